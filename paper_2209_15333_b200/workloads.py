"""Seeded synthetic input generators (NumPy, host) shared by the CUDA path and the test oracle.

This module holds none of the method's arithmetic: it only builds grids (metric fields), gas / scheme
parameters, boundary data and initial conserved fields shaped like the paper's workloads
(PAPER.md:L567-571, L610, L642, L659-667).  The paper's own grids and flow fields are not available
(PAPER.md:L713), so the five BASELINE.json configs below are synthetic stand-ins; DESIGN.md section 5
states each recipe.  The same arrays are handed to both sides, so a generator is never part of parity.

Layout: every field is padded [nz+8][ny+8][nx+8] (x contiguous, 4 ghost layers);
U is [5][nz+8][ny+8][nx+8] with components (rho, rho u, rho v, rho w, E).
Non-dimensional state: rho = T = |u_inf| = 1  =>  p_inf = 1/(gamma Ma^2).
"""
from dataclasses import dataclass, field

import numpy as np

NG = 4


@dataclass
class Case:
    name: str
    nx: int
    ny: int
    nz: int
    grid_kind: str = "uniform"            # "uniform" | "stretched" | "curvilinear"
    dx: float = 1.0
    dy: float = 1.0
    dz: float = 1.0
    metric1d: tuple = None                # stretched: padded 1-D xi_x(i), eta_y(j), zeta_z(k)
    metrics: list = None                  # 10 arrays (nz+8 | 1, ny+8, nx+8): xi_x..zeta_z, J
    gamma: float = 1.4
    Ma: float = 0.1
    Re: float = 1600.0
    Pr: float = 0.72
    T_ref: float = 288.15
    T_suth: float = 110.4
    inviscid: bool = False
    scheme: str = "weno7"                 # "ud7" | "weno7" | "weno5" | "hybrid"
    theta1: float = 0.02
    theta2: float = 0.1
    weno_eps: float = None                # None: set from the grid in __post_init__
    sw_eps: float = 0.0
    bc: list = field(default_factory=lambda: ["periodic"] * 6)
    T_wall: list = field(default_factory=lambda: [1.0] * 6)
    wall_vn: list = field(default_factory=lambda: [None] * 6)
    inflow: list = field(default_factory=lambda: [None] * 6)
    U0: np.ndarray = None
    cfl: float = 0.5
    nsteps: int = 10
    coords: tuple = None                  # optional physical coordinates (x, y, z) of interior points

    def __post_init__(self):
        # The paper prints no WENO epsilon.  The reconstructed quantity is the J^-1-scaled
        # split flux (eq. 6), whose size goes with the cell-face area |grad d|/J, so an absolute 1e-6
        # (Jiang-Shu's value for O(1) data) would swamp the smoothness indicators on fine grids and turn
        # WENO into its linear scheme.  Generators therefore pass eps = 1e-6 * min(|grad d|/J)^2
        # (DESIGN R-10); it is an input of both sides, never part of parity.
        if self.metrics is not None and self.weno_eps is None:
            J = self.metrics[9]
            amin = min(float(np.sqrt(sum((self.metrics[3 * d + c] / J) ** 2 for c in range(3))).min())
                       for d in range(3))
            self.weno_eps = 1e-6 * amin * amin

    @property
    def npoints(self):
        return self.nx * self.ny * self.nz

    @property
    def padded_shape(self):
        return (self.nz + 2 * NG, self.ny + 2 * NG, self.nx + 2 * NG)


# --------------------------------------------------------------------------- helpers
def cons_from_prim(rho, u, v, w, p, gamma):
    """Stack conserved variables (initial-condition bookkeeping only)."""
    return np.stack([rho, rho * u, rho * v, rho * w, p / (gamma - 1.0) + 0.5 * rho * (u * u + v * v + w * w)])


def pad_wrap(a):
    return np.pad(a, NG, mode="wrap")


def uniform_metrics(nx, ny, nz, dx, dy, dz):
    """Metric planes of a uniform Cartesian grid (z-invariant, one padded plane each)."""
    shp = (1, ny + 2 * NG, nx + 2 * NG)
    m = [np.zeros(shp) for _ in range(10)]
    m[0][:] = 1.0 / dx
    m[4][:] = 1.0 / dy
    m[8][:] = 1.0 / dz
    m[9][:] = (1.0 / dx) * (1.0 / dy) * (1.0 / dz)
    return m


def stretched_metrics(kx, ey, zz):
    """Metric fields of a stretched Cartesian grid from padded 1-D xi_x(i), eta_y(j), zeta_z(k).

    Full 3-D fields unless zeta_z is constant (then one plane).  J = xi_x * eta_y * zeta_z (eq. 4)."""
    nxp, nyp, nzp = kx.size, ey.size, zz.size
    planes = 1 if np.all(zz == zz[0]) else nzp
    shp = (planes, nyp, nxp)
    zzp = zz[:planes]
    m = [np.zeros(shp) for _ in range(10)]
    m[0][:] = kx[None, None, :]
    m[4][:] = ey[None, :, None]
    m[8][:] = zzp[:, None, None]
    m[9][:] = (kx[None, None, :] * ey[None, :, None]) * zzp[:, None, None]
    return m


def affine_metrics(nx, ny, nz, A):
    """Constant metrics of the affine map (x,y,z)^T = A (xi,eta,zeta)^T: rows of A^-1, J = det(A^-1)."""
    Ai = np.linalg.inv(np.asarray(A, dtype=np.float64))
    shp = (1, ny + 2 * NG, nx + 2 * NG)
    m = [np.full(shp, Ai[q // 3, q % 3]) for q in range(9)]
    m.append(np.full(shp, np.linalg.det(Ai)))
    return m


def _idx(n):
    return np.arange(-NG, n + NG, dtype=np.float64)


# --------------------------------------------------------------------------- config 1: TGV
def tgv(n=32, seed=20221, scheme="weno7", nsteps=10, perturb=1e-3):
    """3-D Taylor-Green vortex, periodic n^3 on [0,2pi]^3, Ma 0.1, Re 1600 (BASELINE.json config 1)."""
    gamma, Ma = 1.4, 0.1
    h = 2.0 * np.pi / n
    x = h * np.arange(n)
    X = x[None, None, :]
    Y = x[None, :, None]
    Z = x[:, None, None]
    rng = np.random.default_rng(seed)
    u = np.sin(X) * np.cos(Y) * np.cos(Z) + rng.uniform(-perturb, perturb, (n, n, n))
    v = -np.cos(X) * np.sin(Y) * np.cos(Z) + rng.uniform(-perturb, perturb, (n, n, n))
    w = rng.uniform(-perturb, perturb, (n, n, n))
    pinf = 1.0 / (gamma * Ma * Ma)
    p = pinf + (np.cos(2 * X) + np.cos(2 * Y)) * (np.cos(2 * Z) + 2.0) / 16.0
    rho = gamma * Ma * Ma * p  # T = 1
    U = np.stack([pad_wrap(c) for c in cons_from_prim(rho, u, v, w, p + 0 * u, gamma)])
    return Case(name=f"tgv{n}", nx=n, ny=n, nz=n, grid_kind="uniform", dx=h, dy=h, dz=h,
                metrics=uniform_metrics(n, n, n, h, h, h), gamma=gamma, Ma=Ma, Re=1600.0, Pr=0.72,
                T_ref=288.15, scheme=scheme, U0=np.ascontiguousarray(U), cfl=0.5, nsteps=nsteps)


# --------------------------------------------------------------------------- configs 2, 3: HIT
def hit(n=128, Mt=0.5, seed=20222, scheme="weno7", Re_lambda=72.0, k0=4.0, nsteps=100,
        theta1=0.02, theta2=np.inf):
    """Decaying compressible isotropic turbulence, periodic n^3 on [0,2pi]^3 (configs 2 and 3).

    Solenoidal random velocity with shell spectrum E(k) ~ k^4 exp(-2 (k/k0)^2), <u_i u_i> = 3,
    rho = T = 1, Ma = Mt/sqrt(3).  Re from the measured Taylor scale so that Re_lambda is as asked."""
    gamma = 1.4
    rng = np.random.default_rng(seed)
    kf = np.fft.fftfreq(n, 1.0 / n)
    kr = np.fft.rfftfreq(n, 1.0 / n)
    KZ, KY, KX = np.meshgrid(kf, kf, kr, indexing="ij")
    K2 = KX * KX + KY * KY + KZ * KZ
    K = np.sqrt(K2)
    K2s = np.where(K2 == 0, 1.0, K2)
    amp = K * np.exp(-(K / k0) ** 2)          # |u_hat| ~ sqrt(E(k)/(4 pi k^2))
    amp[K > n / 3.0] = 0.0
    a = rng.standard_normal((3,) + K.shape) + 1j * rng.standard_normal((3,) + K.shape)
    kdota = (KX * a[0] + KY * a[1] + KZ * a[2]) / K2s
    uh = [(a[0] - KX * kdota) * amp, (a[1] - KY * kdota) * amp, (a[2] - KZ * kdota) * amp]
    vel = [np.fft.irfftn(c, s=(n, n, n), axes=(0, 1, 2)) for c in uh]
    q2 = sum(np.mean(c * c) for c in vel)
    vel = [c * np.sqrt(3.0 / q2) for c in vel]
    # Taylor scale from the x-derivative of u (spectral), u' = 1
    dudx = np.fft.irfftn(1j * KX * np.fft.rfftn(vel[0], axes=(0, 1, 2)), s=(n, n, n), axes=(0, 1, 2))
    lam = np.sqrt(np.mean(vel[0] ** 2) / np.mean(dudx ** 2))
    uprime = np.sqrt(np.mean(vel[0] ** 2 + vel[1] ** 2 + vel[2] ** 2) / 3.0)
    Re = Re_lambda / (uprime * lam)
    Ma = Mt / np.sqrt(3.0)
    h = 2.0 * np.pi / n
    one = np.ones((n, n, n))
    p = one / (gamma * Ma * Ma)
    U = np.stack([pad_wrap(c) for c in cons_from_prim(one, vel[0], vel[1], vel[2], p, gamma)])
    return Case(name=f"hit{n}_Mt{Mt:g}_{scheme}", nx=n, ny=n, nz=n, grid_kind="uniform", dx=h, dy=h, dz=h,
                metrics=uniform_metrics(n, n, n, h, h, h), gamma=gamma, Ma=Ma, Re=float(Re), Pr=0.72,
                T_ref=288.15, scheme=scheme, theta1=theta1, theta2=theta2,
                U0=np.ascontiguousarray(U), cfl=0.5, nsteps=nsteps)


# --------------------------------------------------------------------------- wall-normal clustering
def _tanh_b(n, Ly, dy1):
    """b of y_j = Ly [1 - tanh(b (1 - j/(n-1)))/tanh b] such that y_1 - y_0 = dy1 (bisection)."""
    def first(b):
        return Ly * (1.0 - np.tanh(b * (1.0 - 1.0 / (n - 1))) / np.tanh(b))
    lo, hi = 1e-3, 20.0
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if first(mid) > dy1:
            lo = mid
        else:
            hi = mid
    return 0.5 * (lo + hi)


def _g_and_dg(j, n, b):
    """g(j) = 1 - tanh(b(1-eta))/tanh b, eta = j/(n-1), and dg/dj; analytic, also outside [0, n-1]."""
    eta = j / (n - 1.0)
    g = 1.0 - np.tanh(b * (1.0 - eta)) / np.tanh(b)
    dg = (b / (n - 1.0)) / np.cosh(b * (1.0 - eta)) ** 2 / np.tanh(b)
    return g, dg


def _blasius_fp(eta):
    """f'(eta) of the Blasius equation f''' + f f''/2 = 0 by RK4 (f''(0) = 0.332057)."""
    def rhs(s):
        return np.array([s[1], s[2], -0.5 * s[0] * s[2]])
    e = np.linspace(0.0, 12.0, 2401)
    s = np.array([0.0, 0.0, 0.332057336])
    out = np.zeros_like(e)
    for q in range(e.size - 1):
        out[q] = s[1]
        hh = e[q + 1] - e[q]
        k1 = rhs(s); k2 = rhs(s + 0.5 * hh * k1); k3 = rhs(s + 0.5 * hh * k2); k4 = rhs(s + hh * k3)
        s = s + hh / 6.0 * (k1 + 2 * k2 + 2 * k3 + k4)
    out[-1] = s[1]
    return np.interp(eta, e, np.minimum(out, 1.0), right=1.0)


def _laminar_profile(y, delta, Tw, gamma, Ma, Pr):
    """Compressible laminar similarity-type profile u(y), T(y): Blasius f' in the Howarth-Dorodnitsyn
    variable, Crocco-Busemann temperature with recovery factor sqrt(Pr) (stand-in, not graded)."""
    Taw = 1.0 + np.sqrt(Pr) * 0.5 * (gamma - 1.0) * Ma * Ma
    eta = np.linspace(0.0, 12.0, 2401)
    fp = _blasius_fp(eta)
    T = Tw + (Taw - Tw) * fp + (1.0 - Taw) * fp * fp
    yphys = np.concatenate([[0.0], np.cumsum(0.5 * (T[1:] + T[:-1]) * np.diff(eta))])
    i99 = np.searchsorted(fp, 0.99)
    yphys *= delta / yphys[i99]
    ya = np.abs(y)
    u = np.interp(ya, yphys, fp, right=1.0) * np.sign(y)
    Tt = np.interp(ya, yphys, T, right=1.0)
    return u, Tt


# --------------------------------------------------------------------------- config 4: flat plate
def flat_plate(nx=1024, ny=128, nz=128, seed=20224, scheme="weno7", nsteps=50, Ly=10.0, dy1=0.004,
               dx=0.1, dz=0.1):
    """Mach 2.9 flat-plate boundary layer on a wall-normal-stretched Cartesian grid (config 4)."""
    gamma, Ma, Re, Pr, T_ref = 1.4, 2.9, 5600.0, 0.72, 108.1
    Tw = 1.0 + np.sqrt(Pr) * 0.5 * (gamma - 1.0) * Ma * Ma
    b = _tanh_b(ny, Ly, dy1)
    g, dg = _g_and_dg(_idx(ny), ny, b)
    y = Ly * g
    ey = 1.0 / (Ly * dg)
    kx = np.full(nx + 2 * NG, 1.0 / dx)
    zz = np.full(nz + 2 * NG, 1.0 / dz)
    u1, T1 = _laminar_profile(y, 1.0, Tw, gamma, Ma, Pr)
    pinf = 1.0 / (gamma * Ma * Ma)
    shp = (nz + 2 * NG, ny + 2 * NG, nx + 2 * NG)
    u = np.broadcast_to(u1[None, :, None], shp).copy()
    T = np.broadcast_to(T1[None, :, None], shp)
    p = np.full(shp, pinf)
    rho = gamma * Ma * Ma * p / T
    zero = np.zeros(shp)
    U = cons_from_prim(rho, u, zero, zero, p, gamma)
    inflow = [None] * 6
    inflow[0] = np.ascontiguousarray(U[:, :, :, NG])         # [5][nz+8][ny+8]
    # blowing / suction strip on the wall (stand-in for ref. [32], formula not in the paper)
    rng = np.random.default_rng(seed)
    xs = dx * _idx(nx)
    zs = dz * _idx(nz)
    win = np.where((xs >= 10.0) & (xs <= 20.0), np.sin(np.pi * (xs - 10.0) / 10.0) ** 2, 0.0)
    Lz = dz * nz
    span = np.zeros_like(zs)
    for m in range(1, 4):
        span += rng.uniform(0.5, 1.0) * np.sin(2.0 * np.pi * m * zs / Lz + rng.uniform(0, 2 * np.pi)) / 3.0
    wall_vn = [None] * 6
    wall_vn[2] = np.ascontiguousarray(0.04 * span[:, None] * win[None, :])   # [nz+8][nx+8]
    T_wall = [1.0] * 6
    T_wall[2] = Tw
    return Case(name=f"plate{nx}x{ny}x{nz}", nx=nx, ny=ny, nz=nz, grid_kind="stretched",
                dx=dx, dy=1.0, dz=dz, metric1d=(kx, ey, zz), metrics=stretched_metrics(kx, ey, zz),
                gamma=gamma, Ma=Ma, Re=Re, Pr=Pr, T_ref=T_ref, scheme=scheme,
                bc=["inflow", "outflow", "wall", "outflow", "periodic", "periodic"],
                T_wall=T_wall, wall_vn=wall_vn, inflow=inflow, U0=np.ascontiguousarray(U),
                cfl=0.5, nsteps=nsteps)


# --------------------------------------------------------------------------- config 5: ramp
def ramp(nx=2048, ny=300, nz=256, seed=20225, scheme="hybrid", theta2=np.inf, nsteps=20, dz=0.1,
         x0=-120.0, x1=84.8, H=60.0, dy1=0.004, nmodes=64, rms=0.05, nshocks=1):
    """Mach 2.9, 24-degree compression-ramp-shaped curvilinear grid, z-extruded 2-D map (config 5).

    Wall y_w(x) = tan24 (x + sqrt(x^2 + d^2))/2 - tan24 d/2 (smoothed corner, d = 2), x uniform,
    y = y_w + (H - y_w) g(eta), tanh clustering g as config 4; metrics analytic via eq. 3-4.

    nshocks > 1 adds a train of nshocks - 1 weak oblique fronts upstream of the ramp shock (normal Mach numbers 1.05 to
    1.35, Rankine-Hugoniot jumps, smeared like the main shock): a stand-in for the shocklets / shock systems that make
    "up to 10 %" of the interfaces leave the linear scheme, used by the bench workloads that measure the
    hybrid kernels at that flagged fraction.  nshocks = 1 is BASELINE.json's config 5."""
    gamma, Ma, Re, Pr, T_ref = 1.4, 2.9, 5600.0, 0.72, 108.1
    Tw = 1.0 + np.sqrt(Pr) * 0.5 * (gamma - 1.0) * Ma * Ma
    dxx = (x1 - x0) / nx
    xs = x0 + dxx * _idx(nx)
    tanA, dl = np.tan(np.deg2rad(24.0)), 2.0
    yw = tanA * 0.5 * (xs + np.sqrt(xs * xs + dl * dl)) - tanA * dl / 2.0
    dyw = tanA * 0.5 * (1.0 + xs / np.sqrt(xs * xs + dl * dl))
    b = _tanh_b(ny, H, dy1)
    g, dg = _g_and_dg(_idx(ny), ny, b)
    Y = yw[None, :] + (H - yw[None, :]) * g[:, None]                 # [ny+8][nx+8]
    y_xi = dyw[None, :] * dxx * (1.0 - g[:, None])
    y_eta = (H - yw[None, :]) * dg[:, None]
    x_xi = dxx
    shp2 = (1, ny + 2 * NG, nx + 2 * NG)
    m = [np.zeros(shp2) for _ in range(10)]
    m[0][0] = 1.0 / x_xi
    m[3][0] = -y_xi / (x_xi * y_eta)
    m[4][0] = 1.0 / y_eta
    m[8][0] = 1.0 / dz
    m[9][0] = 1.0 / (x_xi * y_eta * dz)
    # turbulent-like mean profile: 1/7 power law + Crocco-Busemann temperature, delta = 6.5 mm
    delta = 6.5
    dist = (Y - yw[None, :]) * np.cos(np.arctan(dyw))[None, :]          # approx. wall distance
    s = np.clip(np.abs(dist) / delta, 0.0, 1.0)
    um = s ** (1.0 / 7.0) * np.sign(dist)
    Taw = Tw
    Tm = Tw + (Taw - Tw) * np.abs(um) + (1.0 - Taw) * um * um
    pinf = 1.0 / (gamma * Ma * Ma)
    # velocity fluctuations: random Fourier modes, separable in (x,y) x z, windowed to the layer
    rng = np.random.default_rng(seed)
    Lz = dz * nz
    zs = dz * _idx(nz)
    S = np.zeros((3, nmodes) + Y.shape)
    Zm = np.zeros((nmodes, zs.size))
    wind = np.exp(-((dist / delta - 0.5) / 0.4) ** 2) * (dist > 0)
    for q in range(nmodes):
        kxm = 2.0 * np.pi / delta * rng.uniform(0.3, 2.0)
        kym = 2.0 * np.pi / delta * rng.uniform(0.3, 2.0)
        kzm = 2.0 * np.pi * rng.integers(1, 13) / Lz
        ph = rng.uniform(0, 2 * np.pi, 4)
        amp = rng.standard_normal(3)
        base = np.sin(kxm * xs[None, :] + kym * Y + ph[0])
        for c in range(3):
            S[c, q] = amp[c] * base * wind
        Zm[q] = np.cos(kzm * zs + ph[1])
    shp = (nz + 2 * NG, ny + 2 * NG, nx + 2 * NG)
    fl = [(Zm.T @ S[c].reshape(nmodes, -1)).reshape(shp) for c in range(3)]
    del S
    sc = rms / np.sqrt(np.mean(fl[0][:, wind > 0.5] ** 2) + 1e-300)
    cosw = 1.0 / np.sqrt(1.0 + dyw * dyw)
    sinw = dyw * cosw
    u = (um * cosw[None, :])[None] + sc * fl[0]
    v = (um * sinw[None, :])[None] + sc * fl[1]
    w = sc * fl[2]
    del fl
    # the ramp's oblique shock (weak solution of the theta-beta-M relation for a 24 degree turn), smeared over
    # about three cells with a tanh profile: it is what the shock sensor of the hybrid scheme has to find
    turn = np.deg2rad(24.0)
    lo, hi = np.arcsin(1.0 / Ma) + 1e-6, np.deg2rad(64.0)
    for _ in range(100):
        beta = 0.5 * (lo + hi)
        tb = 2.0 / np.tan(beta) * (Ma ** 2 * np.sin(beta) ** 2 - 1.0) / (Ma ** 2 * (gamma + np.cos(2 * beta)) + 2.0)
        lo, hi = (beta, hi) if tb < np.tan(turn) else (lo, beta)
    m1n2 = (Ma * np.sin(beta)) ** 2
    p_ratio = 1.0 + 2.0 * gamma / (gamma + 1.0) * (m1n2 - 1.0)
    r_ratio = (gamma + 1.0) * m1n2 / ((gamma - 1.0) * m1n2 + 2.0)
    v_ratio = np.sqrt(np.cos(beta) ** 2 + (np.sin(beta) / r_ratio) ** 2)
    dsh = (np.tan(beta) * xs[None, :] - Y) * np.cos(beta)              # > 0 behind the shock
    sh = 0.5 * (1.0 + np.tanh(dsh / (1.5 * dxx)))
    fp_, ft_, fv_ = 1.0 + (p_ratio - 1.0) * sh, 1.0 + (p_ratio / r_ratio - 1.0) * sh, 1.0 + (v_ratio - 1.0) * sh
    for q in range(1, nshocks):
        m1n = 1.05 + 0.1 * (q % 4)                                      # normal Mach number of front q
        bq = np.arcsin(m1n / Ma)
        pq = 1.0 + 2.0 * gamma / (gamma + 1.0) * (m1n ** 2 - 1.0)
        rq = (gamma + 1.0) * m1n ** 2 / ((gamma - 1.0) * m1n ** 2 + 2.0)
        vq = np.sqrt(np.cos(bq) ** 2 + (np.sin(bq) / rq) ** 2)
        xq = -q * 110.0 / nshocks                                       # foot of the front on the plate, upstream
        dq = (np.tan(bq) * (xs[None, :] - xq) - Y) * np.cos(bq)
        sq = 0.5 * (1.0 + np.tanh(dq / (1.5 * dxx)))
        fp_ = fp_ * (1.0 + (pq - 1.0) * sq)
        ft_ = ft_ * (1.0 + (pq / rq - 1.0) * sq)
        fv_ = fv_ * (1.0 + (vq - 1.0) * sq)
    u *= fv_[None]
    v *= fv_[None]
    w *= fv_[None]
    T = np.broadcast_to((Tm * ft_)[None], shp)
    p = np.broadcast_to((pinf * fp_)[None], shp)
    rho = gamma * Ma * Ma * p / T
    U = cons_from_prim(rho, u, v, w, p, gamma)
    inflow = [None] * 6
    inflow[0] = np.ascontiguousarray(U[:, :, :, NG])
    T_wall = [1.0] * 6
    T_wall[2] = Tw
    return Case(name=f"ramp{nx}x{ny}x{nz}", nx=nx, ny=ny, nz=nz, grid_kind="curvilinear",
                dx=dxx, dy=1.0, dz=dz, metrics=m, gamma=gamma, Ma=Ma, Re=Re, Pr=Pr, T_ref=T_ref,
                scheme=scheme, theta1=0.02, theta2=theta2,
                bc=["inflow", "outflow", "wall", "outflow", "periodic", "periodic"],
                T_wall=T_wall, inflow=inflow, U0=np.ascontiguousarray(U), cfl=0.5, nsteps=nsteps)


# --------------------------------------------------------------------------- pin / parity helpers
def vortex_fields(X, Y, gamma, Ma, uinf, vinf, xc, yc, L, beta=5.0):
    """Isentropic vortex (A.10) evaluated at (X,Y) with periodic images of period L."""
    dxp = (X - xc + 0.5 * L) % L - 0.5 * L
    dyp = (Y - yc + 0.5 * L) % L - 0.5 * L
    r2 = dxp * dxp + dyp * dyp
    T = 1.0 - (gamma - 1.0) * Ma * Ma * beta * beta * np.exp(1.0 - r2) / (8.0 * np.pi ** 2)
    rho = T ** (1.0 / (gamma - 1.0))
    p = rho * T / (gamma * Ma * Ma)
    u = uinf - beta / (2 * np.pi) * np.exp(0.5 * (1.0 - r2)) * dyp
    v = vinf + beta / (2 * np.pi) * np.exp(0.5 * (1.0 - r2)) * dxp
    return rho, u, v, p


def vortex(n=32, nz=4, L=10.0, Ma=0.5, uinf=1.0, vinf=0.5, scheme="ud7", A=None, t=0.0):
    """Isentropic vortex on a periodic L x L (x nz h) box; optional affine map A (3x3, in units of h)."""
    gamma = 1.4
    h = L / n
    ii, jj, kk = _idx(n), _idx(n), _idx(nz)
    KK, JJ, II = np.meshgrid(kk, jj, ii, indexing="ij")
    if A is None:
        X, Y = h * II, h * JJ
        met = uniform_metrics(n, n, nz, h, h, h)
        kind = "uniform"
    else:
        A = np.asarray(A, dtype=np.float64) * h
        X = A[0, 0] * II + A[0, 1] * JJ + A[0, 2] * KK
        Y = A[1, 0] * II + A[1, 1] * JJ + A[1, 2] * KK
        met = affine_metrics(n, n, nz, A)
        kind = "curvilinear"
    rho, u, v, p = vortex_fields(X, Y, gamma, Ma, uinf, vinf, 0.5 * L + uinf * t, 0.5 * L + vinf * t, L)
    U = cons_from_prim(rho, u, v, np.zeros_like(u), p, gamma)
    return Case(name=f"vortex{n}", nx=n, ny=n, nz=nz, grid_kind=kind, dx=h, dy=h, dz=h, metrics=met,
                gamma=gamma, Ma=Ma, inviscid=True, scheme=scheme, U0=np.ascontiguousarray(U),
                coords=(X, Y, None))


def smooth_periodic(nx=20, ny=16, nz=12, seed=7, scheme="weno7", Ma=0.8, amp=0.2, inviscid=False,
                    grid="uniform", Re=200.0):
    """Smooth random periodic state (a few seeded Fourier modes per primitive) for parity and invariants.

    grid: "uniform", "stretched" (smooth periodic 1-D stretching) or "wavy" (smooth periodic 3-D
    curvilinear map with all nine metrics populated)."""
    gamma = 1.4
    rng = np.random.default_rng(seed)
    # everything is evaluated on interior indices and wrapped into the ghosts, so it is exactly periodic
    KK, JJ, II = np.meshgrid(np.arange(nz, dtype=np.float64), np.arange(ny, dtype=np.float64),
                             np.arange(nx, dtype=np.float64), indexing="ij")
    a, bq, c = 2 * np.pi * II / nx, 2 * np.pi * JJ / ny, 2 * np.pi * KK / nz

    def field(mean, amplitude):
        f = np.full(II.shape, mean)
        for _ in range(4):
            m = rng.integers(0, 3, 3)
            f = f + amplitude * rng.uniform(-1, 1) * np.cos(m[0] * a + m[1] * bq + m[2] * c + rng.uniform(0, 2 * np.pi))
        return f
    rho = field(1.0, amp * 0.3)
    T = field(1.0, amp * 0.3)
    u, v, w = field(1.0, amp), field(-0.3, amp), field(0.2, amp)
    p = rho * T / (gamma * Ma * Ma)
    U = np.stack([pad_wrap(q) for q in cons_from_prim(rho, u, v, w, p, gamma)])
    hx, hy, hz = 2 * np.pi / nx, 2 * np.pi / ny, 2 * np.pi / nz
    kw = dict(dx=hx, dy=hy, dz=hz)
    metric1d = None
    coords = (hx * II, hy * JJ, hz * KK)
    if grid == "uniform":
        met = uniform_metrics(nx, ny, nz, hx, hy, hz)
        kind = "uniform"
    elif grid == "stretched":
        ia, ja, ka = 2 * np.pi * np.arange(nx) / nx, 2 * np.pi * np.arange(ny) / ny, 2 * np.pi * np.arange(nz) / nz
        kx = np.pad(1.0 / (hx * (1.0 + 0.3 * np.cos(ia))), NG, mode="wrap")
        ey = np.pad(1.0 / (hy * (1.0 + 0.2 * np.sin(ja))), NG, mode="wrap")
        zz = np.pad(1.0 / (hz * (1.0 - 0.25 * np.cos(ka + 0.5))), NG, mode="wrap")
        metric1d = (kx, ey, zz)
        met = stretched_metrics(kx, ey, zz)
        kind = "stretched"
        coords = (hx * (II + 0.3 * nx / (2 * np.pi) * np.sin(a)), hy * (JJ - 0.2 * ny / (2 * np.pi) * np.cos(bq)),
                  hz * (KK - 0.25 * nz / (2 * np.pi) * np.sin(c + 0.5)))
    elif grid == "wavy":
        # x = hx i + e sin(b) sin(c), y = hy j + e sin(a) sin(c), z = hz k + e sin(a) sin(b); analytic Jacobian
        e = 0.08
        sa, sb, sc_ = np.sin(a), np.sin(bq), np.sin(c)
        ca, cb, cc = np.cos(a), np.cos(bq), np.cos(c)
        da, db, dc = 2 * np.pi / nx, 2 * np.pi / ny, 2 * np.pi / nz
        Jm = np.empty(II.shape + (3, 3))
        Jm[..., 0, 0] = hx;               Jm[..., 0, 1] = e * cb * sc_ * db;  Jm[..., 0, 2] = e * sb * cc * dc
        Jm[..., 1, 0] = e * ca * sc_ * da; Jm[..., 1, 1] = hy;                Jm[..., 1, 2] = e * sa * cc * dc
        Jm[..., 2, 0] = e * ca * sb * da;  Jm[..., 2, 1] = e * sa * cb * db;  Jm[..., 2, 2] = hz
        Ji = np.linalg.inv(Jm)
        met = [np.ascontiguousarray(pad_wrap(Ji[..., q // 3, q % 3])) for q in range(9)]
        met.append(np.ascontiguousarray(pad_wrap(np.linalg.det(Ji))))
        kind = "curvilinear"
        coords = (hx * II + e * sb * sc_, hy * JJ + e * sa * sc_, hz * KK + e * sa * sb)
    else:
        raise ValueError(grid)
    return Case(name=f"smooth_{grid}_{scheme}", nx=nx, ny=ny, nz=nz, grid_kind=kind, metric1d=metric1d,
                metrics=met, gamma=gamma, Ma=Ma, Re=Re, Pr=0.72, inviscid=inviscid, scheme=scheme,
                U0=np.ascontiguousarray(U), coords=coords, **kw)


def sod(n=200, scheme="weno7", ny=4, nz=4):
    """1-D Sod shock tube along x on [0,1] (rho,p = 1,1 | 0.125,0.1), outflow ends, inviscid.

    Solver units: Ma = 1/sqrt(gamma) so that p = rho T (T = p/rho)."""
    gamma = 1.4
    Ma = 1.0 / np.sqrt(gamma)
    h = 1.0 / n
    x = h * (_idx(n) + 0.5)
    shp = (nz + 2 * NG, ny + 2 * NG, n + 2 * NG)
    left = np.broadcast_to((x < 0.5)[None, None, :], shp)
    rho = np.where(left, 1.0, 0.125)
    p = np.where(left, 1.0, 0.1)
    z = np.zeros(shp)
    U = cons_from_prim(rho, z, z, z, p, gamma)
    return Case(name=f"sod{n}", nx=n, ny=ny, nz=nz, grid_kind="uniform", dx=h, dy=h, dz=h,
                metrics=uniform_metrics(n, ny, nz, h, h, h), gamma=gamma, Ma=Ma, inviscid=True, scheme=scheme,
                bc=["outflow", "outflow", "periodic", "periodic", "periodic", "periodic"],
                U0=np.ascontiguousarray(U), coords=(x, None, None))


def shocked_periodic(n=24, seed=11, scheme="hybrid", theta1=0.02, theta2=0.1, steep=6.0):
    """Periodic box with a smooth background plus steep pressure/density fronts, so that all three
    levels of the hybrid scheme are exercised.  `steep` sets the front thickness (in units of the box,
    so a bench-sized box passes steep ~ n/7 to keep the fronts a few cells thick)."""
    c = smooth_periodic(n, n, n, seed=seed, scheme=scheme, Ma=1.2, amp=0.15, inviscid=False)
    KK, JJ, II = np.meshgrid(_idx(n), _idx(n), _idx(n), indexing="ij")
    s = 2 * np.pi / n
    front = 0.5 * (1.0 + np.tanh(steep * np.sin(s * II + 0.7 * np.sin(s * JJ)) * np.cos(s * KK * 1.0 + 0.3)))
    U = c.U0.copy()
    fac = 1.0 + 1.5 * front
    U[0] *= fac
    U[1] *= fac
    U[2] *= fac
    U[3] *= fac
    U[4] *= fac * (1.0 + 0.8 * front)
    c.U0 = np.ascontiguousarray(U)
    c.scheme, c.theta1, c.theta2 = scheme, theta1, theta2
    c.name = f"shocked{n}_{scheme}"
    return c
