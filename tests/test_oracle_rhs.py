"""Whole-RHS pins of the oracle: freestream, conservation, symmetry / metric wiring, hybrid limits,
sensor.  CPU only."""
import numpy as np
import pytest

from oracle.oracle import Oracle
from paper_2209_15333_b200 import workloads as W

NG = 4
INT = (slice(None), slice(NG, -NG), slice(NG, -NG), slice(NG, -NG))
SCHEMES = ["ud7", "weno7", "weno5", "hybrid"]


def uniform_state(case, vel=(0.8, -0.3, 0.45), rho=1.1, T=0.9):
    shp = case.padded_shape
    p = rho * T / (case.gamma * case.Ma ** 2)
    one = np.ones(shp)
    return np.ascontiguousarray(W.cons_from_prim(rho * one, vel[0] * one, vel[1] * one, vel[2] * one, p * one, case.gamma))


# ------------------------------------------------------------------ freestream
@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("grid", ["uniform", "stretched", "affine"])
def test_freestream_is_preserved_to_roundoff(grid, scheme):
    case = W.smooth_periodic(12, 10, 8, grid="uniform" if grid == "affine" else grid, scheme=scheme)
    if grid == "affine":
        h = case.dx
        case.metrics = W.affine_metrics(case.nx, case.ny, case.nz,
                                        h * np.array([[1.0, 0.6, 0.1], [-0.2, 0.9, 0.5], [0.3, -0.4, 1.1]]))
    U = uniform_state(case)
    dU = Oracle(case).rhs(U)[INT]
    flux_scale = np.abs(U).max() * max(np.abs(m).max() for m in case.metrics[:9])
    assert np.abs(dU).max() <= 1e-12 * flux_scale
    # the viscous part alone is exactly zero for uniform flow
    case.inviscid = True
    assert np.array_equal(Oracle(case).rhs(U)[INT], dU)


def test_freestream_residual_on_a_curved_grid_is_truncation_level():
    """DESIGN R-18: with analytic metrics and a nonlinear upwind split there is no discrete GCL, so on a
    truly curved grid the uniform-flow residual is truncation error; it must fall at >= 5th order."""
    res = []
    for n in (12, 24):
        case = W.smooth_periodic(n, n, n, grid="wavy", scheme="ud7", inviscid=True)
        dU = Oracle(case).rhs(uniform_state(case))[INT]
        res.append(np.abs(dU).max())
    assert res[1] < 1e-4
    assert res[0] / res[1] > 2.0 ** 5


# ------------------------------------------------------------------ conservation
@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("grid", ["uniform", "stretched", "wavy"])
def test_periodic_conservation(grid, scheme):
    case = W.smooth_periodic(12, 10, 8, grid=grid, scheme=scheme, Re=80.0)
    o = Oracle(case)
    U = o.fill_ghosts(case.U0.copy())
    dU = o.rhs(U)[INT]
    J = np.broadcast_to(case.metrics[9], case.padded_shape)[NG:-NG, NG:-NG, NG:-NG]
    for m in range(5):
        tot = np.sum(dU[m] / J)
        assert abs(tot) <= 1e-12 * np.sum(np.abs(dU[m] / J)) + 1e-13, (m, tot)


# ------------------------------------------------------------------ symmetry / wiring
def test_axis_relabelling_gives_the_same_rhs():
    """x = h eta, y = h zeta, z = h xi: the same flow seen through permuted computational axes must give
    the permuted RHS to round-off.  A swapped eta/zeta label (DESIGN R-4) fails this."""
    case = W.smooth_periodic(10, 12, 14, grid="uniform", scheme="weno7", Re=60.0)
    h = (case.dx, case.dy, case.dz)
    o = Oracle(case)
    U = o.fill_ghosts(case.U0.copy())
    dU = o.rhs(U)
    Up = np.ascontiguousarray(np.transpose(U, (0, 2, 3, 1)))      # U'[k',j',i'] = U[i',k',j']
    nzp, nyp, nxp = Up.shape[1:]
    c2 = W.smooth_periodic(nxp - 2 * NG, nyp - 2 * NG, nzp - 2 * NG, grid="uniform", scheme="weno7", Re=60.0)
    met = [np.zeros((1, nyp, nxp)) for _ in range(10)]
    # xi' runs along physical z, eta' along x, zeta' along y
    met[2][:] = 1.0 / h[2]
    met[3][:] = 1.0 / h[0]
    met[7][:] = 1.0 / h[1]
    met[9][:] = case.metrics[9].ravel()[0]
    c2.metrics = met
    c2.grid_kind = "curvilinear"
    dUp = Oracle(c2).rhs(Up)
    ref = np.transpose(dU, (0, 2, 3, 1))
    assert np.abs(dUp[INT] - ref[INT]).max() <= 1e-12 * np.abs(ref[INT]).max()


@pytest.mark.parametrize("scheme", ["ud7", "weno7", "weno5"])
def test_mirror_symmetry_pins_the_negative_flux_stencil(scheme):
    """Reflect x -> -x (u -> -u): the RHS must be the reflected RHS.  A wrong mirror of the f- stencil
    (f-_{j+4} ... f-_{j-2}) breaks this."""
    case = W.smooth_periodic(14, 8, 6, grid="uniform", scheme=scheme, Re=60.0)
    o = Oracle(case)
    U = o.fill_ghosts(case.U0.copy())
    dU = o.rhs(U)
    Ur = np.ascontiguousarray(U[:, :, :, ::-1])
    Ur[1] *= -1.0
    dUr = o.rhs(Ur)
    ref = dU[:, :, :, ::-1].copy()
    ref[1] *= -1.0
    assert np.abs(dUr[INT] - ref[INT]).max() <= 1e-12 * np.abs(ref[INT]).max()


@pytest.mark.parametrize("option", ["default", "char_recon", "bc_closure", "visc_order8", "all"])
def test_rhs_point_equals_rhs_everywhere_small(option):
    """ora_rhs_point (the sampled-parity entry) is ora_rhs bit for bit, with every option the full-size GPU tests may
    switch on: characteristic variables, the paper's boundary scheme, the 8th-order viscous scheme."""
    for bc_case in ("periodic", "plate", "ramp"):
        if bc_case == "periodic":
            case = W.shocked_periodic(10)
        elif bc_case == "plate":
            case = W.flat_plate(nx=12, ny=10, nz=8, scheme="hybrid")
        else:
            case = W.ramp(nx=12, ny=10, nz=8, nmodes=4, theta2=0.1)
        if option in ("char_recon", "all"):
            case.char_recon = 1
        if option in ("bc_closure", "all"):
            case.bc_closure = 1
        if option in ("visc_order8", "all"):
            case.visc_order = 8
        o = Oracle(case)
        U = o.fill_ghosts(case.U0.copy())
        dU = o.rhs(U)
        ijk = np.array([(i, j, k) for k in range(case.nz) for j in range(case.ny) for i in range(case.nx)], dtype=np.int32)
        pts = o.rhs_points(U, ijk)
        ref = np.stack([dU[m][ijk[:, 2] + NG, ijk[:, 1] + NG, ijk[:, 0] + NG] for m in range(5)], axis=1)
        assert np.array_equal(pts, ref)


def test_rhs_is_a_pure_function_and_leaves_ghosts_alone():
    case = W.smooth_periodic(8, 8, 8)
    o = Oracle(case)
    U = o.fill_ghosts(case.U0.copy())
    U_before = U.copy()
    a, b = o.rhs(U), o.rhs(U)
    assert np.array_equal(a, b) and np.array_equal(U, U_before)
    ghost = np.ones(U.shape, dtype=bool)
    ghost[INT] = False
    assert np.all(a[ghost] == 0.0)


def test_directional_terms_sum_to_inviscid_rhs():
    case = W.smooth_periodic(10, 8, 6, grid="wavy", scheme="weno7", inviscid=True)
    o = Oracle(case)
    U = o.fill_ghosts(case.U0.copy())
    parts = [o.inviscid_dir(U, d) for d in range(3)]
    tot = o.rhs(U)
    assert np.abs((parts[0] + parts[1] + parts[2] - tot)[INT]).max() <= 1e-13 * np.abs(tot[INT]).max()


# ------------------------------------------------------------------ hybrid
def test_hybrid_limits_are_bitwise_the_single_schemes():
    base = W.shocked_periodic(10)
    U = Oracle(base).fill_ghosts(base.U0.copy())
    for (t1, t2), single in (((np.inf, np.inf), "ud7"), ((-1.0, np.inf), "weno7"), ((-1.0, -1.0), "weno5")):
        base.scheme, base.theta1, base.theta2 = "hybrid", t1, t2
        a = Oracle(base).rhs(U)
        base.scheme = single
        b = Oracle(base).rhs(U)
        assert np.array_equal(a, b), single


def test_sensor_formula_and_flags():
    thr = [float(t) for t in open(__file__.replace("test_oracle_rhs.py", "golden/hybrid_thresholds.txt")).read().split("\n")[1].split()]
    case = W.shocked_periodic(12, theta1=thr[0], theta2=thr[1])
    o = Oracle(case)
    U = o.fill_ghosts(case.U0.copy())
    th = o.sensor(U)
    g = case.gamma
    p = (g - 1.0) * (U[4] - 0.5 * (U[1] ** 2 + U[2] ** 2 + U[3] ** 2) / U[0])
    rng = np.random.default_rng(0)
    for _ in range(30):
        i, j, k = (int(rng.integers(0, 12)) + NG for _ in range(3))
        ref = 0.0
        for ax in range(3):
            d = [0, 0, 0]
            d[ax] = 1
            pm, pp = p[k - d[0], j - d[1], i - d[2]], p[k + d[0], j + d[1], i + d[2]]
            ref += abs(-pm + 2 * p[k, j, i] - pp) / (pm + 2 * p[k, j, i] + pp)       # eq. 42
        assert th[k, j, i] == pytest.approx(ref, rel=1e-12)
    # ghosts of theta wrap on periodic axes
    assert np.array_equal(th[NG:-NG, NG:-NG, 0:NG], th[NG:-NG, NG:-NG, -2 * NG:-NG])
    # interface flags: max of the two neighbours against the printed thresholds
    fl = o.flags(th, 0)
    a, b = th[NG:-NG, NG:-NG, NG - 1:-NG], th[NG:-NG, NG:-NG, NG:-NG + 1]
    Th = np.maximum(a, b)
    ref = np.where(Th <= thr[0], 0, np.where(Th <= thr[1], 1, 2))
    assert np.array_equal(fl[NG:-NG, NG:-NG, NG - 1:-NG], ref)
    counts = np.bincount(ref.ravel(), minlength=3)
    assert np.all(counts > 0), counts           # the case exercises all three levels
