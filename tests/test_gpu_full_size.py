"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (same generators, same C-ABI
calls): one `ocfd_rhs` on the full grid, compared with the CPU oracle on SAMPLED outputs that the oracle computes one
by one from U alone (`ora_rhs_points`, which a CPU test proves bit-identical to the array version), plus the whole
array where the oracle finishes in seconds (config 2, 128^3).

The sample is seeded and stratified: uniform random interior points, every corner, and points drawn from the first /
last 8 layers of each direction (where ghost cells, wall closures and ragged tiles live).  The oracle's inputs never
come from the CUDA path: ghosts are filled by the oracle itself.

Error metric as in test_gpu_parity.py: per component, max over the sample of |gpu - ora| divided by
max(max_sample |ora|, 1e-3 Lambda max|U|); bar 1e-11 (north_star).
"""
import numpy as np
import pytest

from paper_2209_15333_b200 import workloads as W

pytestmark = pytest.mark.gpu

NG = 4
TOL_RHS = 1e-11


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_2209_15333_b200 import binding
    binding.load()
    return binding


@pytest.fixture(scope="module")
def Oracle():
    from oracle.oracle import Oracle
    return Oracle


def sample_points(case, n_random, n_face, seed):
    rng = np.random.default_rng(seed)
    n = (case.nx, case.ny, case.nz)
    pts = [rng.integers(0, n, size=(n_random, 3))]
    pts.append(np.array([(i, j, k) for i in (0, n[0] - 1) for j in (0, n[1] - 1) for k in (0, n[2] - 1)]))
    for d in range(3):
        for lo in (True, False):
            q = rng.integers(0, n, size=(n_face, 3))
            layer = rng.integers(0, 8, size=n_face)
            q[:, d] = layer if lo else n[d] - 1 - layer
            pts.append(q)
    return np.unique(np.concatenate(pts).astype(np.int32), axis=0)


def sampled_rhs_error(B, Oracle, case, seed, n_random=3000, n_face=400):
    import torch
    o = Oracle(case)
    U = o.fill_ghosts(case.U0.copy())
    lam = o.max_wavespeed(U)
    ijk = sample_points(case, n_random, n_face, seed)
    ref = o.rhs_points(U, ijk)                                     # [n, 5]
    s = B.Solver(case)
    Ud = s.to_device(U)
    dUd = s.rhs(Ud)
    idx = torch.as_tensor(ijk.astype(np.int64) + NG, device=dUd.device)
    got = dUd[:, idx[:, 2], idx[:, 1], idx[:, 0]].T.cpu().numpy()  # [n, 5]
    assert bool(torch.isfinite(dUd[:, NG:-NG, NG:-NG, NG:-NG]).all())
    s.close()
    floor = 1e-3 * lam * np.abs(U[:, NG:-NG, NG:-NG, NG:-NG]).max()
    err = np.array([np.abs(got[:, m] - ref[:, m]).max() / max(np.abs(ref[:, m]).max(), floor) for m in range(5)])
    return err, ijk.shape[0]


def test_config5_ramp_full_size_sampled(B, Oracle):
    case = W.ramp()                                                # 2048 x 300 x 256, hybrid: bench.py's default workload
    assert (case.nx, case.ny, case.nz) == (2048, 300, 256)
    err, n = sampled_rhs_error(B, Oracle, case, seed=55)
    print(f"config 5 (ramp 2048x300x256, hybrid): {n} sampled points, rel Linf per component {err}")
    assert err.max() <= TOL_RHS


def test_config4_flat_plate_full_size_sampled(B, Oracle):
    case = W.flat_plate()                                          # 1024 x 128 x 128, WENO7
    assert (case.nx, case.ny, case.nz) == (1024, 128, 128)
    err, n = sampled_rhs_error(B, Oracle, case, seed=44)
    print(f"config 4 (plate 1024x128x128, WENO7): {n} sampled points, rel Linf per component {err}")
    assert err.max() <= TOL_RHS


def test_config3_shocklet_hit256_full_size_sampled(B, Oracle):
    case = W.hit(256, Mt=1.0, seed=20223, scheme="hybrid", nsteps=50)
    err, n = sampled_rhs_error(B, Oracle, case, seed=33)
    print(f"config 3 (HIT 256^3, hybrid): {n} sampled points, rel Linf per component {err}")
    assert err.max() <= TOL_RHS


def full_size_flag_report(B, Oracle, case):
    """ocfd_debug_sensor against ora_sensor / ora_flags on the whole grid (north_star: decisions must match at every
    point except those within 1e-12 of a threshold, which are counted and reported; eq. 42)."""
    import torch
    from tests.parity_utils import compare_flags
    o = Oracle(case)
    U = o.fill_ghosts(case.U0.copy())
    th_ref = o.sensor(U)
    fl_ref = [o.flags(th_ref, d) for d in range(3)]
    s = B.Solver(case)
    Ud = s.to_device(U)
    del U
    th_gpu, fl_gpu = s.debug_sensor(Ud)
    torch.cuda.synchronize()
    I = slice(NG, -NG)
    dth = float((th_gpu[I, I, I].cpu() - torch.from_numpy(th_ref[I, I, I])).abs().max())
    fl_gpu = fl_gpu.cpu().numpy()
    del th_gpu, Ud
    s.close()
    bad, near, total, hist = compare_flags(th_ref, fl_ref, fl_gpu, case.theta1, case.theta2)
    print(f"{case.name}: {total} interfaces, max |theta_gpu - theta_ora| {dth:.2e}, {near} within 1e-12 of a threshold "
          f"(excluded), {bad} mismatches outside the band; UD7/WENO7/WENO5 = {hist.tolist()} "
          f"({100.0 * (hist[1] + hist[2]) / hist.sum():.2f} % flagged)")
    assert dth <= 1e-13
    assert bad == 0
    return hist


@pytest.mark.parametrize("theta2", [np.inf, 0.1])
def test_config5_ramp_full_size_sensor_decisions(B, Oracle, theta2):
    hist = full_size_flag_report(B, Oracle, W.ramp(theta2=theta2))
    assert hist[1] > 0 and (np.isinf(theta2) or hist[2] > 0)


@pytest.mark.parametrize("theta2", [np.inf, 0.1])
def test_config3_shocklet_hit256_full_size_sensor_decisions(B, Oracle, theta2):
    full_size_flag_report(B, Oracle, W.hit(256, Mt=1.0, seed=20223, scheme="hybrid", nsteps=50, theta2=theta2))


def test_config2_hit128_whole_array_rhs_and_three_steps(B, Oracle):
    case = W.hit(128)                                              # WENO7
    o = Oracle(case)
    U = o.fill_ghosts(case.U0.copy())
    dt = case.cfl / o.max_wavespeed(U)
    ref = o.rhs(U)
    s = B.Solver(case)
    Ud = s.to_device(U)
    got = s.rhs(Ud).cpu().numpy()
    I = (slice(None), slice(NG, -NG), slice(NG, -NG), slice(NG, -NG))
    err = max(np.abs(got[I][m] - ref[I][m]).max() / np.abs(ref[I][m]).max() for m in range(5))
    print("config 2 (HIT 128^3, WENO7): whole-array RHS rel Linf", err)
    assert err <= TOL_RHS
    for _ in range(3):
        o.rk3_step(U, dt)
        s.rk3_step(Ud, dt)
    got = Ud.cpu().numpy()
    s.close()
    err3 = max(np.abs(got[m] - U[m]).max() / np.abs(U[m]).max() for m in range(5))
    print("config 2: three RK3 steps rel Linf", err3)
    assert err3 <= 1e-10


# ------------------------------------------------------------------ the timed path itself, at full size
def window_case(case, U_full, box):
    """The sub-box [i0,i1) x [j0,j1) x [k0,k1) of `case` as a case of its own, for the CPU side only: state (with the
    true neighbours in its ghost layers), metric planes and boundary data cut out of the full arrays.  A face of the box
    that is a face of the domain keeps the domain's condition and data; an axis the box spans completely stays periodic
    if it was; every other face is a CUT face and gets plain extrapolation, which is wrong there -- the error it makes
    travels 6 points per stage (the reach of the two-pass viscous operator; the inviscid stencils reach 4), so points
    18 or more away from every cut face see none of it after one RK3 step.  Returns (case, cut[6])."""
    import dataclasses
    i0, i1, j0, j1, k0, k1 = box
    lo, hi, n = (i0, j0, k0), (i1, j1, k1), (case.nx, case.ny, case.nz)
    sl = {0: slice(i0, i1 + 2 * NG), 1: slice(j0, j1 + 2 * NG), 2: slice(k0, k1 + 2 * NG)}
    met = []
    for m in case.metrics:
        mk = slice(None) if m.shape[0] == 1 else sl[2]
        met.append(np.ascontiguousarray(m[mk, sl[1], sl[0]]))
    bc, cut = list(case.bc), [False] * 6
    inflow, wall_vn = [None] * 6, [None] * 6
    for d in range(3):
        whole = lo[d] == 0 and hi[d] == n[d]
        for side in range(2):
            f = 2 * d + side
            on_domain_face = lo[d] == 0 if side == 0 else hi[d] == n[d]
            if case.bc[f] == "periodic":
                if not whole:
                    bc[f], cut[f] = "outflow", True
                continue
            if not on_domain_face:
                bc[f], cut[f] = "outflow", True
                continue
            slow, fast = (2, 1) if d == 0 else (2, 0) if d == 1 else (1, 0)      # tangential axes of the face arrays
            if case.inflow[f] is not None:
                inflow[f] = np.ascontiguousarray(case.inflow[f][:, sl[slow], sl[fast]])
            if case.wall_vn[f] is not None:
                wall_vn[f] = np.ascontiguousarray(case.wall_vn[f][sl[slow], sl[fast]])
    sub = dataclasses.replace(case, name=f"{case.name}[{i0}:{i1},{j0}:{j1},{k0}:{k1}]", nx=i1 - i0, ny=j1 - j0, nz=k1 - k0,
                              metrics=met, bc=bc, inflow=inflow, wall_vn=wall_vn, coords=None,
                              U0=np.ascontiguousarray(U_full[:, sl[2], sl[1], sl[0]]))
    assert sub.weno_eps == case.weno_eps
    return sub, cut


def test_config5_full_size_one_rk3_step_whole_windows(B, Oracle):
    """ONE ocfd_rk3_step of config 5 at 2048 x 300 x 256 -- the call, the launch shapes (automatic march segments,
    z chunks of the viscous passes, CTA numbering, rotating state buffers, fused RK3 update) and the grid bench.py
    times -- compared with the CPU reference on WHOLE windows, every point of them that no cut face can have reached:
    the four x-y corners over the full periodic span (inflow / wall / outflow faces, the periodic seam in z, the z-chunk
    seams k = 32, 64, ...), the ragged last tiles in y (300 = 9*32 + 12 = 37*8 + 4), the seam i = 1024 between the two
    segments the automatic rule cuts the x march into, the seam i = 512 between two column groups of the viscous CTA
    numbering, the steepest pressure front of the initial field, and two seeded interior boxes cut in all directions.
    Interfaces whose sensor value comes within 1e-9 of a threshold at any stage may legitimately decide differently;
    they are counted and their domain of influence is left out, as in the stepping tests."""
    import torch
    from tests.parity_utils import near_threshold, dilate
    case = W.ramp()
    assert (case.nx, case.ny, case.nz) == (2048, 300, 256) and case.scheme == "hybrid"
    nx, ny, nz = case.nx, case.ny, case.nz
    o_full = Oracle(case)
    U_full = o_full.fill_ghosts(case.U0.copy())
    dt = case.cfl / o_full.max_wavespeed(U_full)
    s = B.Solver(case)
    Ud = s.to_device(U_full)
    s.rk3_step(Ud, dt)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(Ud[:, NG:-NG, NG:-NG, NG:-NG]).all())
    # where the initial pressure is steepest along x (plane k = 10, away from the faces): the flagged region
    Up = U_full[:, NG + 10, NG:-NG, NG:-NG]
    p = (case.gamma - 1.0) * (Up[4] - 0.5 * (Up[1] ** 2 + Up[2] ** 2 + Up[3] ** 2) / Up[0])
    gp = np.abs(p[40:-40, 42:-38] - p[40:-40, 40:-40]) / p[40:-40, 41:-39]
    jf, i_f = np.unravel_index(int(np.argmax(gp)), gp.shape)
    jf, i_f = int(jf) + 40, int(i_f) + 41
    rng = np.random.default_rng(77)
    boxes = {
        "corner x- y-": (0, 72, 0, 72, 0, nz), "corner x+ y-": (nx - 72, nx, 0, 72, 0, nz),
        "corner x- y+ (ragged y tiles)": (0, 72, ny - 72, ny, 0, nz), "corner x+ y+ (ragged y tiles)": (nx - 72, nx, ny - 72, ny, 0, nz),
        "x march seam i=1024": (1024 - 36, 1024 + 36, 100, 172, 0, nz),
        "column-group seam i=512, top": (512 - 36, 512 + 36, ny - 72, ny, 0, nz),
        "steepest pressure front": (max(0, min(nx - 96, i_f - 48)), max(0, min(nx - 96, i_f - 48)) + 96,
                                    max(0, min(ny - 80, jf - 40)), max(0, min(ny - 80, jf - 40)) + 80, 0, nz),
    }
    for q in range(2):
        a, b, c = int(rng.integers(100, nx - 200)), int(rng.integers(20, ny - 120)), int(rng.integers(8, nz - 140))
        boxes[f"interior box {q}"] = (a, a + 100, b, b + 100, c, c + 130)
    M = 18
    worst, checked, near_total = 0.0, 0, 0
    for tag, box in boxes.items():
        sub, cut = window_case(case, U_full, box)
        o = Oracle(sub)
        U = sub.U0.copy()
        Un = U.copy()
        excl = np.zeros((sub.nz, sub.ny, sub.nx), dtype=bool)
        per = [sub.bc[2 * d] == "periodic" for d in range(3)]
        for st in range(3):                                   # the calls ora_rk3_step makes, with a look at theta per stage
            o.fill_ghosts(U)
            m = near_threshold(o.sensor(U), sub.theta1, sub.theta2, 1e-9)
            if m.any():
                near_total += int(m.sum())
                excl |= dilate(m, M, per)
            o.rk3_update(Un, U, o.rhs(U), dt, st)
        o.fill_ghosts(U)                                      # the step ends with a fill: it resets the wall / inflow nodes
        keep = ~excl
        lo = [M if cut[2 * d] else 0 for d in range(3)]
        hi = [M if cut[2 * d + 1] else 0 for d in range(3)]
        inner = (slice(lo[2], sub.nz - hi[2]), slice(lo[1], sub.ny - hi[1]), slice(lo[0], sub.nx - hi[0]))
        i0, i1, j0, j1, k0, k1 = box
        got = Ud[:, NG + k0:NG + k1, NG + j0:NG + j1, NG + i0:NG + i1].cpu().numpy()
        ref = U[:, NG:-NG, NG:-NG, NG:-NG]
        umax = np.abs(ref).max()
        err = 0.0
        for mcomp in range(5):
            d = np.abs(got[mcomp] - ref[mcomp])[inner][keep[inner]]
            err = max(err, d.max() / max(np.abs(ref[mcomp]).max(), 1e-3 * umax))
        npts = int(keep[inner].sum())
        checked += npts
        worst = max(worst, err)
        print(f"config 5 full size, one RK3 step, window {tag} {box}: {npts} points compared, rel Linf {err:.3e}, "
              f"cut faces {cut}")
        assert npts > 0.15 * sub.nx * sub.ny * sub.nz, tag
        assert err <= 1e-11, (tag, err)
    s.close()
    print(f"config 5 full size: {checked} points in {len(boxes)} windows, worst rel Linf {worst:.3e}, "
          f"{near_total} points next to an interface within 1e-9 of a threshold (their domain of influence left out)")
