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
