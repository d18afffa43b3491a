"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on seeded inputs.

Tolerances (BASELINE.json north_star): relative L-inf <= 1e-11 per RHS, <= 1e-9 after 100 RK3 steps on smooth
cases; hybrid-scheme flags exact except within 1e-12 of a threshold (counted and reported).
Error metric: per conserved component m, max_i |gpu - ora| / max_i |ora| over interior points;
when max|ora_m| is (numerically) zero the error is taken relative to max|U_m|.
DESIGN.md reading R-23 extends "numerically zero" to "zero by cancellation": a component whose max|ora_m| lies below
1e-3 * Lambda * max|U| (0.1 % of the size of the terms that sum to it) is measured against that floor.  Every test that
uses the floor prints the un-floored error of every component beside the floored one and says which were floored.
"""
import json
import os

import numpy as np
import pytest

from paper_2209_15333_b200 import workloads as W

pytestmark = pytest.mark.gpu

NG = 4
INT = (slice(None), slice(NG, -NG), slice(NG, -NG), slice(NG, -NG))
TOL_RHS = 1e-11
TOL_100 = 1e-9


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


def rel_linf(gpu, ora, U, floor=0.0):
    """max|gpu-ora| / max|ora| per component.  `floor` guards components whose exact value is zero or small by
    cancellation (v and w momentum of a 2-D boundary layer, a steady profile): there the round-off of either side
    scales with the terms that cancel, not with their sum, so the denominator is never taken below `floor`
    (callers pass 1e-3 * Lambda_max * max|U|, Lambda = the wavespeed sum of DESIGN section 2, i.e. 0.1 % of the
    size of dU/dt's individual terms).  A component that is identically zero on both sides AND in U (w of a flow with
    no spanwise motion) has error 0 if the two sides agree exactly, else infinity: there is no scale to divide by."""
    errs = []
    for m in range(5):
        den = max(np.abs(ora[m]).max(), floor)
        if den < 1e-300:
            den = np.abs(U[m]).max()
        diff = np.abs(gpu[m] - ora[m]).max()
        errs.append(diff / den if den > 0.0 else (0.0 if diff == 0.0 else np.inf))
    return np.array(errs)


def term_floor(Oracle, case, U_full):
    return 1e-3 * Oracle(case).max_wavespeed(U_full) * np.abs(U_full[INT]).max()


R23_LOG = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out", "r23_errors.jsonl")


def report(tag, got, ref, U, floor):
    """DESIGN R-23 on file: the un-floored error of every component beside the floored one, printed and appended as
    one JSON line to gpurun_out/r23_errors.jsonl (scratch the GPU run leaves behind; the table in profiles/ is made
    from it).  For every component measured against the floor the bar is asserted in its absolute form too:
    |gpu - ora| <= 1e-11 * floor = 1e-14 * Lambda * max|U|.  Returns the floored errors."""
    with np.errstate(invalid="ignore", divide="ignore"):
        raw = rel_linf(got, ref, U)
    flo = rel_linf(got, ref, U, floor)
    absd = np.array([np.abs(got[m] - ref[m]).max() for m in range(5)])
    mx = np.abs(ref).reshape(5, -1).max(axis=1)
    which = [m for m in range(5) if mx[m] < floor]
    print(f"{tag}: rel Linf per component un-floored {raw}, floored {flo}; floor {floor:.3e}, max|ora| {mx}, "
          f"components measured against the floor: {which}")
    for m in which:
        assert absd[m] <= TOL_RHS * floor, (tag, m, absd[m], floor)
    try:
        os.makedirs(os.path.dirname(R23_LOG), exist_ok=True)
        with open(R23_LOG, "a") as f:
            f.write(json.dumps({"case": tag, "floor": floor, "max_abs_ora": mx.tolist(), "abs_err": absd.tolist(),
                                "rel_unfloored": [None if not np.isfinite(v) else float(v) for v in raw],
                                "rel_floored": flo.tolist(), "floored_components": which}) + "\n")
    except OSError:
        pass
    return flo


def run_rhs_both(B, Oracle, case, fill=True):
    o = Oracle(case)
    U = case.U0.copy()
    if fill:
        o.fill_ghosts(U)
    ref = o.rhs(U)
    s = B.Solver(case)
    Ud = s.to_device(U)
    dUd = s.rhs(Ud)
    s.torch.cuda.synchronize()
    got = dUd.cpu().numpy()
    assert np.array_equal(Ud.cpu().numpy(), U), "ocfd_rhs must not modify U"
    ghost = np.ones(got.shape, dtype=bool)
    ghost[INT] = False
    assert np.all(got[ghost] == 0.0), "ocfd_rhs must leave the ghosts of dU untouched"
    s.close()
    return got[INT], ref[INT], U[INT]


# sizes span several tiles of every kernel (x tile 56, y/z tile 20, viscous blocks 32x4x2) with ragged tails
@pytest.mark.parametrize("scheme", ["ud7", "weno7", "weno5", "hybrid"])
@pytest.mark.parametrize("grid", ["uniform", "stretched", "wavy"])
def test_rhs_parity_smooth_periodic(B, Oracle, grid, scheme):
    case = W.smooth_periodic(70, 45, 23, grid=grid, scheme=scheme, Re=150.0, seed=3)
    got, ref, U = run_rhs_both(B, Oracle, case)
    err = rel_linf(got, ref, U)
    assert err.max() <= TOL_RHS, err


@pytest.mark.parametrize("scheme", ["ud7", "weno7", "hybrid"])
def test_rhs_parity_inviscid_only_and_sw_eps(B, Oracle, scheme):
    case = W.smooth_periodic(58, 21, 41, grid="wavy", scheme=scheme, inviscid=True, seed=5)
    case.sw_eps = 0.02
    got, ref, U = run_rhs_both(B, Oracle, case)
    assert rel_linf(got, ref, U).max() <= TOL_RHS


def shocked_box(nx, ny, nz, grid, scheme, aperiodic, seed=9):
    """Inviscid case with steep fronts on any of the smooth_periodic grids (the recipe of W.shocked_periodic on a
    non-cubic, optionally curvilinear box), periodic or with extrapolation on all six faces.  Inputs only."""
    case = W.smooth_periodic(nx, ny, nz, seed=seed, scheme=scheme, Ma=1.2, amp=0.15, inviscid=True, grid=grid)
    KK, JJ, II = np.meshgrid(np.arange(-NG, nz + NG), np.arange(-NG, ny + NG), np.arange(-NG, nx + NG), indexing="ij")
    a, b, c = 2 * np.pi * II / nx, 2 * np.pi * JJ / ny, 2 * np.pi * KK / nz
    front = 0.5 * (1.0 + np.tanh(5.0 * np.sin(a + 0.7 * np.sin(b)) * np.cos(c + 0.3)))
    fac = 1.0 + 1.5 * front
    U = case.U0.copy()
    U[:4] *= fac
    U[4] *= fac * (1.0 + 0.8 * front)
    case.U0 = np.ascontiguousarray(U)
    case.theta1, case.theta2 = 0.02, 0.1
    if aperiodic:
        case.bc = ["outflow"] * 6
    case.name = f"shocked_box_{grid}_{scheme}_{'open' if aperiodic else 'periodic'}"
    return case


@pytest.mark.parametrize("which", ["uniform-periodic", "wavy-open", "stretched-open"])
def test_inviscid_hybrid_standalone_sensor_flags_and_rhs(B, Oracle, which):
    """Runs without viscous terms take theta from the stand-alone sensor kernel (with them it is part of viscous
    pass 1): theta on the interior AND on the first ghost layer of every face (copy rule on aperiodic faces, R-12),
    the per-interface decisions, and the hybrid RHS built on them, against the CPU reference."""
    grid, ends = which.split("-")
    case = shocked_box(70, 45, 23, grid, "hybrid", ends == "open")
    o = Oracle(case)
    U = o.fill_ghosts(case.U0.copy())
    bad, near, total, hist = flag_report(B, Oracle, case, U)
    print(f"{case.name}: {total} interfaces, {near} within 1e-12 of a threshold, {bad} mismatches, "
          f"UD7/WENO7/WENO5 = {hist.tolist()}")
    assert bad == 0 and np.all(hist > 0)
    th_ref = o.sensor(U)
    s = B.Solver(case)
    th_gpu = s.debug_sensor(s.to_device(U))[0].cpu().numpy()
    s.close()
    I = slice(NG, -NG)
    for lo, hi in (((NG - 1, I, I), (-NG, I, I)), ((I, NG - 1, I), (I, -NG, I)), ((I, I, NG - 1), (I, I, -NG))):
        for face in (lo, hi):
            assert np.abs(th_gpu[face] - th_ref[face]).max() <= 1e-13, (which, face)
    got, ref, Ui = run_rhs_both(B, Oracle, case)
    assert rel_linf(got, ref, Ui).max() <= TOL_RHS


@pytest.mark.parametrize("which", ["ud7-wavy-periodic", "weno7-wavy-open", "weno5-stretched-open", "hybrid-uniform-periodic",
                                   "hybrid-wavy-open"])
def test_inviscid_ten_steps_standalone_update(B, Oracle, which):
    """Without viscous terms the RK3 stage update is a kernel of its own (with them it is folded into viscous pass 2)
    working on the rotating state buffers: 10 steps against the CPU reference at the 1e-9 bar, face ghosts included."""
    from tests.parity_utils import step_both_hybrid
    scheme, grid, ends = which.split("-")
    case = shocked_box(46, 30, 20, grid, scheme, ends == "open") if scheme == "hybrid" else \
        W.smooth_periodic(46, 30, 20, grid=grid, scheme=scheme, inviscid=True, seed=12)
    if ends == "open":
        case.bc = ["outflow"] * 6
    res = step_both_hybrid(B, Oracle, case, 10)
    assert res["finite"] and res["flag_mismatches"] == 0
    if res["err_all"] > TOL_100:
        assert res["near"] > 0 and res["excluded_fraction"] < 1.0 and res["err_outside"] <= TOL_100, res
    assert res["err_padded_outside"] <= TOL_100, res
    if scheme == "hybrid":
        assert res["hist0"][0] > 0 and res["hist0"][1] + res["hist0"][2] > 0


def test_rhs_freestream_is_zero_to_roundoff(B, Oracle):
    for grid in ("uniform", "stretched"):
        case = W.smooth_periodic(60, 24, 22, grid=grid, scheme="weno7")
        shp = case.padded_shape
        one = np.ones(shp)
        p = 1.1 * 0.9 / (case.gamma * case.Ma ** 2)
        case.U0 = np.ascontiguousarray(W.cons_from_prim(1.1 * one, 0.8 * one, -0.3 * one, 0.45 * one, p * one, case.gamma))
        got, ref, U = run_rhs_both(B, Oracle, case)
        scale = np.abs(U).max() * max(np.abs(m).max() for m in case.metrics[:9])
        assert np.abs(got).max() <= 1e-12 * scale
        assert np.abs(got - ref).max() <= 1e-12 * scale


def flag_report(B, Oracle, case, U):
    """Compare sensor decisions; returns (mismatches outside the 1e-12 band, interfaces inside the band)."""
    o = Oracle(case)
    th_ref = o.sensor(U)
    s = B.Solver(case)
    th_gpu, fl_gpu = s.debug_sensor(s.to_device(U))
    s.torch.cuda.synchronize()
    th_gpu, fl_gpu = th_gpu.cpu().numpy(), fl_gpu.cpu().numpy()
    s.close()
    I = slice(NG, -NG)
    assert np.abs(th_gpu[I, I, I] - th_ref[I, I, I]).max() <= 1e-13
    bad = near = total = 0
    hist = np.zeros(3, dtype=np.int64)
    for d in range(3):
        fl_ref = o.flags(th_ref, d)
        sl = [I, I, I]
        sl[2 - d] = slice(NG - 1, -NG)                     # interfaces s = -1 .. n-1 along d
        sl = tuple(sl)
        sh = [0, 0, 0]
        sh[2 - d] = 1
        a = th_ref[sl]
        b = np.roll(th_ref, -1, axis=2 - d)[sl]
        Th = np.maximum(a, b)
        band = (np.abs(Th - case.theta1) <= 1e-12) | (np.abs(Th - case.theta2) <= 1e-12)
        diff = fl_gpu[d][sl] != fl_ref[sl]
        bad += int((diff & ~band).sum())
        near += int(band.sum())
        total += diff.size
        hist += np.bincount(fl_ref[sl].ravel(), minlength=3)[:3]
    return bad, near, total, hist


def test_hybrid_sensor_decisions_and_rhs_on_shocked_field(B, Oracle):
    case = W.shocked_periodic(44, theta1=0.02, theta2=0.1)
    o = Oracle(case)
    U = o.fill_ghosts(case.U0.copy())
    bad, near, total, hist = flag_report(B, Oracle, case, U)
    print(f"hybrid flags: {total} interfaces, {near} within 1e-12 of a threshold (excluded), {bad} mismatches; "
          f"UD7/WENO7/WENO5 = {hist.tolist()}")
    assert bad == 0
    assert np.all(hist > 0)
    got, ref, Ui = run_rhs_both(B, Oracle, case)
    assert rel_linf(got, ref, Ui).max() <= TOL_RHS


def test_fill_ghosts_matches_oracle_on_wall_inflow_outflow(B, Oracle):
    for case in (W.flat_plate(nx=60, ny=26, nz=12), W.ramp(nx=48, ny=30, nz=10, nmodes=8)):
        rng = np.random.default_rng(2)
        U = np.ascontiguousarray(case.U0 * (1.0 + 0.02 * rng.uniform(-1, 1, case.U0.shape)))
        ref = Oracle(case).fill_ghosts(U.copy())
        s = B.Solver(case)
        Ud = s.fill_ghosts(s.to_device(U))
        s.torch.cuda.synchronize()
        got = Ud.cpu().numpy()
        s.close()
        # every point the oracle wrote (and only those) must agree; copies are exact, wall arithmetic to round-off
        assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()
        untouched = ref == U                     # edges, corners and the interior away from Dirichlet nodes
        assert np.array_equal(got[untouched], U[untouched])


@pytest.mark.parametrize("which", ["plate", "ramp", "ramp3level"])
def test_rhs_parity_with_walls(B, Oracle, which):
    if which == "plate":
        case = W.flat_plate(nx=72, ny=44, nz=24)
    else:
        case = W.ramp(nx=64, ny=44, nz=24, nmodes=12, theta2=np.inf if which == "ramp" else 0.1)
    got, ref, U = run_rhs_both(B, Oracle, case)
    floor = term_floor(Oracle, case, Oracle(case).fill_ghosts(case.U0.copy()))
    err = report(f"walls/{which}", got, ref, U, floor)
    assert err.max() <= TOL_RHS


@pytest.mark.parametrize("which", ["uniform", "stretched", "wavy", "plate", "ramp"])
def test_rhs_parity_eighth_order_viscous_scheme(B, Oracle, which):
    """visc_order = 8: 9-point central stencils, closure rows 2/2/4/6 on aperiodic axes."""
    if which == "plate":
        case = W.flat_plate(nx=72, ny=44, nz=24)
    elif which == "ramp":
        case = W.ramp(nx=64, ny=44, nz=24, nmodes=12)
    else:
        case = W.smooth_periodic(70, 45, 23, grid=which, scheme="ud7", Re=150.0, seed=5)
    case.visc_order = 8
    got, ref, U = run_rhs_both(B, Oracle, case)
    floor = term_floor(Oracle, case, Oracle(case).fill_ghosts(case.U0.copy()))
    err = report(f"visc8/{which}", got, ref, U, floor)
    assert err.max() <= TOL_RHS
    case.visc_order = 6          # and the two schemes really differ
    ref6 = Oracle(case).rhs(Oracle(case).fill_ghosts(case.U0.copy()))[INT]
    assert rel_linf(ref, ref6, U, floor).max() > 1e-9


@pytest.mark.parametrize("which", ["plate", "ramp", "ramp3level", "box-ud7", "box-weno7", "box-weno5"])
def test_rhs_parity_paper_boundary_scheme(B, Oracle, which):
    """bc_closure = 1: shielded WENO5 next to aperiodic faces, in all three
    sweep kernels (x tile kernel, y / z marching kernels); sizes leave ragged tiles at the far boundaries."""
    if which == "plate":
        case = W.flat_plate(nx=72, ny=44, nz=24)
    elif which.startswith("ramp"):
        case = W.ramp(nx=64, ny=44, nz=24, nmodes=12, theta2=np.inf if which == "ramp" else 0.1)
    else:
        case = W.smooth_periodic(70, 45, 23, grid="wavy", scheme=which.split("-")[1], Re=150.0, seed=6)
        case.bc = ["outflow"] * 6          # every axis aperiodic: closures of all three sweeps and both ends
    case.bc_closure = 1
    got, ref, U = run_rhs_both(B, Oracle, case)
    floor = term_floor(Oracle, case, Oracle(case).fill_ghosts(case.U0.copy()))
    err = report(f"closure/{which}", got, ref, U, floor)
    assert err.max() <= TOL_RHS
    case.bc_closure = 0                # and the closure really changes the result
    o = Oracle(case)
    ref0 = o.rhs(o.fill_ghosts(case.U0.copy()))[INT]
    assert np.abs(ref - ref0).max() > 1e-6 * np.abs(ref0).max()


def test_twenty_steps_paper_boundary_scheme(B, Oracle):
    case = W.flat_plate(nx=64, ny=40, nz=16)
    case.bc_closure = 1
    err, got, ref = step_both(B, Oracle, case, 20)
    print("plate, paper's boundary scheme, 20 steps: rel Linf", err)
    assert err <= 1e-9
    assert np.isfinite(got).all()


@pytest.mark.parametrize("which", ["wavy-ud7", "wavy-weno7", "wavy-weno5", "stretched-hybrid", "uniform-weno7",
                                   "shocked", "plate", "ramp3level", "box-closure", "box-closure-ud7",
                                   "box-closure-hybrid", "plate-closure-ud7", "ramp-closure-hybrid"])
def test_rhs_parity_characteristic_reconstruction(B, Oracle, which):
    """char_recon = 1: all three sweeps in characteristic variables."""
    if which == "plate":
        case = W.flat_plate(nx=72, ny=44, nz=24)
    elif which == "ramp3level":
        case = W.ramp(nx=64, ny=44, nz=24, nmodes=12, theta2=0.1)
    elif which == "shocked":
        case = W.shocked_periodic(44, theta1=0.02, theta2=0.1)
    elif which.startswith("box-closure"):
        # the paper's boundary scheme together with characteristic variables, for the linear and hybrid schemes too:
        # the linear interfaces of a boundary segment that lie outside the boundary band stay with the walkers
        scheme = which.split("-")[2] if which.count("-") == 2 else "weno7"
        case = W.smooth_periodic(70, 45, 23, grid="wavy", scheme=scheme, Re=150.0, seed=6)
        case.bc = ["outflow"] * 6
        case.bc_closure = 1
    elif which == "plate-closure-ud7":
        case = W.flat_plate(nx=72, ny=44, nz=24, scheme="ud7")
        case.bc_closure = 1
    elif which == "ramp-closure-hybrid":
        case = W.ramp(nx=64, ny=44, nz=24, nmodes=12, theta2=0.1)
        case.bc_closure = 1
    else:
        grid, scheme = which.split("-")
        case = W.smooth_periodic(70, 45, 23, grid=grid, scheme=scheme, Re=150.0, seed=8)
    case.char_recon = 1
    got, ref, U = run_rhs_both(B, Oracle, case)
    floor = term_floor(Oracle, case, Oracle(case).fill_ghosts(case.U0.copy()))
    err = report(f"char/{which}", got, ref, U, floor)
    assert err.max() <= TOL_RHS


@pytest.mark.parametrize("dims", [(8, 8, 8), (10, 9, 8), (34, 8, 33), (8, 37, 9)])
@pytest.mark.parametrize("scheme", ["hybrid", "weno7"])
def test_rhs_parity_smallest_and_ragged_grids(B, Oracle, dims, scheme):
    """Edge sizes: the minimum the library accepts (8 points per axis: the march is four chunks, the x tile one
    ragged tile, the viscous tiles mostly empty), and extents one or two past a tile / chunk boundary."""
    nx, ny, nz = dims
    for grid in ("uniform", "wavy"):
        case = W.smooth_periodic(nx, ny, nz, grid=grid, scheme=scheme, Re=120.0, seed=nx + ny + nz)
        got, ref, U = run_rhs_both(B, Oracle, case)
        assert rel_linf(got, ref, U).max() <= TOL_RHS, (dims, grid)


def test_host_buffer_entry_point_equals_the_device_path_and_the_oracle(B, Oracle):
    """ocfd_rk3_steps_host (H2D, n steps, D2H in one call: the end-to-end number of bench.py goes through it)."""
    import torch
    case = W.ramp(nx=64, ny=40, nz=16, nmodes=12)
    o = Oracle(case)
    U = o.fill_ghosts(case.U0.copy())
    dt = case.cfl / o.max_wavespeed(U)
    s = B.Solver(case)
    Ud = s.to_device(U)
    Uh = torch.from_numpy(U.copy()).pin_memory()
    scratch = torch.empty_like(Ud)
    s.rk3_steps_host(Uh, scratch, dt, 2)
    for _ in range(2):
        s.rk3_step(Ud, dt)
        o.rk3_step(U, dt)
    assert bool((Uh == Ud.cpu()).all())
    got = Uh.numpy()
    assert max(np.abs(got[m] - U[m]).max() / np.abs(U[m]).max() for m in range(5)) <= 1e-11
    s.close()


@pytest.mark.parametrize("which", ["plate", "ramp", "wavy"])
def test_max_wavespeed_matches_the_oracle(B, Oracle, which):
    case = (W.flat_plate(nx=72, ny=44, nz=24) if which == "plate" else W.ramp(nx=64, ny=44, nz=24, nmodes=12)
            if which == "ramp" else W.smooth_periodic(70, 45, 23, grid="wavy"))
    o = Oracle(case)
    U = o.fill_ghosts(case.U0.copy())
    s = B.Solver(case)
    lam = s.max_wavespeed(s.to_device(U))
    s.close()
    assert lam == pytest.approx(o.max_wavespeed(U), rel=1e-13)


def test_max_wavespeed_reports_a_blown_up_state_as_nan(B):
    """A NaN anywhere in the interior must not come back as a finite Lambda (a caller would go on with a finite dt)."""
    case = W.smooth_periodic(24, 16, 12, grid="wavy")
    s = B.Solver(case)
    U = case.U0.copy()
    assert np.isfinite(s.max_wavespeed(s.to_device(U)))
    U[4, NG + 5, NG + 7, NG + 11] = np.nan                 # E of one interior point
    assert np.isnan(s.max_wavespeed(s.to_device(U)))
    U = case.U0.copy()
    U[0, NG + 1, NG + 2, NG + 3] = np.nan                  # rho
    assert np.isnan(s.max_wavespeed(s.to_device(U)))
    s.close()


def test_check_state_counts_equal_the_oracle(B, Oracle):
    """ocfd_check_state against ora_check_state (integer counts: exact) on states with bad points of every kind planted
    at seeded places, in the first and last interior planes, rows and columns too; ghosts full of garbage."""
    rng = np.random.default_rng(5)
    for case in (W.smooth_periodic(150, 45, 70, grid="wavy"), W.ramp(nx=64, ny=44, nz=24, nmodes=12), W.tgv(16)):
        o = Oracle(case)
        s = B.Solver(case)
        U = o.fill_ghosts(case.U0.copy())
        assert s.check_state(s.to_device(U)) == o.check_state(U) == (0, 0, 0)
        nz, ny, nx = case.nz, case.ny, case.nx
        spots = np.stack([rng.integers(0, n, 400) for n in (nz, ny, nx)], axis=1)
        spots[:6] = [(0, 0, 0), (nz - 1, ny - 1, nx - 1), (0, ny - 1, 0), (nz - 1, 0, nx - 1), (0, 0, nx - 1), (nz - 1, ny - 1, 0)]
        for q, (k, j, i) in enumerate(spots):
            idx = (k + NG, j + NG, i + NG)
            kind = q % 6
            if kind == 0:
                U[(int(rng.integers(0, 5)),) + idx] = np.nan
            elif kind == 1:
                U[(int(rng.integers(0, 5)),) + idx] = np.inf if q % 4 == 1 else -np.inf
            elif kind == 2:
                U[(0,) + idx] = -abs(U[(0,) + idx])
            elif kind == 3:
                U[(0,) + idx] = 0.0
            elif kind == 4:
                with np.errstate(all="ignore"):               # a collision with an earlier spot may have zeroed rho
                    ke = 0.5 * sum(U[(m,) + idx] ** 2 for m in (1, 2, 3)) / abs(U[(0,) + idx])
                U[(4,) + idx] = 0.5 * ke - 0.01               # E below the kinetic energy: p < 0
            else:
                U[(4,) + idx] = 1.5 * U[(4,) + idx]          # harmless
        U[:, :NG] = np.nan
        U[0, :, :, -NG:] = -1.0
        want = o.check_state(U)
        got = s.check_state(s.to_device(U))
        s.close()
        assert min(want) > 20, want
        assert got == want, (case.name, got, want)


def test_two_contexts_in_one_process_do_not_share_state(B, Oracle):
    """include/ocfd.h: "no global state; several contexts may coexist".  Two contexts with different grids, schemes and
    kernel instantiations, created, used alternately and destroyed in one process (the shared-memory opt-in of the
    kernels is kept per context)."""
    a = W.ramp(nx=48, ny=30, nz=10, nmodes=8)
    b = W.smooth_periodic(40, 24, 18, grid="stretched", scheme="weno7", Re=150.0, seed=4)
    sa, sb = B.Solver(a), B.Solver(b)
    refs, gots = [], []
    for case, s in ((a, sa), (b, sb), (a, sa), (b, sb)):
        o = Oracle(case)
        U = o.fill_ghosts(case.U0.copy())
        refs.append(o.rhs(U)[INT])
        gots.append(s.rhs(s.to_device(U)).cpu().numpy()[INT])
    sa.close()
    sc = B.Solver(a)                                       # a new context after one was destroyed
    U = Oracle(a).fill_ghosts(a.U0.copy())
    gots.append(sc.rhs(sc.to_device(U)).cpu().numpy()[INT])
    refs.append(refs[0])
    sb.close()
    sc.close()
    for got, ref, case in zip(gots, refs, (a, b, a, b, a)):
        U = Oracle(case).fill_ghosts(case.U0.copy())
        floor = term_floor(Oracle, case, U)
        assert rel_linf(got, ref, U[INT], floor).max() <= TOL_RHS
    assert np.array_equal(gots[0], gots[2]) and np.array_equal(gots[1], gots[3]) and np.array_equal(gots[0], gots[4])


def test_debug_sensor_leaves_nan_where_the_sensor_does_not_write(B):
    case = W.shocked_periodic(20)
    s = B.Solver(case)
    th, fl = s.debug_sensor(s.fill_ghosts(s.to_device(case.U0.copy())))
    th = th.cpu().numpy()
    s.close()
    I = slice(NG, -NG)
    assert np.isfinite(th[I, I, I]).all()
    assert np.isfinite(th[NG - 1, I, I]).all() and np.isfinite(th[I, -NG, I]).all() and np.isfinite(th[I, I, NG - 1]).all()
    assert np.isnan(th[0]).all() and np.isnan(th[:, :, 0]).all() and np.isnan(th[NG - 1, NG - 1, :]).all()


def test_results_are_bitwise_reproducible(B):
    """One add per output element and kernel (TMA reduce-add for y and z, in stream order): no atomics race, so two
    evaluations of the same state agree bit for bit (the paper's design accumulates with atomicAdd from several
    streams, and does not have this property)."""
    case = W.ramp(nx=64, ny=44, nz=24, nmodes=12)
    s = B.Solver(case)
    U = s.to_device(case.U0.copy())
    s.fill_ghosts(U)
    a = s.rhs(U).clone()
    b = s.rhs(U).clone()
    assert bool((a == b).all())
    U2 = U.clone()
    s.rk3_step(U, 1e-4)
    s.rk3_step(U2, 1e-4)
    assert bool((U == U2).all())
    s.close()


@pytest.mark.parametrize("which", ["ramp", "periodic"])
def test_launch_shape_knobs_change_no_bit(B, which):
    """ocfd_set_tuning only re-shapes launches: marches cut into segments (every segment re-stages its first 8 rows and
    recomputes the interface fluxes there from the same values in the same order), short z chunks of the viscous
    passes, another CTA numbering.  The result must be the same bits, for one RHS and for a whole RK3 step -- which
    also exercises the segmented march on a grid small enough to compare whole arrays (the automatic rule only cuts
    marches on grids as large as configs 4 and 5)."""
    case = W.ramp(nx=72, ny=44, nz=40, nmodes=12) if which == "ramp" else W.shocked_periodic(40)
    ref = B.Solver(case)
    U0 = ref.to_device(case.U0.copy())
    ref.fill_ghosts(U0)
    dt = 0.3 * case.cfl / ref.max_wavespeed(U0)
    a = ref.rhs(U0).clone()
    Ua = U0.clone()
    ref.rk3_step(Ua, dt)
    ref.close()
    for knobs in ({"march_seg": 3}, {"march_seg": 5, "tile_group": 1}, {"zchunk_flux": 8, "zchunk_div": 8, "tile_group": 2}):
        s = B.Solver(case)
        for k, v in knobs.items():
            s.set_tuning(k, v)
        b = s.rhs(U0).clone()
        Ub = U0.clone()
        s.rk3_step(Ub, dt)
        s.close()
        assert bool((a == b).all()), knobs
        assert bool((Ua == Ub).all()), knobs


@pytest.mark.parametrize("which", ["tgv", "ramp"])
def test_rk3_step_replayed_from_a_cuda_graph_gives_the_same_bits(B, which):
    """ocfd_rk3_step only enqueues kernels on the context's stream, so a caller can capture it into a CUDA graph (after
    one plain call, which does the one-time host-side set-up) and replay the 27 launches of a step as one graph launch:
    what small, launch-bound grids need.  Five replays must equal five plain steps bit for bit."""
    import torch
    case = W.tgv(24) if which == "tgv" else W.ramp(nx=64, ny=40, nz=16, nmodes=8)
    stream = torch.cuda.Stream()                     # not the legacy default stream: that one cannot be captured
    with torch.cuda.stream(stream):
        s = B.Solver(case, stream=stream)
        U = s.to_device(case.U0.copy())
        s.fill_ghosts(U)
        dt = 0.5 * case.cfl / s.max_wavespeed(U)
        plain = U.clone()
        for _ in range(6):
            s.rk3_step(plain, dt)                    # the first of them is the warm-up call as well
        V = U.clone()
        s.rk3_step(V, dt)                            # same buffer as the one captured below
        stream.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=stream):
            s.rk3_step(V, dt)
        # capture enqueues nothing: V still holds the state after one step
        for _ in range(5):
            g.replay()
        stream.synchronize()
        assert bool((V == plain).all())
        assert bool(torch.isfinite(V[:, NG:-NG, NG:-NG, NG:-NG]).all())
        s.close()


def test_set_tuning_refuses_what_the_launchers_would_ignore(B):
    """include/ocfd.h: a zchunk value is 0 (automatic) or at least 8; unknown keys and negative values are errors."""
    s = B.Solver(W.smooth_periodic(8, 8, 8))
    for key in ("zchunk_flux", "zchunk_div", "zchunk_sensor"):
        for v in (1, 7, -1):
            with pytest.raises(B.OcfdError, match="invalid"):
                s.set_tuning(key, v)
        s.set_tuning(key, 8)
        s.set_tuning(key, 0)
    for key in ("xy_fused", "zchunk", ""):
        with pytest.raises(B.OcfdError, match="invalid"):
            s.set_tuning(key, 1)
    s.set_tuning("march_seg", 3)
    s.set_tuning("tile_group", 1)
    s.close()


def test_invalid_parameters_are_refused_without_touching_buffers(B):
    """Argument errors come back as status codes (never exceptions from the library), synchronously."""
    case = W.smooth_periodic(8, 8, 8)
    for field, bad in (("nx", 9), ("nx", 6), ("visc_order", 7), ("bc_closure", 2), ("char_recon", -1)):
        broken = W.smooth_periodic(8, 8, 8)
        if field == "nx":
            broken.nx = bad          # odd, or below the minimum
        else:
            setattr(broken, field, bad)
        with pytest.raises(Exception) as e:
            B.Solver(broken)
        assert "invalid" in str(e.value).lower() or "workspace" in str(e.value).lower() or "shape" in str(e.value).lower()
    s = B.Solver(case)               # and a valid one still works afterwards
    s.close()


def test_ten_steps_characteristic_reconstruction(B, Oracle):
    case = W.tgv(24, nsteps=10)
    case.char_recon = 1
    err, _, _ = step_both(B, Oracle, case, 10, check_every=5)
    print("TGV 24^3, WENO7 in characteristic variables, 10 steps: rel Linf", err)
    assert err <= TOL_100


def test_ten_steps_eighth_order_viscous_scheme(B, Oracle):
    case = W.tgv(24, nsteps=10)
    case.visc_order = 8
    err, _, _ = step_both(B, Oracle, case, 10, check_every=5)
    print("TGV 24^3, 8th-order viscous scheme, 10 steps: rel Linf", err)
    assert err <= TOL_100


def step_both(B, Oracle, case, nsteps, check_every=None):
    o = Oracle(case)
    U = o.fill_ghosts(case.U0.copy())
    dt = case.cfl / o.max_wavespeed(U)
    s = B.Solver(case)
    Ud = s.to_device(U)
    lam = s.max_wavespeed(Ud)
    assert lam == pytest.approx(case.cfl / dt, rel=1e-13)
    worst = 0.0
    for n in range(nsteps):
        o.rk3_step(U, dt)
        s.rk3_step(Ud, dt)
        if check_every and ((n + 1) % check_every == 0 or n == nsteps - 1):
            got = Ud.cpu().numpy()
            worst = max(worst, rel_linf(got[INT], U[INT], U[INT], floor=1e-3 * np.abs(U[INT]).max()).max())
    got = Ud.cpu().numpy()
    s.close()
    umax = np.abs(U[INT]).max()
    err = rel_linf(got[INT], U[INT], U[INT], floor=1e-3 * umax)
    # both sides leave the face ghosts filled; edges and corners are never touched by either
    errg = max(np.abs(got[m] - U[m]).max() / max(np.abs(U[m]).max(), 1e-3 * umax) for m in range(5))
    return max(worst, err.max(), errg), got, U


def test_config1_tgv32_ten_steps(B, Oracle):
    case = W.tgv(32)
    err, _, _ = step_both(B, Oracle, case, case.nsteps, check_every=1)
    print("config 1 (TGV 32^3, 10 steps): rel Linf", err)
    assert err <= TOL_100


def test_hundred_steps_smooth(B, Oracle):
    case = W.tgv(24, nsteps=100)
    err, _, _ = step_both(B, Oracle, case, 100, check_every=25)
    print("TGV 24^3, 100 steps: rel Linf", err)
    assert err <= TOL_100


@pytest.mark.parametrize("which", ["plate", "ramp", "ramp3level"])
def test_twenty_steps_with_walls(B, Oracle, which):
    """20 steps with wall / inflow / outflow faces.  The hybrid cases carry no loosened bar: every interface whose Theta
    comes within 1e-9 of a threshold at any stage is counted, and the 1e-9 bar holds outside its domain of influence
    (everywhere when there is none); the sensor decisions of the two sides are compared at every step."""
    from tests.parity_utils import step_both_hybrid
    if which == "plate":
        case = W.flat_plate(nx=64, ny=40, nz=16)
    else:
        case = W.ramp(nx=64, ny=40, nz=16, nmodes=12, theta2=np.inf if which == "ramp" else 0.1)
    res = step_both_hybrid(B, Oracle, case, 20)
    assert res["finite"] and res["flag_mismatches"] == 0
    if res["err_all"] > TOL_100:
        assert res["near"] > 0 and res["excluded_fraction"] < 1.0 and res["err_outside"] <= TOL_100, res
    assert res["err_padded_outside"] <= TOL_100, res          # face ghosts of the stepped state included
