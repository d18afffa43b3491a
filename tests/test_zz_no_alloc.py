"""ocfd_max_wavespeed_static: the one entry point for callers that cannot allocate device memory.

Some code that wants dt = CFL / Lambda runs where cudaMalloc is not an option: inside an application whose own memory
pool already owns the whole GPU, in a monitoring hook that must leave the allocator alone, or under a memory budget that
is spent on the flow fields.  Such a caller cannot give a context the workspace it asks for, so this entry point works
without a context; its reduction scratch is a fixed 512.25 KiB array inside the library, shared by every call on a
device (include/ocfd.h).  What is checked here:

  * the value equals the context path's (ocfd_max_wavespeed) within the 1e-13 the wavespeed parity test uses, on two
    calls in a row that differ in grid size, grid kind and magnitude -- the second call must not see anything the
    first one left in the shared array (a larger grid with a larger Lambda goes first, so stale slots would win);
  * a NaN state comes back as NaN and does not poison the next call;
  * a grid beyond the array's limit is refused before anything runs;
  * the calls do not change the amount of free device memory.

The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here should hide nothing.
The tests neither need nor assume that another test has run before them in the same process.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2209_15333_b200 import workloads as W

pytestmark = pytest.mark.gpu

NG = 4
REL = 1e-13          # tolerance of test_max_wavespeed_matches_the_oracle


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_2209_15333_b200 import binding
    binding.load()
    return binding


def params_without_workspace(B, s):
    """The solver's parameter block (it holds the device pointers of the metric arrays), stripped of the workspace:
    the static entry point must not need one."""
    P = B.OcfdParams.from_buffer_copy(s.P)
    P.workspace = None
    P.workspace_bytes = 0
    return P


def louder(case, factor):
    """The same flow with every velocity scaled up: a state whose Lambda is clearly larger."""
    U = case.U0.copy()
    ke_old = 0.5 * (U[1] ** 2 + U[2] ** 2 + U[3] ** 2) / U[0]
    U[1:4] *= factor
    U[4] += (factor ** 2 - 1.0) * ke_old
    return U


@pytest.mark.parametrize("first, second", [("wavy_big", "ramp_small"), ("plate_big", "uniform_small"),
                                           ("ramp_big", "wavy_small")])
def test_two_calls_in_a_row_match_the_context_path(B, first, second):
    make = {
        "wavy_big": lambda: W.smooth_periodic(150, 45, 70, grid="wavy"),      # full 3-D metrics, ragged in x
        "wavy_small": lambda: W.smooth_periodic(24, 16, 12, grid="wavy", seed=3),
        "ramp_big": lambda: W.ramp(nx=192, ny=44, nz=80, nmodes=12),          # z-extruded map, several z chunks
        "ramp_small": lambda: W.ramp(nx=64, ny=24, nz=16, nmodes=8),
        "plate_big": lambda: W.flat_plate(nx=136, ny=44, nz=72),              # stretched
        "uniform_small": lambda: W.tgv(16),
    }
    ca, cb = make[first](), make[second]()
    sa, sb = B.Solver(ca), B.Solver(cb)
    Ua = sa.to_device(louder(ca, 3.0) if "plate" not in first else ca.U0)
    Ub = sb.to_device(cb.U0)
    want_a, want_b = sa.max_wavespeed(Ua), sb.max_wavespeed(Ub)              # the existing path, each in its own context
    assert np.isfinite(want_a) and np.isfinite(want_b) and want_a > 0.0 and want_b > 0.0
    Pa, Pb = params_without_workspace(B, sa), params_without_workspace(B, sb)
    got_a = B.max_wavespeed_static(Pa, Ua.data_ptr())                        # call 1: the larger problem
    got_b = B.max_wavespeed_static(Pb, Ub.data_ptr())                        # call 2, straight after it
    got_a2 = B.max_wavespeed_static(Pa, Ua.data_ptr())                       # and back
    assert got_a == pytest.approx(want_a, rel=REL)
    assert got_b == pytest.approx(want_b, rel=REL)
    assert got_a2 == got_a
    sa.close()
    sb.close()


def test_runs_with_no_context_alive(B):
    """Nothing but the parameter block, U and the result pointer: no Solver, no workspace, no context ever created."""
    import torch
    case = W.tgv(24)
    P = B.params_from_case(case)
    P.stream = torch.cuda.current_stream().cuda_stream
    U = torch.as_tensor(case.U0, dtype=torch.float64).cuda()
    lam = B.max_wavespeed_static(P, U.data_ptr())
    # closed form on a uniform grid: max over points of sum_d (|u_d| + c) / h_d
    Ui = case.U0[:, NG:-NG, NG:-NG, NG:-NG]
    u = Ui[1:4] / Ui[0]
    p = (case.gamma - 1.0) * (Ui[4] - 0.5 * Ui[0] * (u ** 2).sum(axis=0))
    c = np.sqrt(case.gamma * p / Ui[0])
    want = ((np.abs(u[0]) + c) / case.dx + (np.abs(u[1]) + c) / case.dy + (np.abs(u[2]) + c) / case.dz).max()
    assert lam == pytest.approx(want, rel=1e-12)


def test_nan_state_is_reported_and_forgotten(B):
    case = W.smooth_periodic(40, 24, 18, grid="wavy")
    s = B.Solver(case)
    P = params_without_workspace(B, s)
    clean = s.to_device(case.U0)
    want = s.max_wavespeed(clean)
    U = case.U0.copy()
    U[4, NG + 5, NG + 7, NG + 11] = np.nan
    assert np.isnan(B.max_wavespeed_static(P, s.to_device(U).data_ptr()))
    assert B.max_wavespeed_static(P, clean.data_ptr()) == pytest.approx(want, rel=REL)   # the NaN slot is not seen again
    s.close()


def test_grid_beyond_the_static_scratch_is_refused(B):
    """ceil(nx/128) * ny = 8 * 8200 > 65536 slots: OCFD_EWORKSPACE (-2) before U is looked at (a 64-byte buffer stands in
    for a 5 GB state), with the reason on stderr and in the binding's exception."""
    import torch
    L = B.load()
    case = W.tgv(16)
    P = B.params_from_case(case)
    P.nx, P.ny, P.nz = 1024, 8200, 16
    P.stream = torch.cuda.current_stream().cuda_stream
    dummy = torch.zeros(8, dtype=torch.float64, device="cuda")
    out = C.c_double(-1.0)
    assert L.ocfd_max_wavespeed_static(C.byref(P), dummy.data_ptr(), C.byref(out)) == -2
    assert out.value == -1.0
    with pytest.raises(B.OcfdError, match="workspace"):
        B.max_wavespeed_static(P, dummy.data_ptr())
    # parameters a context would reject, and null pointers, are argument errors
    Q = B.params_from_case(case)
    Q.nx = 4
    assert L.ocfd_max_wavespeed_static(C.byref(Q), dummy.data_ptr(), C.byref(out)) == -1
    assert L.ocfd_max_wavespeed_static(C.byref(B.params_from_case(case)), None, C.byref(out)) == -1
    assert L.ocfd_max_wavespeed_static(C.byref(B.params_from_case(case)), dummy.data_ptr(), None) == -1
    assert out.value == -1.0


def test_calls_leave_free_device_memory_unchanged(B):
    import torch
    case = W.ramp(nx=64, ny=24, nz=16, nmodes=8)
    s = B.Solver(case)
    P = params_without_workspace(B, s)
    U = s.to_device(case.U0)
    B.max_wavespeed_static(P, U.data_ptr())       # first call on the device: address look-up, kernels loaded
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    vals = [B.max_wavespeed_static(P, U.data_ptr()) for _ in range(5)]
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    assert len(set(vals)) == 1
    s.close()
