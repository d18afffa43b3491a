"""Properties that hold at any size, checked on the CUDA path itself (through the C ABI): the whole pipeline (ghost fill,
RHS, RK3) advects the isentropic vortex at the design order against its analytic solution, and the Sod tube converges to
the exact Riemann solution.  These are the pins of the oracle (tests/test_oracle_time.py) run on the GPU; the exact
solutions are analytic, nothing here comes from the oracle."""
import numpy as np
import pytest

from paper_2209_15333_b200 import workloads as W
from tests.test_oracle_time import exact_sod

pytestmark = pytest.mark.gpu

NG = 4
I3 = (slice(NG, -NG), slice(NG, -NG), slice(NG, -NG))


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_2209_15333_b200 import binding
    binding.load()
    return binding


def _vortex_error(B, n, scheme, t_end=0.5):
    kw = dict(n=n, nz=8, scheme=scheme, uinf=1.0, vinf=1.0, L=16.0)
    case = W.vortex(**kw)
    s = B.Solver(case)
    U = s.to_device(case.U0.copy())
    s.fill_ghosts(U)
    nst = int(np.ceil(t_end * s.max_wavespeed(U) / 0.4))
    for _ in range(nst):
        s.rk3_step(U, t_end / nst)
    got = U.cpu().numpy()
    s.close()
    exact = W.vortex(t=t_end, **kw).U0
    return np.abs(got[0] - exact[0])[I3].max()


@pytest.mark.parametrize("scheme,rate", [("ud7", 4.5), ("weno7", 3.5), ("hybrid", 3.5)])
def test_vortex_advection_on_the_gpu_tracks_the_exact_solution(B, scheme, rate):
    e = [_vortex_error(B, n, scheme) for n in (32, 64)]
    print(scheme, "max density error at n = 32, 64:", e, "observed order", np.log2(e[0] / e[1]))
    assert e[1] < 1e-3
    assert np.log2(e[0] / e[1]) > rate, e


@pytest.mark.parametrize("scheme", ["weno7", "hybrid"])
def test_sod_tube_on_the_gpu_converges_to_the_exact_riemann_solution(B, scheme):
    errs = []
    for n in (100, 200):
        case = W.sod(n=n, scheme=scheme, ny=8, nz=8)
        s = B.Solver(case)
        U = s.to_device(case.U0.copy())
        t_end, dt0 = 0.2, 0.4 * case.dx / 2.2
        nst = int(np.ceil(t_end / dt0))
        for _ in range(nst):
            s.rk3_step(U, t_end / nst)
        got = U.cpu().numpy()
        s.close()
        x = case.coords[0][NG:-NG]
        rho = got[0, NG, NG, NG:-NG]
        er, _, _ = exact_sod(x, t_end)
        errs.append(np.mean(np.abs(rho - er)))
        assert np.abs(got[2:4][(slice(None),) + I3]).max() < 1e-12          # the flow stays one-dimensional
    print(scheme, "L1 density error at n = 100, 200:", errs)
    assert errs[1] < 4e-3
    assert 1.4 < errs[0] / errs[1] < 3.0
    assert rho.max() <= 1.0 + 0.01 and rho.min() >= 0.125 - 0.01 * 0.875
