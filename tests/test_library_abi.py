"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/ocfd.h declares, and validates
arguments synchronously (no kernel is launched here)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2209_15333_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_2209_15333_b200 import build, binding
    build.build()
    binding.load()
    return binding


def test_library_exports_every_declared_symbol(B):
    hdr = open(os.path.join(ROOT, "include", "ocfd.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(ocfd_[a-z0-9_]+)\s*\(", hdr))
    assert declared, "no declarations found"
    L = B.load()
    for name in sorted(declared):
        assert hasattr(L, name), name
    assert declared == set(B.EXPORTS)


def test_params_struct_mirror_and_validation(B):
    L = B.load()
    assert L.ocfd_sizeof_params() == C.sizeof(B.OcfdParams)
    case = W.tgv(16)
    P = B.params_from_case(case)
    nbytes = L.ocfd_workspace_bytes(C.byref(P))
    npad = (16 + 8) ** 3
    assert nbytes >= 23 * npad * 8 and nbytes % 256 == 0      # theta 1 + Fv 12 + U^n 5 + dU 5 fields (no primitive fields)
    case.inviscid = True
    assert L.ocfd_workspace_bytes(C.byref(B.params_from_case(case))) < nbytes   # no viscous-flux fields
    # invalid parameters are rejected without touching anything
    for mutate in (lambda p: setattr(p, "ng", 3), lambda p: setattr(p, "nx", 4), lambda p: setattr(p, "gamma", 1.0),
                   lambda p: setattr(p, "weno_eps", 0.0), lambda p: setattr(p, "weno_eps", 1e-60),
                   lambda p: setattr(p, "scheme", 7),
                   lambda p: p.bc.__setitem__(0, B.BCS["outflow"]),          # periodic not paired
                   lambda p: setattr(p, "grid_kind", B.GRID_KINDS["curvilinear"])):   # metrics missing
        Q = B.params_from_case(W.tgv(16))
        mutate(Q)
        assert L.ocfd_workspace_bytes(C.byref(Q)) == 0
        ctx = C.c_void_p()
        assert L.ocfd_init(C.byref(ctx), C.byref(Q)) == -1 and not ctx.value
    # valid parameters but no workspace
    ctx = C.c_void_p()
    assert L.ocfd_init(C.byref(ctx), C.byref(P)) == -2
    assert L.ocfd_strerror(-2).decode().startswith("workspace")
    # a dead context is refused
    assert L.ocfd_rk3_step(None, None, 0.1) == -5
    assert L.ocfd_launch_count(None) == -1


def test_binding_refuses_to_run_without_a_gpu(B):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        B.Solver(W.tgv(16))


def test_product_path_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2209_15333_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("test oracle", "").replace("the oracle", "").replace("CPU oracle", "") \
                    or f == "workloads.py", f


def test_static_wavespeed_size_limit_is_checked_on_the_host(B):
    """ocfd_max_wavespeed_static (the entry point for callers that cannot allocate device memory) refuses a grid beyond
    its fixed scratch array, and bad arguments, before it touches the GPU: none is needed to see that."""
    L = B.load()
    P = B.params_from_case(W.tgv(16))
    P.nx, P.ny, P.nz = 1024, 8200, 16                      # ceil(1024/128) * 8200 = 65600 > 65536 slots
    never_read = (C.c_double * 8)()
    out = C.c_double(-1.0)
    assert L.ocfd_max_wavespeed_static(C.byref(P), never_read, C.byref(out)) == -2
    P.nx = 6
    assert L.ocfd_max_wavespeed_static(C.byref(P), never_read, C.byref(out)) == -1
    assert L.ocfd_max_wavespeed_static(C.byref(B.params_from_case(W.tgv(16))), None, C.byref(out)) == -1
    assert out.value == -1.0
