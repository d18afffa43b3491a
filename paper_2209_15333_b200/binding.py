"""Thin Python binding of the C-ABI library libocfd_b200.so (include/ocfd.h).

Argument marshalling only: every step of the hot path runs in the library's CUDA kernels.  PyTorch supplies
device memory and the stream.  There is no CPU fallback: `load()` raises if the library has not been built
and `Solver` raises if no CUDA device is present.
"""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "csrc", "libocfd_b200.so")

NG = 4
GRID_KINDS = {"uniform": 0, "stretched": 1, "curvilinear": 2}
SCHEMES = {"ud7": 0, "weno7": 1, "weno5": 2, "hybrid": 3}
BCS = {"periodic": 0, "wall": 1, "inflow": 2, "outflow": 3}
OCFD_OK = 0

EXPORTS = ["ocfd_workspace_bytes", "ocfd_init", "ocfd_destroy", "ocfd_fill_ghosts", "ocfd_rhs", "ocfd_rk3_step",
           "ocfd_rk3_steps_host", "ocfd_max_wavespeed", "ocfd_debug_sensor", "ocfd_timing", "ocfd_timing_read",
           "ocfd_kernel_name", "ocfd_sizeof_params", "ocfd_launch_count", "ocfd_strerror", "ocfd_set_tuning",
           "ocfd_max_wavespeed_static", "ocfd_check_state"]
NKERNELS = 10


class OcfdParams(C.Structure):
    """Mirror of `ocfd_params` in include/ocfd.h."""
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("ng", C.c_int),
        ("grid_kind", C.c_int),
        ("metric", C.c_void_p * 10),
        ("metric_plane_stride", C.c_longlong),
        ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
        ("gamma", C.c_double), ("Ma", C.c_double), ("Re", C.c_double), ("Pr", C.c_double),
        ("T_ref", C.c_double), ("T_suth", C.c_double),
        ("inviscid", C.c_int),
        ("scheme", C.c_int),
        ("theta1", C.c_double), ("theta2", C.c_double),
        ("weno_eps", C.c_double), ("sw_eps", C.c_double),
        ("bc", C.c_int * 6),
        ("T_wall", C.c_double * 6),
        ("wall_vn", C.c_void_p * 6),
        ("inflow", C.c_void_p * 6),
        ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
        ("stream", C.c_void_p),
        ("visc_order", C.c_int),
        ("bc_closure", C.c_int),
        ("char_recon", C.c_int),
    ]


_LIB = None


def load():
    """Load libocfd_b200.so and declare the prototypes of every symbol include/ocfd.h exports."""
    global _LIB
    if _LIB is not None:
        return _LIB
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2209_15333_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    pp = C.POINTER(OcfdParams)
    vp = C.c_void_p
    L.ocfd_workspace_bytes.restype = C.c_size_t
    L.ocfd_workspace_bytes.argtypes = [pp]
    L.ocfd_init.restype = C.c_int
    L.ocfd_init.argtypes = [C.POINTER(vp), pp]
    L.ocfd_destroy.restype = C.c_int
    L.ocfd_destroy.argtypes = [vp]
    L.ocfd_fill_ghosts.restype = C.c_int
    L.ocfd_fill_ghosts.argtypes = [vp, vp]
    L.ocfd_rhs.restype = C.c_int
    L.ocfd_rhs.argtypes = [vp, vp, vp]
    L.ocfd_rk3_step.restype = C.c_int
    L.ocfd_rk3_step.argtypes = [vp, vp, C.c_double]
    L.ocfd_rk3_steps_host.restype = C.c_int
    L.ocfd_rk3_steps_host.argtypes = [vp, vp, vp, C.c_double, C.c_int]
    L.ocfd_max_wavespeed.restype = C.c_int
    L.ocfd_max_wavespeed.argtypes = [vp, vp, C.POINTER(C.c_double)]
    L.ocfd_max_wavespeed_static.restype = C.c_int
    L.ocfd_max_wavespeed_static.argtypes = [pp, vp, C.POINTER(C.c_double)]
    L.ocfd_check_state.restype = C.c_int
    L.ocfd_check_state.argtypes = [vp, vp, C.POINTER(C.c_longlong)]
    L.ocfd_debug_sensor.restype = C.c_int
    L.ocfd_debug_sensor.argtypes = [vp, vp, vp, vp]
    L.ocfd_launch_count.restype = C.c_longlong
    L.ocfd_launch_count.argtypes = [vp]
    L.ocfd_strerror.restype = C.c_char_p
    L.ocfd_strerror.argtypes = [C.c_int]
    L.ocfd_timing.restype = C.c_int
    L.ocfd_timing.argtypes = [vp, C.c_int]
    L.ocfd_timing_read.restype = C.c_int
    L.ocfd_timing_read.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
    L.ocfd_kernel_name.restype = C.c_char_p
    L.ocfd_kernel_name.argtypes = [C.c_int]
    L.ocfd_set_tuning.restype = C.c_int
    L.ocfd_set_tuning.argtypes = [vp, C.c_char_p, C.c_int]
    L.ocfd_sizeof_params.restype = C.c_size_t
    L.ocfd_sizeof_params.argtypes = []
    if L.ocfd_sizeof_params() != C.sizeof(OcfdParams):
        raise RuntimeError("OcfdParams does not mirror ocfd_params (include/ocfd.h)")
    _LIB = L
    return L


class OcfdError(RuntimeError):
    pass


def _check(status):
    if status != OCFD_OK:
        raise OcfdError(f"ocfd status {status}: {load().ocfd_strerror(status).decode()}")


def params_from_case(case):
    """Fill an OcfdParams from a case object (host scalars only; device pointers are set by Solver)."""
    P = OcfdParams()
    P.nx, P.ny, P.nz, P.ng = case.nx, case.ny, case.nz, NG
    P.grid_kind = GRID_KINDS[case.grid_kind]
    P.dx, P.dy, P.dz = case.dx, case.dy, case.dz
    P.gamma, P.Ma, P.Re, P.Pr = case.gamma, case.Ma, case.Re, case.Pr
    P.T_ref, P.T_suth = case.T_ref, case.T_suth
    P.inviscid = 1 if case.inviscid else 0
    P.visc_order = int(getattr(case, "visc_order", 6))
    P.bc_closure = int(getattr(case, "bc_closure", 0))
    P.char_recon = int(getattr(case, "char_recon", 0))
    P.scheme = SCHEMES[case.scheme]
    P.theta1, P.theta2 = case.theta1, case.theta2
    P.weno_eps, P.sw_eps = case.weno_eps, case.sw_eps
    for f in range(6):
        P.bc[f] = BCS[case.bc[f]]
        P.T_wall[f] = case.T_wall[f]
    return P


def max_wavespeed_static(P, U_ptr):
    """ocfd_max_wavespeed_static: Lambda of the state at device address `U_ptr` for the grid and gas an OcfdParams `P`
    describes, with no context and no workspace.  For callers that may not allocate device memory; the scratch is a
    fixed array inside the library (limits and sharing rules: include/ocfd.h)."""
    out = C.c_double(0.0)
    _check(load().ocfd_max_wavespeed_static(C.byref(P), U_ptr, C.byref(out)))
    return out.value


class Solver:
    """One ocfd context on the current CUDA device.  Same method names as the C entry points."""

    def __init__(self, case, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2209_15333_b200 needs a CUDA device (B200, sm_100a); there is no CPU fallback")
        self.torch = torch
        self.L = load()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.case_shape = (5, case.nz + 2 * NG, case.ny + 2 * NG, case.nx + 2 * NG)
        self.npoints = case.nx * case.ny * case.nz
        P = params_from_case(case)
        self._keep = []

        def dev(a):
            t = torch.as_tensor(a, dtype=torch.float64).contiguous().to(self.device)
            self._keep.append(t)
            return t.data_ptr()
        if case.grid_kind == "stretched":
            for q, a in zip((0, 4, 8), case.metric1d):
                P.metric[q] = dev(a)
        elif case.grid_kind == "curvilinear":
            planes = case.metrics[0].shape[0]
            for q in range(10):
                assert case.metrics[q].shape[0] == planes
                P.metric[q] = dev(case.metrics[q])
            P.metric_plane_stride = 0 if planes == 1 else (case.nx + 2 * NG) * (case.ny + 2 * NG)
        for f in range(6):
            if case.wall_vn[f] is not None:
                P.wall_vn[f] = dev(case.wall_vn[f])
            if case.inflow[f] is not None:
                P.inflow[f] = dev(case.inflow[f])
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        P.stream = self.stream.cuda_stream
        nbytes = self.L.ocfd_workspace_bytes(C.byref(P))
        if nbytes == 0:
            raise OcfdError("ocfd_workspace_bytes rejected the parameters")
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = self.workspace.data_ptr()
        P.workspace = (base + 255) // 256 * 256
        P.workspace_bytes = nbytes
        self.P = P
        self.ctx = C.c_void_p()
        _check(self.L.ocfd_init(C.byref(self.ctx), C.byref(P)))

    def close(self):
        if getattr(self, "ctx", None) is not None and self.ctx.value:
            self.L.ocfd_destroy(self.ctx)
            self.ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ------------------------------------------------------------------ helpers
    def to_device(self, U_host):
        t = self.torch.as_tensor(U_host, dtype=self.torch.float64).contiguous().to(self.device)
        assert tuple(t.shape) == self.case_shape, (tuple(t.shape), self.case_shape)
        return t

    def _ptr(self, t):
        assert t.is_cuda and t.dtype == self.torch.float64 and t.is_contiguous() and tuple(t.shape) == self.case_shape
        return t.data_ptr()

    # ------------------------------------------------------------------ the C entry points
    def fill_ghosts(self, U):
        _check(self.L.ocfd_fill_ghosts(self.ctx, self._ptr(U)))
        return U

    def rhs(self, U, dU=None):
        if dU is None:
            dU = self.torch.zeros_like(U)
        _check(self.L.ocfd_rhs(self.ctx, self._ptr(U), self._ptr(dU)))
        return dU

    def rk3_step(self, U, dt):
        _check(self.L.ocfd_rk3_step(self.ctx, self._ptr(U), float(dt)))
        return U

    def rk3_steps_host(self, U_host, U_dev, dt, nsteps=1):
        """U_host: pinned (or pageable) CPU tensor / numpy array of the state, updated in place."""
        if hasattr(U_host, "data_ptr"):
            hp = U_host.data_ptr()
            assert U_host.dtype == self.torch.float64 and U_host.is_contiguous() and tuple(U_host.shape) == self.case_shape
        else:
            assert U_host.dtype.name == "float64" and U_host.flags["C_CONTIGUOUS"] and U_host.shape == self.case_shape
            hp = U_host.ctypes.data
        _check(self.L.ocfd_rk3_steps_host(self.ctx, hp, self._ptr(U_dev), float(dt), int(nsteps)))
        return U_host

    def max_wavespeed(self, U):
        out = C.c_double(0.0)
        _check(self.L.ocfd_max_wavespeed(self.ctx, self._ptr(U), C.byref(out)))
        return out.value

    def check_state(self, U):
        """(points with a non-finite conserved variable, points with rho <= 0, points with p <= 0) over the interior."""
        counts = (C.c_longlong * 3)()
        _check(self.L.ocfd_check_state(self.ctx, self._ptr(U), counts))
        return tuple(int(v) for v in counts)

    def debug_sensor(self, U):
        theta = self.torch.full(self.case_shape[1:], float("nan"), dtype=self.torch.float64, device=self.device)
        flags = self.torch.full((3,) + self.case_shape[1:], 255, dtype=self.torch.uint8, device=self.device)
        _check(self.L.ocfd_debug_sensor(self.ctx, self._ptr(U), theta.data_ptr(), flags.data_ptr()))
        return theta, flags

    def timing(self, enable):
        _check(self.L.ocfd_timing(self.ctx, 1 if enable else 0))

    def timing_read(self):
        """{kernel class name: (total ms, launches)} since the last read."""
        ms = (C.c_double * NKERNELS)()
        n = (C.c_longlong * NKERNELS)()
        _check(self.L.ocfd_timing_read(self.ctx, ms, n))
        return {self.L.ocfd_kernel_name(k).decode(): (ms[k], n[k]) for k in range(NKERNELS)}

    def set_tuning(self, key, value):
        _check(self.L.ocfd_set_tuning(self.ctx, key.encode(), int(value)))

    def launch_count(self):
        return int(self.L.ocfd_launch_count(self.ctx))
