"""ctypes front end of the CPU oracle (oracle/ocfd_oracle.c).  TEST INFRASTRUCTURE, not product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It imports nothing from the CUDA path (paper_2209_15333_b200); a "case" is any object
with the attributes listed in `params_from_case` (the seeded generators in
paper_2209_15333_b200/workloads.py produce such objects for both sides).
"""
import ctypes as C
import os

import numpy as np

NG = 4
SCHEMES = {"ud7": 0, "weno7": 1, "weno5": 2, "hybrid": 3}
BCS = {"periodic": 0, "wall": 1, "inflow": 2, "outflow": 3}

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

_dp = C.POINTER(C.c_double)


class OraParams(C.Structure):
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
        ("met", _dp * 10),
        ("met_sk", C.c_long),
        ("gamma", C.c_double), ("Ma", C.c_double), ("Re", C.c_double), ("Pr", C.c_double),
        ("T_ref", C.c_double), ("T_suth", C.c_double),
        ("inviscid", C.c_int), ("scheme", C.c_int),
        ("theta1", C.c_double), ("theta2", C.c_double), ("weno_eps", C.c_double), ("sw_eps", C.c_double),
        ("bc", C.c_int * 6),
        ("T_wall", C.c_double * 6),
        ("wall_vn", _dp * 6),
        ("inflow", _dp * 6),
        ("visc_order", C.c_int),
        ("bc_closure", C.c_int),
        ("char_recon", C.c_int),
    ]


def lib():
    """Load (building if needed) the oracle shared library."""
    global _LIB
    if _LIB is None:
        import importlib.util
        spec = importlib.util.spec_from_file_location("_ora_build", os.path.join(_HERE, "build.py"))
        mod = importlib.util.module_from_spec(spec)
        spec.loader.exec_module(mod)
        L = C.CDLL(mod.build())
        assert L.ora_sizeof_params() == C.sizeof(OraParams), "ctypes mirror of ora_params is out of date"
        L.ora_ud7.restype = C.c_double
        L.ora_weno7.restype = C.c_double
        L.ora_weno5.restype = C.c_double
        L.ora_mu.restype = C.c_double
        L.ora_max_wavespeed.restype = C.c_double
        L.ora_sizeof_params.restype = C.c_long
        _LIB = L
    return _LIB


def _ptr(a):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_dp)


# ------------------------------------------------------------------ pointwise building blocks
def ud7(f):
    f = np.ascontiguousarray(f, dtype=np.float64)
    assert f.shape == (7,)
    return lib().ora_ud7(_ptr(f))


def weno7(f, eps=1e-6):
    f = np.ascontiguousarray(f, dtype=np.float64)
    assert f.shape == (7,)
    return lib().ora_weno7(_ptr(f), C.c_double(eps))


def weno7_parts(f, eps=1e-6):
    f = np.ascontiguousarray(f, dtype=np.float64)
    q, IS, om = np.zeros(4), np.zeros(4), np.zeros(4)
    lib().ora_weno7_parts(_ptr(f), C.c_double(eps), _ptr(q), _ptr(IS), _ptr(om))
    return q, IS, om


def weno5(f, eps=1e-6):
    f = np.ascontiguousarray(f, dtype=np.float64)
    assert f.shape == (5,)
    return lib().ora_weno5(_ptr(f), C.c_double(eps))


def eigen_matrices(gamma, u, v, w, c, n):
    """S (eq. 35) and S^-1 (eq. 34) of PAPER.md:L236-238 for the unit direction n."""
    n = np.ascontiguousarray(n, dtype=np.float64)
    S, Si = np.zeros((5, 5)), np.zeros((5, 5))
    d = C.c_double
    lib().ora_eigen_matrices(d(gamma), d(u), d(v), d(w), d(c), _ptr(n), _ptr(S), _ptr(Si))
    return S, Si


def weno5_masked(f, keep, nearest, eps=1e-6):
    """Shielded WENO5 of the paper's boundary scheme; bit k of `keep` = candidate k is inside."""
    f = np.ascontiguousarray(f, dtype=np.float64)
    assert f.size == 5
    L = lib()
    L.ora_weno5_masked.restype = C.c_double
    return float(L.ora_weno5_masked(_ptr(f), C.c_double(eps), C.c_int(keep), C.c_double(nearest)))


def weno5_parts(f, eps=1e-6):
    f = np.ascontiguousarray(f, dtype=np.float64)
    q, IS, om = np.zeros(3), np.zeros(3), np.zeros(3)
    lib().ora_weno5_parts(_ptr(f), C.c_double(eps), _ptr(q), _ptr(IS), _ptr(om))
    return q, IS, om


def sw_split(gamma, rho, u, v, w, c, alpha, sw_eps=0.0):
    fp, fm = np.zeros(5), np.zeros(5)
    d = C.c_double
    lib().ora_sw_split(d(gamma), d(sw_eps), d(rho), d(u), d(v), d(w), d(c),
                       d(alpha[0]), d(alpha[1]), d(alpha[2]), _ptr(fp), _ptr(fm))
    return fp, fm


def d1_line(f, periodic, order=6):
    f = np.ascontiguousarray(f, dtype=np.float64)
    out = np.zeros_like(f)
    lib().ora_d1_line(_ptr(f), C.c_int(f.size), C.c_int(1 if periodic else 0), C.c_int(order), _ptr(out))
    return out


# ------------------------------------------------------------------ field-level oracle
def params_from_case(case):
    """Build (OraParams, keepalive list) from a case object.

    Needed attributes: nx ny nz; metrics (list of 10 float64 arrays of shape (nz+8 or 1, ny+8, nx+8));
    gamma Ma Re Pr T_ref T_suth; inviscid; scheme (str); theta1 theta2 weno_eps sw_eps;
    bc (6 str); T_wall (6 floats); wall_vn, inflow (6 arrays or None each).
    """
    P = OraParams()
    keep = []
    P.nx, P.ny, P.nz = case.nx, case.ny, case.nz
    nzp, nyp, nxp = case.nz + 2 * NG, case.ny + 2 * NG, case.nx + 2 * NG
    planes = None
    for q in range(10):
        a = np.ascontiguousarray(case.metrics[q], dtype=np.float64)
        assert a.shape in ((nzp, nyp, nxp), (1, nyp, nxp)), a.shape
        planes = a.shape[0] if planes is None else planes
        assert a.shape[0] == planes
        keep.append(a)
        P.met[q] = _ptr(a)
    P.met_sk = nyp * nxp if planes == nzp else 0
    P.gamma, P.Ma, P.Re, P.Pr = case.gamma, case.Ma, case.Re, case.Pr
    P.T_ref, P.T_suth = case.T_ref, case.T_suth
    P.inviscid = 1 if case.inviscid else 0
    P.visc_order = int(getattr(case, "visc_order", 6))
    P.bc_closure = int(getattr(case, "bc_closure", 0))
    P.char_recon = int(getattr(case, "char_recon", 0))
    P.scheme = SCHEMES[case.scheme]
    P.theta1, P.theta2 = case.theta1, case.theta2
    P.weno_eps, P.sw_eps = case.weno_eps, case.sw_eps
    dims = (case.nx, case.ny, case.nz)
    for f in range(6):
        P.bc[f] = BCS[case.bc[f]]
        P.T_wall[f] = case.T_wall[f]
        d = f // 2
        t1 = 1 if d == 0 else 0
        t2 = 1 if d == 2 else 2
        shape2 = (dims[t2] + 2 * NG, dims[t1] + 2 * NG)
        if case.wall_vn[f] is not None:
            a = np.ascontiguousarray(case.wall_vn[f], dtype=np.float64)
            assert a.shape == shape2, (a.shape, shape2)
            keep.append(a)
            P.wall_vn[f] = _ptr(a)
        if case.inflow[f] is not None:
            a = np.ascontiguousarray(case.inflow[f], dtype=np.float64)
            assert a.shape == (5,) + shape2, (a.shape, shape2)
            keep.append(a)
            P.inflow[f] = _ptr(a)
    return P, keep


class Oracle:
    """The oracle bound to one case's grid, gas and scheme parameters."""

    def __init__(self, case):
        self.P, self._keep = params_from_case(case)
        self.shape = (5, case.nz + 2 * NG, case.ny + 2 * NG, case.nx + 2 * NG)
        self.L = lib()

    def _chk(self, U):
        assert U.dtype == np.float64 and U.flags["C_CONTIGUOUS"] and U.shape == self.shape, (U.shape, self.shape)

    def fill_ghosts(self, U):
        self._chk(U)
        self.L.ora_fill_ghosts(C.byref(self.P), _ptr(U))
        return U

    def rhs(self, U):
        self._chk(U)
        dU = np.zeros_like(U)
        self.L.ora_rhs(C.byref(self.P), _ptr(U), _ptr(dU))
        return dU

    def inviscid_dir(self, U, d):
        self._chk(U)
        dU = np.zeros_like(U)
        self.L.ora_inviscid_dir(C.byref(self.P), _ptr(U), C.c_int(d), _ptr(dU))
        return dU

    def rhs_points(self, U, ijk):
        self._chk(U)
        ijk = np.ascontiguousarray(ijk, dtype=np.int32)
        assert ijk.ndim == 2 and ijk.shape[1] == 3
        out = np.zeros((ijk.shape[0], 5))
        self.L.ora_rhs_points(C.byref(self.P), _ptr(U), C.c_long(ijk.shape[0]),
                              ijk.ctypes.data_as(C.POINTER(C.c_int)), _ptr(out))
        return out

    def rk3_update(self, Un, U, dU, dt, stage):
        self._chk(U)
        self.L.ora_rk3_update(C.byref(self.P), _ptr(Un), _ptr(U), _ptr(dU), C.c_double(dt), C.c_int(stage))
        return U

    def rk3_step(self, U, dt):
        self._chk(U)
        self.L.ora_rk3_step(C.byref(self.P), _ptr(U), C.c_double(dt))
        return U

    def max_wavespeed(self, U):
        self._chk(U)
        return self.L.ora_max_wavespeed(C.byref(self.P), _ptr(U))

    def check_state(self, U):
        """(points with a non-finite conserved variable, points with rho <= 0, points with p <= 0) over the interior."""
        self._chk(U)
        counts = (C.c_longlong * 3)()
        self.L.ora_check_state(C.byref(self.P), _ptr(U), counts)
        return tuple(int(v) for v in counts)

    def sensor(self, U):
        self._chk(U)
        th = np.full(self.shape[1:], np.nan)
        self.L.ora_sensor(C.byref(self.P), _ptr(U), _ptr(th))
        return th

    def flags(self, theta, d):
        fl = np.full(self.shape[1:], 255, dtype=np.uint8)
        self.L.ora_flags(C.byref(self.P), _ptr(theta), C.c_int(d), fl.ctypes.data_as(C.POINTER(C.c_ubyte)))
        return fl

    def mu(self, T):
        return self.L.ora_mu(C.byref(self.P), C.c_double(T))

    def prim_point(self, U5):
        U5 = np.ascontiguousarray(U5, dtype=np.float64)
        out = np.zeros(7)
        self.L.ora_prim_point(C.byref(self.P), _ptr(U5), _ptr(out))
        return out

    def viscous_flux_point(self, g, m, J, u, v, w, T):
        g = np.ascontiguousarray(g, dtype=np.float64)
        m = np.ascontiguousarray(m, dtype=np.float64)
        assert g.shape == (4, 3) and m.shape == (9,)
        out = np.zeros((3, 4))
        d = C.c_double
        self.L.ora_viscous_flux_point(C.byref(self.P), _ptr(g), _ptr(m), d(J), d(u), d(v), d(w), d(T), _ptr(out))
        return out
