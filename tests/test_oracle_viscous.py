"""Pins of the oracle's central differences and viscous terms.  CPU only."""
import numpy as np
import pytest
from numpy.polynomial import polynomial as Pl

from paper_2209_15333_b200 import workloads as W

NG = 4


# ------------------------------------------------------------------ first derivative
def test_d1_interior_is_sixth_order_exact(ora):
    rng = np.random.default_rng(0)
    n = 16
    x = np.arange(n, dtype=np.float64)
    for deg in range(7):
        coef = rng.uniform(-1, 1, deg + 1) / 10.0 ** np.arange(deg + 1)
        d = ora.d1_line(Pl.polyval(x, coef), periodic=False)
        ref = Pl.polyval(x, Pl.polyder(coef))
        assert np.allclose(d[3:n - 3], ref[3:n - 3], atol=1e-11)
    d = ora.d1_line(x ** 7, periodic=False)
    assert abs(d[8] - 7 * x[8] ** 6) > 1.0      # not exact for degree 7


def test_d1_closure_rows_have_the_orders_the_paper_states(ora):
    """one-sided 2nd order at the boundary point; 2nd / 4th / 6th order central at the
    2nd / 3rd / 4th points."""
    n = 12
    x = np.arange(n, dtype=np.float64)
    exact_deg = {0: 2, 1: 2, 2: 4, 3: 6}
    for row, deg in exact_deg.items():
        for dd in range(deg + 1):
            f = (x - 3.3) ** dd
            ref = dd * (x - 3.3) ** max(dd - 1, 0) if dd > 0 else 0 * x
            d = ora.d1_line(f, periodic=False)
            assert d[row] == pytest.approx(ref[row], abs=1e-9), (row, dd)
            assert d[n - 1 - row] == pytest.approx(ref[n - 1 - row], abs=1e-9), (row, dd)
        f = (x - 3.3) ** (deg + 1)
        ref = (deg + 1) * (x - 3.3) ** deg
        d = ora.d1_line(f, periodic=False)
        assert abs(d[row] - ref[row]) > 1e-3, row
    # the closure never reads outside the line: poison the neighbours
    buf = np.full(n + 8, np.nan)
    buf[4:4 + n] = x ** 2
    assert np.all(np.isfinite(ora.d1_line(buf[4:4 + n].copy(), periodic=False)))


def test_d1_periodic_wraps(ora):
    n = 24
    x = 2 * np.pi * np.arange(n) / n
    d = ora.d1_line(np.sin(x), periodic=True) / (2 * np.pi / n)
    assert np.allclose(d, np.cos(x), atol=2e-5)
    d2 = ora.d1_line(np.sin(2 * np.pi * np.arange(2 * n) / (2 * n)), periodic=True) / (2 * np.pi / (2 * n))
    e1 = np.abs(d - np.cos(x)).max()
    e2 = np.abs(d2 - np.cos(2 * np.pi * np.arange(2 * n) / (2 * n))).max()
    assert 50 < e1 / e2 < 80      # 2^6 = 64


# ------------------------------------------------------------------ 8th-order scheme
def test_d1_eighth_order_coefficients_are_the_unique_antisymmetric_nine_point_stencil(ora):
    """The 9-point antisymmetric stencil exact for x, x^3, x^5, x^7 is unique: solve for it and compare with what the
    oracle applies to unit impulses (4/5, -1/5, 4/105, -1/280)."""
    m = np.arange(1, 5, dtype=np.float64)
    A = np.array([2 * m ** (2 * q + 1) for q in range(4)])      # sum_m c_m (m^p - (-m)^p) = p x^(p-1) at x = 0
    c = np.linalg.solve(A, np.array([1.0, 0.0, 0.0, 0.0]))
    assert np.allclose(c, [4 / 5, -1 / 5, 4 / 105, -1 / 280], rtol=1e-12)
    n = 20
    for k, ck in enumerate(c, start=1):
        e = np.zeros(n)
        e[10 + k] = 1.0
        assert ora.d1_line(e, periodic=True, order=8)[10] == pytest.approx(ck, rel=1e-14)
        e[:] = 0.0
        e[10 - k] = 1.0
        assert ora.d1_line(e, periodic=True, order=8)[10] == pytest.approx(-ck, rel=1e-14)


def test_d1_eighth_order_exactness_and_closure_rows(ora):
    rng = np.random.default_rng(8)
    n = 18
    x = np.arange(n, dtype=np.float64)
    for deg in range(9):
        coef = rng.uniform(-1, 1, deg + 1) / 10.0 ** np.arange(deg + 1)
        d = ora.d1_line(Pl.polyval(x, coef), periodic=False, order=8)
        ref = Pl.polyval(x, Pl.polyder(coef))
        assert np.allclose(d[4:n - 4], ref[4:n - 4], atol=1e-10)
    d = ora.d1_line((x - 9.0) ** 9, periodic=False, order=8)
    assert abs(d[11] - 9 * (x[11] - 9.0) ** 8) > 1.0          # not exact for degree 9
    # rows 0..3 and mirrored: one-sided 2nd, central 2nd, 4th, 6th
    for row, deg in {0: 2, 1: 2, 2: 4, 3: 6}.items():
        for dd in range(deg + 1):
            f = (x - 3.3) ** dd
            ref = dd * (x - 3.3) ** max(dd - 1, 0) if dd > 0 else 0 * x
            d = ora.d1_line(f, periodic=False, order=8)
            assert d[row] == pytest.approx(ref[row], abs=1e-8), (row, dd)
            assert d[n - 1 - row] == pytest.approx(ref[n - 1 - row], abs=1e-6 * max(1.0, abs(ref[n - 1 - row]))), (row, dd)
        f = (x - 3.3) ** (deg + 1)
        assert abs(ora.d1_line(f, periodic=False, order=8)[row] - (deg + 1) * (x[row] - 3.3) ** deg) > 1e-3, row
    # rows 0..2 are the same rows as in the 6th-order scheme; the 6th-order scheme has no fourth row
    f = np.sin(0.7 * x)
    d6, d8 = ora.d1_line(f, periodic=False, order=6), ora.d1_line(f, periodic=False, order=8)
    assert np.array_equal(d6[:4], d8[:4]) and np.array_equal(d6[-4:], d8[-4:])
    assert np.all(d6[4:-4] != d8[4:-4])


def test_d1_eighth_order_periodic_convergence(ora):
    errs = []
    for n in (16, 32):
        x = 2 * np.pi * np.arange(n) / n
        d = ora.d1_line(np.sin(x), periodic=True, order=8) / (2 * np.pi / n)
        errs.append(np.abs(d - np.cos(x)).max())
    assert 200 < errs[0] / errs[1] < 300      # 2^8 = 256


# ------------------------------------------------------------------ manufactured viscous RHS
def _manufactured(case, const_T=False):
    """Smooth 2pi-periodic u,v,w,T (rho = 1) and the analytic viscous RHS of rows 2-5, via sympy."""
    import sympy as sp
    x, y, z = sp.symbols("x y z")
    u = 1 + sp.Rational(3, 10) * sp.sin(x) * sp.cos(2 * y) + sp.Rational(1, 5) * sp.cos(z + y)
    v = sp.Rational(-1, 2) + sp.Rational(1, 4) * sp.cos(x + z) * sp.sin(y) + sp.Rational(1, 10) * sp.sin(2 * z)
    w = sp.Rational(1, 5) + sp.Rational(3, 10) * sp.sin(y + 2 * z) + sp.Rational(1, 5) * sp.cos(x) * sp.cos(y)
    T = sp.Integer(1) if const_T else 1 + sp.Rational(1, 5) * sp.sin(x + y) * sp.cos(z) + sp.Rational(1, 10) * sp.cos(2 * x)
    S = sp.Float(case.T_suth) / sp.Float(case.T_ref)
    mu = (1 + S) / (T + S) * T ** sp.Rational(3, 2) / case.Re
    kc = mu / ((case.gamma - 1) * case.Ma ** 2 * case.Pr)
    vel, X = [u, v, w], [x, y, z]
    div = sum(sp.diff(vel[i], X[i]) for i in range(3))
    tau = [[mu * (sp.diff(vel[i], X[j]) + sp.diff(vel[j], X[i])) - (sp.Rational(2, 3) * mu * div if i == j else 0)
            for j in range(3)] for i in range(3)]
    rhs = [sum(sp.diff(tau[i][j], X[j]) for j in range(3)) for i in range(3)]
    rhs.append(sum(sp.diff(sum(vel[i] * tau[i][j] for i in range(3)) + kc * sp.diff(T, X[j]), X[j]) for j in range(3)))
    fn = sp.lambdify((x, y, z), [u, v, w, T] + rhs, "numpy")
    return fn, (sp.lambdify((x, y, z), [sp.diff(vel[i], X[i], 2) * 0 + sum(sp.diff(vel[i], X[j], 2) for j in range(3))
                                       + sp.Rational(1, 3) * sp.diff(div, X[i]) for i in range(3)], "numpy"))


def _viscous_error(ora, grid, n, const_T=False, order=6):
    from oracle.oracle import Oracle
    case = W.smooth_periodic(n, n, n, grid=grid, Re=50.0, Ma=0.6)
    case.visc_order = order
    fn, lap = _manufactured(case, const_T)
    X, Y, Z = case.coords
    u, v, w, T, r1, r2, r3, r4 = [np.broadcast_to(a, X.shape) for a in fn(X, Y, Z)]
    rho = np.ones_like(u)
    p = rho * T / (case.gamma * case.Ma ** 2)
    U = np.stack([W.pad_wrap(c) for c in W.cons_from_prim(rho, u, v, w, p, case.gamma)])
    case.inviscid = False
    full = Oracle(case).rhs(np.ascontiguousarray(U))
    case.inviscid = True
    inv = Oracle(case).rhs(np.ascontiguousarray(U))
    visc = (full - inv)[:, NG:-NG, NG:-NG, NG:-NG]
    assert np.all(visc[0] == 0.0)                      # no viscous flux in the continuity row
    ref = np.stack([r1, r2, r3, r4])
    err = np.abs(visc[1:] - ref).max() / np.abs(ref).max()
    if const_T:  # textbook constant-viscosity form mu/Re (lap u + grad div u / 3)
        l1, l2, l3 = [np.broadcast_to(a, X.shape) for a in lap(X, Y, Z)]
        assert np.allclose(ref[:3], np.stack([l1, l2, l3]) / case.Re, atol=1e-12)
    return err


@pytest.mark.parametrize("grid", ["uniform", "stretched", "wavy"])
def test_viscous_terms_converge_at_sixth_order_to_the_analytic_rhs(ora, grid):
    # the field carries wavenumber-2 modes, so 24 -> 48 points is where the asymptotic rate shows
    e1, e2 = _viscous_error(ora, grid, 24), _viscous_error(ora, grid, 48)
    assert e2 < 1e-4
    assert e1 / e2 > 2.0 ** 5.4, (e1, e2)


@pytest.mark.parametrize("grid", ["uniform", "wavy"])
def test_viscous_terms_eighth_order_scheme_converges_faster(ora, grid):
    """Same manufactured field with the 8th-order central scheme: two applications of an 8th-order derivative.  On the
    wavy grid the analytic metrics are exact, so the rate is that of the scheme."""
    e1, e2 = _viscous_error(ora, grid, 24, order=8), _viscous_error(ora, grid, 48, order=8)
    assert e2 < 3e-6
    assert e1 / e2 > 2.0 ** 7.2, (e1, e2)
    assert e2 < 0.2 * _viscous_error(ora, grid, 48, order=6)


def test_viscous_constant_viscosity_special_case(ora):
    assert _viscous_error(ora, "uniform", 24, const_T=True) < 2e-3


def test_viscous_flux_point_against_hand_formulas(ora):
    """Cartesian metrics, one point: tau_ij and Theta of eq. 12-13 written out by hand."""
    from oracle.oracle import Oracle
    case = W.smooth_periodic(8, 8, 8, Re=100.0, Ma=0.5)
    o = Oracle(case)
    rng = np.random.default_rng(1)
    g = rng.uniform(-1, 1, (4, 3))            # d(u,v,w,T)/d(x,y,z) when metrics are the identity
    m = np.eye(3).ravel()
    u, v, w, T = 0.3, -0.6, 0.9, 1.4
    out = o.viscous_flux_point(g, m, 1.0, u, v, w, T)
    mu = o.mu(T) / case.Re
    kc = o.mu(T) / ((case.gamma - 1) * case.Ma ** 2 * case.Pr * case.Re)   # eq. 14
    div = g[0, 0] + g[1, 1] + g[2, 2]
    tau = np.array([[mu * (g[i, j] + g[j, i]) - (2.0 / 3.0 * mu * div if i == j else 0.0) for j in range(3)]
                    for i in range(3)])
    vel = np.array([u, v, w])
    for d in range(3):
        assert np.allclose(out[d, :3], tau[:, d], rtol=1e-13)
        assert out[d, 3] == pytest.approx(vel @ tau[:, d] + kc * g[3, d], rel=1e-13)
    # J^-1 scaling and metric rotation: a 90-degree relabelling of the axes permutes the fluxes
    out2 = o.viscous_flux_point(g, m, 4.0, u, v, w, T)
    assert np.allclose(out2, out / 4.0, rtol=1e-14)
