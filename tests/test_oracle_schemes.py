"""Pins of the oracle's reconstruction schemes (UD7, WENO7, WENO5) against what the paper prints and
what the definitions fix.  CPU only.  See DESIGN.md section 4 for what each pin can catch."""
import os

import numpy as np
import pytest
from numpy.polynomial import polynomial as Pl

GOLD = os.path.join(os.path.dirname(__file__), "golden")
C7 = np.array([1.0, 12.0, 18.0, 4.0]) / 35.0
C5 = np.array([0.1, 0.6, 0.3])
BIG = 1e40  # eps so large that the nonlinear weights collapse onto the linear ones


def load_rows(name):
    rows = []
    with open(os.path.join(GOLD, name)) as fh:
        for ln in fh:
            if ln.strip() and not ln.startswith("#"):
                rows.append([float(t) for t in ln.split()])
    return rows


def cell_averages(coef, centres):
    """Exact cell averages over [c-1/2, c+1/2] of the polynomial with ascending coefficients coef."""
    anti = Pl.polyint(coef)
    return np.array([Pl.polyval(c + 0.5, anti) - Pl.polyval(c - 0.5, anti) for c in centres])


def candidate_poly(vals, centres):
    """Polynomial (ascending coeffs, degree len(vals)-1) whose cell averages on `centres` equal vals."""
    n = len(vals)
    A = np.zeros((n, n))
    for m in range(n):
        e = np.zeros(n)
        e[m] = 1.0
        A[:, m] = cell_averages(e, centres)
    return np.linalg.solve(A, np.asarray(vals, dtype=np.float64))


def smoothness_by_quadrature(coef):
    """sum_l int_{-1/2}^{1/2} (d^l p / dx^l)^2 dx, l = 1..deg, cell width 1, Gauss-Legendre."""
    xg, wg = np.polynomial.legendre.leggauss(10)
    xg, wg = 0.5 * xg, 0.5 * wg
    total, d = 0.0, np.array(coef, dtype=np.float64)
    for _ in range(len(coef) - 1):
        d = Pl.polyder(d)
        total += np.sum(wg * Pl.polyval(xg, d) ** 2)
    return total


# ----------------------------------------------------------------------------- UD7
def test_ud7_coefficients_are_eq41(ora):
    coef, den = load_rows("ud7_eq41.txt")
    for r in range(7):
        e = np.zeros(7)
        e[r] = 1.0
        assert ora.ud7(e) == pytest.approx(coef[r] / den[0], rel=0, abs=1e-16)


def test_ud7_reproduces_degree6_polynomials(ora):
    rng = np.random.default_rng(1)
    for deg in range(7):
        coef = rng.uniform(-1, 1, deg + 1)
        f = cell_averages(coef, np.arange(-3, 4))
        assert ora.ud7(f) == pytest.approx(Pl.polyval(0.5, coef), abs=2e-13)
    # and not degree 7: the scheme is exactly seventh order
    f = cell_averages(np.eye(8)[7], np.arange(-3, 4))
    assert abs(ora.ud7(f) - 0.5 ** 7) > 1e-3


def test_ud7_flux_difference_is_exact_derivative_for_degree7_point_values(ora):
    # (f^_{j+1/2} - f^_{j-1/2})/h = f'(x_j) for point values of polynomials up to degree 7
    rng = np.random.default_rng(2)
    for deg in range(8):
        coef = rng.uniform(-1, 1, deg + 1)
        pts = Pl.polyval(np.arange(-4, 4, dtype=np.float64), coef)   # f_{j-4..j+3}
        d = ora.ud7(pts[1:8]) - ora.ud7(pts[0:7])
        assert d == pytest.approx(Pl.polyval(0.0, Pl.polyder(coef)), abs=5e-12)


# ----------------------------------------------------------------------------- WENO7
def test_weno7_linear_weights_give_eq41(ora):
    coef, den = load_rows("ud7_eq41.txt")
    Q = np.zeros((4, 7))
    for r in range(7):
        e = np.zeros(7)
        e[r] = 1.0
        Q[:, r] = ora.weno7_parts(e)[0]
    assert np.allclose(C7 @ Q, np.array(coef) / den[0], rtol=0, atol=2e-16)
    rng = np.random.default_rng(3)
    for _ in range(20):
        f = rng.uniform(-2, 2, 7)
        assert ora.weno7(f, BIG) == pytest.approx(ora.ud7(f), abs=1e-14)


def test_weno7_candidates_reproduce_cubics(ora):
    rng = np.random.default_rng(4)
    for _ in range(5):
        coef = rng.uniform(-1, 1, 4)
        q = ora.weno7_parts(cell_averages(coef, np.arange(-3, 4)))[0]
        assert np.allclose(q, Pl.polyval(0.5, coef), atol=1e-13)
    # each candidate only looks at its own four cells
    for k in range(4):
        for r in range(7):
            e = np.zeros(7)
            e[r] = 1.0
            inside = k <= r <= k + 3
            assert (ora.weno7_parts(e)[0][k] != 0.0) == inside


def test_weno7_smoothness_indicators_match_integral_definition(ora):
    rng = np.random.default_rng(5)
    for _ in range(10):
        f = rng.uniform(-3, 3, 7)
        IS = ora.weno7_parts(f)[1]
        for k in range(4):
            cen = np.arange(-3 + k, 1 + k)
            ref = smoothness_by_quadrature(candidate_poly(f[k:k + 4], cen))
            assert IS[k] == pytest.approx(ref, rel=1e-11)


def test_weno7_indicators_zero_on_constants_and_nonnegative(ora):
    assert np.all(ora.weno7_parts(np.full(7, 3.25))[1] == 0.0)
    rng = np.random.default_rng(6)
    for _ in range(200):
        assert np.all(ora.weno7_parts(rng.standard_normal(7))[1] >= 0.0)


def test_weno7_weights_convex_and_definition(ora):
    rng = np.random.default_rng(7)
    for _ in range(50):
        f = rng.uniform(-1, 1, 7)
        eps = 1e-6
        q, IS, om = ora.weno7_parts(f, eps)
        al = C7 / (eps + IS) ** 2
        assert np.allclose(om, al / al.sum(), rtol=1e-14)
        assert om.sum() == pytest.approx(1.0, abs=1e-15) and np.all(om > 0)
        v = ora.weno7(f, eps)
        assert v == pytest.approx(np.dot(om, q), rel=1e-15, abs=1e-16)
        assert q.min() - 1e-14 <= v <= q.max() + 1e-14


def test_weno7_weights_tend_to_linear_on_smooth_data(ora):
    dev = []
    for h in (0.2, 0.1, 0.05):
        x = 0.3 + h * np.arange(-3, 4)
        om = ora.weno7_parts(np.sin(x) + 2.0, 1e-40)[2]
        dev.append(np.abs(om - C7).max())
    assert dev[0] > dev[1] > dev[2]
    assert dev[1] / dev[2] > 2.0 ** 2.5      # at least O(h^3) asymptotically
    assert dev[2] < 1e-3


def test_weno7_eno_property_on_a_step(ora):
    for jump_at in range(1, 7):
        f = np.where(np.arange(7) < jump_at, 0.0, 1.0)
        v = ora.weno7(f, 1e-6)
        # a smooth (constant) sub-stencil exists on one side of the jump unless it sits at j+1/2 itself
        target = f[3] if jump_at != 4 else None
        assert -1e-3 <= v <= 1.0 + 1e-3
        if target is not None and jump_at not in (3, 4):
            assert abs(v - target) < 1e-3 or abs(v - f[4]) < 1e-3


# ----------------------------------------------------------------------------- WENO5
def test_weno5_linear_weights_and_candidates(ora):
    lin = np.array([2.0, -13.0, 47.0, 27.0, -3.0]) / 60.0
    Q = np.zeros((3, 5))
    for r in range(5):
        e = np.zeros(5)
        e[r] = 1.0
        Q[:, r] = ora.weno5_parts(e)[0]
    assert np.allclose(C5 @ Q, lin, atol=2e-16)
    rng = np.random.default_rng(8)
    for deg in range(5):
        coef = rng.uniform(-1, 1, deg + 1)
        f = cell_averages(coef, np.arange(-2, 3))
        assert ora.weno5(f, BIG) == pytest.approx(Pl.polyval(0.5, coef), abs=1e-13)
        if deg <= 2:
            assert np.allclose(ora.weno5_parts(f)[0], Pl.polyval(0.5, coef), atol=1e-13)


def test_weno5_smoothness_indicators_match_integral_definition(ora):
    rng = np.random.default_rng(9)
    for _ in range(10):
        f = rng.uniform(-3, 3, 5)
        IS = ora.weno5_parts(f)[1]
        for k in range(3):
            ref = smoothness_by_quadrature(candidate_poly(f[k:k + 3], np.arange(-2 + k, 1 + k)))
            assert IS[k] == pytest.approx(ref, rel=1e-11)


def test_weno5_weights_convex(ora):
    rng = np.random.default_rng(10)
    for _ in range(50):
        f = rng.uniform(-1, 1, 5)
        q, IS, om = ora.weno5_parts(f, 1e-6)
        al = C5 / (1e-6 + IS) ** 2
        assert np.allclose(om, al / al.sum(), rtol=1e-14)
        v = ora.weno5(f, 1e-6)
        assert q.min() - 1e-14 <= v <= q.max() + 1e-14


def test_weno_same_normalisation_for_5_and_7(ora):
    # DESIGN R-9: both indicator families follow the same integral definition, so on a pure parabola
    # (second difference 1, zero first derivative at x_j) the central candidates agree: 13/12.
    f7 = 0.5 * np.arange(-3, 4, dtype=np.float64) ** 2
    assert ora.weno7_parts(f7)[1][1] == pytest.approx(13.0 / 12.0, rel=1e-14)
    assert ora.weno5_parts(f7[1:6])[1][1] == pytest.approx(13.0 / 12.0, rel=1e-14)
