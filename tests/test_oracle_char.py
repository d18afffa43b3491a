"""Pins of the oracle's flux reconstruction in characteristic variables (section 2.2.2; SURVEY
8(f) NEXT #2; reading DESIGN R-22).  CPU only.

The paper prints S^-1 (eq. 34), S (eq. 35), kappa, kappa1, chi (eq. 36), l (eq. 39) and m (eq. 40).  What fixes them:
S S^-1 = I; S^-1 Lambda S equals the Jacobian of the inviscid flux of eq. 6 in direction n (finite differences), with
Lambda of eq. 33; (l, m, n) orthonormal and right-handed.  What fixes the way they are used: for a linear scheme the
projection cancels (UD7 in characteristic variables = UD7 component by component, to round-off), and on the Sod tube
WENO in characteristic variables keeps the exact-solution bounds better than component-wise WENO.
"""
import numpy as np
import pytest

from paper_2209_15333_b200 import workloads as W

NG = 4
INT = (slice(None), slice(NG, -NG), slice(NG, -NG), slice(NG, -NG))
GAMMA = 1.4


def random_states(seed, k):
    rng = np.random.default_rng(seed)
    out = []
    dirs = [np.array(v, dtype=float) for v in ((1, 0, 0), (0, 1, 0), (0, 0, 1), (0, 0.6, 0.8), (0.6, 0, -0.8))]
    for q in range(k):
        n = dirs[q] if q < len(dirs) else rng.normal(size=3)
        n = n / np.linalg.norm(n)
        out.append((rng.uniform(0.5, 2.0), rng.uniform(-1, 1, 3), rng.uniform(0.5, 2.0), n))
    return out


def flux_n(U, n):
    rho, m, E = U[0], U[1:4], U[4]
    vel = m / rho
    p = (GAMMA - 1.0) * (E - 0.5 * rho * vel @ vel)
    un = vel @ n
    return np.concatenate([[rho * un], m * un + p * n, [(E + p) * un]])


def test_S_times_S_inverse_is_identity_and_frame_is_orthonormal(ora):
    for rho, vel, p, n in random_states(0, 40):
        c = np.sqrt(GAMMA * p / rho)
        S, Si = ora.eigen_matrices(GAMMA, vel[0], vel[1], vel[2], c, n)
        assert np.allclose(S @ Si, np.eye(5), atol=1e-13)
        assert np.allclose(Si @ S, np.eye(5), atol=1e-13)
        l, m = S[1, 1:4], S[2, 1:4]
        assert np.allclose([l @ l, m @ m, l @ m, l @ n, m @ n], [1, 1, 0, 0, 0], atol=1e-14)
        assert np.allclose(np.cross(n, l), m, atol=1e-14)                        # eq. 40
        if abs(n[2]) <= abs(n[1]):                                               # eq. 39
            assert l[2] == 0.0 and np.allclose(l[:2] * np.hypot(n[0], n[1]), [-n[1], n[0]], atol=1e-14)
        else:
            assert l[1] == 0.0 and np.allclose(l[[0, 2]] * np.hypot(n[0], n[2]), [-n[2], n[0]], atol=1e-14)


def test_S_diagonalises_the_flux_jacobian_with_the_eigenvalues_of_eq_33(ora):
    for rho, vel, p, n in random_states(1, 25):
        c = np.sqrt(GAMMA * p / rho)
        U = np.concatenate([[rho], rho * vel, [p / (GAMMA - 1.0) + 0.5 * rho * vel @ vel]])
        A = np.empty((5, 5))
        for k in range(5):
            h = 1e-6 * max(1.0, abs(U[k]))
            e = np.zeros(5)
            e[k] = h
            A[:, k] = (flux_n(U + e, n) - flux_n(U - e, n)) / (2 * h)
        S, Si = ora.eigen_matrices(GAMMA, vel[0], vel[1], vel[2], c, n)
        un = vel @ n
        Lam = np.diag([un, un, un, un - c, un + c])
        assert np.allclose(Si @ Lam @ S, A, atol=2e-8 * np.abs(A).max())


@pytest.mark.parametrize("grid", ["uniform", "wavy"])
def test_linear_scheme_is_unchanged_by_the_projection(grid):
    from oracle.oracle import Oracle
    case = W.smooth_periodic(14, 10, 9, grid=grid, scheme="ud7", inviscid=True)
    o = Oracle(case)
    U = o.fill_ghosts(case.U0.copy())
    a = o.rhs(U)[INT]
    case.char_recon = 1
    b = Oracle(case).rhs(U)[INT]
    assert np.abs(a - b).max() <= 1e-12 * np.abs(a).max()
    assert not np.array_equal(a, b)                      # it did go through the projection


def test_weno_in_characteristic_variables_differs_and_converges_alike():
    from oracle.oracle import Oracle
    case = W.smooth_periodic(16, 10, 9, grid="wavy", scheme="weno7", inviscid=True)
    o = Oracle(case)
    U = o.fill_ghosts(case.U0.copy())
    a = o.rhs(U)[INT]
    case.char_recon = 1
    b = Oracle(case).rhs(U)[INT]
    d = np.abs(a - b).max() / np.abs(a).max()
    assert 1e-9 < d < 5e-2                               # a different nonlinear scheme of the same accuracy


def _sod_run(n, char):
    from oracle.oracle import Oracle
    from tests.test_oracle_time import exact_sod
    case = W.sod(n=n, scheme="weno7")
    case.char_recon = char
    o = Oracle(case)
    U = case.U0.copy()
    t_end, dt0 = 0.2, 0.4 * case.dx / 2.2
    nst = int(np.ceil(t_end / dt0))
    for _ in range(nst):
        o.rk3_step(U, t_end / nst)
    x = case.coords[0][NG:-NG]
    rho = U[0, NG, NG, NG:-NG]
    er, _, _ = exact_sod(x, t_end)
    return rho, er


def test_sod_tube_characteristic_weno_is_at_least_as_monotone():
    rho_c, er = _sod_run(200, 1)
    rho_p, _ = _sod_run(200, 0)
    assert np.mean(np.abs(rho_c - er)) < 4e-3                    # same accuracy bar as the component-wise run
    tv = lambda r: np.abs(np.diff(r)).sum()
    tv_exact = 1.0 - 0.125                                       # monotone exact profile
    assert tv(rho_c) - tv_exact <= tv(rho_p) - tv_exact + 1e-12  # no more spurious variation than component-wise
    assert rho_c.max() <= 1.0 + 1e-3 and rho_c.min() >= 0.125 - 1e-3
