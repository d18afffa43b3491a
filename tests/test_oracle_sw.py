"""Pins of the oracle's Steger-Warming split and thermodynamics.  CPU only."""
import numpy as np
import pytest


def random_state(rng, mach_range=(0.0, 3.0)):
    gamma = rng.choice([1.4, 1.3, 5.0 / 3.0])
    rho, c = rng.uniform(0.2, 3.0), rng.uniform(0.3, 4.0)
    dirn = rng.standard_normal(3)
    dirn /= np.linalg.norm(dirn)
    vel = dirn * c * rng.uniform(*mach_range)
    alpha = rng.standard_normal(3) * rng.uniform(0.1, 5.0)
    return gamma, rho, vel, c, alpha


def exact_flux(gamma, rho, vel, c, alpha):
    """eq. 6 with alpha = (d_x,d_y,d_z)/J:  [rho V, rho u V + a1 p, ..., (E+p) V]."""
    p = rho * c * c / gamma
    E = p / (gamma - 1.0) + 0.5 * rho * vel.dot(vel)
    Vt = alpha.dot(vel)
    return np.array([rho * Vt, *(rho * vel * Vt + alpha * p), (E + p) * Vt])


def paper_eigen_matrices(gamma, vel, c, n):
    """S^-1 (eq. 34) and S (eq. 35) exactly as printed at PAPER.md:L236-238, l and m from eq. 39-40."""
    u, v, w = vel
    n1, n2, n3 = n
    if abs(n3) <= abs(n2):
        l = np.array([-n2, n1, 0.0]) / np.sqrt(n1 * n1 + n2 * n2)
    else:
        l = np.array([-n3, 0.0, n1]) / np.sqrt(n1 * n1 + n3 * n3)
    m = np.cross(n, l)
    un, ul, um = vel.dot(n), vel.dot(l), vel.dot(m)
    V = 0.5 * vel.dot(vel)
    H = V + c * c / (gamma - 1.0)
    kap = (gamma - 1.0) / (c * c)
    k1, chi = 0.5 * kap, 0.5 / c
    Sinv = np.array([
        [1.0, 0.0, 0.0, 1.0, 1.0],
        [u, l[0], m[0], u - c * n1, u + c * n1],
        [v, l[1], m[1], v - c * n2, v + c * n2],
        [w, l[2], m[2], w - c * n3, w + c * n3],
        [V, ul, um, H - c * un, H + c * un]])
    S = np.array([
        [1.0 - kap * V, kap * u, kap * v, kap * w, -kap],
        [-ul, l[0], l[1], l[2], 0.0],
        [-um, m[0], m[1], m[2], 0.0],
        [k1 * V + chi * un, -chi * n1 - k1 * u, -chi * n2 - k1 * v, -chi * n3 - k1 * w, k1],
        [k1 * V - chi * un, chi * n1 - k1 * u, chi * n2 - k1 * v, chi * n3 - k1 * w, k1]])
    return Sinv, S


def test_split_sums_to_exact_flux(ora):
    rng = np.random.default_rng(0)
    for _ in range(200):
        gamma, rho, vel, c, alpha = random_state(rng)
        fp, fm = ora.sw_split(gamma, rho, *vel, c, alpha)
        ref = exact_flux(gamma, rho, vel, c, alpha)
        assert np.allclose(fp + fm, ref, rtol=0, atol=2e-13 * np.abs(ref).max())


def test_split_equals_paper_eigen_decomposition(ora):
    """f+- = S^-1 Lambda+- S U with the matrices printed in the paper (eq. 31-35): pins every row
    of the split flux, including the energy row garbled at PAPER.md:L182 (DESIGN R-5)."""
    rng = np.random.default_rng(1)
    for _ in range(100):
        gamma, rho, vel, c, alpha = random_state(rng)
        sigma = np.linalg.norm(alpha)
        n = alpha / sigma
        Sinv, S = paper_eigen_matrices(gamma, vel, c, n)
        assert np.allclose(S @ Sinv, np.eye(5), atol=1e-12)
        p = rho * c * c / gamma
        Ucons = np.array([rho, *(rho * vel), p / (gamma - 1.0) + 0.5 * rho * vel.dot(vel)])
        un = vel.dot(n)
        lam = sigma * np.array([un, un, un, un - c, un + c])                 # eq. 33
        fp, fm = ora.sw_split(gamma, rho, *vel, c, alpha)
        for sign, f in ((1.0, fp), (-1.0, fm)):
            ref = Sinv @ (0.5 * (lam + sign * np.abs(lam)) * (S @ Ucons))     # eq. 29
            assert np.allclose(f, ref, rtol=0, atol=5e-12 * max(1.0, np.abs(ref).max()))


def test_split_is_one_sided_when_supersonic(ora):
    rng = np.random.default_rng(2)
    seen = 0
    for _ in range(300):
        gamma, rho, vel, c, alpha = random_state(rng, (1.2, 3.0))
        sigma, Vt = np.linalg.norm(alpha), alpha.dot(vel)
        fp, fm = ora.sw_split(gamma, rho, *vel, c, alpha)
        if Vt > 1.01 * c * sigma:
            assert np.all(fm == 0.0)
            seen += 1
        elif Vt < -1.01 * c * sigma:
            assert np.all(fp == 0.0)
            seen += 1
    assert seen > 20


def test_split_jacobians_have_signed_eigenvalues(ora):
    """d f+/dU has eigenvalues >= 0 and d f-/dU <= 0 (finite differences, away from sonic points)."""
    rng = np.random.default_rng(3)
    from oracle.oracle import Oracle
    from paper_2209_15333_b200 import workloads as W
    case = W.smooth_periodic(8, 8, 8)
    done = 0
    while done < 20:
        gamma, rho, vel, c, alpha = random_state(rng, (0.1, 2.0))
        mach_n = alpha.dot(vel) / (c * np.linalg.norm(alpha))
        if min(abs(mach_n), abs(abs(mach_n) - 1.0)) < 0.1:
            continue
        case.gamma, case.Ma = gamma, 0.7
        o = Oracle(case)
        p = rho * c * c / gamma
        U0 = np.array([rho, *(rho * vel), p / (gamma - 1.0) + 0.5 * rho * vel.dot(vel)])

        def F(U):
            q = o.prim_point(U)  # rho u v w p T c
            return ora.sw_split(gamma, q[0], q[1], q[2], q[3], q[6], alpha)
        Jp, Jm = np.zeros((5, 5)), np.zeros((5, 5))
        for m in range(5):
            h = 1e-6 * max(1.0, abs(U0[m]))
            e = np.zeros(5)
            e[m] = h
            (ap, am), (bp, bm) = F(U0 + e), F(U0 - e)
            Jp[:, m], Jm[:, m] = (ap - bp) / (2 * h), (am - bm) / (2 * h)
        scale = (abs(alpha.dot(vel)) + c * np.linalg.norm(alpha))
        assert np.linalg.eigvals(Jp).real.min() > -1e-5 * scale
        assert np.linalg.eigvals(Jm).real.max() < 1e-5 * scale
        done += 1


def test_split_rotational_covariance(ora):
    rng = np.random.default_rng(4)
    for _ in range(50):
        gamma, rho, vel, c, alpha = random_state(rng)
        Q, _ = np.linalg.qr(rng.standard_normal((3, 3)))
        fp, fm = ora.sw_split(gamma, rho, *vel, c, alpha)
        gp, gm = ora.sw_split(gamma, rho, *(Q @ vel), c, Q @ alpha)
        for f, g in ((fp, gp), (fm, gm)):
            s = max(1.0, np.abs(f).max())
            assert g[0] == pytest.approx(f[0], abs=1e-12 * s)
            assert g[4] == pytest.approx(f[4], abs=1e-12 * s)
            assert np.allclose(g[1:4], Q @ f[1:4], atol=1e-12 * s)


def test_sw_eps_smooths_but_keeps_consistency(ora):
    rng = np.random.default_rng(5)
    gamma, rho, vel, c, alpha = random_state(rng)
    fp, fm = ora.sw_split(gamma, rho, *vel, c, alpha, sw_eps=0.05)
    ref = exact_flux(gamma, rho, vel, c, alpha)
    assert np.allclose(fp + fm, ref, atol=1e-12 * np.abs(ref).max())
    fp0, _ = ora.sw_split(gamma, rho, *vel, c, alpha, sw_eps=0.0)
    assert not np.array_equal(fp, fp0)


def test_thermodynamics_and_sutherland(ora):
    from oracle.oracle import Oracle
    from paper_2209_15333_b200 import workloads as W
    case = W.smooth_periodic(8, 8, 8, Ma=0.8)
    o = Oracle(case)
    g, Ma = case.gamma, case.Ma
    rho, u, v, w, T = 1.3, 0.4, -0.2, 0.7, 1.7
    p = rho * T / (g * Ma * Ma)                                    # eq. 16-17
    E = p / (g - 1.0) + 0.5 * rho * (u * u + v * v + w * w)        # eq. 8 as corrected (R-1)
    q = o.prim_point([rho, rho * u, rho * v, rho * w, E])
    assert np.allclose(q, [rho, u, v, w, p, T, np.sqrt(T) / Ma], rtol=1e-14)
    # H = (E+p)/rho = V + c^2/(gamma-1) -- fixes the reading of eq. 8
    assert (E + p) / rho == pytest.approx(0.5 * (u * u + v * v + w * w) + q[6] ** 2 / (g - 1.0), rel=1e-14)
    # Sutherland (eq. 15): mu(1) = 1; mu(T) = T^1.5 (1+S)/(T+S)
    S = case.T_suth / case.T_ref
    assert o.mu(1.0) == pytest.approx(1.0, abs=1e-15)
    assert o.mu(2.5) == pytest.approx(2.5 ** 1.5 * (1 + S) / (2.5 + S), rel=1e-15)
