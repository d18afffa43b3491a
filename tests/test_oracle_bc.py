"""Pins of the oracle's ghost / boundary fill (DESIGN R-16) and max wavespeed (R-17).  CPU only."""
import numpy as np
import pytest

from oracle.oracle import Oracle
from paper_2209_15333_b200 import workloads as W

NG = 4


def prims(case, U):
    g = case.gamma
    rho = U[0]
    u, v, w = U[1] / rho, U[2] / rho, U[3] / rho
    p = (g - 1.0) * (U[4] - 0.5 * rho * (u * u + v * v + w * w))
    T = g * case.Ma ** 2 * p / rho
    return rho, u, v, w, p, T


def test_periodic_ghosts_wrap_exactly():
    case = W.smooth_periodic(9, 7, 6)
    U = case.U0.copy()
    rng = np.random.default_rng(0)
    ghost = np.ones(U.shape, dtype=bool)
    ghost[:, NG:-NG, NG:-NG, NG:-NG] = False
    U[ghost] = rng.uniform(1, 2, ghost.sum())             # scramble every ghost
    before = U.copy()
    Oracle(case).fill_ghosts(U)
    I = slice(NG, -NG)
    assert np.array_equal(U[:, I, I, I], before[:, I, I, I])                      # interior untouched
    assert np.array_equal(U[:, I, I, :NG], U[:, I, I, -2 * NG:-NG])
    assert np.array_equal(U[:, I, I, -NG:], U[:, I, I, NG:2 * NG])
    assert np.array_equal(U[:, I, :NG, I], U[:, I, -2 * NG:-NG, I])
    assert np.array_equal(U[:, :NG, I, I], U[:, -2 * NG:-NG, I, I])
    # edges and corners are never written
    assert np.array_equal(U[:, :NG, :NG, :], before[:, :NG, :NG, :])
    assert np.array_equal(U[:, :, :NG, :NG], before[:, :, :NG, :NG])


def test_plate_boundaries_satisfy_their_invariants():
    case = W.flat_plate(nx=14, ny=12, nz=6)
    # perturb the interior so that nothing is trivially satisfied
    rng = np.random.default_rng(1)
    U = case.U0 * (1.0 + 0.05 * rng.uniform(-1, 1, case.U0.shape))
    U = np.ascontiguousarray(U)
    Oracle(case).fill_ghosts(U)
    rho, u, v, w, p, T = prims(case, U)
    I = slice(NG, -NG)
    Tw = case.T_wall[2]
    # wall node (j = 0): no slip except the prescribed blowing, T = T_w, p from the one-sided formula
    vn = case.wall_vn[2][I, I]
    assert np.allclose(u[I, NG, I], 0.0, atol=1e-14) and np.allclose(w[I, NG, I], 0.0, atol=1e-14)
    assert np.allclose(v[I, NG, I], vn, atol=1e-14)
    assert np.allclose(T[I, NG, I], Tw, rtol=1e-13)
    assert np.allclose(p[I, NG, I], (4 * p[I, NG + 1, I] - p[I, NG + 2, I]) / 3.0, rtol=1e-12)
    for m in range(1, NG + 1):
        for q in (u, v, w):
            assert np.allclose(q[I, NG - m, I] + q[I, NG + m, I], 2 * q[I, NG, I], atol=1e-12)
        assert np.allclose(T[I, NG - m, I] + T[I, NG + m, I], 2 * Tw, rtol=1e-12)
        assert np.allclose(p[I, NG - m, I], p[I, NG + m, I], rtol=1e-12)
    # inflow face: node and ghosts carry the profile (the wall, processed later, owns the shared edge)
    for m in range(0, NG + 1):
        assert np.array_equal(U[:, I, NG + 1:-NG, NG - m], case.inflow[0][:, I, NG + 1:-NG])
    # outflow faces: ghosts copy the last interior node
    for m in range(1, NG + 1):
        assert np.array_equal(U[:, I, I, -NG - 1 + m], U[:, I, I, -NG - 1])
        assert np.array_equal(U[:, I, -NG - 1 + m, I], U[:, I, -NG - 1, I])
    # z periodic
    assert np.array_equal(U[:, :NG, I, I], U[:, -2 * NG:-NG, I, I])


def test_wall_on_a_plus_face_and_tilted_normal():
    """Wall on the y+ face of a sheared grid: blowing velocity follows the unit normal into the fluid."""
    case = W.smooth_periodic(8, 8, 6, grid="uniform")
    h = case.dx
    case.metrics = W.affine_metrics(8, 8, 6, h * np.array([[1.0, 0.4, 0.0], [0.0, 1.0, 0.0], [0.0, 0.2, 1.0]]))
    case.bc = ["periodic", "periodic", "outflow", "wall", "periodic", "periodic"]
    case.T_wall[3] = 1.2
    vn = np.full((6 + 2 * NG, 8 + 2 * NG), 0.03)
    case.wall_vn[3] = vn
    U = case.U0.copy()
    Oracle(case).fill_ghosts(U)
    rho, u, v, w, p, T = prims(case, U)
    I = slice(NG, -NG)
    n = -np.array([case.metrics[3].ravel()[0], case.metrics[4].ravel()[0], case.metrics[5].ravel()[0]])
    n /= np.linalg.norm(n)
    jw = NG + case.ny - 1
    assert np.allclose(u[I, jw, I], 0.03 * n[0], atol=1e-14)
    assert np.allclose(v[I, jw, I], 0.03 * n[1], atol=1e-14)
    assert np.allclose(w[I, jw, I], 0.03 * n[2], atol=1e-14)
    assert np.allclose(T[I, jw, I], 1.2, rtol=1e-13)
    assert np.allclose(T[I, jw + 2, I] + T[I, jw - 2, I], 2.4, rtol=1e-12)


def test_max_wavespeed_closed_form_and_brute_force():
    case = W.smooth_periodic(8, 7, 6, grid="uniform")
    o = Oracle(case)
    shp = case.padded_shape
    one = np.ones(shp)
    rho, T, vel = 1.2, 0.8, (0.7, -0.4, 0.2)
    p = rho * T / (case.gamma * case.Ma ** 2)
    U = np.ascontiguousarray(W.cons_from_prim(rho * one, vel[0] * one, vel[1] * one, vel[2] * one, p * one, case.gamma))
    c = np.sqrt(T) / case.Ma
    ref = (abs(vel[0]) + c) / case.dx + (abs(vel[1]) + c) / case.dy + (abs(vel[2]) + c) / case.dz
    assert o.max_wavespeed(U) == pytest.approx(ref, rel=1e-13)
    # brute force on a curvilinear case
    case = W.smooth_periodic(7, 6, 5, grid="wavy")
    o = Oracle(case)
    U = case.U0
    rho, u, v, w, p, T = prims(case, U)
    cs = np.sqrt(T) / case.Ma
    m = [np.broadcast_to(a, case.padded_shape) for a in case.metrics]
    lam = sum(np.abs(m[3 * d] * u + m[3 * d + 1] * v + m[3 * d + 2] * w)
              + cs * np.sqrt(m[3 * d] ** 2 + m[3 * d + 1] ** 2 + m[3 * d + 2] ** 2) for d in range(3))
    I = slice(NG, -NG)
    assert o.max_wavespeed(U) == pytest.approx(lam[I, I, I].max(), rel=1e-13)
    # ghosts do not take part
    U2 = U.copy()
    U2[:, :NG] *= 3.0
    assert o.max_wavespeed(np.ascontiguousarray(U2)) == o.max_wavespeed(U)


def test_check_state_counts_hand_made_bad_points():
    """ora_check_state (the paper's only statement on divergence is PAPER.md:L305): known numbers of
    points of each kind planted by hand in a clean field; ghosts, edges and corners do not take part."""
    case = W.smooth_periodic(9, 8, 7, grid="wavy")
    o = Oracle(case)
    assert o.check_state(case.U0) == (0, 0, 0)
    U = case.U0.copy()
    g = case.gamma
    pts = lambda *ijk: tuple(NG + q for q in reversed(ijk))          # (i, j, k) -> padded [k][j][i]
    U[(4,) + pts(0, 0, 0)] = np.nan                                    # E NaN: non-finite only
    U[(1,) + pts(8, 7, 6)] = np.inf                                    # rho u inf: non-finite only (last interior point)
    U[(0,) + pts(3, 2, 1)] = np.nan                                    # rho NaN: non-finite, NOT rho <= 0 (NaN compares false)
    U[(0,) + pts(4, 4, 4)] = -0.5                                      # rho < 0: counted once, p not looked at
    U[(0,) + pts(5, 4, 4)] = 0.0                                       # rho == 0 counts as bad
    U[(0,) + pts(6, 1, 2)] = -np.inf                                   # -inf rho: non-finite AND rho <= 0
    for (i, j, k), frac in (((1, 1, 1), 0.5), ((2, 6, 3), 1.0), ((7, 0, 5), 0.999999)):
        idx = pts(i, j, k)                                             # E below / at / just under the kinetic energy
        ke = 0.5 * (U[(1,) + idx] ** 2 + U[(2,) + idx] ** 2 + U[(3,) + idx] ** 2) / U[(0,) + idx]
        U[(4,) + idx] = frac * ke
    # p = (g-1)(E - ke): 0.5 ke and 0.999999 ke give p < 0; E = ke gives p == 0 up to the rounding of ke, planted as exactly
    # zero velocity instead so that p == 0 is exact
    idx = pts(2, 6, 3)
    U[(1,) + idx] = U[(2,) + idx] = U[(3,) + idx] = 0.0
    U[(4,) + idx] = 0.0
    # bad values in ghosts must not count
    U[0, 0, :, :] = -1.0
    U[4, :, :, -1] = np.nan
    assert o.check_state(np.ascontiguousarray(U)) == (4, 3, 3)
    # a healthy pressure just above zero is not counted
    V = case.U0.copy()
    idx = pts(3, 3, 3)
    ke = 0.5 * (V[(1,) + idx] ** 2 + V[(2,) + idx] ** 2 + V[(3,) + idx] ** 2) / V[(0,) + idx]
    V[(4,) + idx] = ke + 1e-9 / (g - 1.0)
    assert o.check_state(V) == (0, 0, 0)
