"""CPU checks of the helpers the GPU parity tests rely on (tests/parity_utils.py): the stage-by-stage stepping of the
oracle is ora_rk3_step bit for bit, and the near-threshold bookkeeping finds, dilates and counts what it should."""
import numpy as np

from oracle.oracle import Oracle
from paper_2209_15333_b200 import workloads as W
from tests.parity_utils import NG, compare_flags, dilate, iface_theta, near_threshold


def test_stagewise_stepping_is_the_oracles_own_step():
    case = W.ramp(nx=16, ny=12, nz=8, nmodes=4, theta2=0.1)
    o = Oracle(case)
    U = o.fill_ghosts(case.U0.copy())
    dt = 0.4 * case.cfl / o.max_wavespeed(U)
    ref = o.rk3_step(U.copy(), dt)
    Un = U.copy()
    for st in range(3):
        if st > 0:
            o.fill_ghosts(U)
        o.rk3_update(Un, U, o.rhs(U), dt, st)
    o.fill_ghosts(U)
    assert np.array_equal(U, ref)


def test_interface_theta_and_flag_comparison_follow_the_definition():
    case = W.shocked_periodic(12, theta1=0.02, theta2=0.1)
    o = Oracle(case)
    U = o.fill_ghosts(case.U0.copy())
    th = o.sensor(U)
    fl = [o.flags(th, d) for d in range(3)]
    for d in range(3):
        Th, sl = iface_theta(th, d)
        want = np.where(Th <= case.theta1, 0, np.where(Th <= case.theta2, 1, 2))
        assert np.array_equal(fl[d][sl], want)              # eq. 42 thresholds, R-11 / R-12
    bad, near, total, hist = compare_flags(th, fl, fl, case.theta1, case.theta2)
    assert (bad, near) == (0, 0) and total == 3 * 13 * 12 * 12 and hist.sum() == total
    wrong = [f.copy() for f in fl]
    wrong[1][NG + 3, NG + 2, NG + 5] ^= 1                   # one flipped decision is one mismatch
    assert compare_flags(th, fl, wrong, case.theta1, case.theta2)[0] == 1
    # ... unless its Theta sits inside the band
    Th, sl = iface_theta(th, 1)
    t1 = float(Th[3, 3, 5])                                 # interface (k=3, s=2 -> row index 3, i=5) along y
    assert compare_flags(th, fl, wrong, t1, np.inf)[0] <= 1


def test_near_threshold_marks_both_points_of_the_interface_and_dilation_respects_walls():
    th = np.zeros((8 + 2 * NG,) * 3)
    th[NG + 2, NG + 3, NG + 4] = 0.5                        # point (i=4, j=3, k=2)
    m = near_threshold(th, 0.5, np.inf, 1e-12)
    pts = set(zip(*np.nonzero(m)))
    # the six interfaces around the point carry Theta = 0.5: the point and its six neighbours
    assert pts == {(2, 3, 4), (1, 3, 4), (3, 3, 4), (2, 2, 4), (2, 4, 4), (2, 3, 3), (2, 3, 5)}
    assert not near_threshold(th, 0.4, np.inf, 1e-3).any()
    one = np.zeros((8, 8, 8), dtype=bool)
    one[0, 4, 7] = True                                     # k=0, j=4, i=7
    d = dilate(one, 2, periodic=[False, True, True])        # x aperiodic, y and z periodic
    assert d[0, 4, 5] and not d[0, 4, 0]                    # no wrap in x
    assert d[6, 4, 7] and d[0, 2, 7] and d[0, 6, 7]         # wraps in z, spreads in y
    assert d.sum() == 3 * 5 * 5
