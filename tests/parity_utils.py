"""Helpers shared by the GPU parity tests: the error metric of SURVEY 8(c) / DESIGN R-23, the comparison of the
hybrid scheme's sensor decisions, and RK3 stepping of both sides with a record of every interface whose sensor value
comes close to a threshold (so that a flipped decision is found, counted and its domain of influence excluded, instead
of being hidden behind a loosened tolerance).

Test infrastructure only; the oracle side of every comparison is computed by oracle/ from inputs the oracle itself
prepared (ghost fill included), never from the CUDA path.
"""
import numpy as np

NG = 4
INT = (slice(None), slice(NG, -NG), slice(NG, -NG), slice(NG, -NG))
I3 = (slice(NG, -NG),) * 3


def rel_linf(gpu, ora, U, floor=0.0):
    """max|gpu-ora| / max(max|ora|, floor) per component; max|U| if that is below 1e-300 (DESIGN R-23)."""
    errs = []
    for m in range(5):
        den = max(np.abs(ora[m]).max(), floor)
        if den < 1e-300:
            den = np.abs(U[m]).max()
        errs.append(np.abs(gpu[m] - ora[m]).max() / den)
    return np.array(errs)


def iface_theta(th, d):
    """Theta of the interfaces s = -1 .. n-1 along direction d (0 x, 1 y, 2 z) of the interior lines: max of the two
    points that share the interface (DESIGN R-12).  Views of `th`, no copies until the maximum."""
    ax = 2 - d
    lo = [slice(NG, -NG)] * 3
    hi = [slice(NG, -NG)] * 3
    lo[ax] = slice(NG - 1, -NG)
    hi[ax] = slice(NG, -NG + 1)
    return np.maximum(th[tuple(lo)], th[tuple(hi)]), tuple(lo)


def compare_flags(th_ref, fl_ref, fl_gpu, theta1, theta2, band=1e-12):
    """Sensor decisions of the two sides on every interface.  fl_ref[d], fl_gpu[d]: padded byte fields, entry of point s
    = scheme of interface s+1/2 along d.  Returns (mismatches outside the band, interfaces inside the band, interfaces,
    histogram of the oracle's decisions)."""
    bad = near = total = 0
    hist = np.zeros(3, dtype=np.int64)
    for d in range(3):
        Th, sl = iface_theta(th_ref, d)
        inband = np.abs(Th - theta1) <= band
        if np.isfinite(theta2):
            inband |= np.abs(Th - theta2) <= band
        diff = fl_gpu[d][sl] != fl_ref[d][sl]
        bad += int((diff & ~inband).sum())
        near += int(inband.sum())
        total += diff.size
        hist += np.bincount(fl_ref[d][sl].ravel(), minlength=3)[:3]
    return bad, near, total, hist


def near_threshold(th, theta1, theta2, band):
    """Interior points that touch an interface whose Theta lies within `band` of a threshold: boolean interior mask."""
    n = tuple(s - 2 * NG for s in th.shape)
    mask = np.zeros(n, dtype=bool)
    for d in range(3):
        Th, _ = iface_theta(th, d)
        close = np.abs(Th - theta1) <= band
        if np.isfinite(theta2):
            close |= np.abs(Th - theta2) <= band
        if not close.any():
            continue
        ax = 2 - d
        # interface s (s = -1 .. n-1) touches points s and s+1
        a = [slice(None)] * 3
        b = [slice(None)] * 3
        a[ax] = slice(1, None)      # interfaces 0 .. n-1   -> points 0 .. n-1 (left point)
        b[ax] = slice(0, -1)        # interfaces -1 .. n-2  -> points 0 .. n-1 (right point)
        mask |= close[tuple(a)] | close[tuple(b)]
    return mask


def dilate(mask, r, periodic):
    """Box dilation of a boolean interior mask by r points along every axis (wrapping on periodic axes)."""
    if not mask.any() or r <= 0:
        return mask
    out = mask
    for ax in range(3):
        n = out.shape[ax]
        rr = min(r, n)
        acc = out.copy()
        for sft in range(1, rr + 1):
            for sg in (1, -1):
                rolled = np.roll(out, sg * sft, axis=ax)
                if not periodic[2 - ax]:
                    idx = [slice(None)] * 3
                    idx[ax] = slice(0, sft) if sg == 1 else slice(n - sft, n)
                    rolled[tuple(idx)] = False
                acc |= rolled
        out = acc
    return out


def step_both_hybrid(B, Oracle, case, nsteps, band=1e-9, check_flags_every=1, log=print):
    """Advance both sides `nsteps` RK3 steps.  The oracle is stepped stage by stage (fill, RHS, update: the same calls
    ora_rk3_step makes) so that its sensor field is seen at EVERY stage: interfaces whose Theta comes within `band` of a
    threshold are the only places where the two sides may legitimately decide differently (their states differ by
    round-off); they are counted, and the points inside their domain of influence (18 points per remaining step: three
    stages of reach 6) are excluded from the comparison.  At the start of every `check_flags_every`-th step the GPU's
    own decisions (ocfd_debug_sensor) are compared with the oracle's, outside the 1e-12 band of north_star.

    Returns dict(err_all, err_outside, err_padded_outside (the same bar over the whole padded array: face ghosts
    included), excluded_fraction, near, flag_mismatches, flag_inband, hist0, hist_end)."""
    o = Oracle(case)
    U = o.fill_ghosts(case.U0.copy())
    dt = case.cfl / o.max_wavespeed(U)
    s = B.Solver(case)
    Ud = s.to_device(U)
    per = [case.bc[2 * d] == "periodic" for d in range(3)]
    excl = np.zeros((case.nz, case.ny, case.nx), dtype=bool)
    near_total = bad_total = inband_total = 0
    hist0 = hist_end = None
    hybrid = case.scheme == "hybrid"
    for n in range(nsteps):
        if hybrid and (n % check_flags_every == 0 or n == nsteps - 1):
            th_ref = o.sensor(U)
            fl_ref = [o.flags(th_ref, d) for d in range(3)]
            th_gpu, fl_gpu = s.debug_sensor(Ud)
            fl_gpu = fl_gpu.cpu().numpy()
            bad, inband, total, hist = compare_flags(th_ref, fl_ref, fl_gpu, case.theta1, case.theta2)
            bad_total += bad
            inband_total += inband
            if hist0 is None:
                hist0 = hist
            del th_gpu, fl_gpu
        Un = U.copy()
        for st in range(3):
            if st > 0:
                o.fill_ghosts(U)
            if hybrid:
                m = near_threshold(o.sensor(U), case.theta1, case.theta2, band)
                if m.any():
                    near_total += int(m.sum())
                    excl |= dilate(m, 18 * (nsteps - n), per)
            dU = o.rhs(U)
            o.rk3_update(Un, U, dU, dt, st)
        o.fill_ghosts(U)
        s.rk3_step(Ud, dt)
    if hybrid:
        th_ref = o.sensor(U)
        hist_end = compare_flags(th_ref, [o.flags(th_ref, d) for d in range(3)],
                                 s.debug_sensor(Ud)[1].cpu().numpy(), case.theta1, case.theta2)[3]
    got = Ud.cpu().numpy()
    s.close()
    gi, ui = got[INT], U[INT]
    umax = np.abs(ui).max()
    floor = 1e-3 * umax
    err_all = rel_linf(gi, ui, ui, floor).max()
    keep = ~excl
    if keep.any():
        den = [max(np.abs(ui[m]).max(), floor) for m in range(5)]
        err_out = max(np.abs(gi[m] - ui[m])[keep].max() / den[m] for m in range(5))
    else:
        err_out = float("nan")
    # the whole padded array as well: both sides leave the face ghosts filled by the last ghost fill of the step (from
    # two different buffers on the GPU side, ocfd_rk3_step rotates them); edges and corners are written by neither and
    # still hold the initial values.  A ghost point counts as excluded if the interior point nearest to it is.
    keep_p = np.pad(keep, NG, mode="edge")
    if keep_p.any():
        err_pad = max(np.abs(got[m] - U[m])[keep_p].max() / max(np.abs(U[m]).max(), floor) for m in range(5))
    else:
        err_pad = float("nan")
    res = dict(err_all=float(err_all), err_outside=float(err_out), err_padded_outside=float(err_pad),
               excluded_fraction=float(excl.mean()),
               near=near_total, flag_mismatches=bad_total, flag_inband=inband_total,
               hist0=None if hist0 is None else hist0.tolist(), hist_end=None if hist_end is None else hist_end.tolist(),
               finite=bool(np.isfinite(got).all()))
    log(f"{case.name}: {nsteps} RK3 steps, rel Linf of U: {err_all:.3e} everywhere, {err_out:.3e} outside the domain of "
        f"influence of {near_total} points next to interfaces within {band:g} of a threshold (excluded fraction "
        f"{excl.mean():.4f}); flag mismatches outside the 1e-12 band {bad_total} (inside it {inband_total}); "
        f"flag histogram UD7/WENO7/WENO5 first {res['hist0']} last {res['hist_end']}")
    return res
