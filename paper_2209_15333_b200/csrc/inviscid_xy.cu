// Rows a2 + a4 + a5 for the x AND y sweeps in ONE marching kernel: primitives from U, Steger-Warming split of both
// directions (eq. 19-29), UD7 / WENO7 / WENO5 reconstruction (eq. 41) and the two
// conservative flux differences, written to dU once.
//
// Why fused: as separate launches the x sweep reads the state and writes dU (88 B/point) and the y sweep reads the
// state again and read-modify-writes dU (128 B/point).  Both work on x-y planes, so one kernel that owns a strip of an
// x-y plane can form both differences from ONE copy of the state in shared memory and write dU once: 48 B/point in
// (U and theta, plus a 25 % x halo that the neighbouring CTA's fetch leaves in the L2) and 40 B/point out.
//
// A CTA owns XC = 32 consecutive x columns of one z plane and walks along y through all ny + 8 padded rows in chunks
// of XR = 4 rows.  Every chunk:
//   TMA      the chunk's U box [5][4 rows][40 columns] (the 32 own columns + 4 halo columns on each side) and, for the
//            hybrid scheme, the theta box arrive in a ring of 3 stages that runs two chunks ahead (one mbarrier each);
//   phase A  one thread per staged point (160 = 4 x 40): u, v, w, c from the conserved variables, then the split fluxes
//            of the xi direction (all 160 points) and of the eta direction (the 128 own points) -> shared memory.
//            Every point is split once per direction and sweep; f+- never reach HBM (the paper materialises them, L549);
//   phase B  y walkers: one thread per (own column, component) keeps the two 7-point windows of the eta fluxes in
//            registers for the whole march as rings of 8 (the chunk loop is unrolled by two so that no value moves
//            between registers), pushes the chunk's 4 rows and completes the 4 points of the PREVIOUS chunk;
//            x walkers: one thread per (row, component, segment of 5 interfaces) slides its windows along the staged
//            row and leaves the 33 interface fluxes of the row in shared memory, where the y walkers of the next chunk
//            pick up h_{i+1/2} - h_{i-1/2} when they complete that row;
//   TMA      the finished 4 x 32 x 5 output tile leaves by one tensor store (the map covers the interior of dU only:
//            ragged tiles, the rows before the first interior point and ghosts are clipped by the hardware).
// Metric data (unit normal k and sigma of both directions, J) are read through the read-only path while the boxes are
// in flight: derived tables of metrics.cu on curvilinear grids (L2-resident planes on a z-extruded grid).
#include "ocfd_internal.cuh"
#include "schemes.cuh"
#include "tma.cuh"

#include <type_traits>

namespace {

constexpr int XC = 32;                  // own columns per CTA
constexpr int XH = OCFD_NG;             // x halo of the staged boxes
constexpr int XW = XC + 2 * XH;         // staged columns
constexpr int XR = 4;                   // rows per chunk
constexpr int XNST = 3;                 // input stages
constexpr int XPTS = XR * XW;           // staged points per chunk
constexpr int XNT = XPTS;               // threads: one per staged point
constexpr int XIN = XR * XC;            // own points per chunk
constexpr int XSL = 5, XNSEG = 7;       // x walkers: segments of 5 interfaces
constexpr int XNIF = XC + 1;            // interfaces per row
constexpr int XHP = XSL * XNSEG + 1;    // pitch of a row of interface fluxes
constexpr int XSTG = 6 * XPTS;          // doubles per input stage: U[5], theta
constexpr int XNW = XR * 5 * XNSEG;     // x walkers
#ifndef XMINB
#define XMINB 3
#endif
static_assert(XSL * XNSEG >= XNIF && XNW <= XNT && XC * 5 == XNT, "walker layout");
static_assert((XSTG * 8) % 128 == 0 && (5 * XPTS * 8) % 128 == 0 && (5 * XIN * 8) % 128 == 0, "TMA alignment");
constexpr size_t X_SMEM =
    sizeof(double) * (size_t)(XNST * XSTG + 2 * 5 * XIN + 10 * XIN + 10 * XPTS + 2 * 5 * XR * XHP) + 8 * XNST + XC * XR;

// KIND: grid kind, SCHEME: ocfd_scheme.  grid = (column tiles, nz).
template <int KIND, int SCHEME>
__global__ void __launch_bounds__(XNT, XMINB)
    k_inviscid_xy(const GridDesc g, const GasDesc gs, const __grid_constant__ CUtensorMap tm_U,
                  const __grid_constant__ CUtensorMap tm_th, const __grid_constant__ CUtensorMap tm_out) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *sIn = reinterpret_cast<double *>(smem_raw);   // [XNST][6][XR][XW]
    double *sO = sIn + XNST * XSTG;                       // [2][5][XR][XC] output tiles
    double *sF = sO + 2 * 5 * XIN;                        // [10][XR][XC]: eta split of the own points, f+ (0..4), f- (5..9)
    double *sFx = sF + 10 * XIN;                          // [10][XR][XW]: xi split of the staged points
    double *sHx = sFx + 10 * XPTS;                        // [2][5][XR][XHP]: xi interface fluxes of this / the previous chunk
    uint64_t *bars = reinterpret_cast<uint64_t *>(sHx + 2 * 5 * XR * XHP);
    unsigned char *sFl = reinterpret_cast<unsigned char *>(bars + XNST);   // [XC][XR] scheme flags of the y interfaces

    const int tid = threadIdx.x;
    const int a0 = blockIdx.x * XC, cross = blockIdx.y;
    const int kp = OCFD_NG + cross;
    const int nd = g.ny, ndp = nd + 2 * OCFD_NG;
    const int nch = (ndp + XR - 1) / XR;

    auto issue = [&](int c) {   // one thread: boxes of chunk c (padded rows XR*c ..) towards stage c % XNST
        const int s = c % XNST;
        double *dst = sIn + s * XSTG;
        tma::mbar_expect_tx(&bars[s], (SCHEME == OCFD_HYBRID ? 6 : 5) * XPTS * 8);
        tma::load4(dst, &tm_U, &bars[s], a0, XR * c, kp, 0);
        if (SCHEME == OCFD_HYBRID) tma::load4(dst + 5 * XPTS, &tm_th, &bars[s], a0, XR * c, kp, 0);
    };
    if (tid == 0) {
#pragma unroll
        for (int q = 0; q < XNST; ++q) tma::mbar_init(&bars[q], 1);
        tma::fence_barrier_init();
        issue(0);
        if (nch > 1) issue(1);
        if (nch > 2) issue(2);
    }

    // phase A role: staged point (row pr, column pc); own points are the columns XH .. XH + XC - 1
    const int pr = tid / XW, pc = tid % XW;
    const int ipA = a0 + pc;                      // padded x index of the staged point
    const bool inner = pc >= XH && pc < XH + XC;
    const int ia = pc - XH;
    // y walker role: own column wa, component wm
    const int wa = tid % XC, wm = tid / XC;
    const int ipW = min(OCFD_NG + a0 + wa, g.nxp - 1);
    // x walker role: segment xs of row xrow, component xm
    const int xs = tid % XNSEG, xrow = (tid / XNSEG) % XR, xm = tid / (XNSEG * XR);

    // register windows of the eta fluxes as rings of 8: padded row r lives in slot r % 8 (two chunks bring every slot
    // back to its place, so the chunk loop is unrolled by two)
    double Wp[8], Wm[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) Wp[e] = Wm[e] = 0.0;
    double hprev = 0.0;
    unsigned pprev = 0;     // packed flags of the previous chunk's y interfaces, 2 bits per row (hybrid)
    __syncthreads();        // barriers initialised before anyone polls them

    auto chunk = [&](const int c, auto ph) {
        constexpr int PH = decltype(ph)::value;
        const int s = c % XNST;
        const double *sU = sIn + s * XSTG;
        const int r0 = XR * c;                    // first padded row of the chunk
        const int rowA = r0 + pr;
        const bool validA = ipA < g.nxp && rowA < ndp;

        // metric data, fetched while the boxes are in flight: k, sigma of both directions at this thread's point ...
        double kx1 = 0.0, kx2 = 0.0, kx3 = 0.0, sgx = 1.0, ky1 = 0.0, ky2 = 0.0, ky3 = 0.0, sgy = 1.0, Jdead;
        if (validA) {
            met_ksJ<KIND, 0>(g, ipA, rowA, kp, kx1, kx2, kx3, sgx, Jdead);
            if (inner) met_ksJ<KIND, 1>(g, ipA, rowA, kp, ky1, ky2, ky3, sgy, Jdead);
        }
        // ... and J of the four points this walker completes in this chunk (padded rows r0-4 .. r0-1)
        double Jw[XR];
#pragma unroll
        for (int e = 0; e < XR; ++e) Jw[e] = jac_at<KIND>(g, ipW, max(r0 - OCFD_NG + e, 0), kp);
        tma::mbar_wait(&bars[s], (c / XNST) & 1);

        // ---- phase A: primitives and split fluxes of the chunk's points; flag of the y interface below each own point
        {
            double *dx = sFx + tid, *dy = sF + pr * XC + ia;
            if (validA) {
                double u, v, w, cc;
                const double rho = sU[tid];
                prim_from_cons(gs, rho, sU[XPTS + tid], sU[2 * XPTS + tid], sU[3 * XPTS + tid], sU[4 * XPTS + tid], u, v, w, cc);
                sw_split_store<KIND, 0>(gs, rho, u, v, w, cc, kx1, kx2, kx3, sgx, dx, XPTS);
                if (inner) sw_split_store<KIND, 1>(gs, rho, u, v, w, cc, ky1, ky2, ky3, sgy, dy, XIN);
            } else {
#pragma unroll
                for (int q = 0; q < 10; ++q) dx[q * XPTS] = 0.0;
                if (inner) {
#pragma unroll
                    for (int q = 0; q < 10; ++q) dy[q * XIN] = 0.0;
                }
            }
            if (SCHEME == OCFD_HYBRID && inner) {
                unsigned char f = 0;
                if (rowA >= OCFD_NG && rowA <= nd + OCFD_NG) {   // interfaces -1/2 .. nd-1/2 (eq. 42, R-12)
                    const double *thp = pr > 0 ? sU + 5 * XPTS + tid - XW
                                               : sIn + ((c + XNST - 1) % XNST) * XSTG + 5 * XPTS + (XR - 1) * XW + pc;
                    f = (unsigned char)iface_flag(gs, *thp, sU[5 * XPTS + tid]);
                }
                sFl[4 * ia + pr] = f;
            }
        }
        __syncthreads();
        // the stage of chunk c-1 is free now (phase A of this chunk read its last theta row)
        if (tid == 0 && c + 2 < nch && c > 0) issue(c + 2);

        // ---- phase B, y walkers: pushing row r completes interface (r-4)+1/2 and with it point r-4
#ifndef XY_NO_Y
        {
            double *so = sO + PH * 5 * XIN + wm * XIN + wa;
            const double *fpn = sF + wm * XIN + wa, *fmn = sF + (wm + 5) * XIN + wa;
            // xi interface fluxes of the rows being completed (left by the x walkers of the previous chunk)
            const double *hx = sHx + ((c + 1) & 1) * 5 * XR * XHP + wm * XR * XHP + wa;
            bool fast = SCHEME == OCFD_UD7;
            unsigned cur = 0;
            if (SCHEME == OCFD_HYBRID) {
                const unsigned w = reinterpret_cast<const unsigned *>(sFl)[wa];
                const unsigned pcur = (w & 3u) | ((w >> 6) & 0xcu) | ((w >> 12) & 0x30u) | ((w >> 18) & 0xc0u);
                // the interfaces completed in this chunk: pf(r0-3), pf(r0-2), pf(r0-1), pf(r0)
                cur = ((pprev >> 2) | (pcur << 6)) & 0xffu;
                pprev = pcur;
                fast = cur == 0;
            }
            // the paper's boundary scheme (ocfd_params.bc_closure): chunks whose interfaces s = r0-8 .. r0-5 come within
            // reach of a boundary (s <= 2 or s >= nd-4) test every interface
            const bool near_bnd = g.closure[1] && (r0 - 2 * OCFD_NG <= 2 || r0 + XR - 1 - 2 * OCFD_NG >= nd - 4);
            if (near_bnd) fast = false;
            double nP[XR], nM[XR], dxh[XR];
#pragma unroll
            for (int e = 0; e < XR; ++e) {
                nP[e] = fpn[e * XC];
                nM[e] = fmn[e * XC];
                dxh[e] = hx[e * XHP + 1] - hx[e * XHP];
            }
            if (fast) {
#pragma unroll
                for (int e = 0; e < XR; ++e) {
                    const int k = 4 * PH + e;
                    Wp[k & 7] = nP[e];
                    Wm[k & 7] = nM[e];
                    const double h = ud7(Wp[(k + 1) & 7], Wp[(k + 2) & 7], Wp[(k + 3) & 7], Wp[(k + 4) & 7], Wp[(k + 5) & 7],
                                         Wp[(k + 6) & 7], Wp[(k + 7) & 7]) +
                                     ud7(Wm[k & 7], Wm[(k + 7) & 7], Wm[(k + 6) & 7], Wm[(k + 5) & 7], Wm[(k + 4) & 7],
                                         Wm[(k + 3) & 7], Wm[(k + 2) & 7]);
                    so[e * XC] = -Jw[e] * ((h - hprev) + dxh[e]);
                    hprev = h;
                }
            } else if (near_bnd) {
#pragma unroll
                for (int e = 0; e < XR; ++e) {
                    const int k = 4 * PH + e;
                    Wp[k & 7] = nP[e];
                    Wm[k & 7] = nM[e];
                    const int flag = SCHEME == OCFD_HYBRID ? (int)((cur >> (2 * e)) & 3u) : 0;
                    const double h = recon_pair_closure<SCHEME>(
                        flag, r0 + e - 2 * OCFD_NG, nd, Wp[(k + 1) & 7], Wp[(k + 2) & 7], Wp[(k + 3) & 7], Wp[(k + 4) & 7],
                        Wp[(k + 5) & 7], Wp[(k + 6) & 7], Wp[(k + 7) & 7], Wm[k & 7], Wm[(k + 7) & 7], Wm[(k + 6) & 7],
                        Wm[(k + 5) & 7], Wm[(k + 4) & 7], Wm[(k + 3) & 7], Wm[(k + 2) & 7], gs.weno_eps);
                    so[e * XC] = -Jw[e] * ((h - hprev) + dxh[e]);
                    hprev = h;
                }
            } else {
#pragma unroll
                for (int e = 0; e < XR; ++e) {
                    const int k = 4 * PH + e;
                    Wp[k & 7] = nP[e];
                    Wm[k & 7] = nM[e];
                    const int flag = SCHEME == OCFD_HYBRID ? (int)((cur >> (2 * e)) & 3u) : 0;
                    const double h = recon_pair<SCHEME>(flag, Wp[(k + 1) & 7], Wp[(k + 2) & 7], Wp[(k + 3) & 7], Wp[(k + 4) & 7],
                                                        Wp[(k + 5) & 7], Wp[(k + 6) & 7], Wp[(k + 7) & 7], Wm[k & 7],
                                                        Wm[(k + 7) & 7], Wm[(k + 6) & 7], Wm[(k + 5) & 7], Wm[(k + 4) & 7],
                                                        Wm[(k + 3) & 7], Wm[(k + 2) & 7], gs.weno_eps);
                    so[e * XC] = -Jw[e] * ((h - hprev) + dxh[e]);
                    hprev = h;
                }
            }
        }

#endif
        // ---- phase B, x walkers: the 33 interface fluxes of every interior row of THIS chunk.  Interface q of a row
        // lies between the staged columns q+3 and q+4 (interior interface index a0 - 1 + q).
#ifndef XY_NO_X
        const int rowX = r0 + xrow;
        if (tid < XNW && rowX >= OCFD_NG && rowX < nd + OCFD_NG) {
            const int q0 = XSL * xs;
            const int nq = min(XSL, XNIF - q0);
            const double *fp = sFx + xm * XPTS + xrow * XW + q0;            // f+ columns q .. q+6
            const double *fm = sFx + (xm + 5) * XPTS + xrow * XW + q0 + 1;  // f- columns q+1 .. q+7
            double *hxo = sHx + (c & 1) * 5 * XR * XHP + (xm * XR + xrow) * XHP + q0;
            double wp[7], wm_[7];
#pragma unroll
            for (int e = 0; e < 6; ++e) {
                wp[e + 1] = fp[e];
                wm_[e + 1] = fm[e];
            }
            unsigned mask = 0u;
            if (SCHEME == OCFD_HYBRID) {
                const double *th = sU + 5 * XPTS + xrow * XW + q0 + 3;
                double ta = th[0];
#pragma unroll
                for (int i = 0; i < XSL; ++i) {
                    const double tb = th[i + 1];     // (the last segment reads two values past its row; they are not used)
                    if (i < nq) mask |= (unsigned)iface_flag(gs, ta, tb) << (2 * i);
                    ta = tb;
                }
            }
            const int s0 = a0 - 1 + q0;   // interior index of the segment's first interface
            const bool near_bnd = g.closure[0] && (s0 <= 2 || s0 + XSL - 1 >= g.nx - 4);
            const bool smooth = !near_bnd && (SCHEME == OCFD_UD7 || (SCHEME == OCFD_HYBRID && mask == 0u));
            if (smooth) {
                // every interface of the segment takes the linear scheme: fully unrolled, the windows slide by renaming
                // (the last segment's extra loads stay inside the shared-memory allocation, only the store is predicated)
#pragma unroll
                for (int i = 0; i < XSL; ++i) {
#pragma unroll
                    for (int e = 0; e < 6; ++e) {
                        wp[e] = wp[e + 1];
                        wm_[e] = wm_[e + 1];
                    }
                    wp[6] = fp[i + 6];
                    wm_[6] = fm[i + 6];
                    const double h = ud7(wp[0], wp[1], wp[2], wp[3], wp[4], wp[5], wp[6]) +
                                     ud7(wm_[6], wm_[5], wm_[4], wm_[3], wm_[2], wm_[1], wm_[0]);
                    if (i < nq) hxo[i] = h;
                }
            } else {
#pragma unroll 1
                for (int i = 0; i < nq; ++i) {
#pragma unroll
                    for (int e = 0; e < 6; ++e) {
                        wp[e] = wp[e + 1];
                        wm_[e] = wm_[e + 1];
                    }
                    wp[6] = fp[i + 6];
                    wm_[6] = fm[i + 6];
                    const int flag = SCHEME == OCFD_HYBRID ? (int)((mask >> (2 * i)) & 3u) : 0;
                    double h;
                    if (near_bnd)
                        h = recon_pair_closure<SCHEME>(flag, s0 + i, g.nx, wp[0], wp[1], wp[2], wp[3], wp[4], wp[5], wp[6],
                                                       wm_[6], wm_[5], wm_[4], wm_[3], wm_[2], wm_[1], wm_[0], gs.weno_eps);
                    else
                        h = recon_pair<SCHEME>(flag, wp[0], wp[1], wp[2], wp[3], wp[4], wp[5], wp[6], wm_[6], wm_[5], wm_[4],
                                               wm_[3], wm_[2], wm_[1], wm_[0], gs.weno_eps);
                    hxo[i] = h;
                }
            }
        }
#endif
        tma::fence_proxy_async();
        __syncthreads();
        if (tid == 0 && r0 + XR - 1 >= 2 * OCFD_NG) {
            const int o = r0 - 2 * OCFD_NG;   // interior row of the first completed point (negative rows are clipped)
            tma::store4(&tm_out, sO + PH * 5 * XIN, a0, o, cross, 0);
            tma::store_commit();
            tma::store_wait_read<1>();   // the other output tile is free for the next chunk
        }
    };
    for (int c = 0; c < nch; c += 2) {
        chunk(c, std::integral_constant<int, 0>());
        if (c + 1 < nch) chunk(c + 1, std::integral_constant<int, 1>());
    }
    if (tid == 0) tma::store_wait_all<0>();
}

template <int KIND, int SCHEME>
ocfd_status launch_xy(ocfd_ctx *c) {
    const GridDesc &g = c->g;
    if (!ocfd_smem_optin(c, (const void *)k_inviscid_xy<KIND, SCHEME>, X_SMEM)) return OCFD_ECUDA;
    dim3 grd((g.nx + XC - 1) / XC, g.nz, 1);
    OCFD_T0(c, K_INV_XY);
    const XYMaps &M = c->xy;
    k_inviscid_xy<KIND, SCHEME><<<grd, XNT, X_SMEM, c->stream>>>(g, c->gas, M.U, M.th, M.out);
    OCFD_CHECK_LAUNCH(c);
    return OCFD_OK;
}

template <int KIND>
ocfd_status launch_xy_kind(ocfd_ctx *c) {
    switch (c->p.scheme) {
        case OCFD_UD7: return launch_xy<KIND, OCFD_UD7>(c);
        case OCFD_WENO7: return launch_xy<KIND, OCFD_WENO7>(c);
        case OCFD_WENO5: return launch_xy<KIND, OCFD_WENO5>(c);
        default: return launch_xy<KIND, OCFD_HYBRID>(c);
    }
}

// input boxes over the whole padded arrays (x halo included), output boxes over the interior of dU
bool encode_xy_maps(ocfd_ctx *c, const double *U, double *dU) {
    const GridDesc &g = c->g;
    XYMaps &M = c->xy;
    const long long full1[4] = {g.nxp, g.nyp, g.nzp, 1}, full5[4] = {g.nxp, g.nyp, g.nzp, 5};
    const long long inner[4] = {g.nx, g.ny, g.nz, 5};
    const int b5[4] = {XW, XR, 1, 5}, b1[4] = {XW, XR, 1, 1}, bo[4] = {XC, XR, 1, 5};
    if (!M.ready && !ocfd_tma_encode(&M.th, c->theta, full1, g.sy, g.sz, g.np, b1)) return false;
    if (M.Up != U && !ocfd_tma_encode(&M.U, U, full5, g.sy, g.sz, g.np, b5)) return false;
    if (M.dUp != dU && !ocfd_tma_encode(&M.out, dU + (long long)OCFD_NG * (g.sz + g.sy + 1), inner, g.sy, g.sz, g.np, bo))
        return false;
    M.ready = true;
    M.Up = U;
    M.dUp = dU;
    return true;
}

}  // namespace

// dU <- -J [(h_{i+1/2} - h_{i-1/2})_xi + (h_{j+1/2} - h_{j-1/2})_eta]; the z sweep accumulates afterwards
ocfd_status launch_inviscid_xy(ocfd_ctx *c, const double *U, double *dU) {
    if (!encode_xy_maps(c, U, dU)) return OCFD_ECUDA;
    switch (c->g.kind) {
        case OCFD_GRID_UNIFORM: return launch_xy_kind<OCFD_GRID_UNIFORM>(c);
        case OCFD_GRID_STRETCHED: return launch_xy_kind<OCFD_GRID_STRETCHED>(c);
        default: return launch_xy_kind<OCFD_GRID_CURVILINEAR>(c);
    }
}
