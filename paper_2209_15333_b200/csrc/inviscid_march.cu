// Rows a2 + a4 + a5 of ONE sweep direction: primitives from U, Steger-Warming split (eq. 19-29),
// UD7 / WENO7 / WENO5 reconstruction (eq. 41) and the conservative flux difference, as a MARCHING
// kernel.  It runs the x, y and z sweeps of every run in component-wise variables.
//
// A CTA owns MAC = 32 pencils (32 consecutive x; for the x sweep 32 consecutive y lines) of one cross index and walks
// along the sweep direction through the padded rows of its segment in chunks of MR = 4 rows.  Per chunk c:
//   TMA      the state of the chunk (the five conserved fields as ONE box; theta if hybrid; on curvilinear grids the
//            metric tables k, sigma and J as one more box) arrives in a ring of 4 (curvilinear) or 6 stages, requested
//            as many chunks ahead as the ring allows by one thread of the warp that has no phase-A work (one mbarrier
//            per stage);
//   phase A  one thread per point of the chunk: u, v, w, c from the conserved variables, then the split fluxes
//            f+-[5] -> shared memory (double-buffered).  Each point is split exactly once per sweep (no halo
//            recomputation) and neither the primitives nor f+- ever reach HBM (the paper materialises f+-, L549);
//   phase B  one thread per (pencil, component): the 7-point windows of f+ and f- live in registers for the whole
//            march, each new row costs two shared-memory loads; h_{i+1/2} is formed as soon as row i+4 has been
//            pushed and -J (h_{i+1/2} - h_{i-1/2}) goes to an output tile in shared memory;
//   TMA      the output tile leaves by one tensor store (x sweep: it writes dU) or one reduce-add (y, z: dU += at the L2).
// Between two CTA barriers the CTA runs phase A of chunk c+1 and phase B of chunk c: ONE barrier per chunk.
// The output tensor map covers the interior of dU only, so the rows before the first interior point, ragged tiles and
// ghosts are clipped by the hardware.
#include "ocfd_internal.cuh"
#include "schemes.cuh"
#include "tma.cuh"

#include <type_traits>

namespace {

constexpr int MAC = 32;             // pencils per CTA (consecutive x)
constexpr int MR = 4;               // rows per chunk
constexpr int MPTS = MAC * MR;      // points per chunk
constexpr int MNT = 5 * MAC;        // threads: one walker per (pencil, component)
// Input ring of one grid kind: a stage holds U[5], theta and, on curvilinear grids, the metric box k1, k2, k3, sigma, J
// of one chunk; as many stages as three CTAs per SM leave room for (the sweeps wait on HBM latency: with 3 stages the
// y / z sweeps of a 256^3 box ran at 0.83 of the HBM peak, with 4 at 0.92).
// MFULL = 0: the z sweep over a z-extruded curvilinear map, whose metric box is one row for the whole chunk.
template <int KIND, int DIR, bool MFULL>
struct MRing {
    static constexpr int MBOX = KIND != OCFD_GRID_CURVILINEAR ? 0 : 5 * (MFULL ? MPTS : MAC);   // doubles of the metric box
    static constexpr int STG = 6 * MPTS + MBOX;                          // doubles per stage
    static constexpr int NST = KIND != OCFD_GRID_CURVILINEAR ? 6 : MFULL ? 4 : 6;   // stages
    // chunks requested ahead.  Curvilinear x sweep: one less than the stages, so that the stage of chunk c-1 still holds
    // its J when phase B of chunk c needs it (the y and z sweeps carry that J in registers instead and use every stage;
    // the x sweep, which keeps its four outputs of a chunk in registers as well, measured slower that way)
    static constexpr int PF = KIND == OCFD_GRID_CURVILINEAR && DIR == 0 ? NST - 1 : NST;
    static constexpr size_t SMEM =
        sizeof(double) * (size_t)(NST * STG + 2 * 10 * MPTS + 2 * 5 * MPTS) + 8 * NST + 2 * 4 * MAC;
    static_assert(3 * (SMEM + 1024) <= 233472, "three CTAs per SM");
};
constexpr int MTMA = MPTS;          // the thread that issues every TMA operation: lane 0 of the warp without phase-A work
static_assert(MPTS <= MNT && (MPTS * 8) % 128 == 0, "chunk shape");

// J along one pencil of the sweep: at(g, i0, e) = J at padded row i0 + e
template <int KIND, int DIR>
struct JRow {
    const double *p;   // curvilinear: J of row 0 of the pencil; stretched: the 1-D metric of the sweep axis
    long long st;      // curvilinear: row stride
    double f0, f1;     // stretched: the two fixed 1-D metrics
    // ap = padded across index (y for the x sweep, else x), crossp = padded cross index (z, z, y for DIR 0, 1, 2)
    __device__ __forceinline__ JRow(const GridDesc &g, int ap, int crossp) : p(nullptr), st(0), f0(0.0), f1(0.0) {
        if (KIND == OCFD_GRID_STRETCHED) {
            f0 = __ldg(g.met[DIR == 0 ? 4 : 0] + ap);
            f1 = __ldg(g.met[DIR == 2 ? 4 : 8] + crossp);
            p = g.met[4 * DIR];
        } else if (KIND == OCFD_GRID_CURVILINEAR) {
            st = DIR == 0 ? 1 : DIR == 1 ? g.sy : g.msk;
            p = g.atab[0] + 4 * g.atab_fs +
                (DIR == 0 ? (long long)crossp * g.msk + (long long)ap * g.sy
                          : (DIR == 1 ? (long long)crossp * g.msk : (long long)crossp * g.sy) + ap);
        }
    }
    __device__ __forceinline__ double at(const GridDesc &g, int i0, int e) const {
        if (KIND == OCFD_GRID_UNIFORM) return g.uJ;
        if (KIND == OCFD_GRID_STRETCHED) {
            const double m = __ldg(p + i0 + e);
            return DIR == 0 ? (m * f0) * f1 : DIR == 1 ? (f0 * m) * f1 : (f0 * f1) * m;   // (xi_x eta_y) zeta_z
        }
        return __ldg(p + (long long)(i0 + e) * st);
    }
};

// KIND: grid kind, SCHEME: ocfd_scheme, DIR: 0 x, 1 y, 2 z.  grid = (tiles across, cross extent).
// DIR 0: the 32 pencils are 32 consecutive y lines and a chunk is 4 x-points of each (boxes of 32-byte rows; the tensor
// maps of the x sweep ask the L2 for 256-byte fills, so that the 8 chunks that share them find them there).  The
// shared arrays keep the box order (x fastest), the split fluxes are stored with an XOR swizzle of the pencil index so
// that both the point-wise phase and the walkers are free of bank conflicts, and the output tile is written as two
// 16-byte stores per walker and leaves by a TMA store (the x sweep writes dU, y and z accumulate).
// Occupancy: 3 CTAs per SM (128 registers, 74 KB of shared memory each): the hybrid scheme's three code paths need the
// 128 registers to keep the unrolled linear path free of spills (measured: 3.8 ms against 4.5 ms per sweep on config 5).
template <int KIND, int SCHEME, int DIR, bool MFULL>
__global__ void __launch_bounds__(MNT, 3)
    k_inviscid_march(const GridDesc g, const GasDesc gs, const __grid_constant__ CUtensorMap tm_U,
                     const __grid_constant__ CUtensorMap tm_th,
                     const __grid_constant__ CUtensorMap tm_out, const __grid_constant__ CUtensorMap tm_met,
                     const int seglen) {
    constexpr bool mfull = MFULL;
    constexpr int MNST = MRing<KIND, DIR, MFULL>::NST, MSTG = MRing<KIND, DIR, MFULL>::STG, MPF = MRing<KIND, DIR, MFULL>::PF;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *sIn = reinterpret_cast<double *>(smem_raw);   // [MNST][NF][MR][MAC]
    double *sF = sIn + MNST * MSTG;                       // [2][10][MR][MAC]: f+ (0..4), f- (5..9) of chunk c in buffer c % 2
    double *sO = sF + 2 * 10 * MPTS;                      // [2][5][MR][MAC] output tiles
    uint64_t *bars = reinterpret_cast<uint64_t *>(sO + 2 * 5 * MPTS);
    unsigned char *sFl = reinterpret_cast<unsigned char *>(bars + MNST);   // [2][MAC][MR] scheme flags pf of chunk c % 2

    const int tid = threadIdx.x;
    const int a0 = blockIdx.x * MAC, cross = blockIdx.y;
    const int nd = DIR == 0 ? g.nx : DIR == 1 ? g.ny : g.nz;
    const int nap = DIR == 0 ? g.nyp : g.nxp;   // padded extent across
    const int ndp = nd + 2 * OCFD_NG;
    // blockIdx.z = segment of the march: interior rows [o0, o1) (seglen is a multiple of MR; short segments keep the
    // CTAs short, which evens out the end of the launch when the cross-section gives few CTAs).  A segment stages the
    // padded rows o0 .. o1 + 7, i.e. the chunks [cbeg, cend); every per-chunk slot below is indexed by lc = c - cbeg.
    const int o0 = blockIdx.z * seglen, o1 = min(o0 + seglen, nd);
    const int cbeg = o0 / MR, cend = (o1 + 2 * OCFD_NG + MR - 1) / MR, nch = cend - cbeg;

    auto issue = [&](int lc) {   // one thread: boxes of chunk c (padded rows MR*c ..) towards stage lc % MNST
        const int c = cbeg + lc, s = lc % MNST;
        double *dst = sIn + s * MSTG;
        const int c0 = DIR == 0 ? MR * c : OCFD_NG + a0;
        const int c1 = DIR == 0 ? OCFD_NG + a0 : DIR == 1 ? MR * c : OCFD_NG + cross;
        const int c2 = DIR == 2 ? MR * c : OCFD_NG + cross;
        // curvilinear grids: the metric tables k1, k2, k3, sigma and J of the chunk come the same way (mfull = 0: a
        // z-extruded map swept along z, one row serves the whole chunk)
        const uint32_t mbytes = KIND == OCFD_GRID_CURVILINEAR ? 5u * (mfull ? MPTS : MAC) * 8u : 0u;
        tma::mbar_expect_tx(&bars[s], (SCHEME == OCFD_HYBRID ? 6 : 5) * MPTS * 8 + mbytes);
        if (KIND == OCFD_GRID_CURVILINEAR) {
            const int m2 = DIR == 2 ? (mfull ? MR * c : 0) : (g.msk ? OCFD_NG + cross : 0);
            // (x sweep: the copy of the table with y contiguous, so the box is [4 x][32 lines])
            // z-extruded tables are a few planes that every cross index reads again: ask the L2 to keep them
            const uint64_t keep = tma::policy_evict_last();
            tma::load4_hint(dst + 6 * MPTS, &tm_met, &bars[s], DIR == 0 ? c1 : c0, DIR == 0 ? c0 : c1, m2, 0, keep);
        }
        tma::load4(dst, &tm_U, &bars[s], c0, c1, c2, 0);
        if (SCHEME == OCFD_HYBRID) tma::load4(dst + 5 * MPTS, &tm_th, &bars[s], c0, c1, c2, 0);
    };
    if (tid == MTMA) {
#pragma unroll
        for (int q = 0; q < MNST; ++q) tma::mbar_init(&bars[q], 1);
        tma::fence_barrier_init();
        issue(0);
        if (nch > 1) issue(1);
#pragma unroll
        for (int q = 2; q < MPF; ++q)
            if (nch > q) issue(q);
    }

    // phase A role: point (row pr, pencil pa) of every chunk; walker role: pencil wa, component wm
    // (in both cases the point of thread tid sits at position tid of a staged box)
    const int pr = DIR == 0 ? tid % MR : tid / MAC, pa = DIR == 0 ? (tid / MR) % MAC : tid % MAC;
    const bool producer = tid < MPTS;
    const int wa = tid % MAC, wm = tid / MAC;
    const int apA = OCFD_NG + a0 + pa;
    const bool x_ok = apA < nap - OCFD_NG;   // pencils past the last interior line hold zero-filled state
    const JRow<KIND, DIR> jrow(g, min(OCFD_NG + a0 + wa, nap - 1), OCFD_NG + cross);
    const int sfi = DIR == 0 ? pr * MAC + (pa ^ (pr << 2)) : tid;   // this thread's point inside a split-flux field

    // Register windows as rings of 8: padded row r lives in slot r % 8.  Two chunks (8 rows) bring every slot back to
    // its place, so the chunk loop is unrolled by two and no value is ever moved between registers.
    double Wp[8], Wm[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) Wp[e] = Wm[e] = 0.0;
    double hprev = 0.0;
    double Jnext[MR] = {0.0, 0.0, 0.0, 0.0};   // curvilinear: J of the rows of the chunk whose phase B ran last (see phase B)
    unsigned pprev = 0;     // packed scheme flags pf(r) of the previous chunk's rows, 2 bits per row (hybrid)
    __syncthreads();        // barriers initialised before anyone polls them

    // ---- phase A of chunk c: split fluxes of the chunk's points -> sF[c % 2]; pf(r) = scheme flag of the interface
    // between rows r-1 and r -> sFl[c % 2]
    auto phaseA = [&](const int lc) {
        const int s = lc % MNST;
        const double *sU = sIn + s * MSTG;
        const int rowA = MR * (cbeg + lc) + pr;
        const bool validA = producer && x_ok && rowA < ndp;
        // metric data of this thread's point, fetched while the boxes are in flight
        double k1 = 0.0, k2 = 0.0, k3 = 0.0, sig = 1.0, Jdead;
        if (KIND != OCFD_GRID_CURVILINEAR && validA)
            met_ksJ<KIND, DIR>(g, DIR == 0 ? rowA : apA, DIR == 0 ? apA : DIR == 1 ? rowA : OCFD_NG + cross,
                               DIR == 2 ? rowA : OCFD_NG + cross, k1, k2, k3, sig, Jdead);
        tma::mbar_wait(&bars[s], (lc / MNST) & 1);   // every thread: the walkers read J of this stage one chunk later
        if (!producer) return;
        if (KIND == OCFD_GRID_CURVILINEAR && validA) {
            // the metric box lands densely: field stride = its own row count x MAC
            const int mi = DIR == 0 ? pr * MAC + pa : mfull ? tid : pa, mfs = mfull ? MPTS : MAC;
            const double *mp = sU + 6 * MPTS + mi;
            k1 = mp[0]; k2 = mp[mfs]; k3 = mp[2 * mfs]; sig = mp[3 * mfs];
        }
        double *dst = sF + (lc & 1) * 10 * MPTS + sfi;
        if (validA) {
            double u, v, w, cc;
            const double rho = sU[tid];
            prim_from_cons(gs, rho, sU[MPTS + tid], sU[2 * MPTS + tid], sU[3 * MPTS + tid], sU[4 * MPTS + tid], u, v, w, cc);
            sw_split_store<KIND, DIR>(gs, rho, u, v, w, cc, k1, k2, k3, sig, dst, MPTS);
        } else {
#pragma unroll
            for (int q = 0; q < 10; ++q) dst[q * MPTS] = 0.0;
        }
        if (SCHEME == OCFD_HYBRID) {
            unsigned char f = 0;
            // interfaces -1/2 .. nd-1/2 (eq. 42, R-12) of live pencils: a pencil past the last interior line would read
            // theta from ghost rows nobody wrote, and one lane on the non-linear path costs its whole warp that path
            if (x_ok && rowA >= OCFD_NG && rowA <= nd + OCFD_NG) {
                const double *thp =
                    pr > 0 ? sU + 5 * MPTS + tid - (DIR == 0 ? 1 : MAC)
                           : sIn + ((lc + MNST - 1) % MNST) * MSTG + 5 * MPTS + (DIR == 0 ? tid + MR - 1 : (MR - 1) * MAC + pa);
                f = (unsigned char)iface_flag(gs, *thp, sU[5 * MPTS + tid]);
            }
            sFl[(lc & 1) * 4 * MAC + 4 * pa + pr] = f;
        }
    };

    // ---- phase B of chunk c (PH = c % 2 fixes the ring slots at compile time): push the chunk's rows through the
    // register windows.  Pushing row r completes interface (r-4)+1/2 (f+ rows r-7..r-1, f- rows r-6..r) and point r-4.
    auto phaseB = [&](const int lc, auto ph) {
        constexpr int PH = decltype(ph)::value;
        const int r0 = MR * (cbeg + lc);   // first padded row of the chunk
        // J of the four points this walker completes in this chunk (padded rows r0-4 .. r0-1; the first chunk
        // completes nothing that is kept)
        double Jw[MR];
        if (KIND != OCFD_GRID_CURVILINEAR) {
            const int i0 = max(r0 - OCFD_NG, 0);
#pragma unroll
            for (int e = 0; e < MR; ++e) Jw[e] = jrow.at(g, i0, e);
        } else {
            // J of rows r0-4 .. r0-1 arrived with chunk c-1, whose stage is being refilled by now: this walker took it
            // into registers during its previous phase B, and now takes the J of this chunk's rows for the next one
            // (the stage of chunk c is intact until the barrier that ends this interval)
            if (DIR == 0) {   // (x sweep: straight from the stage of chunk c-1, see MRing::PF)
                const double *jp = sIn + ((lc + MNST - 1) % MNST) * MSTG + 10 * MPTS;
#pragma unroll
                for (int e = 0; e < MR; ++e) Jw[e] = jp[e * MAC + wa];
            } else {
                const double *jp = sIn + (lc % MNST) * MSTG + 6 * MPTS + 4 * (mfull ? MPTS : MAC);
#pragma unroll
                for (int e = 0; e < MR; ++e) {
                    Jw[e] = Jnext[e];
                    Jnext[e] = jp[(mfull ? e * MAC : 0) + wa];
                }
            }
        }
        double *so = sO + PH * 5 * MPTS + wm * MPTS + (DIR == 0 ? wa * MR : wa);
        const double *fpn = sF + PH * 10 * MPTS + wm * MPTS, *fmn = fpn + 5 * MPTS;
        double out[MR];
        bool fast = SCHEME == OCFD_UD7;
        unsigned cur = 0;
        if (SCHEME == OCFD_HYBRID) {
            const unsigned w = reinterpret_cast<const unsigned *>(sFl + PH * 4 * MAC)[wa];
            const unsigned pc = (w & 3u) | ((w >> 6) & 0xcu) | ((w >> 12) & 0x30u) | ((w >> 18) & 0xc0u);
            // the interfaces completed in this chunk: pf(r0-3), pf(r0-2), pf(r0-1), pf(r0)
            cur = ((pprev >> 2) | (pc << 6)) & 0xffu;
            pprev = pc;
            fast = cur == 0;
        }
        // the paper's boundary scheme (ocfd_params.bc_closure): the chunks whose interfaces s = r0-8 .. r0-5 come within
        // reach of a boundary (s <= 2 or s >= nd-4) take the out-of-line path, which tests every interface
        const bool near_bnd = g.closure[DIR] && (r0 - 2 * OCFD_NG <= 2 || r0 + MR - 1 - 2 * OCFD_NG >= nd - 4);
        if (near_bnd) fast = false;
        double nP[MR], nM[MR];   // the chunk's new rows (loaded up front, entered into the rings one by one)
#pragma unroll
        for (int e = 0; e < MR; ++e) {
            const int q = e * MAC + (DIR == 0 ? wa ^ (e << 2) : wa);
            nP[e] = fpn[q];
            nM[e] = fmn[q];
        }
        if (fast) {
#pragma unroll
            for (int e = 0; e < MR; ++e) {
                const int k = 4 * PH + e;
                Wp[k & 7] = nP[e];
                Wm[k & 7] = nM[e];
                const double h = ud7(Wp[(k + 1) & 7], Wp[(k + 2) & 7], Wp[(k + 3) & 7], Wp[(k + 4) & 7], Wp[(k + 5) & 7],
                                     Wp[(k + 6) & 7], Wp[(k + 7) & 7]) +
                                 ud7(Wm[k & 7], Wm[(k + 7) & 7], Wm[(k + 6) & 7], Wm[(k + 5) & 7], Wm[(k + 4) & 7],
                                     Wm[(k + 3) & 7], Wm[(k + 2) & 7]);
                if (DIR == 0) out[e] = -Jw[e] * (h - hprev);
                else so[e * MAC] = -Jw[e] * (h - hprev);
                hprev = h;
            }
        } else if (near_bnd) {
            // chunks next to an aperiodic boundary under the paper's boundary scheme: every interface is tested (a
            // branch of its own, so that the out-of-line call does not weigh on the general path below)
#pragma unroll
            for (int e = 0; e < MR; ++e) {
                const int k = 4 * PH + e;
                Wp[k & 7] = nP[e];
                Wm[k & 7] = nM[e];
                const int flag = SCHEME == OCFD_HYBRID ? (int)((cur >> (2 * e)) & 3u) : 0;
                const double h = recon_pair_closure<SCHEME>(
                    flag, r0 + e - 2 * OCFD_NG, nd, Wp[(k + 1) & 7], Wp[(k + 2) & 7], Wp[(k + 3) & 7], Wp[(k + 4) & 7],
                    Wp[(k + 5) & 7], Wp[(k + 6) & 7], Wp[(k + 7) & 7], Wm[k & 7], Wm[(k + 7) & 7], Wm[(k + 6) & 7],
                    Wm[(k + 5) & 7], Wm[(k + 4) & 7], Wm[(k + 3) & 7], Wm[(k + 2) & 7], gs.weno_eps);
                if (DIR == 0) out[e] = -Jw[e] * (h - hprev);
                else so[e * MAC] = -Jw[e] * (h - hprev);
                hprev = h;
            }
        } else {
#pragma unroll
            for (int e = 0; e < MR; ++e) {
                const int k = 4 * PH + e;
                Wp[k & 7] = nP[e];
                Wm[k & 7] = nM[e];
                const int flag = SCHEME == OCFD_HYBRID ? (int)((cur >> (2 * e)) & 3u) : 0;
                const double h = recon_pair<SCHEME>(flag, Wp[(k + 1) & 7], Wp[(k + 2) & 7], Wp[(k + 3) & 7], Wp[(k + 4) & 7],
                                                    Wp[(k + 5) & 7], Wp[(k + 6) & 7], Wp[(k + 7) & 7], Wm[k & 7],
                                                    Wm[(k + 7) & 7], Wm[(k + 6) & 7], Wm[(k + 5) & 7], Wm[(k + 4) & 7],
                                                    Wm[(k + 3) & 7], Wm[(k + 2) & 7], gs.weno_eps);
                if (DIR == 0) out[e] = -Jw[e] * (h - hprev);
                else so[e * MAC] = -Jw[e] * (h - hprev);
                hprev = h;
            }
        }
        if (DIR == 0) {
            reinterpret_cast<double2 *>(so)[0] = make_double2(out[0], out[1]);
            reinterpret_cast<double2 *>(so)[1] = make_double2(out[2], out[3]);
        }
    };

    // One CTA barrier per chunk: between two barriers the CTA runs phase A of chunk c+1 and phase B of chunk c (the
    // split fluxes are double-buffered), so the warp that has no phase-A work and the warps that finish early always
    // find work of the other kind.  After the barrier: the output tile of chunk c leaves, and the boxes of chunk
    // c + MNST are requested into the stage of chunk c (phase A of chunk c+1 has read its last theta row).
    auto interval = [&](const int lc, auto ph) {
        constexpr int PH = decltype(ph)::value;
        if (lc + 1 < nch) phaseA(lc + 1);
        phaseB(lc, ph);
        tma::fence_proxy_async();
        // the store of chunk c-1 has finished reading the tile that phase B of chunk c+1 is about to overwrite (it was
        // issued one interval ago)
        if (tid == MTMA) tma::store_wait_read<0>();
        __syncthreads();
        if (tid == MTMA) {
            const int o = MR * (cbeg + lc) - 2 * OCFD_NG;   // interior index of the first point completed by this chunk
            if (o >= o0) {                                  // (the first two chunks of a segment only fill the windows)
                if (DIR == 0) tma::store4(&tm_out, sO + PH * 5 * MPTS, o, a0, cross, 0);
                else tma::reduce_add4(&tm_out, sO + PH * 5 * MPTS, a0, DIR == 1 ? o : cross, DIR == 2 ? o : cross, 0);
                tma::store_commit();
            }
            if (lc + MPF < nch) issue(lc + MPF);
        }
    };
    phaseA(0);
    __syncthreads();
    for (int lc = 0; lc < nch; lc += 2) {
        interval(lc, std::integral_constant<int, 0>());
        if (lc + 1 < nch) interval(lc + 1, std::integral_constant<int, 1>());
    }
    if (tid == MTMA) tma::store_wait_all<0>();
}

template <int KIND, int SCHEME, int DIR, bool MFULL>
ocfd_status launch_march_m(ocfd_ctx *c) {
    const GridDesc &g = c->g;
    constexpr size_t M_SMEM = MRing<KIND, DIR, MFULL>::SMEM;
    if (!ocfd_smem_optin(c, (const void *)k_inviscid_march<KIND, SCHEME, DIR, MFULL>, M_SMEM)) return OCFD_ECUDA;
    const int ncross = DIR == 2 ? g.ny : g.nz;
    if (ncross > 65535) return OCFD_EINVAL;
    const int nd = DIR == 0 ? g.nx : DIR == 1 ? g.ny : g.nz, ntile = ((DIR == 0 ? g.ny : g.nx) + MAC - 1) / MAC;
    // Segments along the march: as few as give every SM's three CTA slots about eight CTAs to work through (a CTA that
    // marches 2000 rows runs for a millisecond, and the SMs that finish their last one early then idle), never shorter
    // than 128 rows (each segment re-stages 8 rows); "march_seg" of ocfd_set_tuning overrides (A/B runs).
    int nseg = 1;
    while ((long long)ntile * ncross * nseg < 24ll * c->nsm && nd / (nseg + 1) >= 128) ++nseg;
    if (c->tune.march_seg > 0) nseg = c->tune.march_seg;
    int seglen = ((nd + nseg - 1) / nseg + MR - 1) / MR * MR;
    if (seglen < 2 * MR) seglen = 2 * MR;
    nseg = (nd + seglen - 1) / seglen;
    dim3 grd(ntile, ncross, nseg);
    OCFD_T0(c, K_INV_X + DIR);
    const MarchMaps &M = c->march;
    k_inviscid_march<KIND, SCHEME, DIR, MFULL><<<grd, MNT, M_SMEM, c->stream>>>(g, c->gas, M.U[DIR], M.th[DIR], M.out[DIR],
                                                                               M.met[DIR], seglen);
    OCFD_CHECK_LAUNCH(c);
    return OCFD_OK;
}

// the z sweep over a z-extruded curvilinear map has an instance of its own (one metric row per chunk: smaller stages,
// more of them)
template <int KIND, int SCHEME, int DIR>
ocfd_status launch_march(ocfd_ctx *c) {
    if (KIND == OCFD_GRID_CURVILINEAR && DIR == 2 && c->g.msk == 0) return launch_march_m<KIND, SCHEME, DIR, false>(c);
    return launch_march_m<KIND, SCHEME, DIR, true>(c);
}

template <int KIND, int SCHEME>
ocfd_status launch_march_dir(ocfd_ctx *c, int dir) {
    return dir == 0 ? launch_march<KIND, SCHEME, 0>(c) : dir == 1 ? launch_march<KIND, SCHEME, 1>(c) : launch_march<KIND, SCHEME, 2>(c);
}

template <int KIND>
ocfd_status launch_march_kind(ocfd_ctx *c, int dir) {
    switch (c->p.scheme) {
        case OCFD_UD7: return launch_march_dir<KIND, OCFD_UD7>(c, dir);
        case OCFD_WENO7: return launch_march_dir<KIND, OCFD_WENO7>(c, dir);
        case OCFD_WENO5: return launch_march_dir<KIND, OCFD_WENO5>(c, dir);
        default: return launch_march_dir<KIND, OCFD_HYBRID>(c, dir);
    }
}

// input boxes over the whole padded arrays, output boxes over the interior of dU
bool encode_march_maps(ocfd_ctx *c, const double *U, double *dU) {
    const GridDesc &g = c->g;
    MarchMaps &M = c->march;
    const long long full1[4] = {g.nxp, g.nyp, g.nzp, 1}, full5[4] = {g.nxp, g.nyp, g.nzp, 5};
    const long long inner[4] = {g.nx, g.ny, g.nz, 5};
    for (int d = 0; d < 3; ++d) {
        const int bx = d == 0 ? MR : MAC, by = d == 0 ? MAC : d == 1 ? MR : 1, bz = d == 2 ? MR : 1;
        const int b1[4] = {bx, by, bz, 1}, bo[4] = {bx, by, bz, 5};
        if (!M.ready) {
            if (g.kind == OCFD_GRID_CURVILINEAR) {
                // the derived metric table of this direction: [5][planes][nyp][nxp], one plane if z-extruded
                const long long mdim[4] = {g.nxp, g.nyp, g.msk ? g.nzp : 1, 5};
                const int mz = d == 2 && g.msk ? MR : 1;
                const int m5[4] = {bx, by, mz, 5};   // k1, k2, k3, sigma, J as one box
                if (d == 0) {   // y-contiguous copy [5][planes][nxp][nypT]: boxes of 4 rows of 32 lines
                    const long long tdim[4] = {g.nyp, g.nxp, g.msk ? g.nzp : 1, 5};
                    const int t5[4] = {MAC, MR, 1, 5};
                    if (!ocfd_tma_encode(&M.met[d], g.atabT, tdim, g.nypT, (long long)g.nxp * g.nypT, g.atabT_fs, t5)) return false;
                } else {
                    if (!ocfd_tma_encode(&M.met[d], g.atab[d], mdim, g.sy, g.sz, g.atab_fs, m5)) return false;
                }
            } else {   // unused, but the kernel takes the parameters
                M.met[d] = CUtensorMap();
            }
            if (!ocfd_tma_encode(&M.th[d], c->theta, full1, g.sy, g.sz, g.np, b1, d == 0)) return false;
        }
        if (M.Up != U && !ocfd_tma_encode(&M.U[d], U, full5, g.sy, g.sz, g.np, bo, d == 0)) return false;
        if (M.dUp != dU &&
            !ocfd_tma_encode(&M.out[d], dU + (long long)OCFD_NG * (g.sz + g.sy + 1), inner, g.sy, g.sz, g.np, bo))
            return false;
    }
    M.ready = true;
    M.Up = U;
    M.dUp = dU;
    return true;
}

}  // namespace

ocfd_status launch_inviscid_march(ocfd_ctx *c, const double *U, double *dU, int dir) {
    if (dir < 0 || dir > 2) return OCFD_EINVAL;
    if (!encode_march_maps(c, U, dU)) return OCFD_ECUDA;
    switch (c->g.kind) {
        case OCFD_GRID_UNIFORM: return launch_march_kind<OCFD_GRID_UNIFORM>(c, dir);
        case OCFD_GRID_STRETCHED: return launch_march_kind<OCFD_GRID_STRETCHED>(c, dir);
        default: return launch_march_kind<OCFD_GRID_CURVILINEAR>(c, dir);
    }
}
