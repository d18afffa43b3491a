// Rows a6 + a7 (+ a8 fused): viscous and heat-flux terms (eq. 9-15) by the 6th-order central
// first derivative applied twice (DESIGN R-15): pass 1 forms the viscous fluxes at interior
// points, pass 2 differences them and accumulates into dU (and, inside ocfd_rk3_step, applies the RK3 stage update
// of eq. 45 in the same kernel so that dU is not written and re-read).
//
// Pass 1 reads the conserved variables and forms T, u, v, w itself (row a2; no primitive field exists in HBM); for the
// hybrid scheme it also writes the shock sensor (row a3), whose inputs it has staged anyway.
//
// Both passes are 2.5-D marching kernels: a CTA owns a 32 x 8 tile in x-y and walks along z.  Every z-plane of every
// input is fetched exactly once, by TMA box loads into a ring of shared-memory stages that run two or more planes
// ahead of the arithmetic (one elected thread issues them, completion is signalled on one mbarrier per stage), so the
// HBM pipe stays full without tying up registers.  The seven z-planes the zeta-derivative needs live in a register
// window per thread; the x / y neighbours of the current plane are read from the staged box (3-point halos; the box is
// 4 wider in x on each side because a TMA box of doubles must start at an even x index).
#include "ocfd_internal.cuh"
#include "schemes.cuh"
#include "tma.cuh"


namespace {

constexpr int TX = 32, TY = 8, VNT = TX * TY;  // own points of a tile = threads

// Tile of a CTA.  The hardware hands out CTAs in the order of their linear index; with the plain x-fastest numbering
// the CTAs resident at one time form two or three full rows of tiles, and most y halos are fetched from HBM twice.
// Numbering the tiles column group by column group (gw tiles wide, y fastest between the rows of a group) makes the
// resident set a compact block whose inner halos are found in the L2; rows of a group stay contiguous in memory.
__device__ __forceinline__ void tile_of_block(int gw, int &bx, int &by) {
    const int nxt = gridDim.x, nyt = gridDim.y;
    const int L = blockIdx.x + nxt * blockIdx.y;
    const int nfull = nxt / gw, rem = nxt - nfull * gw;
    if (L < nfull * gw * nyt) {
        const int grp = L / (gw * nyt), r = L - grp * gw * nyt;
        by = r / gw;
        bx = grp * gw + (r - by * gw);
    } else {
        const int r = L - nfull * gw * nyt;
        by = r / rem;
        bx = nfull * gw + (r - by * rem);
    }
}
constexpr int BXW = TX + 8;                    // x extent of a box with x halos (i0-4 .. i0+TX+3)
template <int ORDER>
struct VG {                                    // geometry of the scheme of order ORDER (6 or 8)
    static constexpr int H = ORDER / 2;        // stencil reach
    static constexpr int BYH = TY + 2 * H;     // y extent of a box with y halos (j0-H .. j0+TY+H-1)
    static constexpr int W = 2 * H + 1;        // z window
};

// central-difference coefficients in constant memory: every DFMA takes its coefficient as a constant-bank operand (an
// immediate fp64 constant costs two moves per use)
__constant__ double c_d6[3] = {45.0 / 60.0, -9.0 / 60.0, 1.0 / 60.0};                               // 6th order (L313)
__constant__ double c_d8[4] = {672.0 / 840.0, -168.0 / 840.0, 32.0 / 840.0, -3.0 / 840.0};         // 8th order: 4/5, -1/5, 4/105, -1/280

__device__ __forceinline__ double d1c(double m3, double m2, double m1, double p1, double p2, double p3) {
    return fma(c_d6[2], p3 - m3, fma(c_d6[1], p2 - m2, c_d6[0] * (p1 - m1)));
}
__device__ __forceinline__ double d1c8(double m4, double m3, double m2, double m1, double p1, double p2, double p3,
                                       double p4) {
    return fma(c_d8[3], p4 - m4, fma(c_d8[2], p3 - m3, fma(c_d8[1], p2 - m2, c_d8[0] * (p1 - m1))));
}
// interior stencil of order ORDER on a line (p points at the position, stride st)
template <int ORDER>
__device__ __forceinline__ double d1_int(const double *p, int st) {
    if (ORDER == 8) return d1c8(p[-4 * st], p[-3 * st], p[-2 * st], p[-st], p[st], p[2 * st], p[3 * st], p[4 * st]);
    return d1c(p[-3 * st], p[-2 * st], p[-st], p[st], p[2 * st], p[3 * st]);
}
// first derivative at position s of a line of n; closure rows of an aperiodic axis (one-sided 2nd order
// at the boundary point, central 2nd / 4th / 6th order at the 2nd / 3rd / 4th point) only touch values inside the line
template <int ORDER>
__device__ __forceinline__ double d1_line(const double *p, int st, int s, int n, int periodic) {
    constexpr int H = ORDER / 2;
    if (periodic || (s >= H && s <= n - 1 - H)) return d1_int<ORDER>(p, st);
    if (s == 0) return (-3.0 * p[0] + 4.0 * p[st] - p[2 * st]) * 0.5;
    if (s == n - 1) return (3.0 * p[0] - 4.0 * p[-st] + p[-2 * st]) * 0.5;
    if (s == 1 || s == n - 2) return (p[st] - p[-st]) * 0.5;
    if (s == 2 || s == n - 3) return (8.0 * (p[st] - p[-st]) - (p[2 * st] - p[-2 * st])) * (1.0 / 12.0);
    return d1c(p[-3 * st], p[-2 * st], p[-st], p[st], p[2 * st], p[3 * st]);   // ORDER 8, s == 3 or n-4
}
// the same from a register window v[0..2H] = f_{s-H..s+H}
template <int ORDER>
__device__ __forceinline__ double d1_win(const double *v, int s, int n, int periodic) {
    constexpr int H = ORDER / 2;
    if (periodic || (s >= H && s <= n - 1 - H)) {
        if (ORDER == 8) return d1c8(v[0], v[1], v[2], v[3], v[5], v[6], v[7], v[8]);
        return d1c(v[0], v[1], v[2], v[4], v[5], v[6]);
    }
    if (s == 0) return (-3.0 * v[H] + 4.0 * v[H + 1] - v[H + 2]) * 0.5;
    if (s == n - 1) return (3.0 * v[H] - 4.0 * v[H - 1] + v[H - 2]) * 0.5;
    if (s == 1 || s == n - 2) return (v[H + 1] - v[H - 1]) * 0.5;
    if (s == 2 || s == n - 3) return (8.0 * (v[H + 1] - v[H - 1]) - (v[H + 2] - v[H - 2])) * (1.0 / 12.0);
    return d1c(v[H - 3], v[H - 2], v[H - 1], v[H + 1], v[H + 2], v[H + 3]);
}

// ------------------------------------------------------------------------------------------------ a6 (+ a2, a3)
// Input: the conserved variables U (valid on interior + face ghosts).  Every staged plane is converted IN PLACE to
// (T, u, v, w, p) by the whole CTA as soon as it lands (row a2 lives here and in the sweeps; no primitive field exists
// in HBM).  Output Fv[12][np] at interior points, plus, on periodic axes, the three image planes each direction's flux
// needs beyond the faces (pass 2 fetches plain boxes and cannot wrap).
// SENSOR (hybrid scheme): the kernel also writes the shock sensor theta (row a3, eq. 42; R-11, R-12)
// of its points: p of the x / y neighbours sits in the converted plane, p of plane k+1 in the ring, p of plane k-1 in a
// register, so the sensor costs no HBM read at all, only its 8 B/point write.  ocfd_rk3_step therefore runs this
// kernel BEFORE the inviscid sweeps of the stage (it depends on U only).
template <int ORDER>
struct VF {
    static constexpr int NST = VG<ORDER>::H + 2;                 // ring: planes k..k+H+1 (the newest being converted)
    static constexpr int FLD = VG<ORDER>::BYH * BXW;             // doubles per staged field
    static constexpr int STAGE = 5 * FLD;                        // doubles per stage
    static constexpr size_t SMEM = sizeof(double) * NST * STAGE + 8 * NST;
    static_assert((STAGE * 8) % 128 == 0, "TMA destinations must stay 128-byte aligned");
};

// (rho, rho u, rho v, rho w, E) -> (T, u, v, w, p) of one staged plane, in place.  Only the points a stencil reaches are
// converted: the own rows with their x halo and the y-halo rows above the own columns (496 of the 560 staged points
// for the 6th-order scheme: two rounds of the 256 threads instead of three); the corners stay raw and are never read.
// The positions a thread converts are the same in every plane: convert_slots works them out once (-1 = none).
template <int ORDER>
struct ConvSlots {
    static constexpr int H = VG<ORDER>::H, WX = TX + 2 * H, N1 = TY * WX, N = N1 + 2 * H * TX, ROUNDS = (N + VNT - 1) / VNT;
    int p[ROUNDS];
};
template <int ORDER>
__device__ __forceinline__ ConvSlots<ORDER> convert_slots(int tid) {
    using C = ConvSlots<ORDER>;
    C c;
#pragma unroll
    for (int r = 0; r < C::ROUNDS; ++r) {
        const int q = tid + r * VNT;
        int row, col;
        if (q < C::N1) {
            row = C::H + q / C::WX;
            col = 4 - C::H + q % C::WX;
        } else {
            const int hr = (q - C::N1) / TX;
            row = hr < C::H ? hr : hr + TY;
            col = 4 + (q - C::N1) % TX;
        }
        c.p[r] = q < C::N ? row * BXW + col : -1;
    }
    return c;
}
template <int ORDER>
__device__ __forceinline__ void convert_plane(const GasDesc &gs, double *st, const ConvSlots<ORDER> &slots) {
    constexpr int FLD = VF<ORDER>::FLD;
#pragma unroll
    for (int r = 0; r < ConvSlots<ORDER>::ROUNDS; ++r) {
        const int p = slots.p[r];
        if (p < 0) continue;
        const double rho = st[p];
        const double ir = fast_rcp_pos(rho);
        const double u = st[FLD + p] * ir, v = st[2 * FLD + p] * ir, w = st[3 * FLD + p] * ir;
        const double pr = gs.gm1 * (st[4 * FLD + p] - 0.5 * rho * (u * u + v * v + w * w));
        st[p] = gs.gM2 * pr * ir;
        st[FLD + p] = u;
        st[2 * FLD + p] = v;
        st[3 * FLD + p] = w;
        st[4 * FLD + p] = pr;
    }
}

template <int KIND, int ORDER, bool SENSOR>
__global__ void __launch_bounds__(VNT, ORDER == 8 ? 1 : 2)
    k_viscous_flux(const GridDesc g, const GasDesc gs, const __grid_constant__ CUtensorMap tm_U,
                   const double *__restrict__ U, double *__restrict__ Fv, double *__restrict__ theta, int zchunk,
                   int tgroup) {
    constexpr int H = VG<ORDER>::H, VF_NST = VF<ORDER>::NST, VF_STAGE = VF<ORDER>::STAGE, FLD = VF<ORDER>::FLD;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *ring = reinterpret_cast<double *>(smem_raw);
    uint64_t *bars = reinterpret_cast<uint64_t *>(ring + VF_NST * VF_STAGE);
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * TX + tx;
    int tbx, tby;
    tile_of_block(tgroup, tbx, tby);
    const int i0 = tbx * TX, j0 = tby * TY;
    const int i = i0 + tx, j = j0 + ty;
    const bool own = i < g.nx && j < g.ny;
    const int k0 = blockIdx.z * zchunk, k1 = min(k0 + zchunk, g.nz);
    const int last = k1 + H - 1;  // last plane the window needs
    auto issue = [&](int plane) {  // plane k (interior index) -> stage (k - k0) % NST
        const int s = (plane - k0) % VF_NST;
        tma::mbar_expect_tx(&bars[s], VF_STAGE * 8);
        tma::load4_hint(ring + s * VF_STAGE, &tm_U, &bars[s], i0, j0 + OCFD_NG - H, plane + OCFD_NG, 0,
                        tma::policy_evict_last());   // the halo of this box is a neighbouring tile's interior
    };
    if (tid == 0) {
        for (int s = 0; s < VF_NST; ++s) tma::mbar_init(&bars[s], 1);
        tma::fence_barrier_init();
        for (int q = 0; q < VF_NST; ++q)
            if (k0 + q <= last) issue(k0 + q);
    }
    // z window: planes k-H .. k+H of T,u,v,w at this thread's column.  The H planes below the chunk come straight from
    // global memory (converted here), everything else through the ring.
    const int ipc = min(i, g.nx - 1) + OCFD_NG, jpc = min(j, g.ny - 1) + OCFD_NG;
    const long long col = (long long)jpc * g.sy + ipc;
    const int ctr = (ty + H) * BXW + tx + 4;  // own point inside a staged field
    // Only the H planes BELOW the current one live in registers (wlo[a][q] = plane k-H+q); the current plane and the H
    // planes above it are read from the ring, where they sit converted anyway: 12 registers of window per field set
    // instead of 28, and 3 values to shift per field and plane instead of 6.
    double wlo[4][H];
    double pm = 0.0;                           // p of plane k-1 (sensor)
#pragma unroll
    for (int q = 0; q < H; ++q) {
        const long long id = (long long)(k0 - H + q + OCFD_NG) * g.sz + col;
        const double rho = __ldg(U + id), ir = fast_rcp_pos(rho);
        const double u = __ldg(U + g.np + id) * ir, v = __ldg(U + 2 * g.np + id) * ir, ww = __ldg(U + 3 * g.np + id) * ir;
        const double pr = gs.gm1 * (__ldg(U + 4 * g.np + id) - 0.5 * rho * (u * u + v * v + ww * ww));
        wlo[0][q] = gs.gM2 * pr * ir; wlo[1][q] = u; wlo[2][q] = v; wlo[3][q] = ww;
        pm = pr;
    }
    const ConvSlots<ORDER> slots = convert_slots<ORDER>(tid);
    __syncthreads();  // barriers initialised
    // planes k0 .. k0+H: convert, then take the own column of the first H into the window
#pragma unroll 1
    for (int q = 0; q <= H; ++q) {
        if (k0 + q > last) break;
        tma::mbar_wait(&bars[q], 0);
        convert_plane<ORDER>(gs, ring + q * VF_STAGE, slots);
    }
    // convert_plane writes a TMA destination in place (generic proxy); a later box load overwrites the same bytes through
    // the async proxy, so every thread orders its writes before the barrier that lets tid 0 issue that load
    tma::fence_proxy_async();
    __syncthreads();
    // whole-tile tests: away from aperiodic faces every point takes the central stencil and no row test is needed
    const bool xin = g.periodic[0] || (i0 >= H && i0 + TX <= g.nx - H);
    const bool yin = g.periodic[1] || (j0 >= H && j0 + TY <= g.ny - H);
    // z-extruded metrics (one plane): fetched once for the whole march
    const bool hoist = KIND == OCFD_GRID_CURVILINEAR && g.msk == 0;
    double m[3][3], iJ = 0.0;
    if (hoist && own) {
#pragma unroll
        for (int d = 0; d < 3; ++d) Met<KIND>::row(g, d, i + OCFD_NG, j + OCFD_NG, 0, m[d][0], m[d][1], m[d][2]);
        iJ = 1.0 / Met<KIND>::J(g, i + OCFD_NG, j + OCFD_NG, 0);
    }
    const int ip = i + OCFD_NG, jp = j + OCFD_NG;
    long long id = (long long)(k0 + OCFD_NG) * g.sz + (long long)jp * g.sy + ip;   // this thread's point of plane k
    int sk = 0;                                                                    // ring stage of plane k
    // periodic images in x and y: fixed per thread
    const int imx = !g.periodic[0] ? 0 : i < H ? 1 : i >= g.nx - H ? -1 : 0;
    const int imy = !g.periodic[1] ? 0 : j < H ? 1 : j >= g.ny - H ? -1 : 0;
    double *Fp = Fv + id;
    const bool xy_edge = i == 0 || j == 0 || i == g.nx - 1 || j == g.ny - 1;   // touches a face in x or y (theta ghosts)
    for (int k = k0; k < k1; ++k, id += g.sz, Fp += g.sz, sk = sk + 1 == VF_NST ? 0 : sk + 1) {
        const int kp = k + OCFD_NG;
        const bool zin = g.periodic[2] || (k >= H && k <= g.nz - 1 - H);   // central stencil along z in this plane
        if (own) {
            const double *sp = ring + sk * VF_STAGE + ctr;
            // z window of the four fields: planes k-H .. k-1 from registers, k .. k+H from the ring (plane k+H was
            // converted during the previous iteration, or before the loop)
            double w[4][2 * H + 1];
#pragma unroll
            for (int a = 0; a < 4; ++a) {
#pragma unroll
                for (int q = 0; q < H; ++q) w[a][q] = wlo[a][q];
#pragma unroll
                for (int q = 0; q <= H; ++q) {
                    const int sq = sk + q < VF_NST ? sk + q : sk + q - VF_NST;
                    w[a][H + q] = ring[sq * VF_STAGE + a * FLD + ctr];
                }
#pragma unroll
                for (int q = 0; q + 1 < H; ++q) wlo[a][q] = wlo[a][q + 1];
                wlo[a][H - 1] = w[a][H];
            }
            if (SENSOR) {
                // theta = phi_i + phi_j + phi_k, phi = |p- - 2 p0 + p+| / (p- + 2 p0 + p+); one division for the three
                const double *cp = sp + 4 * FLD;
                const double p0 = cp[0], pp = ring[(sk + 1 < VF_NST ? sk + 1 : 0) * VF_STAGE + 4 * FLD + ctr];
                const double t0 = p0 + p0;
                const double ni = fabs(t0 - cp[-1] - cp[1]), di = t0 + cp[-1] + cp[1];
                const double nj = fabs(t0 - cp[-BXW] - cp[BXW]), dj = t0 + cp[-BXW] + cp[BXW];
                const double nk = fabs(t0 - pm - pp), dk = t0 + pm + pp;
                const double dij = di * dj;
                const double th = fast_div_pos(ni * (dj * dk) + nj * (di * dk) + nk * dij, dij * dk);
                pm = p0;
                theta[id] = th;
                if (xy_edge || k == 0 || k == g.nz - 1) {
                    // first ghost layer of theta: wrap on periodic axes, else the nearest interior value (R-12)
                    const int cc[3] = {i, j, k};
                    const int n[3] = {g.nx, g.ny, g.nz};
                    const long long st[3] = {1, g.sy, g.sz};
#pragma unroll
                    for (int d = 0; d < 3; ++d) {
                        if (cc[d] == 0) theta[g.periodic[d] ? id + n[d] * st[d] : id - st[d]] = th;
                        if (cc[d] == n[d] - 1) theta[g.periodic[d] ? id - n[d] * st[d] : id + st[d]] = th;
                    }
                }
            }
            double gr[4][3];
#pragma unroll
            for (int a = 0; a < 4; ++a) {
                const double *q = sp + a * FLD;
                gr[a][0] = xin ? d1_int<ORDER>(q, 1) : d1_line<ORDER>(q, 1, i, g.nx, 0);
                gr[a][1] = yin ? d1_int<ORDER>(q, BXW) : d1_line<ORDER>(q, BXW, j, g.ny, 0);
                gr[a][2] = zin ? d1_win<ORDER>(w[a], H, 2 * H + 1, 1) : d1_win<ORDER>(w[a], k, g.nz, 0);
            }
            if (!hoist) {
#pragma unroll
                for (int d = 0; d < 3; ++d) Met<KIND>::row(g, d, ip, jp, kp, m[d][0], m[d][1], m[d][2]);
                iJ = 1.0 / Met<KIND>::J(g, ip, jp, kp);
            }
            double gx[4], gy[4], gz[4];  // Cartesian gradients of T,u,v,w (chain rule)
#pragma unroll
            for (int a = 0; a < 4; ++a) {
                gx[a] = m[0][0] * gr[a][0] + m[1][0] * gr[a][1] + m[2][0] * gr[a][2];
                gy[a] = m[0][1] * gr[a][0] + m[1][1] * gr[a][1] + m[2][1] * gr[a][2];
                gz[a] = m[0][2] * gr[a][0] + m[1][2] * gr[a][1] + m[2][2] * gr[a][2];
            }
            const double T = w[0][H], u = w[1][H], v = w[2][H], ww = w[3][H];
            const double mu0 = fast_div_pos((1.0 + gs.suth) * (T * fast_sqrt_pos(T)), T + gs.suth);  // eq. 15
            const double mu = mu0 * gs.invRe, kc = mu0 * gs.kfac;              // eq. 14
            const double div = gx[1] + gy[2] + gz[3];
            const double txx = mu * (2.0 * gx[1] - (2.0 / 3.0) * div);         // eq. 13
            const double tyy = mu * (2.0 * gy[2] - (2.0 / 3.0) * div);
            const double tzz = mu * (2.0 * gz[3] - (2.0 / 3.0) * div);
            const double txy = mu * (gy[1] + gx[2]), txz = mu * (gz[1] + gx[3]), tyz = mu * (gz[2] + gy[3]);
            const double thx = u * txx + v * txy + ww * txz + kc * gx[0];      // eq. 12 (R-2)
            const double thy = u * txy + v * tyy + ww * tyz + kc * gy[0];
            const double thz = u * txz + v * tyz + ww * tzz + kc * gz[0];
            // periodic image of this point beyond the faces of each direction's own axis: +1 / -1 period, 0 = none
            const int imz = !g.periodic[2] ? 0 : k < H ? 1 : k >= g.nz - H ? -1 : 0;
            const int ims[3] = {imx, imy, imz};
            const long long period[3] = {g.nx, (long long)g.ny * g.sy, (long long)g.nz * g.sz};
            double *F = Fp;                                                     // field 4 d of this point
#pragma unroll
            for (int d = 0; d < 3; ++d, F += 4 * g.np) {                        // eq. 9-11
                const double dx = m[d][0] * iJ, dy = m[d][1] * iJ, dz = m[d][2] * iJ;
                const double f0 = dx * txx + dy * txy + dz * txz, f1 = dx * txy + dy * tyy + dz * tyz;
                const double f2 = dx * txz + dy * tyz + dz * tzz, f3 = dx * thx + dy * thy + dz * thz;
                __stcs(F, f0); __stcs(F + g.np, f1); __stcs(F + 2 * g.np, f2); __stcs(F + 3 * g.np, f3);
                if (ims[d] != 0) {
                    double *G = F + (ims[d] > 0 ? period[d] : -period[d]);
                    G[0] = f0; G[g.np] = f1; G[2 * g.np] = f2; G[3 * g.np] = f3;
                }
            }
        }
        // the plane after the newest one of the window: convert it now, so that ONE barrier per plane both publishes it
        // and releases the stage of plane k
        if (k + H + 1 <= last) {
            const int sc = (k + H + 1 - k0) % VF_NST;
            tma::mbar_wait(&bars[sc], ((k + H + 1 - k0) / VF_NST) & 1);
            convert_plane<ORDER>(gs, ring + sc * VF_STAGE, slots);
        }
        tma::fence_proxy_async();   // generic writes of convert_plane before the async-proxy refill of a stage
        __syncthreads();
        if (tid == 0 && k + VF_NST <= last) issue(k + VF_NST);
    }
}

// ------------------------------------------------------------------------------------------------ a7 (+ a8)
// RK: 0 = plain accumulate into dU (ocfd_rhs); 1..3 = also apply RK3 stage RK-1 (eq. 45) to U, dU is not written.
// One stage holds, for plane k: F with x halos, G with y halos, dU, U, U^n of the tile, and H of plane k+3.
constexpr int VD_NST = 3;
constexpr int VD_F = 4 * TY * BXW, VD_H = 4 * TY * TX, VD_C = 5 * TY * TX;
template <int ORDER>
struct VD {
    static constexpr int G = 4 * VG<ORDER>::BYH * TX;
    static constexpr int STAGE = VD_F + G + VD_H + 3 * VD_C;
    static constexpr size_t SMEM = sizeof(double) * VD_NST * STAGE + 8 * VD_NST;
    static_assert((VD_F * 8) % 128 == 0 && (G * 8) % 128 == 0 && (VD_H * 8) % 128 == 0 && (VD_C * 8) % 128 == 0 &&
                  (STAGE * 8) % 128 == 0, "TMA destinations must stay 128-byte aligned");
};

template <int KIND, int RK, int ORDER>
__global__ void __launch_bounds__(VNT, 1)
    k_viscous_div(const GridDesc g, const __grid_constant__ CUtensorMap tm_F, const __grid_constant__ CUtensorMap tm_G,
                  const __grid_constant__ CUtensorMap tm_H, const __grid_constant__ CUtensorMap tm_dU,
                  const __grid_constant__ CUtensorMap tm_U, const __grid_constant__ CUtensorMap tm_Un,
                  const double *__restrict__ Fv, double *__restrict__ dU, double *Uout, double dt, int zchunk,
                  int tgroup) {
    constexpr int HH = VG<ORDER>::H, BYH = VG<ORDER>::BYH, VD_G = VD<ORDER>::G, VD_STAGE = VD<ORDER>::STAGE;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *ring = reinterpret_cast<double *>(smem_raw);
    uint64_t *bars = reinterpret_cast<uint64_t *>(ring + VD_NST * VD_STAGE);
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * TX + tx;
    int tbx, tby;
    tile_of_block(tgroup, tbx, tby);
    const int i0 = tbx * TX, j0 = tby * TY;
    const int i = i0 + tx, j = j0 + ty;
    const bool own = i < g.nx && j < g.ny;
    const int k0 = blockIdx.z * zchunk, k1 = min(k0 + zchunk, g.nz);
    constexpr bool LD_U = RK != 0, LD_UN = RK >= 2;
    constexpr uint32_t BYTES = 8u * (VD_F + VD_G + VD_H + VD_C + (LD_U ? VD_C : 0) + (LD_UN ? VD_C : 0));
    auto issue = [&](int k) {
        const int s = (k - k0) % VD_NST;
        double *b = ring + s * VD_STAGE;
        const int xp = i0 + OCFD_NG, yp = j0 + OCFD_NG, kp = k + OCFD_NG;
        tma::mbar_expect_tx(&bars[s], BYTES);
        // (plain loads: L2 eviction hints on these boxes were measured and cost 10 %, profiles/r01_c)
        tma::load4(b, &tm_F, &bars[s], xp - 4, yp, kp, 0);
        tma::load4(b + VD_F, &tm_G, &bars[s], xp, yp - HH, kp, 4);
        tma::load4(b + VD_F + VD_G, &tm_H, &bars[s], xp, yp, kp + HH, 8);
        tma::load4(b + VD_F + VD_G + VD_H, &tm_dU, &bars[s], xp, yp, kp, 0);
        if (LD_U) tma::load4(b + VD_F + VD_G + VD_H + VD_C, &tm_U, &bars[s], xp, yp, kp, 0);
        if (LD_UN) tma::load4(b + VD_F + VD_G + VD_H + 2 * VD_C, &tm_Un, &bars[s], xp, yp, kp, 0);
    };
    if (tid == 0) {
        for (int s = 0; s < VD_NST; ++s) tma::mbar_init(&bars[s], 1);
        tma::fence_barrier_init();
        for (int q = 0; q < VD_NST; ++q)
            if (k0 + q < k1) issue(k0 + q);
    }
    // z window of the zeta-direction flux H: planes k-H .. k+H-1 from global memory, plane k+H arrives with stage k
    const int ipc = min(i, g.nx - 1) + OCFD_NG, jpc = min(j, g.ny - 1) + OCFD_NG;
    const long long col = (long long)jpc * g.sy + ipc;
    const double *H = Fv + 8 * g.np;
    double w[4][2 * HH + 1];
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int q = 0; q < 2 * HH; ++q) w[r][q + 1] = __ldg(H + r * g.np + (long long)(k0 - HH + q + OCFD_NG) * g.sz + col);
    __syncthreads();  // barriers initialised
    const int ctr = ty * TX + tx;
    for (int k = k0; k < k1; ++k) {
        const int s = (k - k0) % VD_NST;
        const double *b = ring + s * VD_STAGE;
        tma::mbar_wait(&bars[s], ((k - k0) / VD_NST) & 1);
#pragma unroll
        for (int r = 0; r < 4; ++r) {
#pragma unroll
            for (int q = 0; q < 2 * HH; ++q) w[r][q] = w[r][q + 1];
            w[r][2 * HH] = b[VD_F + VD_G + r * TY * TX + ctr];
        }
        if (own) {
            const int ip = i + OCFD_NG, jp = j + OCFD_NG, kp = k + OCFD_NG;
            const long long id = (long long)kp * g.sz + (long long)jp * g.sy + ip;
            const double J = Met<KIND>::J(g, ip, jp, kp);
            const double *sdU = b + VD_F + VD_G + VD_H, *sU = sdU + VD_C, *sUn = sU + VD_C;
            double acc[5];
            acc[0] = sdU[ctr];
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                double sum = d1_line<ORDER>(b + (r * TY + ty) * BXW + tx + 4, 1, i, g.nx, g.periodic[0]);
                sum += d1_line<ORDER>(b + VD_F + (r * BYH + ty + HH) * TX + tx, TX, j, g.ny, g.periodic[1]);
                sum += d1_win<ORDER>(w[r], k, g.nz, g.periodic[2]);
                acc[r + 1] = sdU[(r + 1) * TY * TX + ctr] + J * sum;
            }
            if (RK == 0) {
#pragma unroll
                for (int r = 1; r < 5; ++r) dU[r * g.np + id] = acc[r];
            } else {
#pragma unroll
                for (int m = 0; m < 5; ++m) {
                    const long long q = m * g.np + id;
                    const double u = sU[m * TY * TX + ctr];
                    // (Uout may be the buffer tm_U or tm_Un reads: the boxes of this plane have landed, and no other
                    // CTA reads these points)
                    if (RK == 1) {
                        __stcs(Uout + q, u + dt * acc[m]);
                    } else if (RK == 2) {
                        __stcs(Uout + q, 0.75 * sUn[m * TY * TX + ctr] + 0.25 * (u + dt * acc[m]));
                    } else {
                        __stcs(Uout + q, (1.0 / 3.0) * sUn[m * TY * TX + ctr] + (2.0 / 3.0) * (u + dt * acc[m]));
                    }
                }
            }
        }
        __syncthreads();  // stage s is free again
        if (tid == 0 && k + VD_NST < k1) issue(k + VD_NST);
    }
}

// width of the column groups of tile_of_block: 16 tiles (512 points of x), "tile_group" of ocfd_set_tuning overrides
int tile_group(const ocfd_ctx *c, unsigned nxt) {
    int gw = c->tune.tile_group > 0 ? c->tune.tile_group : 16;
    if (gw > (int)nxt) gw = (int)nxt;
    return gw;
}

int pick_zchunk(const ocfd_ctx *c, int pass) {
    const GridDesc &g = c->g;
    // enough blocks to fill the SMs a few times over ...
    const long long tiles = (long long)((g.nx + TX - 1) / TX) * ((g.ny + TY - 1) / TY);
    int zc = g.nz;
    while (zc > 32 && tiles * ((g.nz + zc - 1) / zc) < c->nsm * 8) zc = (zc + 1) / 2;
    // ... and short enough that tiles which share a halo stay close in z: CTAs drift apart while they march, and a
    // halo plane the neighbour read long ago has left the L2.  Measured on config 5 (profiles/r01_c): chunks of 64
    // planes for pass 1 (4.94 -> 4.73 ms) and 32 for pass 2 (7.99 -> 7.02 ms); the prologue planes of a chunk come from L2.
    const int cap = pass == 1 ? 64 : 32;
    if (zc > cap) zc = cap;
    const int v = pass == 1 ? c->tune.zchunk_f : c->tune.zchunk_d;   // ocfd_set_tuning (A/B runs)
    if (v >= 8) zc = v < g.nz ? v : g.nz;
    return zc;
}

// tensor maps of pass 1 (U boxes with x-y halos) and of pass 2
bool encode_flux_map(ocfd_ctx *c, const double *U) {
    const GridDesc &g = c->g;
    ViscMaps &M = c->visc;
    if (M.Ufp == U) return true;
    const long long d5[4] = {g.nxp, g.nyp, g.nzp, 5};
    const int bp[4] = {BXW, TY + c->visc_order, 1, 5};   // TY + 2 H rows
    if (!ocfd_tma_encode(&M.Uf, U, d5, g.sy, g.sz, g.np, bp)) return false;
    M.Ufp = U;
    return true;
}

// M.Un describes the context's second state buffer, M.U the caller's U (re-encoded when the pointer changes)
bool encode_div_maps(ocfd_ctx *c, const double *dU, const double *U) {
    const GridDesc &g = c->g;
    ViscMaps &M = c->visc;
    const long long d12[4] = {g.nxp, g.nyp, g.nzp, 12}, d5[4] = {g.nxp, g.nyp, g.nzp, 5};
    const int BYH = TY + c->visc_order;   // TY + 2 H
    const int bF[4] = {BXW, TY, 1, 4}, bG[4] = {TX, BYH, 1, 4}, bH[4] = {TX, TY, 1, 4};
    const int bC[4] = {TX, TY, 1, 5};
    if (!M.ready) {
        if (!ocfd_tma_encode(&M.F, c->Fv, d12, g.sy, g.sz, g.np, bF)) return false;
        if (!ocfd_tma_encode(&M.G, c->Fv, d12, g.sy, g.sz, g.np, bG)) return false;
        if (!ocfd_tma_encode(&M.H, c->Fv, d12, g.sy, g.sz, g.np, bH)) return false;
        if (!ocfd_tma_encode(&M.Un, c->Un, d5, g.sy, g.sz, g.np, bC)) return false;
        M.ready = true;
    }
    if (M.dUp != dU) {
        if (!ocfd_tma_encode(&M.dU, dU, d5, g.sy, g.sz, g.np, bC)) return false;
        M.dUp = dU;
    }
    if (U && M.Up != U) {
        if (!ocfd_tma_encode(&M.U, U, d5, g.sy, g.sz, g.np, bC)) return false;
        M.Up = U;
    }
    return true;
}

template <int KIND, int RK, int ORDER>
ocfd_status launch_div(ocfd_ctx *c, dim3 grd, dim3 blk, double *dU, const RkBufs &rk, double dt, int zc) {
    if (!ocfd_smem_optin(c, (const void *)k_viscous_div<KIND, RK, ORDER>, VD<ORDER>::SMEM)) return OCFD_ECUDA;
    const ViscMaps &M = c->visc;
    auto map_of = [&](const double *p) -> const CUtensorMap & { return p == c->Un ? M.Un : M.U; };
    k_viscous_div<KIND, RK, ORDER><<<grd, blk, VD<ORDER>::SMEM, c->stream>>>(
        c->g, M.F, M.G, M.H, M.dU, RK ? map_of(rk.Uin) : M.dU, RK >= 2 ? map_of(rk.Un) : M.dU, c->Fv, dU, rk.out, dt, zc,
        tile_group(c, grd.x));
    return OCFD_OK;
}

template <int KIND, int ORDER>
ocfd_status launch_div_kind(ocfd_ctx *c, double *dU, const RkBufs &rk, double dt, int rk_stage) {
    const GridDesc &g = c->g;
    // the caller's U is whichever of the stage's buffers is not the context's own
    const double *user = rk_stage < 0 ? nullptr : rk.Uin != c->Un ? rk.Uin : rk.Un;
    if (!encode_div_maps(c, dU, user)) return OCFD_ECUDA;
    const int zcd = pick_zchunk(c, 2);
    dim3 blk(TX, TY, 1), grdd((g.nx + TX - 1) / TX, (g.ny + TY - 1) / TY, (g.nz + zcd - 1) / zcd);
    OCFD_T0(c, K_VISC_DIV);
    ocfd_status st;
    switch (rk_stage) {
        case 0: st = launch_div<KIND, 1, ORDER>(c, grdd, blk, dU, rk, dt, zcd); break;
        case 1: st = launch_div<KIND, 2, ORDER>(c, grdd, blk, dU, rk, dt, zcd); break;
        case 2: st = launch_div<KIND, 3, ORDER>(c, grdd, blk, dU, rk, dt, zcd); break;
        default: st = launch_div<KIND, 0, ORDER>(c, grdd, blk, dU, rk, 0.0, zcd);
    }
    if (st != OCFD_OK) return st;
    OCFD_CHECK_LAUNCH(c);
    return OCFD_OK;
}

template <int KIND, int ORDER, bool SENSOR>
ocfd_status launch_flux(ocfd_ctx *c, const double *U) {
    const GridDesc &g = c->g;
    if (!encode_flux_map(c, U)) return OCFD_ECUDA;
    if (!ocfd_smem_optin(c, (const void *)k_viscous_flux<KIND, ORDER, SENSOR>, VF<ORDER>::SMEM)) return OCFD_ECUDA;
    const int zc = pick_zchunk(c, 1);
    dim3 blk(TX, TY, 1), grd((g.nx + TX - 1) / TX, (g.ny + TY - 1) / TY, (g.nz + zc - 1) / zc);
    OCFD_T0(c, K_VISC_FLUX);
    k_viscous_flux<KIND, ORDER, SENSOR><<<grd, blk, VF<ORDER>::SMEM, c->stream>>>(g, c->gas, c->visc.Uf, U, c->Fv, c->theta, zc,
                                                                                  tile_group(c, grd.x));
    OCFD_CHECK_LAUNCH(c);
    return OCFD_OK;
}

template <int KIND, int ORDER>
ocfd_status launch_flux_kind(ocfd_ctx *c, const double *U, bool sensor) {
    return sensor ? launch_flux<KIND, ORDER, true>(c, U) : launch_flux<KIND, ORDER, false>(c, U);
}

}  // namespace

// Pass 1 (a6): Fv <- viscous fluxes of U; with `sensor` also theta <- shock sensor of U (a3).  Depends on U only.
ocfd_status launch_viscous_flux(ocfd_ctx *c, const double *U, bool sensor) {
    if (c->visc_order == 8) {
        switch (c->g.kind) {
            case OCFD_GRID_UNIFORM: return launch_flux_kind<OCFD_GRID_UNIFORM, 8>(c, U, sensor);
            case OCFD_GRID_STRETCHED: return launch_flux_kind<OCFD_GRID_STRETCHED, 8>(c, U, sensor);
            default: return launch_flux_kind<OCFD_GRID_CURVILINEAR, 8>(c, U, sensor);
        }
    }
    switch (c->g.kind) {
        case OCFD_GRID_UNIFORM: return launch_flux_kind<OCFD_GRID_UNIFORM, 6>(c, U, sensor);
        case OCFD_GRID_STRETCHED: return launch_flux_kind<OCFD_GRID_STRETCHED, 6>(c, U, sensor);
        default: return launch_flux_kind<OCFD_GRID_CURVILINEAR, 6>(c, U, sensor);
    }
}

// Pass 2 (a7): rk_stage < 0: dU += viscous terms.  rk_stage = 0,1,2: the same, then rk.out <- RK3 stage update (a8) in
// the same kernel.
ocfd_status launch_viscous_div(ocfd_ctx *c, double *dU, const RkBufs &rk, double dt, int rk_stage) {
    if (c->visc_order == 8) {
        switch (c->g.kind) {
            case OCFD_GRID_UNIFORM: return launch_div_kind<OCFD_GRID_UNIFORM, 8>(c, dU, rk, dt, rk_stage);
            case OCFD_GRID_STRETCHED: return launch_div_kind<OCFD_GRID_STRETCHED, 8>(c, dU, rk, dt, rk_stage);
            default: return launch_div_kind<OCFD_GRID_CURVILINEAR, 8>(c, dU, rk, dt, rk_stage);
        }
    }
    switch (c->g.kind) {
        case OCFD_GRID_UNIFORM: return launch_div_kind<OCFD_GRID_UNIFORM, 6>(c, dU, rk, dt, rk_stage);
        case OCFD_GRID_STRETCHED: return launch_div_kind<OCFD_GRID_STRETCHED, 6>(c, dU, rk, dt, rk_stage);
        default: return launch_div_kind<OCFD_GRID_CURVILINEAR, 6>(c, dU, rk, dt, rk_stage);
    }
}
