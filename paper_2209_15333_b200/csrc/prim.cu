// Rows a3 (shock sensor, stand-alone form) and a9 (max wavespeed); row a2 (primitives) lives inside its consumers.
#include "ocfd_internal.cuh"
#include "schemes.cuh"
#include "tma.cuh"


namespace {

// a3 (stand-alone form, for runs without viscous terms; with them the sensor is part of viscous pass 1, viscous.cu):
// theta = phi_i + phi_j + phi_k at interior points (eq. 42, R-11) and its first ghost layer (R-12).
// phi_d = |p_- - 2 p_0 + p_+| / (p_- + 2 p_0 + p_+); the three quotients share one division:
// theta = (n_i d_j d_k + n_j d_i d_k + n_k d_i d_j) / (d_i d_j d_k).
//
// 2.5-D marching kernel: a CTA owns an ST x SY tile in x-y and walks along z; every plane of U (with its 1-point x-y
// halo) is fetched once by a TMA box load into a ring of shared-memory stages that runs ahead of the arithmetic; the
// CTA turns each landed plane into p in place (row a2: no primitive field exists in HBM), so U is read once from HBM
// (40 B/point) and theta written once (8 B/point).
constexpr int ST = 32, SY = 8, SNT = ST * SY;
constexpr int SBX = ST + 4, SBY = SY + 2;          // box with halo; 2 wider in x on each side: a box of doubles starts at an even x
constexpr int S_FLD = SBX * SBY;                   // doubles per staged field
constexpr int S_NST = 4;                           // ring: planes k, k+1 live, k+2 being converted, one more in flight
constexpr int S_STAGE = (5 * S_FLD * 8 + 127) / 128 * 128 / 8;   // doubles per stage, 128-byte aligned
constexpr size_t S_SMEM = sizeof(double) * S_NST * S_STAGE + 8 * S_NST;

// p of the points of one staged plane of U, left in the slot of rho
__device__ __forceinline__ void pressure_plane(const GasDesc &gs, double *st, int tid) {
    for (int q = tid; q < S_FLD; q += SNT) {
        const double rho = st[q], ir = fast_rcp_pos(rho);
        const double u = st[S_FLD + q] * ir, v = st[2 * S_FLD + q] * ir, w = st[3 * S_FLD + q] * ir;
        st[q] = gs.gm1 * (st[4 * S_FLD + q] - 0.5 * rho * (u * u + v * v + w * w));
    }
}

__global__ void __launch_bounds__(SNT) k_sensor(GridDesc g, GasDesc gs, const __grid_constant__ CUtensorMap tm_U,
                                                const double *__restrict__ U, double *__restrict__ theta, int zchunk) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *ring = reinterpret_cast<double *>(smem_raw);
    uint64_t *bars = reinterpret_cast<uint64_t *>(ring + S_NST * S_STAGE);
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * ST + tx;
    const int i0 = blockIdx.x * ST, j0 = blockIdx.y * SY;
    const int i = i0 + tx, j = j0 + ty;
    const bool own = i < g.nx && j < g.ny;
    const int k0 = blockIdx.z * zchunk, k1 = min(k0 + zchunk, g.nz);
    const int last = k1;   // last plane needed (k1 - 1 + 1)
    auto issue = [&](int plane) {   // interior plane index -> stage (plane - k0) % S_NST
        const int s = (plane - k0) % S_NST;
        tma::mbar_expect_tx(&bars[s], 5 * S_FLD * 8);
        tma::load4(ring + s * S_STAGE, &tm_U, &bars[s], i0 + OCFD_NG - 2, j0 + OCFD_NG - 1, plane + OCFD_NG, 0);
    };
    if (tid == 0) {
        for (int s = 0; s < S_NST; ++s) tma::mbar_init(&bars[s], 1);
        tma::fence_barrier_init();
        for (int q = 0; q < S_NST; ++q)
            if (k0 + q <= last) issue(k0 + q);
    }
    // p of plane k0-1 at this thread's column, straight from global memory
    double pm;
    {
        const int ipc = min(i, g.nx - 1) + OCFD_NG, jpc = min(j, g.ny - 1) + OCFD_NG;
        const long long id = (long long)(k0 - 1 + OCFD_NG) * g.sz + (long long)jpc * g.sy + ipc;
        const double rho = __ldg(U + id), ir = fast_rcp_pos(rho);
        const double u = __ldg(U + g.np + id) * ir, v = __ldg(U + 2 * g.np + id) * ir, w = __ldg(U + 3 * g.np + id) * ir;
        pm = gs.gm1 * (__ldg(U + 4 * g.np + id) - 0.5 * rho * (u * u + v * v + w * w));
    }
    __syncthreads();   // barriers initialised
    for (int q = 0; q < 2; ++q) {   // planes k0, k0+1 (both exist: k0+1 <= k1)
        tma::mbar_wait(&bars[q], 0);
        pressure_plane(gs, ring + q * S_STAGE, tid);
    }
    // pressure_plane writes a TMA destination in place (generic proxy); the box load that later refills the stage goes
    // through the async proxy: every thread orders its writes before the barrier that lets tid 0 issue that load
    tma::fence_proxy_async();
    __syncthreads();
    const int ctr = (ty + 1) * SBX + tx + 2;
    for (int k = k0; k < k1; ++k) {
        const double *c = ring + ((k - k0) % S_NST) * S_STAGE + ctr;
        const double p0 = c[0], pp = ring[((k + 1 - k0) % S_NST) * S_STAGE + ctr];
        if (own) {
            const double t0 = p0 + p0;
            const double ni = fabs(t0 - c[-1] - c[1]), di = t0 + c[-1] + c[1];
            const double nj = fabs(t0 - c[-SBX] - c[SBX]), dj = t0 + c[-SBX] + c[SBX];
            const double nk = fabs(t0 - pm - pp), dk = t0 + pm + pp;
            const double dij = di * dj;
            const double th = fast_div_pos(ni * (dj * dk) + nj * (di * dk) + nk * dij, dij * dk);
            const long long id = pidx(g, i + OCFD_NG, j + OCFD_NG, k + OCFD_NG);
            theta[id] = th;
            const int cc[3] = {i, j, k};
            const int n[3] = {g.nx, g.ny, g.nz};
            const long long st[3] = {1, g.sy, g.sz};
            const bool face = i == 0 || j == 0 || k == 0 || i == g.nx - 1 || j == g.ny - 1 || k == g.nz - 1;
#pragma unroll
            for (int d = 0; d < 3 && face; ++d) {
                if (cc[d] == 0) theta[g.periodic[d] ? id + n[d] * st[d] : id - st[d]] = th;
                if (cc[d] == n[d] - 1) theta[g.periodic[d] ? id - n[d] * st[d] : id + st[d]] = th;
            }
        }
        pm = p0;
        if (k + 2 <= last) {   // the plane after next: turn it into p now, one barrier publishes it and frees plane k
            const int sc = (k + 2 - k0) % S_NST;
            tma::mbar_wait(&bars[sc], ((k + 2 - k0) / S_NST) & 1);
            pressure_plane(gs, ring + sc * S_STAGE, tid);
        }
        tma::fence_proxy_async();
        __syncthreads();
        if (tid == 0 && k + S_NST <= last) issue(k + S_NST);
    }
}

// per-interface scheme flags for the parity report (the inviscid kernels recompute them on the fly)
__global__ void k_flags(GridDesc g, GasDesc gs, int scheme, const double *__restrict__ theta, unsigned char *__restrict__ flags) {
    int ip = blockIdx.x * blockDim.x + threadIdx.x;
    int jp = blockIdx.y * blockDim.y + threadIdx.y;
    int kp = blockIdx.z;
    if (ip >= g.nxp || jp >= g.nyp) return;
    const int c[3] = {ip - OCFD_NG, jp - OCFD_NG, kp - OCFD_NG};
    const int n[3] = {g.nx, g.ny, g.nz};
    const long long s[3] = {1, g.sy, g.sz};
    long long id = pidx(g, ip, jp, kp);
    for (int d = 0; d < 3; ++d) {
        bool ok = true;
        for (int e = 0; e < 3; ++e) ok = ok && (e == d ? (c[e] >= -1 && c[e] < n[e]) : (c[e] >= 0 && c[e] < n[e]));
        unsigned char f = 255;
        if (ok) {
            if (scheme != OCFD_HYBRID) f = (unsigned char)scheme;
            else {
                double Th = fmax(theta[id], theta[id + s[d]]);
                f = Th <= gs.theta1 ? 0 : (Th <= gs.theta2 ? 1 : 2);
            }
        }
        flags[d * g.np + id] = f;
    }
}

// a9: Lambda = max sum_d (|d_x u + d_y v + d_z w| + c |grad d|) over interior points (R-17).
// A thread owns one (i, j) column and walks a chunk of z planes: coalesced along x, no index division per point, and on
// grids whose metrics do not depend on z (uniform; z-extruded curvilinear maps) the nine metric values and the three
// square roots |grad d| are fetched and formed once per column instead of once per point.
constexpr int WS_NT = 128;
template <int KIND>
__global__ void __launch_bounds__(WS_NT) k_wavespeed(GridDesc g, GasDesc gs, const double *__restrict__ U,
                                                     unsigned long long *__restrict__ out, int zchunk) {
    const int i = blockIdx.x * WS_NT + threadIdx.x, j = blockIdx.y;
    const int k0 = blockIdx.z * zchunk, k1 = min(k0 + zchunk, g.nz);
    double best = 0.0;
    bool bad = false;
    if (i < g.nx) {
        const int ip = i + OCFD_NG, jp = j + OCFD_NG;
        const bool fixed = KIND == OCFD_GRID_UNIFORM || (KIND == OCFD_GRID_CURVILINEAR && g.msk == 0);
        double a[3][3], len[3];
        auto fetch = [&](int kp) {
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                Met<KIND>::row(g, d, ip, jp, kp, a[d][0], a[d][1], a[d][2]);
                len[d] = sqrt(a[d][0] * a[d][0] + a[d][1] * a[d][1] + a[d][2] * a[d][2]);
            }
        };
        if (fixed) fetch(OCFD_NG);
        long long id = pidx(g, ip, jp, k0 + OCFD_NG);
        // seeded reciprocal and square root (schemes.cuh: within an ulp or two; a NaN, zero or negative argument still
        // ends as a non-finite s): the library 1/x and sqrt were half of this kernel's instructions; two planes per
        // trip keep ten loads in flight per thread
#pragma unroll 2
        for (int k = k0; k < k1; ++k, id += g.sz) {
            if (!fixed) fetch(k + OCFD_NG);
            const double rho = __ldcs(U + id), ir = fast_rcp_pos(rho);
            const double u = __ldcs(U + g.np + id) * ir, v = __ldcs(U + 2 * g.np + id) * ir, w = __ldcs(U + 3 * g.np + id) * ir;
            const double p = gs.gm1 * (__ldcs(U + 4 * g.np + id) - 0.5 * rho * (u * u + v * v + w * w));
            const double c = fast_sqrt_pos(gs.gM2 * p * ir) * gs.invMa;
            double s = 0.0;
#pragma unroll
            for (int d = 0; d < 3; ++d) s += fabs(a[d][0] * u + a[d][1] * v + a[d][2] * w) + c * len[d];
            // fmax drops a NaN operand: a blown-up state (NaN rho or p) must not come back as a finite Lambda
            bad |= !(s == s);
            best = fmax(best, s);
        }
    }
    // warp-shuffle max, then one atomic per warp on the ordered bit pattern (all values are >= 0; the quiet-NaN
    // pattern orders above +inf, so one bad point makes the result NaN)
    for (int o = 16; o > 0; o >>= 1) best = fmax(best, __shfl_xor_sync(0xffffffffu, best, o));
    bad = __any_sync(0xffffffffu, bad);
    if ((threadIdx.x & 31) == 0)
        atomicMax(out, bad ? 0x7ff8000000000000ull : (unsigned long long)__double_as_longlong(best));
}

// State guard: counts of interior points with a non-finite conserved variable, with rho <= 0, with p <= 0 (p looked at
// only where the five values are finite and rho > 0).  Same launch shape as the wavespeed march: one (i, j) column per
// thread, coalesced along x, 40 B/point read once.  Integer counts: warp-reduced, then one atomic per warp and counter.
__global__ void __launch_bounds__(WS_NT) k_check_state(GridDesc g, GasDesc gs, const double *__restrict__ U,
                                                       unsigned long long *__restrict__ counts, int zchunk) {
    const int i = blockIdx.x * WS_NT + threadIdx.x, j = blockIdx.y;
    const int k0 = blockIdx.z * zchunk, k1 = min(k0 + zchunk, g.nz);
    unsigned int n_nonfinite = 0, n_rho = 0, n_p = 0;
    if (i < g.nx) {
        long long id = pidx(g, i + OCFD_NG, j + OCFD_NG, k0 + OCFD_NG);
        for (int k = k0; k < k1; ++k, id += g.sz) {
            const double rho = U[id], m1 = U[g.np + id], m2 = U[2 * g.np + id], m3 = U[3 * g.np + id], E = U[4 * g.np + id];
            const bool finite = isfinite(rho) && isfinite(m1) && isfinite(m2) && isfinite(m3) && isfinite(E);
            n_nonfinite += !finite;
            n_rho += rho <= 0.0;
            if (finite && rho > 0.0) {
                const double u = m1 / rho, v = m2 / rho, w = m3 / rho;
                n_p += gs.gm1 * (E - 0.5 * rho * (u * u + v * v + w * w)) <= 0.0;
            }
        }
    }
    n_nonfinite = __reduce_add_sync(0xffffffffu, n_nonfinite);
    n_rho = __reduce_add_sync(0xffffffffu, n_rho);
    n_p = __reduce_add_sync(0xffffffffu, n_p);
    if ((threadIdx.x & 31) == 0) {
        if (n_nonfinite) atomicAdd(counts, (unsigned long long)n_nonfinite);
        if (n_rho) atomicAdd(counts + 1, (unsigned long long)n_rho);
        if (n_p) atomicAdd(counts + 2, (unsigned long long)n_p);
    }
}

}  // namespace

ocfd_status launch_sensor(ocfd_ctx *c, const double *U) {
    const GridDesc &g = c->g;
    if (c->sens_U != U) {
        const long long d5[4] = {g.nxp, g.nyp, g.nzp, 5};
        const int bx[4] = {SBX, SBY, 1, 5};
        if (!ocfd_tma_encode(&c->sens_map, U, d5, g.sy, g.sz, g.np, bx)) return OCFD_ECUDA;
        c->sens_U = U;
    }
    if (!ocfd_smem_optin(c, (const void *)k_sensor, S_SMEM)) return OCFD_ECUDA;
    // enough blocks to fill the SMs a few times over, chunks long enough that the prologue planes stay cheap
    const long long tiles = (long long)((g.nx + ST - 1) / ST) * ((g.ny + SY - 1) / SY);
    int zc = g.nz;
    while (zc > 32 && tiles * ((g.nz + zc - 1) / zc) < c->nsm * 16) zc = (zc + 1) / 2;
    if (zc > 64) zc = 64;   // short marches keep halo-sharing tiles close in z (as in the viscous kernels)
    if (c->tune.zchunk_s >= 8) zc = c->tune.zchunk_s < g.nz ? c->tune.zchunk_s : g.nz;
    dim3 blk(ST, SY, 1), grd((g.nx + ST - 1) / ST, (g.ny + SY - 1) / SY, (g.nz + zc - 1) / zc);
    OCFD_T0(c, K_SENSOR);
    k_sensor<<<grd, blk, S_SMEM, c->stream>>>(g, c->gas, c->sens_map, U, c->theta, zc);
    OCFD_CHECK_LAUNCH(c);
    return OCFD_OK;
}

ocfd_status launch_flags(ocfd_ctx *c, unsigned char *flags) {
    const GridDesc &g = c->g;
    dim3 blk(32, 8, 1), grd((g.nxp + 31) / 32, (g.nyp + 7) / 8, g.nzp);
    OCFD_T0(c, K_SENSOR);
    k_flags<<<grd, blk, 0, c->stream>>>(g, c->gas, (int)c->p.scheme, c->theta, flags);
    OCFD_CHECK_LAUNCH(c);
    return OCFD_OK;
}

ocfd_status launch_wavespeed(ocfd_ctx *c, const double *U, double *host_out) {
    const GridDesc &g = c->g;
    unsigned long long *out = (unsigned long long *)c->scal;
    if (cudaMemsetAsync(out, 0, sizeof(unsigned long long), c->stream) != cudaSuccess) return OCFD_ECUDA;
    if (g.ny > 65535) return OCFD_EINVAL;
    // z chunks: long enough to amortise the per-column metric work, short enough to fill the SMs a few times over
    int zc = g.nz;
    const long long cols = (long long)((g.nx + WS_NT - 1) / WS_NT) * g.ny;
    while (zc > 32 && cols * ((g.nz + zc - 1) / zc) < 8ll * c->nsm) zc = (zc + 1) / 2;
    if (zc > 64) zc = 64;
    const dim3 grd((g.nx + WS_NT - 1) / WS_NT, g.ny, (g.nz + zc - 1) / zc);
    OCFD_T0(c, K_WAVE);
    switch (g.kind) {
        case OCFD_GRID_UNIFORM: k_wavespeed<OCFD_GRID_UNIFORM><<<grd, WS_NT, 0, c->stream>>>(g, c->gas, U, out, zc); break;
        case OCFD_GRID_STRETCHED: k_wavespeed<OCFD_GRID_STRETCHED><<<grd, WS_NT, 0, c->stream>>>(g, c->gas, U, out, zc); break;
        default: k_wavespeed<OCFD_GRID_CURVILINEAR><<<grd, WS_NT, 0, c->stream>>>(g, c->gas, U, out, zc);
    }
    OCFD_CHECK_LAUNCH(c);
    if (cudaMemcpyAsync(host_out, out, sizeof(double), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) return OCFD_ECUDA;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return OCFD_ECUDA;
    return OCFD_OK;
}

ocfd_status launch_check_state(ocfd_ctx *c, const double *U, long long *host_counts) {
    const GridDesc &g = c->g;
    unsigned long long *cnt = (unsigned long long *)c->scal + 1;   // word 0 of the scalar area is the wavespeed result
    if (g.ny > 65535) return OCFD_EINVAL;
    if (cudaMemsetAsync(cnt, 0, 3 * sizeof(unsigned long long), c->stream) != cudaSuccess) return OCFD_ECUDA;
    int zc = g.nz;
    const long long cols = (long long)((g.nx + WS_NT - 1) / WS_NT) * g.ny;
    while (zc > 32 && cols * ((g.nz + zc - 1) / zc) < 8ll * c->nsm) zc = (zc + 1) / 2;
    if (zc > 64) zc = 64;
    const dim3 grd((g.nx + WS_NT - 1) / WS_NT, g.ny, (g.nz + zc - 1) / zc);
    OCFD_T0(c, K_CHECK);
    k_check_state<<<grd, WS_NT, 0, c->stream>>>(g, c->gas, U, cnt, zc);
    OCFD_CHECK_LAUNCH(c);
    if (cudaMemcpyAsync(host_counts, cnt, 3 * sizeof(long long), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess)
        return OCFD_ECUDA;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return OCFD_ECUDA;
    return OCFD_OK;
}
