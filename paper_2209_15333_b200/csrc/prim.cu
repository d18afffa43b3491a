// Rows a2 (primitives), a3 (shock sensor) and a9 (max wavespeed).
#include "ocfd_internal.cuh"

namespace {

// a2: u,v,w,T,c,p at every padded point (eq. 8 as corrected, eq. 16).  Edge / corner ghosts
// hold whatever the caller left there; their primitives are computed but never read.
__global__ void __launch_bounds__(256) k_prim(long long np, GasDesc gs, const double *__restrict__ U,
                                              double *__restrict__ prim) {
    long long stride = (long long)gridDim.x * blockDim.x;
    for (long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x; id < np; id += stride) {
        // true divisions (not a reciprocal multiply): this kernel is HBM-bound, and the pressure that feeds
        // the shock-sensor decisions then rounds exactly as the definition does
        double rho = U[id];
        double u = U[np + id] / rho, v = U[2 * np + id] / rho, w = U[3 * np + id] / rho;
        double p = gs.gm1 * (U[4 * np + id] - 0.5 * rho * (u * u + v * v + w * w));
        double T = gs.gM2 * p / rho;
        prim[P_U * np + id] = u;
        prim[P_V * np + id] = v;
        prim[P_W * np + id] = w;
        prim[P_T * np + id] = T;
        prim[P_C * np + id] = sqrt(T) * gs.invMa;
        prim[P_P * np + id] = p;
    }
}

__device__ __forceinline__ double phi_of(double pm, double p0, double pp) {
    return fabs(-pm + 2.0 * p0 - pp) / (pm + 2.0 * p0 + pp);  // eq. 42
}

// a3: theta = phi_i + phi_j + phi_k at interior points (eq. 42, R-11) and its first ghost layer (R-12)
__global__ void __launch_bounds__(256) k_sensor(GridDesc g, const double *__restrict__ p, double *__restrict__ theta) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    int j = blockIdx.y * blockDim.y + threadIdx.y;
    int k = blockIdx.z * blockDim.z + threadIdx.z;
    if (i >= g.nx || j >= g.ny || k >= g.nz) return;
    long long id = pidx(g, i + OCFD_NG, j + OCFD_NG, k + OCFD_NG);
    double p0 = p[id];
    double th = phi_of(p[id - 1], p0, p[id + 1]);
    th += phi_of(p[id - g.sy], p0, p[id + g.sy]);
    th += phi_of(p[id - g.sz], p0, p[id + g.sz]);
    theta[id] = th;
    const int c[3] = {i, j, k};
    const int n[3] = {g.nx, g.ny, g.nz};
    const long long s[3] = {1, g.sy, g.sz};
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        if (c[d] == 0) theta[g.periodic[d] ? id + n[d] * s[d] : id - s[d]] = th;
        if (c[d] == n[d] - 1) theta[g.periodic[d] ? id - n[d] * s[d] : id + s[d]] = th;
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

// a9: Lambda = max sum_d (|d_x u + d_y v + d_z w| + c |grad d|) over interior points (R-17)
template <int KIND>
__global__ void __launch_bounds__(256) k_wavespeed(GridDesc g, GasDesc gs, const double *__restrict__ U,
                                                   unsigned long long *__restrict__ out) {
    long long n = (long long)g.nx * g.ny * g.nz;
    long long stride = (long long)gridDim.x * blockDim.x;
    double best = 0.0;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += stride) {
        int i = (int)(q % g.nx), j = (int)((q / g.nx) % g.ny), k = (int)(q / ((long long)g.nx * g.ny));
        int ip = i + OCFD_NG, jp = j + OCFD_NG, kp = k + OCFD_NG;
        long long id = pidx(g, ip, jp, kp);
        double rho = U[id], ir = 1.0 / rho;
        double u = U[g.np + id] * ir, v = U[2 * g.np + id] * ir, w = U[3 * g.np + id] * ir;
        double p = gs.gm1 * (U[4 * g.np + id] - 0.5 * rho * (u * u + v * v + w * w));
        double c = sqrt(gs.gM2 * p * ir) * gs.invMa;
        double s = 0.0;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            double a1, a2, a3;
            Met<KIND>::row(g, d, ip, jp, kp, a1, a2, a3);
            s += fabs(a1 * u + a2 * v + a3 * w) + c * sqrt(a1 * a1 + a2 * a2 + a3 * a3);
        }
        best = fmax(best, s);
    }
    // warp-shuffle max, then one atomic per warp on the ordered bit pattern (all values are >= 0)
    for (int o = 16; o > 0; o >>= 1) best = fmax(best, __shfl_xor_sync(0xffffffffu, best, o));
    if ((threadIdx.x & 31) == 0) atomicMax(out, (unsigned long long)__double_as_longlong(best));
}

}  // namespace

ocfd_status launch_prim(ocfd_ctx *c, const double *U) {
    long long np = c->g.np;
    int blocks = (int)((np + 255) / 256);
    if (blocks > 148 * 32) blocks = 148 * 32;
    OCFD_T0(c, K_PRIM);
    k_prim<<<blocks, 256, 0, c->stream>>>(np, c->gas, U, c->prim);
    OCFD_CHECK_LAUNCH(c);
    return OCFD_OK;
}

ocfd_status launch_sensor(ocfd_ctx *c, const double *U) {
    (void)U;
    const GridDesc &g = c->g;
    dim3 blk(32, 4, 2), grd((g.nx + 31) / 32, (g.ny + 3) / 4, (g.nz + 1) / 2);
    OCFD_T0(c, K_SENSOR);
    k_sensor<<<grd, blk, 0, c->stream>>>(g, c->prim + (long long)P_P * g.np, c->theta);
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
    long long n = (long long)g.nx * g.ny * g.nz;
    int blocks = (int)((n + 255) / 256);
    if (blocks > 148 * 16) blocks = 148 * 16;
    OCFD_T0(c, K_WAVE);
    switch (g.kind) {
        case OCFD_GRID_UNIFORM: k_wavespeed<OCFD_GRID_UNIFORM><<<blocks, 256, 0, c->stream>>>(g, c->gas, U, out); break;
        case OCFD_GRID_STRETCHED: k_wavespeed<OCFD_GRID_STRETCHED><<<blocks, 256, 0, c->stream>>>(g, c->gas, U, out); break;
        default: k_wavespeed<OCFD_GRID_CURVILINEAR><<<blocks, 256, 0, c->stream>>>(g, c->gas, U, out);
    }
    OCFD_CHECK_LAUNCH(c);
    if (cudaMemcpyAsync(host_out, out, sizeof(double), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) return OCFD_ECUDA;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return OCFD_ECUDA;
    return OCFD_OK;
}
