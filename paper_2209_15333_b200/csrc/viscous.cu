// Rows a6 + a7: viscous and heat-flux terms (eq. 9-15) by the 6th-order central first
// derivative applied twice (DESIGN R-15): pass 1 forms the viscous fluxes at interior points,
// pass 2 differences them and accumulates into dU.
#include "ocfd_internal.cuh"

namespace {

__device__ __forceinline__ double d1_int(const double *__restrict__ f, long long st) {
    return (45.0 * (f[st] - f[-st]) - 9.0 * (f[2 * st] - f[-2 * st]) + (f[3 * st] - f[-3 * st])) * (1.0 / 60.0);
}
// closure rows of an aperiodic axis; f points at element s of a line of n
__device__ __forceinline__ double d1_closure(const double *__restrict__ f, long long st, int s, int n) {
    if (s == 0) return (-3.0 * f[0] + 4.0 * f[st] - f[2 * st]) * 0.5;
    if (s == n - 1) return (3.0 * f[0] - 4.0 * f[-st] + f[-2 * st]) * 0.5;
    if (s == 1 || s == n - 2) return (f[st] - f[-st]) * 0.5;
    if (s == 2 || s == n - 3) return (8.0 * (f[st] - f[-st]) - (f[2 * st] - f[-2 * st])) * (1.0 / 12.0);
    return d1_int(f, st);
}
// pass 1: periodic axes read the (valid) ghost values of the primitives
__device__ __forceinline__ double d1_ghost(const double *__restrict__ f, long long st, int s, int n, int periodic) {
    if (periodic || (s >= 3 && s <= n - 4)) return d1_int(f, st);
    return d1_closure(f, st, s, n);
}
// pass 2: the fluxes exist at interior points only; periodic axes wrap the index
__device__ __forceinline__ double d1_wrap(const double *__restrict__ f, long long st, int s, int n, int periodic) {
    if (s >= 3 && s <= n - 4) return d1_int(f, st);
    if (!periodic) return d1_closure(f, st, s, n);
    double v[7];
#pragma unroll
    for (int o = -3; o <= 3; ++o) {
        int q = s + o;
        q = q < 0 ? q + n : (q >= n ? q - n : q);
        v[o + 3] = f[(long long)(q - s) * st];
    }
    return (45.0 * (v[4] - v[2]) - 9.0 * (v[5] - v[1]) + (v[6] - v[0])) * (1.0 / 60.0);
}

// a6
template <int KIND>
__global__ void __launch_bounds__(256) k_viscous_flux(GridDesc g, GasDesc gs, const double *__restrict__ prim,
                                                      double *__restrict__ Fv) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z * blockDim.z + threadIdx.z;
    if (i >= g.nx || j >= g.ny || k >= g.nz) return;
    const int ip = i + OCFD_NG, jp = j + OCFD_NG, kp = k + OCFD_NG;
    const long long id = pidx(g, ip, jp, kp);
    double gr[4][3];
#pragma unroll
    for (int a = 0; a < 4; ++a) {
        const double *f = prim + a * g.np + id;  // P_U, P_V, P_W, P_T
        gr[a][0] = d1_ghost(f, 1, i, g.nx, g.periodic[0]);
        gr[a][1] = d1_ghost(f, g.sy, j, g.ny, g.periodic[1]);
        gr[a][2] = d1_ghost(f, g.sz, k, g.nz, g.periodic[2]);
    }
    double m[3][3];
#pragma unroll
    for (int d = 0; d < 3; ++d) Met<KIND>::row(g, d, ip, jp, kp, m[d][0], m[d][1], m[d][2]);
    const double iJ = 1.0 / Met<KIND>::J(g, ip, jp, kp);
    double gx[4], gy[4], gz[4];
#pragma unroll
    for (int a = 0; a < 4; ++a) {  // chain rule
        gx[a] = m[0][0] * gr[a][0] + m[1][0] * gr[a][1] + m[2][0] * gr[a][2];
        gy[a] = m[0][1] * gr[a][0] + m[1][1] * gr[a][1] + m[2][1] * gr[a][2];
        gz[a] = m[0][2] * gr[a][0] + m[1][2] * gr[a][1] + m[2][2] * gr[a][2];
    }
    const double u = prim[P_U * g.np + id], v = prim[P_V * g.np + id], w = prim[P_W * g.np + id], T = prim[P_T * g.np + id];
    const double mu0 = (1.0 + gs.suth) / (T + gs.suth) * T * sqrt(T);  // eq. 15
    const double mu = mu0 * gs.invRe, kc = mu0 * gs.kfac;              // eq. 14
    const double div = gx[0] + gy[1] + gz[2];
    const double txx = mu * (2.0 * gx[0] - (2.0 / 3.0) * div);         // eq. 13
    const double tyy = mu * (2.0 * gy[1] - (2.0 / 3.0) * div);
    const double tzz = mu * (2.0 * gz[2] - (2.0 / 3.0) * div);
    const double txy = mu * (gy[0] + gx[1]), txz = mu * (gz[0] + gx[2]), tyz = mu * (gz[1] + gy[2]);
    const double thx = u * txx + v * txy + w * txz + kc * gx[3];       // eq. 12 (R-2)
    const double thy = u * txy + v * tyy + w * tyz + kc * gy[3];
    const double thz = u * txz + v * tyz + w * tzz + kc * gz[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {                                       // eq. 9-11
        const double dx = m[d][0] * iJ, dy = m[d][1] * iJ, dz = m[d][2] * iJ;
        Fv[(4 * d + 0) * g.np + id] = dx * txx + dy * txy + dz * txz;
        Fv[(4 * d + 1) * g.np + id] = dx * txy + dy * tyy + dz * tyz;
        Fv[(4 * d + 2) * g.np + id] = dx * txz + dy * tyz + dz * tzz;
        Fv[(4 * d + 3) * g.np + id] = dx * thx + dy * thy + dz * thz;
    }
}

// a7
template <int KIND>
__global__ void __launch_bounds__(256) k_viscous_div(GridDesc g, const double *__restrict__ Fv, double *__restrict__ dU) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z * blockDim.z + threadIdx.z;
    if (i >= g.nx || j >= g.ny || k >= g.nz) return;
    const int ip = i + OCFD_NG, jp = j + OCFD_NG, kp = k + OCFD_NG;
    const long long id = pidx(g, ip, jp, kp);
    const double J = Met<KIND>::J(g, ip, jp, kp);
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        double s = d1_wrap(Fv + (0 + r) * g.np + id, 1, i, g.nx, g.periodic[0]);
        s += d1_wrap(Fv + (4 + r) * g.np + id, g.sy, j, g.ny, g.periodic[1]);
        s += d1_wrap(Fv + (8 + r) * g.np + id, g.sz, k, g.nz, g.periodic[2]);
        dU[(r + 1) * g.np + id] += J * s;
    }
}

template <int KIND>
ocfd_status launch_kind(ocfd_ctx *c, double *dU) {
    const GridDesc &g = c->g;
    dim3 blk(32, 4, 2), grd((g.nx + 31) / 32, (g.ny + 3) / 4, (g.nz + 1) / 2);
    OCFD_T0(c, K_VISC_FLUX);
    k_viscous_flux<KIND><<<grd, blk, 0, c->stream>>>(g, c->gas, c->prim, c->Fv);
    OCFD_CHECK_LAUNCH(c);
    OCFD_T0(c, K_VISC_DIV);
    k_viscous_div<KIND><<<grd, blk, 0, c->stream>>>(g, c->Fv, dU);
    OCFD_CHECK_LAUNCH(c);
    return OCFD_OK;
}

}  // namespace

ocfd_status launch_viscous(ocfd_ctx *c, const double *U, double *dU) {
    (void)U;
    switch (c->g.kind) {
        case OCFD_GRID_UNIFORM: return launch_kind<OCFD_GRID_UNIFORM>(c, dU);
        case OCFD_GRID_STRETCHED: return launch_kind<OCFD_GRID_STRETCHED>(c, dU);
        default: return launch_kind<OCFD_GRID_CURVILINEAR>(c, dU);
    }
}
