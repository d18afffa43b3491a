// Rows a6 + a7 (+ a8 fused): viscous and heat-flux terms (eq. 9-15) by the 6th-order central
// first derivative applied twice (DESIGN R-15): pass 1 forms the viscous fluxes at interior
// points, pass 2 differences them and accumulates into dU (and, inside ocfd_rk3_step, applies the RK3 stage update
// of eq. 45 in the same kernel so that dU is not written and re-read).
//
// Both passes are 2.5-D marching kernels: a block owns an x-y tile and walks along z.  Each thread keeps the seven
// z-planes its zeta-derivative needs in registers, so every field value is fetched from HBM once; the x and y
// neighbours of the current plane are exchanged through a shared-memory tile with 3-point halos.
#include "ocfd_internal.cuh"

namespace {

constexpr int TX = 32, TY = 8;               // threads = tile of own points
constexpr int SXW = TX + 6, SYW = TY + 6;    // shared tile with 3-point halos

__device__ __forceinline__ double d1c(double m3, double m2, double m1, double p1, double p2, double p3) {
    return (45.0 * (p1 - m1) - 9.0 * (p2 - m2) + (p3 - m3)) * (1.0 / 60.0);
}
// first derivative at position s of a line of n from the seven values v[0..6] = f_{s-3..s+3}; closure rows of an
// aperiodic axis only touch values inside the line
__device__ __forceinline__ double d1_seven(const double v[7], int s, int n, int periodic) {
    if (periodic || (s >= 3 && s <= n - 4)) return d1c(v[0], v[1], v[2], v[4], v[5], v[6]);
    if (s == 0) return (-3.0 * v[3] + 4.0 * v[4] - v[5]) * 0.5;
    if (s == n - 1) return (3.0 * v[3] - 4.0 * v[2] + v[1]) * 0.5;
    if (s == 1 || s == n - 2) return (v[4] - v[2]) * 0.5;
    return (8.0 * (v[4] - v[2]) - (v[5] - v[1])) * (1.0 / 12.0);  // s == 2 or n-3
}
// the same from a shared-memory line (p points at position s, stride st)
__device__ __forceinline__ double d1_line(const double *p, int st, int s, int n, int periodic) {
    if (periodic || (s >= 3 && s <= n - 4)) return d1c(p[-3 * st], p[-2 * st], p[-st], p[st], p[2 * st], p[3 * st]);
    if (s == 0) return (-3.0 * p[0] + 4.0 * p[st] - p[2 * st]) * 0.5;
    if (s == n - 1) return (3.0 * p[0] - 4.0 * p[-st] + p[-2 * st]) * 0.5;
    if (s == 1 || s == n - 2) return (p[st] - p[-st]) * 0.5;
    return (8.0 * (p[st] - p[-st]) - (p[2 * st] - p[-2 * st])) * (1.0 / 12.0);
}

__device__ __forceinline__ int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }
__device__ __forceinline__ int wrapi(int v, int n) { return v < 0 ? v + n : (v >= n ? v - n : v); }

// ------------------------------------------------------------------------------------------------ a6
// prim: padded fields u,v,w,T (valid on interior + face ghosts).  Fv: [12][np], written at interior points.
template <int KIND>
__global__ void __launch_bounds__(TX *TY, 2) k_viscous_flux(GridDesc g, GasDesc gs, const double *__restrict__ prim,
                                                         double *__restrict__ Fv, int zchunk) {
    __shared__ double sp[4][SYW][SXW];
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * TX + tx;
    const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY;
    const int i = i0 + tx, j = j0 + ty;
    const bool own = i < g.nx && j < g.ny;
    // threads past the ragged edge still stage their (ghost) column: the last own points differentiate through it
    const int ip = min(i, g.nx + OCFD_NG - 1) + OCFD_NG, jp = min(j, g.ny + OCFD_NG - 1) + OCFD_NG;
    const int k0 = blockIdx.z * zchunk, k1 = min(k0 + zchunk, g.nz);
    const long long col = (long long)jp * g.sy + ip;  // padded offset within a plane
    // z window: planes k-3 .. k+3 of the four fields at this thread's column
    double w[4][7];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int q = 0; q < 6; ++q) w[a][q + 1] = prim[a * g.np + (long long)(k0 - 3 + q + OCFD_NG) * g.sz + col];
    // metrics of this column are needed every step; for z-extruded grids they do not depend on k
    for (int k = k0; k < k1; ++k) {
        const int kp = k + OCFD_NG;
#pragma unroll
        for (int a = 0; a < 4; ++a) {
#pragma unroll
            for (int q = 0; q < 6; ++q) w[a][q] = w[a][q + 1];
            w[a][6] = prim[a * g.np + (long long)(kp + 3) * g.sz + col];
        }
        __syncthreads();  // previous plane's tile is no longer read
#pragma unroll
        for (int a = 0; a < 4; ++a) sp[a][ty + 3][tx + 3] = w[a][3];
        // halo cells of plane k (x: 2x3 columns, y: 2x3 rows; corners are not needed)
        for (int c = tid; c < 2 * 3 * TY + 2 * 3 * TX; c += TX * TY) {
            int hx, hy;
            if (c < 6 * TY) { hx = (c % 6 < 3) ? c % 6 : TX + c % 6; hy = 3 + c / 6; }
            else { const int e = c - 6 * TY; hx = 3 + e % TX; hy = (e / TX < 3) ? e / TX : TY + e / TX; }
            const int gi = clampi(i0 - 3 + hx, -OCFD_NG, g.nx + OCFD_NG - 1) + OCFD_NG;
            const int gj = clampi(j0 - 3 + hy, -OCFD_NG, g.ny + OCFD_NG - 1) + OCFD_NG;
            const long long id = (long long)kp * g.sz + (long long)gj * g.sy + gi;
#pragma unroll
            for (int a = 0; a < 4; ++a) sp[a][hy][hx] = __ldg(prim + a * g.np + id);
        }
        __syncthreads();
        if (!own) continue;
        double gr[4][3];
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            gr[a][0] = d1_line(&sp[a][ty + 3][tx + 3], 1, i, g.nx, g.periodic[0]);
            gr[a][1] = d1_line(&sp[a][ty + 3][tx + 3], SXW, j, g.ny, g.periodic[1]);
            gr[a][2] = d1_seven(w[a], k, g.nz, g.periodic[2]);
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
        const double u = w[0][3], v = w[1][3], ww = w[2][3], T = w[3][3];
        const double mu0 = (1.0 + gs.suth) / (T + gs.suth) * T * sqrt(T);  // eq. 15
        const double mu = mu0 * gs.invRe, kc = mu0 * gs.kfac;              // eq. 14
        const double div = gx[0] + gy[1] + gz[2];
        const double txx = mu * (2.0 * gx[0] - (2.0 / 3.0) * div);         // eq. 13
        const double tyy = mu * (2.0 * gy[1] - (2.0 / 3.0) * div);
        const double tzz = mu * (2.0 * gz[2] - (2.0 / 3.0) * div);
        const double txy = mu * (gy[0] + gx[1]), txz = mu * (gz[0] + gx[2]), tyz = mu * (gz[1] + gy[2]);
        const double thx = u * txx + v * txy + ww * txz + kc * gx[3];      // eq. 12 (R-2)
        const double thy = u * txy + v * tyy + ww * tyz + kc * gy[3];
        const double thz = u * txz + v * tyz + ww * tzz + kc * gz[3];
        const long long id = (long long)kp * g.sz + col;
#pragma unroll
        for (int d = 0; d < 3; ++d) {                                       // eq. 9-11
            const double dx = m[d][0] * iJ, dy = m[d][1] * iJ, dz = m[d][2] * iJ;
            Fv[(4 * d + 0) * g.np + id] = dx * txx + dy * txy + dz * txz;
            Fv[(4 * d + 1) * g.np + id] = dx * txy + dy * tyy + dz * tyz;
            Fv[(4 * d + 2) * g.np + id] = dx * txz + dy * tyz + dz * tzz;
            Fv[(4 * d + 3) * g.np + id] = dx * thx + dy * thy + dz * thz;
        }
    }
}

// ------------------------------------------------------------------------------------------------ a7 (+ a8)
// RK: 0 = plain accumulate into dU (ocfd_rhs); 1..3 = also apply RK3 stage RK-1 (eq. 45) to U, dU is not written.
template <int KIND, int RK>
__global__ void __launch_bounds__(TX *TY, 2) k_viscous_div(GridDesc g, const double *__restrict__ Fv, double *__restrict__ dU,
                                                        double *__restrict__ U, double *__restrict__ Un, double dt,
                                                        int zchunk) {
    __shared__ double sF[4][TY][SXW];   // xi-direction flux with x halos
    __shared__ double sG[4][SYW][TX];   // eta-direction flux with y halos
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * TX + tx;
    const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY;
    const int i = i0 + tx, j = j0 + ty;
    const bool own = i < g.nx && j < g.ny;
    const int ip = (own ? i : g.nx - 1) + OCFD_NG, jp = (own ? j : g.ny - 1) + OCFD_NG;
    const int k0 = blockIdx.z * zchunk, k1 = min(k0 + zchunk, g.nz);
    const long long col = (long long)jp * g.sy + ip;
    const double *H = Fv + 8 * g.np;
    // z window of the zeta-direction flux: interior planes only; periodic axes wrap, aperiodic ones never read outside
    auto zplane = [&](int k) -> long long {
        const int kk = g.periodic[2] ? wrapi(k, g.nz) : clampi(k, 0, g.nz - 1);
        return (long long)(kk + OCFD_NG) * g.sz;
    };
    double w[4][7];
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int q = 0; q < 6; ++q) w[r][q + 1] = H[r * g.np + zplane(k0 - 3 + q) + col];
    for (int k = k0; k < k1; ++k) {
        const int kp = k + OCFD_NG;
        const long long pl = (long long)kp * g.sz;
#pragma unroll
        for (int r = 0; r < 4; ++r) {
#pragma unroll
            for (int q = 0; q < 6; ++q) w[r][q] = w[r][q + 1];
            w[r][6] = H[r * g.np + zplane(k + 3) + col];
        }
        __syncthreads();
        // own values + halos of F (x) and G (y) for plane k
        for (int c = tid; c < TY * SXW; c += TX * TY) {
            const int hx = c % SXW, hy = c / SXW;
            int gi = i0 - 3 + hx;
            gi = g.periodic[0] ? wrapi(gi, g.nx) : clampi(gi, 0, g.nx - 1);
            const int gj = min(j0 + hy, g.ny - 1);
            const long long id = pl + (long long)(gj + OCFD_NG) * g.sy + gi + OCFD_NG;
#pragma unroll
            for (int r = 0; r < 4; ++r) sF[r][hy][hx] = __ldg(Fv + r * g.np + id);
        }
        for (int c = tid; c < SYW * TX; c += TX * TY) {
            const int hx = c % TX, hy = c / TX;
            int gj = j0 - 3 + hy;
            gj = g.periodic[1] ? wrapi(gj, g.ny) : clampi(gj, 0, g.ny - 1);
            const int gi = min(i0 + hx, g.nx - 1);
            const long long id = pl + (long long)(gj + OCFD_NG) * g.sy + gi + OCFD_NG;
#pragma unroll
            for (int r = 0; r < 4; ++r) sG[r][hy][hx] = __ldg(Fv + (4 + r) * g.np + id);
        }
        __syncthreads();
        if (!own) continue;
        const long long id = pl + col;
        const double J = Met<KIND>::J(g, ip, jp, kp);
        double acc[5];
        acc[0] = dU[id];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            // interior stencils wrap through the staged halos, so "periodic" is passed as 1 only when the axis is
            double s = d1_line(&sF[r][ty][tx + 3], 1, i, g.nx, g.periodic[0]);
            s += d1_line(&sG[r][ty + 3][tx], TX, j, g.ny, g.periodic[1]);
            s += d1_seven(w[r], k, g.nz, g.periodic[2]);
            acc[r + 1] = dU[(r + 1) * g.np + id] + J * s;
        }
        if (RK == 0) {
#pragma unroll
            for (int r = 1; r < 5; ++r) dU[r * g.np + id] = acc[r];
        } else {
#pragma unroll
            for (int m = 0; m < 5; ++m) {
                const long long q = m * g.np + id;
                const double u = U[q];
                if (RK == 1) {
                    Un[q] = u;
                    U[q] = u + dt * acc[m];
                } else if (RK == 2) {
                    U[q] = 0.75 * Un[q] + 0.25 * (u + dt * acc[m]);
                } else {
                    U[q] = (1.0 / 3.0) * Un[q] + (2.0 / 3.0) * (u + dt * acc[m]);
                }
            }
        }
    }
}

int pick_zchunk(const GridDesc &g) {
    // enough blocks to fill 148 SMs a few times over, chunks long enough that the 6 halo planes stay cheap
    const long long tiles = (long long)((g.nx + TX - 1) / TX) * ((g.ny + TY - 1) / TY);
    int zc = g.nz;
    while (zc > 32 && tiles * ((g.nz + zc - 1) / zc) < 148 * 8) zc = (zc + 1) / 2;
    return zc;
}

template <int KIND>
ocfd_status launch_kind(ocfd_ctx *c, double *dU, double *U, double dt, int rk_stage) {
    const GridDesc &g = c->g;
    const int zc = pick_zchunk(g);
    dim3 blk(TX, TY, 1), grd((g.nx + TX - 1) / TX, (g.ny + TY - 1) / TY, (g.nz + zc - 1) / zc);
    OCFD_T0(c, K_VISC_FLUX);
    k_viscous_flux<KIND><<<grd, blk, 0, c->stream>>>(g, c->gas, c->prim, c->Fv, zc);
    OCFD_CHECK_LAUNCH(c);
    OCFD_T0(c, K_VISC_DIV);
    switch (rk_stage) {
        case 0: k_viscous_div<KIND, 1><<<grd, blk, 0, c->stream>>>(g, c->Fv, dU, U, c->Un, dt, zc); break;
        case 1: k_viscous_div<KIND, 2><<<grd, blk, 0, c->stream>>>(g, c->Fv, dU, U, c->Un, dt, zc); break;
        case 2: k_viscous_div<KIND, 3><<<grd, blk, 0, c->stream>>>(g, c->Fv, dU, U, c->Un, dt, zc); break;
        default: k_viscous_div<KIND, 0><<<grd, blk, 0, c->stream>>>(g, c->Fv, dU, nullptr, nullptr, 0.0, zc);
    }
    OCFD_CHECK_LAUNCH(c);
    return OCFD_OK;
}

}  // namespace

// rk_stage < 0: dU += viscous terms.  rk_stage = 0,1,2: the same, then U <- RK3 stage update in the same kernel.
ocfd_status launch_viscous(ocfd_ctx *c, double *dU, double *U, double dt, int rk_stage) {
    switch (c->g.kind) {
        case OCFD_GRID_UNIFORM: return launch_kind<OCFD_GRID_UNIFORM>(c, dU, U, dt, rk_stage);
        case OCFD_GRID_STRETCHED: return launch_kind<OCFD_GRID_STRETCHED>(c, dU, U, dt, rk_stage);
        default: return launch_kind<OCFD_GRID_CURVILINEAR>(c, dU, U, dt, rk_stage);
    }
}
