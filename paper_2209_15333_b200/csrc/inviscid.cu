// Rows a4 + a5: Steger-Warming split (eq. 19-29) computed in-kernel for a tile plus its
// 4-point halos, staged in shared memory, then UD7 / WENO7 / WENO5 reconstruction (eq. 41) of
// both split fluxes at every interface of the tile and the conservative flux difference.
//
// Unlike the paper's design (one kernel materialises f+- of all directions in global memory, then
// a difference kernel per direction re-reads them), the split fluxes never leave the SM: that removes
// 160 B/point/direction of HBM traffic.  See DESIGN.md section 7.
#include "ocfd_internal.cuh"

namespace {

// ------------------------------------------------------------------------------------------ schemes
__device__ __forceinline__ double ud7(double a, double b, double c, double d, double e, double f, double g) {
    // eq. 41
    return (-3.0 * a + 25.0 * b - 101.0 * c + 319.0 * d + 214.0 * e - 38.0 * f + 4.0 * g) * (1.0 / 420.0);
}

// WENO7.  Inputs f_{j-3..j+3} in upwind order; one division per reconstruction:
// sum_k w_k q_k = (sum_k C_k P_k q_k) / (sum_k C_k P_k), P_k = prod_{m != k} (eps + IS_m)^2.
__device__ __forceinline__ double weno7(double a, double b, double c, double d, double e, double f, double g, double eps) {
    // undivided differences
    const double d1a = b - a, d1b = c - b, d1c = d - c, d1d = e - d, d1e = f - e, d1f = g - f;
    const double d2a = d1b - d1a, d2b = d1c - d1b, d2c = d1d - d1c, d2d = d1e - d1d, d2e = d1f - d1e;
    const double s30 = d2b - d2a, s31 = d2c - d2b, s32 = d2d - d2c, s33 = d2e - d2d;  // third derivatives
    // second derivatives of the four cubics at x_j
    const double s20 = d2b + s30, s21 = d2c, s22 = d2c, s23 = d2d - s33;
    // first derivatives at x_j
    const double s10 = (-7.0 * a + 33.0 * b - 69.0 * c + 43.0 * d) * (1.0 / 24.0);
    const double s11 = (5.0 * b - 27.0 * c + 15.0 * d + 7.0 * e) * (1.0 / 24.0);
    const double s12 = (-7.0 * c - 15.0 * d + 27.0 * e - 5.0 * f) * (1.0 / 24.0);
    const double s13 = (-43.0 * d + 69.0 * e - 33.0 * f + 7.0 * g) * (1.0 / 24.0);
    const double k2 = 13.0 / 12.0, k3 = 1043.0 / 960.0, k13 = 1.0 / 12.0;
    double i0 = s10 * (s10 + k13 * s30) + k2 * s20 * s20 + k3 * s30 * s30 + eps;
    double i1 = s11 * (s11 + k13 * s31) + k2 * s21 * s21 + k3 * s31 * s31 + eps;
    double i2 = s12 * (s12 + k13 * s32) + k2 * s22 * s22 + k3 * s32 * s32 + eps;
    double i3 = s13 * (s13 + k13 * s33) + k2 * s23 * s23 + k3 * s33 * s33 + eps;
    i0 *= i0; i1 *= i1; i2 *= i2; i3 *= i3;
    const double p01 = i0 * i1, p23 = i2 * i3;
    const double w0 = (1.0 / 35.0) * (i1 * p23), w1 = (12.0 / 35.0) * (i0 * p23);
    const double w2 = (18.0 / 35.0) * (p01 * i3), w3 = (4.0 / 35.0) * (p01 * i2);
    const double q0 = (-3.0 * a + 13.0 * b - 23.0 * c + 25.0 * d) * (1.0 / 12.0);
    const double q1 = (b - 5.0 * c + 13.0 * d + 3.0 * e) * (1.0 / 12.0);
    const double q2 = (-c + 7.0 * d + 7.0 * e - f) * (1.0 / 12.0);
    const double q3 = (3.0 * d + 13.0 * e - 5.0 * f + g) * (1.0 / 12.0);
    return (w0 * q0 + w1 * q1 + w2 * q2 + w3 * q3) / (w0 + w1 + w2 + w3);
}

// WENO5 (Jiang-Shu), inputs f_{j-2..j+2}
__device__ __forceinline__ double weno5(double b, double c, double d, double e, double f, double eps) {
    double t0 = b - 2.0 * c + d, t1 = b - 4.0 * c + 3.0 * d;
    double i0 = (13.0 / 12.0) * t0 * t0 + 0.25 * t1 * t1 + eps;
    t0 = c - 2.0 * d + e; t1 = c - e;
    double i1 = (13.0 / 12.0) * t0 * t0 + 0.25 * t1 * t1 + eps;
    t0 = d - 2.0 * e + f; t1 = 3.0 * d - 4.0 * e + f;
    double i2 = (13.0 / 12.0) * t0 * t0 + 0.25 * t1 * t1 + eps;
    i0 *= i0; i1 *= i1; i2 *= i2;
    const double w0 = 0.1 * (i1 * i2), w1 = 0.6 * (i0 * i2), w2 = 0.3 * (i0 * i1);
    const double q0 = (2.0 * b - 7.0 * c + 11.0 * d) * (1.0 / 6.0);
    const double q1 = (-c + 5.0 * d + 2.0 * e) * (1.0 / 6.0);
    const double q2 = (2.0 * d + 5.0 * e - f) * (1.0 / 6.0);
    return (w0 * q0 + w1 * q1 + w2 * q2) / (w0 + w1 + w2);
}

template <int SCHEME>
__device__ __forceinline__ double recon(int flag, double a, double b, double c, double d, double e, double f, double g,
                                        double eps) {
    if (SCHEME == OCFD_UD7) return ud7(a, b, c, d, e, f, g);
    if (SCHEME == OCFD_WENO7) return weno7(a, b, c, d, e, f, g, eps);
    if (SCHEME == OCFD_WENO5) return weno5(b, c, d, e, f, eps);
    if (flag == 0) return ud7(a, b, c, d, e, f, g);
    if (flag == 1) return weno7(a, b, c, d, e, f, g, eps);
    return weno5(b, c, d, e, f, eps);
}

// numerical flux h[5] of one interface from the staged split fluxes: sF[c*cs + p*ps], c = 0..4 f+, 5..9 f-;
// p .. p+7 are the eight points j-3 .. j+4 around the interface
template <int SCHEME>
__device__ __forceinline__ void iface_flux(const double *__restrict__ sF, int cs, int ps, int flag, double eps, double h[5]) {
#pragma unroll
    for (int m = 0; m < 5; ++m) {
        const double *fp = sF + m * cs, *fm = sF + (m + 5) * cs;
        double hp = recon<SCHEME>(flag, fp[0], fp[ps], fp[2 * ps], fp[3 * ps], fp[4 * ps], fp[5 * ps], fp[6 * ps], eps);
        double hm = recon<SCHEME>(flag, fm[7 * ps], fm[6 * ps], fm[5 * ps], fm[4 * ps], fm[3 * ps], fm[2 * ps], fm[ps], eps);
        h[m] = hp + hm;
    }
}

__device__ __forceinline__ int iface_flag(const GasDesc &gs, double tha, double thb) {
    double Th = fmax(tha, thb);
    return Th <= gs.theta1 ? 0 : (Th <= gs.theta2 ? 1 : 2);
}

// ------------------------------------------------------------------------------------------ Steger-Warming
// Split fluxes of direction DIR at one point, written to sF[c*cs], c = 0..9 (eq. 19-29 with the
// readings R-4, R-5, R-7).  (a1,a2,a3) = (d_x,d_y,d_z)/J.
template <int KIND, int DIR>
__device__ __forceinline__ void sw_split_store(const GasDesc &gs, double rho, double u, double v, double w, double c,
                                               double a1, double a2, double a3, double *__restrict__ sF, int cs) {
    double sigma, k1, k2, k3, Vt;
    if (KIND == OCFD_GRID_CURVILINEAR) {
        sigma = sqrt(a1 * a1 + a2 * a2 + a3 * a3);
        double is = 1.0 / sigma;
        k1 = a1 * is; k2 = a2 * is; k3 = a3 * is;
        Vt = a1 * u + a2 * v + a3 * w;
    } else {  // Cartesian: alpha has one non-zero component
        double a = DIR == 0 ? a1 : DIR == 1 ? a2 : a3;
        sigma = fabs(a);
        double sg = a < 0.0 ? -1.0 : 1.0;
        k1 = DIR == 0 ? sg : 0.0; k2 = DIR == 1 ? sg : 0.0; k3 = DIR == 2 ? sg : 0.0;
        Vt = a * (DIR == 0 ? u : DIR == 1 ? v : w);
    }
    const double cs_ = c * sigma;
    const double l1 = Vt, l4 = Vt - cs_, l5 = Vt + cs_;
    double l1p, l4p, l5p;
    if (gs.sw_eps == 0.0) {  // eq. 29
        l1p = 0.5 * (l1 + fabs(l1)); l4p = 0.5 * (l4 + fabs(l4)); l5p = 0.5 * (l5 + fabs(l5));
    } else {
        const double e2 = gs.sw_eps * gs.sw_eps;
        l1p = 0.5 * (l1 + sqrt(l1 * l1 + e2)); l4p = 0.5 * (l4 + sqrt(l4 * l4 + e2)); l5p = 0.5 * (l5 + sqrt(l5 * l5 + e2));
    }
    const double l1m = l1 - l1p, l4m = l4 - l4p, l5m = l5 - l5p;
    const double um = u - c * k1, vm = v - c * k2, wm = w - c * k3;
    const double up = u + c * k1, vp = v + c * k2, wp = w + c * k3;
    const double vc1 = 0.5 * (um * um + vm * vm + wm * wm), vc2 = 0.5 * (up * up + vp * vp + wp * wp);
    const double q2 = u * u + v * v + w * w, c2w = gs.w0 * c * c;
    const double h = rho * gs.inv2g;
    {
        const double t = gs.tgm1 * l1p;
        sF[0] = h * (t + l4p + l5p);
        sF[cs] = h * (t * u + l4p * um + l5p * up);
        sF[2 * cs] = h * (t * v + l4p * vm + l5p * vp);
        sF[3 * cs] = h * (t * w + l4p * wm + l5p * wp);
        sF[4 * cs] = h * (gs.gm1 * l1p * q2 + l4p * vc1 + l5p * vc2 + c2w * (l4p + l5p));
    }
    {
        const double t = gs.tgm1 * l1m;
        sF[5 * cs] = h * (t + l4m + l5m);
        sF[6 * cs] = h * (t * u + l4m * um + l5m * up);
        sF[7 * cs] = h * (t * v + l4m * vm + l5m * vp);
        sF[8 * cs] = h * (t * w + l4m * wm + l5m * wp);
        sF[9 * cs] = h * (gs.gm1 * l1m * q2 + l4m * vc1 + l5m * vc2 + c2w * (l4m + l5m));
    }
}

// split fluxes at padded point (ip,jp,kp) from the primitive fields
template <int KIND, int DIR>
__device__ __forceinline__ void split_point(const GridDesc &g, const GasDesc &gs, const double *__restrict__ U,
                                            const double *__restrict__ prim, int ip, int jp, int kp,
                                            double *__restrict__ sF, int cs) {
    const long long id = pidx(g, ip, jp, kp);
    const double rho = __ldg(U + id);
    const double u = __ldg(prim + P_U * g.np + id), v = __ldg(prim + P_V * g.np + id), w = __ldg(prim + P_W * g.np + id);
    const double c = __ldg(prim + P_C * g.np + id);
    double a1, a2, a3;
    Met<KIND>::row(g, DIR, ip, jp, kp, a1, a2, a3);
    const double iJ = 1.0 / Met<KIND>::J(g, ip, jp, kp);
    sw_split_store<KIND, DIR>(gs, rho, u, v, w, c, a1 * iJ, a2 * iJ, a3 * iJ, sF, cs);
}

// ------------------------------------------------------------------------------------------ x sweep
// Block: XT threads along x (one per point of a 64-point window: 56 outputs + 4-point halos) x XL lines.
constexpr int XT = 64, XL = 4, XOUT = XT - 8;

template <int KIND, int SCHEME>
__global__ void __launch_bounds__(XT *XL) k_inviscid_x(GridDesc g, GasDesc gs, const double *__restrict__ U,
                                                         const double *__restrict__ prim, const double *__restrict__ theta,
                                                         double *__restrict__ dU) {
    __shared__ double sF[10][XL][XT];
    __shared__ double sH[5][XL][XT];
    const int t = threadIdx.x, l = threadIdx.y;
    const int line = blockIdx.y * XL + l;
    const bool line_ok = line < g.ny * g.nz;
    const int j = line_ok ? line % g.ny : 0, k = line_ok ? line / g.ny : 0;
    const int jp = j + OCFD_NG, kp = k + OCFD_NG;
    const int ip = blockIdx.x * XOUT + t;  // padded x index of this thread's point
    const int i = ip - OCFD_NG;            // interior index
    const bool pt_ok = line_ok && ip < g.nxp;
    if (pt_ok) split_point<KIND, 0>(g, gs, U, prim, ip, jp, kp, &sF[0][l][t], XL * XT);
    __syncthreads();
    // interface i+1/2 uses points t-3 .. t+4
    if (pt_ok && t >= 3 && t <= XT - 5 && i >= -1 && i <= g.nx - 1) {
        int flag = 0;
        if (SCHEME == OCFD_HYBRID) {
            const long long id = pidx(g, ip, jp, kp);
            flag = iface_flag(gs, __ldg(theta + id), __ldg(theta + id + 1));
        }
        double h[5];
        iface_flux<SCHEME>(&sF[0][l][t - 3], XL * XT, 1, flag, gs.weno_eps, h);
#pragma unroll
        for (int m = 0; m < 5; ++m) sH[m][l][t] = h[m];
    }
    __syncthreads();
    if (pt_ok && t >= 4 && t <= XT - 5 && i >= 0 && i < g.nx) {
        const long long id = pidx(g, ip, jp, kp);
        const double J = Met<KIND>::J(g, ip, jp, kp);
#pragma unroll
        for (int m = 0; m < 5; ++m) dU[m * g.np + id] = -J * (sH[m][l][t] - sH[m][l][t - 1]);
    }
}

// ------------------------------------------------------------------------------------------ y / z sweeps
// Block: 32 lanes along x (coalesced rows) x YR rows of threads; the tile holds YP = YS + 8 points along the sweep
// (YS outputs).  YP and YS + 1 are multiples of YR = 7, so the split-flux pass (YP/YR points per thread) and the
// reconstruction pass ((YS+1)/YR interfaces per thread) are both perfectly balanced.
constexpr int YW = 32, YR = 7, YS = 20, YP = YS + 8, YI = YS + 1;
static_assert(YP % YR == 0 && YI % YR == 0, "tile shape");

template <int KIND, int SCHEME, int DIR>
__global__ void __launch_bounds__(YW *YR) k_inviscid_yz(GridDesc g, GasDesc gs, const double *__restrict__ U,
                                                          const double *__restrict__ prim, const double *__restrict__ theta,
                                                          double *__restrict__ dU) {
    extern __shared__ double smem[];  // sF[10][YP][YW], later aliased by sH[5][YI][YW]
    double *sF = smem;
    const int x = threadIdx.x, r = threadIdx.y;
    const int ip = blockIdx.x * YW + x + OCFD_NG;
    const bool x_ok = ip < g.nx + OCFD_NG;
    const int s0 = blockIdx.y * YS;                       // first interior sweep index of the tile
    const int nd = DIR == 1 ? g.ny : g.nz;
    const int cp = blockIdx.z + OCFD_NG;                  // padded cross index (k for the y sweep, j for z)
    const long long sd = DIR == 1 ? g.sy : g.sz;
    // pass 1: split fluxes at tile points p = 0..YP-1  <->  padded sweep index s0 + p
    if (x_ok) {
#pragma unroll
        for (int q = 0; q < YP / YR; ++q) {
            const int p = r + q * YR;
            int sp = s0 + p;
            if (sp > nd + 2 * OCFD_NG - 1) sp = nd + 2 * OCFD_NG - 1;  // ragged tail: stay inside the array
            const int jp = DIR == 1 ? sp : cp, kp = DIR == 1 ? cp : sp;
            split_point<KIND, DIR>(g, gs, U, prim, ip, jp, kp, sF + p * YW + x, YP * YW);
        }
    }
    __syncthreads();
    // pass 2: interfaces q = 0..YI-1 between tile points q+3 and q+4 (interior sweep index s0-1+q)
    double h[YI / YR][5];
#pragma unroll
    for (int qq = 0; qq < YI / YR; ++qq) {
        const int q = r + qq * YR;
        const int s = s0 - 1 + q;
        if (x_ok && s <= nd - 1) {
            int flag = 0;
            if (SCHEME == OCFD_HYBRID) {
                const int sp = s + OCFD_NG;
                const long long id = pidx(g, ip, DIR == 1 ? sp : cp, DIR == 1 ? cp : sp);
                flag = iface_flag(gs, __ldg(theta + id), __ldg(theta + id + sd));
            }
            iface_flux<SCHEME>(sF + q * YW + x, YP * YW, YW, flag, gs.weno_eps, h[qq]);
        }
    }
    __syncthreads();
    double *sH = smem;  // [5][YI][YW]
#pragma unroll
    for (int qq = 0; qq < YI / YR; ++qq) {
        const int q = r + qq * YR;
#pragma unroll
        for (int m = 0; m < 5; ++m) sH[(m * YI + q) * YW + x] = h[qq][m];
    }
    __syncthreads();
    // pass 3: outputs o = 0..YS-1 (interior sweep index s0+o): dU -= J (h_{o+1} - h_o)
    if (x_ok) {
        for (int o = r; o < YS; o += YR) {
            const int s = s0 + o;
            if (s >= nd) break;
            const int sp = s + OCFD_NG;
            const int jp = DIR == 1 ? sp : cp, kp = DIR == 1 ? cp : sp;
            const long long id = pidx(g, ip, jp, kp);
            const double J = Met<KIND>::J(g, ip, jp, kp);
#pragma unroll
            for (int m = 0; m < 5; ++m)
                dU[m * g.np + id] -= J * (sH[(m * YI + o + 1) * YW + x] - sH[(m * YI + o) * YW + x]);
        }
    }
}

template <int KIND, int SCHEME>
ocfd_status launch_kind_scheme(ocfd_ctx *c, const double *U, double *dU) {
    const GridDesc &g = c->g;
    {
        dim3 blk(XT, XL), grd((g.nx + XOUT - 1) / XOUT, (g.ny * g.nz + XL - 1) / XL);
        OCFD_T0(c, K_INV_X);
        k_inviscid_x<KIND, SCHEME><<<grd, blk, 0, c->stream>>>(g, c->gas, U, c->prim, c->theta, dU);
        OCFD_CHECK_LAUNCH(c);
    }
    const size_t shm = sizeof(double) * 10 * YP * YW;
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(k_inviscid_yz<KIND, SCHEME, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)shm) != cudaSuccess) return OCFD_ECUDA;
        if (cudaFuncSetAttribute(k_inviscid_yz<KIND, SCHEME, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)shm) != cudaSuccess) return OCFD_ECUDA;
        attr_set = true;
    }
    {
        dim3 blk(YW, YR), grd((g.nx + YW - 1) / YW, (g.ny + YS - 1) / YS, g.nz);
        OCFD_T0(c, K_INV_Y);
        k_inviscid_yz<KIND, SCHEME, 1><<<grd, blk, shm, c->stream>>>(g, c->gas, U, c->prim, c->theta, dU);
        OCFD_CHECK_LAUNCH(c);
    }
    {
        dim3 blk(YW, YR), grd((g.nx + YW - 1) / YW, (g.nz + YS - 1) / YS, g.ny);
        OCFD_T0(c, K_INV_Z);
        k_inviscid_yz<KIND, SCHEME, 2><<<grd, blk, shm, c->stream>>>(g, c->gas, U, c->prim, c->theta, dU);
        OCFD_CHECK_LAUNCH(c);
    }
    return OCFD_OK;
}

template <int KIND>
ocfd_status launch_kind(ocfd_ctx *c, const double *U, double *dU) {
    switch (c->p.scheme) {
        case OCFD_UD7: return launch_kind_scheme<KIND, OCFD_UD7>(c, U, dU);
        case OCFD_WENO7: return launch_kind_scheme<KIND, OCFD_WENO7>(c, U, dU);
        case OCFD_WENO5: return launch_kind_scheme<KIND, OCFD_WENO5>(c, U, dU);
        default: return launch_kind_scheme<KIND, OCFD_HYBRID>(c, U, dU);
    }
}

}  // namespace

// dU <- -J sum_d (h_{s+1/2} - h_{s-1/2}); the x sweep writes, y and z accumulate (same order as the definition)
ocfd_status launch_inviscid(ocfd_ctx *c, const double *U, double *dU) {
    switch (c->g.kind) {
        case OCFD_GRID_UNIFORM: return launch_kind<OCFD_GRID_UNIFORM>(c, U, dU);
        case OCFD_GRID_STRETCHED: return launch_kind<OCFD_GRID_STRETCHED>(c, U, dU);
        default: return launch_kind<OCFD_GRID_CURVILINEAR>(c, U, dU);
    }
}
