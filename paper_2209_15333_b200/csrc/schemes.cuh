// Device functions shared by the inviscid sweep kernels: the reconstructions of eq. 41 / L286-305 (UD7, WENO7, WENO5),
// the hybrid interface flag (eq. 42, R-12) and the Steger-Warming split of one point (eq. 19-29).
#pragma once
#include "ocfd_internal.cuh"

namespace {

// ------------------------------------------------------------------------------------------ schemes
// eq. 41 coefficients / 420, in constant memory so that every DFMA takes its coefficient as a constant-bank operand
__constant__ double c_ud7[7] = {-3.0 / 420.0, 25.0 / 420.0, -101.0 / 420.0, 319.0 / 420.0, 214.0 / 420.0, -38.0 / 420.0, 4.0 / 420.0};

__device__ __forceinline__ double ud7(double a, double b, double c, double d, double e, double f, double g) {
    // eq. 41, as two fused-multiply-add chains
    const double lo = fma(c_ud7[2], c, fma(c_ud7[1], b, c_ud7[0] * a));
    const double hi = fma(c_ud7[6], g, fma(c_ud7[5], f, fma(c_ud7[4], e, c_ud7[3] * d)));
    return lo + hi;
}

// 1/x for x > 0 in the normal range: hardware seed (about 20 bits) and two Newton steps; a quotient num/den formed
// with it and corrected once by the residual is within a few ulp of the exact one (the bar on the sweeps is 1e-11)
__device__ __forceinline__ double fast_div_pos(double num, double den) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(den));
    r = fma(fma(-den, r, 1.0), r, r);
    r = fma(fma(-den, r, 1.0), r, r);
    const double q = num * r;
    return fma(fma(-den, q, num), r, q);
}

// 1/x for x > 0 in the normal range, within an ulp or two (same seed and Newton steps as fast_div_pos)
__device__ __forceinline__ double fast_rcp_pos(double x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    r = fma(fma(-x, r, 1.0), r, r);
    r = fma(fma(-x, r, 1.0), r, r);
    return r;
}

// sqrt(x) for x > 0 in the normal range: hardware seed of 1/sqrt(x), two Newton steps, one correction of the product
// (within an ulp or two; the library sqrt costs about twice the instructions)
__device__ __forceinline__ double fast_sqrt_pos(double x) {
    double r;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    const double hx = 0.5 * x;
    r = fma(fma(-hx * r, r, 0.5), r, r);
    r = fma(fma(-hx * r, r, 0.5), r, r);
    const double s = x * r;
    return fma(fma(-s, s, x), 0.5 * r, s);
}

// Row a2 inside its consumers: velocity and speed of sound of one point from the conserved variables (eq. 8 as
// corrected, DESIGN R-1; eq. 16: c^2 = T / Ma^2 = gamma p / rho).  No primitive field is ever written to HBM: every
// kernel that needs u, v, w, c (or T, p) forms them from the U box it has staged anyway.
__device__ __forceinline__ void prim_from_cons(const GasDesc &gs, double rho, double ru, double rv, double rw, double E,
                                               double &u, double &v, double &w, double &c) {
    const double ir = fast_rcp_pos(rho);
    u = ru * ir; v = rv * ir; w = rw * ir;
    const double p = gs.gm1 * (E - 0.5 * rho * (u * u + v * v + w * w));
    c = sqrt(gs.gamma * p * ir);
}

// WENO7.  Inputs f_{j-3..j+3} in upwind order; one division per reconstruction:
// sum_k w_k q_k = (sum_k P_k C_k q_k) / (sum_k C_k P_k), P_k = prod_{m != k} (eps + IS_m)^2.
// Everything is written on the undivided differences of the window (the derivatives s1, s2, s3 of the four cubics at
// x_j and the candidates C_k q_k are short combinations of them), about 100 fp64 instructions per reconstruction.
__device__ __forceinline__ double weno7(double a, double b, double c, double d, double e, double f, double g, double eps) {
    const double d1a = b - a, d1b = c - b, d1c = d - c, d1d = e - d, d1e = f - e, d1f = g - f;
    const double d2a = d1b - d1a, d2b = d1c - d1b, d2c = d1d - d1c, d2d = d1e - d1d, d2e = d1f - d1e;
    const double s30 = d2b - d2a, s31 = d2c - d2b, s32 = d2d - d2c, s33 = d2e - d2d;  // third derivatives
    // second derivatives of the four cubics at x_j
    const double s20 = d2b + s30, s21 = d2c, s23 = d2d - s33;
    // first derivatives at x_j: (-7a+33b-69c+43d)/24 = d1c + d2b/2 + 7 s30/24, (5b-27c+15d+7e)/24 = (d1c+d1d)/2 - 5 s31/24,
    // (-7c-15d+27e-5f)/24 = (d1c+d1d)/2 - 5 s32/24, (-43d+69e-33f+7g)/24 = d1d - d2d/2 + 7 s33/24
    const double mid = 0.5 * (d1c + d1d);
    const double s10 = fma(7.0 / 24.0, s30, fma(0.5, d2b, d1c));
    const double s11 = fma(-5.0 / 24.0, s31, mid);
    const double s12 = fma(-5.0 / 24.0, s32, mid);
    const double s13 = fma(7.0 / 24.0, s33, fma(-0.5, d2d, d1d));
    const double k2 = 13.0 / 12.0, k3 = 1043.0 / 960.0, k13 = 1.0 / 12.0;
    double i0 = fma(s10, fma(k13, s30, s10), fma(k2 * s20, s20, fma(k3 * s30, s30, eps)));
    double i1 = fma(s11, fma(k13, s31, s11), fma(k2 * s21, s21, fma(k3 * s31, s31, eps)));
    double i2 = fma(s12, fma(k13, s32, s12), fma(k2 * s21, s21, fma(k3 * s32, s32, eps)));
    double i3 = fma(s13, fma(k13, s33, s13), fma(k2 * s23, s23, fma(k3 * s33, s33, eps)));
    i0 *= i0; i1 *= i1; i2 *= i2; i3 *= i3;
    const double p01 = i0 * i1, p23 = i2 * i3;
    const double P0 = i1 * p23, P1 = i0 * p23, P2 = p01 * i3, P3 = p01 * i2;
    // candidates times their linear weights C = (1, 12, 18, 4)/35
    const double q0 = fma(25.0 / 420.0, d, fma(-23.0 / 420.0, c, fma(13.0 / 420.0, b, (-3.0 / 420.0) * a)));
    const double q1 = fma(36.0 / 420.0, e, fma(156.0 / 420.0, d, fma(-60.0 / 420.0, c, (12.0 / 420.0) * b)));
    const double q2 = fma(-18.0 / 420.0, f, fma(126.0 / 420.0, e, fma(126.0 / 420.0, d, (-18.0 / 420.0) * c)));
    const double q3 = fma(4.0 / 420.0, g, fma(-20.0 / 420.0, f, fma(52.0 / 420.0, e, (12.0 / 420.0) * d)));
    const double num = fma(P3, q3, fma(P2, q2, fma(P1, q1, P0 * q0)));
    const double den = fma(4.0 / 35.0, P3, fma(18.0 / 35.0, P2, fma(12.0 / 35.0, P1, (1.0 / 35.0) * P0)));
    return fast_div_pos(num, den);
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
    return fast_div_pos(w0 * q0 + w1 * q1 + w2 * q2, w0 + w1 + w2);
}

// WENO5 with shielded candidates (the paper's boundary scheme; DESIGN R-20): bit k of `keep` set =
// candidate k lies inside the domain; the others get weight 0 and are not evaluated.  keep == 0: `nearest` (R-21).
__device__ __forceinline__ double weno5_masked(double b, double c, double d, double e, double f, double eps, int keep,
                                               double nearest) {
    if ((keep & 7) == 0) return nearest;
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, q0 = 0.0, q1 = 0.0, q2 = 0.0;
    if (keep & 1) {
        const double t0 = b - 2.0 * c + d, t1 = b - 4.0 * c + 3.0 * d;
        const double is = (13.0 / 12.0) * t0 * t0 + 0.25 * t1 * t1 + eps;
        a0 = 0.1 / (is * is);
        q0 = (2.0 * b - 7.0 * c + 11.0 * d) * (1.0 / 6.0);
    }
    if (keep & 2) {
        const double t0 = c - 2.0 * d + e, t1 = c - e;
        const double is = (13.0 / 12.0) * t0 * t0 + 0.25 * t1 * t1 + eps;
        a1 = 0.6 / (is * is);
        q1 = (-c + 5.0 * d + 2.0 * e) * (1.0 / 6.0);
    }
    if (keep & 4) {
        const double t0 = d - 2.0 * e + f, t1 = 3.0 * d - 4.0 * e + f;
        const double is = (13.0 / 12.0) * t0 * t0 + 0.25 * t1 * t1 + eps;
        a2 = 0.3 / (is * is);
        q2 = (2.0 * d + 5.0 * e - f) * (1.0 / 6.0);
    }
    return (a0 * q0 + a1 * q1 + a2 * q2) / (a0 + a1 + a2);
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

__device__ __forceinline__ int iface_flag(const GasDesc &gs, double tha, double thb) {
    double Th = fmax(tha, thb);
    return Th <= gs.theta1 ? 0 : (Th <= gs.theta2 ? 1 : 2);
}

// h_{s+1/2} of an interface near an aperiodic boundary under the paper's boundary scheme.  s = interior index of the
// interface (s + 1/2), n = points of the axis; p0..p6 = f+ of points s-3..s+3, m0..m6 = f- of points s+4..s-2.  A flux
// whose 7-point stencil stays inside [0, n-1] takes the regular scheme `flag`.  Out of line: it runs on the few
// interfaces next to a boundary only.
__device__ __forceinline__ int inside3(int a, int n) { return a >= 0 && a + 2 <= n - 1; }
template <int SCHEME>
__device__ __noinline__ double recon_pair_closure(int flag, int s, int n, double p0, double p1, double p2, double p3,
                                                  double p4, double p5, double p6, double m0, double m1, double m2,
                                                  double m3, double m4, double m5, double m6, double eps) {
    const bool near_p = s - 3 < 0 || s + 3 > n - 1, near_m = s - 2 < 0 || s + 4 > n - 1;
    // f+ candidates {s-2,s-1,s}, {s-1,s,s+1}, {s,s+1,s+2}; f- (mirrored) {s+3,s+2,s+1}, {s+2,s+1,s}, {s+1,s,s-1}
    const int keep_p = inside3(s - 2, n) | inside3(s - 1, n) << 1 | inside3(s, n) << 2;
    const int keep_m = inside3(s + 1, n) | inside3(s, n) << 1 | inside3(s - 1, n) << 2;
    // all shielded only at s = -1 (f+: nearest node 0 = p4) and s = n-1 (f-: nearest node n-1 = m4)
    const double hp = near_p ? weno5_masked(p1, p2, p3, p4, p5, eps, keep_p, p4) : recon<SCHEME>(flag, p0, p1, p2, p3, p4, p5, p6, eps);
    const double hm = near_m ? weno5_masked(m1, m2, m3, m4, m5, eps, keep_m, m4) : recon<SCHEME>(flag, m0, m1, m2, m3, m4, m5, m6, eps);
    return hp + hm;
}

// h_{i+1/2} = recon(f+ window) + recon(mirrored f- window); out of line for the hybrid scheme (rare path, one copy)
template <int SCHEME>
__device__ __noinline__ double recon_pair_slow(int flag, double p0, double p1, double p2, double p3, double p4, double p5,
                                               double p6, double m0, double m1, double m2, double m3, double m4, double m5,
                                               double m6, double eps) {
    return recon<SCHEME>(flag, p0, p1, p2, p3, p4, p5, p6, eps) + recon<SCHEME>(flag, m0, m1, m2, m3, m4, m5, m6, eps);
}
template <int SCHEME>
__device__ __forceinline__ double recon_pair(int flag, double p0, double p1, double p2, double p3, double p4, double p5,
                                             double p6, double m0, double m1, double m2, double m3, double m4, double m5,
                                             double m6, double eps) {
    if (SCHEME == OCFD_HYBRID) return recon_pair_slow<SCHEME>(flag, p0, p1, p2, p3, p4, p5, p6, m0, m1, m2, m3, m4, m5, m6, eps);
    return recon<SCHEME>(flag, p0, p1, p2, p3, p4, p5, p6, eps) + recon<SCHEME>(flag, m0, m1, m2, m3, m4, m5, m6, eps);
}

// J at a padded point (the factor of the flux difference, eq. 1)
template <int KIND>
__device__ __forceinline__ double jac_at(const GridDesc &g, int ip, int jp, int kp) {
    if (KIND == OCFD_GRID_UNIFORM) return g.uJ;
    if (KIND == OCFD_GRID_STRETCHED) return (__ldg(g.met[0] + ip) * __ldg(g.met[4] + jp)) * __ldg(g.met[8] + kp);
    return __ldg(g.atab[0] + 4 * g.atab_fs + (long long)kp * g.msk + (long long)jp * g.sy + ip);
}

// ------------------------------------------------------------------------------------------ characteristic variables
// Eigenvector frame of one interface: unit direction n, l by eq. 39, m = n x l (eq. 40), the
// averaged state u, v, w, c (eq. 32) and the scalars of eq. 36.  Row k of S (eq. 35) and column k of S^-1 (eq. 34)
// are produced on demand, so that a thread never holds the two 5 x 5 matrices.
struct CharFrame {
    double u, v, w, c, V, H, un, ul, um, kap, chi;
    double n[3], l[3], m[3];
    __device__ __forceinline__ void set(double gamma, double u_, double v_, double w_, double c_, double n0, double n1,
                                        double n2) {
        u = u_; v = v_; w = w_; c = c_;
        n[0] = n0; n[1] = n1; n[2] = n2;
        if (fabs(n2) <= fabs(n1)) {
            const double r = rsqrt(n0 * n0 + n1 * n1);
            l[0] = -n1 * r; l[1] = n0 * r; l[2] = 0.0;
        } else {
            const double r = rsqrt(n0 * n0 + n2 * n2);
            l[0] = -n2 * r; l[1] = 0.0; l[2] = n0 * r;
        }
        m[0] = n[1] * l[2] - n[2] * l[1]; m[1] = n[2] * l[0] - n[0] * l[2]; m[2] = n[0] * l[1] - n[1] * l[0];
        V = 0.5 * (u * u + v * v + w * w);
        H = V + c * c / (gamma - 1.0);
        un = u * n[0] + v * n[1] + w * n[2]; ul = u * l[0] + v * l[1] + w * l[2]; um = u * m[0] + v * m[1] + w * m[2];
        kap = (gamma - 1.0) / (c * c);
        chi = 0.5 / c;
    }
    // row K of S
    template <int K>
    __device__ __forceinline__ void row(double s[5]) const {
        const double k1 = 0.5 * kap;
        if (K == 0) { s[0] = 1.0 - kap * V; s[1] = kap * u; s[2] = kap * v; s[3] = kap * w; s[4] = -kap; }
        if (K == 1) { s[0] = -ul; s[1] = l[0]; s[2] = l[1]; s[3] = l[2]; s[4] = 0.0; }
        if (K == 2) { s[0] = -um; s[1] = m[0]; s[2] = m[1]; s[3] = m[2]; s[4] = 0.0; }
        if (K == 3) { s[0] = k1 * V + chi * un; s[1] = -chi * n[0] - k1 * u; s[2] = -chi * n[1] - k1 * v; s[3] = -chi * n[2] - k1 * w; s[4] = k1; }
        if (K == 4) { s[0] = k1 * V - chi * un; s[1] = chi * n[0] - k1 * u; s[2] = chi * n[1] - k1 * v; s[3] = chi * n[2] - k1 * w; s[4] = k1; }
    }
    // column K of S^-1
    template <int K>
    __device__ __forceinline__ void col(double r[5]) const {
        if (K == 0) { r[0] = 1.0; r[1] = u; r[2] = v; r[3] = w; r[4] = V; }
        if (K == 1) { r[0] = 0.0; r[1] = l[0]; r[2] = l[1]; r[3] = l[2]; r[4] = ul; }
        if (K == 2) { r[0] = 0.0; r[1] = m[0]; r[2] = m[1]; r[3] = m[2]; r[4] = um; }
        if (K == 3) { r[0] = 1.0; r[1] = u - c * n[0]; r[2] = v - c * n[1]; r[3] = w - c * n[2]; r[4] = H - c * un; }
        if (K == 4) { r[0] = 1.0; r[1] = u + c * n[0]; r[2] = v + c * n[1]; r[3] = w + c * n[2]; r[4] = H + c * un; }
    }
};

// One characteristic component K of one interface (eq. 31): project the split fluxes of the 8 stencil rows with row K
// of S (f+ of rows 0..6, f- of rows 1..7, read from shared memory: fp/fm point at row 0 of component 0, `cs` =
// component stride, `rs` = row stride), reconstruct, and add column K of S^-1 times the result to h[5].
template <int SCHEME, int K>
__device__ __noinline__ void char_component(const CharFrame &F, int flag, bool closure, int s, int n,
                                               const double *fp, const double *fm, int cs, int rs, double eps,
                                               double h[5]) {
    double sk[5], wp[7], wm[7];
    F.row<K>(sk);
#pragma unroll
    for (int r = 0; r < 7; ++r) {
        double a = 0.0, b = 0.0;
#pragma unroll
        for (int q = 0; q < 5; ++q) {
            a = fma(sk[q], fp[q * cs + r * rs], a);
            b = fma(sk[q], fm[q * cs + (r + 1) * rs], b);
        }
        wp[r] = a;
        wm[r] = b;
    }
    const double hw = closure ? recon_pair_closure<SCHEME>(flag, s, n, wp[0], wp[1], wp[2], wp[3], wp[4], wp[5], wp[6],
                                                           wm[6], wm[5], wm[4], wm[3], wm[2], wm[1], wm[0], eps)
                              : recon<SCHEME>(flag, wp[0], wp[1], wp[2], wp[3], wp[4], wp[5], wp[6], eps) +
                                    recon<SCHEME>(flag, wm[6], wm[5], wm[4], wm[3], wm[2], wm[1], wm[0], eps);
    double rk[5];
    F.col<K>(rk);
#pragma unroll
    for (int q = 0; q < 5; ++q) h[q] = fma(rk[q], hw, h[q]);
}

// ------------------------------------------------------------------------------------------ Steger-Warming
// Split fluxes of direction DIR at one point, written to sF[c*cs], c = 0..9 (eq. 19-29 with the
// readings R-4, R-5, R-7).  k = alpha/|alpha| (unit), sigma = |alpha|, alpha = (d_x,d_y,d_z)/J.
//
// With |k| = 1 the bracket of eq. 23-26 collapses: writing A = 2(gamma-1) lam1, S = lam4 + lam5, D = lam5 - lam4,
//   f1   = h (A + S),                      h = rho / (2 gamma)
//   f2-4 = u_i f1 + k_i (h c D)
//   f5   = (q^2/2) f1 + (k.u)(h c D) + (1/2 + (3-gamma)/(2(gamma-1))) c^2 h S
// (expand (u -+ c k)^2/2 = q^2/2 -+ c k.u + c^2/2), which is 15 instructions per sign instead of 37.
template <int KIND, int DIR>
__device__ __forceinline__ void sw_split_store(const GasDesc &gs, double rho, double u, double v, double w, double c,
                                               double k1, double k2, double k3, double sigma,
                                               double *__restrict__ sF, int cs) {
    const double Vn = KIND == OCFD_GRID_CURVILINEAR ? k1 * u + k2 * v + k3 * w
                                                     : (DIR == 0 ? k1 * u : DIR == 1 ? k2 * v : k3 * w);
    const double l1 = sigma * Vn, cs_ = c * sigma;
    const double l4 = l1 - cs_, l5 = l1 + cs_;
    double l1p, l4p, l5p;
    if (gs.sw_eps == 0.0) {  // eq. 29
        l1p = 0.5 * (l1 + fabs(l1)); l4p = 0.5 * (l4 + fabs(l4)); l5p = 0.5 * (l5 + fabs(l5));
    } else {
        const double e2 = gs.sw_eps * gs.sw_eps;
        l1p = 0.5 * (l1 + sqrt(l1 * l1 + e2)); l4p = 0.5 * (l4 + sqrt(l4 * l4 + e2)); l5p = 0.5 * (l5 + sqrt(l5 * l5 + e2));
    }
    const double l1m = l1 - l1p, l4m = l4 - l4p, l5m = l5 - l5p;
    const double h = rho * gs.inv2g;
    const double hq = 0.5 * (u * u + v * v + w * w);
    const double hc = h * c, hcc = hc * (c * gs.w1);
    {
        const double S = l4p + l5p;
        const double f1 = h * (gs.tgm1 * l1p + S), D = hc * (l5p - l4p);
        sF[0] = f1;
        sF[cs] = KIND == OCFD_GRID_CURVILINEAR || DIR == 0 ? u * f1 + k1 * D : u * f1;
        sF[2 * cs] = KIND == OCFD_GRID_CURVILINEAR || DIR == 1 ? v * f1 + k2 * D : v * f1;
        sF[3 * cs] = KIND == OCFD_GRID_CURVILINEAR || DIR == 2 ? w * f1 + k3 * D : w * f1;
        sF[4 * cs] = hq * f1 + (Vn * D + hcc * S);
    }
    {
        const double S = l4m + l5m;
        const double f1 = h * (gs.tgm1 * l1m + S), D = hc * (l5m - l4m);
        sF[5 * cs] = f1;
        sF[6 * cs] = KIND == OCFD_GRID_CURVILINEAR || DIR == 0 ? u * f1 + k1 * D : u * f1;
        sF[7 * cs] = KIND == OCFD_GRID_CURVILINEAR || DIR == 1 ? v * f1 + k2 * D : v * f1;
        sF[8 * cs] = KIND == OCFD_GRID_CURVILINEAR || DIR == 2 ? w * f1 + k3 * D : w * f1;
        sF[9 * cs] = hq * f1 + (Vn * D + hcc * S);
    }
}

}  // namespace
