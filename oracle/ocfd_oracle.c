/*
 * oracle/ocfd_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU restatement of the right-hand side of the finite-difference
 * compressible Navier-Stokes solver described in /root/reference/PAPER.md
 * (arxiv 2209.15333, "OpenCFD-SCU Part 1"), written from the paper's equations.
 * It follows the algorithm step by step in the paper's order and notation: plain loops,
 * no tiling, no fusion, no reordering.  It shares no code with the CUDA path in
 * paper_2209_15333_b200/csrc/ and is only imported by tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs.
 *
 * Compile:  gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC  (see oracle/build.py).
 * No fast-math, no FMA contraction: every operation rounds as written.
 *
 * Citations "PAPER.md:Lnnn" are line numbers of /root/reference/PAPER.md; "DESIGN R-n" are the
 * readings of garbled/silent passages registered in DESIGN.md section 3.
 *
 * Array layout: every 3-D field is a padded box
 * [nz+8][ny+8][nx+8], x contiguous, LAP = 4 ghost layers per face.  Conserved variables
 * U = (rho, rho u, rho v, rho w, E) (eq. 5) are stored component-major
 * [5][nz+8][ny+8][nx+8].  Computational spacing is 1 in xi, eta, zeta.
 *
 * Parity pins (tests/test_oracle_*.py, all run with -m "not gpu"):
 *   ora_ud7                 eq. 41 coefficients printed at PAPER.md:L282 (tests/golden/ud7_eq41.txt)
 *   ora_weno7 / ora_weno5   linear weights reproduce eq. 41 / the 5th-order upwind formula;
 *                           polynomial reproduction; smoothness indicators against brute-force
 *                           quadrature of their integral definition; convexity / ENO property
 *   ora_sw_split            f+ + f- == exact flux of eq. 6; one-sidedness when supersonic;
 *                           eigenvalue signs of the split Jacobians; rotational covariance
 *   ora_d1_line             polynomial exactness of interior and closure rows, 6th and 8th order
 *   viscous terms           manufactured solution differentiated symbolically (sympy), 6th / 8th order
 *   ora_rk3_update          y' = lambda y closed form 1 + z + z^2/2 + z^3/6 (eq. 45)
 *   ora_rhs (whole)         freestream, conservation, isentropic-vortex order, Sod vs exact Riemann,
 *                           skewed-grid equivalence, hybrid limits
 *   ora_weno5_masked        (paper boundary scheme, bc_closure) candidate exactness, renormalised weights, no
 *                           out-of-domain reads; the all-shielded value (DESIGN R-21) is PARITY UNPINNED
 *   ora_max_wavespeed       uniform-flow closed form; brute force
 *   ora_check_state         hand-made fields with known numbers of bad points of each kind (tests/test_oracle_bc.py)
 *   ora_fill_ghosts         BC invariants
 * Unpinned (no data in the container): agreement with the authors' own program output.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#define NG 4 /* LAP */

enum { ORA_UD7 = 0, ORA_WENO7 = 1, ORA_WENO5 = 2, ORA_HYBRID = 3 };
enum { ORA_BC_PERIODIC = 0, ORA_BC_WALL = 1, ORA_BC_INFLOW = 2, ORA_BC_OUTFLOW = 3 };

typedef struct {
    int nx, ny, nz;          /* interior dimensions */
    const double *met[10];   /* xi_x xi_y xi_z eta_x eta_y eta_z zeta_x zeta_y zeta_z J (eq. 3, 4); padded fields */
    long met_sk;             /* k-plane stride of the metric fields in doubles: (nx+8)*(ny+8), or 0 when
                                the grid is a 2-D map extruded in z (one padded plane per metric) */
    double gamma, Ma, Re, Pr, T_ref, T_suth;
    int inviscid;            /* 1: skip viscous terms */
    int scheme;              /* ORA_UD7 / WENO7 / WENO5 / HYBRID */
    double theta1, theta2;   /* hybrid thresholds */
    double weno_eps;         /* DESIGN R-10 */
    double sw_eps;           /* 0 = eq. 29 exactly, DESIGN R-6 */
    int bc[6];               /* x-, x+, y-, y+, z-, z+ */
    double T_wall[6];
    const double *wall_vn[6];
    const double *inflow[6];
    int visc_order;          /* 6 (default; 0 means 6) or 8: order of the central scheme of the viscous terms,
                                PAPER.md:L313 "two such schemes, of sixth and eighth order" */
    int bc_closure;          /* 0: ghost cells feed the full stencils (north_star; DESIGN R-14);
                                1: the paper's boundary scheme, PAPER.md:L307-309 (DESIGN R-20, R-21) */
    int char_recon;          /* 1: flux reconstruction in characteristic variables, PAPER.md:L212-263 (section 2.2.2) */
} ora_params;
static int vorder(const ora_params *P) { return P->visc_order == 8 ? 8 : 6; }

/* ---------------------------------------------------------------- indexing */
static long SX(const ora_params *P) { (void)P; return 1; }
static long SY(const ora_params *P) { return P->nx + 2 * NG; }
static long SZ(const ora_params *P) { return (long)(P->nx + 2 * NG) * (P->ny + 2 * NG); }
static long NP(const ora_params *P) { return SZ(P) * (P->nz + 2 * NG); }
static long IDX(const ora_params *P, int i, int j, int k) {
    return (long)(k + NG) * SZ(P) + (long)(j + NG) * SY(P) + (i + NG);
}
static long MIDX(const ora_params *P, int i, int j, int k) {
    return (long)(k + NG) * P->met_sk + (long)(j + NG) * SY(P) + (i + NG);
}
static int dim_n(const ora_params *P, int d) { return d == 0 ? P->nx : d == 1 ? P->ny : P->nz; }
static long dim_stride(const ora_params *P, int d) { return d == 0 ? SX(P) : d == 1 ? SY(P) : SZ(P); }
static int periodic(const ora_params *P, int d) { return P->bc[2 * d] == ORA_BC_PERIODIC; }

/* ------------------------------------------------- thermodynamics (A.2) */
typedef struct { double rho, u, v, w, p, T, c; } ora_prim;

/* E = p/(gamma-1) + rho q^2/2 (eq. 8 PAPER.md:L113 as corrected, DESIGN R-1);
 * p = rho T/(gamma Ma^2), c^2 = T/Ma^2 (eq. 16). */
static ora_prim prim_of(const ora_params *P, double r, double ru, double rv, double rw, double E) {
    ora_prim q;
    q.rho = r;
    q.u = ru / r;
    q.v = rv / r;
    q.w = rw / r;
    q.p = (P->gamma - 1.0) * (E - 0.5 * r * (q.u * q.u + q.v * q.v + q.w * q.w));
    q.T = P->gamma * P->Ma * P->Ma * q.p / r;
    q.c = sqrt(q.T) / P->Ma;
    return q;
}
static ora_prim prim_at(const ora_params *P, const double *U, long id) {
    long np = NP(P);
    return prim_of(P, U[id], U[np + id], U[2 * np + id], U[3 * np + id], U[4 * np + id]);
}
void ora_prim_point(const ora_params *P, const double U5[5], double out7[7]) {
    ora_prim q = prim_of(P, U5[0], U5[1], U5[2], U5[3], U5[4]);
    out7[0] = q.rho; out7[1] = q.u; out7[2] = q.v; out7[3] = q.w; out7[4] = q.p; out7[5] = q.T; out7[6] = q.c;
}

/* Sutherland, eq. 15 with C = T_suth the Sutherland constant (DESIGN R-8). */
double ora_mu(const ora_params *P, double T) {
    double S = P->T_suth / P->T_ref;
    return (1.0 + S) / (T + S) * T * sqrt(T);
}

/* ----------------------------------------- Steger-Warming split (A.3) */
/* PAPER.md:L161-202, eq. 19-29, with the readings DESIGN R-4, R-5, R-7.
 * alpha = (d_x, d_y, d_z)/J for direction d.  fp = f(lambda+), fm = f(lambda-). */
void ora_sw_split(double gamma, double sw_eps, double rho, double u, double v, double w, double c,
                  double a1, double a2, double a3, double fp[5], double fm[5]) {
    double sigma = sqrt(a1 * a1 + a2 * a2 + a3 * a3);            /* eq. 22 */
    double k1 = a1 / sigma, k2 = a2 / sigma, k3 = a3 / sigma;    /* eq. 27 */
    double Vt = a1 * u + a2 * v + a3 * w;                        /* eq. 21 */
    double lam[3] = { Vt, Vt - c * sigma, Vt + c * sigma };      /* eq. 20: lambda_1, lambda_4, lambda_5 */
    double q2 = u * u + v * v + w * w;
    for (int s = 0; s < 2; ++s) {
        double sgn = s == 0 ? 1.0 : -1.0;
        double l1 = 0.5 * (lam[0] + sgn * sqrt(lam[0] * lam[0] + sw_eps * sw_eps)); /* eq. 29 */
        double l4 = 0.5 * (lam[1] + sgn * sqrt(lam[1] * lam[1] + sw_eps * sw_eps));
        double l5 = 0.5 * (lam[2] + sgn * sqrt(lam[2] * lam[2] + sw_eps * sw_eps));
        double um = u - c * k1, vm = v - c * k2, wm = w - c * k3;
        double up = u + c * k1, vp = v + c * k2, wp = w + c * k3;
        double W = (3.0 - gamma) * (l4 + l5) * c * c / (2.0 * (gamma - 1.0)); /* eq. 26 */
        double vc1 = 0.5 * (um * um + vm * vm + wm * wm);
        double vc2 = 0.5 * (up * up + vp * vp + wp * wp);
        double h = rho / (2.0 * gamma);
        double *f = s == 0 ? fp : fm;
        f[0] = h * (2.0 * (gamma - 1.0) * l1 + l4 + l5);
        f[1] = h * (2.0 * (gamma - 1.0) * l1 * u + l4 * um + l5 * up);
        f[2] = h * (2.0 * (gamma - 1.0) * l1 * v + l4 * vm + l5 * vp);
        f[3] = h * (2.0 * (gamma - 1.0) * l1 * w + l4 * wm + l5 * wp);
        f[4] = h * ((gamma - 1.0) * l1 * q2 + l4 * vc1 + l5 * vc2 + W);
    }
}

/* ----------------------------------------------- reconstructions (A.4-A.5) */
/* All take the POSITIVE-flux orientation: f[0..6] = f_{j-3..j+3}, result at j+1/2.
 * The negative flux is reconstructed by mirroring the stencil about j+1/2. */

/* eq. 41 */
double ora_ud7(const double f[7]) {
    return (-3.0 * f[0] + 25.0 * f[1] - 101.0 * f[2] + 319.0 * f[3] + 214.0 * f[4] - 38.0 * f[5] + 4.0 * f[6]) / 420.0;
}

/* WENO7 of Jiang-Shu type (ref. [21]); formulas derived from the definition
 * (DESIGN R-9): four cubic candidates, linear weights (1,12,18,4)/35, smoothness indicators
 * IS_k = sum_{l=1..3} int_{x_j-1/2}^{x_j+1/2} h^{2l-1} (d^l p_k/dx^l)^2 dx written with the
 * derivatives s1,s2,s3 of candidate k at x_j:  IS = s1^2 + 13/12 s2^2 + 1043/960 s3^2 + s1 s3/12. */
void ora_weno7_parts(const double f[7], double eps, double q[4], double IS[4], double om[4]) {
    static const double C[4] = { 1.0 / 35.0, 12.0 / 35.0, 18.0 / 35.0, 4.0 / 35.0 };
    double s1[4], s2[4], s3[4], al[4], sum = 0.0;
    q[0] = (-3.0 * f[0] + 13.0 * f[1] - 23.0 * f[2] + 25.0 * f[3]) / 12.0;
    q[1] = (f[1] - 5.0 * f[2] + 13.0 * f[3] + 3.0 * f[4]) / 12.0;
    q[2] = (-f[2] + 7.0 * f[3] + 7.0 * f[4] - f[5]) / 12.0;
    q[3] = (3.0 * f[3] + 13.0 * f[4] - 5.0 * f[5] + f[6]) / 12.0;
    s1[0] = (-7.0 * f[0] + 33.0 * f[1] - 69.0 * f[2] + 43.0 * f[3]) / 24.0;
    s2[0] = -f[0] + 4.0 * f[1] - 5.0 * f[2] + 2.0 * f[3];
    s3[0] = -f[0] + 3.0 * f[1] - 3.0 * f[2] + f[3];
    s1[1] = (5.0 * f[1] - 27.0 * f[2] + 15.0 * f[3] + 7.0 * f[4]) / 24.0;
    s2[1] = f[2] - 2.0 * f[3] + f[4];
    s3[1] = -f[1] + 3.0 * f[2] - 3.0 * f[3] + f[4];
    s1[2] = (-7.0 * f[2] - 15.0 * f[3] + 27.0 * f[4] - 5.0 * f[5]) / 24.0;
    s2[2] = f[2] - 2.0 * f[3] + f[4];
    s3[2] = -f[2] + 3.0 * f[3] - 3.0 * f[4] + f[5];
    s1[3] = (-43.0 * f[3] + 69.0 * f[4] - 33.0 * f[5] + 7.0 * f[6]) / 24.0;
    s2[3] = 2.0 * f[3] - 5.0 * f[4] + 4.0 * f[5] - f[6];
    s3[3] = -f[3] + 3.0 * f[4] - 3.0 * f[5] + f[6];
    for (int k = 0; k < 4; ++k) {
        IS[k] = s1[k] * s1[k] + 13.0 / 12.0 * s2[k] * s2[k] + 1043.0 / 960.0 * s3[k] * s3[k] + s1[k] * s3[k] / 12.0;
        al[k] = C[k] / ((eps + IS[k]) * (eps + IS[k]));
        sum += al[k];
    }
    for (int k = 0; k < 4; ++k) om[k] = al[k] / sum;
}
double ora_weno7(const double f[7], double eps) {
    double q[4], IS[4], om[4];
    ora_weno7_parts(f, eps, q, IS, om);
    return om[0] * q[0] + om[1] * q[1] + om[2] * q[2] + om[3] * q[3];
}

/* WENO5 (Jiang-Shu), f[0..4] = f_{j-2..j+2} (A.5). */
void ora_weno5_parts(const double f[5], double eps, double q[3], double IS[3], double om[3]) {
    static const double C[3] = { 0.1, 0.6, 0.3 };
    double al[3], sum = 0.0, a, b;
    q[0] = (2.0 * f[0] - 7.0 * f[1] + 11.0 * f[2]) / 6.0;
    q[1] = (-f[1] + 5.0 * f[2] + 2.0 * f[3]) / 6.0;
    q[2] = (2.0 * f[2] + 5.0 * f[3] - f[4]) / 6.0;
    a = f[0] - 2.0 * f[1] + f[2]; b = f[0] - 4.0 * f[1] + 3.0 * f[2];
    IS[0] = 13.0 / 12.0 * a * a + 0.25 * b * b;
    a = f[1] - 2.0 * f[2] + f[3]; b = f[1] - f[3];
    IS[1] = 13.0 / 12.0 * a * a + 0.25 * b * b;
    a = f[2] - 2.0 * f[3] + f[4]; b = 3.0 * f[2] - 4.0 * f[3] + f[4];
    IS[2] = 13.0 / 12.0 * a * a + 0.25 * b * b;
    for (int k = 0; k < 3; ++k) { al[k] = C[k] / ((eps + IS[k]) * (eps + IS[k])); sum += al[k]; }
    for (int k = 0; k < 3; ++k) om[k] = al[k] / sum;
}
double ora_weno5(const double f[5], double eps) {
    double q[3], IS[3], om[3];
    ora_weno5_parts(f, eps, q, IS, om);
    return om[0] * q[0] + om[1] * q[1] + om[2] * q[2];
}

/* scheme of one interface: 0 UD7, 1 WENO7, 2 WENO5.  Theta = max(theta_j, theta_j+1)
 * (DESIGN R-12); Theta <= theta1 -> UD7; theta1 < Theta <= theta2 -> WENO7; else WENO5 (R-11). */
static int iface_scheme(const ora_params *P, double th_a, double th_b) {
    if (P->scheme != ORA_HYBRID) return P->scheme;
    double Th = th_a > th_b ? th_a : th_b;
    if (Th <= P->theta1) return ORA_UD7;
    if (Th <= P->theta2) return ORA_WENO7;
    return ORA_WENO5;
}
/* one numerical flux value from a 7-point window already oriented upwind */
static double recon(int scheme, const double f[7], double eps) {
    if (scheme == ORA_UD7) return ora_ud7(f);
    if (scheme == ORA_WENO7) return ora_weno7(f, eps);
    return ora_weno5(f + 1, eps);
}

/* ------------------------------------- central first derivative (A.7) */
/* 6th-order central.  f points at element 0 of a line with stride st.
 * Periodic axis: neighbours are read through the stride (ghost or wrapped values must be
 * there; see callers).  Aperiodic axis of length n: one-sided 2nd order at the boundary
 * point, 2nd / 4th order central at the 2nd / 3rd point, no ghost used. */
static double d1_interior(const double *f, long st) {
    return (45.0 * (f[st] - f[-st]) - 9.0 * (f[2 * st] - f[-2 * st]) + (f[3 * st] - f[-3 * st])) / 60.0;
}
/* 8th-order central (the second scheme of PAPER.md:L313; the standard coefficients 4/5, -1/5, 4/105, -1/280 of the
 * 9-point antisymmetric stencil, pinned by polynomial exactness up to degree 8) */
static double d1_interior8(const double *f, long st) {
    return (672.0 * (f[st] - f[-st]) - 168.0 * (f[2 * st] - f[-2 * st]) + 32.0 * (f[3 * st] - f[-3 * st])
            - 3.0 * (f[4 * st] - f[-4 * st])) / 840.0;
}
static double d1_int(const double *f, long st, int order) {
    return order == 8 ? d1_interior8(f, st) : d1_interior(f, st);
}
/* aperiodic axis: "second-order unilateral at the boundary point, second-, fourth- and sixth-order
 * central at the second, third and fourth boundary points"; the fourth row only exists for the 8th-order scheme
 * (for the 6th-order scheme the fourth point already takes the interior stencil) */
static double d1_closure(const double *f, long st, int s, int n, int order) {
    /* f points at element s of the line */
    if (s == 0) return (-3.0 * f[0] + 4.0 * f[st] - f[2 * st]) / 2.0;
    if (s == n - 1) return (3.0 * f[0] - 4.0 * f[-st] + f[-2 * st]) / 2.0;
    if (s == 1 || s == n - 2) return (f[st] - f[-st]) / 2.0;
    if (s == 2 || s == n - 3) return (8.0 * (f[st] - f[-st]) - (f[2 * st] - f[-2 * st])) / 12.0;
    if (order == 8 && (s == 3 || s == n - 4)) return d1_interior(f, st);
    return d1_int(f, st, order);
}
/* derivative of a whole line, for the pins; periodic lines wrap */
void ora_d1_line(const double *f, int n, int is_periodic, int order, double *out) {
    for (int s = 0; s < n; ++s) {
        if (is_periodic) {
            double w[9];
            for (int m = -4; m <= 4; ++m) w[m + 4] = f[((s + m) % n + n) % n];
            out[s] = d1_int(w + 4, 1, order == 8 ? 8 : 6);
        } else {
            out[s] = d1_closure(f + s, 1, s, n, order == 8 ? 8 : 6);
        }
    }
}

/* --------------------------------------------------- ghost fill (A.8) */
/* The paper gives no formulas; DESIGN R-16 defines them.
 * Faces are processed in the order x-, x+, y-, y+, z-, z+: first all Dirichlet nodes
 * (wall, inflow), then all ghost layers.  Only face ghosts are written (no edges/corners). */
static void face_axes(int f, int *d, int *t1, int *t2) {
    *d = f / 2;
    *t1 = *d == 0 ? 1 : 0; /* fast tangential axis */
    *t2 = *d == 2 ? 1 : 2; /* slow tangential axis */
}
static void set_cons(const ora_params *P, double *U, long id, double rho, double u, double v, double w, double p) {
    long np = NP(P);
    U[id] = rho;
    U[np + id] = rho * u;
    U[2 * np + id] = rho * v;
    U[3 * np + id] = rho * w;
    U[4 * np + id] = p / (P->gamma - 1.0) + 0.5 * rho * (u * u + v * v + w * w);
}
void ora_fill_ghosts(const ora_params *P, double *U) {
    long np = NP(P);
    double gM2 = P->gamma * P->Ma * P->Ma;
    for (int pass = 0; pass < 2; ++pass)
        for (int f = 0; f < 6; ++f) {
            int d, t1, t2;
            face_axes(f, &d, &t1, &t2);
            int n = dim_n(P, d), n1 = dim_n(P, t1), n2 = dim_n(P, t2);
            long sd = dim_stride(P, d), s1 = dim_stride(P, t1), s2 = dim_stride(P, t2);
            int lo = (f % 2 == 0);
            long in = lo ? sd : -sd;            /* step into the domain */
            int b = lo ? 0 : n - 1;             /* boundary node along d */
            long pitch2 = n1 + 2 * NG;          /* padded 2-D face arrays: [n2+8][n1+8] */
            for (int c2 = 0; c2 < n2; ++c2)
                for (int c1 = 0; c1 < n1; ++c1) {
                    long id0 = (long)NG * (SX(P) + SY(P) + SZ(P)) + (long)b * sd + (long)c1 * s1 + (long)c2 * s2;
                    long fid = (long)(c2 + NG) * pitch2 + (c1 + NG);
                    long fnp = (long)(n2 + 2 * NG) * pitch2;
                    int bc = P->bc[f];
                    if (pass == 0) { /* Dirichlet nodes */
                        if (bc == ORA_BC_WALL) {
                            ora_prim q1 = prim_at(P, U, id0 + in), q2 = prim_at(P, U, id0 + 2 * in);
                            double p0 = (4.0 * q1.p - q2.p) / 3.0;
                            double Tw = P->T_wall[f];
                            double rho0 = gM2 * p0 / Tw;
                            double u = 0.0, v = 0.0, w = 0.0;
                            if (P->wall_vn[f]) { /* (u,v,w) = v_n * unit normal into the fluid */
                                int i = (int)((id0 % SY(P))) - NG, j = (int)((id0 / SY(P)) % (P->ny + 2 * NG)) - NG,
                                    k = (int)(id0 / SZ(P)) - NG;
                                long mi = MIDX(P, i, j, k);
                                double a1 = P->met[3 * d][mi], a2 = P->met[3 * d + 1][mi], a3 = P->met[3 * d + 2][mi];
                                double s = sqrt(a1 * a1 + a2 * a2 + a3 * a3), sg = lo ? 1.0 : -1.0;
                                double vn = P->wall_vn[f][fid];
                                u = vn * sg * a1 / s; v = vn * sg * a2 / s; w = vn * sg * a3 / s;
                            }
                            set_cons(P, U, id0, rho0, u, v, w, p0);
                        } else if (bc == ORA_BC_INFLOW) {
                            for (int m = 0; m < 5; ++m) U[m * np + id0] = P->inflow[f][m * fnp + fid];
                        }
                    } else { /* ghost layers */
                        for (int g = 1; g <= NG; ++g) {
                            long idg = id0 - g * in;
                            if (bc == ORA_BC_PERIODIC) {
                                long src = idg + (lo ? (long)n * sd : -(long)n * sd);
                                for (int m = 0; m < 5; ++m) U[m * np + idg] = U[m * np + src];
                            } else if (bc == ORA_BC_OUTFLOW) {
                                for (int m = 0; m < 5; ++m) U[m * np + idg] = U[m * np + id0];
                            } else if (bc == ORA_BC_INFLOW) {
                                for (int m = 0; m < 5; ++m) U[m * np + idg] = P->inflow[f][m * fnp + fid];
                            } else { /* wall: u mirrored about the wall value, T about T_w, p even */
                                ora_prim q0 = prim_at(P, U, id0), qm = prim_at(P, U, id0 + g * in);
                                double Tw = P->T_wall[f];
                                double u = 2.0 * q0.u - qm.u, v = 2.0 * q0.v - qm.v, w = 2.0 * q0.w - qm.w;
                                double T = 2.0 * Tw - qm.T, p = qm.p;
                                set_cons(P, U, idg, gM2 * p / T, u, v, w, p);
                            }
                        }
                    }
                }
        }
}

/* ------------------------------------------------ shock sensor (A.6) */
/* eq. 42 with theta = phi_i + phi_j + phi_k (DESIGN R-11) at interior
 * points; ghosts of theta: periodic wrap, else copy of the nearest interior value (R-12).
 * theta is a padded field; points that are not interior or face ghosts are left untouched. */
static double phi_of(double pm, double p0, double pp) { return fabs(-pm + 2.0 * p0 - pp) / (pm + 2.0 * p0 + pp); }
static double theta_point(const ora_params *P, const double *U, int i, int j, int k) {
    long id = IDX(P, i, j, k);
    double p0 = prim_at(P, U, id).p, th = 0.0;
    for (int d = 0; d < 3; ++d) {
        long st = dim_stride(P, d);
        th += phi_of(prim_at(P, U, id - st).p, p0, prim_at(P, U, id + st).p);
    }
    return th;
}
/* theta at a point that may lie in a face-ghost layer of direction d (index s along d) */
static double theta_ext(const ora_params *P, const double *U, int d, int i, int j, int k) {
    int c[3] = { i, j, k };
    int n = dim_n(P, d);
    if (c[d] < 0) c[d] = periodic(P, d) ? c[d] + n : 0;
    else if (c[d] >= n) c[d] = periodic(P, d) ? c[d] - n : n - 1;
    return theta_point(P, U, c[0], c[1], c[2]);
}
void ora_sensor(const ora_params *P, const double *U, double *theta) {
#pragma omp parallel for collapse(2)
    for (int k = 0; k < P->nz; ++k)
        for (int j = 0; j < P->ny; ++j)
            for (int i = 0; i < P->nx; ++i) theta[IDX(P, i, j, k)] = theta_point(P, U, i, j, k);
    for (int d = 0; d < 3; ++d) {
        int n = dim_n(P, d);
        for (int k = (d == 2 ? -NG : 0); k < (d == 2 ? P->nz + NG : P->nz); ++k)
            for (int j = (d == 1 ? -NG : 0); j < (d == 1 ? P->ny + NG : P->ny); ++j)
                for (int i = (d == 0 ? -NG : 0); i < (d == 0 ? P->nx + NG : P->nx); ++i) {
                    int c[3] = { i, j, k };
                    if (c[d] >= 0 && c[d] < n) continue;
                    int s[3] = { i, j, k };
                    s[d] = c[d] < 0 ? (periodic(P, d) ? c[d] + n : 0) : (periodic(P, d) ? c[d] - n : n - 1);
                    theta[IDX(P, i, j, k)] = theta[IDX(P, s[0], s[1], s[2])];
                }
    }
}
/* flag[IDX(point s)] = scheme of interface s+1/2 along d, s = -1 .. n-1 */
void ora_flags(const ora_params *P, const double *theta, int d, unsigned char *flag) {
    long st = dim_stride(P, d);
    int n = dim_n(P, d);
    int lo[3] = { 0, 0, 0 }, hi[3] = { P->nx, P->ny, P->nz };
    lo[d] = -1; hi[d] = n;
    for (int k = lo[2]; k < hi[2]; ++k)
        for (int j = lo[1]; j < hi[1]; ++j)
            for (int i = lo[0]; i < hi[0]; ++i) {
                long id = IDX(P, i, j, k);
                flag[id] = (unsigned char)iface_scheme(P, theta[id], theta[id + st]);
            }
}

/* ------------------------------------------- inviscid term, one direction */
/* split fluxes of direction d at a point (interior or face ghost of direction d) */
static void split_at(const ora_params *P, const double *U, int d, int i, int j, int k, double fp[5], double fm[5]) {
    ora_prim q = prim_at(P, U, IDX(P, i, j, k));
    long mi = MIDX(P, i, j, k);
    double J = P->met[9][mi];
    double a1 = P->met[3 * d][mi] / J, a2 = P->met[3 * d + 1][mi] / J, a3 = P->met[3 * d + 2][mi] / J;
    ora_sw_split(P->gamma, P->sw_eps, q.rho, q.u, q.v, q.w, q.c, a1, a2, a3, fp, fm);
}
/* Paper's boundary scheme: "uses the fifth-order WENO scheme to calculate the numerical flux near
 * the boundary.  When a subtemplate of the WENO scheme uses grid points outside the boundary, the weight of the
 * subtemplate is forced to 0".  f[0..4] is the upwind-oriented WENO5 window, keep bit k set = candidate k lies inside
 * the domain.  Candidates that are shielded are not evaluated at all (no value outside the domain is read).  If every
 * candidate is shielded (the interface on the boundary itself, for the flux whose upwind side is outside) the value
 * of the boundary node `nearest` is taken (DESIGN R-21; the paper is silent). */
double ora_weno5_masked(const double f[5], double eps, int keep, double nearest) {
    static const double C[3] = { 0.1, 0.6, 0.3 };
    double q[3] = { 0, 0, 0 }, al[3] = { 0, 0, 0 }, sum = 0.0, a, b, IS;
    if ((keep & 7) == 0) return nearest;
    if (keep & 1) {
        q[0] = (2.0 * f[0] - 7.0 * f[1] + 11.0 * f[2]) / 6.0;
        a = f[0] - 2.0 * f[1] + f[2]; b = f[0] - 4.0 * f[1] + 3.0 * f[2];
        IS = 13.0 / 12.0 * a * a + 0.25 * b * b;
        al[0] = C[0] / ((eps + IS) * (eps + IS));
    }
    if (keep & 2) {
        q[1] = (-f[1] + 5.0 * f[2] + 2.0 * f[3]) / 6.0;
        a = f[1] - 2.0 * f[2] + f[3]; b = f[1] - f[3];
        IS = 13.0 / 12.0 * a * a + 0.25 * b * b;
        al[1] = C[1] / ((eps + IS) * (eps + IS));
    }
    if (keep & 4) {
        q[2] = (2.0 * f[2] + 5.0 * f[3] - f[4]) / 6.0;
        a = f[2] - 2.0 * f[3] + f[4]; b = 3.0 * f[2] - 4.0 * f[3] + f[4];
        IS = 13.0 / 12.0 * a * a + 0.25 * b * b;
        al[2] = C[2] / ((eps + IS) * (eps + IS));
    }
    sum = al[0] + al[1] + al[2];
    return (al[0] / sum) * q[0] + (al[1] / sum) * q[1] + (al[2] / sum) * q[2];
}
static int inside3(int a, int n) { return a >= 0 && a + 2 <= n - 1; } /* points a, a+1, a+2 all in [0, n-1] */
/* numerical flux h_{s+1/2}[5] along direction d, from the split fluxes of the 8 points s-3..s+4
 * (fp, fm are [8][5], row r = point s-3+r). f+ uses s-3..s+3; f- uses the mirror s+4..s-2.
 * closure != 0 (aperiodic axis of n points with the paper's boundary scheme, DESIGN R-20): a flux whose 7-point
 * stencil reaches outside [0, n-1] is replaced by the shielded WENO5 above, separately for f+ and f-. */
static void iface_flux(int scheme, double eps, const double fp[8][5], const double fm[8][5], double h[5],
                       int closure, int s, int n) {
    const int near_p = closure && (s - 3 < 0 || s + 3 > n - 1);
    const int near_m = closure && (s - 2 < 0 || s + 4 > n - 1);
    /* f+ candidates {s-2,s-1,s}, {s-1,s,s+1}, {s,s+1,s+2}; f- (mirrored) {s+3,s+2,s+1}, {s+2,s+1,s}, {s+1,s,s-1} */
    const int keep_p = inside3(s - 2, n) | inside3(s - 1, n) << 1 | inside3(s, n) << 2;
    const int keep_m = inside3(s + 1, n) | inside3(s, n) << 1 | inside3(s - 1, n) << 2;
    const int np_ = s < 0 ? 0 : s > n - 1 ? n - 1 : s;             /* boundary node nearest to the upwind side of f+ */
    const int nm_ = s + 1 < 0 ? 0 : s + 1 > n - 1 ? n - 1 : s + 1; /* ... of f- */
    for (int m = 0; m < 5; ++m) {
        double a[7], b[7];
        for (int r = 0; r < 7; ++r) { a[r] = fp[r][m]; b[r] = fm[7 - r][m]; }
        const double hp = near_p ? ora_weno5_masked(a + 1, eps, keep_p, fp[np_ - (s - 3)][m]) : recon(scheme, a, eps);
        const double hm = near_m ? ora_weno5_masked(b + 1, eps, keep_m, fm[nm_ - (s - 3)][m]) : recon(scheme, b, eps);
        h[m] = hp + hm;
    }
}
/* ---------------------------------- reconstruction in characteristic variables (section 2.2.2) */
/* Left / right eigenvector matrices S (eq. 35) and S^-1 (eq. 34) of the flux Jacobian in the unit direction n, for
 * the state (u, v, w, c); V = q^2/2 (eq. 25), H = V + c^2/(gamma-1), kappa = (gamma-1)/c^2, kappa1 = kappa/2,
 * chi = 1/(2c) (eq. 36); l by eq. 39, m = n x l (eq. 40). */
void ora_eigen_matrices(double gamma, double u, double v, double w, double c, const double n[3], double S[5][5],
                        double Si[5][5]) {
    double l[3], m[3];
    if (fabs(n[2]) <= fabs(n[1])) {
        double r = sqrt(n[0] * n[0] + n[1] * n[1]);
        l[0] = -n[1] / r; l[1] = n[0] / r; l[2] = 0.0;
    } else {
        double r = sqrt(n[0] * n[0] + n[2] * n[2]);
        l[0] = -n[2] / r; l[1] = 0.0; l[2] = n[0] / r;
    }
    m[0] = n[1] * l[2] - n[2] * l[1]; m[1] = n[2] * l[0] - n[0] * l[2]; m[2] = n[0] * l[1] - n[1] * l[0];
    const double V = 0.5 * (u * u + v * v + w * w), H = V + c * c / (gamma - 1.0);
    const double un = u * n[0] + v * n[1] + w * n[2], ul = u * l[0] + v * l[1] + w * l[2], um = u * m[0] + v * m[1] + w * m[2];
    const double kap = (gamma - 1.0) / (c * c), k1 = 0.5 * kap, chi = 1.0 / (2.0 * c);
    const double vel[3] = { u, v, w };
    /* S^-1: columns are the right eigenvectors (eq. 34) */
    Si[0][0] = 1.0; Si[0][1] = 0.0; Si[0][2] = 0.0; Si[0][3] = 1.0; Si[0][4] = 1.0;
    for (int r = 0; r < 3; ++r) {
        Si[r + 1][0] = vel[r]; Si[r + 1][1] = l[r]; Si[r + 1][2] = m[r];
        Si[r + 1][3] = vel[r] - c * n[r]; Si[r + 1][4] = vel[r] + c * n[r];
    }
    Si[4][0] = V; Si[4][1] = ul; Si[4][2] = um; Si[4][3] = H - c * un; Si[4][4] = H + c * un;
    /* S: rows are the left eigenvectors (eq. 35) */
    S[0][0] = 1.0 - kap * V; S[0][4] = -kap;
    S[1][0] = -ul; S[1][4] = 0.0;
    S[2][0] = -um; S[2][4] = 0.0;
    S[3][0] = k1 * V + chi * un; S[3][4] = k1;
    S[4][0] = k1 * V - chi * un; S[4][4] = k1;
    for (int r = 0; r < 3; ++r) {
        S[0][r + 1] = kap * vel[r];
        S[1][r + 1] = l[r];
        S[2][r + 1] = m[r];
        S[3][r + 1] = -chi * n[r] - k1 * vel[r];
        S[4][r + 1] = chi * n[r] - k1 * vel[r];
    }
}
/* S, S^-1 of interface s+1/2 along d: state from the simple average of the conserved variables of its two points
 * (eq. 32); direction n = (alpha_s + alpha_s+1) normalised, alpha = grad(d)/J (the paper does not say where the
 * metrics of the interface come from: DESIGN R-22). */
static void iface_eigen(const ora_params *P, const double *U, int d, const int c0[3], double S[5][5], double Si[5][5]) {
    int c1[3] = { c0[0], c0[1], c0[2] };
    c1[d] += 1;
    long np = NP(P), ia = IDX(P, c0[0], c0[1], c0[2]), ib = IDX(P, c1[0], c1[1], c1[2]);
    double Ua[5], n[3] = { 0, 0, 0 };
    for (int m = 0; m < 5; ++m) Ua[m] = 0.5 * (U[m * np + ia] + U[m * np + ib]);
    ora_prim q = prim_of(P, Ua[0], Ua[1], Ua[2], Ua[3], Ua[4]);
    long ma = MIDX(P, c0[0], c0[1], c0[2]), mb = MIDX(P, c1[0], c1[1], c1[2]);
    for (int r = 0; r < 3; ++r) n[r] = P->met[3 * d + r][ma] / P->met[9][ma] + P->met[3 * d + r][mb] / P->met[9][mb];
    double len = sqrt(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]);
    for (int r = 0; r < 3; ++r) n[r] /= len;
    ora_eigen_matrices(P->gamma, q.u, q.v, q.w, q.c, n, S, Si);
}
/* iface_flux in characteristic variables (eq. 31): the split fluxes of every stencil point are projected with the S
 * of the interface, each characteristic component is reconstructed by the scheme, the sum is projected back. */
static void iface_flux_char(int scheme, double eps, const double fp[8][5], const double fm[8][5], double h[5],
                            int closure, int s, int n, const double S[5][5], const double Si[5][5]) {
    double wp[8][5], wm[8][5], hw[5];
    for (int r = 0; r < 8; ++r)
        for (int k = 0; k < 5; ++k) {
            double a = 0.0, b = 0.0;
            for (int m = 0; m < 5; ++m) { a += S[k][m] * fp[r][m]; b += S[k][m] * fm[r][m]; }
            wp[r][k] = a; wm[r][k] = b;
        }
    iface_flux(scheme, eps, (const double(*)[5])wp, (const double(*)[5])wm, hw, closure, s, n);
    for (int m = 0; m < 5; ++m) {
        double a = 0.0;
        for (int k = 0; k < 5; ++k) a += Si[m][k] * hw[k];
        h[m] = a;
    }
}
static int closure_on(const ora_params *P, int d) { return P->bc_closure && !periodic(P, d); }
/* dU -= J (h_{s+1/2} - h_{s-1/2}) over all interior points, direction d  (A.1, A.6) */
static void inviscid_dir(const ora_params *P, const double *U, const double *theta, int d, double *dU) {
    long np = NP(P);
    int n = dim_n(P, d);
    int t1 = d == 0 ? 1 : 0, t2 = d == 2 ? 1 : 2;
    int n1 = dim_n(P, t1), n2 = dim_n(P, t2);
#pragma omp parallel
    {
        double(*fp)[5] = malloc(sizeof(double[5]) * (n + 2 * NG));
        double(*fm)[5] = malloc(sizeof(double[5]) * (n + 2 * NG));
        double(*h)[5] = malloc(sizeof(double[5]) * (n + 1));
#pragma omp for collapse(2)
        for (int c2 = 0; c2 < n2; ++c2)
            for (int c1 = 0; c1 < n1; ++c1) {
                int c[3];
                c[t1] = c1; c[t2] = c2;
                for (int s = -NG; s < n + NG; ++s) {
                    c[d] = s;
                    split_at(P, U, d, c[0], c[1], c[2], fp[s + NG], fm[s + NG]);
                }
                for (int s = -1; s < n; ++s) { /* interface s+1/2 */
                    c[d] = s;
                    long id = IDX(P, c[0], c[1], c[2]);
                    int sch = P->scheme == ORA_HYBRID ? iface_scheme(P, theta[id], theta[id + dim_stride(P, d)]) : P->scheme;
                    if (P->char_recon) {
                        double S[5][5], Si[5][5];
                        iface_eigen(P, U, d, c, S, Si);
                        iface_flux_char(sch, P->weno_eps, (const double(*)[5])(fp + (s - 3 + NG)),
                                        (const double(*)[5])(fm + (s - 3 + NG)), h[s + 1], closure_on(P, d), s, n,
                                        (const double(*)[5])S, (const double(*)[5])Si);
                    } else
                        iface_flux(sch, P->weno_eps, (const double(*)[5])(fp + (s - 3 + NG)),
                                   (const double(*)[5])(fm + (s - 3 + NG)), h[s + 1], closure_on(P, d), s, n);
                }
                for (int s = 0; s < n; ++s) {
                    c[d] = s;
                    long id = IDX(P, c[0], c[1], c[2]);
                    double J = P->met[9][MIDX(P, c[0], c[1], c[2])];
                    for (int m = 0; m < 5; ++m) dU[m * np + id] -= J * (h[s + 1][m] - h[s][m]);
                }
            }
        free(fp); free(fm); free(h);
    }
}

/* ------------------------------------------------- viscous terms (A.7) */
/* Viscous fluxes (rows 2-5 of eq. 9-11) at one point from the twelve
 * computational-space derivatives g[phi][d] of phi = u,v,w,T, the metrics m[9], J, and u,v,w,T.
 * out[d][r], d = xi,eta,zeta, r = 0..3 (momentum x,y,z and energy rows). */
void ora_viscous_flux_point(const ora_params *P, const double g[4][3], const double m[9], double J,
                            double u, double v, double w, double T, double out[3][4]) {
    double gx[4], gy[4], gz[4];
    for (int a = 0; a < 4; ++a) { /* chain rule */
        gx[a] = m[0] * g[a][0] + m[3] * g[a][1] + m[6] * g[a][2];
        gy[a] = m[1] * g[a][0] + m[4] * g[a][1] + m[7] * g[a][2];
        gz[a] = m[2] * g[a][0] + m[5] * g[a][1] + m[8] * g[a][2];
    }
    double mu = ora_mu(P, T) / P->Re;                                            /* mu/Re */
    double kc = ora_mu(P, T) / ((P->gamma - 1.0) * P->Ma * P->Ma * P->Pr * P->Re); /* eq. 14 */
    double div = gx[0] + gy[1] + gz[2];
    double txx = mu * (2.0 * gx[0] - 2.0 / 3.0 * div);                            /* eq. 13 */
    double tyy = mu * (2.0 * gy[1] - 2.0 / 3.0 * div);
    double tzz = mu * (2.0 * gz[2] - 2.0 / 3.0 * div);
    double txy = mu * (gy[0] + gx[1]);
    double txz = mu * (gz[0] + gx[2]);
    double tyz = mu * (gz[1] + gy[2]);
    double Thx = u * txx + v * txy + w * txz + kc * gx[3];                        /* eq. 12, DESIGN R-2 */
    double Thy = u * txy + v * tyy + w * tyz + kc * gy[3];
    double Thz = u * txz + v * tyz + w * tzz + kc * gz[3];
    for (int d = 0; d < 3; ++d) {
        double dx = m[3 * d], dy = m[3 * d + 1], dz = m[3 * d + 2];
        out[d][0] = (dx * txx + dy * txy + dz * txz) / J;
        out[d][1] = (dx * txy + dy * tyy + dz * tyz) / J;
        out[d][2] = (dx * txz + dy * tyz + dz * tzz) / J;
        out[d][3] = (dx * Thx + dy * Thy + dz * Thz) / J;
    }
}
/* first derivative along d of a padded field at interior point (i,j,k) following A.7:
 * periodic axis -> interior stencil through ghost values; aperiodic -> closure rows. */
static double d1_field(const ora_params *P, const double *f, int d, int i, int j, int k) {
    long id = IDX(P, i, j, k), st = dim_stride(P, d);
    int s = d == 0 ? i : d == 1 ? j : k;
    return periodic(P, d) ? d1_int(f + id, st, vorder(P)) : d1_closure(f + id, st, s, dim_n(P, d), vorder(P));
}
/* pass 1 at one interior point: prim arrays pu,pv,pw,pT are padded fields valid on interior+face ghosts */
static void viscous_flux_at(const ora_params *P, const double *pu, const double *pv, const double *pw,
                            const double *pT, int i, int j, int k, double out[3][4]) {
    const double *ph[4] = { pu, pv, pw, pT };
    double g[4][3], m[9];
    for (int a = 0; a < 4; ++a)
        for (int d = 0; d < 3; ++d) g[a][d] = d1_field(P, ph[a], d, i, j, k);
    long mi = MIDX(P, i, j, k), id = IDX(P, i, j, k);
    for (int q = 0; q < 9; ++q) m[q] = P->met[q][mi];
    ora_viscous_flux_point(P, g, m, P->met[9][mi], pu[id], pv[id], pw[id], pT[id], out);
}

/* ------------------------------------------------------- whole RHS (A.1) */
/* dU = L(U) on interior points; ghosts of U must be valid (ora_fill_ghosts); ghosts of dU are
 * left untouched.  Order of accumulation: 0, -xi, -eta, -zeta inviscid, + viscous.
 * work: optional; if non-NULL must hold 17 padded fields (4 prims + 12 Fv + theta). */
void ora_rhs(const ora_params *P, const double *U, double *dU) {
    long np = NP(P);
    double *theta = NULL;
    for (int m = 0; m < 5; ++m)
        for (int k = 0; k < P->nz; ++k)
            for (int j = 0; j < P->ny; ++j)
                for (int i = 0; i < P->nx; ++i) dU[m * np + IDX(P, i, j, k)] = 0.0;
    if (P->scheme == ORA_HYBRID) {
        theta = malloc(sizeof(double) * np);
        ora_sensor(P, U, theta);
    }
    for (int d = 0; d < 3; ++d) inviscid_dir(P, U, theta, d, dU);
    free(theta);
    if (P->inviscid) return;

    /* primitives u,v,w,T on interior + face ghosts (NaN elsewhere so that misuse shows) */
    double *pr = malloc(sizeof(double) * 4 * np);
    double *Fv = malloc(sizeof(double) * 12 * np);
    for (long q = 0; q < 4 * np; ++q) pr[q] = NAN;
    for (long q = 0; q < 12 * np; ++q) Fv[q] = NAN;
#pragma omp parallel for collapse(2)
    for (int k = -NG; k < P->nz + NG; ++k)
        for (int j = -NG; j < P->ny + NG; ++j)
            for (int i = -NG; i < P->nx + NG; ++i) {
                int out = (i < 0 || i >= P->nx) + (j < 0 || j >= P->ny) + (k < 0 || k >= P->nz);
                if (out > 1) continue;
                long id = IDX(P, i, j, k);
                ora_prim q = prim_at(P, U, id);
                pr[id] = q.u; pr[np + id] = q.v; pr[2 * np + id] = q.w; pr[3 * np + id] = q.T;
            }
    /* pass 1: viscous fluxes at interior points */
#pragma omp parallel for collapse(2)
    for (int k = 0; k < P->nz; ++k)
        for (int j = 0; j < P->ny; ++j)
            for (int i = 0; i < P->nx; ++i) {
                double o[3][4];
                viscous_flux_at(P, pr, pr + np, pr + 2 * np, pr + 3 * np, i, j, k, o);
                long id = IDX(P, i, j, k);
                for (int d = 0; d < 3; ++d)
                    for (int r = 0; r < 4; ++r) Fv[(4 * d + r) * np + id] = o[d][r];
            }
    /* periodic axes: wrap the flux of that direction into the ghost layers its stencil reaches (3 or 4) */
    const int H = vorder(P) / 2;
    for (int d = 0; d < 3; ++d) {
        if (!periodic(P, d)) continue;
        int n = dim_n(P, d);
        for (int k = (d == 2 ? -H : 0); k < (d == 2 ? P->nz + H : P->nz); ++k)
            for (int j = (d == 1 ? -H : 0); j < (d == 1 ? P->ny + H : P->ny); ++j)
                for (int i = (d == 0 ? -H : 0); i < (d == 0 ? P->nx + H : P->nx); ++i) {
                    int c[3] = { i, j, k };
                    if (c[d] >= 0 && c[d] < n) continue;
                    int s[3] = { i, j, k };
                    s[d] = c[d] < 0 ? c[d] + n : c[d] - n;
                    for (int r = 0; r < 4; ++r)
                        Fv[(4 * d + r) * np + IDX(P, i, j, k)] = Fv[(4 * d + r) * np + IDX(P, s[0], s[1], s[2])];
                }
    }
    /* pass 2: dU += J (D_xi Fv + D_eta Gv + D_zeta Hv), rows 2-5 (row 1 is zero) */
#pragma omp parallel for collapse(2)
    for (int k = 0; k < P->nz; ++k)
        for (int j = 0; j < P->ny; ++j)
            for (int i = 0; i < P->nx; ++i) {
                long id = IDX(P, i, j, k);
                double J = P->met[9][MIDX(P, i, j, k)];
                for (int r = 0; r < 4; ++r) {
                    double s = 0.0;
                    for (int d = 0; d < 3; ++d) s += d1_field(P, Fv + (4 * d + r) * np, d, i, j, k);
                    dU[(r + 1) * np + id] += J * s;
                }
            }
    free(pr); free(Fv);
}

/* Same L(U) at ONE interior point, computed from U alone with no stored intermediates, for sampled
 * parity on grids too large for ora_rhs.  tests/ check that it equals ora_rhs bit for bit. */
static void fv_dir_at(const ora_params *P, const double *U, int d, int i, int j, int k, double out4[4]) {
    /* viscous flux of direction d at interior point (i,j,k), derivatives straight from U */
    double g[4][3], m[9];
    for (int e = 0; e < 3; ++e) {
        long st = dim_stride(P, e);
        int s = e == 0 ? i : e == 1 ? j : k, n = dim_n(P, e);
        double line[4][9]; /* u,v,w,T at offsets -H..H along e (only those the stencil touches) */
        const int H = vorder(P) / 2;
        int lo = -H, hi = H;
        if (!periodic(P, e)) { if (s + lo < 0) lo = -s; if (s + hi > n - 1) hi = n - 1 - s; }
        for (int a = 0; a < 4; ++a) for (int o = 0; o < 9; ++o) line[a][o] = NAN;
        for (int o = lo; o <= hi; ++o) {
            ora_prim q = prim_at(P, U, IDX(P, i, j, k) + o * st);
            line[0][o + 4] = q.u; line[1][o + 4] = q.v; line[2][o + 4] = q.w; line[3][o + 4] = q.T;
        }
        for (int a = 0; a < 4; ++a)
            g[a][e] = periodic(P, e) ? d1_int(&line[a][4], 1, vorder(P)) : d1_closure(&line[a][4], 1, s, n, vorder(P));
    }
    long mi = MIDX(P, i, j, k);
    for (int q = 0; q < 9; ++q) m[q] = P->met[q][mi];
    ora_prim q0 = prim_at(P, U, IDX(P, i, j, k));
    double o[3][4];
    ora_viscous_flux_point(P, g, m, P->met[9][mi], q0.u, q0.v, q0.w, q0.T, o);
    for (int r = 0; r < 4; ++r) out4[r] = o[d][r];
}
void ora_rhs_point(const ora_params *P, const double *U, int i, int j, int k, double out[5]) {
    for (int m = 0; m < 5; ++m) out[m] = 0.0;
    double J = P->met[9][MIDX(P, i, j, k)];
    for (int d = 0; d < 3; ++d) {
        int c[3] = { i, j, k };
        int s0 = c[d];
        double fp[9][5], fm[9][5], h[2][5]; /* points s0-4 .. s0+4 */
        for (int r = 0; r < 9; ++r) {
            c[d] = s0 - 4 + r;
            split_at(P, U, d, c[0], c[1], c[2], fp[r], fm[r]);
        }
        for (int e = 0; e < 2; ++e) { /* interfaces s0-1/2 (e=0) and s0+1/2 (e=1) */
            int sch = P->scheme;
            if (P->scheme == ORA_HYBRID) {
                int a[3] = { i, j, k }, b[3] = { i, j, k };
                a[d] = s0 - 1 + e; b[d] = s0 + e;
                sch = iface_scheme(P, theta_ext(P, U, d, a[0], a[1], a[2]), theta_ext(P, U, d, b[0], b[1], b[2]));
            }
            if (P->char_recon) {
                double S[5][5], Si[5][5];
                int ci[3] = { i, j, k };
                ci[d] = s0 - 1 + e;
                iface_eigen(P, U, d, ci, S, Si);
                iface_flux_char(sch, P->weno_eps, (const double(*)[5])(fp + e), (const double(*)[5])(fm + e), h[e],
                                closure_on(P, d), s0 - 1 + e, dim_n(P, d), (const double(*)[5])S, (const double(*)[5])Si);
            } else
                iface_flux(sch, P->weno_eps, (const double(*)[5])(fp + e), (const double(*)[5])(fm + e), h[e],
                           closure_on(P, d), s0 - 1 + e, dim_n(P, d));
        }
        for (int m = 0; m < 5; ++m) out[m] -= J * (h[1][m] - h[0][m]);
    }
    if (P->inviscid) return;
    double acc[4] = { 0, 0, 0, 0 };
    double dsum[3][4];
    for (int d = 0; d < 3; ++d) {
        int c[3] = { i, j, k };
        int s0 = c[d], n = dim_n(P, d);
        double line[4][9];
        for (int r = 0; r < 4; ++r) for (int o = 0; o < 9; ++o) line[r][o] = NAN;
        const int H = vorder(P) / 2;
        int lo = -H, hi = H;
        if (!periodic(P, d)) { if (s0 + lo < 0) lo = -s0; if (s0 + hi > n - 1) hi = n - 1 - s0; }
        for (int o = lo; o <= hi; ++o) {
            int s = s0 + o;
            if (periodic(P, d)) s = (s % n + n) % n;
            c[d] = s;
            double f4[4];
            fv_dir_at(P, U, d, c[0], c[1], c[2], f4);
            for (int r = 0; r < 4; ++r) line[r][o + 4] = f4[r];
        }
        for (int r = 0; r < 4; ++r)
            dsum[d][r] = periodic(P, d) ? d1_int(&line[r][4], 1, vorder(P)) : d1_closure(&line[r][4], 1, s0, n, vorder(P));
    }
    for (int r = 0; r < 4; ++r) {
        acc[r] = 0.0;
        for (int d = 0; d < 3; ++d) acc[r] += dsum[d][r];
        out[r + 1] += J * acc[r];
    }
}
void ora_rhs_points(const ora_params *P, const double *U, long npts, const int *ijk, double *out) {
#pragma omp parallel for schedule(dynamic, 16)
    for (long q = 0; q < npts; ++q) ora_rhs_point(P, U, ijk[3 * q], ijk[3 * q + 1], ijk[3 * q + 2], out + 5 * q);
}

/* ------------------------------------------------------ time marching (A.8) */
/* TVD RK3, eq. 45: stage s: U <- a_s U^n + b_s (U + dt L(U)),
 * (a,b) = (0,1), (3/4,1/4), (1/3,2/3).  Interior points only. */
void ora_rk3_update(const ora_params *P, const double *Un, double *U, const double *dU, double dt, int stage) {
    static const double A[3] = { 0.0, 3.0 / 4.0, 1.0 / 3.0 }, B[3] = { 1.0, 1.0 / 4.0, 2.0 / 3.0 };
    long np = NP(P);
    for (int m = 0; m < 5; ++m)
        for (int k = 0; k < P->nz; ++k)
            for (int j = 0; j < P->ny; ++j)
                for (int i = 0; i < P->nx; ++i) {
                    long id = m * np + IDX(P, i, j, k);
                    U[id] = A[stage] * Un[id] + B[stage] * (U[id] + dt * dU[id]);
                }
}
/* one full step: 3 x (fill ghosts, RHS, update), then a final ghost fill */
void ora_rk3_step(const ora_params *P, double *U, double dt) {
    long np = NP(P);
    double *Un = malloc(sizeof(double) * 5 * np), *dU = malloc(sizeof(double) * 5 * np);
    ora_fill_ghosts(P, U);
    memcpy(Un, U, sizeof(double) * 5 * np);
    for (int s = 0; s < 3; ++s) {
        if (s > 0) ora_fill_ghosts(P, U);
        ora_rhs(P, U, dU);
        ora_rk3_update(P, Un, U, dU, dt, s);
    }
    ora_fill_ghosts(P, U);
    free(Un); free(dU);
}

/* ------------------------------------------------------- wavespeed (A.9) */
/* Lambda = max over interior points of sum_d ( |d_x u + d_y v + d_z w| + c |grad d| ); the paper
 * gives no time-step rule, DESIGN R-17.  dt = CFL / Lambda. */
double ora_max_wavespeed(const ora_params *P, const double *U) {
    double best = 0.0;
    for (int k = 0; k < P->nz; ++k)
        for (int j = 0; j < P->ny; ++j)
            for (int i = 0; i < P->nx; ++i) {
                ora_prim q = prim_at(P, U, IDX(P, i, j, k));
                long mi = MIDX(P, i, j, k);
                double s = 0.0;
                for (int d = 0; d < 3; ++d) {
                    double a1 = P->met[3 * d][mi], a2 = P->met[3 * d + 1][mi], a3 = P->met[3 * d + 2][mi];
                    s += fabs(a1 * q.u + a2 * q.v + a3 * q.w) + q.c * sqrt(a1 * a1 + a2 * a2 + a3 * a3);
                }
                if (s > best) best = s;
            }
    return best;
}

/* ------------------------------------------------------- state guard */
/* The paper has no divergence handling: the scheme "can be guaranteed not to diverge, provided the time step is
 * appropriate".  The guard a caller can afford every few steps is a count over interior points:
 *   counts[0]  points with a NaN or an infinity in any of the five conserved variables,
 *   counts[1]  points with rho <= 0,
 *   counts[2]  points with p <= 0, p by eq. 8 (DESIGN R-1) as in prim_of; looked at only where the five values are
 *              finite and rho > 0 (elsewhere p has no meaning).
 * A NaN compares false, so a point with NaN rho is in counts[0] only. */
void ora_check_state(const ora_params *P, const double *U, long long counts[3]) {
    long np = NP(P);
    counts[0] = counts[1] = counts[2] = 0;
    for (int k = 0; k < P->nz; ++k)
        for (int j = 0; j < P->ny; ++j)
            for (int i = 0; i < P->nx; ++i) {
                long id = IDX(P, i, j, k);
                int finite = 1;
                for (int m = 0; m < 5; ++m) finite = finite && isfinite(U[m * np + id]);
                if (!finite) counts[0]++;
                if (U[id] <= 0.0) counts[1]++;
                if (finite && U[id] > 0.0 && prim_at(P, U, id).p <= 0.0) counts[2]++;
            }
}

/* inviscid term of a single direction only (dU zeroed first), for direction-wise parity tests */
void ora_inviscid_dir(const ora_params *P, const double *U, int d, double *dU) {
    long np = NP(P);
    double *theta = NULL;
    for (int m = 0; m < 5; ++m)
        for (int k = 0; k < P->nz; ++k)
            for (int j = 0; j < P->ny; ++j)
                for (int i = 0; i < P->nx; ++i) dU[m * np + IDX(P, i, j, k)] = 0.0;
    if (P->scheme == ORA_HYBRID) { theta = malloc(sizeof(double) * np); ora_sensor(P, U, theta); }
    inviscid_dir(P, U, theta, d, dU);
    free(theta);
}

long ora_sizeof_params(void) { return (long)sizeof(ora_params); }
