// Internal declarations shared by the CUDA translation units of libocfd_b200 (not part of the C ABI).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>

#include <vector>

#include "ocfd.h"

#define OCFD_NG 4

// Grid description handed to kernels by value.
struct GridDesc {
    int nx, ny, nz;        // interior
    int nxp, nyp, nzp;     // padded
    long long sy, sz, np;  // strides in doubles (x stride is 1), padded points per field
    int kind;              // ocfd_grid_kind
    const double *met[10];
    long long msk;         // metric k-plane stride (curvilinear)
    double ux, uy, uz;     // uniform: 1/dx, 1/dy, 1/dz
    double uJ;             // uniform: J
    int periodic[3];
    int closure[3];        // 1: the paper's shielded-WENO5 boundary scheme on this (aperiodic) axis (ocfd_params.bc_closure)
    // derived metric data built once at init (launch_metric_tables), so that no kernel divides by J per point:
    //   curvilinear: atab[d] = [5][planes][nyp][nxp] fields (k1, k2, k3, sigma, J) with alpha = (d_x, d_y, d_z)/J,
    //                sigma = |alpha|, k = alpha/sigma; k-plane stride msk (0 if extruded)
    //   stretched:   rmet[d] = 1-D arrays 1/xi_x(i), 1/eta_y(j), 1/zeta_z(k)
    //   uniform:     ua[d] = dx dy dz / spacing of axis d  (= d_d/J)
    const double *atab[3];
    long long atab_fs;     // field stride of atab (doubles)
    // curvilinear: the table of direction 0 once more with y contiguous, [5][planes][nxp][nypT] (nypT = nyp rounded up
    // to even): the x sweep stages 32 lines x 4 x-points per chunk, which are 4 rows of 256 bytes in this copy instead
    // of 32 rows of 32 bytes (the TMA engine works row by row)
    const double *atabT;
    long long atabT_fs;
    int nypT;
    const double *rmet[3];
    double ua[3];
};

// Gas / scheme constants handed to kernels by value.
struct GasDesc {
    double gamma, gm1, Ma, gM2, invMa;  // gM2 = gamma Ma^2
    double inv2g;                       // 1/(2 gamma)
    double w0;                          // (3-gamma)/(2(gamma-1))   (eq. 26)
    double w1;                          // w0 + 1/2
    double tgm1;                        // 2(gamma-1)
    double suth;                        // T_suth/T_ref
    double invRe, kfac;                 // 1/Re, 1/((gamma-1) Ma^2 Pr Re)
    double weno_eps, sw_eps, theta1, theta2;
};

// kernel classes, for ocfd_timing_read / ocfd_kernel_name (K_INV_X + d = the sweep of direction d as its own launch)
enum { K_GHOST = 0, K_SENSOR, K_INV_X, K_INV_Y, K_INV_Z, K_VISC_FLUX, K_VISC_DIV, K_RK, K_WAVE, K_CHECK, K_COUNT };
static_assert(K_COUNT == OCFD_NKERNELS, "kernel class count");

struct TimedLaunch { cudaEvent_t a, b; int id; };

// TMA tensor maps of the tile sweeps (characteristic variables; per direction), re-encoded only when the caller's
// U / dU pointers change
struct InvMaps {
    const double *Up, *dUp;
    bool ready;
    CUtensorMap U[3], th[3], out[3];
};
// ... of the marching sweeps (inviscid_march.cu), same roles, other box shapes
struct MarchMaps {
    const double *Up, *dUp;
    bool ready;
    CUtensorMap U[3], th[3], out[3], met[3];
};
// ... and of the two viscous passes
struct ViscMaps {
    const double *Ufp, *Up, *dUp;
    bool ready;
    CUtensorMap Uf, F, G, H, dU, U, Un;
};

// Tuning knobs of one context (ocfd_set_tuning): launch-shape choices that change no result beyond round-off.
struct Tuning {
    int zchunk_f;    // planes per CTA of viscous pass 1 (0 automatic)
    int zchunk_d;    // ... of viscous pass 2
    int zchunk_s;    // ... of the shock sensor
    int march_seg;   // segments per pencil of the marching sweeps (0 automatic)
    int tile_group;  // tiles per column group in the CTA numbering of the viscous passes (0: 16; >= tiles per row: x-fastest)
};

struct ocfd_ctx {
    uint64_t magic;
    ocfd_params p;
    GridDesc g;
    GasDesc gas;
    cudaStream_t stream;
    int visc_order;  // 6 or 8 (ocfd_params.visc_order, 0 -> 6)
    int nsm;         // SM count of the device (persistent kernels launch a multiple of it)
    Tuning tune;
    std::vector<const void *> smem_optin;   // kernels whose dynamic shared-memory limit has been raised in this context
    // workspace carve-up (device pointers)
    double *theta;   // [np]
    double *Fv;      // [12][np]
    double *Un;      // [5][np]: the second state buffer of ocfd_rk3_step (holds U^(1), U^(2); the user's U keeps U^n)
    double *dUw;     // [5][np]
    double *scal;    // small scalar area (wavespeed result)
    double *mtab;    // derived metric tables (see GridDesc)
    unsigned char *flags;  // [3][np] bytes (debug only)
    InvMaps inv;
    MarchMaps march;
    CUtensorMap sens_map;   // U with a 1-point x-y halo (stand-alone shock sensor)
    const double *sens_U;
    ViscMaps visc;
    long long launches;
    // optional per-launch timing with CUDA events on the launch stream (ocfd_timing)
    int timing;
    std::vector<TimedLaunch> tl;
    size_t tl_used;
};

// bracket one kernel launch: OCFD_T0 before it, OCFD_CHECK_LAUNCH after it
inline void ocfd_t0(ocfd_ctx *c, int id) {
    if (!c->timing) return;
    if (c->tl_used == c->tl.size()) {
        TimedLaunch t;
        cudaEventCreate(&t.a);
        cudaEventCreate(&t.b);
        c->tl.push_back(t);
    }
    c->tl[c->tl_used].id = id;
    cudaEventRecord(c->tl[c->tl_used].a, c->stream);
}
inline void ocfd_t1(ocfd_ctx *c) {
    if (!c->timing) return;
    cudaEventRecord(c->tl[c->tl_used].b, c->stream);
    c->tl_used++;
}
#define OCFD_T0(ctx, id) ocfd_t0((ctx), (id))

// ---------------------------------------------------------------- metric access
// padded linear index of (ip,jp,kp)
__device__ __forceinline__ long long pidx(const GridDesc &g, int ip, int jp, int kp) {
    return (long long)kp * g.sz + (long long)jp * g.sy + ip;
}

template <int KIND>
struct Met {
    // metric row of direction d at padded point (ip,jp,kp): (d_x, d_y, d_z)
    __device__ __forceinline__ static void row(const GridDesc &g, int d, int ip, int jp, int kp, double &a, double &b,
                                               double &c) {
        if (KIND == OCFD_GRID_UNIFORM) {
            a = d == 0 ? g.ux : 0.0;
            b = d == 1 ? g.uy : 0.0;
            c = d == 2 ? g.uz : 0.0;
        } else if (KIND == OCFD_GRID_STRETCHED) {
            a = d == 0 ? __ldg(g.met[0] + ip) : 0.0;
            b = d == 1 ? __ldg(g.met[4] + jp) : 0.0;
            c = d == 2 ? __ldg(g.met[8] + kp) : 0.0;
        } else {
            long long mi = (long long)kp * g.msk + (long long)jp * g.sy + ip;
            a = __ldg(g.met[3 * d] + mi);
            b = __ldg(g.met[3 * d + 1] + mi);
            c = __ldg(g.met[3 * d + 2] + mi);
        }
    }
    __device__ __forceinline__ static double J(const GridDesc &g, int ip, int jp, int kp) {
        if (KIND == OCFD_GRID_UNIFORM) return g.uJ;
        if (KIND == OCFD_GRID_STRETCHED) return (__ldg(g.met[0] + ip) * __ldg(g.met[4] + jp)) * __ldg(g.met[8] + kp);
        return __ldg(g.met[9] + (long long)kp * g.msk + (long long)jp * g.sy + ip);
    }
};

// Unit normal k = alpha/|alpha| and length sigma = |alpha| of alpha = (d_x, d_y, d_z)/J (eq. 20-22) of direction DIR,
// and J itself, at a padded point.
template <int KIND, int DIR>
__device__ __forceinline__ void met_ksJ(const GridDesc &g, int ip, int jp, int kp, double &k1, double &k2, double &k3,
                                        double &sigma, double &J) {
    if (KIND == OCFD_GRID_UNIFORM) {
        const double a = g.ua[DIR];
        const double sg = a < 0.0 ? -1.0 : 1.0;
        k1 = DIR == 0 ? sg : 0.0;
        k2 = DIR == 1 ? sg : 0.0;
        k3 = DIR == 2 ? sg : 0.0;
        sigma = fabs(a);
        J = g.uJ;
    } else if (KIND == OCFD_GRID_STRETCHED) {
        const double rx = __ldg(g.rmet[0] + ip), ry = __ldg(g.rmet[1] + jp), rz = __ldg(g.rmet[2] + kp);
        const double a = DIR == 0 ? ry * rz : DIR == 1 ? rx * rz : rx * ry;
        const double sg = a < 0.0 ? -1.0 : 1.0;
        k1 = DIR == 0 ? sg : 0.0;
        k2 = DIR == 1 ? sg : 0.0;
        k3 = DIR == 2 ? sg : 0.0;
        sigma = fabs(a);
        J = (__ldg(g.met[0] + ip) * __ldg(g.met[4] + jp)) * __ldg(g.met[8] + kp);
    } else {
        const double *t = g.atab[DIR] + (long long)kp * g.msk + (long long)jp * g.sy + ip;
        k1 = __ldg(t);
        k2 = __ldg(t + g.atab_fs);
        k3 = __ldg(t + 2 * g.atab_fs);
        sigma = __ldg(t + 3 * g.atab_fs);
        J = __ldg(t + 4 * g.atab_fs);
    }
}

// ---------------------------------------------------------------- kernel launchers (host side)
ocfd_status launch_metric_tables(ocfd_ctx *c);
ocfd_status launch_fill_ghosts(ocfd_ctx *c, double *U);
ocfd_status launch_sensor(ocfd_ctx *c, const double *U);
ocfd_status launch_flags(ocfd_ctx *c, unsigned char *flags);
ocfd_status launch_inviscid(ocfd_ctx *c, const double *U, double *dU);
ocfd_status launch_inviscid_march(ocfd_ctx *c, const double *U, double *dU, int dir);
ocfd_status launch_viscous_flux(ocfd_ctx *c, const double *U, bool sensor);
// RK3 buffers of one stage (eq. 45): out <- a_s Un + b_s (Uin + dt dU); ocfd_rk3_step rotates them so that no stage
// copies the state (stage 0: user's U -> second buffer; stage 1: in place in the second buffer; stage 2: -> user's U)
struct RkBufs { const double *Un, *Uin; double *out; };
ocfd_status launch_viscous_div(ocfd_ctx *c, double *dU, const RkBufs &rk, double dt, int rk_stage);
ocfd_status launch_rk_update(ocfd_ctx *c, const double *Un, const double *Uin, double *out, const double *dU, double dt,
                             int stage);
ocfd_status launch_wavespeed(ocfd_ctx *c, const double *U, double *host_out);
ocfd_status launch_check_state(ocfd_ctx *c, const double *U, long long *host_counts);

// Raise the dynamic shared-memory limit of `kernel` to `bytes` once per context (the attribute lives in the device
// context of the function, so a process-wide flag would leave a second device without it).
inline bool ocfd_smem_optin(ocfd_ctx *c, const void *kernel, size_t bytes) {
    for (const void *k : c->smem_optin)
        if (k == kernel) return true;
    if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) != cudaSuccess) return false;
    c->smem_optin.push_back(kernel);
    return true;
}

// a failed launch is reported on stderr with the CUDA error text (the C ABI only carries OCFD_ECUDA)
inline bool ocfd_launch_failed(const char *file, int line) {
    const cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) return false;
    fprintf(stderr, "libocfd_b200: CUDA error at %s:%d: %s\n", file, line, cudaGetErrorString(e));
    return true;
}
#define OCFD_CHECK_LAUNCH(ctx)                                        \
    do {                                                              \
        ocfd_t1(ctx);                                                 \
        (ctx)->launches++;                                            \
        if (ocfd_launch_failed(__FILE__, __LINE__)) return OCFD_ECUDA; \
    } while (0)
