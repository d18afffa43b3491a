// C ABI of libocfd_b200 (include/ocfd.h): argument validation, workspace carve-up, step orchestration.
#include <math.h>
#include <new>
#include <string.h>

#include "ocfd_internal.cuh"

namespace {

const uint64_t kMagic = 0x4f43464442323030ull;  // "OCFDB200"

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

bool valid_params(const ocfd_params *p) {
    if (!p) return false;
    if (p->ng != OCFD_NG) return false;
    if (p->nx < 8 || p->ny < 8 || p->nz < 8) return false;
    if (p->nx > OCFD_MAX_EXTENT || p->ny > OCFD_MAX_EXTENT || p->nz > OCFD_MAX_EXTENT) return false;  // grid dimensions of the launches
    if (p->nx % 2) return false;  // TMA: row pitch (nx+8)*8 bytes must be a multiple of 16
    if ((long long)(p->nx + 8) * (p->ny + 8) * (p->nz + 8) > (1ll << 40)) return false;
    if (!(p->gamma > 1.0) || !(p->Ma > 0.0) || !(p->weno_eps >= 1e-50) || !(p->sw_eps >= 0.0)) return false;  // (eps+IS)^6 must stay normal
    if (!p->inviscid && (!(p->Re > 0.0) || !(p->Pr > 0.0) || !(p->T_ref > 0.0) || !(p->T_suth >= 0.0))) return false;
    if (p->scheme < OCFD_UD7 || p->scheme > OCFD_HYBRID) return false;
    if (p->visc_order != 0 && p->visc_order != 6 && p->visc_order != 8) return false;
    if (p->bc_closure != 0 && p->bc_closure != 1) return false;
    if (p->char_recon != 0 && p->char_recon != 1) return false;
    if (p->scheme == OCFD_HYBRID && (isnan(p->theta1) || isnan(p->theta2) || p->theta1 > p->theta2)) return false;
    switch (p->grid_kind) {
        case OCFD_GRID_UNIFORM:
            if (!(p->dx > 0.0) || !(p->dy > 0.0) || !(p->dz > 0.0)) return false;
            break;
        case OCFD_GRID_STRETCHED:
            if (!p->metric[0] || !p->metric[4] || !p->metric[8]) return false;
            break;
        case OCFD_GRID_CURVILINEAR:
            for (int q = 0; q < 10; ++q)
                if (!p->metric[q]) return false;
            if (p->metric_plane_stride != 0 && p->metric_plane_stride != (long long)(p->nx + 8) * (p->ny + 8)) return false;
            break;
        default: return false;
    }
    for (int f = 0; f < 6; ++f) {
        if (p->bc[f] < OCFD_BC_PERIODIC || p->bc[f] > OCFD_BC_EXTRAP_OUTFLOW) return false;
        if (p->bc[f] == OCFD_BC_SUPERSONIC_INFLOW && !p->inflow[f]) return false;
        if (p->bc[f] == OCFD_BC_WALL_ISOTHERMAL && !(p->T_wall[f] > 0.0)) return false;
    }
    for (int d = 0; d < 3; ++d)
        if ((p->bc[2 * d] == OCFD_BC_PERIODIC) != (p->bc[2 * d + 1] == OCFD_BC_PERIODIC)) return false;
    return true;
}

struct Carve { size_t theta, Fv, Un, dUw, scal, mtab, total; };

Carve carve(const ocfd_params *p) {
    const size_t np = (size_t)(p->nx + 8) * (p->ny + 8) * (p->nz + 8);
    const size_t fb = align_up(np * sizeof(double), 256);
    Carve c;
    size_t off = 0;
    c.theta = off; off += fb;
    c.Fv = off; off += p->inviscid ? 0 : align_up(12 * np * sizeof(double), 256);
    c.Un = off; off += align_up(5 * np * sizeof(double), 256);
    c.dUw = off; off += align_up(5 * np * sizeof(double), 256);
    c.scal = off; off += 256;
    c.mtab = off;
    if (p->grid_kind == OCFD_GRID_CURVILINEAR) {
        const size_t planes = p->metric_plane_stride ? (size_t)(p->nz + 8) : 1;
        off += align_up(15 * planes * (size_t)(p->nx + 8) * (p->ny + 8) * sizeof(double), 256);
        off += align_up(5 * planes * (size_t)(p->nx + 8) * (size_t)((p->ny + 9) & ~1) * sizeof(double), 256);  // atabT
    } else if (p->grid_kind == OCFD_GRID_STRETCHED) {
        off += align_up((size_t)(p->nx + p->ny + p->nz + 24) * sizeof(double), 256);
    }
    c.total = off;
    return c;
}

bool live(const ocfd_ctx *c) { return c && c->magic == kMagic; }

}  // namespace

extern "C" {

size_t ocfd_workspace_bytes(const ocfd_params *p) {
    if (!valid_params(p)) return 0;
    return carve(p).total;
}

ocfd_status ocfd_init(ocfd_ctx **out, const ocfd_params *p) {
    if (!out) return OCFD_EINVAL;
    *out = nullptr;
    if (!valid_params(p)) return OCFD_EINVAL;
    const Carve cv = carve(p);
    if (!p->workspace || ((uintptr_t)p->workspace & 255) || p->workspace_bytes < cv.total) return OCFD_EWORKSPACE;
    int dev = 0, major = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return OCFD_ECUDA;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) return OCFD_ECUDA;
    if (major < 10) return OCFD_EUNSUPPORTED;  // sm_100a only; there is no other code path
    int nsm = 0;
    if (cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || nsm <= 0) return OCFD_ECUDA;
    ocfd_ctx *c = new (std::nothrow) ocfd_ctx();
    if (!c) return OCFD_EINVAL;
    c->magic = kMagic;
    c->p = *p;
    c->stream = (cudaStream_t)p->stream;
    c->nsm = nsm;
    c->tune = Tuning();
    c->visc_order = p->visc_order == 8 ? 8 : 6;
    GridDesc &g = c->g;
    g.nx = p->nx; g.ny = p->ny; g.nz = p->nz;
    g.nxp = p->nx + 8; g.nyp = p->ny + 8; g.nzp = p->nz + 8;
    g.sy = g.nxp; g.sz = (long long)g.nxp * g.nyp; g.np = g.sz * g.nzp;
    g.kind = p->grid_kind;
    for (int q = 0; q < 10; ++q) g.met[q] = p->metric[q];
    g.msk = p->metric_plane_stride;
    g.ux = g.uy = g.uz = g.uJ = 0.0;
    if (p->grid_kind == OCFD_GRID_UNIFORM) {
        g.ux = 1.0 / p->dx; g.uy = 1.0 / p->dy; g.uz = 1.0 / p->dz;
        g.uJ = (g.ux * g.uy) * g.uz;
    }
    for (int d = 0; d < 3; ++d) g.periodic[d] = p->bc[2 * d] == OCFD_BC_PERIODIC;
    for (int d = 0; d < 3; ++d) g.closure[d] = p->bc_closure && !g.periodic[d];
    GasDesc &s = c->gas;
    s.gamma = p->gamma; s.gm1 = p->gamma - 1.0; s.Ma = p->Ma; s.gM2 = p->gamma * p->Ma * p->Ma; s.invMa = 1.0 / p->Ma;
    s.inv2g = 1.0 / (2.0 * p->gamma);
    s.w0 = (3.0 - p->gamma) / (2.0 * (p->gamma - 1.0));
    s.w1 = s.w0 + 0.5;
    s.tgm1 = 2.0 * (p->gamma - 1.0);
    s.suth = p->inviscid ? 0.0 : p->T_suth / p->T_ref;
    s.invRe = p->inviscid ? 0.0 : 1.0 / p->Re;
    s.kfac = p->inviscid ? 0.0 : 1.0 / ((p->gamma - 1.0) * p->Ma * p->Ma * p->Pr * p->Re);
    s.weno_eps = p->weno_eps; s.sw_eps = p->sw_eps; s.theta1 = p->theta1; s.theta2 = p->theta2;
    char *w = (char *)p->workspace;
    c->theta = (double *)(w + cv.theta);
    c->Fv = (double *)(w + cv.Fv);
    c->Un = (double *)(w + cv.Un);
    c->dUw = (double *)(w + cv.dUw);
    c->scal = (double *)(w + cv.scal);
    c->mtab = (double *)(w + cv.mtab);
    for (int d = 0; d < 3; ++d) { g.atab[d] = nullptr; g.rmet[d] = nullptr; g.ua[d] = 0.0; }
    g.atab_fs = 0;
    g.atabT = nullptr; g.atabT_fs = 0; g.nypT = (g.nyp + 1) & ~1;
    if (p->grid_kind == OCFD_GRID_UNIFORM) {
        g.ua[0] = g.ux / g.uJ; g.ua[1] = g.uy / g.uJ; g.ua[2] = g.uz / g.uJ;
    } else if (p->grid_kind == OCFD_GRID_STRETCHED) {
        g.rmet[0] = c->mtab; g.rmet[1] = c->mtab + g.nxp; g.rmet[2] = c->mtab + g.nxp + g.nyp;
    } else {
        g.atab_fs = (g.msk ? (long long)g.nzp : 1ll) * g.sz;
        for (int d = 0; d < 3; ++d) g.atab[d] = c->mtab + 5 * d * g.atab_fs;
        g.atabT_fs = (g.msk ? (long long)g.nzp : 1ll) * g.nxp * g.nypT;
        g.atabT = c->mtab + (align_up(15 * (size_t)g.atab_fs * sizeof(double), 256) / sizeof(double));
    }
    c->flags = nullptr;
    c->launches = 0;
    c->inv.ready = false;
    c->inv.Up = c->inv.dUp = nullptr;
    c->march.ready = false;
    c->march.Up = c->march.dUp = nullptr;
    c->sens_U = nullptr;
    c->visc.ready = false;
    c->visc.Ufp = c->visc.Up = c->visc.dUp = nullptr;
    c->timing = 0;
    c->tl_used = 0;
    if (launch_metric_tables(c) != OCFD_OK) { delete c; return OCFD_ECUDA; }
    *out = c;
    return OCFD_OK;
}

ocfd_status ocfd_destroy(ocfd_ctx *c) {
    if (!live(c)) return OCFD_ESTATE;
    c->magic = 0;
    for (auto &t : c->tl) { cudaEventDestroy(t.a); cudaEventDestroy(t.b); }
    delete c;
    return OCFD_OK;
}

ocfd_status ocfd_fill_ghosts(ocfd_ctx *c, double *U) {
    if (!live(c)) return OCFD_ESTATE;
    if (!U) return OCFD_EINVAL;
    return launch_fill_ghosts(c, U);
}

// theta of U for the hybrid scheme: part of viscous pass 1 (which has staged everything the sensor needs), or the
// stand-alone sensor kernel when there are no viscous terms
static ocfd_status flux_and_sensor(ocfd_ctx *c, const double *U) {
    const bool hybrid = c->p.scheme == OCFD_HYBRID;
    if (!c->p.inviscid) return launch_viscous_flux(c, U, hybrid);
    return hybrid ? launch_sensor(c, U) : OCFD_OK;
}

// rows a2-a7; rk_stage >= 0 additionally folds the RK3 stage update (a8) into the last kernel that touches dU.
// Order: viscous pass 1 (+ sensor) first -- it depends on U only --, then the sweeps, then viscous pass 2 (+ RK3).
static ocfd_status rhs_impl(ocfd_ctx *c, const double *U, double *dU, int rk_stage, double dt, const RkBufs &rk) {
    ocfd_status st;
    if ((st = flux_and_sensor(c, U)) != OCFD_OK) return st;
    if ((st = launch_inviscid(c, U, dU)) != OCFD_OK) return st;
    if (!c->p.inviscid) return launch_viscous_div(c, dU, rk, dt, rk_stage);
    if (rk_stage >= 0) return launch_rk_update(c, rk.Un, rk.Uin, rk.out, dU, dt, rk_stage);
    return OCFD_OK;
}

ocfd_status ocfd_rhs(ocfd_ctx *c, const double *U, double *dU) {
    if (!live(c)) return OCFD_ESTATE;
    if (!U || !dU || U == dU) return OCFD_EINVAL;
    return rhs_impl(c, U, dU, -1, 0.0, RkBufs{nullptr, nullptr, nullptr});  // rk_stage < 0: no update
}

ocfd_status ocfd_rk3_step(ocfd_ctx *c, double *U, double dt) {
    if (!live(c)) return OCFD_ESTATE;
    if (!U || !(dt == dt)) return OCFD_EINVAL;
    ocfd_status st;
    // eq. 45 without a copy of the state: U keeps U^n through the step, the intermediate states live in the second
    // buffer B, and the last stage writes U^(n+1) over U^n (point-wise, so in place is safe)
    double *B = c->Un;
    const RkBufs rk[3] = {{nullptr, U, B}, {U, B, B}, {U, B, U}};
    for (int s = 0; s < 3; ++s) {
        double *cur = s == 0 ? U : B;
        if ((st = launch_fill_ghosts(c, cur)) != OCFD_OK) return st;
        if ((st = rhs_impl(c, cur, c->dUw, s, dt, rk[s])) != OCFD_OK) return st;
    }
    return launch_fill_ghosts(c, U);
}

ocfd_status ocfd_rk3_steps_host(ocfd_ctx *c, double *U_host, double *U_dev, double dt, int nsteps) {
    if (!live(c)) return OCFD_ESTATE;
    if (!U_host || !U_dev || nsteps < 0) return OCFD_EINVAL;
    const size_t bytes = (size_t)5 * c->g.np * sizeof(double);
    if (cudaMemcpyAsync(U_dev, U_host, bytes, cudaMemcpyHostToDevice, c->stream) != cudaSuccess) return OCFD_ECUDA;
    for (int n = 0; n < nsteps; ++n) {
        ocfd_status st = ocfd_rk3_step(c, U_dev, dt);
        if (st != OCFD_OK) return st;
    }
    if (cudaMemcpyAsync(U_host, U_dev, bytes, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) return OCFD_ECUDA;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return OCFD_ECUDA;
    return OCFD_OK;
}

ocfd_status ocfd_max_wavespeed(ocfd_ctx *c, const double *U, double *host_out) {
    if (!live(c)) return OCFD_ESTATE;
    if (!U || !host_out) return OCFD_EINVAL;
    return launch_wavespeed(c, U, host_out);
}

ocfd_status ocfd_check_state(ocfd_ctx *c, const double *U, long long *host_counts) {
    if (!live(c)) return OCFD_ESTATE;
    if (!U || !host_counts) return OCFD_EINVAL;
    return launch_check_state(c, U, host_counts);
}

ocfd_status ocfd_debug_sensor(ocfd_ctx *c, const double *U, double *theta, unsigned char *flag_xyz) {
    if (!live(c)) return OCFD_ESTATE;
    if (!U) return OCFD_EINVAL;
    ocfd_status st;
    // all-ones bytes are a NaN: what the sensor does not write (everything but the interior and the first ghost layer
    // of each face) comes back as NaN
    if (cudaMemsetAsync(c->theta, 0xff, c->g.np * sizeof(double), c->stream) != cudaSuccess) return OCFD_ECUDA;
    // the same kernel that computes theta inside ocfd_rhs / ocfd_rk3_step for this context
    if ((st = c->p.inviscid ? launch_sensor(c, U) : launch_viscous_flux(c, U, true)) != OCFD_OK) return st;
    if (theta && cudaMemcpyAsync(theta, c->theta, c->g.np * sizeof(double), cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess)
        return OCFD_ECUDA;
    if (flag_xyz && (st = launch_flags(c, flag_xyz)) != OCFD_OK) return st;
    return OCFD_OK;
}

ocfd_status ocfd_timing(ocfd_ctx *c, int enable) {
    if (!live(c)) return OCFD_ESTATE;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return OCFD_ECUDA;
    c->timing = enable ? 1 : 0;
    c->tl_used = 0;
    return OCFD_OK;
}

ocfd_status ocfd_timing_read(ocfd_ctx *c, double *ms, long long *launches) {
    if (!live(c)) return OCFD_ESTATE;
    if (!ms || !launches) return OCFD_EINVAL;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return OCFD_ECUDA;
    for (int k = 0; k < OCFD_NKERNELS; ++k) { ms[k] = 0.0; launches[k] = 0; }
    for (size_t q = 0; q < c->tl_used; ++q) {
        float t = 0.f;
        if (cudaEventElapsedTime(&t, c->tl[q].a, c->tl[q].b) != cudaSuccess) return OCFD_ECUDA;
        ms[c->tl[q].id] += t;
        launches[c->tl[q].id]++;
    }
    c->tl_used = 0;
    return OCFD_OK;
}

const char *ocfd_kernel_name(int id) {
    static const char *names[OCFD_NKERNELS] = {"ghost_fill", "shock_sensor", "inviscid_x", "inviscid_y",
                                               "inviscid_z", "viscous_flux", "viscous_div", "rk3_update", "max_wavespeed",
                                               "check_state"};
    return id >= 0 && id < OCFD_NKERNELS ? names[id] : "?";
}

size_t ocfd_sizeof_params(void) { return sizeof(ocfd_params); }

ocfd_status ocfd_set_tuning(ocfd_ctx *c, const char *key, int value) {
    if (!live(c)) return OCFD_ESTATE;
    if (!key || value < 0) return OCFD_EINVAL;
    const bool zchunk = !strncmp(key, "zchunk_", 7);
    if (zchunk && value > 0 && value < 8) return OCFD_EINVAL;   // the marches need chunks of at least 8 planes
    if (!strcmp(key, "zchunk_flux")) c->tune.zchunk_f = value;
    else if (!strcmp(key, "zchunk_div")) c->tune.zchunk_d = value;
    else if (!strcmp(key, "zchunk_sensor")) c->tune.zchunk_s = value;
    else if (!strcmp(key, "march_seg")) c->tune.march_seg = value;
    else if (!strcmp(key, "tile_group")) c->tune.tile_group = value;
    else return OCFD_EINVAL;
    return OCFD_OK;
}

long long ocfd_launch_count(const ocfd_ctx *c) { return live(c) ? c->launches : -1; }

const char *ocfd_strerror(ocfd_status s) {
    switch (s) {
        case OCFD_OK: return "ok";
        case OCFD_EINVAL: return "invalid argument";
        case OCFD_EWORKSPACE: return "workspace missing, misaligned or too small";
        case OCFD_ECUDA: return "CUDA runtime or launch error";
        case OCFD_EUNSUPPORTED: return "unsupported (this library runs on sm_100a only)";
        case OCFD_ESTATE: return "invalid or destroyed context";
    }
    return "unknown status";
}

}  // extern "C"
