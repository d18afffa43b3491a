/*
 * ocfd.h -- C ABI of the B200-native RHS / RK3 hot path of the OpenCFD-SCU finite-difference DNS method
 * (arxiv 2209.15333; citations "PAPER.md:Lnnn" are lines of /root/reference/PAPER.md, "DESIGN R-n" are the
 * readings registered in DESIGN.md section 3).
 *
 * One structured block on ONE GPU (sm_100a), fp64 throughout.  All field pointers are DEVICE
 * pointers unless a name says "host".  The library allocates no field memory: the caller (PyTorch in the Python
 * binding) owns U, dU, the metric fields, the boundary data and one scratch workspace.  Every call except
 * ocfd_max_wavespeed and ocfd_rk3_steps_host only enqueues work on the stream given at init and returns.
 *
 * Layout: a field is a padded box [nz+8][ny+8][nx+8], x contiguous, 4 ghost layers per
 * face (LAP = 4, the reach of the 7th-order stencils).  U and dU are component-major [5][nz+8][ny+8][nx+8] with
 * components (rho, rho u, rho v, rho w, E) (eq. 5).  Interior index (i,j,k) lives at padded
 * (i+4, j+4, k+4).  Edge and corner ghosts are never read nor written by any entry point.
 *
 * Errors: every entry point returns an ocfd_status; argument errors are detected synchronously and leave all
 * buffers untouched; CUDA launch errors map to OCFD_ECUDA.  No global state (the one exception is the fixed scratch array
 * of ocfd_max_wavespeed_static, see there); several contexts may coexist.
 * There is no CPU fallback of any kind.
 */
#ifndef OCFD_H
#define OCFD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ocfd_ctx ocfd_ctx; /* opaque; owns no device memory */

#define OCFD_MAX_EXTENT 65527 /* largest interior extent per axis (an extent + 8 is a CUDA grid dimension) */

typedef enum {
    OCFD_OK = 0,
    OCFD_EINVAL = -1,       /* bad argument (null pointer, bad size, inconsistent boundary pairing ...) */
    OCFD_EWORKSPACE = -2,   /* workspace missing, misaligned or smaller than ocfd_workspace_bytes() */
    OCFD_ECUDA = -3,        /* a CUDA runtime call or kernel launch failed */
    OCFD_EUNSUPPORTED = -4, /* valid request this build does not implement */
    OCFD_ESTATE = -5        /* call order violated (e.g. destroyed context) */
} ocfd_status;

typedef enum { OCFD_GRID_UNIFORM = 0, OCFD_GRID_STRETCHED = 1, OCFD_GRID_CURVILINEAR = 2 } ocfd_grid_kind;

/* Inviscid reconstruction (Table 2 rows 6, 4, 2 and the hybrid of eq. 42). */
typedef enum { OCFD_UD7 = 0, OCFD_WENO7 = 1, OCFD_WENO5 = 2, OCFD_HYBRID = 3 } ocfd_scheme;

/* Boundary treatment of one face (DESIGN R-16; the paper prints no formulas). */
typedef enum {
    OCFD_BC_PERIODIC = 0,
    OCFD_BC_WALL_ISOTHERMAL = 1,
    OCFD_BC_SUPERSONIC_INFLOW = 2,
    OCFD_BC_EXTRAP_OUTFLOW = 3
} ocfd_bc;

typedef struct {
    int nx, ny, nz;   /* interior dimensions, each >= 8 and <= OCFD_MAX_EXTENT; nx must be even (rows of the padded
                         fields must stay 16-byte aligned for the TMA tensor maps); anything else is OCFD_EINVAL */
    int ng;           /* ghost layers; must be 4 */
    ocfd_grid_kind grid_kind;
    /* Metric data (eq. 3-4), device pointers, caller-owned, must outlive the context.
     *   CURVILINEAR: metric[0..8] = xi_x xi_y xi_z eta_x eta_y eta_z zeta_x zeta_y zeta_z, metric[9] = J,
     *                each a padded field including ghost values; consecutive k-planes are
     *                metric_plane_stride doubles apart: (nx+8)*(ny+8) for full 3-D fields, 0 for a 2-D map
     *                extruded in z (one padded plane per metric, the shape of the paper's ramp and
     *                flat-plate grids).
     *   STRETCHED:   metric[0], metric[4], metric[8] = padded 1-D arrays xi_x(i), eta_y(j), zeta_z(k) of
     *                nx+8, ny+8, nz+8 doubles; the rest NULL.  J = (xi_x * eta_y) * zeta_z.
     *   UNIFORM:     all NULL; spacing dx, dy, dz below.  xi_x = 1/dx ..., J = ((1/dx)(1/dy))(1/dz). */
    const double *metric[10];
    long long metric_plane_stride;
    double dx, dy, dz;
    /* Gas / flow parameters: ratio of specific heats, reference Mach, Reynolds and Prandtl
     * numbers, reference temperature [K] and Sutherland constant [K] (DESIGN R-8: 110.4). */
    double gamma, Ma, Re, Pr, T_ref, T_suth;
    int inviscid;            /* 1: skip the viscous terms (rows a6, a7) */
    ocfd_scheme scheme;
    double theta1, theta2;   /* hybrid thresholds (0.02, 0.1), theta1 <= theta2; theta2 = +inf gives two
                                levels */
    /* epsilon of the WENO weights, applied to the J^-1-scaled split flux (DESIGN R-10).  Range: the kernels form the
     * WENO7 weights with ONE division, as sum_k P_k C_k q_k / sum_k C_k P_k with P_k a product of three (eps + IS_m)^2,
     * i.e. of size (eps + IS)^6, and divide by seeded reciprocals that flush subnormal inputs to zero.  That stays in
     * the normal fp64 range for 1e-50 <= eps + IS <= 1e50, i.e. weno_eps >= 1e-50 (smaller values are OCFD_EINVAL) and
     * J^-1-scaled split fluxes below about 1e25 in magnitude: any grid and unit system whose cell-face areas lie
     * between 1e-22 and 1e22 with O(1) non-dimensional flow variables. */
    double weno_eps;
    double sw_eps;           /* 0: eigenvalue split exactly as eq. 29; > 0: (lambda +- sqrt(lambda^2+eps^2))/2 */
    ocfd_bc bc[6];           /* x-, x+, y-, y+, z-, z+; PERIODIC must be set on both faces of an axis */
    double T_wall[6];        /* non-dimensional wall temperature of WALL faces */
    /* Optional prescribed wall-normal velocity (blowing / suction) of WALL faces: padded 2-D device array over
     * the two tangential axes, [slow+8][fast+8] with fast = x (or y on x-faces), else NULL. */
    const double *wall_vn[6];
    /* INFLOW faces: 5 padded 2-D device arrays of conserved variables, component-major [5][slow+8][fast+8]. */
    const double *inflow[6];
    void *workspace;         /* device scratch, 256-byte aligned, at least ocfd_workspace_bytes() */
    size_t workspace_bytes;
    void *stream;            /* cudaStream_t to enqueue on (0 = default stream) */
    /* Order of the central scheme of the viscous terms ("two such schemes, of sixth and eighth
     * order"): 6 (also 0) or 8.  On aperiodic axes the boundary rows are one-sided 2nd order at the boundary point
     * and central 2nd / 4th (/ 6th for the 8th-order scheme) at the following points. */
    int visc_order;
    /* Inviscid boundary scheme on aperiodic axes.  0: the ghost cells written by ocfd_fill_ghosts feed the full
     * stencils (default).  1: the paper's scheme: a flux whose 7-point stencil reaches outside
     * the domain is computed by WENO5 with the candidate sub-stencils that contain an outside point shielded
     * (weight 0, the others renormalised); no value outside the domain is read by the sweeps.  If all three
     * candidates are shielded (the boundary interface itself, for the wave that enters) the boundary node's split
     * flux is taken (DESIGN R-21).  The paper does not say what happens there: that value is a choice of this build,
     * matched by the test reference but pinned by nothing in the paper. */
    int bc_closure;
    /* 1: flux reconstruction in characteristic variables (section 2.2.2): at every interface the
     * split fluxes of the stencil are projected with the left eigenvectors S (eq. 35) of the averaged state (eq. 32),
     * reconstructed component by component and projected back with S^-1 (eq. 34).  0: component-wise (default). */
    int char_recon;
} ocfd_params;

/* Bytes of device scratch a context with these parameters needs; 0 if the parameters are invalid.  Pure. */
size_t ocfd_workspace_bytes(const ocfd_params *p);

/* Validate, copy the parameters, carve the workspace, build the derived metric tables (one small launch on the stream).
 * No field memory is allocated.  Errors: OCFD_EINVAL (parameters), OCFD_EWORKSPACE, OCFD_EUNSUPPORTED (not an sm_100
 * device), OCFD_ECUDA.  The library reads no environment variable and keeps no state outside its contexts. */
ocfd_status ocfd_init(ocfd_ctx **out, const ocfd_params *p);
ocfd_status ocfd_destroy(ocfd_ctx *ctx);

/* Row a1.  Set Dirichlet nodes (wall, inflow) then fill the 4 ghost layers of every face of U, in place,
 * faces in the order x-, x+, y-, y+, z-, z+ (DESIGN R-16). */
ocfd_status ocfd_fill_ghosts(ocfd_ctx *ctx, double *U);

/* Rows a2-a7.  dU <- L(U) = -J sum_d d(F_d)/d(d) + J sum_d d(Fv_d)/d(d) (eq. 1) on interior points.
 * Ghosts of U must be valid; ghosts of dU are left untouched; U is not modified (pure function of U). */
ocfd_status ocfd_rhs(ocfd_ctx *ctx, const double *U, double *dU);

/* Rows a1-a8.  One TVD-RK3 step (eq. 45): 3 x (fill ghosts, RHS, stage update), then a
 * final ghost fill, in place on U.  The call only enqueues kernels on the context's stream (27 launches with viscous
 * terms): after one plain call with the same U pointer (one-time host-side set-up: tensor maps, shared-memory opt-in) it
 * can be captured into a CUDA graph on a non-default stream and replayed, which is what launch-bound small grids need
 * (tests/test_gpu_parity.py replays it bit for bit; `bench.py --graph` times it). */
ocfd_status ocfd_rk3_step(ocfd_ctx *ctx, double *U, double dt);

/* The same nsteps steps end to end from HOST memory: copy U_host (5 padded fields, pinned or pageable) into the
 * device buffer U_dev, step, copy back, synchronise the stream. */
ocfd_status ocfd_rk3_steps_host(ocfd_ctx *ctx, double *U_host, double *U_dev, double dt, int nsteps);

/* Row a9.  Lambda = max over interior points of sum_d (|d_x u + d_y v + d_z w| + c |grad d|) (DESIGN R-17);
 * the caller sets dt = CFL / Lambda.  Writes one double to host_out and synchronises the stream. */
ocfd_status ocfd_max_wavespeed(ocfd_ctx *ctx, const double *U, double *host_out);

/* State guard.  The paper handles no divergence: the scheme "can be guaranteed not to diverge,
 * provided the time step is appropriate"; ocfd_max_wavespeed turns a NaN state into a NaN Lambda, but a
 * negative density or pressure only shows up as a NaN one stage later, without a place or a count.  This call counts,
 * over the interior points of U (device pointer; ghosts are not looked at):
 *   host_counts[0]  points with a NaN or an infinity in any of the five conserved variables,
 *   host_counts[1]  points with rho <= 0 (a NaN rho compares false and is in [0] only; -inf is in both),
 *   host_counts[2]  points with p = (gamma-1)(E - rho (u^2+v^2+w^2)/2) <= 0, evaluated only where all five values are
 *                   finite and rho > 0.
 * One kernel (40 B/point read once), one 24-byte device-to-host copy; returns after the stream has drained. */
ocfd_status ocfd_check_state(ocfd_ctx *ctx, const double *U, long long host_counts[3]);

/* Row a9 for callers that cannot allocate device memory.  Everything else in this header needs a context, and a
 * context needs a workspace of several fields from the caller; code that must not call cudaMalloc -- a callback inside
 * an application whose own pool already owns all of HBM, a monitoring hook that may not disturb the allocator, a job
 * whose memory budget is spent on the flow fields -- cannot supply one.  This call needs neither: pass the same
 * parameter block a context would get (only nx, ny, nz, ng, grid_kind, metric, metric_plane_stride, dx, dy, dz, gamma,
 * Ma and stream are used; workspace may be NULL; the block must still be one ocfd_init would accept), the state U
 * (device pointer, ghosts not read) and a host pointer for the result.  Same value as ocfd_max_wavespeed (a maximum
 * does not depend on the order it is taken in), NaN for a state with a non-finite wavespeed, and like it the call
 * returns after the stream has drained.  It calls no cudaMalloc, cudaFree or allocating library routine.
 *
 * The reduction's scratch is a fixed array inside the library image: (OCFD_STATIC_WAVESPEED_SLOTS + 32) * 8 bytes =
 * 512.25 KiB on every GPU that loads the library, held until the process exits.  Limits and rules that follow:
 *   - ceil(nx / 128) * ny must not exceed OCFD_STATIC_WAVESPEED_SLOTS; a larger grid is refused with OCFD_EWORKSPACE
 *     and one line on stderr, before anything is launched (use ocfd_max_wavespeed with a context for such grids);
 *   - all calls on one device share the array.  No call depends on what an earlier one left in it, but two calls that
 *     run on the same GPU at the same time (from two threads or on two streams) corrupt each other's result: serialise
 *     them.  Calls made one after the other from one thread are safe, since each returns only when its work is done;
 *   - the first call on each device also looks up the array's device address (host-side work, no allocation); the
 *     device the stream belongs to must be current, and that first call should be made before any stream capture.
 * Errors: OCFD_EINVAL (null pointer, parameters ocfd_init would reject, ny > 65535), OCFD_EWORKSPACE (grid beyond the
 * limit above), OCFD_EUNSUPPORTED (not an sm_100 device), OCFD_ECUDA. */
#define OCFD_STATIC_WAVESPEED_SLOTS 65536
ocfd_status ocfd_max_wavespeed_static(const ocfd_params *p, const double *U, double *host_out);

/* Hybrid-scheme parity report: theta (padded field, interior + the first ghost layer of each face written) and
 * the per-interface scheme flags (0 UD7, 1 WENO7, 2 WENO5): flag_xyz is [3][nz+8][ny+8][nx+8] bytes and
 * flag_xyz[d][point s] is the scheme of interface s+1/2 along direction d, s = -1 .. n-1.  Either output
 * may be NULL.  Device pointers. */
ocfd_status ocfd_debug_sensor(ocfd_ctx *ctx, const double *U, double *theta, unsigned char *flag_xyz);

/* Launch-shape knobs of one context, for A/B measurements; they change no result beyond round-off.  Keys:
 * "zchunk_flux", "zchunk_div", "zchunk_sensor" (planes a CTA of
 * the viscous passes / the stand-alone sensor marches; 0 automatic, else >= 8), "march_seg" (segments a pencil of the
 * marching sweeps is cut into; 0 automatic), "tile_group" (tiles per column group in the CTA numbering of the viscous
 * passes; 0 = 16, a value >= the tiles per row gives the plain x-fastest order).  Unknown key, negative value or a
 * zchunk value between 1 and 7: OCFD_EINVAL. */
ocfd_status ocfd_set_tuning(ocfd_ctx *ctx, const char *key, int value);

/* sizeof(ocfd_params) as compiled, so that a foreign-language mirror of the struct can check itself. */
size_t ocfd_sizeof_params(void);

/* Per-kernel-class device timing with CUDA events recorded on the launch stream around every kernel launch.
 * ocfd_timing(ctx, 1) switches it on (and clears the record), ocfd_timing(ctx, 0) off.  ocfd_timing_read
 * synchronises the stream, adds up the elapsed milliseconds and launch counts per class since the last read
 * into ms[OCFD_NKERNELS] / launches[OCFD_NKERNELS] (host arrays) and clears the record.  Class names:
 * ocfd_kernel_name(id), id = 0 .. OCFD_NKERNELS-1. */
#define OCFD_NKERNELS 10
ocfd_status ocfd_timing(ocfd_ctx *ctx, int enable);
ocfd_status ocfd_timing_read(ocfd_ctx *ctx, double *ms, long long *launches);
const char *ocfd_kernel_name(int id);

/* Number of kernels this context has launched so far (for the bench's gpu_launches claim). */
long long ocfd_launch_count(const ocfd_ctx *ctx);

const char *ocfd_strerror(ocfd_status s);

#ifdef __cplusplus
}
#endif
#endif /* OCFD_H */
