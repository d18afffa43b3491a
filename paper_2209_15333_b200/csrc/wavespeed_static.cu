// ocfd_max_wavespeed_static (include/ocfd.h): row a9 once more, for callers that cannot allocate device memory.
//
// Who that is: every other entry point needs an ocfd_ctx, and a context needs a caller-supplied workspace of several
// fields.  Code that runs where cudaMalloc is off limits has no way to get one: a callback of an application that has
// handed all of HBM to its own pool, a monitoring hook that must not disturb the allocator's state, a process working
// under a fixed memory budget that is already spent on the flow fields.  Such a caller still holds U and the metric
// arrays (they are its own data) and wants Lambda for dt = CFL / Lambda.  This entry point takes exactly those and
// nothing else: no context, no workspace, and it calls no cudaMalloc / cudaFree / allocating library routine.
//
// The scratch the reduction needs (one partial maximum per thread block, then the result) lives in a file-scope
// __device__ array of fixed size below.  Consequences a caller has to know:
//   * the array is part of the library image: every GPU that loads libocfd_b200.so holds its 512.25 KiB until the
//     process exits, whether this entry point is ever called or not;
//   * its size bounds the grid: ceil(nx/128) * ny columns of thread blocks must not exceed
//     OCFD_STATIC_WAVESPEED_SLOTS (65536), otherwise the call is refused (OCFD_EWORKSPACE, with a line on stderr);
//   * all calls on one device share it.  Nothing in it has to start at zero -- a call writes every slot before it
//     reads it, so what the previous call left behind is never seen -- but two calls that are in flight on the same GPU
//     at the same time (two host threads, or two streams) overwrite each other's partial maxima.  A call returns only
//     after its stream has drained, so calls made one after the other from one thread never overlap; anything else the
//     caller must serialise;
//   * the first call on each device looks up the array's device address (a host-side query, no kernel, no allocation).
//     Make that first call outside any stream capture.
#include <mutex>

#include "ocfd_internal.cuh"
#include "schemes.cuh"

namespace {

constexpr int WSS_NT = 128;                                  // threads per block, one (i, j) column each
constexpr int WSS_SLOTS = OCFD_STATIC_WAVESPEED_SLOTS;       // partial maxima (one per thread block)
constexpr int WSS_RESULT = WSS_SLOTS;                        // slot of the final value, on a 256-byte line of its own
constexpr unsigned long long WSS_NAN = 0x7ff8000000000000ull;

// The scratch.  In device code this name is the array; in host code it is only a handle for cudaGetSymbolAddress.
static __device__ __align__(256) unsigned long long g_wss_scratch[WSS_SLOTS + 32];

// Same march as k_wavespeed (prim.cu): a thread owns one (i, j) column and walks a chunk of z planes (R-17).  Instead of
// an atomic on one word the block leaves its maximum, as the ordered bit pattern of a non-negative double, in the slot
// of its own linear index.
template <int KIND>
__global__ void __launch_bounds__(WSS_NT) k_wavespeed_partials(GridDesc g, GasDesc gs, const double *__restrict__ U,
                                                               unsigned long long *__restrict__ partial, int zchunk) {
    __shared__ unsigned long long warp_best[WSS_NT / 32];
    const int i = blockIdx.x * WSS_NT + threadIdx.x, j = blockIdx.y;
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
            bad |= !(s == s);   // fmax would drop a NaN: a blown-up state must come back as NaN, not as a finite Lambda
            best = fmax(best, s);
        }
    }
    for (int o = 16; o > 0; o >>= 1) best = fmax(best, __shfl_xor_sync(0xffffffffu, best, o));
    bad = __any_sync(0xffffffffu, bad);
    if ((threadIdx.x & 31) == 0) warp_best[threadIdx.x >> 5] = bad ? WSS_NAN : (unsigned long long)__double_as_longlong(best);
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long m = warp_best[0];
        for (int q = 1; q < WSS_NT / 32; ++q) m = max(m, warp_best[q]);
        partial[((long long)blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x] = m;
    }
}

// One block folds the n partial maxima into the result slot.  Device code may name the array directly.
__global__ void __launch_bounds__(1024) k_wavespeed_fold(int n) {
    __shared__ unsigned long long warp_best[32];
    unsigned long long m = 0;
    for (int q = threadIdx.x; q < n; q += 1024) m = max(m, g_wss_scratch[q]);
    for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) warp_best[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x < 32) {
        m = warp_best[threadIdx.x];
        for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (threadIdx.x == 0) g_wss_scratch[WSS_RESULT] = m;
    }
}

// Per-device set-up, done by the first call on that device with that device current: the device address of the
// scratch array (the host-side name is not one) and the SM count the launch shape is sized for.
constexpr int WSS_MAX_DEVICES = 64;
struct DeviceSetup { unsigned long long *scratch; int nsm; };
DeviceSetup g_setup[WSS_MAX_DEVICES] = {};
std::mutex g_setup_lock;

ocfd_status device_setup(DeviceSetup *out) {
    int dev = 0, major = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return OCFD_ECUDA;
    if (dev < 0 || dev >= WSS_MAX_DEVICES) return OCFD_EUNSUPPORTED;
    std::lock_guard<std::mutex> hold(g_setup_lock);
    if (!g_setup[dev].scratch) {
        if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) return OCFD_ECUDA;
        if (major < 10) return OCFD_EUNSUPPORTED;   // sm_100a only, as everywhere in this library
        if (cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || nsm <= 0) return OCFD_ECUDA;
        void *ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&ptr, g_wss_scratch);
        if (e != cudaSuccess || !ptr) {
            fprintf(stderr, "libocfd_b200: ocfd_max_wavespeed_static: cudaGetSymbolAddress failed on device %d: %s\n", dev,
                    cudaGetErrorString(e));
            return OCFD_ECUDA;
        }
        g_setup[dev].nsm = nsm;
        g_setup[dev].scratch = (unsigned long long *)ptr;
    }
    *out = g_setup[dev];
    return OCFD_OK;
}

}  // namespace

extern "C" ocfd_status ocfd_max_wavespeed_static(const ocfd_params *p, const double *U, double *host_out) {
    if (!U || !host_out) return OCFD_EINVAL;
    if (ocfd_workspace_bytes(p) == 0) return OCFD_EINVAL;   // the validation every context goes through (pure, host only)
    if (p->ny > 65535) return OCFD_EINVAL;                  // ny is a grid dimension of the launch
    // the limit of the fixed scratch, checked before anything touches the GPU
    const long long cols = (long long)((p->nx + WSS_NT - 1) / WSS_NT) * p->ny;
    if (cols > WSS_SLOTS) {
        fprintf(stderr, "libocfd_b200: ocfd_max_wavespeed_static: grid %d x %d x %d needs ceil(nx/%d) * ny = %lld scratch "
                        "slots, the static array holds %d; use ocfd_max_wavespeed with a context instead\n",
                p->nx, p->ny, p->nz, WSS_NT, cols, WSS_SLOTS);
        return OCFD_EWORKSPACE;
    }
    DeviceSetup ds;
    ocfd_status st = device_setup(&ds);
    if (st != OCFD_OK) return st;

    GridDesc g = {};
    g.nx = p->nx; g.ny = p->ny; g.nz = p->nz;
    g.nxp = p->nx + 8; g.nyp = p->ny + 8; g.nzp = p->nz + 8;
    g.sy = g.nxp; g.sz = (long long)g.nxp * g.nyp; g.np = g.sz * g.nzp;
    g.kind = p->grid_kind;
    for (int q = 0; q < 10; ++q) g.met[q] = p->metric[q];
    g.msk = p->metric_plane_stride;
    if (p->grid_kind == OCFD_GRID_UNIFORM) {
        g.ux = 1.0 / p->dx; g.uy = 1.0 / p->dy; g.uz = 1.0 / p->dz;
        g.uJ = (g.ux * g.uy) * g.uz;
    }
    GasDesc gs = {};
    gs.gamma = p->gamma; gs.gm1 = p->gamma - 1.0; gs.Ma = p->Ma; gs.gM2 = p->gamma * p->Ma * p->Ma; gs.invMa = 1.0 / p->Ma;

    // z chunks as in the context path (long enough to amortise the per-column metric work, short enough to fill the
    // SMs a few times over), then lengthened until the thread blocks fit the scratch slots
    int zc = g.nz;
    while (zc > 32 && cols * ((g.nz + zc - 1) / zc) < 8ll * ds.nsm) zc = (zc + 1) / 2;
    if (zc > 64) zc = 64;
    while (cols * ((g.nz + zc - 1) / zc) > WSS_SLOTS) zc = zc * 2 < g.nz ? zc * 2 : g.nz;   // ends: cols <= WSS_SLOTS
    const dim3 grd((g.nx + WSS_NT - 1) / WSS_NT, g.ny, (g.nz + zc - 1) / zc);
    const int nblocks = (int)(cols * grd.z);
    cudaStream_t stream = (cudaStream_t)p->stream;
    switch (g.kind) {
        case OCFD_GRID_UNIFORM: k_wavespeed_partials<OCFD_GRID_UNIFORM><<<grd, WSS_NT, 0, stream>>>(g, gs, U, ds.scratch, zc); break;
        case OCFD_GRID_STRETCHED: k_wavespeed_partials<OCFD_GRID_STRETCHED><<<grd, WSS_NT, 0, stream>>>(g, gs, U, ds.scratch, zc); break;
        default: k_wavespeed_partials<OCFD_GRID_CURVILINEAR><<<grd, WSS_NT, 0, stream>>>(g, gs, U, ds.scratch, zc);
    }
    if (ocfd_launch_failed(__FILE__, __LINE__)) return OCFD_ECUDA;
    k_wavespeed_fold<<<1, 1024, 0, stream>>>(nblocks);
    if (ocfd_launch_failed(__FILE__, __LINE__)) return OCFD_ECUDA;
    if (cudaMemcpyAsync(host_out, ds.scratch + WSS_RESULT, sizeof(double), cudaMemcpyDeviceToHost, stream) != cudaSuccess)
        return OCFD_ECUDA;
    if (cudaStreamSynchronize(stream) != cudaSuccess) return OCFD_ECUDA;
    return OCFD_OK;
}
