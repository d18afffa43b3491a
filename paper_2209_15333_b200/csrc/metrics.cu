// Derived metric data, built once per context (ocfd_init): for curvilinear grids sigma = |alpha_d| and the unit normal
// k_d = alpha_d/sigma of alpha_d = (d_x, d_y, d_z)/J (eq. 20-22); reciprocal 1-D spacings for
// stretched grids.  The sweeps then never divide nor take a square root for the metrics.
#include "ocfd_internal.cuh"

namespace {

__global__ void k_alpha_tables(GridDesc g, double *__restrict__ tab, double *__restrict__ tabT, long long npts) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x; id < npts; id += stride) {
        const double J = g.met[9][id];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            double *t = tab + 5 * d * g.atab_fs + id;
            const double a1 = g.met[3 * d][id] / J, a2 = g.met[3 * d + 1][id] / J, a3 = g.met[3 * d + 2][id] / J;
            const double sigma = sqrt(a1 * a1 + a2 * a2 + a3 * a3);
            t[0] = a1 / sigma;
            t[g.atab_fs] = a2 / sigma;
            t[2 * g.atab_fs] = a3 / sigma;
            t[3 * g.atab_fs] = sigma;
            t[4 * g.atab_fs] = J;
            if (d == 0) {   // the copy of direction 0 with y contiguous (x sweep)
                const int ip = (int)(id % g.nxp), jp = (int)((id / g.nxp) % g.nyp);
                const long long pl = id / g.sz;
                double *tt = tabT + (pl * g.nxp + ip) * g.nypT + jp;
                tt[0] = a1 / sigma;
                tt[g.atabT_fs] = a2 / sigma;
                tt[2 * g.atabT_fs] = a3 / sigma;
                tt[3 * g.atabT_fs] = sigma;
                tt[4 * g.atabT_fs] = J;
            }
        }
    }
}

__global__ void k_recip_1d(const double *__restrict__ a, double *__restrict__ r, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) r[i] = 1.0 / a[i];
}

}  // namespace

ocfd_status launch_metric_tables(ocfd_ctx *c) {
    const GridDesc &g = c->g;
    if (g.kind == OCFD_GRID_CURVILINEAR) {
        const long long npts = g.atab_fs;
        int blocks = (int)((npts + 255) / 256);
        if (blocks > c->nsm * 16) blocks = c->nsm * 16;
        k_alpha_tables<<<blocks, 256, 0, c->stream>>>(g, c->mtab, const_cast<double *>(g.atabT), npts);
        if (cudaGetLastError() != cudaSuccess) return OCFD_ECUDA;
    } else if (g.kind == OCFD_GRID_STRETCHED) {
        const int n[3] = {g.nxp, g.nyp, g.nzp};
        for (int d = 0; d < 3; ++d) {
            k_recip_1d<<<(n[d] + 255) / 256, 256, 0, c->stream>>>(g.met[4 * d], const_cast<double *>(g.rmet[d]), n[d]);
            if (cudaGetLastError() != cudaSuccess) return OCFD_ECUDA;
        }
    }
    return OCFD_OK;
}
