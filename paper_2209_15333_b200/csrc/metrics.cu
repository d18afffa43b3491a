// Derived metric data, built once per context (ocfd_init): alpha_d = (d_x, d_y, d_z)/J of eq. 20-22 (PAPER.md:L161-
// 176) for curvilinear grids, reciprocal 1-D spacings for stretched grids.  The sweeps then never divide by J.
#include "ocfd_internal.cuh"

namespace {

__global__ void k_alpha_tables(GridDesc g, double *__restrict__ tab, long long npts) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x; id < npts; id += stride) {
        const double J = g.met[9][id];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            double *t = tab + 4 * d * g.atab_fs + id;
            t[0] = g.met[3 * d][id] / J;
            t[g.atab_fs] = g.met[3 * d + 1][id] / J;
            t[2 * g.atab_fs] = g.met[3 * d + 2][id] / J;
            t[3 * g.atab_fs] = J;
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
        if (blocks > 148 * 16) blocks = 148 * 16;
        k_alpha_tables<<<blocks, 256, 0, c->stream>>>(g, c->mtab, npts);
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
