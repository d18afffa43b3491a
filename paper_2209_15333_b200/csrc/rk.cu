// Row a8: TVD RK3 stage update, eq. 45: U <- a_s U^n + b_s (U + dt L(U)), interior points.
#include "ocfd_internal.cuh"

namespace {

// out <- a_s Un + b_s (Uin + dt dU).  The buffers rotate (ocfd_rk3_step): no stage copies the state, Uin may be out.
template <int STAGE>
__global__ void __launch_bounds__(256) k_rk_update(GridDesc g, const double *Un, const double *Uin, double *out,
                                                   const double *__restrict__ dU, double dt) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= g.nx || j >= g.ny) return;
    const long long id = pidx(g, i + OCFD_NG, j + OCFD_NG, k + OCFD_NG);
#pragma unroll
    for (int m = 0; m < 5; ++m) {
        const long long q = m * g.np + id;
        const double u = Uin[q], r = dU[q];
        if (STAGE == 0) {
            out[q] = u + dt * r;
        } else if (STAGE == 1) {
            out[q] = 0.75 * Un[q] + 0.25 * (u + dt * r);
        } else {
            out[q] = (1.0 / 3.0) * Un[q] + (2.0 / 3.0) * (u + dt * r);
        }
    }
}

}  // namespace

ocfd_status launch_rk_update(ocfd_ctx *c, const double *Un, const double *Uin, double *out, const double *dU, double dt,
                             int stage) {
    const GridDesc &g = c->g;
    dim3 blk(64, 4, 1), grd((g.nx + 63) / 64, (g.ny + 3) / 4, g.nz);
    OCFD_T0(c, K_RK);
    if (stage == 0) k_rk_update<0><<<grd, blk, 0, c->stream>>>(g, Un, Uin, out, dU, dt);
    else if (stage == 1) k_rk_update<1><<<grd, blk, 0, c->stream>>>(g, Un, Uin, out, dU, dt);
    else k_rk_update<2><<<grd, blk, 0, c->stream>>>(g, Un, Uin, out, dU, dt);
    OCFD_CHECK_LAUNCH(c);
    return OCFD_OK;
}
