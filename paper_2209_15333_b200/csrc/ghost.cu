// Row a1: Dirichlet boundary nodes and ghost-layer fill (DESIGN section 2 "Ghost fill", R-16).
#include "ocfd_internal.cuh"

namespace {

struct FaceGeom {
    int d, lo;          // normal axis, 1 for the minus face
    int n, n1, n2;      // points along normal, fast tangential, slow tangential axes
    long long sd, s1, s2;
    long long in;       // step into the domain
    int b;              // boundary node index along d
    long long pitch2, fnp;  // padded 2-D face arrays: [n2+8][n1+8]
};

__host__ FaceGeom face_geom(const GridDesc &g, int f) {
    FaceGeom F;
    F.d = f / 2;
    F.lo = (f % 2 == 0);
    int t1 = F.d == 0 ? 1 : 0, t2 = F.d == 2 ? 1 : 2;
    const int n[3] = {g.nx, g.ny, g.nz};
    const long long s[3] = {1, g.sy, g.sz};
    F.n = n[F.d]; F.n1 = n[t1]; F.n2 = n[t2];
    F.sd = s[F.d]; F.s1 = s[t1]; F.s2 = s[t2];
    F.in = F.lo ? F.sd : -F.sd;
    F.b = F.lo ? 0 : F.n - 1;
    F.pitch2 = F.n1 + 2 * OCFD_NG;
    F.fnp = (long long)(F.n2 + 2 * OCFD_NG) * F.pitch2;
    return F;
}

struct Prim5 { double rho, u, v, w, p, T; };

__device__ __forceinline__ Prim5 prim_at(const GasDesc &gs, const double *U, long long np, long long id) {
    Prim5 q;
    q.rho = U[id];
    double ir = 1.0 / q.rho;
    q.u = U[np + id] * ir;
    q.v = U[2 * np + id] * ir;
    q.w = U[3 * np + id] * ir;
    q.p = gs.gm1 * (U[4 * np + id] - 0.5 * q.rho * (q.u * q.u + q.v * q.v + q.w * q.w));
    q.T = gs.gM2 * q.p * ir;
    return q;
}
__device__ __forceinline__ void set_cons(const GasDesc &gs, double *U, long long np, long long id, double rho, double u,
                                         double v, double w, double p) {
    U[id] = rho;
    U[np + id] = rho * u;
    U[2 * np + id] = rho * v;
    U[3 * np + id] = rho * w;
    U[4 * np + id] = p / gs.gm1 + 0.5 * rho * (u * u + v * v + w * w);
}

__device__ __forceinline__ long long node_index(const GridDesc &g, const FaceGeom &F, int c1, int c2) {
    return (long long)OCFD_NG * (1 + g.sy + g.sz) + (long long)F.b * F.sd + (long long)c1 * F.s1 + (long long)c2 * F.s2;
}

// Dirichlet nodes of one face (wall or inflow)
template <int KIND>
__global__ void k_bc_nodes(GridDesc g, GasDesc gs, FaceGeom F, int bc, double Tw, const double *__restrict__ wall_vn,
                           const double *__restrict__ inflow, double *__restrict__ U) {
    int c1 = blockIdx.x * blockDim.x + threadIdx.x;
    int c2 = blockIdx.y * blockDim.y + threadIdx.y;
    if (c1 >= F.n1 || c2 >= F.n2) return;
    long long id0 = node_index(g, F, c1, c2);
    long long fid = (long long)(c2 + OCFD_NG) * F.pitch2 + (c1 + OCFD_NG);
    if (bc == OCFD_BC_WALL_ISOTHERMAL) {
        Prim5 q1 = prim_at(gs, U, g.np, id0 + F.in), q2 = prim_at(gs, U, g.np, id0 + 2 * F.in);
        double p0 = (4.0 * q1.p - q2.p) / 3.0;
        double rho0 = gs.gM2 * p0 / Tw;
        double u = 0.0, v = 0.0, w = 0.0;
        if (wall_vn) {
            int ip = (int)(id0 % g.sy), jp = (int)((id0 / g.sy) % g.nyp), kp = (int)(id0 / g.sz);
            double a1, a2, a3;
            Met<KIND>::row(g, F.d, ip, jp, kp, a1, a2, a3);
            double s = sqrt(a1 * a1 + a2 * a2 + a3 * a3), sg = F.lo ? 1.0 : -1.0;
            double vn = wall_vn[fid];
            u = vn * sg * a1 / s; v = vn * sg * a2 / s; w = vn * sg * a3 / s;
        }
        set_cons(gs, U, g.np, id0, rho0, u, v, w, p0);
    } else {  // inflow
        for (int m = 0; m < 5; ++m) U[m * g.np + id0] = inflow[m * F.fnp + fid];
    }
}

// ghost layers of one face
__global__ void k_bc_ghosts(GridDesc g, GasDesc gs, FaceGeom F, int bc, double Tw, const double *__restrict__ inflow,
                            double *__restrict__ U) {
    int c1 = blockIdx.x * blockDim.x + threadIdx.x;
    int c2 = blockIdx.y * blockDim.y + threadIdx.y;
    int gl = blockIdx.z + 1;  // ghost layer 1..4
    if (c1 >= F.n1 || c2 >= F.n2) return;
    long long id0 = node_index(g, F, c1, c2);
    long long idg = id0 - gl * F.in;
    if (bc == OCFD_BC_PERIODIC) {
        long long src = idg + (F.lo ? (long long)F.n * F.sd : -(long long)F.n * F.sd);
        for (int m = 0; m < 5; ++m) U[m * g.np + idg] = U[m * g.np + src];
    } else if (bc == OCFD_BC_EXTRAP_OUTFLOW) {
        for (int m = 0; m < 5; ++m) U[m * g.np + idg] = U[m * g.np + id0];
    } else if (bc == OCFD_BC_SUPERSONIC_INFLOW) {
        long long fid = (long long)(c2 + OCFD_NG) * F.pitch2 + (c1 + OCFD_NG);
        for (int m = 0; m < 5; ++m) U[m * g.np + idg] = inflow[m * F.fnp + fid];
    } else {  // isothermal wall: u mirrored about the wall value, T about T_w, p even
        Prim5 q0 = prim_at(gs, U, g.np, id0), qm = prim_at(gs, U, g.np, id0 + gl * F.in);
        double u = 2.0 * q0.u - qm.u, v = 2.0 * q0.v - qm.v, w = 2.0 * q0.w - qm.w;
        double T = 2.0 * Tw - qm.T, p = qm.p;
        set_cons(gs, U, g.np, idg, gs.gM2 * p / T, u, v, w, p);
    }
}

}  // namespace

ocfd_status launch_fill_ghosts(ocfd_ctx *c, double *U) {
    const GridDesc &g = c->g;
    for (int pass = 0; pass < 2; ++pass)
        for (int f = 0; f < 6; ++f) {
            FaceGeom F = face_geom(g, f);
            int bc = c->p.bc[f];
            // x-faces: the fast tangential axis is y (strided); keep blocks small there
            dim3 blk(F.d == 0 ? 8 : 32, F.d == 0 ? 16 : 4, 1);
            dim3 grd((F.n1 + blk.x - 1) / blk.x, (F.n2 + blk.y - 1) / blk.y, 1);
            if (pass == 0) {
                if (bc != OCFD_BC_WALL_ISOTHERMAL && bc != OCFD_BC_SUPERSONIC_INFLOW) continue;
                OCFD_T0(c, K_GHOST);
                switch (g.kind) {
                    case OCFD_GRID_UNIFORM:
                        k_bc_nodes<OCFD_GRID_UNIFORM><<<grd, blk, 0, c->stream>>>(g, c->gas, F, bc, c->p.T_wall[f], c->p.wall_vn[f], c->p.inflow[f], U);
                        break;
                    case OCFD_GRID_STRETCHED:
                        k_bc_nodes<OCFD_GRID_STRETCHED><<<grd, blk, 0, c->stream>>>(g, c->gas, F, bc, c->p.T_wall[f], c->p.wall_vn[f], c->p.inflow[f], U);
                        break;
                    default:
                        k_bc_nodes<OCFD_GRID_CURVILINEAR><<<grd, blk, 0, c->stream>>>(g, c->gas, F, bc, c->p.T_wall[f], c->p.wall_vn[f], c->p.inflow[f], U);
                }
            } else {
                grd.z = OCFD_NG;
                OCFD_T0(c, K_GHOST);
                k_bc_ghosts<<<grd, blk, 0, c->stream>>>(g, c->gas, F, bc, c->p.T_wall[f], c->p.inflow[f], U);
            }
            OCFD_CHECK_LAUNCH(c);
        }
    return OCFD_OK;
}
