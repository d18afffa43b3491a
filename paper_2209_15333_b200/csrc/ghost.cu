// Row a1: Dirichlet boundary nodes and the ghost shell (DESIGN section 2 "Ghost fill", R-16).
//
// Two kinds of launches per fill:
//   k_dirichlet<AXIS>   one launch per wall / inflow face, in the face order x-, x+, y-, y+, z-, z+ (a node on an edge
//                       shared by two such faces belongs to the later one, and a wall node next to an inflow face reads
//                       that face's nodes): one thread per node of the face, addressed by its padded coordinates;
//   k_shell             ONE launch for the ghost layers of all six faces.  It is written from the ghost point's side:
//                       every thread owns one point of the shell (the 4-deep slabs beyond the faces, edges and corners
//                       excluded), finds which face it lies behind and how deep, and fetches what that face's condition
//                       prescribes.  Ghost points read interior points only, so the six faces are independent here.
#include "ocfd_internal.cuh"

namespace {

// padded extents / interior extents / strides as small arrays indexed by axis
struct Box {
    int n[3];
    long long st[3];
    long long np;
};
__host__ __device__ inline Box box_of(const GridDesc &g) {
    Box b;
    b.n[0] = g.nx; b.n[1] = g.ny; b.n[2] = g.nz;
    b.st[0] = 1; b.st[1] = g.sy; b.st[2] = g.sz;
    b.np = g.np;
    return b;
}

// what every face prescribes (by value to the kernels): condition, wall temperature, boundary data
struct FaceTable {
    int bc[6];
    double Tw[6];
    const double *inflow[6];   // [5][n_slow + 8][n_fast + 8], conserved variables
    const double *vn[6];       // [n_slow + 8][n_fast + 8] wall-normal velocity or null
};

struct State { double rho, u, v, w, p; };

__device__ __forceinline__ State load_state(const GasDesc &gs, const double *U, long long np, long long at) {
    State s;
    s.rho = U[at];
    const double r = 1.0 / s.rho;
    s.u = U[np + at] * r;
    s.v = U[2 * np + at] * r;
    s.w = U[3 * np + at] * r;
    s.p = gs.gm1 * (U[4 * np + at] - 0.5 * s.rho * (s.u * s.u + s.v * s.v + s.w * s.w));
    return s;
}
__device__ __forceinline__ void store_state(const GasDesc &gs, double *U, long long np, long long at, const State &s) {
    U[at] = s.rho;
    U[np + at] = s.rho * s.u;
    U[2 * np + at] = s.rho * s.v;
    U[3 * np + at] = s.rho * s.w;
    U[4 * np + at] = s.p / gs.gm1 + 0.5 * s.rho * (s.u * s.u + s.v * s.v + s.w * s.w);
}

// position of padded point (ip, jp, kp) inside the 2-D boundary arrays of a face normal to AXIS: the two tangential
// padded coordinates, lower axis fastest
template <int AXIS>
__device__ __forceinline__ long long face_slot(const GridDesc &g, int ip, int jp, int kp) {
    if (AXIS == 0) return (long long)kp * g.nyp + jp;
    if (AXIS == 1) return (long long)kp * g.nxp + ip;
    return (long long)jp * g.nxp + ip;
}
template <int AXIS>
__device__ __forceinline__ long long face_size(const GridDesc &g) {
    if (AXIS == 0) return (long long)g.nzp * g.nyp;
    if (AXIS == 1) return (long long)g.nzp * g.nxp;
    return (long long)g.nyp * g.nxp;
}

// Dirichlet nodes of the face normal to AXIS on side `high` (0: index 0, 1: index n-1).  (a, b) run over the two
// tangential axes, lower axis on threadIdx.x.
template <int KIND, int AXIS>
__global__ void k_dirichlet(const GridDesc g, const GasDesc gs, const int high, const int bc, const double Tw,
                            const double *__restrict__ vn, const double *__restrict__ inflow, double *__restrict__ U) {
    const Box bx = box_of(g);
    constexpr int TA = AXIS == 0 ? 1 : 0, TB = AXIS == 2 ? 1 : 2;
    const int a = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y * blockDim.y + threadIdx.y;
    if (a >= bx.n[TA] || b >= bx.n[TB]) return;
    int c[3];
    c[AXIS] = OCFD_NG + (high ? bx.n[AXIS] - 1 : 0);
    c[TA] = OCFD_NG + a;
    c[TB] = OCFD_NG + b;
    const long long at = pidx(g, c[0], c[1], c[2]);
    const long long slot = face_slot<AXIS>(g, c[0], c[1], c[2]);
    if (bc == OCFD_BC_SUPERSONIC_INFLOW) {
        const long long fs = face_size<AXIS>(g);
#pragma unroll
        for (int m = 0; m < 5; ++m) U[m * bx.np + at] = inflow[m * fs + slot];
        return;
    }
    // isothermal wall: T = T_w, zero pressure gradient to second order (p0 = (4 p1 - p2)/3), velocity = blowing /
    // suction along the unit normal that points into the fluid (zero without it)
    const long long inward = high ? -bx.st[AXIS] : bx.st[AXIS];
    const State s1 = load_state(gs, U, bx.np, at + inward), s2 = load_state(gs, U, bx.np, at + 2 * inward);
    State s;
    s.p = (4.0 * s1.p - s2.p) / 3.0;
    s.rho = gs.gM2 * s.p / Tw;
    s.u = s.v = s.w = 0.0;
    if (vn) {
        double m1, m2, m3;
        Met<KIND>::row(g, AXIS, c[0], c[1], c[2], m1, m2, m3);
        const double len = sqrt(m1 * m1 + m2 * m2 + m3 * m3), sgn = high ? -1.0 : 1.0;
        const double q = vn[slot];
        s.u = q * sgn * m1 / len;
        s.v = q * sgn * m2 / len;
        s.w = q * sgn * m3 / len;
    }
    store_state(gs, U, bx.np, at, s);
}

// One ghost point behind the face normal to AXIS: `depth` = 1..4 layers outside, `high` = side.
template <int AXIS>
__device__ __forceinline__ void fill_ghost_point(const GridDesc &g, const GasDesc &gs, const FaceTable &ft, double *U,
                                                 int ip, int jp, int kp, int high, int depth) {
    const Box bx = box_of(g);
    const int face = 2 * AXIS + high;
    const long long at = pidx(g, ip, jp, kp);
    const long long inward = high ? -bx.st[AXIS] : bx.st[AXIS];
    const long long node = at + depth * inward;           // the boundary node this ghost point hangs on
    const int bc = ft.bc[face];
    if (bc == OCFD_BC_PERIODIC) {                           // image: one period further in
        const long long src = at + (long long)bx.n[AXIS] * inward;
#pragma unroll
        for (int m = 0; m < 5; ++m) U[m * bx.np + at] = U[m * bx.np + src];
    } else if (bc == OCFD_BC_EXTRAP_OUTFLOW) {              // zeroth-order extrapolation
#pragma unroll
        for (int m = 0; m < 5; ++m) U[m * bx.np + at] = U[m * bx.np + node];
    } else if (bc == OCFD_BC_SUPERSONIC_INFLOW) {           // the prescribed profile
        const long long slot = face_slot<AXIS>(g, ip, jp, kp), fs = face_size<AXIS>(g);
        const double *in = ft.inflow[face];
#pragma unroll
        for (int m = 0; m < 5; ++m) U[m * bx.np + at] = in[m * fs + slot];
    } else {                                                // wall: velocity odd about the wall value, T about T_w, p even
        const State w0 = load_state(gs, U, bx.np, node), im = load_state(gs, U, bx.np, node + depth * inward);
        const double Tim = gs.gM2 * im.p / im.rho;
        State s;
        s.u = 2.0 * w0.u - im.u;
        s.v = 2.0 * w0.v - im.v;
        s.w = 2.0 * w0.w - im.w;
        s.p = im.p;
        s.rho = gs.gM2 * s.p / (2.0 * ft.Tw[face] - Tim);
        store_state(gs, U, bx.np, at, s);
    }
}

// The whole ghost shell.  Threads are numbered through three slab families: points behind the x faces (8 per interior
// (j, k) line, the ghost index fastest), behind the y faces and behind the z faces (x fastest in both).
__global__ void k_shell(const GridDesc g, const GasDesc gs, const FaceTable ft, double *__restrict__ U) {
    const long long cx = 8ll * g.ny * g.nz, cy = 8ll * g.nx * g.nz, cz = 8ll * g.nx * g.ny;
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t < cx) {
        const int e = (int)(t % 8), j = (int)((t / 8) % g.ny), k = (int)(t / (8ll * g.ny));
        const int high = e >= OCFD_NG, depth = high ? e - OCFD_NG + 1 : OCFD_NG - e;
        fill_ghost_point<0>(g, gs, ft, U, high ? g.nx + OCFD_NG + e - OCFD_NG : e, j + OCFD_NG, k + OCFD_NG, high, depth);
        return;
    }
    t -= cx;
    if (t < cy) {
        const int i = (int)(t % g.nx), e = (int)((t / g.nx) % 8), k = (int)(t / (8ll * g.nx));
        const int high = e >= OCFD_NG, depth = high ? e - OCFD_NG + 1 : OCFD_NG - e;
        fill_ghost_point<1>(g, gs, ft, U, i + OCFD_NG, high ? g.ny + OCFD_NG + e - OCFD_NG : e, k + OCFD_NG, high, depth);
        return;
    }
    t -= cy;
    if (t < cz) {
        const int i = (int)(t % g.nx), j = (int)((t / g.nx) % g.ny), e = (int)(t / ((long long)g.nx * g.ny));
        const int high = e >= OCFD_NG, depth = high ? e - OCFD_NG + 1 : OCFD_NG - e;
        fill_ghost_point<2>(g, gs, ft, U, i + OCFD_NG, j + OCFD_NG, high ? g.nz + OCFD_NG + e - OCFD_NG : e, high, depth);
    }
}

template <int KIND>
void launch_dirichlet(ocfd_ctx *c, int face, double *U) {
    const GridDesc &g = c->g;
    const int axis = face / 2, high = face % 2, bc = c->p.bc[face];
    const int n[3] = {g.nx, g.ny, g.nz};
    const int na = n[axis == 0 ? 1 : 0], nb = n[axis == 2 ? 1 : 2];
    // x faces: threadIdx.x runs along y (strided in memory): narrow blocks
    const dim3 blk(axis == 0 ? 8 : 32, axis == 0 ? 16 : 4, 1), grd((na + blk.x - 1) / blk.x, (nb + blk.y - 1) / blk.y, 1);
    const double Tw = c->p.T_wall[face];
    const double *vn = c->p.wall_vn[face], *in = c->p.inflow[face];
    if (axis == 0) k_dirichlet<KIND, 0><<<grd, blk, 0, c->stream>>>(g, c->gas, high, bc, Tw, vn, in, U);
    else if (axis == 1) k_dirichlet<KIND, 1><<<grd, blk, 0, c->stream>>>(g, c->gas, high, bc, Tw, vn, in, U);
    else k_dirichlet<KIND, 2><<<grd, blk, 0, c->stream>>>(g, c->gas, high, bc, Tw, vn, in, U);
}

}  // namespace

ocfd_status launch_fill_ghosts(ocfd_ctx *c, double *U) {
    const GridDesc &g = c->g;
    FaceTable ft;
    for (int f = 0; f < 6; ++f) {
        ft.bc[f] = c->p.bc[f];
        ft.Tw[f] = c->p.T_wall[f];
        ft.inflow[f] = c->p.inflow[f];
        ft.vn[f] = c->p.wall_vn[f];
    }
    for (int f = 0; f < 6; ++f) {
        if (ft.bc[f] != OCFD_BC_WALL_ISOTHERMAL && ft.bc[f] != OCFD_BC_SUPERSONIC_INFLOW) continue;
        OCFD_T0(c, K_GHOST);
        switch (g.kind) {
            case OCFD_GRID_UNIFORM: launch_dirichlet<OCFD_GRID_UNIFORM>(c, f, U); break;
            case OCFD_GRID_STRETCHED: launch_dirichlet<OCFD_GRID_STRETCHED>(c, f, U); break;
            default: launch_dirichlet<OCFD_GRID_CURVILINEAR>(c, f, U);
        }
        OCFD_CHECK_LAUNCH(c);
    }
    const long long total = 8ll * ((long long)g.ny * g.nz + (long long)g.nx * g.nz + (long long)g.nx * g.ny);
    const int nt = 256;
    OCFD_T0(c, K_GHOST);
    k_shell<<<(unsigned)((total + nt - 1) / nt), nt, 0, c->stream>>>(g, c->gas, ft, U);
    OCFD_CHECK_LAUNCH(c);
    return OCFD_OK;
}
