// mg_project_kernels.cuh -- the two steps either side of the pressure solve in the projection
// method (eq. 1-2, BASELINE.json north_star):
//   k_project_rhs     : f = div(u*)/dt from the staggered velocity                 (C10)
//   k_project_correct : u -= dt * beta_face * grad p with the level-0 faces         (C11)
// Staggering (R21): u[i,j,k] sits on the MINUS x-face of cell (i,j,k), v on the minus y-face,
// w on the minus z-face; a cell's plus face is the next cell's minus face (wrap).  On a
// Neumann axis the wrap face is the wall: its beta is 0, so the correction never moves it.
//
// Both are single streaming passes with 16-byte accesses: a thread owns an aligned x-pair,
// the x-neighbour word comes from the adjacent lane by shuffle (edge lanes load one scalar),
// the y / z neighbours are one more row / plane load each (L1 / L2 hits).
// Algorithmic bytes per cell: rhs 24 + 8; correct 16 (p, a) + 48 (u, v, w read and written).
#pragma once
#include "mg_common.cuh"

namespace mg {

struct PjArgs {
    int nx, ny, nz;
    int bcx, bcy, bcz;
    double sc;                 // rhs: 1/(h*dt);  correct: dt/h
    const double *a;           // correct: a = 0.5/rho
    const double *p;           // correct
    double *u, *v, *w;         // rhs: read;  correct: read and written
    double *f;                 // rhs: out
};

__device__ __forceinline__ double2 pj_ld2(const double *base, size_t idx)
{
    return *reinterpret_cast<const double2 *>(base + idx);
}

// grid: (ceil(nx/64), ceil(ny/8), nz), block (32, 8)
__global__ void __launch_bounds__(256) k_project_rhs(PjArgs A)
{
    const int lx = threadIdx.x;
    const int x0r = (blockIdx.x * 32 + lx) * 2, jr = blockIdx.y * 8 + threadIdx.y, k = blockIdx.z;
    const bool valid = x0r < A.nx && jr < A.ny;
    const int x0 = min(x0r, A.nx - 2), j = min(jr, A.ny - 1);
    const int xr = x0 + 2 == A.nx ? 0 : x0 + 2;
    const int jp = j == A.ny - 1 ? 0 : j + 1, kp = k == A.nz - 1 ? 0 : k + 1;
    const size_t plane = (size_t)A.nx * A.ny;
    const size_t c = (size_t)x0 + (size_t)A.nx * j + plane * k;
    const double2 u0 = pj_ld2(A.u, c);
    const double2 v0 = pj_ld2(A.v, c), v1 = pj_ld2(A.v, (size_t)x0 + (size_t)A.nx * jp + plane * k);
    const double2 w0 = pj_ld2(A.w, c), w1 = pj_ld2(A.w, (size_t)x0 + (size_t)A.nx * j + plane * kp);
    double ur = __shfl_down_sync(0xffffffffu, u0.x, 1);          // u on the plus face of the odd cell
    if (lx == 31 || x0 + 2 >= A.nx) ur = A.u[(size_t)xr + (size_t)A.nx * j + plane * k];
    if (!valid) return;
    double2 f;
    f.x = __dmul_rn(__dadd_rn(__dadd_rn(__dsub_rn(u0.y, u0.x), __dsub_rn(v1.x, v0.x)), __dsub_rn(w1.x, w0.x)), A.sc);
    f.y = __dmul_rn(__dadd_rn(__dadd_rn(__dsub_rn(ur, u0.y), __dsub_rn(v1.y, v0.y)), __dsub_rn(w1.y, w0.y)), A.sc);
    *reinterpret_cast<double2 *>(A.f + c) = f;
}

__global__ void __launch_bounds__(256) k_project_correct(PjArgs A)
{
    const int lx = threadIdx.x;
    const int x0r = (blockIdx.x * 32 + lx) * 2, jr = blockIdx.y * 8 + threadIdx.y, k = blockIdx.z;
    const bool valid = x0r < A.nx && jr < A.ny;
    const int x0 = min(x0r, A.nx - 2), j = min(jr, A.ny - 1);
    const int xl = x0 == 0 ? A.nx - 1 : x0 - 1;
    const int jm = j == 0 ? A.ny - 1 : j - 1, km = k == 0 ? A.nz - 1 : k - 1;
    const size_t plane = (size_t)A.nx * A.ny;
    const size_t c = (size_t)x0 + (size_t)A.nx * j + plane * k;
    const size_t cym = (size_t)x0 + (size_t)A.nx * jm + plane * k, czm = (size_t)x0 + (size_t)A.nx * j + plane * km;
    const double2 pc = pj_ld2(A.p, c), pym = pj_ld2(A.p, cym), pzm = pj_ld2(A.p, czm);
    const double2 ac = pj_ld2(A.a, c), aym = pj_ld2(A.a, cym), azm = pj_ld2(A.a, czm);
    double pl = __shfl_up_sync(0xffffffffu, pc.y, 1), al = __shfl_up_sync(0xffffffffu, ac.y, 1);
    if (lx == 0) {
        const size_t cl = (size_t)xl + (size_t)A.nx * j + plane * k;
        pl = A.p[cl]; al = A.a[cl];
    }
    if (!valid) return;
    const bool wx = A.bcx && x0 == 0, wy = A.bcy && j == 0, wz = A.bcz && k == 0;
    // level-0 minus faces (C2): beta = a_c + a_nb, wall face +0.0
    const double bx0 = wx ? 0.0 : __dadd_rn(ac.x, al), bx1 = __dadd_rn(ac.y, ac.x);
    const double by0 = wy ? 0.0 : __dadd_rn(ac.x, aym.x), by1 = wy ? 0.0 : __dadd_rn(ac.y, aym.y);
    const double bz0 = wz ? 0.0 : __dadd_rn(ac.x, azm.x), bz1 = wz ? 0.0 : __dadd_rn(ac.y, azm.y);
    const double g = -A.sc;
    double2 u = pj_ld2(A.u, c), v = pj_ld2(A.v, c), w = pj_ld2(A.w, c);
    u.x = __fma_rn(g, __dmul_rn(bx0, __dsub_rn(pc.x, pl)), u.x);
    u.y = __fma_rn(g, __dmul_rn(bx1, __dsub_rn(pc.y, pc.x)), u.y);
    v.x = __fma_rn(g, __dmul_rn(by0, __dsub_rn(pc.x, pym.x)), v.x);
    v.y = __fma_rn(g, __dmul_rn(by1, __dsub_rn(pc.y, pym.y)), v.y);
    w.x = __fma_rn(g, __dmul_rn(bz0, __dsub_rn(pc.x, pzm.x)), w.x);
    w.y = __fma_rn(g, __dmul_rn(bz1, __dsub_rn(pc.y, pzm.y)), w.y);
    *reinterpret_cast<double2 *>(A.u + c) = u;
    *reinterpret_cast<double2 *>(A.v + c) = v;
    *reinterpret_cast<double2 *>(A.w + c) = w;
}

} // namespace mg
