// mg_common.cuh -- device-side level descriptor, canonical stencil arithmetic and
// deterministic block reductions shared by all kernels of libmg (CUDA path only;
// nothing here is shared with oracle/).
//
// Arithmetic follows DESIGN.md §3 (C1-C9) with explicit
// round-to-nearest intrinsics (__dadd_rn/__dmul_rn/__fma_rn/__ddiv_rn), which the
// compiler never contracts or reassociates, so every field is reproducible bit for
// bit regardless of how kernels are fused or tiled.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mg {

// One grid level as the kernels see it (passed by value).
struct Lv {
    int nx, ny, nz;
    int bcx, bcy, bcz;          // 1 = homogeneous Neumann on that axis, 0 = periodic
    double h2, ih2;             // C1: h_l^2 and 1/h_l^2
    const double *a;            // level 0: a = 0.5/rho per cell (faces formed on the fly, C2)
    const double *bx, *by, *bz; // levels >= 1: stored minus-face coefficients (C3)
    // R24 (mg_create6): one boundary type per side.  gen != 0 selects the wall logic of the
    // level-generic kernels: wall face = stored wall value, neighbour value 0.0.
    int gen;
    int bcm[3], bcp[3];         // MG_BC_* of the minus / plus side of x, y, z
    const double *wx, *wy, *wz; // levels >= 1: plus-wall face coefficients (wx[j + ny*k], wy[i + nx*k], wz[i + nx*j])
};

// C2w: Dirichlet wall face of a cell with coefficient a (ghost = -p_c, ghost density the cell's)
__device__ __forceinline__ double wall_face(int bc_side, double ac)
{
    return bc_side == 2 ? __dmul_rn(2.0, __dadd_rn(ac, ac)) : 0.0;
}

__device__ __forceinline__ size_t cidx(const Lv &L, int i, int j, int k)
{
    return (size_t)i + (size_t)L.nx * ((size_t)j + (size_t)L.ny * (size_t)k);
}

// The six face coefficients of cell (i,j,k), order x-,x+,y-,y+,z-,z+.
// CELL = true : level 0, beta = a[c] + a[nb], wall face = +0.0 (C2)
// CELL = false: stored minus faces; plus face = neighbour's minus face (wrap); a
//               Neumann axis stores 0 in its wrap face.
template <bool CELL>
__device__ __forceinline__ void faces(const Lv &L, int i, int j, int k, size_t c, size_t cxm,
                                      size_t cxp, size_t cym, size_t cyp, size_t czm, size_t czp,
                                      double b[6])
{
    if (L.gen) {
        // R24: walls of a non-periodic axis carry their own coefficient (bcx/bcy/bcz = walled)
        if (CELL) {
            const double ac = L.a[c];
            b[0] = (L.bcx && i == 0) ? wall_face(L.bcm[0], ac) : __dadd_rn(ac, L.a[cxm]);
            b[1] = (L.bcx && i == L.nx - 1) ? wall_face(L.bcp[0], ac) : __dadd_rn(ac, L.a[cxp]);
            b[2] = (L.bcy && j == 0) ? wall_face(L.bcm[1], ac) : __dadd_rn(ac, L.a[cym]);
            b[3] = (L.bcy && j == L.ny - 1) ? wall_face(L.bcp[1], ac) : __dadd_rn(ac, L.a[cyp]);
            b[4] = (L.bcz && k == 0) ? wall_face(L.bcm[2], ac) : __dadd_rn(ac, L.a[czm]);
            b[5] = (L.bcz && k == L.nz - 1) ? wall_face(L.bcp[2], ac) : __dadd_rn(ac, L.a[czp]);
        } else {
            b[0] = L.bx[c];
            b[1] = (L.bcx && i == L.nx - 1) ? L.wx[(size_t)j + (size_t)L.ny * (size_t)k] : L.bx[cxp];
            b[2] = L.by[c];
            b[3] = (L.bcy && j == L.ny - 1) ? L.wy[(size_t)i + (size_t)L.nx * (size_t)k] : L.by[cyp];
            b[4] = L.bz[c];
            b[5] = (L.bcz && k == L.nz - 1) ? L.wz[(size_t)i + (size_t)L.nx * (size_t)j] : L.bz[czp];
        }
    } else if (CELL) {
        const double ac = L.a[c];
        b[0] = (L.bcx && i == 0) ? 0.0 : __dadd_rn(ac, L.a[cxm]);
        b[1] = (L.bcx && i == L.nx - 1) ? 0.0 : __dadd_rn(ac, L.a[cxp]);
        b[2] = (L.bcy && j == 0) ? 0.0 : __dadd_rn(ac, L.a[cym]);
        b[3] = (L.bcy && j == L.ny - 1) ? 0.0 : __dadd_rn(ac, L.a[cyp]);
        b[4] = (L.bcz && k == 0) ? 0.0 : __dadd_rn(ac, L.a[czm]);
        b[5] = (L.bcz && k == L.nz - 1) ? 0.0 : __dadd_rn(ac, L.a[czp]);
    } else {
        b[0] = L.bx[c];  b[1] = L.bx[cxp];
        b[2] = L.by[c];  b[3] = L.by[cyp];
        b[4] = L.bz[c];  b[5] = L.bz[czp];
    }
}

// C4: S = sum beta*p_nb (nested fma, order x-,x+,y-,y+,z-,z+), D = sum beta (left to right)
__device__ __forceinline__ double stencil_S(const double b[6], double pxm, double pxp, double pym,
                                            double pyp, double pzm, double pzp)
{
    return __fma_rn(b[5], pzp,
           __fma_rn(b[4], pzm,
           __fma_rn(b[3], pyp,
           __fma_rn(b[2], pym,
           __fma_rn(b[1], pxp, __dmul_rn(b[0], pxm))))));
}
__device__ __forceinline__ double stencil_D(const double b[6])
{
    return __dadd_rn(__dadd_rn(__dadd_rn(__dadd_rn(__dadd_rn(b[0], b[1]), b[2]), b[3]), b[4]), b[5]);
}
// C5: Gauss-Seidel value; C6: residual
__device__ __forceinline__ double gs_value(double h2, double f, double S, double D)
{
    return __dmul_rn(__fma_rn(-h2, f, S), __ddiv_rn(1.0, D));
}
// same value through the correctly rounded reciprocal instruction sequence: 1.0/D and
// rcp(D) are both the round-to-nearest reciprocal, hence identical bits
__device__ __forceinline__ double gs_value_rcp(double h2, double f, double S, double D)
{
    return __dmul_rn(__fma_rn(-h2, f, S), __drcp_rn(D));
}
__device__ __forceinline__ double resid_value(double ih2, double f, double S, double D, double p)
{
    return __fma_rn(-ih2, __fma_rn(-D, p, S), f);
}
// C8
__device__ __forceinline__ double lerp(double near, double far)
{
    return __fma_rn(0.25, far, __dmul_rn(0.75, near));
}

// Straightforward global-memory evaluation of S and D at one cell (reference kernels).
template <bool CELL>
__device__ __forceinline__ void stencil_global(const Lv &L, const double *__restrict__ p, int i,
                                               int j, int k, double &S, double &D)
{
    const int im = i == 0 ? L.nx - 1 : i - 1, ip = i == L.nx - 1 ? 0 : i + 1;
    const int jm = j == 0 ? L.ny - 1 : j - 1, jp = j == L.ny - 1 ? 0 : j + 1;
    const int km = k == 0 ? L.nz - 1 : k - 1, kp = k == L.nz - 1 ? 0 : k + 1;
    const size_t c = cidx(L, i, j, k);
    const size_t cxm = cidx(L, im, j, k), cxp = cidx(L, ip, j, k);
    const size_t cym = cidx(L, i, jm, k), cyp = cidx(L, i, jp, k);
    const size_t czm = cidx(L, i, j, km), czp = cidx(L, i, j, kp);
    double b[6];
    faces<CELL>(L, i, j, k, c, cxm, cxp, cym, cyp, czm, czp, b);
    if (L.gen) {            // a wall's neighbour value is 0.0 (C2)
        S = stencil_S(b, (L.bcx && i == 0) ? 0.0 : p[cxm], (L.bcx && i == L.nx - 1) ? 0.0 : p[cxp],
                      (L.bcy && j == 0) ? 0.0 : p[cym], (L.bcy && j == L.ny - 1) ? 0.0 : p[cyp],
                      (L.bcz && k == 0) ? 0.0 : p[czm], (L.bcz && k == L.nz - 1) ? 0.0 : p[czp]);
    } else {
        S = stencil_S(b, p[cxm], p[cxp], p[cym], p[cyp], p[czm], p[czp]);
    }
    D = stencil_D(b);
}

// ---------------------------------------------------------------------------
// Deterministic block reduction (warp shuffles, then one warp over the per-warp
// partials; fixed tree, no atomics).  Result valid in thread 0.
// ---------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = __dadd_rn(v, __shfl_down_sync(0xffffffffu, v, o));
    return v;
}

__device__ __forceinline__ double block_sum(double v, double *smem32)
{
    const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    const int lane = tid & 31, warp = tid >> 5;
    const int nwarp = (blockDim.x * blockDim.y * blockDim.z + 31) >> 5;
    v = warp_sum(v);
    __syncthreads();                    // smem32 may be reused by consecutive calls
    if (lane == 0) smem32[warp] = v;
    __syncthreads();
    if (warp == 0) {
        v = lane < nwarp ? smem32[lane] : 0.0;
        v = warp_sum(v);
    }
    return v;
}

} // namespace mg
