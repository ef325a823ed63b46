// mg_pcg_kernels.cuh -- the pieces of the MG-preconditioned conjugate gradient iteration
// (R22, C12-C14) that the V-cycle path does not have: the adjoint
// restriction R' = (1/8) P^T of the trilinear prolongation, the operator application, and the
// vector updates and dot products of the CG recurrence.  Level-generic, straight global-memory
// kernels: the symmetric cycle is the weaker preconditioner on the paper's workloads (DESIGN.md
// section 8), so this path is built for completeness and parity, not tuned.
#pragma once
#include "mg_common.cuh"
#include "mg_ref_kernels.cuh"

namespace mg {

// C14: the four fine indices 2I-1 .. 2I+2 that can carry coarse index I in the prolongation,
// wrapped, or (beyond a Neumann wall) absent: weight 0.  w_q = 0.75 [near(i_q) = I] + 0.25 [far(i_q) = I].
__device__ __forceinline__ void pt_stencil(int I, int fn, int cn, int neumann, int idx[4], double w[4])
{
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        int i = 2 * I - 1 + q;
        bool outside = false;
        if (i < 0) { if (neumann) { outside = true; i = 0; } else i += fn; }
        if (i >= fn) { if (neumann) { outside = true; i = fn - 1; } else i -= fn; }
        idx[q] = i;
        const int near = i >> 1;
        const int far = far_index(near, i & 1, cn, neumann);
        w[q] = outside ? 0.0 : __dadd_rn(near == I ? 0.75 : 0.0, far == I ? 0.25 : 0.0);
    }
}

// fc = 0.125 * sum_z wz * (sum_y wy * (sum_x wx * r)), each sum t = w0*r0; t = fma(w1,r1,t); ...
__global__ void k_restrict_adj(Lv F, int cnx, int cny, int cnz, const double *__restrict__ r,
                               double *__restrict__ fc)
{
    const int I = blockIdx.x * blockDim.x + threadIdx.x;
    const int J = blockIdx.y * blockDim.y + threadIdx.y;
    const int K = blockIdx.z;
    if (I >= cnx || J >= cny) return;
    int ix[4], iy[4], iz[4];
    double wx[4], wy[4], wz[4];
    pt_stencil(I, F.nx, cnx, F.bcx, ix, wx);
    pt_stencil(J, F.ny, cny, F.bcy, iy, wy);
    pt_stencil(K, F.nz, cnz, F.bcz, iz, wz);
    double tz = 0.0;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        double ty = 0.0;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const double *row = r + (size_t)F.nx * ((size_t)iy[b] + (size_t)F.ny * (size_t)iz[c]);
            double tx = __dmul_rn(wx[0], row[ix[0]]);
            tx = __fma_rn(wx[1], row[ix[1]], tx);
            tx = __fma_rn(wx[2], row[ix[2]], tx);
            tx = __fma_rn(wx[3], row[ix[3]], tx);
            ty = b == 0 ? __dmul_rn(wy[0], tx) : __fma_rn(wy[b], tx, ty);
        }
        tz = c == 0 ? __dmul_rn(wz[0], ty) : __fma_rn(wz[c], ty, tz);
    }
    fc[(size_t)I + (size_t)cnx * ((size_t)J + (size_t)cny * (size_t)K)] = __dmul_rn(0.125, tz);
}

// C12: out = A d = ih2 * fma(-D, d, S)
template <bool CELL>
__global__ void k_apply(Lv L, const double *__restrict__ d, double *__restrict__ out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= L.nx || j >= L.ny) return;
    double S, D;
    stencil_global<CELL>(L, d, i, j, k, S, D);
    const size_t c = cidx(L, i, j, k);
    out[c] = __dmul_rn(L.ih2, __fma_rn(-D, d[c], S));
}

// first stage of x.y (fixed grid-stride order, fixed block tree)
__global__ void k_dot(const double *__restrict__ x, const double *__restrict__ y, size_t n,
                      double *__restrict__ partial)
{
    __shared__ double red[32];
    double s = 0.0;
    for (size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x; c < n; c += (size_t)gridDim.x * blockDim.x)
        s = __fma_rn(x[c], y[c], s);
    s = block_sum(s, red);
    if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

// C13: p = fma(alpha, d, p); r = fma(-alpha, q, r); first stage of sum r^2 in the same pass
__global__ void k_pcg_update(double alpha, const double *__restrict__ d, const double *__restrict__ q,
                             double *__restrict__ p, double *__restrict__ r, size_t n,
                             double *__restrict__ partial)
{
    __shared__ double red[32];
    double s = 0.0;
    for (size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x; c < n; c += (size_t)gridDim.x * blockDim.x) {
        p[c] = __fma_rn(alpha, d[c], p[c]);
        const double rv = __fma_rn(-alpha, q[c], r[c]);
        r[c] = rv;
        s = __fma_rn(rv, rv, s);
    }
    s = block_sum(s, red);
    if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

// C13: d = fma(beta, d, z)
__global__ void k_pcg_direction(double beta, const double *__restrict__ z, double *__restrict__ d, size_t n)
{
    for (size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x; c < n; c += (size_t)gridDim.x * blockDim.x)
        d[c] = __fma_rn(beta, d[c], z[c]);
}

} // namespace mg
