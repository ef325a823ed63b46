// mg_ref_kernels.cuh -- level-generic reference kernels: one launch per half-sweep /
// transfer / reduction, any even nx,ny,nz, straight global-memory stencils.
// They are the correctness baseline of the CUDA path (MG_OPT_KERNELS = 0), the
// fallback for shapes the streaming kernels do not tile, and the setup kernels
// (coefficients, reductions) of every configuration.
#pragma once
#include "mg_common.cuh"

namespace mg {

// ---- A0: coefficients -----------------------------------------------------
// a = 0.5/rho (C2); flags[0] |= 1 if some rho is not a finite positive number; flags[1] |= 1 if
// some a lies outside [2^-900, 2^900].
__global__ void k_cell_coef(const double *__restrict__ rho, double *__restrict__ a, size_t n,
                            int *__restrict__ flags)
{
    bool bad = false, wide = false;
    for (size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x; c < n;
         c += (size_t)gridDim.x * blockDim.x) {
        const double r = rho[c];
        bad |= !(r > 0.0) || isinf(r);
        const double av = __ddiv_rn(0.5, r);
        wide |= !(av >= 0x1p-900 && av <= 0x1p900);      // outside the range of the branch-free reciprocal
        a[c] = av;
    }
    if (__syncthreads_or(bad) && threadIdx.x == 0) atomicOr(flags, 1);
    if (__syncthreads_or(wide) && threadIdx.x == 0) atomicOr(flags + 1, 1);
}

// minus faces of a CELL level written out explicitly (mg_level_faces on level 0)
__global__ void k_faces_from_cell(Lv L, double *__restrict__ bx, double *__restrict__ by,
                                  double *__restrict__ bz)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= L.nx || j >= L.ny) return;
    const size_t c = cidx(L, i, j, k);
    const double ac = L.a[c];
    bx[c] = (L.bcx && i == 0) ? wall_face(L.gen ? L.bcm[0] : 1, ac) : __dadd_rn(ac, L.a[cidx(L, i == 0 ? L.nx - 1 : i - 1, j, k)]);
    by[c] = (L.bcy && j == 0) ? wall_face(L.gen ? L.bcm[1] : 1, ac) : __dadd_rn(ac, L.a[cidx(L, i, j == 0 ? L.ny - 1 : j - 1, k)]);
    bz[c] = (L.bcz && k == 0) ? wall_face(L.gen ? L.bcm[2] : 1, ac) : __dadd_rn(ac, L.a[cidx(L, i, j, k == 0 ? L.nz - 1 : k - 1)]);
}

// C3: coarse minus faces = mean of the 4 finer minus faces of the even children.
// FINE_CELL: the finer level is level 0 (faces formed from a on the fly).
template <bool FINE_CELL>
__device__ __forceinline__ double fine_face(const Lv &F, int axis, int i, int j, int k)
{
    const size_t c = cidx(F, i, j, k);
    if (!FINE_CELL) return axis == 0 ? F.bx[c] : (axis == 1 ? F.by[c] : F.bz[c]);
    if (axis == 0) {
        if (F.bcx && i == 0) return wall_face(F.gen ? F.bcm[0] : 1, F.a[c]);
        return __dadd_rn(F.a[c], F.a[cidx(F, i == 0 ? F.nx - 1 : i - 1, j, k)]);
    }
    if (axis == 1) {
        if (F.bcy && j == 0) return wall_face(F.gen ? F.bcm[1] : 1, F.a[c]);
        return __dadd_rn(F.a[c], F.a[cidx(F, i, j == 0 ? F.ny - 1 : j - 1, k)]);
    }
    if (F.bcz && k == 0) return wall_face(F.gen ? F.bcm[2] : 1, F.a[c]);
    return __dadd_rn(F.a[c], F.a[cidx(F, i, j, k == 0 ? F.nz - 1 : k - 1)]);
}

template <bool FINE_CELL>
__global__ void k_coarsen_faces(Lv F, int cnx, int cny, int cnz, double *__restrict__ cbx,
                                double *__restrict__ cby, double *__restrict__ cbz)
{
    const int I = blockIdx.x * blockDim.x + threadIdx.x;
    const int J = blockIdx.y * blockDim.y + threadIdx.y;
    const int K = blockIdx.z;
    if (I >= cnx || J >= cny) return;
    const int i = 2 * I, j = 2 * J, k = 2 * K;
    const size_t c = (size_t)I + (size_t)cnx * ((size_t)J + (size_t)cny * (size_t)K);
    cbx[c] = __dmul_rn(0.25, __dadd_rn(
        __dadd_rn(fine_face<FINE_CELL>(F, 0, i, j, k),     fine_face<FINE_CELL>(F, 0, i, j + 1, k)),
        __dadd_rn(fine_face<FINE_CELL>(F, 0, i, j, k + 1), fine_face<FINE_CELL>(F, 0, i, j + 1, k + 1))));
    cby[c] = __dmul_rn(0.25, __dadd_rn(
        __dadd_rn(fine_face<FINE_CELL>(F, 1, i, j, k),     fine_face<FINE_CELL>(F, 1, i + 1, j, k)),
        __dadd_rn(fine_face<FINE_CELL>(F, 1, i, j, k + 1), fine_face<FINE_CELL>(F, 1, i + 1, j, k + 1))));
    cbz[c] = __dmul_rn(0.25, __dadd_rn(
        __dadd_rn(fine_face<FINE_CELL>(F, 2, i, j, k),     fine_face<FINE_CELL>(F, 2, i + 1, j, k)),
        __dadd_rn(fine_face<FINE_CELL>(F, 2, i, j + 1, k), fine_face<FINE_CELL>(F, 2, i + 1, j + 1, k))));
}

// R24: plus-wall faces of the coarse level = mean of the four finer plus-wall faces lying on
// them, pairs in the order of C3 (over the faster in-plane axis first).  One thread per coarse
// wall cell of one axis (blockIdx.z = axis); (u, v) = the two in-plane indices, u faster.
template <bool FINE_CELL>
__device__ __forceinline__ double fine_wall(const Lv &F, int axis, int u, int v)
{
    if (!FINE_CELL)
        return axis == 0 ? F.wx[(size_t)u + (size_t)F.ny * (size_t)v]
                         : (axis == 1 ? F.wy[(size_t)u + (size_t)F.nx * (size_t)v] : F.wz[(size_t)u + (size_t)F.nx * (size_t)v]);
    const size_t c = axis == 0 ? cidx(F, F.nx - 1, u, v) : (axis == 1 ? cidx(F, u, F.ny - 1, v) : cidx(F, u, v, F.nz - 1));
    return wall_face(F.bcp[axis], F.a[c]);
}

template <bool FINE_CELL>
__global__ void k_coarsen_walls(Lv F, int cnx, int cny, int cnz, double *__restrict__ cwx,
                                double *__restrict__ cwy, double *__restrict__ cwz)
{
    const int axis = blockIdx.z;
    const int nu = axis == 0 ? cny : cnx, nv = axis == 2 ? cny : cnz;
    const int U = blockIdx.x * blockDim.x + threadIdx.x, V = blockIdx.y * blockDim.y + threadIdx.y;
    if (U >= nu || V >= nv) return;
    const double w = __dmul_rn(0.25, __dadd_rn(
        __dadd_rn(fine_wall<FINE_CELL>(F, axis, 2 * U, 2 * V),     fine_wall<FINE_CELL>(F, axis, 2 * U + 1, 2 * V)),
        __dadd_rn(fine_wall<FINE_CELL>(F, axis, 2 * U, 2 * V + 1), fine_wall<FINE_CELL>(F, axis, 2 * U + 1, 2 * V + 1))));
    double *dst = axis == 0 ? cwx : (axis == 1 ? cwy : cwz);
    dst[(size_t)U + (size_t)nu * (size_t)V] = w;
}

// ---- A1/A6: one colour of a red-black Gauss-Seidel sweep (C4, C5) ------------
template <bool CELL>
__global__ void k_smooth_half(Lv L, int colour, const double *__restrict__ f, double *p)
{
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    const int i = 2 * (blockIdx.x * blockDim.x + threadIdx.x) + ((j + k + colour) & 1);
    if (i >= L.nx || j >= L.ny) return;
    double S, D;
    stencil_global<CELL>(L, p, i, j, k, S, D);
    const size_t c = cidx(L, i, j, k);
    p[c] = gs_value(L.h2, f[c], S, D);
}

// ---- A2: residual field (C6) -------------------------------------------------
template <bool CELL>
__global__ void k_residual(Lv L, const double *__restrict__ f, const double *__restrict__ p,
                           double *__restrict__ r)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= L.nx || j >= L.ny) return;
    double S, D;
    stencil_global<CELL>(L, p, i, j, k, S, D);
    const size_t c = cidx(L, i, j, k);
    r[c] = resid_value(L.ih2, f[c], S, D, p[c]);
}

// ---- A7: sum of squared residuals, first stage (optionally also writes r) ---------
// Fixed grid; thread t visits cells t, t+T, ... so the summation tree is fixed.
template <bool CELL>
__global__ void k_residual_norm2(Lv L, const double *__restrict__ f, const double *__restrict__ p,
                                 double *__restrict__ r_or_null, double *__restrict__ partial)
{
    __shared__ double red[32];
    const size_t n = (size_t)L.nx * L.ny * L.nz;
    const size_t plane = (size_t)L.nx * L.ny;
    double acc = 0.0;
    for (size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x; c < n;
         c += (size_t)gridDim.x * blockDim.x) {
        const int k = (int)(c / plane);
        const int rem = (int)(c - (size_t)k * plane);
        const int j = rem / L.nx, i = rem - j * L.nx;
        double S, D;
        stencil_global<CELL>(L, p, i, j, k, S, D);
        const double r = resid_value(L.ih2, f[c], S, D, p[c]);
        if (r_or_null) r_or_null[c] = r;
        acc = __fma_rn(r, r, acc);
    }
    acc = block_sum(acc, red);
    if (threadIdx.x == 0) partial[blockIdx.x] = acc;
}

// ---- A2+A3: residual fused with 8-child-mean restriction (C6, C7) ----------------
template <bool CELL>
__global__ void k_residual_restrict(Lv L, const double *__restrict__ f,
                                    const double *__restrict__ p, int cnx, int cny,
                                    double *__restrict__ fc)
{
    const int I = blockIdx.x * blockDim.x + threadIdx.x;
    const int J = blockIdx.y * blockDim.y + threadIdx.y;
    const int K = blockIdx.z;
    if (I >= cnx || J >= cny) return;
    double r[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const int i = 2 * I + (q & 1), j = 2 * J + ((q >> 1) & 1), k = 2 * K + (q >> 2);
        double S, D;
        stencil_global<CELL>(L, p, i, j, k, S, D);
        const size_t c = cidx(L, i, j, k);
        r[q] = resid_value(L.ih2, f[c], S, D, p[c]);
    }
    // r[q], q = x + 2y + 4z: ((r000+r100)+(r010+r110)) + ((r001+r101)+(r011+r111))
    fc[(size_t)I + (size_t)cnx * ((size_t)J + (size_t)cny * (size_t)K)] = __dmul_rn(
        0.125, __dadd_rn(__dadd_rn(__dadd_rn(r[0], r[1]), __dadd_rn(r[2], r[3])),
                         __dadd_rn(__dadd_rn(r[4], r[5]), __dadd_rn(r[6], r[7]))));
}

// ---- A5: p += trilinear prolongation of e (C8) -----------------------------------
__device__ __forceinline__ int far_index(int I, int side, int n, int neumann)
{
    int Ip = I + 2 * side - 1;
    if (Ip < 0) Ip = neumann ? 0 : n - 1;
    if (Ip >= n) Ip = neumann ? n - 1 : 0;
    return Ip;
}

// R24: the far coarse index beyond a wall is the boundary cell itself; beyond a Dirichlet wall its
// value enters with sign -1 (ghost = -e_boundary)
__device__ __forceinline__ int far_index6(int I, int side, int n, int bc_minus, int bc_plus, double &sign)
{
    int Ip = I + 2 * side - 1;
    sign = 1.0;
    if (Ip < 0) {
        if (bc_minus == 0) Ip = n - 1;
        else { Ip = 0; if (bc_minus == 2) sign = -1.0; }
    }
    if (Ip >= n) {
        if (bc_plus == 0) Ip = 0;
        else { Ip = n - 1; if (bc_plus == 2) sign = -1.0; }
    }
    return Ip;
}

__device__ __forceinline__ double prolong_value(const Lv &L, const double *__restrict__ e, int cnx,
                                                int cny, int cnz, int i, int j, int k)
{
    const int I = i >> 1, J = j >> 1, K = k >> 1;
    if (L.gen) {
        double sx, sy, sz;
        const int Ip = far_index6(I, i & 1, cnx, L.bcm[0], L.bcp[0], sx);
        const int Jp = far_index6(J, j & 1, cny, L.bcm[1], L.bcp[1], sy);
        const int Kp = far_index6(K, k & 1, cnz, L.bcm[2], L.bcp[2], sz);
        const double sxy = __dmul_rn(sx, sy), sxz = __dmul_rn(sx, sz), syz = __dmul_rn(sy, sz);
#define E_(ii, jj, kk) e[(size_t)(ii) + (size_t)cnx * ((size_t)(jj) + (size_t)cny * (size_t)(kk))]
        return lerp(lerp(lerp(E_(I, J, K), __dmul_rn(sx, E_(Ip, J, K))),
                         lerp(__dmul_rn(sy, E_(I, Jp, K)), __dmul_rn(sxy, E_(Ip, Jp, K)))),
                    lerp(lerp(__dmul_rn(sz, E_(I, J, Kp)), __dmul_rn(sxz, E_(Ip, J, Kp))),
                         lerp(__dmul_rn(syz, E_(I, Jp, Kp)), __dmul_rn(__dmul_rn(sxy, sz), E_(Ip, Jp, Kp)))));
#undef E_
    }
    const int Ip = far_index(I, i & 1, cnx, L.bcx);
    const int Jp = far_index(J, j & 1, cny, L.bcy);
    const int Kp = far_index(K, k & 1, cnz, L.bcz);
#define E_(ii, jj, kk) e[(size_t)(ii) + (size_t)cnx * ((size_t)(jj) + (size_t)cny * (size_t)(kk))]
    const double v =
        lerp(lerp(lerp(E_(I, J, K),   E_(Ip, J, K)),  lerp(E_(I, Jp, K),  E_(Ip, Jp, K))),
             lerp(lerp(E_(I, J, Kp),  E_(Ip, J, Kp)), lerp(E_(I, Jp, Kp), E_(Ip, Jp, Kp))));
#undef E_
    return v;
}

__global__ void k_prolong_add(Lv L, const double *__restrict__ e, int cnx, int cny, int cnz,
                              double *__restrict__ p)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= L.nx || j >= L.ny) return;
    const size_t c = cidx(L, i, j, k);
    p[c] = __dadd_rn(p[c], prolong_value(L, e, cnx, cny, cnz, i, j, k));
}

// ---- reductions ------------------------------------------------------------------
// first stage of sum(x) and sum(x^2)
__global__ void k_sum_sumsq(const double *__restrict__ x, size_t n, double *__restrict__ partial_sum,
                            double *__restrict__ partial_sq)
{
    __shared__ double red[32];
    double s = 0.0, q = 0.0;
    for (size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x; c < n;
         c += (size_t)gridDim.x * blockDim.x) {
        const double v = x[c];
        s = __dadd_rn(s, v);
        q = __fma_rn(v, v, q);
    }
    s = block_sum(s, red);
    q = block_sum(q, red);
    if (threadIdx.x == 0) {
        partial_sum[blockIdx.x] = s;
        if (partial_sq) partial_sq[blockIdx.x] = q;
    }
}

// second stage: out[slot] = sum(partial[0..m)), one block
__global__ void k_final_sum(const double *__restrict__ partial, int m, double *__restrict__ out)
{
    __shared__ double red[32];
    double s = 0.0;
    for (int t = threadIdx.x; t < m; t += blockDim.x) s = __dadd_rn(s, partial[t]);
    s = block_sum(s, red);
    if (threadIdx.x == 0) *out = s;
}

// x -= (*sum)/n
__global__ void k_subtract_mean(double *__restrict__ x, size_t n, const double *__restrict__ sum)
{
    const double mean = __ddiv_rn(*sum, (double)n);
    for (size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x; c < n;
         c += (size_t)gridDim.x * blockDim.x)
        x[c] = __dsub_rn(x[c], mean);
}

__global__ void k_fill_zero(double *__restrict__ x, size_t n)
{
    for (size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x; c < n;
         c += (size_t)gridDim.x * blockDim.x)
        x[c] = 0.0;
}

} // namespace mg
