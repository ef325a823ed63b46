// mg_coarse_kernel.cuh -- A4: the trailing levels of the hierarchy (<= 16^3 and below)
// inside ONE persistent CTA (BASELINE.json north_star "coarse levels <=16^3 in a single
// persistent CTA").
//
// Every array of every level handled here (p, f, bx, by, bz and the reciprocal diagonal
// invD = rcp(D), D from C4) lives in shared memory for the whole kernel: 6 arrays x 4096
// doubles at 16^3 + 8^3 + 4^3 = 224 256 B of the 232 448 B a CTA may own.  The kernel
// runs the complete sub-V-cycle -- nu1 sweeps, residual + 8-child restriction, ...,
// coarse_sweeps sweeps on the coarsest level, prolongation + correction, nu2 sweeps --
// with __syncthreads() between half-sweeps instead of kernel launches, reads the rhs of
// its top level from global memory once and writes the correction back once.
//
// Arithmetic: the same expression trees as the level-generic kernels (C3-C8 of
// DESIGN.md §3), so the result is bit-identical to running those levels launch by
// launch (MG_OPT_COARSE_CTA = 0), which the GPU tests check.  invD = __drcp_rn(D) is the
// correctly rounded reciprocal, the same bits as the 1.0/D of C5; it depends on the
// coefficients only, so it is formed once per launch and reused by every sweep.
#pragma once
#include "mg_common.cuh"
#include "mg_ref_kernels.cuh"     // far_index6: prolongation ghosts beyond walls (R24)

namespace mg {

constexpr int kCoarseMaxLevels = 4;
constexpr int kCoarseThreads = 1024;
constexpr size_t kCoarseSmemMax = 232448;      // 227 KB: opt-in dynamic shared memory per CTA

struct CoarseArgs {
    int nlev;
    int n[kCoarseMaxLevels][3];
    double h2[kCoarseMaxLevels], ih2[kCoarseMaxLevels];
    const double *bx[kCoarseMaxLevels], *by[kCoarseMaxLevels], *bz[kCoarseMaxLevels];
    int bc[3];           // axis has walls (not periodic)
    // R24 (mg_create6 with a Dirichlet side): wall logic as in the level-generic kernels.  The
    // plus-wall planes stay in global memory (n^2 values per axis, read through L1).
    int gen;
    int bcm[3], bcp[3];
    const double *wx[kCoarseMaxLevels], *wy[kCoarseMaxLevels], *wz[kCoarseMaxLevels];
    int nu1, nu2, coarse_sweeps;
    int cycle_type;      // 0 = V, 1 = F, 2 = W (R23)
    int warm;            // 0: initial guess 0; 1: a later visit, the guess is read from p
    const double *f;     // rhs of the top level handled here (global, read once)
    double *p;           // correction of that level (global, written once)
};

inline size_t coarse_cta_bytes(int (*n)[3], int nlev)
{
    size_t cells = 0;
    for (int q = 0; q < nlev; ++q) cells += (size_t)n[q][0] * n[q][1] * n[q][2];
    return cells * 6 * sizeof(double);
}

inline bool coarse_cta_fits(int (*n)[3], int nlev)
{
    return nlev >= 1 && nlev <= kCoarseMaxLevels && coarse_cta_bytes(n, nlev) <= kCoarseSmemMax;
}

// one level as the CTA sees it: everything in shared memory
struct CLv {
    int nx, ny, nz;
    double h2, ih2;
    double *p, *f, *bx, *by, *bz, *id;
    int gen, wallx, wally, wallz;          // R24: walls with their own coefficient
    const double *wx, *wy, *wz;
};

__device__ __forceinline__ CLv coarse_level(const CoarseArgs &A, int q, double *sm)
{
    size_t off = 0;
    for (int r = 0; r < q; ++r) off += (size_t)A.n[r][0] * A.n[r][1] * A.n[r][2] * 6;
    CLv L;
    L.nx = A.n[q][0]; L.ny = A.n[q][1]; L.nz = A.n[q][2];
    L.h2 = A.h2[q]; L.ih2 = A.ih2[q];
    const size_t n = (size_t)L.nx * L.ny * L.nz;
    L.p = sm + off; L.f = L.p + n; L.bx = L.f + n; L.by = L.bx + n; L.bz = L.by + n; L.id = L.bz + n;
    L.gen = A.gen; L.wallx = A.gen && A.bc[0]; L.wally = A.gen && A.bc[1]; L.wallz = A.gen && A.bc[2];
    L.wx = A.wx[q]; L.wy = A.wy[q]; L.wz = A.wz[q];
    return L;
}

// S (C4) of cell (i,j,k) from the shared-memory arrays; stored minus faces, the plus
// face is the wrapped neighbour's minus face (0 on a Neumann wall)
__device__ __forceinline__ double coarse_S(const CLv &L, const double *p, int i, int j, int k, int c)
{
    const int sx = 1, sy = L.nx, sz = L.nx * L.ny;
    const int cxm = i == 0 ? c + (L.nx - 1) * sx : c - sx, cxp = i == L.nx - 1 ? c - (L.nx - 1) * sx : c + sx;
    const int cym = j == 0 ? c + (L.ny - 1) * sy : c - sy, cyp = j == L.ny - 1 ? c - (L.ny - 1) * sy : c + sy;
    const int czm = k == 0 ? c + (L.nz - 1) * sz : c - sz, czp = k == L.nz - 1 ? c - (L.nz - 1) * sz : c + sz;
    if (L.gen) {        // R24: a plus wall has its own coefficient, the value beyond any wall is 0.0
        const bool xm = L.wallx && i == 0, xp = L.wallx && i == L.nx - 1;
        const bool ym = L.wally && j == 0, yp = L.wally && j == L.ny - 1;
        const bool zm = L.wallz && k == 0, zp = L.wallz && k == L.nz - 1;
        double b[6] = { L.bx[c], xp ? L.wx[j + L.ny * k] : L.bx[cxp], L.by[c], yp ? L.wy[i + L.nx * k] : L.by[cyp],
                        L.bz[c], zp ? L.wz[i + L.nx * j] : L.bz[czp] };
        return stencil_S(b, xm ? 0.0 : p[cxm], xp ? 0.0 : p[cxp], ym ? 0.0 : p[cym], yp ? 0.0 : p[cyp],
                         zm ? 0.0 : p[czm], zp ? 0.0 : p[czp]);
    }
    double b[6] = { L.bx[c], L.bx[cxp], L.by[c], L.by[cyp], L.bz[c], L.bz[czp] };
    return stencil_S(b, p[cxm], p[cxp], p[cym], p[cyp], p[czm], p[czp]);
}

__device__ __forceinline__ double coarse_D(const CLv &L, int i, int j, int k, int c)
{
    const int sy = L.nx, sz = L.nx * L.ny;
    const int cxp = i == L.nx - 1 ? c - (L.nx - 1) : c + 1;
    const int cyp = j == L.ny - 1 ? c - (L.ny - 1) * sy : c + sy;
    const int czp = k == L.nz - 1 ? c - (L.nz - 1) * sz : c + sz;
    if (L.gen) {
        double b[6] = { L.bx[c], (L.wallx && i == L.nx - 1) ? L.wx[j + L.ny * k] : L.bx[cxp],
                        L.by[c], (L.wally && j == L.ny - 1) ? L.wy[i + L.nx * k] : L.by[cyp],
                        L.bz[c], (L.wallz && k == L.nz - 1) ? L.wz[i + L.nx * j] : L.bz[czp] };
        return stencil_D(b);
    }
    double b[6] = { L.bx[c], L.bx[cxp], L.by[c], L.by[cyp], L.bz[c], L.bz[czp] };
    return stencil_D(b);
}

// one colour of a red-black sweep (R9, C4, C5); caller synchronises afterwards
__device__ __forceinline__ void coarse_half(const CLv &L, int colour, int tid, int nthr)
{
    const int hx = L.nx >> 1;
    const int nh = hx * L.ny * L.nz;
    for (int q = tid; q < nh; q += nthr) {
        const int ih = q % hx, r = q / hx;
        const int j = r % L.ny, k = r / L.ny;
        const int i = 2 * ih + ((j + k + colour) & 1);
        const int c = i + L.nx * (j + L.ny * k);
        const double S = coarse_S(L, L.p, i, j, k, c);
        L.p[c] = __dmul_rn(__fma_rn(-L.h2, L.f[c], S), L.id[c]);
    }
}

__device__ __forceinline__ void coarse_sweeps(const CLv &L, int sweeps, int tid, int nthr)
{
    for (int s = 0; s < sweeps; ++s) {
        coarse_half(L, 0, tid, nthr);
        __syncthreads();
        coarse_half(L, 1, tid, nthr);
        __syncthreads();
    }
}

// residual (C6) of one cell; D is recomputed (the residual needs D itself, not 1/D)
__device__ __forceinline__ double coarse_resid(const CLv &L, int i, int j, int k)
{
    const int c = i + L.nx * (j + L.ny * k);
    const double S = coarse_S(L, L.p, i, j, k, c);
    const double D = coarse_D(L, i, j, k, c);
    return resid_value(L.ih2, L.f[c], S, D, L.p[c]);
}

// A2+A3: f_coarse = 8-child mean of the residual (C7); e_coarse = 0
__device__ __forceinline__ void coarse_residual_restrict(const CLv &L, const CLv &C, int tid, int nthr)
{
    const int nc = C.nx * C.ny * C.nz;
    for (int q = tid; q < nc; q += nthr) {
        const int I = q % C.nx, r = q / C.nx;
        const int J = r % C.ny, K = r / C.ny;
        double v[8];
#pragma unroll
        for (int t = 0; t < 8; ++t)
            v[t] = coarse_resid(L, 2 * I + (t & 1), 2 * J + ((t >> 1) & 1), 2 * K + (t >> 2));
        C.f[q] = __dmul_rn(0.125, __dadd_rn(__dadd_rn(__dadd_rn(v[0], v[1]), __dadd_rn(v[2], v[3])),
                                           __dadd_rn(__dadd_rn(v[4], v[5]), __dadd_rn(v[6], v[7]))));
        C.p[q] = 0.0;
    }
}

__device__ __forceinline__ int coarse_far(int I, int side, int n, int neumann)
{
    int Ip = I + 2 * side - 1;
    if (Ip < 0) Ip = neumann ? 0 : n - 1;
    if (Ip >= n) Ip = neumann ? n - 1 : 0;
    return Ip;
}

// A5: p += trilinear prolongation of the coarse correction (C8)
__device__ __forceinline__ void coarse_prolong_add(const CLv &L, const CLv &C, const CoarseArgs &A, int tid,
                                                   int nthr)
{
    const int *bc = A.bc;
    const int n = L.nx * L.ny * L.nz;
    const double *e = C.p;
    for (int c = tid; c < n; c += nthr) {
        const int i = c % L.nx, r = c / L.nx;
        const int j = r % L.ny, k = r / L.ny;
        const int I = i >> 1, J = j >> 1, K = k >> 1;
        if (A.gen) {        // R24: the value beyond a Dirichlet wall is -e_boundary (signs multiply over the axes)
            double sx, sy, sz;
            const int Ip = far_index6(I, i & 1, C.nx, A.bcm[0], A.bcp[0], sx);
            const int Jp = far_index6(J, j & 1, C.ny, A.bcm[1], A.bcp[1], sy);
            const int Kp = far_index6(K, k & 1, C.nz, A.bcm[2], A.bcp[2], sz);
            const double sxy = __dmul_rn(sx, sy), sxz = __dmul_rn(sx, sz), syz = __dmul_rn(sy, sz);
#define CE_(ii, jj, kk) e[(ii) + C.nx * ((jj) + C.ny * (kk))]
            const double v =
                lerp(lerp(lerp(CE_(I, J, K), __dmul_rn(sx, CE_(Ip, J, K))),
                          lerp(__dmul_rn(sy, CE_(I, Jp, K)), __dmul_rn(sxy, CE_(Ip, Jp, K)))),
                     lerp(lerp(__dmul_rn(sz, CE_(I, J, Kp)), __dmul_rn(sxz, CE_(Ip, J, Kp))),
                          lerp(__dmul_rn(syz, CE_(I, Jp, Kp)), __dmul_rn(__dmul_rn(sxy, sz), CE_(Ip, Jp, Kp)))));
#undef CE_
            L.p[c] = __dadd_rn(L.p[c], v);
            continue;
        }
        const int Ip = coarse_far(I, i & 1, C.nx, bc[0]);
        const int Jp = coarse_far(J, j & 1, C.ny, bc[1]);
        const int Kp = coarse_far(K, k & 1, C.nz, bc[2]);
#define CE_(ii, jj, kk) e[(ii) + C.nx * ((jj) + C.ny * (kk))]
        const double v =
            lerp(lerp(lerp(CE_(I, J, K),  CE_(Ip, J, K)),  lerp(CE_(I, Jp, K),  CE_(Ip, Jp, K))),
                 lerp(lerp(CE_(I, J, Kp), CE_(Ip, J, Kp)), lerp(CE_(I, Jp, Kp), CE_(Ip, Jp, Kp))));
#undef CE_
        L.p[c] = __dadd_rn(L.p[c], v);
    }
}

// F- and W-cycles (R23) below the top level of the CTA: the recursion of the cycle index walked
// with an explicit stack (at most kCoarseMaxLevels frames), every thread of the CTA in step.
// A frame is (level, cycle type, stage): 0 = entered, 1 = first visit of the coarse problem done,
// 2 = both done.
__device__ __forceinline__ void coarse_cycle(const CoarseArgs &A, double *sm, int type, int tid, int nthr)
{
    int fq[kCoarseMaxLevels + 1], fty[kCoarseMaxLevels + 1], fst[kCoarseMaxLevels + 1];
    int sp = 0;
    fq[0] = 0; fty[0] = type; fst[0] = 0;
    while (sp >= 0) {
        const int q = fq[sp], ty = fty[sp];
        const CLv L = coarse_level(A, q, sm);
        if (q == A.nlev - 1) {                               // R13
            coarse_sweeps(L, A.coarse_sweeps, tid, nthr);
            --sp;
            continue;
        }
        const CLv C = coarse_level(A, q + 1, sm);
        if (fst[sp] == 0) {
            coarse_sweeps(L, A.nu1, tid, nthr);
            coarse_residual_restrict(L, C, tid, nthr);
            __syncthreads();
            fst[sp] = 1;
            ++sp; fq[sp] = q + 1; fty[sp] = ty; fst[sp] = 0;
            continue;
        }
        if (fst[sp] == 1) {
            fst[sp] = 2;
            if (q + 1 < A.nlev - 1 && ty != 0) {             // second visit: W again, or V after F
                ++sp; fq[sp] = q + 1; fty[sp] = ty == 2 ? 2 : 0; fst[sp] = 0;
                continue;
            }
        }
        coarse_prolong_add(L, C, A, tid, nthr);
        __syncthreads();
        coarse_sweeps(L, A.nu2, tid, nthr);
        --sp;
    }
}

__global__ void __launch_bounds__(kCoarseThreads, 1) k_coarse_cta(CoarseArgs A)
{
    extern __shared__ __align__(16) double coarse_sm[];
    const int tid = threadIdx.x, nthr = blockDim.x;

    // ---- stage coefficients of every level, rhs of the top level, zero initial guess
    for (int q = 0; q < A.nlev; ++q) {
        const CLv L = coarse_level(A, q, coarse_sm);
        const int n = L.nx * L.ny * L.nz;
        const double *gx = A.bx[q], *gy = A.by[q], *gz = A.bz[q];
        for (int c = tid; c < n; c += nthr) {
            L.bx[c] = gx[c]; L.by[c] = gy[c]; L.bz[c] = gz[c];
            if (q == 0) { L.f[c] = A.f[c]; L.p[c] = A.warm ? A.p[c] : 0.0; }
        }
    }
    __syncthreads();
    for (int q = 0; q < A.nlev; ++q) {
        const CLv L = coarse_level(A, q, coarse_sm);
        const int n = L.nx * L.ny * L.nz;
        for (int c = tid; c < n; c += nthr) {
            const int i = c % L.nx, r = c / L.nx;
            L.id[c] = __drcp_rn(coarse_D(L, i, r % L.ny, r / L.ny, c));
        }
    }
    __syncthreads();

    if (A.cycle_type != 0) {
        coarse_cycle(A, coarse_sm, A.cycle_type, tid, nthr);
    } else {
    // ---- down
    for (int q = 0; q + 1 < A.nlev; ++q) {
        const CLv L = coarse_level(A, q, coarse_sm);
        const CLv C = coarse_level(A, q + 1, coarse_sm);
        coarse_sweeps(L, A.nu1, tid, nthr);
        coarse_residual_restrict(L, C, tid, nthr);
        __syncthreads();
    }
    // ---- coarsest level (R13)
    {
        const CLv L = coarse_level(A, A.nlev - 1, coarse_sm);
        coarse_sweeps(L, A.coarse_sweeps, tid, nthr);
    }
    // ---- up
    for (int q = A.nlev - 2; q >= 0; --q) {
        const CLv L = coarse_level(A, q, coarse_sm);
        const CLv C = coarse_level(A, q + 1, coarse_sm);
        coarse_prolong_add(L, C, A, tid, nthr);
        __syncthreads();
        coarse_sweeps(L, A.nu2, tid, nthr);
    }
    }
    // ---- correction of the top level back to global memory
    {
        const CLv L = coarse_level(A, 0, coarse_sm);
        const int n = L.nx * L.ny * L.nz;
        for (int c = tid; c < n; c += nthr) A.p[c] = L.p[c];
    }
}

// opt-in to the dynamic shared memory the kernel needs; per device, called from mg_create
inline int coarse_cta_prepare_device()
{
    return cudaFuncSetAttribute(k_coarse_cta, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)kCoarseSmemMax) == cudaSuccess ? 0 : -1;
}

inline int launch_coarse_cta(const CoarseArgs &a, cudaStream_t st)
{
    int n[kCoarseMaxLevels][3];
    for (int q = 0; q < a.nlev; ++q) { n[q][0] = a.n[q][0]; n[q][1] = a.n[q][1]; n[q][2] = a.n[q][2]; }
    const size_t bytes = coarse_cta_bytes(n, a.nlev);
    if (bytes > kCoarseSmemMax) return -1;
    k_coarse_cta<<<1, kCoarseThreads, bytes, st>>>(a);
    return 0;
}

} // namespace mg
