// mg_stream_kernels.cuh -- fused 2.5-D streaming kernels for the large levels.
//
// One launch = one full red-black Gauss-Seidel sweep (red half-sweep, then black) read
// from p_in and written to p_out (ping-pong: tiles of other CTAs must see the old
// iterate), i.e. 32 B/cell of compulsory HBM traffic on level 0 (p in, p out, f, a)
// instead of 64 B for two half-sweep launches.  Optional fused tails:
//   TAIL_RESTRICT : r = f - A p_out on the fly, 8-child mean written to the coarse rhs
//                   (A2+A3 fused into the last pre-smoothing sweep; r never materialised)
//   TAIL_NORM     : sum r^2 per CTA (A7 fused into the last post-smoothing sweep)
// Optional fused head:
//   HEAD_PROLONG  : p_in + P e is smoothed instead of p_in (A5 fused into the first
//                   post-smoothing sweep)
//
// Geometry.  A CTA owns an (x,y) tile and marches along z through a z-chunk.  Thread
// (lx,ly) owns the column of the x-PAIR (2 lx, 2 lx+1) of tile row ly: one cell of the
// pair is red, the other black, so every thread does exactly one red update (plane t)
// and one black update (plane t-2) per step, and all global loads/stores are coalesced
// 16-byte double2 accesses.  The thread keeps its own column's z-window (planes t+1 ..
// t-3 of p and a) in registers; only in-plane neighbours go through shared memory
// (4 plane slots, even-x and odd-x cells de-interleaved so that every LDS is
// conflict-free).  The tile is loaded with a halo of 2 cells: ring 2 only supplies
// data, ring 1 additionally recomputes the red update (the value the neighbouring CTA
// also computes -- same expression tree, same inputs, same bits), the interior does
// both colours.  Exact global red->black semantics are kept (SURVEY §7 "temporal
// blocking must keep exact global semantics").
//
// Boundaries.  Indices outside the domain are wrapped (periodic) or mirrored (Neumann)
// at load time.  A Neumann ghost cell carries a = -a(mirror), so the canonical face
// beta = a_c + a_nb evaluates to exactly +0.0 on a wall face (C2) with no wall logic in
// the update; ghost cells themselves are never updated.
#pragma once
#include "mg_common.cuh"

namespace mg {

constexpr int SK_LX = 32;            // thread columns (x pairs): 64 cells loaded
constexpr int SK_LY = 16;            // thread rows loaded
constexpr int SK_OX = 60;            // output cells per tile in x (pairs 1..30)
constexpr int SK_OY = 12;            // output rows per tile (rows 2..13)
constexpr int SK_THREADS = SK_LX * SK_LY;

struct SkSlot {                      // one z-plane of the tile in shared memory
    double pe[SK_LY][SK_LX];         // p of even-x cells
    double po[SK_LY][SK_LX];         // p of odd-x cells
    double ae[SK_LY][SK_LX];         // a (level 0) of even-x cells
    double ao[SK_LY][SK_LX];
};

enum { SK_TAIL_NONE = 0, SK_TAIL_RESTRICT = 1, SK_TAIL_NORM = 2 };

struct SkArgs {
    Lv L;
    const double *f;
    const double *pin;
    double *pout;
    int zchunk;
    // HEAD_PROLONG: coarse correction e (level+1) with its dims
    const double *e;
    int cnx, cny, cnz;
    // TAIL_RESTRICT: coarse rhs;  TAIL_NORM: per-CTA partial sums
    double *fc;
    double *partial;
};

// source index of global coordinate g along an axis of n cells: in range as is, else
// wrapped (periodic) or mirrored (Neumann, ghost = true)
__device__ __forceinline__ int sk_map(int g, int n, int neumann, bool &ghost)
{
    ghost = false;
    if (g >= 0 && g < n) return g;
    if (!neumann) { g %= n; return g < 0 ? g + n : g; }
    ghost = true;
    int m = g < 0 ? -1 - g : 2 * n - 1 - g;
    if (m < 0 || m >= n) { m %= n; if (m < 0) m += n; }      // far ghost: value irrelevant
    return m;
}

template <bool CELL, bool HEAD_PROLONG, int TAIL>
__global__ void __launch_bounds__(SK_THREADS, 1) k_stream_sweep(SkArgs A)
{
    extern __shared__ __align__(16) unsigned char sk_smem_raw[];
    SkSlot *slots = reinterpret_cast<SkSlot *>(sk_smem_raw);
    const Lv &L = A.L;
    const int lx = threadIdx.x, ly = threadIdx.y;
    const int ox = blockIdx.x * SK_OX, oy = blockIdx.y * SK_OY;
    const int kz0 = blockIdx.z * A.zchunk;
    const int kz1 = min(L.nz, kz0 + A.zchunk);

    // ---- this thread's column: source indices of its pair and row
    const int gx = ox - 2 + 2 * lx;              // global x of the pair's even cell (may be outside)
    const int gy = oy - 2 + ly;
    bool ghost_x0, ghost_x1, ghost_y;
    const int sx0 = sk_map(gx, L.nx, L.bcx, ghost_x0);
    const int sx1 = sk_map(gx + 1, L.nx, L.bcx, ghost_x1);
    const int sy = sk_map(gy, L.ny, L.bcy, ghost_y);
    const bool swapx = sx1 < sx0;                 // mirrored pair: (sx1, sx0) is the aligned pair
    const int sxp = swapx ? sx1 : sx0;            // aligned pair start (even)
    const bool ghost_xy = ghost_x0 || ghost_y;    // ghost_x0 == ghost_x1 (pairs never straddle a wall)
    const size_t col = (size_t)sxp + (size_t)L.nx * (size_t)sy;
    const size_t plane_stride = (size_t)L.nx * L.ny;

    // region flags
    const bool is_out = lx >= 1 && lx <= 30 && ly >= 2 && ly <= 13 && gx < L.nx && gy < L.ny &&
                        gx >= 0 && gy >= 0;                   // owns output cells (both of the pair)
    const bool row_r1 = ly >= 1 && ly <= 14 && !ghost_y;      // rows where red is (re)computed

    // register z-window: index 0 = plane t+1, 1 = t, 2 = t-1, 3 = t-2, 4 = t-3
    double2 P[5], Aa[5], F[4];
#pragma unroll
    for (int q = 0; q < 5; ++q) { P[q] = make_double2(0.0, 0.0); Aa[q] = make_double2(0.0, 0.0); }
#pragma unroll
    for (int q = 0; q < 4; ++q) F[q] = make_double2(0.0, 0.0);

    auto load_plane = [&](int k, double2 &p2, double2 &a2, double2 &f2) {
        bool ghost_z;
        const int sk = sk_map(k, L.nz, L.bcz, ghost_z);
        const size_t idx = col + plane_stride * (size_t)sk;
        p2 = *reinterpret_cast<const double2 *>(A.pin + idx);
        f2 = *reinterpret_cast<const double2 *>(A.f + idx);
        if (CELL) a2 = *reinterpret_cast<const double2 *>(L.a + idx);
        if (swapx) {
            double t_ = p2.x; p2.x = p2.y; p2.y = t_;
            t_ = f2.x; f2.x = f2.y; f2.y = t_;
            if (CELL) { t_ = a2.x; a2.x = a2.y; a2.y = t_; }
        }
        if (CELL && (ghost_xy || ghost_z)) { a2.x = -a2.x; a2.y = -a2.y; }
        if (HEAD_PROLONG) {
            // p_in + P e (C8) for both cells of the pair; ghosts keep the mirrored value,
            // which is what the in-domain neighbour needs (it is multiplied by beta = 0)
            p2.x = __dadd_rn(p2.x, prolong_value(L, A.e, A.cnx, A.cny, A.cnz, sx0, sy, sk));
            p2.y = __dadd_rn(p2.y, prolong_value(L, A.e, A.cnx, A.cny, A.cnz, sx1, sy, sk));
        }
    };
    auto store_slot = [&](int k, const double2 &p2, const double2 &a2) {
        SkSlot &S = slots[k & 3];
        S.pe[ly][lx] = p2.x; S.po[ly][lx] = p2.y;
        if (CELL) { S.ae[ly][lx] = a2.x; S.ao[ly][lx] = a2.y; }
    };

    // one Gauss-Seidel update (MODE 0) or residual (MODE 1) of cell `c` (0 = even-x cell,
    // 1 = odd-x cell) of this thread's pair at the plane held in window index W (slot of
    // plane k), using the window entries W-1 (plane k+1) and W+1 (plane k-1).
    auto cell_SD = [&](int c, int k, int ks, const double2 &Pm, const double2 &Pc, const double2 &Pp,
                       const double2 &Am, const double2 &Ac, const double2 &Ap, double &S_, double &D_) {
        // Pm/Am: plane k-1, Pc/Ac: plane k, Pp/Ap: plane k+1
        const SkSlot &S = slots[k & 3];
        const double *own_p = c ? &S.po[0][0] : &S.pe[0][0];      // same x: y neighbours
        const double *oth_p = c ? &S.pe[0][0] : &S.po[0][0];      // other parity: x neighbour
        const int o = ly * SK_LX + lx;
        const double p_partner = c ? Pc.x : Pc.y;
        const double p_xnb = oth_p[o + (c ? 1 : -1)];
        const double pxm = c ? p_partner : p_xnb;
        const double pxp = c ? p_xnb : p_partner;
        const double pym = own_p[o - SK_LX], pyp = own_p[o + SK_LX];
        const double pzm = c ? Pm.y : Pm.x, pzp = c ? Pp.y : Pp.x;
        double b[6];
        if (CELL) {
            const double *own_a = c ? &S.ao[0][0] : &S.ae[0][0];
            const double *oth_a = c ? &S.ae[0][0] : &S.ao[0][0];
            const double a_c = c ? Ac.y : Ac.x;
            const double a_partner = c ? Ac.x : Ac.y;
            const double a_xnb = oth_a[o + (c ? 1 : -1)];
            b[0] = __dadd_rn(a_c, c ? a_partner : a_xnb);
            b[1] = __dadd_rn(a_c, c ? a_xnb : a_partner);
            b[2] = __dadd_rn(a_c, own_a[o - SK_LX]);
            b[3] = __dadd_rn(a_c, own_a[o + SK_LX]);
            b[4] = __dadd_rn(a_c, c ? Am.y : Am.x);
            b[5] = __dadd_rn(a_c, c ? Ap.y : Ap.x);
        } else {
            // stored minus faces, read through L1/L2 at the (wrapped) source position
            const int x = c ? sx1 : sx0;
            const int xp = x == L.nx - 1 ? 0 : x + 1;
            const int yp = sy == L.ny - 1 ? 0 : sy + 1;
            const int kp = ks == L.nz - 1 ? 0 : ks + 1;
            const size_t cc = (size_t)x + (size_t)L.nx * ((size_t)sy + (size_t)L.ny * (size_t)ks);
            b[0] = __ldg(L.bx + cc);
            b[1] = __ldg(L.bx + ((size_t)xp + (size_t)L.nx * ((size_t)sy + (size_t)L.ny * (size_t)ks)));
            b[2] = __ldg(L.by + cc);
            b[3] = __ldg(L.by + ((size_t)x + (size_t)L.nx * ((size_t)yp + (size_t)L.ny * (size_t)ks)));
            b[4] = __ldg(L.bz + cc);
            b[5] = __ldg(L.bz + ((size_t)x + (size_t)L.nx * ((size_t)sy + (size_t)L.ny * (size_t)kp)));
        }
        S_ = stencil_S(b, pxm, pxp, pym, pyp, pzm, pzp);
        D_ = stencil_D(b);
    };

    // ---- prologue: planes kz0-2, kz0-1, kz0 into window indices 2,1,0 of step t = kz0-1
    {
        double2 a2 = make_double2(0.0, 0.0);
        load_plane(kz0 - 2, P[2], a2, F[2]); Aa[2] = a2; store_slot(kz0 - 2, P[2], Aa[2]);
        load_plane(kz0 - 1, P[1], a2, F[1]); Aa[1] = a2; store_slot(kz0 - 1, P[1], Aa[1]);
        load_plane(kz0,     P[0], a2, F[0]); Aa[0] = a2; store_slot(kz0,     P[0], Aa[0]);
    }
    __syncthreads();

    for (int t = kz0 - 1; t <= kz1 + 1; ++t) {
        // prefetch plane t+2 (consumed at the end of this step)
        double2 pn = make_double2(0.0, 0.0), an = make_double2(0.0, 0.0), fn = make_double2(0.0, 0.0);
        const bool need_next = t + 2 <= kz1 + 1;
        if (need_next) load_plane(t + 2, pn, an, fn);

        // -------- red half-sweep at plane t (window index 1)
        {
            const int cr = (oy + ly + t) & 1;          // which cell of the pair is red (x+y+z even)
            bool ghost_z;
            const int kt = sk_map(t, L.nz, L.bcz, ghost_z);
            const int xl = 2 * lx + cr;                // local x of the red cell
            const bool can = row_r1 && !ghost_x0 && !ghost_z && xl >= 1 && xl <= 62 && t <= kz1;
            if (can) {
                double S_, D_;
                // the slot is keyed by the plane number t, the face arrays by the wrapped plane kt
                cell_SD(cr, t, kt, P[2], P[1], P[0], Aa[2], Aa[1], Aa[0], S_, D_);
                const double fv = cr ? F[1].y : F[1].x;
                const double pv = gs_value(L.h2, fv, S_, D_);
                if (cr) { P[1].y = pv; slots[t & 3].po[ly][lx] = pv; }
                else    { P[1].x = pv; slots[t & 3].pe[ly][lx] = pv; }
            }
        }
        // -------- black half-sweep at plane t-2 (window index 3)
        {
            const int kb = t - 2;
            const int cb = ((oy + ly + t) & 1) ^ 1;
            const bool can = is_out && kb >= kz0 && kb < kz1;
            if (can) {
                double S_, D_;
                cell_SD(cb, kb, kb, P[4], P[3], P[2], Aa[4], Aa[3], Aa[2], S_, D_);
                const double fv = cb ? F[3].y : F[3].x;
                const double pv = gs_value(L.h2, fv, S_, D_);
                if (cb) P[3].y = pv; else P[3].x = pv;
                *reinterpret_cast<double2 *>(A.pout + col + plane_stride * (size_t)kb) = P[3];
            }
        }
        __syncthreads();
        // rotate the window and publish plane t+2
#pragma unroll
        for (int q = 4; q > 0; --q) { P[q] = P[q - 1]; Aa[q] = Aa[q - 1]; }
#pragma unroll
        for (int q = 3; q > 0; --q) F[q] = F[q - 1];
        P[0] = pn; Aa[0] = an; F[0] = fn;
        if (need_next) store_slot(t + 2, pn, an);
    }
}

// ------------------------------------------------------------------------------ host side
inline bool stream_sweep_supported(int nx, int ny, int nz)
{
    // any even dims work; below 32^3 the launch is latency-bound and the reference /
    // single-CTA kernels are used instead
    return nx >= 32 && ny >= 32 && nz >= 32;
}

inline int sk_zchunk(int nx, int ny, int nz, int num_sms)
{
    const int tiles = ((nx + SK_OX - 1) / SK_OX) * ((ny + SK_OY - 1) / SK_OY);
    int chunks = (4 * num_sms + tiles - 1) / tiles;     // aim at >= 4 CTAs per SM over the launch
    if (chunks < 1) chunks = 1;
    int zc = (nz + chunks - 1) / chunks;
    if (zc < 16) zc = 16;
    if (zc > 64) zc = 64;
    if (zc > nz) zc = nz;
    return zc;
}

template <bool CELL>
inline int sk_launch_plain(const SkArgs &a, int num_sms, cudaStream_t st)
{
    static bool attr_done = false;
    auto kern = k_stream_sweep<CELL, false, SK_TAIL_NONE>;
    const size_t smem = 4 * sizeof(SkSlot);
    if (!attr_done) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return -1;
        attr_done = true;
    }
    SkArgs b = a;
    b.zchunk = sk_zchunk(a.L.nx, a.L.ny, a.L.nz, num_sms);
    dim3 grid((a.L.nx + SK_OX - 1) / SK_OX, (a.L.ny + SK_OY - 1) / SK_OY, (a.L.nz + b.zchunk - 1) / b.zchunk);
    kern<<<grid, dim3(SK_LX, SK_LY, 1), smem, st>>>(b);
    return 0;
}

// one full red-black sweep p_in -> p_out
inline int launch_stream_sweep(Lv L, bool cell, const double *f, const double *pin, double *pout,
                               int num_sms, cudaStream_t st)
{
    SkArgs a;
    a.L = L; a.f = f; a.pin = pin; a.pout = pout; a.zchunk = 0;
    a.e = nullptr; a.cnx = a.cny = a.cnz = 0; a.fc = nullptr; a.partial = nullptr;
    return cell ? sk_launch_plain<true>(a, num_sms, st) : sk_launch_plain<false>(a, num_sms, st);
}

} // namespace mg
