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
    double p[2][SK_LY][SK_LX];       // p by pair component (see "components" below)
    double a[2][SK_LY][SK_LX];       // a = 0.5/rho (level 0 only)
};

constexpr int SK_DEPTH = 3;           // planes in flight beyond the one being collected
constexpr int SK_NSTAGE = SK_DEPTH + 1;
struct SkStage {                     // raw global layout of one plane of the tile (cp.async target)
    double2 p[SK_LY][SK_LX];
    double2 f[SK_LY][SK_LX];
    double2 a[SK_LY][SK_LX];
};
constexpr size_t SK_SMEM_BYTES = 4 * sizeof(SkSlot) + SK_NSTAGE * sizeof(SkStage);

__device__ __forceinline__ void sk_cp_async16(unsigned d, const void *gmem_src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void sk_cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void sk_cp_async_wait()
{
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory");
}

enum { SK_TAIL_NONE = 0, SK_TAIL_RESTRICT = 1, SK_TAIL_NORM = 2 };

struct SkArgs {
    Lv L;
    const double *f;
    const double *pin;
    double *pout;
    int zchunk;                      // even
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
// same for planes, which are never further than n away from the domain (no division)
__device__ __forceinline__ int sk_map_near(int k, int n, int neumann, bool &ghost)
{
    ghost = false;
    if (k < 0) { ghost = neumann; return neumann ? -1 - k : k + n; }
    if (k >= n) { ghost = neumann; return neumann ? 2 * n - 1 - k : k - n; }
    return k;
}

template <int V> struct SkInt { static constexpr int value = V; };

// Components.  Thread (lx,ly) owns the cells (2lx, 2lx+1) of tile row ly, held as
// component 0/1 such that component c has x-parity c ^ (ly & 1).  With the tile origin
// even in x, y and the z-chunk origin even, the colour of component c at plane k is
// (c + k) & 1 for EVERY thread: which component is red is a compile-time property of
// the (6-fold unrolled) step, so the z-window lives in registers addressed by constants
// (no rotation moves) and colour never costs a select.
template <bool CELL, bool HEAD_PROLONG, int TAIL, int RP>
__device__ __forceinline__ void sk_body(const SkArgs &A, unsigned char *sk_smem_raw)
{
    SkSlot *slots = reinterpret_cast<SkSlot *>(sk_smem_raw);
    SkStage *stages = reinterpret_cast<SkStage *>(sk_smem_raw + 4 * sizeof(SkSlot));
    const Lv &L = A.L;
    const int lx = threadIdx.x, ly = threadIdx.y;
    constexpr int rp = RP;                       // row parity = ly & 1 (warp-uniform)
    const int ox = blockIdx.x * SK_OX, oy = blockIdx.y * SK_OY;
    const int kz0 = blockIdx.z * A.zchunk;
    const int kz1 = min(L.nz, kz0 + A.zchunk);
    const int so = ly * SK_LX + lx;              // offset inside one smem component plane

    // ---- this thread's column
    const int gx = ox - 2 + 2 * lx;              // global x of the pair's even cell (may be outside)
    const int gy = oy - 2 + ly;
    bool ghost_x, ghost_x1, ghost_y;
    const int sx0 = sk_map(gx, L.nx, L.bcx, ghost_x);
    const int sx1 = sk_map(gx + 1, L.nx, L.bcx, ghost_x1);   // ghost_x1 == ghost_x (nx even)
    const int sy = sk_map(gy, L.ny, L.bcy, ghost_y);
    const int xs0 = rp ? sx1 : sx0, xs1 = rp ? sx0 : sx1;    // source x of component 0 / 1
    const size_t rowoff = (size_t)L.nx * (size_t)sy;
    const size_t plane_stride = (size_t)L.nx * L.ny;
    const bool ghost_xy = ghost_x || ghost_y;
    // x neighbour of component c lives in component c^1 of the thread at lx + dx(c)
    constexpr int dx0 = rp ? 1 : -1, dx1 = -dx0;
    // smem offsets of the in-plane neighbours, clamped into the tile: edge threads read a
    // valid (meaningless) word instead of branching; their results are never stored
    const int so_x0 = min(max(so + dx0, 0), SK_LY * SK_LX - 1);
    const int so_x1 = min(max(so + dx1, 0), SK_LY * SK_LX - 1);
    const int so_ym = ly > 0 ? so - SK_LX : so;
    const int so_yp = ly < SK_LY - 1 ? so + SK_LX : so;
    // region flags
    const bool is_out = lx >= 1 && lx <= 30 && ly >= 2 && ly <= 13 && gx >= 0 && gx < L.nx &&
                        gy >= 0 && gy < L.ny;
    const bool row_r1 = ly >= 1 && ly <= 14 && !ghost_xy;
    // component c sits at local x = 2lx + (c^rp); red is recomputed on local x in [1,62]
    const bool red_ok0 = row_r1 && !(lx == 0 && rp == 0) && !(lx == 31 && rp == 1);
    const bool red_ok1 = row_r1 && !(lx == 0 && rp == 1) && !(lx == 31 && rp == 0);

    // register z-window: ring of 6 planes; plane (t + d) of unrolled step U sits in (U+d) mod 6
    double P[6][2], Aa[6][2], F[6][2];
#pragma unroll
    for (int q = 0; q < 6; ++q)
        for (int c = 0; c < 2; ++c) { P[q][c] = 0.0; Aa[q][c] = 0.0; F[q][c] = 0.0; }

    const unsigned stage_addr = (unsigned)__cvta_generic_to_shared(&stages[0].p[ly][lx]);
    // aligned pair holding this thread's two cells, and which half is component 0
    const int xpair = min(sx0, sx1);
    const int c0_hi = xs0 > xs1 ? 1 : 0;          // component 0 is the odd-x (upper) word of the pair
    // asynchronous copy of this thread's words of plane k into its staging buffer (LDGSTS:
    // no registers are tied up, SK_DEPTH planes stay in flight per CTA)
    // per-thread base pointers of the three streams; a plane is one 32x32->64 bit
    // multiply-add away (plane stride in bytes < 2^32, checked on the host)
    const unsigned plane_bytes = (unsigned)(plane_stride * sizeof(double));
    const char *src_p = reinterpret_cast<const char *>(A.pin + (size_t)xpair + rowoff);
    const char *src_f = reinterpret_cast<const char *>(A.f + (size_t)xpair + rowoff);
    const char *src_a = CELL ? reinterpret_cast<const char *>(L.a + (size_t)xpair + rowoff) : nullptr;
    auto issue = [&](int k) {
        bool gz;
        const unsigned sk = (unsigned)sk_map_near(k, L.nz, L.bcz, gz);
        const size_t off = (size_t)sk * plane_bytes;
        const unsigned g = stage_addr + (unsigned)(k & (SK_NSTAGE - 1)) * (unsigned)sizeof(SkStage);
        sk_cp_async16(g, src_p + off);
        sk_cp_async16(g + (unsigned)sizeof(double2) * SK_LY * SK_LX, src_f + off);
        if (CELL) sk_cp_async16(g + 2u * (unsigned)sizeof(double2) * SK_LY * SK_LX, src_a + off);
        sk_cp_async_commit();
    };
    // pick the landed words of plane k out of the staging buffer into a ring entry
    auto collect = [&](int k, double *p2, double *a2, double *f2, bool &ghost_z) {
        const int sk = sk_map_near(k, L.nz, L.bcz, ghost_z);
        const SkStage &G = stages[k & (SK_NSTAGE - 1)];
        const double *gp = reinterpret_cast<const double *>(&G.p[ly][lx]);
        const double *gf = reinterpret_cast<const double *>(&G.f[ly][lx]);
        p2[0] = gp[c0_hi]; p2[1] = gp[c0_hi ^ 1];
        f2[0] = gf[c0_hi]; f2[1] = gf[c0_hi ^ 1];
        if (CELL) {
            const double *ga = reinterpret_cast<const double *>(&G.a[ly][lx]);
            a2[0] = ga[c0_hi]; a2[1] = ga[c0_hi ^ 1];
        }
        if (HEAD_PROLONG) {
            p2[0] = __dadd_rn(p2[0], prolong_value(L, A.e, A.cnx, A.cny, A.cnz, xs0, sy, sk));
            p2[1] = __dadd_rn(p2[1], prolong_value(L, A.e, A.cnx, A.cny, A.cnz, xs1, sy, sk));
        }
    };
    // finish a loaded plane: ghost sign of a, publish to the plane's smem slot
    auto publish = [&](int k, double *p2, double *a2, bool ghost_z) {
        SkSlot &S = slots[k & 3];
        if (CELL) {
            if (ghost_xy || ghost_z) { a2[0] = -a2[0]; a2[1] = -a2[1]; }
            (&S.a[0][0][0])[so] = a2[0]; (&S.a[1][0][0])[so] = a2[1];
        }
        (&S.p[0][0][0])[so] = p2[0]; (&S.p[1][0][0])[so] = p2[1];
    };

    // S and D (C4) of component C of this thread's pair at plane k (smem slot k & 3; face
    // arrays at wrapped plane ks); Pm/Pc/Pp = ring entries of planes k-1, k, k+1
    auto cell_SD = [&](auto Cc, int k, int ks, const double *Pm, const double *Pc, const double *Pp,
                       const double *Am, const double *Ac, const double *Ap, double &S_, double &D_) {
        constexpr int C = decltype(Cc)::value;
        const SkSlot &S = slots[k & 3];
        const double *oth_p = &S.p[C ^ 1][0][0];
        constexpr bool left_is_smem = (C ? dx1 : dx0) < 0;
        const double p_xnb = oth_p[C ? so_x1 : so_x0];
        const double p_partner = Pc[C ^ 1];
        const double pxm = left_is_smem ? p_xnb : p_partner;
        const double pxp = left_is_smem ? p_partner : p_xnb;
        const double pym = oth_p[so_ym], pyp = oth_p[so_yp];
        const double pzm = Pm[C], pzp = Pp[C];
        double b[6];
        if (CELL) {
            const double *oth_a = &S.a[C ^ 1][0][0];
            const double a_c = Ac[C];
            const double a_xnb = oth_a[C ? so_x1 : so_x0];
            const double a_partner = Ac[C ^ 1];
            b[0] = __dadd_rn(a_c, left_is_smem ? a_xnb : a_partner);
            b[1] = __dadd_rn(a_c, left_is_smem ? a_partner : a_xnb);
            b[2] = __dadd_rn(a_c, oth_a[so_ym]);
            b[3] = __dadd_rn(a_c, oth_a[so_yp]);
            b[4] = __dadd_rn(a_c, Am[C]);
            b[5] = __dadd_rn(a_c, Ap[C]);
        } else {
            // stored minus faces, read through L1/L2 at the (wrapped) source position
            const int x = C ? xs1 : xs0;
            const int xp = x == L.nx - 1 ? 0 : x + 1;
            const int yp = sy == L.ny - 1 ? 0 : sy + 1;
            const int kp = ks == L.nz - 1 ? 0 : ks + 1;
            const size_t pl = plane_stride * (size_t)ks;
            const size_t cc = (size_t)x + rowoff + pl;
            b[0] = __ldg(L.bx + cc);
            b[1] = __ldg(L.bx + ((size_t)xp + rowoff + pl));
            b[2] = __ldg(L.by + cc);
            b[3] = __ldg(L.by + ((size_t)x + (size_t)L.nx * (size_t)yp + pl));
            b[4] = __ldg(L.bz + cc);
            b[5] = __ldg(L.bz + ((size_t)x + rowoff + plane_stride * (size_t)kp));
        }
        S_ = stencil_S(b, pxm, pxp, pym, pyp, pzm, pzp);
        D_ = stencil_D(b);
    };

    const int t0 = kz0 - 1, t_end = kz1 + 1;
    // ---- prologue: planes t0-1 .. t0+1 -> ring entries 5, 0, 1; SK_DEPTH more in flight
    {
        static_assert(SK_NSTAGE == 4, "prologue stages exactly four planes");
        issue(t0 - 1); issue(t0); issue(t0 + 1); issue(min(t0 + 2, kz1 + 1));
        sk_cp_async_wait<1>();
        bool gz;
        collect(t0 - 1, P[5], Aa[5], F[5], gz); publish(t0 - 1, P[5], Aa[5], gz);
        collect(t0,     P[0], Aa[0], F[0], gz); publish(t0,     P[0], Aa[0], gz);
        collect(t0 + 1, P[1], Aa[1], F[1], gz); publish(t0 + 1, P[1], Aa[1], gz);
        // their buffers are free again: bring the pipeline to SK_DEPTH planes in flight
#pragma unroll
        for (int d = 3; d <= 1 + SK_DEPTH; ++d) issue(min(t0 + d, kz1 + 1));
    }
    __syncthreads();

    // one step: red at plane t (ring U), black at plane t-2 (ring U+4), load plane t+2 (ring U+2)
    auto step = [&](auto Uc, int t) {
        constexpr int U = decltype(Uc)::value;
        constexpr int R_P1 = (U + 1) % 6, R_0 = U % 6, R_M1 = (U + 5) % 6, R_M2 = (U + 4) % 6,
                      R_M3 = (U + 3) % 6, R_P2 = (U + 2) % 6;
        constexpr int RC = (1 + U) & 1;          // red component at plane t (t0 is odd)
        constexpr int BC = RC ^ 1;               // black component at plane t-2
        // keep SK_DEPTH planes in flight: plane t+2+SK_DEPTH goes into the staging buffer that
        // plane t+1 left at the end of the previous step (always issued, clamped at the end)
        issue(min(t + 2 + SK_DEPTH, kz1 + 1));

        // both updates are evaluated unconditionally (independent chains interleave);
        // only the stores are predicated
        bool ghost_z, ghost_zb;
        const int kt = sk_map_near(t, L.nz, L.bcz, ghost_z);
        const int kb = t - 2;
        const int kbs = sk_map_near(kb, L.nz, L.bcz, ghost_zb);
        double Sr, Dr, Sb, Db;
        cell_SD(SkInt<RC>{}, t, kt, P[R_M1], P[R_0], P[R_P1], Aa[R_M1], Aa[R_0], Aa[R_P1], Sr, Dr);
        cell_SD(SkInt<BC>{}, kb, kbs, P[R_M3], P[R_M2], P[R_M1], Aa[R_M3], Aa[R_M2], Aa[R_M1], Sb, Db);
        const double pr = gs_value_rcp(L.h2, F[R_0][RC], Sr, Dr);
        const double pb = gs_value_rcp(L.h2, F[R_M2][BC], Sb, Db);
        // -------- red half-sweep at plane t
        if ((RC ? red_ok1 : red_ok0) && !ghost_z && t <= kz1) {
            P[R_0][RC] = pr;
            (&slots[t & 3].p[RC][0][0])[so] = pr;
        }
        // -------- black half-sweep at plane t-2
        if (is_out && kb >= kz0 && kb < kz1) {
            P[R_M2][BC] = pb;
            double2 o2;
            o2.x = rp ? P[R_M2][1] : P[R_M2][0];
            o2.y = rp ? P[R_M2][0] : P[R_M2][1];
            *reinterpret_cast<double2 *>(A.pout + (size_t)gx + rowoff + plane_stride * (size_t)kb) = o2;
        }
        __syncthreads();
        // plane t+2 has landed (all but the SK_DEPTH newest groups are complete)
        sk_cp_async_wait<SK_DEPTH>();
        bool gz_next;
        collect(min(t + 2, kz1 + 1), P[R_P2], Aa[R_P2], F[R_P2], gz_next);
        publish(t + 2, P[R_P2], Aa[R_P2], gz_next);
    };

    for (int tb = t0; tb <= t_end; tb += 6) {
        step(SkInt<0>{}, tb);
        if (tb + 1 > t_end) break;
        step(SkInt<1>{}, tb + 1);
        if (tb + 2 > t_end) break;
        step(SkInt<2>{}, tb + 2);
        if (tb + 3 > t_end) break;
        step(SkInt<3>{}, tb + 3);
        if (tb + 4 > t_end) break;
        step(SkInt<4>{}, tb + 4);
        if (tb + 5 > t_end) break;
        step(SkInt<5>{}, tb + 5);
    }
}

template <bool CELL, bool HEAD_PROLONG, int TAIL>
__global__ void __launch_bounds__(SK_THREADS, 1) k_stream_sweep(SkArgs A)
{
    extern __shared__ __align__(16) unsigned char sk_smem_raw[];
    // a warp is one tile row, so the row parity is warp-uniform: two specialised bodies
    if (threadIdx.y & 1) sk_body<CELL, HEAD_PROLONG, TAIL, 1>(A, sk_smem_raw);
    else                 sk_body<CELL, HEAD_PROLONG, TAIL, 0>(A, sk_smem_raw);
}

// ------------------------------------------------------------------------------ host side
inline bool stream_sweep_supported(int nx, int ny, int nz)
{
    // any even dims work; below 32^3 the launch is latency-bound and the reference /
    // single-CTA kernels are used instead
    return nx >= 32 && ny >= 32 && nz >= 32 && (size_t)nx * ny * sizeof(double) < 0xffffffffull;
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
    return (zc + 1) & ~1;            // even: the colour of a component must not depend on the chunk
}

template <bool CELL>
inline int sk_launch_plain(const SkArgs &a, int num_sms, cudaStream_t st)
{
    static bool attr_done = false;
    auto kern = k_stream_sweep<CELL, false, SK_TAIL_NONE>;
    const size_t smem = SK_SMEM_BYTES;
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
