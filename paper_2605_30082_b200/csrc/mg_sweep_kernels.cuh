// mg_sweep_kernels.cuh -- the level-0 smoother: one full red-black Gauss-Seidel sweep (red
// half-sweep, then black, R9) in ONE streaming pass, read from p_in and written to p_out:
// 32 B per cell of compulsory HBM traffic (p in, p out, f, a).
//
// Geometry.  A CTA owns an (x,y) tile of 64 x S3_TY cells including a halo of 2 and marches
// through a z-chunk.  A warp is one tile row; thread (lx,ly) owns the column of the aligned
// x-pair (2lx, 2lx+1) of row ly and keeps the z-window of its two cells (planes t+3 .. t-3 of
// p, a, f) in a compile-time-indexed register ring (6-fold unrolled step).  At step t it
// updates its red cell of plane t and its black cell of plane t-2; ring 1 of the tile
// recomputes the red values the neighbouring CTA also computes (same expression tree, same
// inputs, same bits), so exact global red->black semantics are kept; rows 0 and S3_TY-1
// (ring 2) only move data.
//
// Data movement (history and measurements: profiles/r1b_sweep.md, r1d_cycle.md):
//   * p and a: cp.async (16 B, .ca) of the thread's own pair into private staging slots, three
//     planes in flight; a thread only reads back what it copied itself, so staging needs no
//     barrier, only cp.async.wait_group;
//   * f never needs to be shared: LDG.128 straight into the ring three steps before its first
//     use, with an L2 prefetch one plane further;
//   * exchange planes in shared memory hold (p, a) as one 16-byte entry per cell, split by
//     colour class: one conflict-free LDS.128 fetches a neighbour's value AND its coefficient
//     (6 neighbour reads + 2 staging reads + 3 stores, all 128-bit, per thread and step);
//   * six exchange slots = the ring length, so every shared-memory address of the unrolled
//     loop is a per-thread base plus a compile-time offset;
//   * everything a step writes to shared memory is first read two steps later and every slot
//     it overwrites was last read two steps earlier: ONE barrier every SECOND step;
//   * steady-state steps (all touched planes inside the domain and the chunk) carry no index
//     mapping and no range tests; the z-chunk length is chosen so that the CTAs fill whole
//     waves of the machine (s3_zchunk).
//
// Boundaries.  Indices outside the domain are wrapped (periodic) or mirrored (Neumann) at
// load time.  A Neumann ghost cell carries a = -a(mirror), so the canonical face
// beta = a_c + a_nb evaluates to exactly +0.0 on a wall face (C2) with no wall logic in the
// update (one XOR with a per-thread sign mask); ghost cells themselves are never updated.  A
// mirrored x-pair arrives reversed: its two publish addresses are swapped (free).
//
// Only the CELL = true instance (level 0) is built.  The stored-face branch (CELL = false) of
// the template lost against the half-sweep launches on every level size (profiles/r1d_cycle.md)
// and is not instantiated; the cycle uses k_smooth_half on levels >= 1.
#pragma once
#include "mg_common.cuh"

namespace mg {

constexpr int S3_LX = 32;                 // lanes: 32 x-pairs = 64 cells loaded in x
constexpr int S3_TY = 16;                 // tile rows loaded
constexpr int S3_OX = 2 * S3_LX - 4;      // 60 output cells in x
constexpr int S3_OY = S3_TY - 4;          // 12 output rows
constexpr int S3_THREADS = S3_LX * S3_TY;
constexpr int S3_NSLOT = 6;
#ifndef S3_FDIRECT
#define S3_FDIRECT 1
#endif
#ifndef S3_BAR2
#define S3_BAR2 1
#endif
constexpr int S3_FAHEAD = 3;              // f is loaded this many steps before its first use
constexpr int S3_FPF = 1;                 // L2 prefetch distance of the f stream beyond that load (measured: 1 < 2 < 4 < none)
#ifndef S3_NST_
#define S3_NST_ 3
#endif
constexpr int S3_NST = S3_NST_;                 // staging planes in flight (cp.async)

constexpr int S3_COMP_BYTES = S3_TY * S3_LX * 16;        // one colour class of one plane
constexpr int S3_SLOT_BYTES = 2 * S3_COMP_BYTES;
constexpr int S3_PAD_BYTES = S3_LX * 16;                   // one row before and after the slots
constexpr int S3_STAGE_OFF = S3_NSLOT * S3_SLOT_BYTES + 2 * S3_PAD_BYTES;
constexpr int S3_STAGE_BYTES = (S3_FDIRECT ? 2 : 3) * S3_COMP_BYTES;         // p and a words of one plane, raw (lo, hi) pairs
constexpr size_t S3_SMEM_BYTES = (size_t)S3_STAGE_OFF + (size_t)S3_NST * S3_STAGE_BYTES;

struct S3Args {
    Lv L;
    const double *f;
    const double *pin;
    double *pout;
    int zchunk;                           // even
};

// source index of global coordinate g along an axis of n cells: in range as is, else
// wrapped (periodic) or mirrored (Neumann, ghost = true)
__device__ __forceinline__ int s3_map(int g, int n, int neumann, bool &ghost)
{
    ghost = false;
    if (g >= 0 && g < n) return g;
    if (!neumann) { g %= n; return g < 0 ? g + n : g; }
    ghost = true;
    int m = g < 0 ? -1 - g : 2 * n - 1 - g;
    if (m < 0 || m >= n) { m %= n; if (m < 0) m += n; }      // far ghost: value irrelevant
    return m;
}
// planes are never further than n away from the domain (no division)
__device__ __forceinline__ int s3_zmap(int k, int n, int neumann, unsigned &sign)
{
    sign = 0u;
    if (k < 0) { sign = neumann ? 0x80000000u : 0u; return neumann ? -1 - k : k + n; }
    if (k >= n) { sign = neumann ? 0x80000000u : 0u; return neumann ? 2 * n - 1 - k : k - n; }
    return k;
}

__device__ __forceinline__ double s3_xor_sign(double v, unsigned m)
{
    return __hiloint2double(__double2hiint(v) ^ (int)m, __double2loint(v));
}
template <int OFF> __device__ __forceinline__ double2 s3_lds128(unsigned addr)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2+%3];\n" : "=d"(v.x), "=d"(v.y) : "r"(addr), "n"(OFF));
    return v;
}
template <int OFF> __device__ __forceinline__ void s3_sts128(unsigned addr, double x, double y)
{
    asm volatile("st.shared.v2.f64 [%0+%1], {%2, %3};\n" ::"r"(addr), "n"(OFF), "d"(x), "d"(y) : "memory");
}
__device__ __forceinline__ double2 s3_ldg128(const char *p)
{
    double2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];\n" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ void s3_prefetch_l2(const char *p)
{
    asm volatile("prefetch.global.L2 [%0];\n" ::"l"(p));
}
template <int OFF> __device__ __forceinline__ void s3_cp_async16(unsigned dst, const char *src)
{
    asm volatile("cp.async.ca.shared.global [%0+%1], [%2], 16;\n" ::"r"(dst), "n"(OFF), "l"(src) : "memory");
}
__device__ __forceinline__ void s3_cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void s3_cp_async_wait()
{
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory");
}

template <int V> struct S3Int { static constexpr int value = V; };

// Components.  Thread (lx,ly) holds its two cells as component 0/1 such that component c
// has x-parity c ^ (ly & 1).  Tile origin and z-chunk origin are even, so the colour of
// component c at plane k is (c + k) & 1 for EVERY thread: which component is red is a
// compile-time property of the unrolled step.  The in-plane neighbours of a cell of
// component c are all of component c^1: rows ly-1, ly+1 at the same lane, and lane
// lx-1 (cell at x-parity 0) or lx+1 (x-parity 1); the other x-neighbour is the thread's
// own partner cell.
template <bool CELL, int RP>
__device__ __forceinline__ void s3_body(const S3Args &A, unsigned smem_base)
{
    const Lv &L = A.L;
    const int lx = threadIdx.x, ly = threadIdx.y;
    const int ox = blockIdx.x * S3_OX, oy = blockIdx.y * S3_OY;
    const int kz0 = blockIdx.z * A.zchunk;
    const int kz1 = min(L.nz, kz0 + A.zchunk);

    // ---- this thread's column
    const int gx = ox - 2 + 2 * lx;              // global x of the pair's even cell (may be outside)
    const int gy = oy - 2 + ly;
    bool ghost_x, ghost_x1, ghost_y;
    const int sx0 = s3_map(gx, L.nx, L.bcx, ghost_x);
    const int sx1 = s3_map(gx + 1, L.nx, L.bcx, ghost_x1);   // same ghost state (nx even)
    const int sy = s3_map(gy, L.ny, L.bcy, ghost_y);
    const bool mirrored = sx0 > sx1;             // Neumann x-ghost pair: (lo,hi) words are reversed
    const int xpair = min(sx0, sx1);             // even: 16-byte aligned pair
    const bool ghost_xy = ghost_x || ghost_y;
    const unsigned sign_xy = ghost_xy ? 0x80000000u : 0u;
    const size_t plane_stride = (size_t)L.nx * L.ny;
    const size_t plane_bytes = plane_stride * sizeof(double);
    // byte offset of this thread's pair inside a plane; every stream address is formed at
    // its use as (kernel-parameter base) + offset, so only the offset lives in registers
    const size_t col_bytes = ((size_t)xpair + (size_t)L.nx * (size_t)sy) * sizeof(double);
    const char *base_p = reinterpret_cast<const char *>(A.pin);
    const char *base_f = reinterpret_cast<const char *>(A.f);
    const char *base_a = reinterpret_cast<const char *>(L.a);
    // the loaded pair is (lo, hi) = cells (xpair, xpair+1); the cell at x-parity 0 is
    // component RP, the one at x-parity 1 component RP^1
    constexpr int C_LO = RP, C_HI = RP ^ 1;

    // ---- shared-memory addresses (bytes).  Entry of (comp, row, lane) inside a slot; the
    // neighbour entries are compile-time offsets from `self` (+-16: lane, +-512: row).
    // Edge threads read a valid, meaningless entry (a pad of one row precedes and follows
    // the slots) instead of branching; their results are never stored.
    const unsigned self = smem_base + (unsigned)(S3_PAD_BYTES + (ly * S3_LX + lx) * 16);
    // publish addresses of the lo / hi word (swapped for a reversed ghost pair)
    const unsigned pub_lo = self + (unsigned)((mirrored ? C_HI : C_LO) * S3_COMP_BYTES);
    const unsigned pub_hi = self + (unsigned)((mirrored ? C_LO : C_HI) * S3_COMP_BYTES);

    // ---- region predicates
    const bool is_out = lx >= 1 && lx <= S3_LX - 2 && ly >= 2 && ly <= S3_TY - 3 && gx >= 0 && gx < L.nx &&
                        gy >= 0 && gy < L.ny;
    const bool w_work = ly >= 1 && ly <= S3_TY - 2;       // warp-uniform: rows that compute at all
    const bool row_r1 = w_work && !ghost_xy;
    // red is recomputed on local x in [1, 62]: everything but the outermost cell of the edge lanes
    const bool red_ok_lo = row_r1 && lx != 0;               // cell at local x = 2lx
    const bool red_ok_hi = row_r1 && lx != S3_LX - 1;       // cell at local x = 2lx + 1
    const bool red_ok0 = C_LO == 0 ? red_ok_lo : red_ok_hi;
    const bool red_ok1 = C_LO == 1 ? red_ok_lo : red_ok_hi;

    // register z-window: ring of 6 planes; plane (t + d) of unrolled step U sits in (U+d) mod 6
    double P[6][2], Aa[6][2], F[6][2];
#pragma unroll
    for (int q = 0; q < 6; ++q)
        for (int c = 0; c < 2; ++c) { P[q][c] = 0.0; Aa[q][c] = 0.0; F[q][c] = 0.0; }

    // ---- global -> shared staging: cp.async (LDGSTS) of this thread's own 16-byte words, S3_NST
    // planes in flight per CTA (3 x 24 KB: the bytes in flight that HBM latency asks for;
    // generation 3a kept one plane in registers and was latency-bound at 3.6 TB/s of loads).
    // A thread only ever reads back what it copied itself, so the staging buffers need no
    // barrier, only cp.async.wait_group.  Plane k uses staging slot (k - t0) mod 3.
    const unsigned stage_self = smem_base + (unsigned)(S3_STAGE_OFF + (ly * S3_LX + lx) * 16);
    auto issue_at = [&](auto Sc, size_t off) __attribute__((always_inline)) {
        constexpr int SLOT = decltype(Sc)::value;
        s3_cp_async16<SLOT * S3_STAGE_BYTES>(stage_self, base_p + off);
        if (CELL) s3_cp_async16<SLOT * S3_STAGE_BYTES + S3_COMP_BYTES>(stage_self, base_a + off);
        if (!S3_FDIRECT) s3_cp_async16<SLOT * S3_STAGE_BYTES + 2 * S3_COMP_BYTES>(stage_self, base_f + off);
        s3_cp_async_commit();
    };
    auto issue = [&](auto Sc, int k) __attribute__((always_inline)) {   // any plane: wrapped / mirrored at the z ends
        unsigned sg;
        issue_at(Sc, col_bytes + (size_t)s3_zmap(k, L.nz, L.bcz, sg) * plane_bytes);
    };
    // steady state: one running offset (plane t+5 of this thread's pair), one 64-bit add per
    // step; the store of plane t-2 is seven planes behind it (is_out threads load and store
    // the same pair)
    size_t roff = col_bytes;
    const size_t back_store = (size_t)(S3_NST + 4) * plane_bytes, back_f = (size_t)(S3_NST + 2 - S3_FAHEAD) * plane_bytes;
    // move a landed plane from staging slot SLOT into ring entry R and publish it to exchange slot R
    auto take = [&](auto Rc, auto Sc, unsigned sign) __attribute__((always_inline)) {
        constexpr int R = decltype(Rc)::value;
        constexpr int SLOT = decltype(Sc)::value;
        const double2 vp = s3_lds128<SLOT * S3_STAGE_BYTES>(stage_self);
        P[R][C_LO] = vp.x; P[R][C_HI] = vp.y;
        if (!S3_FDIRECT) {
            const double2 vf = s3_lds128<SLOT * S3_STAGE_BYTES + 2 * S3_COMP_BYTES>(stage_self);
            F[R][C_LO] = vf.x; F[R][C_HI] = vf.y;
        }
        if (CELL) {
            const double2 va = s3_lds128<SLOT * S3_STAGE_BYTES + S3_COMP_BYTES>(stage_self);
            Aa[R][C_LO] = s3_xor_sign(va.x, sign);
            Aa[R][C_HI] = s3_xor_sign(va.y, sign);
        }
        s3_sts128<R * S3_SLOT_BYTES>(pub_lo, P[R][C_LO], Aa[R][C_LO]);
        s3_sts128<R * S3_SLOT_BYTES>(pub_hi, P[R][C_HI], Aa[R][C_HI]);
    };
    // f never needs to be shared: its pair of plane t+1 is loaded straight into the ring one
    // step ahead of its first use (red half-sweep of plane t+1); an L2 prefetch runs S3_FPF
    // planes further ahead so that this load is an L2 hit
    auto load_f = [&](auto Rc, size_t off) __attribute__((always_inline)) {
        constexpr int R = decltype(Rc)::value;
        const double2 vf = s3_ldg128(base_f + off);
        F[R][C_LO] = vf.x; F[R][C_HI] = vf.y;
    };
    auto zoff = [&](int k) -> size_t { unsigned sg; return col_bytes + (size_t)s3_zmap(k, L.nz, L.bcz, sg) * plane_bytes; };
    auto zsign = [&](int k) -> unsigned { unsigned sg; s3_zmap(k, L.nz, L.bcz, sg); return sg ^ sign_xy; };

    // Gauss-Seidel value (C4, C5) of component C at plane k = ring entry RK = exchange slot RK;
    // ks = source plane of k (face arrays of the coarse levels)
    auto gs = [&](auto Cc, auto RKc, int ks) __attribute__((always_inline)) -> double {
        constexpr int C = decltype(Cc)::value;
        constexpr int RK = decltype(RKc)::value, RM = (RK + 5) % 6, RPL = (RK + 1) % 6;
        constexpr bool x_even = (C == C_LO);       // cell at x-parity 0: left neighbour is in lane lx-1
        constexpr int so = RK * S3_SLOT_BYTES + (C ^ 1) * S3_COMP_BYTES;
        const double2 xn = s3_lds128<so + (x_even ? -16 : 16)>(self);
        const double2 ym = s3_lds128<so - S3_LX * 16>(self);
        const double2 yp = s3_lds128<so + S3_LX * 16>(self);
        const double p_partner = P[RK][C ^ 1];
        const double pxm = x_even ? xn.x : p_partner;
        const double pxp = x_even ? p_partner : xn.x;
        double b[6];
        if (CELL) {
            const double a_c = Aa[RK][C];
            const double a_partner = Aa[RK][C ^ 1];
            b[0] = __dadd_rn(a_c, x_even ? xn.y : a_partner);
            b[1] = __dadd_rn(a_c, x_even ? a_partner : xn.y);
            b[2] = __dadd_rn(a_c, ym.y);
            b[3] = __dadd_rn(a_c, yp.y);
            b[4] = __dadd_rn(a_c, Aa[RM][C]);
            b[5] = __dadd_rn(a_c, Aa[RPL][C]);
        } else {
            // stored minus faces, read through L1/L2 at the (wrapped) source position
            const int x = x_even ? xpair : xpair + 1;
            const int xp = x == L.nx - 1 ? 0 : x + 1;
            const int yp_ = sy == L.ny - 1 ? 0 : sy + 1;
            const int kp = ks == L.nz - 1 ? 0 : ks + 1;
            const size_t pl = plane_stride * (size_t)ks;
            const size_t row = (size_t)L.nx * (size_t)sy;
            const size_t cc = (size_t)x + row + pl;
            b[0] = __ldg(L.bx + cc);
            b[1] = __ldg(L.bx + ((size_t)xp + row + pl));
            b[2] = __ldg(L.by + cc);
            b[3] = __ldg(L.by + ((size_t)x + (size_t)L.nx * (size_t)yp_ + pl));
            b[4] = __ldg(L.bz + cc);
            b[5] = __ldg(L.bz + ((size_t)x + row + plane_stride * (size_t)kp));
        }
        const double S = stencil_S(b, pxm, pxp, ym.x, yp.x, P[RM][C], P[RPL][C]);
        const double D = stencil_D(b);
        return gs_value_rcp(L.h2, F[RK][C], S, D);
    };

    const int t0 = kz0 - 1, t_end = kz1 + 1;
    // ---- prologue: planes t0-1, t0, t0+1 -> ring entries 5, 0, 1; plane t0+2 in flight
    // (plane k uses staging slot (k - t0) mod S3_NST)
    static_assert(S3_FAHEAD == 3, "the prologue loads f of exactly three planes");
    static_assert(S3_NST == 3 || S3_NST == 6, "staging depth must divide the unroll factor");
    issue(S3Int<S3_NST - 1>{}, t0 - 1); issue(S3Int<0>{}, t0); issue(S3Int<1>{}, t0 + 1);
    if (S3_FDIRECT) {
        load_f(S3Int<0>{}, zoff(t0)); load_f(S3Int<1>{}, zoff(t0 + 1));
        load_f(S3Int<2>{}, zoff(min(t0 + 2, kz1 + 1)));
    }
    s3_cp_async_wait<0>();
    take(S3Int<5>{}, S3Int<S3_NST - 1>{}, zsign(t0 - 1));
    take(S3Int<0>{}, S3Int<0>{}, zsign(t0));
    take(S3Int<1>{}, S3Int<1>{}, zsign(t0 + 1));
    issue(S3Int<2 % S3_NST>{}, min(t0 + 2, kz1 + 1));
    issue(S3Int<3 % S3_NST>{}, min(t0 + 3, kz1 + 1));
    issue(S3Int<4 % S3_NST>{}, min(t0 + 4, kz1 + 1));
    if (S3_NST == 6) {
        issue(S3Int<5 % S3_NST>{}, min(t0 + 5, kz1 + 1));
        issue(S3Int<6 % S3_NST>{}, min(t0 + 6, kz1 + 1));
        issue(S3Int<7 % S3_NST>{}, min(t0 + 7, kz1 + 1));
    }
    __syncthreads();

    // one step: red at plane t (ring U), black at plane t-2 (ring U+4), plane t+2 enters ring
    // U+2.  STEADY: every plane touched (t-3 .. t+3) lies inside the domain and inside this
    // CTA's chunk (t-3 .. t+5), so there is no mapping, no range test, and the loads use a running offset.
    auto step = [&](auto Uc, auto Steady, int t) __attribute__((always_inline)) {
        constexpr int U = decltype(Uc)::value;
        constexpr bool STEADY = decltype(Steady)::value != 0;
        constexpr int R_0 = U % 6, R_M2 = (U + 4) % 6, R_P2 = (U + 2) % 6;
        constexpr int RC = (1 + U) & 1;          // red component at plane t (t0 is odd)
        constexpr int BC = RC ^ 1;               // black component at plane t-2
        unsigned sg_t = 0u, sg_b = 0u;
        const int kb = t - 2;
        const int kt = STEADY ? t : s3_zmap(t, L.nz, L.bcz, sg_t);
        const int kbs = STEADY ? kb : s3_zmap(kb, L.nz, L.bcz, sg_b);
        // f of plane t+3 -> ring, three steps before its first use (the entry it overwrites, plane
        // t-3, was last read by the black update of step t-1); measured 2 steps: 1.04 ms, 3: 0.96 ms
        if (!S3_FDIRECT) {
        } else if (STEADY) {
            load_f(S3Int<(U + S3_FAHEAD) % 6>{}, roff - back_f);
            s3_prefetch_l2(base_f + (roff - back_f) + S3_FPF * plane_bytes);
        } else {
            load_f(S3Int<(U + S3_FAHEAD) % 6>{}, zoff(min(t + S3_FAHEAD, kz1 + 1)));
        }
        // Ring-2 rows (the first and the last warp) only move data.  Everywhere else both
        // updates are evaluated unconditionally (two independent chains interleave); only
        // the stores are predicated.
        if (w_work) {
        const double pr = gs(S3Int<RC>{}, S3Int<R_0>{}, kt);
        const double pb = gs(S3Int<BC>{}, S3Int<R_M2>{}, kbs);
        // -------- red half-sweep at plane t
        if ((RC ? red_ok1 : red_ok0) && (STEADY || (sg_t == 0u && t <= kz1))) {
            P[R_0][RC] = pr;
            s3_sts128<R_0 * S3_SLOT_BYTES + RC * S3_COMP_BYTES>(self, pr, Aa[R_0][RC]);
        }
        // -------- black half-sweep at plane t-2
        if (is_out && (STEADY || (kb >= kz0 && kb < kz1))) {
            P[R_M2][BC] = pb;
            double2 o2;
            o2.x = P[R_M2][C_LO];
            o2.y = P[R_M2][C_HI];
            if (STEADY) *reinterpret_cast<double2 *>(reinterpret_cast<char *>(A.pout) + (roff - back_store)) = o2;
            else *reinterpret_cast<double2 *>(A.pout + (size_t)gx + (size_t)L.nx * (size_t)gy +
                                              plane_stride * (size_t)kb) = o2;
        }
        }
        // -------- plane t+2 (in flight for three steps) enters the ring and its exchange
        // slot (last read two barriers ago); plane t+5 goes in flight into the freed staging slot
        constexpr int SLOT = (U + 2) % S3_NST;
        s3_cp_async_wait<S3_NST - 1>();
        take(S3Int<R_P2>{}, S3Int<SLOT>{}, STEADY ? sign_xy : zsign(min(t + 2, kz1 + 1)));
        if (STEADY) { issue_at(S3Int<SLOT>{}, roff); roff += plane_bytes; }
        else issue(S3Int<SLOT>{}, min(t + 2 + S3_NST, kz1 + 1));
        // Shared-memory writes of step t (red values of plane t, publication of plane t+2) are
        // first read in step t+2, and the exchange slot written in step t was last read in step
        // t-2: one barrier every second step orders both.
        if (!S3_BAR2 || (U & 1)) __syncthreads();
    };
    auto generic_steps = [&](int &t, int t_last) __attribute__((always_inline)) {
        for (; t <= t_last; ++t) {
            switch ((t - t0) % 6) {
            case 0: step(S3Int<0>{}, S3Int<0>{}, t); break;
            case 1: step(S3Int<1>{}, S3Int<0>{}, t); break;
            case 2: step(S3Int<2>{}, S3Int<0>{}, t); break;
            case 3: step(S3Int<3>{}, S3Int<0>{}, t); break;
            case 4: step(S3Int<4>{}, S3Int<0>{}, t); break;
            default: step(S3Int<5>{}, S3Int<0>{}, t); break;
            }
        }
    };

    int t = t0;
    // steady steps: t in [kz0+2, ts_end]; entered at ring position 3 (t0 + 3 = kz0 + 2)
    const int ts_end = min(kz1 - 1 - S3_NST, L.nz - 3 - S3_NST);
    generic_steps(t, min(kz0 + 1, t_end));
    if (t + 5 <= ts_end) {
        roff = col_bytes + (size_t)(t + 2 + S3_NST) * plane_bytes;
        for (; t + 5 <= ts_end; t += 6) {
            step(S3Int<3>{}, S3Int<1>{}, t);
            step(S3Int<4>{}, S3Int<1>{}, t + 1);
            step(S3Int<5>{}, S3Int<1>{}, t + 2);
            step(S3Int<0>{}, S3Int<1>{}, t + 3);
            step(S3Int<1>{}, S3Int<1>{}, t + 4);
            step(S3Int<2>{}, S3Int<1>{}, t + 5);
        }
    }
    generic_steps(t, t_end);
}

template <bool CELL>
__global__ void __launch_bounds__(S3_THREADS, 1) k_sweep3(S3Args A)
{
    extern __shared__ __align__(16) unsigned char s3_smem_raw[];
    const unsigned base = (unsigned)__cvta_generic_to_shared(s3_smem_raw);
    // a warp is one tile row, so the row parity is warp-uniform: two specialised bodies
    if (threadIdx.y & 1) s3_body<CELL, 1>(A, base);
    else                 s3_body<CELL, 0>(A, base);
}

// ------------------------------------------------------------------------------ host side
inline bool sweep3_supported(int nx, int ny, int nz)
{
    // any even dims work; below 32^3 the launch is latency-bound and the reference /
    // single-CTA kernels are used instead
    return nx >= 32 && ny >= 32 && nz >= 32;
}

inline int s3_zchunk(int nx, int ny, int nz, int num_sms)
{
    // Long z-chunks amortise the four halo planes and the prologue of a CTA (512^3: 1.14 ms
    // per sweep with 64-plane chunks, 1.05 ms with 172), but the launch must still fill the
    // machine in whole waves (one CTA per SM): over all chunk counts (chunks of at least 16
    // planes) take the one that maximises (filled share of the waves) x (output planes per
    // step): 512^3 -> 3 chunks of 172, 256^3 -> 4 of 64, 1024^3 -> 2 of 512.
    const int tiles = ((nx + S3_OX - 1) / S3_OX) * ((ny + S3_OY - 1) / S3_OY);
    const int max_chunks = nz / 16 > 0 ? nz / 16 : 1;
    int best_c = 1;
    double best_eff = -1.0;
    for (int c = 1; c <= max_chunks; ++c) {
        int zc = ((nz + c - 1) / c + 1) & ~1;
        const int ctas = tiles * ((nz + zc - 1) / zc);
        const int waves = (ctas + num_sms - 1) / num_sms;
        // fraction of SM-time slots that hold a CTA x fraction of a CTA's steps that are output planes
        const double eff = (double)ctas / ((double)waves * num_sms) * (double)zc / (double)(zc + 6);
        if (eff > best_eff + 1e-12) { best_eff = eff; best_c = c; }
    }
    int zc = ((nz + best_c - 1) / best_c + 1) & ~1;   // even: the colour of a component must not depend on the chunk
    if (zc > nz) zc = nz;
    return zc;
}

// opt-in to the dynamic shared memory of k_sweep3; per device, called from mg_create
inline int sweep3_prepare_device()
{
    return cudaFuncSetAttribute(k_sweep3<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)S3_SMEM_BYTES) == cudaSuccess ? 0 : -1;
}

template <bool CELL>
inline int s3_launch(const S3Args &a, int num_sms, cudaStream_t st)
{
    auto kern = k_sweep3<CELL>;
    S3Args b = a;
    b.zchunk = s3_zchunk(a.L.nx, a.L.ny, a.L.nz, num_sms);
    dim3 grid((a.L.nx + S3_OX - 1) / S3_OX, (a.L.ny + S3_OY - 1) / S3_OY, (a.L.nz + b.zchunk - 1) / b.zchunk);
    kern<<<grid, dim3(S3_LX, S3_TY, 1), S3_SMEM_BYTES, st>>>(b);
    return 0;
}

// one full red-black sweep p_in -> p_out
inline int launch_sweep3(Lv L, bool cell, const double *f, const double *pin, double *pout, int num_sms,
                         cudaStream_t st)
{
    S3Args a;
    a.L = L; a.f = f; a.pin = pin; a.pout = pout; a.zchunk = 0;
    if (!cell) return -1;                 // stored-face levels use the half-sweep kernels
    return s3_launch<true>(a, num_sms, st);
}

} // namespace mg
