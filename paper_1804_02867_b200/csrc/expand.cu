// Frontier expansion kernels.  One level of the traversal is
//   k_order        lists the parents of the level by kind: first visit of i* / revisit of i* (the producer of an entry
//                  stored i*, E = EF_i* and the index of the visited record of i* in its header)
//   k_expand       EVALUATES every child (discard tests, beam key):
//                    first visit (PROC1/1', Eq 3): one warp per parent staged in shared memory by a bulk
//                      asynchronous copy, ONE LANE PER OR-ALTERNATIVE of i*; a child on a new arc of a pathway whose
//                      integers are far from the 2^62 guard needs lane-local work only (scale k = c / gcd(|E|, c), its own
//                      column of S for the new unbalanced count, the linear state hash); alternatives that are arcs of the
//                      support take the warp-cooperative general routine;
//                    revisit (PROC2-4, Eq 4 / Eq 5): exactly one child; 8 lanes per parent, four
//                      parents per warp, parents read in place;
//                  a child costs an 8-byte key and an 8-byte tag (general routine: plus a 64-byte task)
//   k_select_*     beam threshold over the keys (post.cu)
//   k_compact      lists the survivors, sizes them and reserves their places in the next frontier / candidate buffer
//   k_materialise  builds every surviving child from its parent (8 lanes per child)
// All grids are sized for the machine, the work is found through the device-resident control block: the host enqueues
// whole batches of levels without reading anything back.
#include <climits>

#include "device_common.cuh"
#include "launch.hpp"

namespace efm {

enum { CH_OK = 0, CH_NONPOS = 1, CH_OVERFLOW = 2 };
#ifndef EFM_MIN_BLOCKS
#define EFM_MIN_BLOCKS 24   // resident one-warp blocks per SM the register allocation aims at (80 registers)
#endif
// Work items are small: the dynamic distribution then evens out the very different costs of parents (measured on genome,
// cap 2^18, k_expand per step: 4 / 8 / 16 / 32 revisits per item 30.6 / 31.9 / 34.3 / 38.8 ms; 2 / 4 / 8 / 16 first visits
// 30.0 / 30.1 / 30.6 / 32.3 ms)
#ifndef EFM_RPI
#define EFM_RPI 4
#endif
#ifndef EFM_PPI
#define EFM_PPI 4
#endif
constexpr int kParentsPerItem = EFM_PPI;    // first-visit parents a warp takes per work item
constexpr int kRevisitPerItem = EFM_RPI;    // revisit parents a warp takes per work item (four at a time, 8 lanes each)
#ifndef EFM_STAGE_BYTES
#define EFM_STAGE_BYTES 1024   // 1 / 1.5 / 2 KB: 28.9 / 29.5 / 29.8 ms (the shared memory not used is L1 for the graph)
#endif
constexpr int kStageBytes = EFM_STAGE_BYTES;   // staging buffer per parent (larger entries are read in place)
constexpr u32 FULL = 0xffffffffu;
constexpr u64 kSmall = 1ULL << 40;   // fast arithmetic: every flux and extra flux of the parent below this ...
constexpr int kSmallCoef = 1 << 20;  // ... and every coefficient below this: no product can reach 2^62
constexpr u32 kTaskChunk = 16;       // task slots a warp reserves per atomic

// ------------------------------------------------------------------ collectives over a group of G consecutive lanes
template <int G>
__device__ __forceinline__ u64 g_sum(u32 m, u64 v) {
#pragma unroll
    for (int o = G / 2; o; o >>= 1) v += __shfl_xor_sync(m, v, o);
    return v;
}
__device__ __forceinline__ u64 g_max(u32 m, u64 v) {   // two 32-bit redux instead of 64-bit shuffle rounds
    const u32 hi = (u32)(v >> 32);
    const u32 mh = __reduce_max_sync(m, hi);
    const u32 ml = __reduce_max_sync(m, hi == mh ? (u32)v : 0u);
    return ((u64)mh << 32) | ml;
}
__device__ __forceinline__ u64 g_min(u32 m, u64 v) { return ~g_max(m, ~v); }

// ------------------------------------------------------------------ integer helpers
// The rarely taken arithmetic (64-bit division, gcd) stays out of line.
__device__ __noinline__ u64 udiv64(u64 a, u64 b) { return a / b; }
__device__ __noinline__ u64 umod64(u64 a, u64 b) { return a % b; }
__device__ __noinline__ i64 sdiv64(i64 a, i64 b) { return a / b; }
__device__ __noinline__ u64 gcd64(u64 a, u64 b) {   // binary gcd
    if (a == 0) return b;
    if (b == 0) return a;
    const int sh = __ffsll((i64)(a | b)) - 1;
    a >>= (__ffsll((i64)a) - 1);
    do {
        b >>= (__ffsll((i64)b) - 1);
        if (a > b) { u64 t = a; a = b; b = t; }
        b -= a;
    } while (b);
    return a << sh;
}
struct S128 { u64 lo; i64 hi; };
__device__ __forceinline__ S128 mul_s(i64 a, i64 b) { S128 r; r.lo = (u64)a * (u64)b; r.hi = __mul64hi(a, b); return r; }
__device__ __forceinline__ S128 add_s(S128 a, S128 b) {
    S128 r; r.lo = a.lo + b.lo; r.hi = a.hi + b.hi + (i64)(r.lo < a.lo); return r;
}
__device__ __forceinline__ bool abs_gt_guard(S128 x) {   // |x| > 2^62
    if (x.hi < 0) { x.lo = ~x.lo + 1ULL; x.hi = ~x.hi + (i64)(x.lo == 0); }
    return x.hi != 0 || x.lo > EFM_GUARD;
}
__device__ __forceinline__ bool umul_gt_guard(u64 a, u64 b) {  // a*b > 2^62, a, b >= 0
    return __umul64hi(a, b) != 0 || a * b > EFM_GUARD;
}
__device__ __forceinline__ u64 abs64(i64 v) { return (u64)(v < 0 ? -v : v); }
__device__ __forceinline__ u64 arc_mult(const DevGraph& g, u32 a) { return __ldg(&g.arc_mix[a]); }
// x mod r, r > 0: one 32-bit division when both fit, the out-of-line 64-bit routine otherwise
__device__ __forceinline__ u64 mod_any(u64 x, u64 r) {
    if (((x | r) >> 32) == 0) return (u64)((u32)x % (u32)r);
    return umod64(x, r);
}
// gcd(E, c), E / gcd and c / gcd; c = 1, 2, 3 without a division
__device__ __forceinline__ void scale_of(u64 absE, u32 c, u64& k, u64& d) {
    if (c == 1) { k = 1; d = absE; return; }
    if (c == 2) { const bool ev = (absE & 1ULL) == 0; k = ev ? 1u : 2u; d = ev ? absE >> 1 : absE; return; }
    if (c == 3) { const u64 qd = absE / 3ULL; const bool dv = qd * 3ULL == absE; k = dv ? 1u : 3u; d = dv ? qd : absE; return; }
    const u64 gg = gcd64(umod64(absE, (u64)c), (u64)c);
    k = (u64)(c / (u32)gg); d = gg == 1 ? absE : udiv64(absE, gg);
}

// Common divisor g of the un-normalised child (reading G10): g = gcd(T, k f_t for t != ia) over the group's lanes.
// Remainders instead of a gcd per element: with r = T, the smallest non-zero remainder of the k f_t modulo r is divided
// by everything g divides, so r shrinks to it; r = 1 settles g = 1 (the usual case), no non-zero remainder means every
// k f_t is a multiple of r, and then g = gcd(T, r) (g divides r, r divides every k f_t).
template <int G>
__device__ __forceinline__ u64 common_divisor(u32 gmask, int gl, const i64* flux, int ns, int ia, u64 k, u64 T) {
    if (T == 1) return 1;
    u64 r = T;
#pragma unroll 1
    for (;;) {
        u64 mn = ~0ULL;
#pragma unroll 1
        for (int t0 = 0; t0 < ns; t0 += G) {   // group-uniform trip count
            const int t = t0 + gl;
            u64 m = 0;
            if (t < ns && t != ia) m = mod_any(k * (u64)flux[t], r);   // k f_t <= 2^62 (no overflow was found before)
            if (__any_sync(gmask, m == 1)) return 1;
            if (m) mn = min(mn, m);
        }
        mn = g_min(gmask, mn);
        if (mn == ~0ULL) return r == T ? T : gcd64(T, r);
        if (mn == 1) return 1;
        r = mn;   // strictly smaller: the loop ends
    }
}

// ------------------------------------------------------------------ asynchronous staging (bulk copy + mbarrier)
__device__ __forceinline__ u32 smem_u32(const void* p) { return (u32)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(u64* bar, u32 count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(u64* bar, u32 bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, u32 bytes, u64* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(u64* bar, u32 parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}

__device__ __forceinline__ bool sbit(const u32* bits, int a) { return (bits[a >> 5] >> (a & 31)) & 1u; }

// Per-warp chunked reservation of child slots: one atomic per kKeyChunk keys.  A round that does not fit the rest of the
// chunk takes the rest and continues in a fresh chunk: no slot is stranded before the warp finishes.
constexpr u64 kNoSlot = ~0ULL;
struct KeyOut {
    u64 base; u32 left;
    // one slot for every lane with want = true (others, and everyone after an overflow, get kNoSlot); warp-wide call
    __device__ __forceinline__ u64 reserve(const ExpandArgs& A, LevelCtl* lv, int lane, bool want) {
        const u32 m = __ballot_sync(FULL, want);
        const u32 cnt = (u32)__popc(m);
        if (cnt == 0) return kNoSlot;
        const u32 rank = (u32)__popc(m & ((1u << lane) - 1u));
        u64 slot;
        if (cnt > left) {
            u64 b = 0;
            if (lane == 0) b = atomicAdd(&lv->n_slots, (u64)kKeyChunk);
            b = __shfl_sync(FULL, b, 0);
            if (__builtin_expect(b + kKeyChunk > A.max_keys, 0)) {
                if (lane == 0) atomicOr(&A.ctl->error, (u32)ERR_KEYS);
                for (u32 t = lane; t < left; t += 32) A.keys[base + t] = kKeySentinel;
                left = 0;
                return kNoSlot;
            }
            slot = rank < left ? base + rank : b + (rank - left);
            base = b + (cnt - left); left = kKeyChunk - (cnt - left);
        } else {
            slot = base + rank;
            base += cnt; left -= cnt;
        }
        return want ? slot : kNoSlot;
    }
    __device__ __forceinline__ void finish(const ExpandArgs& A, int lane) {
        for (u32 t = lane; t < left; t += 32) A.keys[base + t] = kKeySentinel;
        left = 0;
    }
};
struct TaskOut {   // task slots need not be dense: a warp takes kTaskChunk at a time, unused ones are never referenced
    u64 base; u32 left;
    // warp-uniform call: `cnt` slots (<= kTaskChunk); returns the first or kNoSlot
    __device__ __forceinline__ u64 reserve(const ExpandArgs& A, LevelCtl* lv, int lane, u32 cnt) {
        if (cnt > left) {
            u64 b = 0;
            if (lane == 0) b = atomicAdd(&lv->n_tasks, (u64)kTaskChunk);
            b = __shfl_sync(FULL, b, 0);
            if (__builtin_expect(b + kTaskChunk > A.max_tasks, 0)) {
                if (lane == 0) atomicOr(&A.ctl->error, (u32)ERR_KEYS);
                left = 0;
                return kNoSlot;
            }
            base = b; left = kTaskChunk;
        }
        const u64 s = base;
        base += cnt; left -= cnt;
        return s;
    }
};

// ------------------------------------------------------------------ k_order: parents of the level by kind
// Reads the offset of every entry of the level (allocation order), its size (offset of the next entry) and two header
// words, and appends it to the first-visit list (front of plist) or the revisit list (back of plist).  Thread 0 clears the
// counters of the other level set: nothing of the previous level is needed any more, and the children of this level
// allocate there.
constexpr int kOrderItems = 4;
__global__ void __launch_bounds__(256) k_order(const __grid_constant__ ExpandArgs A) {
    __shared__ u32 s_w[2][8];
    __shared__ u64 s_base[2];
    Ctl* ctl = A.ctl;
    LevelCtl* lv = &ctl->lv[A.par];
    const u64 alloc = lv->alloc;
    // after a capacity error the frontier is incomplete: the remaining levels of the batch do nothing
    const u64 n = ctl->error ? 0ULL : alloc >> kAllocShift, total_units = alloc & kAllocUnitMask;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        LevelCtl* o = &ctl->lv[A.par ^ 1];
        o->alloc = 0; o->nF = 0; o->nR = 0; o->work = 0; o->n_slots = 0; o->n_tasks = 0; o->n_keys = 0; o->n_done = 0; o->n_surv = 0;
        if (n) atomicAdd(&ctl->st[ST_EXPANDED], n);
        if (A.level >= A.max_levels && n) atomicOr(&ctl->error, (u32)ERR_LEVELS);
    }
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    constexpr u64 kTile = 256 * kOrderItems;
    u64 bytes = 0;
    for (u64 tile = (u64)blockIdx.x * kTile; tile < n; tile += (u64)gridDim.x * kTile) {
        u64 word[kOrderItems];
        u32 isF = 0, isR = 0;
#pragma unroll
        for (int j = 0; j < kOrderItems; ++j) {
            const u64 i = tile + (u64)j * 256 + threadIdx.x;
            word[j] = 0;
            if (i < n) {
                const u64 off = __ldg(&A.cur_off[i]);
                const u64 nx = i + 1 < n ? __ldg(&A.cur_off[i + 1]) : total_units;
                const u32* h = (const u32*)(A.cur + (off << 4));
                const u32 w0 = __ldg(h), w10 = __ldg(h + 10);
                word[j] = off | ((nx - off) << kListShift);
                bytes += algo_entry_bytes(w0 & 0xffffu, w0 >> 16);
                if (w10 >> 16) isR |= 1u << j; else isF |= 1u << j;
            }
        }
        u32 v[2] = {(u32)__popc(isF), (u32)__popc(isR)}, ex[2];
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            u32 x = v[c];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const u32 y = __shfl_up_sync(FULL, x, o); if (lane >= o) x += y; }
            ex[c] = x - v[c];
            if (lane == 31) s_w[c][wib] = x;
        }
        __syncthreads();
        if (threadIdx.x < 2) {
            const int c = threadIdx.x;
            u32 tot = 0;
            for (int w = 0; w < 8; ++w) { const u32 t = s_w[c][w]; s_w[c][w] = tot; tot += t; }
            s_base[c] = tot ? atomicAdd(c == 0 ? &lv->nF : &lv->nR, (u64)tot) : 0ULL;
        }
        __syncthreads();
        u64 pf = s_base[0] + s_w[0][wib] + ex[0], pr = s_base[1] + s_w[1][wib] + ex[1];
#pragma unroll
        for (int j = 0; j < kOrderItems; ++j) {
            if ((isF >> j) & 1u) A.plist[pf++] = word[j];
            else if ((isR >> j) & 1u) A.plist[A.max_frontier - 1 - (pr++)] = word[j];
        }
        __syncthreads();
    }
    bytes = g_sum<32>(FULL, bytes);
    if (lane == 0 && bytes) atomicAdd(&ctl->st[ST_ALGO_BYTES], bytes);
}

// ------------------------------------------------------------------ k_expand
struct WarpAcc { u32 children, done, general; };   // warp-uniform counters kept in registers, flushed once per warp

// Header of an entry (three 16-byte words) decoded into registers.
struct Hdr {
    int ns, nv, nu, istar, vk, ones;
    u32 cand;
    u64 hs, hv, big;
    i64 E;
};
__device__ __forceinline__ Hdr decode_hdr(const uint4 h0, const uint4 h1, const uint4 h2) {
    Hdr H;
    H.ns = (int)(h0.x & 0xffffu); H.nv = (int)(h0.x >> 16); H.nu = (int)(h0.y & 0xffffu); H.ones = (int)(h0.y >> 16);
    H.hs = (u64)h0.z | ((u64)h0.w << 32);
    H.hv = (u64)h1.x | ((u64)h1.y << 32);
    H.big = (u64)h1.z | ((u64)h1.w << 32);
    H.E = (i64)((u64)h2.x | ((u64)h2.y << 32));
    H.istar = (int)(h2.z & 0xffffu); H.vk = (int)(h2.z >> 16) - 1;
    H.cand = h2.w;
    return H;
}
__device__ __forceinline__ void write_task(const ExpandArgs& A, u64 ti, int ca, int cia, int cnu, u32 flags, u64 ck, u64 cd, u64 cT, u64 cg,
                                           u64 chs, u64 chv, u64 newrec) {
    uint4* tk = A.tasks + 4 * ti;
    __stcs(tk + 0, make_uint4(0u, (u32)ca | ((u32)(cia & 0xffff) << 16), (u32)cnu | (flags << 16), (u32)ck));
    __stcs(tk + 1, make_uint4((u32)cd, (u32)(cd >> 32), (u32)cT, (u32)(cT >> 32)));
    __stcs(tk + 2, make_uint4((u32)cg, (u32)(cg >> 32), (u32)chs, (u32)(chs >> 32)));
    __stcs(tk + 3, make_uint4((u32)chv, (u32)(chv >> 32), (u32)newrec, (u32)(newrec >> 32)));
}

// ---- revisit parents (PROC2-4; readings G2-G5): 8 lanes per parent, read in place.
// MODES: the build with the sampling mode (8(f)-1), the reaction mask (8(f)-2) and the per-candidate end records; the
// plain exhaustive traversal runs the build without them.
template <bool MODES>
__device__ __forceinline__ void expand_revisits(const ExpandArgs& A, LevelCtl* lv, u64 first, u64 nR, int lane, KeyOut& ko, TaskOut& to,
                                                WarpAcc& acc) {
    constexpr int G = 8;
    const int gl = lane & 7, grp = lane >> 3;
    const u32 gmask = 0xffu << (grp * 8);
    Ctl* ctl = A.ctl;
    const bool small_graph = A.g.max_coef < kSmallCoef;
    // list words of the item's parents: lane l holds parent l.  The entries are read in place; while four parents are
    // processed, the lines of the next four are requested into L1 (one 128-byte line per lane and step).
    const u64 mylw = first + (u64)lane < nR ? __ldg(&A.plist[A.max_frontier - 1 - (first + (u64)lane)]) : 0ULL;
    auto request = [&](int r) {
        const u64 w = __shfl_sync(FULL, mylw, (4 * r + grp) & 31);
        const unsigned char* e = A.cur + ((w & kListOffMask) << 4);
        const u32 bytes = (u32)((w >> kListShift) << 4);
#pragma unroll 1
        for (u32 o = (u32)gl * 128u; o < bytes; o += 1024u) asm volatile("prefetch.global.L1 [%0];\n" ::"l"(e + o));
    };
    request(0);
#pragma unroll 1
    for (int r = 0; r < kRevisitPerItem / 4; ++r) {
        const u64 idx = first + (u64)(4 * r + grp);
        const bool live = idx < nR;
        if (!__any_sync(FULL, live)) break;
        if (r + 1 < kRevisitPerItem / 4) request(r + 1);
        const u64 pid = A.max_frontier - 1 - (live ? idx : first);
        const u64 lw = __shfl_sync(FULL, mylw, live ? 4 * r + grp : 0);
        const unsigned char* eb = A.cur + ((lw & kListOffMask) << 4);
        const Hdr H = decode_hdr(__ldg((const uint4*)eb), __ldg((const uint4*)eb + 1), __ldg((const uint4*)eb + 2));
        const int ns = H.ns, nv = H.nv, nu = H.nu, istar = H.istar;
        const i64* flux = (const i64*)(eb + kHdr);
        const u64* vis = (const u64*)(flux + ns);
        const i64* ef = (const i64*)(vis + nv);
        const u16* arc = (const u16*)(ef + nu);
        const u16* efmet = arc + ns;
        const i64 E = H.E;
        const bool fwd = E > 0;
        const u64 absE = abs64(E);
        const u64 rec = vis[H.vk];
        const int cntv = (int)(rec >> 48) + 1;
        bool act = live;
        if (live && cntv > A.max_loop) {
            act = false;
            if (gl == 0) { atomicAdd(&ctl->st[ST_NOT_EFM], 1ULL); if (MODES && A.cand_end) A.cand_end[H.cand] = END_NOTEFM | ((u64)A.level << 8); }
        }
        const int PI = (int)((rec >> 16) & 0xffffu), PO = (int)(rec & 0xffffu);
        // position and coefficient of PI in I[i*] and of PO in O[i*]: from the columns of the two arcs
        int lPI = -1, lPO = -1, cPI = 0, cPO = 0;
        {
            const int a0 = __ldg(&A.g.col_ptr[PI]), a1 = __ldg(&A.g.col_ptr[PI + 1]);
            const int b0 = __ldg(&A.g.col_ptr[PO]), b1 = __ldg(&A.g.col_ptr[PO + 1]);
#pragma unroll 1
            for (int q = a0 + gl; q < a1; q += G) { const int2 e = __ldg(&A.g.col[q]); if (col_met(e) == istar && e.y > 0) { lPI = col_pos(e); cPI = e.y; } }
#pragma unroll 1
            for (int q = b0 + gl; q < b1; q += G) { const int2 e = __ldg(&A.g.col[q]); if (col_met(e) == istar && e.y < 0) { lPO = col_pos(e); cPO = -e.y; } }
            lPI = __reduce_max_sync(gmask, lPI); cPI = __reduce_max_sync(gmask, cPI);
            lPO = __reduce_max_sync(gmask, lPO); cPO = __reduce_max_sync(gmask, cPO);
        }
        // Def 11: forward PO ~ SI, backward PI ~ SO, secondary = any arc of that side in the support (G5).
        // The support is scanned once: arcs that produce (forward) / consume (backward) i* are looked up in the table,
        // and the positions of PI and PO in the support come along.
        const int nI = __ldg(&A.g.node[istar]).y;
        const i64 doff = __ldg(&A.g.dep_off[istar]);
        // the pair (PO, PI) itself is one of the candidates in either direction: its bit often settles the test
        const i64 b0 = doff + (i64)lPO * nI + lPI;
        const bool dep0 = ((__ldg(&A.g.dep_bits[b0 >> 5]) >> (b0 & 31)) & 1u) != 0;
        bool dep = dep0;
        int iaPI = -1, iaPO = -1;
        const u64* sig = A.g.colsig + (fwd ? 0 : 1);   // metabolites an arc produces / consumes
#pragma unroll 1
        for (int t = gl; t < ns; t += G) {
            const int a = arc[t];
            if (a == PI) { iaPI = t; continue; }
            if (a == PO) { iaPO = t; continue; }
            if (dep0 || !((__ldg(&sig[2 * a]) >> (istar & 63)) & 1ULL)) continue;   // the column of a does not hold i* on that side
            const int q0 = __ldg(&A.g.col_ptr[a]), q1 = __ldg(&A.g.col_ptr[a + 1]);
#pragma unroll 1
            for (int q = q0; q < q1; ++q) {
                const int2 e = __ldg(&A.g.col[q]);
                if (col_met(e) != istar) continue;
                if (fwd && e.y > 0) { const i64 b = doff + (i64)lPO * nI + col_pos(e); dep = dep || ((__ldg(&A.g.dep_bits[b >> 5]) >> (b & 31)) & 1u); }
                if (!fwd && e.y < 0) { const i64 b = doff + (i64)col_pos(e) * nI + lPI; dep = dep || ((__ldg(&A.g.dep_bits[b >> 5]) >> (b & 31)) & 1u); }
            }
        }
        dep = __any_sync(gmask, dep);
        iaPI = __reduce_max_sync(gmask, iaPI); iaPO = __reduce_max_sync(gmask, iaPO);
        int ca, cc, csign, cia;
        if (fwd) { if (!dep) { ca = PO; cc = cPO; csign = +1; cia = iaPO; } else { ca = PI; cc = cPI; csign = -1; cia = iaPI; } }   // Eq 4 / Eq 5
        else     { if (!dep) { ca = PI; cc = cPI; csign = +1; cia = iaPI; } else { ca = PO; cc = cPO; csign = -1; cia = iaPO; } }
        const u64 newrec = vis_pack((u32)istar, (u32)PI, (u32)PO, (u32)cntv);
        // ---- bump(f, a, sign |E| / c) of SURVEY.md 8(c) O6
        u64 ck, cd;
        scale_of(absE, (u32)max(cc, 1), ck, cd);
        const u64 fa = (u64)flux[max(cia, 0)];
        const bool smallP = small_graph && H.big < kSmall;   // no product can reach the guard
        bool ovf = false, nonpos = false;
        u64 cT;
        {
            const u64 lo = ck * fa, hi = smallP ? 0ULL : __umul64hi(ck, fa);
            if (csign > 0) { cT = lo + cd; const u64 hi2 = hi + (cT < lo); ovf = hi2 != 0 || cT > EFM_GUARD; }
            else if (hi == 0 && lo <= cd) { nonpos = true; cT = 0; }   // k f_a - d <= 0
            else { cT = lo - cd; const u64 hi2 = hi - (lo < cd); ovf = hi2 != 0 || cT > EFM_GUARD; }
        }
        const bool bigk = !smallP && ck > 1 && umul_gt_guard(ck, H.big);
        if (__builtin_expect(act && bigk, 0)) {   // exact: the largest flux among t != ia
            u64 mx = 0;
#pragma unroll 1
            for (int t = gl; t < ns; t += G) if (t != cia) mx = max(mx, (u64)flux[t]);
            mx = g_max(gmask, mx);
            ovf = ovf || umul_gt_guard(ck, mx);
        }
        int status = ovf ? CH_OVERFLOW : (nonpos ? CH_NONPOS : CH_OK);   // Prop 3, G11
        // extra fluxes of the un-normalised child: EF'_i = k EF_i + sign d s_ia (Eq 2 on the scaled fluxes)
        int cnu = nu;
        const int qa0 = __ldg(&A.g.col_ptr[ca]), qa1 = __ldg(&A.g.col_ptr[ca + 1]);
        if (act && status == CH_OK) {
            bool ovf2 = false;
            if (__builtin_expect(bigk, 0)) {   // exact sweep over the unbalanced metabolites outside col(a)
#pragma unroll 1
                for (int t = gl; t < nu; t += G) {
                    const int i = efmet[t];
                    bool in_a = false;
#pragma unroll 1
                    for (int q = qa0; q < qa1; ++q) in_a = in_a || col_met(__ldg(&A.g.col[q])) == i;
                    if (!in_a) ovf2 = ovf2 || abs_gt_guard(mul_s((i64)ck, ef[t]));
                }
            }
            int delta = 0;
            const i64 sdd = csign > 0 ? (i64)cd : -(i64)cd;
#pragma unroll 1
            for (int q = qa0 + gl; q < qa1; q += G) {
                const int2 e = __ldg(&A.g.col[q]);
                const int met = col_met(e);
                i64 efp = 0;
#pragma unroll 1
                for (int t = 0; t < nu; ++t) if ((int)efmet[t] == met) efp = ef[t];
                bool nz;
                if (smallP) nz = ((i64)ck * efp + sdd * (i64)e.y) != 0;
                else {
                    const S128 x = add_s(mul_s((i64)ck, efp), mul_s(sdd, (i64)e.y));
                    ovf2 = ovf2 || abs_gt_guard(x);
                    nz = (x.lo | (u64)x.hi) != 0;
                }
                delta += (int)nz - (int)(efp != 0);
            }
            if (__any_sync(gmask, ovf2)) status = CH_OVERFLOW;
            else cnu = nu + __reduce_add_sync(gmask, delta);
        }
        if (act && status != CH_OK) {
            if (gl == 0) {
                atomicAdd(&ctl->st[status == CH_OVERFLOW ? ST_OVERFLOW : ST_NONPOS], 1ULL);
                if (MODES && A.cand_end) A.cand_end[H.cand] = (status == CH_OVERFLOW ? END_OVERFLOW : END_NONPOS) | ((u64)A.level << 8);
            }
            act = false;
        }
        // gcd normalisation (reading G10): g = gcd(T, k f_t for t != a)
        // A flux of 1 on another arc settles it: g divides k then, and gcd(T, k) = gcd(d, k) = 1.
        u64 cg = 1;
        if (act && H.ones - (int)(fa == 1) <= 0) cg = common_divisor<G>(gmask, gl, flux, ns, cia, ck, cT);
        u64 chs;
        if (cg == 1) chs = ck * H.hs + arc_mult(A.g, (u32)ca) * (cT - ck * fa);   // linear arc part of the state hash
        else {
            chs = 0;
#pragma unroll 1
            for (int t = gl; t < ns; t += G) {
                const u64 F = t == cia ? cT : ck * (u64)flux[t];
                chs += arc_mult(A.g, (u32)arc[t]) * udiv64(F, cg);
            }
            chs = g_sum<G>(gmask, chs);
        }
        const u64 chv = H.hv + vis_term(newrec) - vis_term(rec);
        const bool cdone = cnu == 0;
        // ---- emit: key + tag + task
        const bool emit = act && gl == 0;
        const u32 em = __ballot_sync(FULL, emit);
        const u32 ne = (u32)__popc(em);
        acc.children += ne; acc.general += ne; acc.done += (u32)__popc(__ballot_sync(FULL, emit && cdone));
        if (ne) {
            const u64 slot = ko.reserve(A, lv, lane, emit);
            const u64 tb = to.reserve(A, lv, lane, ne);
            if (emit && slot != kNoSlot) {
                if (tb == kNoSlot) __stcs(&A.keys[slot], kKeySentinel);
                else {
                    const u64 ti = tb + (u64)__popc(em & ((1u << lane) - 1u));
                    __stcs(&A.keys[slot], cdone ? kKeyDone : beam_key((u32)cnu, mix64(chs + chv)));
                    __stcs(&A.tags[slot], (pid << kTagParentShift) | ((u64)TK_TASK << 32) | ti);
                    write_task(A, ti, ca, cia, cnu, (csign < 0 ? (u32)TF_NEG : 0u) | (u32)TF_INSUPP, ck, cd, cT, cg, chs, chv, newrec);
                }
            }
        }
    }
}

// ---- first-visit parents (PROC1 / PROC1', Eq 3; readings G1, G13, G14, G15, G22)
struct WarpSmem {
    unsigned char* stage[2]; u64* bar; u32* sbits; u16* upos;
};

template <bool MODES>
__device__ __forceinline__ void expand_first_visits(const ExpandArgs& A, LevelCtl* lv, u64 first, u64 nF, int lane, const WarpSmem& S,
                                                    u32& phase, KeyOut& ko, TaskOut& to, WarpAcc& acc) {
    Ctl* ctl = A.ctl;
    const bool fast_graph = !A.no_fast && A.g.max_coef < kSmallCoef;
    const int cnt = (int)min((u64)kParentsPerItem, nF - first);
    // list words of the item's parents: lane j holds parent j
    const u64 mylw = lane < cnt ? __ldg(&A.plist[first + lane]) : 0ULL;
    auto staged_of = [&](u64 lw) -> bool { return !A.force_inplace && ((lw >> kListShift) << 4) <= (u64)A.sm_stage_bytes; };
    auto prefetch = [&](int j, int b) {
        const u64 lw = __shfl_sync(FULL, mylw, j);
        if (staged_of(lw) && lane == 0) {
            const u32 bytes = (u32)((lw >> kListShift) << 4);
            mbar_expect_tx(&S.bar[b], bytes);
            bulk_g2s(S.stage[b], A.cur + ((lw & kListOffMask) << 4), bytes, &S.bar[b]);
        }
    };
    prefetch(0, 0);
#pragma unroll 1
    for (int j = 0; j < cnt; ++j) {
        const int sb = j & 1;
        const u64 lw = __shfl_sync(FULL, mylw, j);
        const u64 pid = first + (u64)j;
        if (j + 1 < cnt) prefetch(j + 1, sb ^ 1);
        const bool staged = staged_of(lw);
        const unsigned char* eb = A.cur + ((lw & kListOffMask) << 4);
        if (__builtin_expect(staged, 1)) {
            mbar_wait(&S.bar[sb], (phase >> sb) & 1u);
            phase ^= 1u << sb;
            eb = S.stage[sb];
        }
        const uint4* e4 = (const uint4*)eb;
        const Hdr H = decode_hdr(e4[0], e4[1], e4[2]);
        const int ns = H.ns, nv = H.nv, nu = H.nu, istar = H.istar;
        const i64* flux = (const i64*)(eb + kHdr);
        const u64* vis = (const u64*)(flux + ns);
        const i64* ef = (const i64*)(vis + nv);
        const u16* arc = (const u16*)(ef + nu);
        const u16* efmet = arc + ns;
        const i64 E = H.E;
        const bool fwd = E > 0;
        const u64 absE = abs64(E);
        u32* sbits = S.sbits; u16* upos = S.upos;
        // the graph data of i* is requested before the tables are built: slices of I / O, the first 32 OR-alternative
        // records and the first 32 arcs of the primary search
        const int4 nd = __ldg(&A.g.node[istar]);
        const int in0 = nd.x, nI = nd.y, out0 = nd.z, nO = nd.w;
        const int2* alist = fwd ? A.g.out_e + out0 : A.g.in_e + in0;
        const uint4* altl = fwd ? A.g.out_alt + 2 * (size_t)out0 : A.g.in_alt + 2 * (size_t)in0;
        const int alen = fwd ? nO : nI;
        const int2* plist = fwd ? A.g.in_e + in0 : A.g.out_e + out0;
        const int plen = fwd ? nI : nO;
        uint4 r0n = make_uint4(0, 0, 0, 0), r1n = r0n;
        if (lane < alen) { r0n = __ldg(&altl[2 * lane]); r1n = __ldg(&altl[2 * lane + 1]); }
        int pan = lane < plen ? __ldg(&plist[lane]).x : -1;
        // ---- support bitset, EF index table
#pragma unroll 1
        for (int t = lane; t < ns; t += 32) { const u32 a = arc[t]; atomicOr(&sbits[a >> 5], 1u << (a & 31)); }
#pragma unroll 1
        for (int t = lane; t < nu; t += 32) upos[efmet[t]] = (u16)(t + 1);
        __syncwarp();
        auto ef_of = [&](int met) -> i64 { const u32 u = upos[met]; return u ? ef[u - 1] : 0; };
        int n_adm = 0;
        if (nv >= A.V) {
            if (lane == 0) { atomicAdd(&ctl->st[ST_VISITED], 1ULL); if (MODES && A.cand_end) A.cand_end[H.cand] = END_VISITED | ((u64)A.level << 8); }
        } else {
            // primary on the side the flux arrives from: lowest arc of that side in the support (G13)
            int prim = -1;
#pragma unroll 1
            for (int base = 0; base < plen && prim < 0; base += 32) {
                const int pa = pan;
                const int qn = base + 32 + lane;
                pan = qn < plen ? __ldg(&plist[qn]).x : -1;
                const u32 bal = __ballot_sync(FULL, pa >= 0 && sbit(sbits, pa));
                if (bal) prim = __shfl_sync(FULL, pa, __ffs(bal) - 1);
            }
            if (lane == 0) A.pprim[pid] = (u32)prim;
            const bool fastP = fast_graph && H.big < kSmall;
            // visited record of i* without the chosen arc (PI = primary / chosen arc, PO = chosen arc / primary)
            const u64 vbase = vis_pack((u32)istar, fwd ? (u32)prim : 0u, fwd ? 0u : (u32)prim, 0u);
            const int ashift = fwd ? 0 : 16;
            auto admissible = [&](u32 a, u32 tw, bool insup) -> bool {   // readings G14, G15 and the reaction mask of 8(f)-2
                return !(tw != 0xffffu && sbit(sbits, (int)tw)) && (insup || ns < A.D) && (!MODES || !A.amask || ((__ldg(&A.amask[a >> 5]) >> (a & 31)) & 1u));
            };
            // 8(f)-1 sampling: count the admissible alternatives, then take exactly one of them
            int pick_idx = -1, seen = 0;
            if (MODES && A.sample) {
                int tot = 0;
#pragma unroll 1
                for (int base = 0; base < alen; base += 32) {
                    const int q = base + lane;
                    bool ad = false;
                    if (q < alen) { const uint4 r = __ldg(&altl[2 * q]); const u32 a = r.x & 0xffffu; ad = admissible(a, r.y & 0xffffu, sbit(sbits, (int)a)); }
                    tot += __popc(__ballot_sync(FULL, ad));
                }
                if (tot > 0) pick_idx = (int)(sample_pick(A.sample_seed, H.cand, (u32)istar) % (u64)tot);
            }
#pragma unroll 1
            for (int base = 0; base < alen; base += 32) {
                const int q = base + lane;
                int a = -1, c = 1;
                bool adm = false, insup = false, generic = false;
                const uint4 r0 = r0n, r1 = r1n;   // requested one round ahead
                if (q + 32 < alen) { r0n = __ldg(&altl[2 * (q + 32)]); r1n = __ldg(&altl[2 * (q + 32) + 1]); }
                if (q < alen) {   // one 32-byte record per OR-alternative: arc, c, twin and the column of the arc
                    a = (int)(r0.x & 0xffffu); c = (int)(r0.x >> 16);
                    const u32 tw = r0.y & 0xffffu;
                    generic = (r0.y >> 24) & 1u;
                    if (__builtin_expect(generic, 0)) c = __ldg(&alist[q]).y;   // the coefficient may not fit the record
                    insup = sbit(sbits, a);
                    adm = admissible((u32)a, tw, insup);
                }
                u32 adm_m = __ballot_sync(FULL, adm);
                if (adm_m == 0) continue;
                n_adm += __popc(adm_m);
                if (MODES && A.sample) {   // only the sampled alternative goes on
                    const int here = __popc(adm_m);
                    const int sel = (pick_idx >= seen && pick_idx < seen + here) ? (int)__fns(adm_m, 0, pick_idx - seen + 1) : -1;
                    seen += here;
                    adm = adm && lane == sel;
                    adm_m = sel >= 0 ? 1u << sel : 0u;
                    if (adm_m == 0) continue;
                }
                // ---- lane-parallel evaluation: new arc, small integers => no overflow, no common factor
                const bool fast = adm && !insup && fastP && !generic;
                const u32 fast_m = __ballot_sync(FULL, fast);
                if (fast_m) {
                    u64 key = 0;
                    int nu2 = nu;
                    if (fast) {
                        u64 k, d;
                        scale_of(absE, (u32)c, k, d);
                        const int ncol = (int)((r0.y >> 16) & 0xffu);
                        const u32 cw[6] = {r0.z, r0.w, r1.x, r1.y, r1.z, r1.w};
#pragma unroll
                        for (int e = 0; e < 6; ++e) {
                            if (e < ncol) {
                                const u32 u = upos[cw[e] & 0xffffu];
                                if (u == 0) ++nu2;   // balanced in the parent: d s != 0 unbalances it
                                else {
                                    const i64 x = (i64)k * ef[u - 1] + (i64)d * (i64)(short)(cw[e] >> 16);   // |.| < 2^60 + 2^60
                                    nu2 -= (int)(x == 0);
                                }
                            }
                        }
                        const u64 hs2 = k * H.hs + arc_mult(A.g, (u32)a) * d;
                        const u64 hv2 = H.hv + vis_term(vbase | ((u64)(u32)a << ashift));
                        key = nu2 == 0 ? kKeyDone : beam_key((u32)nu2, mix64(hs2 + hv2));
                    }
                    acc.children += (u32)__popc(fast_m);
                    acc.done += (u32)__popc(__ballot_sync(FULL, fast && nu2 == 0));
                    const u64 slot = ko.reserve(A, lv, lane, fast);
                    if (fast && slot != kNoSlot) {
                        __stcs(&A.keys[slot], key);
                        __stcs(&A.tags[slot], (pid << kTagParentShift) | ((u64)TK_FAST << 32) | ((u64)(u32)q << 16) | (u64)(u32)nu2);
                    }
                }
                // ---- one child at a time: general evaluation (arc of the support, large integers, wide column)
                u32 slow_m = adm_m & ~fast_m;
#pragma unroll 1
                while (slow_m) {
                    const int l = __ffs(slow_m) - 1;
                    slow_m &= slow_m - 1;
                    const int ca = __shfl_sync(FULL, a, l);
                    const int cc = __shfl_sync(FULL, c, l);
                    const u64 newrec = vbase | ((u64)(u32)ca << ashift);
                    const int qa0 = __ldg(&A.g.col_ptr[ca]), qa1 = __ldg(&A.g.col_ptr[ca + 1]);
                    u64 ck, cd;
                    scale_of(absE, (u32)cc, ck, cd);
                    const bool cin = sbit(sbits, ca);
                    int cia = -1;
                    if (cin) {   // position of the arc in the sorted support
#pragma unroll 1
                        for (int b2 = 0; b2 < ns && cia < 0; b2 += 32) {
                            const int t = b2 + lane;
                            const u32 hit = __ballot_sync(FULL, t < ns && arc[t] == ca);
                            if (hit) cia = b2 + __ffs(hit) - 1;
                        }
                    }
                    // scaled fluxes F_t = k f_t, F_a = k f_a + d: overflow first, then the extra fluxes (order of O6).
                    // big >= every flux and |EF| of the parent: products below the guard with it need no exact sweep.
                    const bool bigk = ck > 1 && umul_gt_guard(ck, H.big);
                    bool ovf = false;
                    u64 cT = cd;
                    const u64 fa = cin ? (u64)flux[cia] : 0ULL;
                    if (cin) {
                        const u64 lo = ck * fa, hi = __umul64hi(ck, fa);
                        cT = lo + cd;
                        const u64 hi2 = hi + (cT < lo);
                        ovf = hi2 != 0 || cT > EFM_GUARD;
                    }
                    if (__builtin_expect(bigk, 0)) {   // exact: the largest flux among t != ia (a new arc carries d <= |E| <= 2^62)
                        u64 mx = 0;
#pragma unroll 1
                        for (int t = lane; t < ns; t += 32) if (t != cia) mx = max(mx, (u64)flux[t]);
                        mx = g_max(FULL, mx);
                        ovf = ovf || umul_gt_guard(ck, mx);
                    }
                    int cnu = nu;
                    if (!ovf) {
                        bool ovf2 = false;
                        if (__builtin_expect(bigk, 0)) {   // exact sweep over the unbalanced metabolites outside col(a)
#pragma unroll 1
                            for (int t = lane; t < nu; t += 32) {
                                const int i = efmet[t];
                                bool in_a = false;
#pragma unroll 1
                                for (int r = qa0; r < qa1; ++r) in_a = in_a || col_met(__ldg(&A.g.col[r])) == i;
                                if (!in_a) ovf2 = ovf2 || abs_gt_guard(mul_s((i64)ck, ef[t]));
                            }
                        }
                        int delta = 0;
#pragma unroll 1
                        for (int qq = qa0 + lane; qq < qa1; qq += 32) {
                            const int2 e = __ldg(&A.g.col[qq]);
                            const i64 efp = ef_of(col_met(e));
                            const S128 x = add_s(mul_s((i64)ck, efp), mul_s((i64)cd, (i64)e.y));
                            ovf2 = ovf2 || abs_gt_guard(x);
                            delta += (int)((x.lo | (u64)x.hi) != 0) - (int)(efp != 0);
                        }
                        ovf = __any_sync(FULL, ovf2);
                        cnu = nu + __reduce_add_sync(FULL, delta);
                    }
                    if (__builtin_expect(ovf, 0)) {
                        if (lane == 0) { atomicAdd(&ctl->st[ST_OVERFLOW], 1ULL); if (MODES && A.cand_end) A.cand_end[H.cand] = END_OVERFLOW | ((u64)A.level << 8); }
                        continue;
                    }
                    // gcd normalisation (reading G10).  A new arc cannot introduce a common factor: gcd_t(k f_t) = k and
                    // gcd(k, d) = 1.  An arc of the support: g = gcd(T, k f_t for t != a).
                    u64 cg = 1;
                    if (cin && H.ones - (int)(fa == 1) <= 0) cg = common_divisor<32>(FULL, lane, flux, ns, cia, ck, cT);   // a unit flux elsewhere: g = 1
                    u64 chs;
                    if (cg == 1) chs = ck * H.hs + arc_mult(A.g, (u32)ca) * (cT - ck * fa);
                    else {
                        chs = 0;
#pragma unroll 1
                        for (int t = lane; t < ns; t += 32) {
                            const u64 F = t == cia ? cT : ck * (u64)flux[t];
                            chs += arc_mult(A.g, (u32)arc[t]) * udiv64(F, cg);
                        }
                        chs = g_sum<32>(FULL, chs);
                    }
                    const u64 chv = H.hv + vis_term(newrec);
                    const bool cdone = cnu == 0;
                    acc.children++; acc.general++; acc.done += cdone;
                    const u64 slot = ko.reserve(A, lv, lane, lane == 0);
                    const u64 ti = to.reserve(A, lv, lane, 1);
                    if (lane == 0 && slot != kNoSlot) {
                        if (ti == kNoSlot) __stcs(&A.keys[slot], kKeySentinel);
                        else {
                            __stcs(&A.keys[slot], cdone ? kKeyDone : beam_key((u32)cnu, mix64(chs + chv)));
                            __stcs(&A.tags[slot], (pid << kTagParentShift) | ((u64)TK_TASK << 32) | ti);
                            write_task(A, ti, ca, cia, cnu, (u32)TF_FIRST | (cin ? (u32)TF_INSUPP : 0u), ck, cd, cT, cg, chs, chv, newrec);
                        }
                    }
                }
            }
            if (n_adm == 0 && lane == 0) {   // no admissible alternative
                atomicAdd(&ctl->st[ST_DEAD_END], 1ULL);
                if (MODES && A.cand_end) A.cand_end[H.cand] = END_DEAD | ((u64)A.level << 8);
            }
        }
        // ---- restore the shared tables to zero for the next parent
        __syncwarp();
#pragma unroll 1
        for (int t = lane; t < nu; t += 32) upos[efmet[t]] = 0;
#pragma unroll 1
        for (int i = lane; i < (A.g.W32 + 3) / 4; i += 32) ((uint4*)sbits)[i] = make_uint4(0, 0, 0, 0);
        __syncwarp();
    }
}

template <bool MODES>
__global__ void __launch_bounds__(32, EFM_MIN_BLOCKS) k_expand(const __grid_constant__ ExpandArgs A) {
    extern __shared__ uint4 smem4[];
    const int lane = threadIdx.x;
    unsigned char* gs = (unsigned char*)smem4;
    WarpSmem S;
    S.stage[0] = gs; S.stage[1] = gs + A.sm_stage_bytes;
    S.sbits = (u32*)(gs + A.sm_sbits);
    S.upos = (u16*)(gs + A.sm_upos);
    S.bar = (u64*)(gs + A.sm_misc);
    Ctl* ctl = A.ctl;
    LevelCtl* lv = &ctl->lv[A.par];
    const u64 nF = lv->nF, nR = lv->nR;
    const u64 nRi = (nR + kRevisitPerItem - 1) / kRevisitPerItem, nFi = (nF + kParentsPerItem - 1) / kParentsPerItem;
    const u64 total = nRi + nFi;
    if (blockIdx.x == 0 && lane == 0 && nF) atomicAdd(&ctl->st[ST_FIRST], nF);
    if ((u64)blockIdx.x >= total) return;
    u32 phase = 0;
    if (nFi) {
#pragma unroll 1
        for (int i = lane; i < (A.g.W32 + 3) / 4; i += 32) ((uint4*)S.sbits)[i] = make_uint4(0, 0, 0, 0);
#pragma unroll 1
        for (int i = lane; i < (A.g.M + 8) / 8; i += 32) ((uint4*)S.upos)[i] = make_uint4(0, 0, 0, 0);
        if (lane == 0) { mbar_init(&S.bar[0], 1); mbar_init(&S.bar[1], 1); }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        __syncwarp();
    }
    KeyOut ko; ko.base = 0; ko.left = 0;
    TaskOut to; to.base = 0; to.left = 0;
    WarpAcc acc; acc.children = 0; acc.done = 0; acc.general = 0;
    // dynamic distribution: revisit items first (they are the longer ones), then first-visit items
#pragma unroll 1
    for (;;) {
        u64 w = 0;
        if (lane == 0) w = atomicAdd(&lv->work, 1ULL);
        w = __shfl_sync(FULL, w, 0);
        if (w >= total) break;
        if (w < nRi) expand_revisits<MODES>(A, lv, w * kRevisitPerItem, nR, lane, ko, to, acc);
        else expand_first_visits<MODES>(A, lv, (w - nRi) * kParentsPerItem, nF, lane, S, phase, ko, to, acc);
    }
    ko.finish(A, lane);
    if (lane == 0) {
        if (acc.children) { atomicAdd(&ctl->st[ST_CHILDREN], (u64)acc.children); atomicAdd(&ctl->st[ST_ALGO_BYTES], 8ULL * acc.children); }
        if (acc.done) atomicAdd(&lv->n_done, (u64)acc.done);
        if (acc.children - acc.done) atomicAdd(&lv->n_keys, (u64)(acc.children - acc.done));
        if (acc.general) atomicAdd(&ctl->st[ST_GENERAL], (u64)acc.general);
    }
}

// ------------------------------------------------------------------ survivors of the beam -> list of slots
// Balanced children (kKeyDone) and active children with key < X (all of them when the beam does not bind).  A block
// appends the survivors of a tile with ONE atomic per counter; the order of the list does not matter.  Besides listing
// the survivors, the kernel sizes every child (tag / task + parent header) and reserves its place: an entry index and
// 16-byte units in the next frontier, or a candidate slot.  k_materialise then needs no coordination at all.
constexpr int kCompactItems = 4;   // keys per thread: a block handles the survivors of 1024 keys with one atomic per counter
__global__ void __launch_bounds__(256) k_compact(const __grid_constant__ ExpandArgs A) {
    __shared__ u32 s_w[4][8];      // per warp totals: survivors, frontier children, frontier units, candidates
    __shared__ u64 s_base[4];
    Ctl* ctl = A.ctl;
    LevelCtl* lv = &ctl->lv[A.par];
    LevelCtl* nx = &ctl->lv[A.par ^ 1];
    const u64 n = min(lv->n_slots, A.max_keys);
    const bool notrunc = A.cap == 0 || lv->n_keys <= A.cap;
    const u64 X = ctl->X;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    constexpr u64 kTile = 256 * kCompactItems;
    for (u64 tile = (u64)blockIdx.x * kTile; tile < n; tile += (u64)gridDim.x * kTile) {   // block-uniform trip count
        // item j of a thread is key tile + j * 256 + threadIdx.x (coalesced loads)
        u32 takes = 0, my_front = 0, my_units = 0, my_cand = 0, my_bytes = 0;
        u32 units[kCompactItems];
        u64 poff[kCompactItems];
        // the four items of a thread advance together through the chain key -> tag -> (task word) -> parent offset ->
        // parent header, so that a thread waits for four memory latencies, not sixteen
#pragma unroll
        for (int j = 0; j < kCompactItems; ++j) {
            const u64 i = tile + (u64)j * 256 + threadIdx.x;
            const u64 key = i < n ? __ldcs(&A.keys[i]) : kKeySentinel;
            if (key == kKeyDone || (key != kKeySentinel && (notrunc || key < X))) takes |= 1u << j;
        }
        u64 tag[kCompactItems];
        u32 qz[kCompactItems], w0[kCompactItems];
#pragma unroll
        for (int j = 0; j < kCompactItems; ++j) tag[j] = ((takes >> j) & 1u) ? __ldcs(&A.tags[tile + (u64)j * 256 + threadIdx.x]) : 0ULL;
#pragma unroll
        for (int j = 0; j < kCompactItems; ++j) {
            qz[j] = 0; poff[j] = 0;
            if ((takes >> j) & 1u) {
                if (((tag[j] >> 32) & 3ULL) == TK_TASK) qz[j] = __ldg(&A.tasks[4 * (u64)(u32)tag[j]].z);
                else qz[j] = ((u32)tag[j] & 0xffffu) | ((u32)TF_FIRST << 16);
                poff[j] = __ldg(&A.plist[tag[j] >> kTagParentShift]) & kListOffMask;
            }
        }
#pragma unroll
        for (int j = 0; j < kCompactItems; ++j) w0[j] = ((takes >> j) & 1u) ? __ldg((const u32*)(A.cur + (poff[j] << 4))) : 0u;
#pragma unroll
        for (int j = 0; j < kCompactItems; ++j) {
            units[j] = 0;
            if ((takes >> j) & 1u) {
                const u32 ns = w0[j] & 0xffffu, nv = w0[j] >> 16, cnu = qz[j] & 0xffffu, fl = qz[j] >> 16;
                const u32 n2 = ns + ((fl & TF_INSUPP) ? 0u : 1u), nv2 = nv + ((fl & TF_FIRST) ? 1u : 0u);
                my_bytes += algo_entry_bytes(n2, nv2);
                if (cnu == 0) my_cand++;
                else { units[j] = entry_bytes(n2, nv2, cnu) >> 4; my_front++; my_units += units[j]; }
            }
        }
        // exclusive prefix over the threads of the block for the four counters (warp scan + warp totals)
        u32 v[4] = {(u32)__popc(takes), my_front, my_units, my_cand};
        u32 ex[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            u32 x = v[c];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const u32 y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
            ex[c] = x - v[c];
            if (lane == 31) s_w[c][wib] = x;
        }
        my_bytes = __reduce_add_sync(0xffffffffu, my_bytes);
        __syncthreads();
        if (threadIdx.x < 4) {
            const int c = threadIdx.x;
            u32 tot = 0;
            for (int w = 0; w < 8; ++w) { const u32 t = s_w[c][w]; s_w[c][w] = tot; tot += t; }
            if (c == 0) s_base[0] = tot ? atomicAdd(&lv->n_surv, (u64)tot) : 0ULL;
            if (c == 1) s_base[1] = tot;                      // frontier children of the block (combined with c == 2 below)
            if (c == 2) s_base[2] = tot;
            if (c == 3) s_base[3] = tot ? atomicAdd(&ctl->n_cand, (u64)tot) : 0ULL;
        }
        if (lane == 0 && my_bytes) atomicAdd(&ctl->st[ST_ALGO_BYTES], (u64)my_bytes);
        __syncthreads();
        if (threadIdx.x == 0) {
            const u64 nf = s_base[1], nu = s_base[2];
            const u64 old = nf ? atomicAdd(&nx->alloc, (nf << kAllocShift) | nu) : 0ULL;
            s_base[1] = old >> kAllocShift; s_base[2] = old & kAllocUnitMask;
        }
        __syncthreads();
        u64 pos = s_base[0] + s_w[0][wib] + ex[0];
        u64 fidx = s_base[1] + s_w[1][wib] + ex[1], foff = s_base[2] + s_w[2][wib] + ex[2];
        u64 cidx = s_base[3] + s_w[3][wib] + ex[3];
#pragma unroll
        for (int j = 0; j < kCompactItems; ++j) {
            if ((takes >> j) & 1u) {
                const u64 i = tile + (u64)j * 256 + threadIdx.x;
                u64 dst;
                if (units[j] == 0) {   // candidate
                    if (cidx >= A.max_cand) { atomicOr(&ctl->error, (u32)ERR_CAND); dst = ~0ULL; }
                    else dst = (1ULL << 63) | cidx;
                    ++cidx;
                } else {
                    if (fidx >= A.max_frontier || foff + units[j] > A.frontier_units) { atomicOr(&ctl->error, (u32)ERR_FRONTIER); dst = ~0ULL; }
                    else { dst = foff; A.nxt_off[fidx] = foff; }
                    ++fidx; foff += units[j];
                }
                if (pos < A.max_surv) { A.surv[pos] = make_ulonglong2(i, poff[j]); A.surv_dst[pos] = dst; }
                else atomicOr(&ctl->error, dst == ~0ULL ? 0u : (u32)ERR_FRONTIER);
                ++pos;
            }
        }
        __syncthreads();   // the shared arrays are reused by the next tile
    }
}

// ------------------------------------------------------------------ materialise: G lanes per surviving child
// Reads the tag (and the task of a child of the general routine; a lane-parallel child is re-derived from the parent's
// header, its OR-alternative record and the primary arc k_expand stored), reads the parent entry straight from HBM / L2
// (every element is needed once) and writes the child: a candidate slot if it is balanced, otherwise a packed entry of the
// next frontier, with i*, E and the visited record of i* found for its own expansion.  G = 8 (four children per warp)
// suits entries of a few dozen arcs: the per-child control flow and address arithmetic is shared by four children.
#ifndef EFM_MAT_BLOCKS
#define EFM_MAT_BLOCKS 4
#endif
#ifndef EFM_MAT_GROUP
#define EFM_MAT_GROUP 8    // lanes per child (measured k_compact + k_materialise per step: 32 -> 22.9 ms, 16 -> 20.3, 8 -> 19.0, 4 -> 21.6)
#endif
constexpr int kMatThreads = 256;
template <int G>
__global__ void __launch_bounds__(kMatThreads, EFM_MAT_BLOCKS) k_materialise(const __grid_constant__ ExpandArgs A) {
    constexpr int kMatWarps = kMatThreads / G;   // children per block
    const u32 gbits = G == 32 ? 0xffffffffu : ((1u << (G & 31)) - 1u);
    const u32 gmask = gbits << (threadIdx.x & 31 & ~(G - 1));   // lanes of this child
    const int gshift = threadIdx.x & 31 & ~(G - 1);
    auto gballot = [&](bool pred) -> u32 { return (__ballot_sync(gmask, pred) >> gshift) & gbits; };
    auto gany = [&](bool pred) -> bool { return __any_sync(gmask, pred) != 0; };
    const int lane = threadIdx.x & (G - 1), wib = threadIdx.x / G;   // lane within the child's group, group within the block
    const u32 lt = (1u << lane) - 1u;
    Ctl* ctl = A.ctl;
    LevelCtl* lv = &ctl->lv[A.par];
    const u64 n_surv = min(lv->n_surv, A.max_surv);
    if (blockIdx.x == 0 && threadIdx.x == 0 && A.level + 1 < A.max_levels) {   // the record of this level for the host
        LevelStats* rec = &A.lvl[A.level + 1];
        rec->parents = lv->nF + lv->nR; rec->active_children = lv->n_keys; rec->done_children = lv->n_done;
        rec->kept = ctl->lv[A.par ^ 1].alloc >> kAllocShift; rec->surv = lv->n_surv;
    }
    // k_compact reserved the place of every child: the groups work on their own, no block-wide step is left
    for (u64 sidx = (u64)blockIdx.x * kMatWarps + wib; sidx < n_surv; sidx += (u64)gridDim.x * kMatWarps) {
    // ---- the tag, the reserved place, the header of the parent
    const ulonglong2 sv = __ldcs(&A.surv[sidx]);
    const u64 dstrec = __ldcs(&A.surv_dst[sidx]);
    const u64 slot = sv.x;
    const unsigned char* pe = A.cur + (sv.y << 4);
    const u64 tag = __ldcs(&A.tags[slot]);
    const Hdr P = decode_hdr(__ldg((const uint4*)pe), __ldg((const uint4*)pe + 1), __ldg((const uint4*)pe + 2));
    int ca, cia, cnu;
    u32 flags;
    u64 ck, cd, cT, cg, chs, chv, newrec;
    if (((tag >> 32) & 3ULL) == TK_TASK) {
        const uint4* tk = A.tasks + 4 * (u64)(u32)tag;
        const uint4 q0 = __ldcs(tk), q1 = __ldcs(tk + 1), q2 = __ldcs(tk + 2), q3 = __ldcs(tk + 3);
        ca = (int)(q0.y & 0xffffu);
        cia = (q0.y >> 16) == 0xffffu ? -1 : (int)(q0.y >> 16);
        cnu = (int)(q0.z & 0xffffu);
        flags = q0.z >> 16;
        ck = q0.w;
        cd = (u64)q1.x | ((u64)q1.y << 32); cT = (u64)q1.z | ((u64)q1.w << 32);
        cg = (u64)q2.x | ((u64)q2.y << 32); chs = (u64)q2.z | ((u64)q2.w << 32);
        chv = (u64)q3.x | ((u64)q3.y << 32); newrec = (u64)q3.z | ((u64)q3.w << 32);
    } else {
        // lane-parallel child of a first visit: new arc a = alternative q of i*, Eq 3: k = c / gcd(|E|, c),
        // d = |E| / gcd, no common divisor
        const u32 q = ((u32)tag >> 16) & 0xffffu;
        cnu = (int)((u32)tag & 0xffffu);
        const bool fwd = P.E > 0;
        const int4 nd = __ldg(&A.g.node[P.istar]);
        const uint4 r0 = __ldg(fwd ? &A.g.out_alt[2 * (size_t)(nd.z + (int)q)] : &A.g.in_alt[2 * (size_t)(nd.x + (int)q)]);
        ca = (int)(r0.x & 0xffffu);
        scale_of(abs64(P.E), r0.x >> 16, ck, cd);
        const u32 prim = __ldg(&A.pprim[tag >> kTagParentShift]);
        newrec = vis_pack((u32)P.istar, fwd ? prim : (u32)ca, fwd ? (u32)ca : prim, 0u);
        cT = cd; cg = 1; cia = -1; flags = TF_FIRST;
        chs = ck * P.hs + arc_mult(A.g, (u32)ca) * cd;
        chv = P.hv + vis_term(newrec);
    }
    const bool cin = (flags & TF_INSUPP) != 0, firstv = (flags & TF_FIRST) != 0;
    const u64 sd = (flags & TF_NEG) ? (u64)0 - cd : cd;
    // ---- the parent
    const int ns = P.ns, nv = P.nv, nu = P.nu;
    const i64* flux = (const i64*)(pe + kHdr);
    const u64* vis = (const u64*)(flux + ns);
    const i64* ef = (const i64*)(vis + nv);
    const u16* arc = (const u16*)(ef + nu);
    const u16* efmet = arc + ns;
    const bool to_cand = cnu == 0;
    const int n2 = ns + (cin ? 0 : 1);
    const int nv2 = to_cand ? 0 : nv + (firstv ? 1 : 0);
    const int nu2 = to_cand ? 0 : cnu;
    // ---- every element of the parent this lane will need, requested before anything waits: the loads overlap each
    // other (entries beyond 2 G arcs / records are loaded where they are used)
    u32 pa0 = 0xffffffffu, pa1 = 0xffffffffu, pm0 = 0xffffffffu;
    i64 pf0 = 0, pf1 = 0, pe0 = 0;
    u64 pv0 = 0, pv1 = 0;
    int pcol0 = 0, pcol1 = 0;
    {
        if (lane < ns) { pa0 = arc[lane]; pf0 = flux[lane]; }
        if (lane + G < ns) { pa1 = arc[lane + G]; pf1 = flux[lane + G]; }
        if (!to_cand) {
            if (lane < nv) pv0 = vis[lane];
            if (lane + G < nv) pv1 = vis[lane + G];
            if (lane < nu) { pm0 = efmet[lane]; pe0 = ef[lane]; }
            pcol0 = __ldg(&A.g.col_ptr[ca]); pcol1 = __ldg(&A.g.col_ptr[ca + 1]);
        }
    }
    const bool ok = dstrec != ~0ULL;   // ~0: a capacity error was flagged by k_compact
    unsigned char* dst = (dstrec >> 63) ? A.cand + (dstrec & ~(1ULL << 63)) * A.cand_stride : A.nxt + (dstrec << 4);
    if (ok) {
    // ---- write
    int ins = 0;   // a new arc goes where the ascending order puts it
    if (!cin)
        for (int b2 = 0; b2 < ns; b2 += G) {
            const int t = b2 + lane;
            const u32 at = b2 == 0 ? pa0 : (b2 == G ? pa1 : (t < ns ? (u32)arc[t] : 0xffffffffu));
            ins += __popc(gballot(at < (u32)ca));
        }
    i64* flux2 = (i64*)(dst + kHdr);
    u64* vis2 = (u64*)(flux2 + n2);
    i64* ef2 = (i64*)(vis2 + nv2);
    u16* arc2 = (u16*)(ef2 + nu2);
    u16* efmet2 = arc2 + n2;
    u64 mx = cin ? 0ULL : cT;   // a new arc never comes with a common divisor
    int ones = 0;               // fluxes equal to 1 (the expansion of the child skips its gcd sweep when another arc carries 1)
    for (int t = lane; t < ns; t += G) {
        const u64 ft = t < G ? (u64)pf0 : (t < 2 * G ? (u64)pf1 : (u64)flux[t]);
        u64 F = t == cia ? cT : ck * ft;
        if (cg > 1) F = udiv64(F, cg);
        const int pos = t + ((!cin && t >= ins) ? 1 : 0);
        flux2[pos] = (i64)F;
        arc2[pos] = (u16)(t < G ? pa0 : (t < 2 * G ? pa1 : (u32)arc[t]));
        mx = max(mx, F);
        ones += (int)(F == 1);
    }
    if (!cin && lane == 0) { flux2[ins] = (i64)cT; arc2[ins] = (u16)ca; ones += (int)(cT == 1); }
    ones = __reduce_add_sync(gmask, ones);
    u32 best = 0xffffffffu;   // lowest unbalanced metabolite of the child (reading G12): met << 16 | position in its list
    i64 bestE = 0;
    int vk2 = -1;
    if (!to_cand) {
        // EF list of the child: EF' = (k EF + sign d s_.a) / g over the parent's list, then the metabolites of col(a)
        // that were balanced in the parent.  k_expand established that nothing exceeds 2^62, so the wrapping 64-bit
        // arithmetic is exact.
        const int qa0 = pcol0, qa1 = pcol1;
        int wbase = 0;
        u32 seen = 0;   // bit q - qa0: metabolite of col(a)[q] is in the parent's list (columns longer than 32: see below)
        const int nc = qa1 - qa0;
        // the column of the arc in registers (up to six entries, the usual case): an element of the parent's list meets it
        // with compares only, and which column entries were met is one group-wide OR at the end
        int cm[6]; i64 cs[6];
#pragma unroll
        for (int q = 0; q < 6; ++q) {
            cm[q] = -2; cs[q] = 0;
            if (q < nc && nc <= 6) { const int2 e = __ldg(&A.g.col[qa0 + q]); cm[q] = col_met(e); cs[q] = (i64)e.y; }
        }
        for (int t0 = 0; t0 < nu; t0 += G) {
            const int t = t0 + lane;
            const bool valid = t < nu;
            i64 x = 0;
            int met = -1;
            if (nc <= 6) {
                i64 s = 0;
                if (valid) met = t0 == 0 ? (int)pm0 : (int)efmet[t];
#pragma unroll
                for (int q = 0; q < 6; ++q) if (met == cm[q]) { s = cs[q]; seen |= 1u << q; }
                if (valid) {
                    x = (i64)(ck * (u64)(t0 == 0 ? pe0 : ef[t]) + sd * (u64)s);
                    if (cg > 1) x = sdiv64(x, (i64)cg);
                }
            } else {
                if (valid) {
                    met = t0 == 0 ? (int)pm0 : (int)efmet[t];
                    i64 s = 0;
                    for (int qq = qa0; qq < qa1; ++qq) { const int2 e = __ldg(&A.g.col[qq]); if (col_met(e) == met) s = e.y; }
                    x = (i64)(ck * (u64)(t0 == 0 ? pe0 : ef[t]) + sd * (u64)s);
                    if (cg > 1) x = sdiv64(x, (i64)cg);
                }
                for (int qq = qa0; qq < qa1 && qq < qa0 + 32; ++qq)
                    if (gany(valid && col_met(__ldg(&A.g.col[qq])) == met)) seen |= 1u << (qq - qa0);
            }
            const u32 nz = gballot(valid && x != 0);
            if (valid && x != 0) {
                const int pos = wbase + __popc(nz & lt);
                ef2[pos] = x; efmet2[pos] = (u16)met;
                mx = max(mx, abs64(x));
                const u32 bk = ((u32)met << 16) | (u32)pos;
                if (bk < best) { best = bk; bestE = x; }
            }
            wbase += __popc(nz);
        }
        if (nc <= 6) seen = __reduce_or_sync(gmask, seen);   // the lanes noted their own matches
        for (int qq = qa0; qq < qa1; ++qq) {   // warp-uniform, a handful of entries
            const int2 e = __ldg(&A.g.col[qq]);
            const int emet = col_met(e);
            bool in_parent;
            if (qq < qa0 + 32) in_parent = (seen >> (qq - qa0)) & 1u;
            else {   // columns longer than 32 entries: scan the parent's list again
                bool f = false;
                for (int t = lane; t < nu; t += G) f = f || (int)efmet[t] == emet;
                in_parent = gany(f);
            }
            if (!in_parent) {
                i64 x = (i64)(sd * (u64)(i64)e.y);
                if (cg > 1) x = sdiv64(x, (i64)cg);
                if (lane == 0) {
                    ef2[wbase] = x; efmet2[wbase] = (u16)emet;
                    const u32 bk = ((u32)emet << 16) | (u32)wbase;
                    if (bk < best) { best = bk; bestE = x; }
                }
                mx = max(mx, abs64(x));
                ++wbase;
            }
        }
        // i* of the child and its E: the group's smallest (metabolite, position); the owner lane passes E on
        const u32 gbest = __reduce_min_sync(gmask, best);
        const u32 owner = gballot(best == gbest);
        bestE = __shfl_sync(gmask, bestE, (__ffs(owner) - 1) + gshift);
        best = gbest;
        // the visited record of the parent's i* is appended (first visit) or replaced (revisit); the record of the
        // child's own i*, if it has one, is noted for its expansion
        const u32 met_star = (u32)((newrec >> 32) & 0xffffu), met2 = best >> 16;
        for (int u = lane; u < nv; u += G) {
            const u64 r = u < G ? pv0 : (u < 2 * G ? pv1 : vis[u]);
            const u32 rm = (u32)((r >> 32) & 0xffffu);
            vis2[u] = (!firstv && rm == met_star) ? newrec : r;
            if (rm == met2) vk2 = u;
        }
        if (firstv && lane == 0) vis2[nv] = newrec;
        vk2 = __reduce_max_sync(gmask, vk2);
    }
    mx = g_max(gmask, mx);
    if (lane == 0) {
        uint4* h4 = (uint4*)dst;
        h4[0] = make_uint4((u32)n2 | ((u32)nv2 << 16), (u32)nu2 | ((u32)min(ones, 0xffff) << 16), (u32)chs, (u32)(chs >> 32));
        h4[1] = make_uint4((u32)chv, (u32)(chv >> 32), (u32)mx, (u32)(mx >> 32));
        h4[2] = make_uint4((u32)(u64)bestE, (u32)((u64)bestE >> 32), to_cand ? 0u : ((best >> 16) | ((u32)(vk2 + 1) << 16)),
                          to_cand ? A.level + 1u : P.cand);   // a balanced pathway keeps its step count, an active one its origin
        if (to_cand && A.cand_end) A.cand_end[P.cand] = END_DONE | ((u64)(A.level + 1u) << 8);
    }
    }   // ok
    }
}

// ------------------------------------------------------------------ roots (INIT kernel of the paper)
// One thread per seed set.  BUILD: every seed arc gets flux 1, the extra fluxes follow from Eq 2; the
// root is classified like any other entry (balanced -> candidate, otherwise its beam key).  Seed sets are tiny, so
// the quadratic duplicate scan below is cheaper than any scatter.  WRITE: the roots the beam keeps become level 0.
// The roots play the children of a level "-1": their key counters live in control set 1, they allocate in set 0.
template <bool WRITE>
__global__ void __launch_bounds__(128) k_roots(const RootArgs R) {
    const u64 r = (u64)blockIdx.x * blockDim.x + threadIdx.x;
    const DevGraph& g = R.g;
    Ctl* ctl = R.ctl;
    LevelCtl* lv = &ctl->lv[1];
    if (WRITE && r == 0) {
        LevelStats* rec = &R.lvl[0];
        rec->parents = 0; rec->active_children = lv->n_keys; rec->done_children = lv->n_done; rec->surv = 0;
    }
    if (r >= R.n_roots) return;
    unsigned char* e = R.stage + (R.stage_off[r] << 4);
    if (WRITE) {
        const u64 key = R.keys[r];
        const bool notrunc = R.cap == 0 || lv->n_keys <= R.cap;
        if (key == kKeySentinel || !(notrunc || key < ctl->X)) return;
        const u32 w0 = *(const u32*)e, nu = ((const u32*)e)[1] & 0xffffu;
        const u64 units = entry_bytes(w0 & 0xffffu, w0 >> 16, nu) >> 4;
        const u64 old = atomicAdd(&ctl->lv[0].alloc, (1ULL << kAllocShift) | units);
        const u64 slot = old >> kAllocShift, off = old & kAllocUnitMask;
        if (slot >= R.max_frontier || off + units > R.frontier_units) { atomicOr(&ctl->error, (u32)ERR_FRONTIER); return; }
        R.nxt_off[slot] = off;
        uint4* dst = (uint4*)(R.nxt + (off << 4));
        for (u64 c = 0; c < units; ++c) dst[c] = ((const uint4*)e)[c];
        return;
    }
    if (r == 0) lv->n_slots = R.n_roots;
    const int s0 = R.seed_ptr[r], ns = R.seed_ptr[r + 1] - s0;
    const int* arcs = R.seed_arc + s0;
    // Eq 2 with every flux = 1: EF_i = sum of s_ia over the seed arcs; (t, q) is the first occurrence of its metabolite
    auto ef_at = [&](int t, int q, i64& sum) -> bool {
        const int met = col_met(g.col[q]);
        sum = 0;
        for (int t2 = 0; t2 < ns; ++t2)
            for (int q2 = g.col_ptr[arcs[t2]]; q2 < g.col_ptr[arcs[t2] + 1]; ++q2)
                if (col_met(g.col[q2]) == met) {
                    if (t2 < t || (t2 == t && q2 < q)) return false;
                    sum += g.col[q2].y;
                }
        return sum != 0;
    };
    int nu = 0;
    for (int t = 0; t < ns; ++t)
        for (int q = g.col_ptr[arcs[t]]; q < g.col_ptr[arcs[t] + 1]; ++q) { i64 s; if (ef_at(t, q, s)) ++nu; }
    i64* flux = (i64*)(e + kHdr);
    i64* ef = flux + ns;          // n_vis = 0
    u16* arc = (u16*)(ef + nu);
    u16* efmet = arc + ns;
    u64 hs = 0, big = 1;
    for (int t = 0; t < ns; ++t) { flux[t] = 1; arc[t] = (u16)arcs[t]; hs += arc_term((u32)arcs[t], 1ULL); }
    int w = 0;
    u32 istar = 0xffffffffu;
    i64 E = 0;
    for (int t = 0; t < ns; ++t)
        for (int q = g.col_ptr[arcs[t]]; q < g.col_ptr[arcs[t] + 1]; ++q) {
            i64 s;
            if (ef_at(t, q, s)) {
                const u32 met = (u32)col_met(g.col[q]);
                ef[w] = s; efmet[w] = (u16)met; big = max(big, abs64(s)); ++w;
                if (met < istar) { istar = met; E = s; }   // lowest unbalanced metabolite (reading G12)
            }
        }
    ((u32*)e)[0] = (u32)ns; ((u32*)e)[1] = (u32)nu | ((u32)ns << 16);   // every flux is 1
    ((u64*)e)[1] = hs; ((u64*)e)[2] = 0; ((u64*)e)[3] = big;
    ((u64*)e)[4] = (u64)E; ((u32*)e)[10] = nu ? istar : 0u;   // no visited record yet: first visit
    ((u32*)e)[11] = nu ? (u32)r : 0u;   // origin of the pathway; a root that is balanced at once took 0 expansions
    if (nu == 0) {   // balanced at once (arbiter "Done")
        R.keys[r] = kKeySentinel;
        atomicAdd(&lv->n_done, 1ULL);
        if (R.cand_end) R.cand_end[r] = END_DONE;
        const u64 slot = atomicAdd(&ctl->n_cand, 1ULL);
        if (slot >= R.max_cand) { atomicOr(&ctl->error, (u32)ERR_CAND); return; }
        unsigned char* dst = R.cand + slot * R.cand_stride;
        const u32 bytes = entry_bytes((u32)ns, 0, 0);
        for (u32 c = 0; c < bytes / 16; ++c) ((uint4*)dst)[c] = ((const uint4*)e)[c];
    } else {
        R.keys[r] = beam_key((u32)nu, mix64(hs));
        atomicAdd(&lv->n_keys, 1ULL);
    }
}

// ------------------------------------------------------------------ host launchers
static size_t align16(size_t x) { return (x + 15) & ~(size_t)15; }

void expand_smem_layout(ExpandArgs& a) {
    // staging: the largest entry if it is small, otherwise 1.5 KB (larger entries are rare and read in place);
    // the smaller the per-warp footprint, the more of the graph stays in L1
    a.sm_stage_bytes = (u32)align16(a.max_entry < (u32)kStageBytes ? (a.max_entry < 64u ? 64u : a.max_entry) : (u32)kStageBytes);
    size_t off = 2 * (size_t)a.sm_stage_bytes;   // two staging buffers
    a.sm_sbits = (u32)off; off = align16(off + (size_t)a.g.W32 * 4 + 16);   // zeroed in 16-byte chunks
    a.sm_upos = (u32)off;  off = align16(off + (size_t)a.g.M * 2 + 16);
    a.sm_misc = (u32)off;  off = align16(off + 16);                          // two mbarriers
    a.sm_group = (u32)off;
}

// key slots the evaluation can leave unused: every warp of the grid strands at most the rest of one chunk
u64 expand_key_slack(int sm_count) { return (u64)sm_count * EFM_MIN_BLOCKS * kKeyChunk; }
u64 expand_task_slack(int sm_count) { return (u64)sm_count * EFM_MIN_BLOCKS * kTaskChunk; }

cudaError_t launch_order(const ExpandArgs& a, int sm_count, cudaStream_t s) {
    u64 blocks = (a.max_frontier + 1023) / 1024;
    if (blocks > (u64)sm_count * 4) blocks = (u64)sm_count * 4;
    if (blocks < 1) blocks = 1;
    k_order<<<(unsigned)blocks, 256, 0, s>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_expand(const ExpandArgs& a, int sm_count, cudaStream_t s) {
    const size_t smem = a.sm_group;
    if (smem > 227 * 1024) return cudaErrorInvalidValue;
    // per device: the attribute belongs to the function on the current device
    const bool modes = a.sample || a.amask || a.cand_end;
    cudaError_t e = modes ? cudaFuncSetAttribute(k_expand<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024)
                          : cudaFuncSetAttribute(k_expand<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    int per_sm = EFM_MIN_BLOCKS;
    while (per_sm > 1 && (size_t)per_sm * (smem + 1024) > 220 * 1024) --per_sm;
    if (modes) k_expand<true><<<(unsigned)(sm_count * per_sm), 32, smem, s>>>(a);
    else k_expand<false><<<(unsigned)(sm_count * per_sm), 32, smem, s>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_compact(const ExpandArgs& a, int sm_count, cudaStream_t s) {
    u64 blocks = (a.max_keys + 1023) / 1024;   // one tile of 256 x kCompactItems keys per block and round
    if (blocks > (u64)sm_count * 16) blocks = (u64)sm_count * 16;
    if (blocks < 1) blocks = 1;
    k_compact<<<(unsigned)blocks, 256, 0, s>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_materialise(const ExpandArgs& a, int sm_count, cudaStream_t s) {
    k_materialise<EFM_MAT_GROUP><<<(unsigned)(sm_count * 16), kMatThreads, 0, s>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_roots(bool write, const RootArgs& r, cudaStream_t s) {
    const unsigned blocks = (unsigned)((r.n_roots + 127) / 128);
    if (write) k_roots<true><<<blocks, 128, 0, s>>>(r);
    else k_roots<false><<<blocks, 128, 0, s>>>(r);
    return cudaGetLastError();
}

}  // namespace efm
