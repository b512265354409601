// Frontier expansion kernels: one warp owns one partial pathway at a time.
// The warp stages the packed parent entry in shared memory.  The entry carries its non-zero extra fluxes EF_i
// (Eq 2) as a short list, so the lowest unbalanced metabolite i* (reading G12) is a warp min and no
// scatter over the support is needed; children update the list incrementally, EF' = (k EF + sign d s_.a) / g.
//   first visit (PROC1/1', Eq 3): fans out over the OR-alternatives of i*, ONE LANE PER
//       ALTERNATIVE -- a child that adds a new arc to a pathway whose integers are far from the 2^62 guard needs only
//       lane-local work (scale k = c/gcd(|E|,c), its own column of S for the new unbalanced count, an incremental
//       state hash); anything else (arc already in the support, large integers) takes the warp-cooperative general
//       routine eval_child();
//   revisit (PROC2-4, Eq 4 / Eq 5): exactly one child, general routine.
// Children are classified where they are generated (balanced -> candidate; otherwise beam key).  Three modes:
//   COUNT  : count children, write their 8-byte beam keys and the balanced children (pass 1 of a level the beam may cut)
//   WRITE  : regenerate the children of parents that have a survivor and materialise those with key < X  (pass 2)
//   DIRECT : single pass, every child is materialised                     (beam cannot bind)
#include <climits>

#include "device_common.cuh"
#include "launch.hpp"

namespace efm {

enum { CH_OK = 0, CH_NONPOS = 1, CH_OVERFLOW = 2 };
#ifndef EFM_MIN_BLOCKS
#define EFM_MIN_BLOCKS 24   // resident one-warp blocks per SM the register allocation aims at (80 registers)
#endif
#ifndef EFM_KBLOCK
#define EFM_KBLOCK 32
#endif
constexpr int kBlock = EFM_KBLOCK;    // one warp per block: a finished warp frees its slot at once (parents differ a lot in cost)
constexpr int kWarps = kBlock / 32;
#ifndef EFM_PPW
#define EFM_PPW 8
#endif
constexpr int kParentsPerWarp = EFM_PPW;
#ifndef EFM_STAGE_BYTES
#define EFM_STAGE_BYTES 1536
#endif
constexpr int kStageBytes = EFM_STAGE_BYTES;   // staging buffer per parent (larger entries are read in place)
static_assert(kParentsPerWarp <= 8, "SS_OFF holds 8 parent offsets");
#ifndef EFM_PREFETCH
#define EFM_PREFETCH EFM_STAGE_BYTES
#endif
constexpr int kPrefetch = EFM_PREFETCH;   // bytes of the next parent requested ahead (1536 = the whole staging buffer: 41.7 ms, 1024: 42.2 ms)
constexpr u32 FULL = 0xffffffffu;
constexpr u64 kSmall = 1ULL << 40;   // fast path: every flux and extra flux of the parent below this ...
constexpr int kSmallCoef = 1 << 20;  // ... and every coefficient below this: no product can reach 2^62

// ------------------------------------------------------------------ warp collectives
// Collectives over a group of G consecutive lanes (G = 32: the warp); `m` is the lane mask of the group.
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
__device__ __forceinline__ u64 w_max(u64 v) {   // two 32-bit redux instead of five 64-bit shuffle rounds
    const u32 hi = (u32)(v >> 32);
    const u32 mh = __reduce_max_sync(FULL, hi);
    const u32 ml = __reduce_max_sync(FULL, hi == mh ? (u32)v : 0u);
    return ((u64)mh << 32) | ml;
}
__device__ __forceinline__ u64 w_min(u64 v) { return ~w_max(~v); }
__device__ __forceinline__ u64 w_bcast(u64 v, int src) { return __shfl_sync(FULL, v, src); }

// ------------------------------------------------------------------ integer helpers
// The rarely taken arithmetic (64-bit division, gcd) stays out of line: inlined at every site it was almost half of the
// kernel's instructions and the hot path paid for it in instruction-cache misses.
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
__device__ __noinline__ u32 gcd32(u32 a, u32 b) {
    if (a == 0) return b;
    if (b == 0) return a;
    const int sh = __ffs((int)(a | b)) - 1;
    a >>= (__ffs((int)a) - 1);
    do {
        b >>= (__ffs((int)b) - 1);
        if (a > b) { u32 t = a; a = b; b = t; }
        b -= a;
    } while (b);
    return a << sh;
}
template <int G>
__device__ __forceinline__ u64 g_gcd(u32 m, u64 v, bool narrow) {
    if (narrow) {   // every value below 2^32
        u32 x = (u32)v;
#pragma unroll
        for (int o = G / 2; o; o >>= 1) { const u32 w = __shfl_xor_sync(m, x, o); x = gcd32(x, w); }
        return x;
    }
#pragma unroll
    for (int o = G / 2; o; o >>= 1) { const u64 w = __shfl_xor_sync(m, v, o); v = gcd64(v, w); }
    return v;
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
// arc term of the state hash through the per-arc table of multipliers (device_common.cuh: arc_term)
__device__ __forceinline__ u64 arc_term_t(const DevGraph& g, u32 a, u64 f) { return __ldg(&g.arc_mix[a]) * f; }

// Per-warp chunked reservation of beam-key slots: one atomic per kKeyChunk keys instead of one per child.
constexpr u64 kNoSlot = ~0ULL;
template <int G>
struct KeyOut {
    u64 base; u32 left;
    u32 gmask; int gshift;   // lanes of the group that owns the chunk
    // one slot for every lane with want = true (others, and everyone after an overflow, get kNoSlot)
    __device__ __forceinline__ u64 reserve(const ExpandArgs& A, int lane, bool want) {
        const u32 m = (__ballot_sync(gmask, want) >> gshift) & (G == 32 ? 0xffffffffu : ((1u << (G & 31)) - 1u));
        const u32 cnt = (u32)__popc(m);
        if (cnt == 0) return kNoSlot;
        if (cnt > left) {
#pragma unroll 1
            for (u32 t = lane; t < left; t += G) A.keys[base + t] = kKeySentinel;
            u64 b = 0;
            if (lane == 0) b = atomicAdd(&A.ctl->n_slots, (u64)kKeyChunk);
            b = __shfl_sync(gmask, b, 0, G);
            if (__builtin_expect(b + kKeyChunk > A.max_keys, 0)) {
                if (lane == 0) atomicOr(&A.ctl->error, (u32)ERR_KEYS);
                left = 0;
                return kNoSlot;
            }
            base = b; left = kKeyChunk;
        }
        const u64 slot = want ? base + __popc(m & ((1u << lane) - 1u)) : kNoSlot;
        base += cnt; left -= cnt;
        return slot;
    }
    __device__ __forceinline__ void finish(const ExpandArgs& A, int lane) {
        for (u32 t = lane; t < left; t += G) A.keys[base + t] = kKeySentinel;
        left = 0;
    }
};

// gcd(E, c), E / gcd and c / gcd for the small coefficients of the fast path (c < 2^20); c = 2, 3 without a division
__device__ __forceinline__ void scale_small(u64 absE, u32 c, u32& k, u64& d) {
    if (c == 2) { const bool ev = (absE & 1ULL) == 0; k = ev ? 1u : 2u; d = ev ? absE >> 1 : absE; return; }
    if (c == 3) { const u64 qd = absE / 3ULL; const bool dv = qd * 3ULL == absE; k = dv ? 1u : 3u; d = dv ? qd : absE; return; }
    const u32 gg = (u32)gcd64(umod64(absE, (u64)c), (u64)c);
    k = c / gg; d = udiv64(absE, (u64)gg);
}

// 16-byte asynchronous copy global -> shared (LDGSTS): no register staging, completion awaited with cp_async_wait()
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem_src));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group 0;\n" ::: "memory"); }

__device__ __forceinline__ bool sbit(const u32* bits, int a) { return (bits[a >> 5] >> (a & 31)) & 1u; }

// per-warp statistics live in shared memory (one u64 each), flushed to the control block once per warp
enum { SS_EXPANDED = 0, SS_CHILDREN, SS_DONE, SS_ACTIVE, SS_DEAD, SS_NOTEFM, SS_NONPOS, SS_OVF, SS_VISITED, SS_BYTES,
       SS_ROUNDS, SS_FIRST, SS_GENERAL, SS_SATURATED,
       SS_OFF,   // kParentsPerWarp words: offsets of the parents of this group
       SS_WORDS = SS_OFF + 8 };

// One kernel body, every routine inlined once: the staged parent is addressed through shared-memory pointers the
// compiler can track.  The kernel only EVALUATES: every child that passes the discard tests gets a slot holding its
// beam key and a 64-byte task (what k_materialise needs to build it from its parent); nothing is written to the next
// frontier here, so a parent with hundreds of surviving children costs this warp no more than one without any.
template <int G>
__global__ void __launch_bounds__(kBlock, EFM_MIN_BLOCKS) k_expand(const __grid_constant__ ExpandArgs A) {
    extern __shared__ uint4 smem4[];
    // a group of G consecutive lanes owns a parent (G = 32: the warp; G = 16: two parents per warp share the issue slots
    // of the control flow they have in common)
    const int lane = threadIdx.x & (G - 1);
    const int wib = threadIdx.x / G;
    const u32 gbits = G == 32 ? 0xffffffffu : ((1u << (G & 31)) - 1u);
    const int gshift = threadIdx.x & 31 & ~(G - 1);
    const u32 gmask = gbits << gshift;
    auto gballot = [&](bool pred) -> u32 { return (__ballot_sync(gmask, pred) >> gshift) & gbits; };
    unsigned char* gs = (unsigned char*)smem4 + (size_t)wib * A.sm_group;
    uint4* stage = (uint4*)gs;
    u32* sbits = (u32*)(gs + A.sm_sbits);   // support bitset over arcs
    u16* upos = (u16*)(gs + A.sm_upos);     // metabolite -> 1 + index in the EF list of the parent, 0 = balanced
    u64* sst = (u64*)(gs + A.sm_misc);
    #pragma unroll 1
    for (int i = lane; i < A.g.W32; i += G) sbits[i] = 0;
    #pragma unroll 1
    for (int i = lane; i < (A.g.M + 8) / 8; i += G) ((uint4*)upos)[i] = make_uint4(0, 0, 0, 0);
    for (int i = lane; i < SS_WORDS; i += G) sst[i] = 0;
    __syncwarp(gmask);

    Ctl* ctl = A.ctl;
    const bool fast_graph = !A.no_fast && A.g.max_coef < kSmallCoef;
    KeyOut<G> ko; ko.base = 0; ko.left = 0; ko.gmask = gmask; ko.gshift = gshift;
    // a warp owns A.ppw (<= kParentsPerWarp) consecutive parents; the grid covers the level and the block scheduler evens out the
    // very different costs of parents (skipped / first visit over a hub / revisit)
    const u64 p0 = ((u64)blockIdx.x * (blockDim.x / G) + wib) * A.ppw;
    const u64 p1 = min(p0 + A.ppw, A.n_cur);

    // Double-buffered staging: while parent p is processed, the first kPrefetch bytes of parent p + 1 travel to the other
    // staging buffer with asynchronous copies (no registers, no waiting); the frontier buffers end in spare bytes so that
    // the fixed-size copy may run past the end of a short entry.
    u64* soff = sst + SS_OFF;
    if (lane < kParentsPerWarp) soff[lane] = p0 + lane < p1 ? __ldcs(&A.cur_off[p0 + lane]) : 0ULL;
    __syncwarp(gmask);
    const u32 pre_chunks = min(A.sm_stage_bytes, (u32)kPrefetch) / 16;
    auto prefetch = [&](u64 p, int b) {
        const unsigned char* gsrc = A.cur + (soff[p - p0] << 4);
        unsigned char* sdst = gs + (size_t)b * A.sm_stage_bytes;
        #pragma unroll 1
        for (u32 c = lane; c < pre_chunks; c += G) cp_async16(sdst + 16 * c, gsrc + 16 * c);
        cp_async_commit();
    };
    if (p0 < p1) prefetch(p0, 0);
#pragma unroll 1
    for (u64 p = p0; p < p1; ++p) {
        // ---- the parent: its first kPrefetch bytes are on their way already, the rest follows once the header is known
        const int sb = (int)(p - p0) & 1;
        const uint4* src = (const uint4*)(A.cur + (soff[p - p0] << 4));
        cp_async_wait();
        __syncwarp(gmask);
        if (p + 1 < p1) prefetch(p + 1, sb ^ 1);
        stage = (uint4*)(gs + (size_t)sb * A.sm_stage_bytes);
        const uint4 h0 = stage[0], h1 = stage[1];
        const int ns = (int)(h0.x & 0xffffu), nv = (int)(h0.x >> 16);
        const int nu = (int)h0.y;
        const u32 nch = entry_bytes((u32)ns, (u32)nv, (u32)nu) / 16;
        // entries that fit the staging buffer are read from shared memory; the rare larger ones are read in place
        const bool staged = !A.force_inplace && nch * 16 <= A.sm_stage_bytes;
        if (__builtin_expect(staged, 1)) {
            #pragma unroll 1
            for (u32 c = pre_chunks + lane; c < nch; c += G) stage[c] = __ldcs(src + c);   // streaming: the frontier must not evict the graph from L1
        }
        __syncwarp(gmask);
        const u64 Phs = (u64)h0.z | ((u64)h0.w << 32);
        const u64 Phv = (u64)h1.x | ((u64)h1.y << 32);
        const u64 Pbig = (u64)h1.z | ((u64)h1.w << 32);
        const unsigned char* eb = staged ? (const unsigned char*)stage : (const unsigned char*)src;
        const i64* flux = (const i64*)(eb + kHdr);
        const u64* vis = (const u64*)(flux + ns);
        const i64* ef = (const i64*)(vis + nv);
        const u16* arc = (const u16*)(ef + nu);
        const u16* efmet = arc + ns;

        // ---- support bitset, EF index table, PROC0: lowest unbalanced metabolite i* (reading G12)
        #pragma unroll 1
        for (int t = lane; t < ns; t += G) { const u32 a = arc[t]; atomicOr(&sbits[a >> 5], 1u << (a & 31)); }
        u32 best = 0xffffffffu;
        #pragma unroll 1
        for (int t = lane; t < nu; t += G) {
            const u32 i = efmet[t];
            upos[i] = (u16)(t + 1);
            best = min(best, (i << 16) | (u32)t);
        }
        best = __reduce_min_sync(gmask, best);
        __syncwarp(gmask);
        const int istar = (int)(best >> 16);
        const i64 E = ef[best & 0xffffu];
        const bool fwd = E > 0;
        const u64 absE = abs64(E);
        auto ef_of = [&](int met) -> i64 { const u32 u = upos[met]; return u ? ef[u - 1] : 0; };
        if (lane == 0) { sst[SS_EXPANDED]++; sst[SS_BYTES] += algo_entry_bytes((u32)ns, (u32)nv); }
        // visited?
        int vk = -1;
        #pragma unroll 1
        for (int base = 0; base < nv && vk < 0; base += G) {
            const int u = base + lane;
            const u32 hit = gballot(u < nv && (int)((vis[u] >> 32) & 0xffffu) == istar);
            if (hit) vk = base + __ffs(hit) - 1;
        }
        const bool firstv = vk < 0;
        if (lane == 0) { sst[SS_FIRST] += firstv; sst[SS_SATURATED] += ns >= A.D; }
        const int in0 = __ldg(&A.g.in_ptr[istar]), nI = __ldg(&A.g.in_ptr[istar + 1]) - in0;
        const int out0 = __ldg(&A.g.out_ptr[istar]), nO = __ldg(&A.g.out_ptr[istar + 1]) - out0;

        // ---- what to branch over: the OR-alternatives of i* (first visit) or the single Eq 4 / Eq 5 bump (revisit)
        const int2* alist = nullptr;
        const uint4* altl = nullptr;
        int alen = 0, prim = -1;
        int r_a = 0, r_c = 1, r_sign = +1;
        u64 rec = 0, r_newrec = 0;
        if (firstv) {
            // PROC1 / PROC1' (Eq 3; readings G1, G13, G14, G15, G22)
            if (nv >= A.V) {
                if (lane == 0) sst[SS_VISITED]++;
            } else {
                // primary on the side the flux arrives from: lowest arc of that side in the support (G13)
                const int2* plist = fwd ? A.g.in_e + in0 : A.g.out_e + out0;
                const int plen = fwd ? nI : nO;
                #pragma unroll 1
                for (int base = 0; base < plen && prim < 0; base += G) {
                    const int q = base + lane;
                    const int pa = q < plen ? __ldg(&plist[q]).x : -1;
                    const u32 bal = gballot(pa >= 0 && sbit(sbits, pa));
                    if (bal) prim = __shfl_sync(gmask, pa, __ffs(bal) - 1, G);
                }
                alist = fwd ? A.g.out_e + out0 : A.g.in_e + in0;
                altl = fwd ? A.g.out_alt + 2 * (size_t)out0 : A.g.in_alt + 2 * (size_t)in0;
                alen = fwd ? nO : nI;
            }
        } else {
            // PROC2-4 (readings G2-G5)
            rec = vis[vk];
            const int cntv = (int)(rec >> 48) + 1;
            if (cntv > A.max_loop) {
                if (lane == 0) sst[SS_NOTEFM]++;
            } else {
                const int PI = (int)((rec >> 16) & 0xffffu), PO = (int)(rec & 0xffffu);
                int lPI = -1, lPO = -1, cPI = 0, cPO = 0;
                #pragma unroll 1
                for (int q = lane; q < nI; q += G) { const int2 e = __ldg(&A.g.in_e[in0 + q]); if (e.x == PI) { lPI = q; cPI = e.y; } }
                #pragma unroll 1
                for (int q = lane; q < nO; q += G) { const int2 e = __ldg(&A.g.out_e[out0 + q]); if (e.x == PO) { lPO = q; cPO = e.y; } }
                lPI = __reduce_max_sync(gmask, lPI); cPI = __reduce_max_sync(gmask, cPI);
                lPO = __reduce_max_sync(gmask, lPO); cPO = __reduce_max_sync(gmask, cPO);
                // Def 11: forward PO ~ SI, backward PI ~ SO, secondary = any arc of that side in the support (G5)
                bool dep = false;
                const i64 doff = __ldg(&A.g.dep_off[istar]);
                if (fwd) {
                    #pragma unroll 1
                    for (int q = lane; q < nI; q += G) {
                        const i64 b = doff + (i64)lPO * nI + q;
                        dep = dep || (sbit(sbits, __ldg(&A.g.in_e[in0 + q]).x) && ((__ldg(&A.g.dep_bits[b >> 5]) >> (b & 31)) & 1u));
                    }
                } else {
                    #pragma unroll 1
                    for (int q = lane; q < nO; q += G) {
                        const i64 b = doff + (i64)q * nI + lPI;
                        dep = dep || (sbit(sbits, __ldg(&A.g.out_e[out0 + q]).x) && ((__ldg(&A.g.dep_bits[b >> 5]) >> (b & 31)) & 1u));
                    }
                }
                dep = __any_sync(gmask, dep);
                if (fwd) { if (!dep) { r_a = PO; r_c = cPO; r_sign = +1; } else { r_a = PI; r_c = cPI; r_sign = -1; } }   // Eq 4 / Eq 5
                else     { if (!dep) { r_a = PI; r_c = cPI; r_sign = +1; } else { r_a = PO; r_c = cPO; r_sign = -1; } }
                r_newrec = vis_pack((u32)istar, (u32)PI, (u32)PO, (u32)cntv);
                alen = 1;
            }
        }
        const bool fastP = firstv && fast_graph && Pbig < kSmall;
        int n_adm = 0;
        #pragma unroll 1
        for (int base = 0; base < alen; base += G) {
            const int q = base + lane;
            int a = -1, c = 1;
            bool adm = false, insup = false, generic = false;
            uint4 r0 = make_uint4(0, 0, 0, 0), r1 = r0;
            if (firstv) {
                if (q < alen) {   // one 32-byte record per OR-alternative: arc, c, twin and the column of the arc
                    r0 = __ldg(&altl[2 * q]); r1 = __ldg(&altl[2 * q + 1]);
                    a = (int)(r0.x & 0xffffu); c = (int)(r0.x >> 16);
                    const u32 tw = r0.y & 0xffffu;
                    generic = (r0.y >> 24) & 1u;
                    if (__builtin_expect(generic, 0)) c = __ldg(&alist[q]).y;   // the coefficient may not fit the record
                    insup = sbit(sbits, a);
                    adm = !(tw != 0xffffu && sbit(sbits, (int)tw)) && (insup || ns < A.D);
                }
            } else if (lane == 0) {
                a = r_a; c = r_c; adm = true; insup = true;   // PI / PO are arcs of the support
            }
            if (lane == 0) sst[SS_ROUNDS]++;
            const u32 adm_m = gballot(adm);
            if (__builtin_expect(adm_m == 0, 0)) continue;
            n_adm += __popc(adm_m);
            // ---- lane-parallel evaluation: new arc, small integers => no overflow, no common factor
            const bool fast = adm && !insup && fastP && !generic;
            const u32 fast_m = gballot(fast);
            u32 k = 1; u64 d = absE;
            int nu2 = nu;
            u64 hs2 = 0, hv2 = 0, key = 0;
            if (fast_m) {
                if (fast) {
                    if (c != 1) scale_small(absE, (u32)c, k, d);
                    const int ncol = (int)((r0.y >> 16) & 0xffu);
                    const u32 cw[6] = {r0.z, r0.w, r1.x, r1.y, r1.z, r1.w};
#pragma unroll
                    for (int e = 0; e < 6; ++e) {
                        if (e < ncol) {
                            const i64 efp = ef_of((int)(cw[e] & 0xffffu));
                            const i64 x = (i64)k * efp + (i64)d * (i64)(short)(cw[e] >> 16);   // |.| < 2^60 + 2^60
                            nu2 += (int)(x != 0) - (int)(efp != 0);
                        }
                    }
                }
                const u64 hsb = (u64)k * Phs;   // the arc part of the state hash is linear in the fluxes
                if (fast) {
                    const u64 newrec = vis_pack((u32)istar, (u32)(fwd ? prim : a), (u32)(fwd ? a : prim), 0u);
                    hs2 = hsb + arc_term_t(A.g, (u32)a, d);
                    hv2 = Phv + vis_term(newrec);
                    key = beam_key((u32)nu2, mix64(hs2 + hv2));
                }
            }
            const u32 done_m = gballot(fast && nu2 == 0);
            if (lane == 0) {
                const int nf = __popc(fast_m);
                sst[SS_CHILDREN] += nf; sst[SS_BYTES] += 8 * nf; sst[SS_DONE] += __popc(done_m); sst[SS_ACTIVE] += __popc(fast_m & ~done_m);
            }
            // ---- emit the lane-parallel children: one slot each (beam key + task)
            if (fast_m) {
                const u64 slot = ko.reserve(A, lane, fast);
                if (fast && slot != kNoSlot) {
                    const u64 newrec = vis_pack((u32)istar, (u32)(fwd ? prim : a), (u32)(fwd ? a : prim), 0u);
                    __stcs(&A.keys[slot], nu2 == 0 ? kKeyDone : key);
                    __stcs(&A.t0[slot], make_uint4((u32)p, (u32)a | 0xffff0000u, (u32)nu2 | ((u32)TF_FIRST << 16), k));
                    __stcs(&A.t1[slot], make_uint4((u32)d, (u32)(d >> 32), (u32)d, (u32)(d >> 32)));
                    __stcs(&A.t2[slot], make_uint4(1u, 0u, (u32)hs2, (u32)(hs2 >> 32)));
                    __stcs(&A.t3[slot], make_uint4((u32)hv2, (u32)(hv2 >> 32), (u32)newrec, (u32)(newrec >> 32)));
                }
            }
            // ---- one child at a time: general evaluation (arc of the support, large integers)
            u32 slow_m = adm_m & ~fast_m;
            #pragma unroll 1
            while (slow_m) {
                const int l = __ffs(slow_m) - 1;
                slow_m &= slow_m - 1;
                // warp-uniform description of the child relative to its parent
                const int ca = __shfl_sync(gmask, a, l, G);
                u64 ck, cd, cT, cg = 1, chs, chv;   // scale, |E| / gcd(|E|, c), un-normalised new flux of ca, common divisor, hash sums
                int cnu = nu, csign = +1, cia = -1;
                bool cin = false;
                const u64 newrec = firstv ? vis_pack((u32)istar, (u32)(fwd ? prim : ca), (u32)(fwd ? ca : prim), 0u) : r_newrec;
                const int qa0 = __ldg(&A.g.col_ptr[ca]), qa1 = __ldg(&A.g.col_ptr[ca + 1]);
                {
                // bump(f, a, sign*|E|/c) of SURVEY.md 8(c) O6 with the whole warp
                const int cc = __shfl_sync(gmask, c, l, G);
                csign = firstv ? +1 : r_sign;
                const u64 gg = cc == 1 ? 1ULL : gcd64(absE, (u64)cc);
                ck = gg == 1 ? (u64)cc : (u64)((u32)cc / (u32)gg);
                cd = gg == 1 ? absE : udiv64(absE, gg);
                cin = sbit(sbits, ca);
                if (cin) {   // position of the arc in the sorted support
                    #pragma unroll 1
                    for (int b2 = 0; b2 < ns && cia < 0; b2 += G) {
                        const int t = b2 + lane;
                        const u32 hit = gballot(t < ns && arc[t] == ca);
                        if (hit) cia = b2 + __ffs(hit) - 1;
                    }
                }
                // scaled fluxes F_t = k f_t, F_a = k f_a +- d: overflow first, then non-positive (order of O6).
                // Pbig >= every flux and |EF| of the parent: products below the guard with it need no exact sweep.
                const bool bigk = ck > 1 && umul_gt_guard(ck, Pbig);
                bool ovf = false, nonpos = false;
                cT = cd;
                if (cin) {
                    const u64 fa = (u64)flux[cia];
                    const u64 lo = ck * fa, hi = __umul64hi(ck, fa);
                    if (csign > 0) {
                        cT = lo + cd;
                        const u64 hi2 = hi + (cT < lo);
                        ovf = hi2 != 0 || cT > EFM_GUARD;
                    } else {
                        if (hi == 0 && lo <= cd) { nonpos = true; cT = 0; }           // k f_a - d <= 0
                        else { cT = lo - cd; const u64 hi2 = hi - (lo < cd); ovf = hi2 != 0 || cT > EFM_GUARD; }
                    }
                }
                if (__builtin_expect(bigk, 0)) {   // exact: the largest flux among t != ia (a new arc carries d <= |E| <= 2^62)
                    u64 mx = 0;
                    #pragma unroll 1
                    for (int t = lane; t < ns; t += G) if (t != cia) mx = max(mx, (u64)flux[t]);
                    mx = g_max(gmask, mx);
                    ovf = ovf || umul_gt_guard(ck, mx);
                }
                int status = ovf ? CH_OVERFLOW : (nonpos ? CH_NONPOS : CH_OK);   // Prop 3, G11
                if (status == CH_OK) {
                    // extra fluxes of the un-normalised child: EF'_i = k EF_i + sign d s_ia (Eq 2 on the scaled fluxes)
                    bool ovf2 = false;
                    if (__builtin_expect(bigk, 0)) {   // exact sweep over the unbalanced metabolites outside col(a)
                        #pragma unroll 1
                        for (int t = lane; t < nu; t += G) {
                            const int i = efmet[t];
                            bool in_a = false;
                            #pragma unroll 1
                            for (int r = qa0; r < qa1; ++r) in_a = in_a || __ldg(&A.g.col[r]).x == i;
                            if (!in_a) ovf2 = ovf2 || abs_gt_guard(mul_s((i64)ck, ef[t]));
                        }
                    }
                    int delta = 0;
                    #pragma unroll 1
                    for (int qq = qa0 + lane; qq < qa1; qq += G) {
                        const int2 e = __ldg(&A.g.col[qq]);
                        const i64 efp = ef_of(e.x);
                        const S128 x = add_s(mul_s((i64)ck, efp), mul_s(csign > 0 ? (i64)cd : -(i64)cd, (i64)e.y));
                        ovf2 = ovf2 || abs_gt_guard(x);
                        delta += (int)((x.lo | (u64)x.hi) != 0) - (int)(efp != 0);
                    }
                    if (__any_sync(gmask, ovf2)) status = CH_OVERFLOW;
                    else cnu = nu + __reduce_add_sync(gmask, delta);
                }
                if (__builtin_expect(status != CH_OK, 0)) {
                    if (lane == 0) sst[status == CH_OVERFLOW ? SS_OVF : SS_NONPOS]++;
                    continue;
                }
                // gcd normalisation (reading G10).  A new arc cannot introduce a common factor: gcd_t(k f_t) = k and
                // gcd(k, d) = 1.  An arc of the support: g = gcd(T, k f_t for t != a).
                if (cin && cT != 1) {
                    // every lane folds its scaled fluxes into r = gcd(T, k f_t, ...); r divides T, and one lane with
                    // r = 1 settles g = 1 (the usual case: T is small and some flux is coprime to it)
                    const bool narrow = cT < (1ULL << 32);
                    u64 r = cT;
                    #pragma unroll 1
                    for (int t = lane; t < ns; t += G) {
                        if (t == cia) continue;
                        const u64 x = ck * (u64)flux[t];   // <= 2^62 (no overflow was found above)
                        if (narrow) {
                            const u32 r32 = (u32)r;
                            r = gcd32(r32, (x >> 32) == 0 ? (u32)x % r32 : (u32)umod64(x, (u64)r32));
                        } else r = gcd64(r, x);
                    }
                    if (__builtin_expect(!__any_sync(gmask, r == 1), 0)) cg = g_gcd<G>(gmask, r, narrow);
                }
                if (cg == 1) {   // linear: sum of m_t (k f_t) with the term of arc a replaced by m_a T
                    chs = ck * Phs + arc_term_t(A.g, (u32)ca, cT - (cin ? ck * (u64)flux[cia] : 0ULL));
                } else {
                    chs = 0;
                    #pragma unroll 1
                    for (int t = lane; t < ns; t += G) {
                        u64 F = t == cia ? cT : ck * (u64)flux[t];
                        if (cg > 1) F = udiv64(F, cg);
                        chs += arc_term_t(A.g, (u32)arc[t], F);
                    }
                    chs = g_sum<G>(gmask, chs);
                    if (!cin) chs += arc_term_t(A.g, (u32)ca, cT);
                }
                chv = Phv + vis_term(newrec) - (firstv ? 0ULL : vis_term(rec));
                }
                // account for the child and emit it
                const bool cdone = cnu == 0;
                if (lane == 0) { sst[SS_CHILDREN]++; sst[SS_GENERAL]++; sst[SS_BYTES] += 8; sst[cdone ? SS_DONE : SS_ACTIVE]++; }
                const u64 slot = ko.reserve(A, lane, lane == 0);
                if (lane == 0 && slot != kNoSlot) {
                    const u32 flags = (csign < 0 ? TF_NEG : 0u) | (firstv ? TF_FIRST : 0u) | (cin ? TF_INSUPP : 0u);
                    __stcs(&A.keys[slot], cdone ? kKeyDone : beam_key((u32)cnu, mix64(chs + chv)));
                    __stcs(&A.t0[slot], make_uint4((u32)p, (u32)ca | ((u32)(cia & 0xffff) << 16), (u32)cnu | (flags << 16), (u32)ck));
                    __stcs(&A.t1[slot], make_uint4((u32)cd, (u32)(cd >> 32), (u32)cT, (u32)(cT >> 32)));
                    __stcs(&A.t2[slot], make_uint4((u32)cg, (u32)(cg >> 32), (u32)chs, (u32)(chs >> 32)));
                    __stcs(&A.t3[slot], make_uint4((u32)chv, (u32)(chv >> 32), (u32)newrec, (u32)(newrec >> 32)));
                }
            }
        }
        if (firstv && nv < A.V && n_adm == 0 && lane == 0) sst[SS_DEAD]++;   // no admissible alternative
        // ---- restore the shared tables to zero for the next parent
        __syncwarp(gmask);
        #pragma unroll 1
        for (int t = lane; t < ns; t += G) sbits[arc[t] >> 5] = 0;
        #pragma unroll 1
        for (int t = lane; t < nu; t += G) upos[efmet[t]] = 0;
        __syncwarp(gmask);
    }
    ko.finish(A, lane);
    __syncwarp(gmask);
    if (lane == 0) {
        u64* st = ctl->st;
        if (sst[SS_EXPANDED]) { atomicAdd(&st[ST_EXPANDED], sst[SS_EXPANDED]); atomicAdd(&ctl->lvl_expanded, sst[SS_EXPANDED]); }
        if (sst[SS_CHILDREN]) { atomicAdd(&st[ST_CHILDREN], sst[SS_CHILDREN]); atomicAdd(&ctl->lvl_children, sst[SS_CHILDREN]); }
        if (sst[SS_DONE]) atomicAdd(&ctl->lvl_done, sst[SS_DONE]);
        if (sst[SS_ACTIVE]) atomicAdd(&ctl->n_keys, sst[SS_ACTIVE]);
        if (sst[SS_DEAD]) atomicAdd(&st[ST_DEAD_END], sst[SS_DEAD]);
        if (sst[SS_NOTEFM]) atomicAdd(&st[ST_NOT_EFM], sst[SS_NOTEFM]);
        if (sst[SS_NONPOS]) atomicAdd(&st[ST_NONPOS], sst[SS_NONPOS]);
        if (sst[SS_OVF]) atomicAdd(&st[ST_OVERFLOW], sst[SS_OVF]);
        if (sst[SS_VISITED]) atomicAdd(&st[ST_VISITED], sst[SS_VISITED]);
        if (sst[SS_BYTES]) atomicAdd(&st[ST_ALGO_BYTES], sst[SS_BYTES]);
        if (sst[SS_ROUNDS]) atomicAdd(&st[ST_ROUNDS], sst[SS_ROUNDS]);
        if (sst[SS_FIRST]) atomicAdd(&st[ST_FIRST], sst[SS_FIRST]);
        if (sst[SS_GENERAL]) atomicAdd(&st[ST_GENERAL], sst[SS_GENERAL]);
        if (sst[SS_SATURATED]) atomicAdd(&st[ST_SATURATED], sst[SS_SATURATED]);
    }
}

// ------------------------------------------------------------------ survivors of the beam -> list of slots
// Balanced children (kKeyDone) and active children with key < X (all of them when the beam does not bind).  A block
// appends the survivors of a tile with ONE atomic (a warp-level atomic per 32 keys serialised on the counter); the order
// of the list does not matter.
constexpr int kCompactItems = 4;   // keys per thread: a block handles the survivors of 1024 keys with one atomic per counter
// Besides listing the survivors, the kernel sizes every child (task + parent header) and reserves its place: an entry
// index and 16-byte units in the next frontier, or a candidate slot.  k_materialise then needs no coordination at all.
__global__ void __launch_bounds__(256) k_compact(const __grid_constant__ ExpandArgs A) {
    __shared__ u32 s_w[4][8];      // per warp totals: survivors, frontier children, frontier units, candidates
    __shared__ u64 s_base[4];
    Ctl* ctl = A.ctl;
    const u64 n = min(ctl->n_slots, A.max_keys);
    const bool notrunc = ctl->notrunc != 0;
    const u64 X = ctl->X;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    constexpr u64 kTile = 256 * kCompactItems;
    for (u64 tile = (u64)blockIdx.x * kTile; tile < n; tile += (u64)gridDim.x * kTile) {   // block-uniform trip count
        // item j of a thread is key tile + j * 256 + threadIdx.x (coalesced loads)
        u32 takes = 0, my_front = 0, my_units = 0, my_cand = 0, my_bytes = 0;
        u32 units[kCompactItems];
        u64 poff[kCompactItems];
        // the four items of a thread advance together through the chain key -> task word -> parent offset -> parent header,
        // so that a thread waits for three memory latencies, not twelve
#pragma unroll
        for (int j = 0; j < kCompactItems; ++j) {
            const u64 i = tile + (u64)j * 256 + threadIdx.x;
            const u64 key = i < n ? __ldcs(&A.keys[i]) : kKeySentinel;
            if (key == kKeyDone || (key != kKeySentinel && (notrunc || key < X))) takes |= 1u << j;
        }
        u32 qx[kCompactItems], qz[kCompactItems], w0[kCompactItems];
#pragma unroll
        for (int j = 0; j < kCompactItems; ++j) {
            qx[j] = 0; qz[j] = 0;
            if ((takes >> j) & 1u) { const uint4 q0 = __ldcs(&A.t0[tile + (u64)j * 256 + threadIdx.x]); qx[j] = q0.x; qz[j] = q0.z; }
        }
#pragma unroll
        for (int j = 0; j < kCompactItems; ++j) poff[j] = ((takes >> j) & 1u) ? __ldg(&A.cur_off[qx[j]]) : 0ULL;
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
            if (c == 0) s_base[0] = tot ? atomicAdd(&ctl->n_surv, (u64)tot) : 0ULL;
            if (c == 1) s_base[1] = tot;                      // frontier children of the block (combined with c == 2 below)
            if (c == 2) s_base[2] = tot;
            if (c == 3) s_base[3] = tot ? atomicAdd(&ctl->n_cand, (u64)tot) : 0ULL;
        }
        if (lane == 0 && my_bytes) atomicAdd(&ctl->st[ST_ALGO_BYTES], (u64)my_bytes);
        __syncthreads();
        if (threadIdx.x == 0) {
            const u64 nf = s_base[1], nu = s_base[2];
            const u64 old = nf ? atomicAdd(&ctl->n_next, (nf << kAllocShift) | nu) : 0ULL;
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
                A.surv[pos] = make_ulonglong2(i, poff[j]);
                A.surv_dst[pos] = dst;
                ++pos;
            }
        }
        __syncthreads();   // the shared arrays are reused by the next tile
    }
}

// ------------------------------------------------------------------ materialise: G lanes per surviving child
// Reads the task, reads the parent entry straight from HBM / L2 (every element is needed once) and writes the child:
// a candidate slot if it is balanced, otherwise a packed entry of the next frontier.  A block of 256 / G children
// takes the places k_compact reserved.  G = 8 (four children per warp) suits entries of a few dozen arcs:
// the per-child control flow and address arithmetic is shared by a quarter as many instructions.
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
    const u64 n_surv = A.ctl->n_surv;
    // k_compact reserved the place of every child: the groups work on their own, no block-wide step is left
    for (u64 sidx = (u64)blockIdx.x * kMatWarps + wib; sidx < n_surv; sidx += (u64)gridDim.x * kMatWarps) {
    // ---- the task, the reserved place, the header of the parent
    const ulonglong2 sv = __ldcs(&A.surv[sidx]);
    const u64 dstrec = __ldcs(&A.surv_dst[sidx]);
    const u64 slot = sv.x;
    const unsigned char* pe = A.cur + (sv.y << 4);
    const uint4 q0 = __ldcs(&A.t0[slot]), q1 = __ldcs(&A.t1[slot]), q2 = __ldcs(&A.t2[slot]), q3 = __ldcs(&A.t3[slot]);
    const uint4 h0 = __ldg((const uint4*)pe);
    const int ca = (int)(q0.y & 0xffffu);
    const int cia = (q0.y >> 16) == 0xffffu ? -1 : (int)(q0.y >> 16);
    const int cnu = (int)(q0.z & 0xffffu);
    const u32 flags = q0.z >> 16;
    const bool cin = (flags & TF_INSUPP) != 0, firstv = (flags & TF_FIRST) != 0;
    const u64 ck = q0.w;
    const u64 cd = (u64)q1.x | ((u64)q1.y << 32), cT = (u64)q1.z | ((u64)q1.w << 32);
    const u64 cg = (u64)q2.x | ((u64)q2.y << 32), chs = (u64)q2.z | ((u64)q2.w << 32);
    const u64 chv = (u64)q3.x | ((u64)q3.y << 32), newrec = (u64)q3.z | ((u64)q3.w << 32);
    const u64 sd = (flags & TF_NEG) ? (u64)0 - cd : cd;
    // ---- the parent
    const int ns = (int)(h0.x & 0xffffu), nv = (int)(h0.x >> 16), nu = (int)h0.y;
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
    for (int t = lane; t < ns; t += G) {
        const u64 ft = t < G ? (u64)pf0 : (t < 2 * G ? (u64)pf1 : (u64)flux[t]);
        u64 F = t == cia ? cT : ck * ft;
        if (cg > 1) F = udiv64(F, cg);
        const int pos = t + ((!cin && t >= ins) ? 1 : 0);
        flux2[pos] = (i64)F;
        arc2[pos] = (u16)(t < G ? pa0 : (t < 2 * G ? pa1 : (u32)arc[t]));
        mx = max(mx, F);
    }
    if (!cin && lane == 0) { flux2[ins] = (i64)cT; arc2[ins] = (u16)ca; }
    if (!to_cand) {
        // the visited record of i* is appended (first visit) or replaced (revisit)
        const u32 met_star = (u32)((newrec >> 32) & 0xffffu);
        for (int u = lane; u < nv; u += G) {
            const u64 r = u < G ? pv0 : (u < 2 * G ? pv1 : vis[u]);
            vis2[u] = (!firstv && (u32)((r >> 32) & 0xffffu) == met_star) ? newrec : r;
        }
        if (firstv && lane == 0) vis2[nv] = newrec;
        // EF list of the child: EF' = (k EF + sign d s_.a) / g over the parent's list, then the metabolites of col(a)
        // that were balanced in the parent.  k_expand established that nothing exceeds 2^62, so the wrapping 64-bit
        // arithmetic is exact.
        const int qa0 = pcol0, qa1 = pcol1;
        int wbase = 0;
        u32 seen = 0;   // bit q - qa0: metabolite of col(a)[q] is in the parent's list (columns longer than 32: see below)
        for (int t0 = 0; t0 < nu; t0 += G) {
            const int t = t0 + lane;
            const bool valid = t < nu;
            i64 x = 0;
            int met = -1;
            if (valid) {
                met = t0 == 0 ? (int)pm0 : (int)efmet[t];
                i64 s = 0;
                for (int qq = qa0; qq < qa1; ++qq) { const int2 e = __ldg(&A.g.col[qq]); if (e.x == met) s = e.y; }
                x = (i64)(ck * (u64)(t0 == 0 ? pe0 : ef[t]) + sd * (u64)s);
                if (cg > 1) x = sdiv64(x, (i64)cg);
            }
            for (int qq = qa0; qq < qa1 && qq < qa0 + 32; ++qq)
                if (gany(valid && __ldg(&A.g.col[qq]).x == met)) seen |= 1u << (qq - qa0);
            const u32 nz = gballot(valid && x != 0);
            if (valid && x != 0) {
                const int pos = wbase + __popc(nz & lt);
                ef2[pos] = x; efmet2[pos] = (u16)met;
                mx = max(mx, abs64(x));
            }
            wbase += __popc(nz);
        }
        for (int qq = qa0; qq < qa1; ++qq) {   // warp-uniform, a handful of entries
            const int2 e = __ldg(&A.g.col[qq]);
            bool in_parent;
            if (qq < qa0 + 32) in_parent = (seen >> (qq - qa0)) & 1u;
            else {   // columns longer than 32 entries: scan the parent's list again
                bool f = false;
                for (int t = lane; t < nu; t += G) f = f || (int)efmet[t] == e.x;
                in_parent = gany(f);
            }
            if (!in_parent) {
                i64 x = (i64)(sd * (u64)(i64)e.y);
                if (cg > 1) x = sdiv64(x, (i64)cg);
                if (lane == 0) { ef2[wbase] = x; efmet2[wbase] = (u16)e.x; }
                mx = max(mx, abs64(x));
                ++wbase;
            }
        }
        {   // maximum over the lanes of the child
            const u32 hi = (u32)(mx >> 32);
            const u32 mh = __reduce_max_sync(gmask, hi);
            const u32 ml = __reduce_max_sync(gmask, hi == mh ? (u32)mx : 0u);
            mx = ((u64)mh << 32) | ml;
        }
    }
    if (lane == 0) {
        uint4* h4 = (uint4*)dst;
        h4[0] = make_uint4((u32)n2 | ((u32)nv2 << 16), (u32)nu2, (u32)chs, (u32)(chs >> 32));
        h4[1] = make_uint4((u32)chv, (u32)(chv >> 32), (u32)mx, (u32)(mx >> 32));
    }
    }   // ok
    }
}

__global__ void k_level_begin(Ctl* ctl) {
    ctl->n_next = 0; ctl->n_keys = 0; ctl->n_slots = 0; ctl->n_surv = 0; ctl->lvl_done = 0; ctl->lvl_children = 0; ctl->lvl_expanded = 0;
}

// ------------------------------------------------------------------ roots (INIT kernel of the paper)
// One thread per seed set.  BUILD: every seed arc gets flux 1, the extra fluxes follow from Eq 2; the
// root is classified like any other entry (balanced -> candidate, otherwise its beam key).  Seed sets are tiny, so
// the quadratic duplicate scan below is cheaper than any scatter.  WRITE: the roots the beam keeps become level 0.
template <bool WRITE>
__global__ void __launch_bounds__(128) k_roots(const RootArgs R) {
    const u64 r = (u64)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= R.n_roots) return;
    const DevGraph& g = R.g;
    Ctl* ctl = R.ctl;
    unsigned char* e = R.stage + (R.stage_off[r] << 4);
    if (WRITE) {
        const u64 key = R.keys[r];
        if (key == kKeySentinel || !(ctl->notrunc || key < ctl->X)) return;
        const u32 w0 = *(const u32*)e, nu = ((const u32*)e)[1];
        const u64 units = entry_bytes(w0 & 0xffffu, w0 >> 16, nu) >> 4;
        const u64 old = atomicAdd(&ctl->n_next, (1ULL << kAllocShift) | units);
        const u64 slot = old >> kAllocShift, off = old & kAllocUnitMask;
        if (slot >= R.max_frontier || off + units > R.frontier_units) { atomicOr(&ctl->error, (u32)ERR_FRONTIER); return; }
        R.nxt_off[slot] = off;
        uint4* dst = (uint4*)(R.nxt + (off << 4));
        for (u64 c = 0; c < units; ++c) dst[c] = ((const uint4*)e)[c];
        return;
    }
    if (r == 0) ctl->n_slots = R.n_roots;
    const int s0 = R.seed_ptr[r], ns = R.seed_ptr[r + 1] - s0;
    const int* arcs = R.seed_arc + s0;
    // Eq 2 with every flux = 1: EF_i = sum of s_ia over the seed arcs; (t, q) is the first occurrence of its metabolite
    auto ef_at = [&](int t, int q, i64& sum) -> bool {
        const int met = g.col[q].x;
        sum = 0;
        for (int t2 = 0; t2 < ns; ++t2)
            for (int q2 = g.col_ptr[arcs[t2]]; q2 < g.col_ptr[arcs[t2] + 1]; ++q2)
                if (g.col[q2].x == met) {
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
    for (int t = 0; t < ns; ++t)
        for (int q = g.col_ptr[arcs[t]]; q < g.col_ptr[arcs[t] + 1]; ++q) {
            i64 s;
            if (ef_at(t, q, s)) { ef[w] = s; efmet[w] = (u16)g.col[q].x; big = max(big, abs64(s)); ++w; }
        }
    ((u32*)e)[0] = (u32)ns; ((u32*)e)[1] = (u32)nu;
    ((u64*)e)[1] = hs; ((u64*)e)[2] = 0; ((u64*)e)[3] = big;
    if (nu == 0) {   // balanced at once (arbiter "Done")
        R.keys[r] = kKeySentinel;
        atomicAdd(&ctl->lvl_done, 1ULL);
        const u64 slot = atomicAdd(&ctl->n_cand, 1ULL);
        if (slot >= R.max_cand) { atomicOr(&ctl->error, (u32)ERR_CAND); return; }
        unsigned char* dst = R.cand + slot * R.cand_stride;
        const u32 bytes = entry_bytes((u32)ns, 0, 0);
        for (u32 c = 0; c < bytes / 16; ++c) ((uint4*)dst)[c] = ((const uint4*)e)[c];
    } else {
        R.keys[r] = beam_key((u32)nu, mix64(hs));
        atomicAdd(&ctl->n_keys, 1ULL);
    }
}

// ------------------------------------------------------------------ host launchers
static size_t align16(size_t x) { return (x + 15) & ~(size_t)15; }

void expand_smem_layout(ExpandArgs& a) {
    // staging: the largest entry if it is small, otherwise 1.5 KB (larger entries are rare and read in place);
    // the smaller the per-warp footprint, the more of the graph stays in L1
    a.sm_stage_bytes = (u32)align16(a.max_entry < (u32)kStageBytes ? (a.max_entry < 32u ? 32u : a.max_entry) : (u32)kStageBytes);
    size_t off = 2 * (size_t)a.sm_stage_bytes;   // two staging buffers
    a.sm_sbits = (u32)off; off = align16(off + (size_t)a.g.W32 * 4);
    a.sm_upos = (u32)off;  off = align16(off + (size_t)a.g.M * 2 + 16);   // zeroed in 16-byte chunks
    a.sm_misc = (u32)off;  off = align16(off + (size_t)SS_WORDS * 8);
    a.sm_group = (u32)off;
}

// key slots the count pass can leave unused: every warp of the largest grid may strand one chunk
// every warp may strand one chunk of key slots; a warp covers kParentsPerWarp parents
u64 expand_key_slack(u64 max_parents) { return (max_parents / kParentsPerWarp + 32768) * kKeyChunk; }

#ifndef EFM_EXP_GROUP
#define EFM_EXP_GROUP 32   // lanes per parent in k_expand (measured on genome / cap 262144: 32 -> 44 ms, 16 -> 64 ms, 8 -> 119 ms:
                           // the parents of a warp diverge too much to share issue slots, unlike k_materialise)
#endif
cudaError_t launch_expand(const ExpandArgs& a, int sm_count, cudaStream_t s) {
    constexpr int G = EFM_EXP_GROUP;
    // groups per block: as many as fit beside the per-group staging (huge networks fall back to fewer warps)
    int warps = kWarps;
    while (warps > 1 && (size_t)a.sm_group * warps * (32 / G) > 200 * 1024) warps >>= 1;
    const int groups = warps * (32 / G);
    const size_t smem = (size_t)a.sm_group * groups;
    if (smem > 227 * 1024) return cudaErrorInvalidValue;
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(k_expand<G>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    // small levels: fewer parents per group so that every SM still gets its share of warps
    u64 ppw = a.n_cur / ((u64)sm_count * 32 * (32 / G));
    ppw = ppw < 1 ? 1 : (ppw > (u64)kParentsPerWarp ? (u64)kParentsPerWarp : ppw);
    ExpandArgs a2 = a;
    a2.ppw = (u32)ppw;
    const u64 per_block = (u64)groups * ppw;
    const u64 need = (a.n_cur + per_block - 1) / per_block;
    if (need > 0x7fffffffULL) return cudaErrorInvalidValue;
    k_expand<G><<<(unsigned)(need ? need : 1), warps * 32, smem, s>>>(a2);
    return cudaGetLastError();
}

// survivors of the level -> next frontier / candidates.  n_hint bounds the key slots in use (host side estimate).
cudaError_t launch_materialise(const ExpandArgs& a, u64 n_slots_hint, u64 n_surv, int sm_count, cudaStream_t s, int phase) {
    if (phase == 0) {   // compact
        u64 blocks = (n_slots_hint + 1023) / 1024;   // one tile of 256 x kCompactItems keys per block and round
        if (blocks > (u64)sm_count * 64) blocks = (u64)sm_count * 64;
        if (blocks < 1) blocks = 1;
        k_compact<<<(unsigned)blocks, 256, 0, s>>>(a);
        return cudaGetLastError();
    }
    (void)n_surv;   // read on the device (ctl->n_surv): no host round trip between the two kernels
    k_materialise<EFM_MAT_GROUP><<<(unsigned)(sm_count * 32), kMatThreads, 0, s>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_roots(bool write, const RootArgs& r, cudaStream_t s) {
    const unsigned blocks = (unsigned)((r.n_roots + 127) / 128);
    if (write) k_roots<true><<<blocks, 128, 0, s>>>(r);
    else k_roots<false><<<blocks, 128, 0, s>>>(r);
    return cudaGetLastError();
}

cudaError_t launch_level_begin(Ctl* ctl, cudaStream_t s) {
    k_level_begin<<<1, 1, 0, s>>>(ctl);
    return cudaGetLastError();
}

}  // namespace efm
