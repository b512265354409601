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

enum { MODE_COUNT = 0, MODE_WRITE = 1, MODE_DIRECT = 2 };
enum { CH_OK = 0, CH_NONPOS = 1, CH_OVERFLOW = 2 };
#ifndef EFM_MIN_BLOCKS
#define EFM_MIN_BLOCKS 16   // resident one-warp blocks per SM the register allocation aims at (128 registers)
#endif
constexpr int kBlock = 32;    // one warp per block: a finished warp frees its slot at once (parents differ a lot in cost)
constexpr int kWarps = kBlock / 32;
#ifndef EFM_PPW
#define EFM_PPW 8
#endif
constexpr int kParentsPerWarp = EFM_PPW;
constexpr u32 FULL = 0xffffffffu;
constexpr u64 kSmall = 1ULL << 40;   // fast path: every flux and extra flux of the parent below this ...
constexpr int kSmallCoef = 1 << 20;  // ... and every coefficient below this: no product can reach 2^62

// ------------------------------------------------------------------ warp collectives
__device__ __forceinline__ u64 w_sum(u64 v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
    return v;
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
__device__ __forceinline__ u64 gcd64(u64 a, u64 b) {   // binary gcd
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
__device__ __forceinline__ u32 gcd32(u32 a, u32 b) {
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
__device__ __forceinline__ u64 w_gcd(u64 v, bool narrow) {
    if (narrow) {   // every value below 2^32
        u32 x = (u32)v;
#pragma unroll
        for (int o = 16; o; o >>= 1) { const u32 w = __shfl_xor_sync(FULL, x, o); x = gcd32(x, w); }
        return x;
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) { const u64 w = __shfl_xor_sync(FULL, v, o); v = gcd64(v, w); }
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
// arc term of the state hash through the per-arc table of inner mixes (device_common.cuh: arc_term)
__device__ __forceinline__ u64 arc_term_t(const DevGraph& g, u32 a, u64 f) { return mix64(__ldg(&g.arc_mix[a]) + f); }

// Per-warp chunked reservation of beam-key slots: one atomic per kKeyChunk keys instead of one per child.
struct KeyOut {
    u64 base; u32 left;
    __device__ __forceinline__ void push(const ExpandArgs& A, int lane, bool want, u64 key) {
        const u32 m = __ballot_sync(FULL, want);
        const u32 cnt = (u32)__popc(m);
        if (cnt == 0) return;
        if (cnt > left) {
#pragma unroll 1
            for (u32 t = lane; t < left; t += 32) A.keys[base + t] = kKeySentinel;
            u64 b = 0;
            if (lane == 0) b = atomicAdd(&A.ctl->n_slots, (u64)kKeyChunk);
            b = w_bcast(b, 0);
            if (b + kKeyChunk > A.max_keys) {
                if (lane == 0) atomicOr(&A.ctl->error, (u32)ERR_KEYS);
                left = 0;
                return;
            }
            base = b; left = kKeyChunk;
        }
        if (want) __stcs(&A.keys[base + __popc(m & ((1u << lane) - 1u))], key);
        base += cnt; left -= cnt;
    }
    __device__ __forceinline__ void finish(const ExpandArgs& A, int lane) {
        for (u32 t = lane; t < left; t += 32) A.keys[base + t] = kKeySentinel;
        left = 0;
    }
};

// gcd(E, c), E / gcd and c / gcd for the small coefficients of the fast path (c < 2^20); c = 2, 3 without a division
__device__ __forceinline__ void scale_small(u64 absE, u32 c, u32& k, u64& d) {
    if (c == 2) { const bool ev = (absE & 1ULL) == 0; k = ev ? 1u : 2u; d = ev ? absE >> 1 : absE; return; }
    if (c == 3) { const u64 qd = absE / 3ULL; const bool dv = qd * 3ULL == absE; k = dv ? 1u : 3u; d = dv ? qd : absE; return; }
    const u32 gg = (u32)gcd64(absE % (u64)c, (u64)c);
    k = c / gg; d = absE / (u64)gg;
}

__device__ __forceinline__ bool sbit(const u32* bits, int a) { return (bits[a >> 5] >> (a & 31)) & 1u; }

// per-warp statistics live in shared memory (one u64 each), flushed to the control block once per warp
enum { SS_EXPANDED = 0, SS_CHILDREN, SS_DONE, SS_ACTIVE, SS_DEAD, SS_NOTEFM, SS_NONPOS, SS_OVF, SS_VISITED, SS_BYTES,
       SS_ROUNDS, SS_FIRST, SS_GENERAL, SS_SATURATED, SS_WRITE_PARENTS,
       SS_KC,   // 4 words: the hash sums of the k-scaled support for the last two scales k (k0, s0, k1, s1)
       SS_WORDS = SS_KC + 4 };

// One kernel body, every routine inlined once: the staged parent is addressed through shared-memory pointers the
// compiler can track, and both kinds of children (lane-parallel "fast" ones and warp-cooperative "general" ones) funnel
// into a single evaluate / place / write sequence.
template <int MODE>
__global__ void __launch_bounds__(kBlock, EFM_MIN_BLOCKS) k_expand(const __grid_constant__ ExpandArgs A) {
    extern __shared__ uint4 smem4[];
    const int lane = threadIdx.x & 31;
    const int wib = threadIdx.x >> 5;
    const u32 lt = (1u << lane) - 1u;
    unsigned char* gs = (unsigned char*)smem4 + (size_t)wib * A.sm_group;
    uint4* stage = (uint4*)gs;
    u32* sbits = (u32*)(gs + A.sm_sbits);   // support bitset over arcs
    u16* upos = (u16*)(gs + A.sm_upos);     // metabolite -> 1 + index in the EF list of the parent, 0 = balanced
    u64* sst = (u64*)(gs + A.sm_misc);
    #pragma unroll 1
    for (int i = lane; i < A.g.W32; i += 32) sbits[i] = 0;
    #pragma unroll 1
    for (int i = lane; i < (A.g.M + 8) / 8; i += 32) ((uint4*)upos)[i] = make_uint4(0, 0, 0, 0);
    if (lane < SS_WORDS) sst[lane] = 0;
    __syncwarp();

    Ctl* ctl = A.ctl;
    const bool notrunc = MODE == MODE_WRITE ? ctl->notrunc != 0 : true;
    const u64 X = MODE == MODE_WRITE ? ctl->X : 0;
    const bool fast_graph = !A.no_fast && A.g.max_coef < kSmallCoef;
    KeyOut ko; ko.base = 0; ko.left = 0;
    // a warp owns A.ppw (<= kParentsPerWarp) consecutive parents; the grid covers the level and the block scheduler evens out the
    // very different costs of parents (skipped / first visit over a hub / revisit)
    const u64 p0 = ((u64)blockIdx.x * (blockDim.x >> 5) + wib) * A.ppw;
    const u64 p1 = min(p0 + A.ppw, A.n_cur);

#pragma unroll 1
    for (u64 p = p0; p < p1; ++p) {
        if (MODE == MODE_WRITE && !notrunc && __ldcs(&A.pmin[p]) >= X) continue;   // no child of p survives the beam
        // ---- stage the parent: the first 32 16-byte chunks speculatively, the rest once the header is known
        const uint4* src = (const uint4*)(A.cur + (__ldcs(&A.cur_off[p]) << 4));
        const uint4 first16 = __ldcs(src + lane);   // the buffers end in 512 spare bytes
        const u32 hdr = __shfl_sync(FULL, first16.x, 0);
        const int ns = (int)(hdr & 0xffffu), nv = (int)(hdr >> 16);
        const int nu = (int)__shfl_sync(FULL, first16.y, 0);
        const u32 nch = entry_bytes((u32)ns, (u32)nv, (u32)nu) / 16;
        if ((u32)lane < nch) stage[lane] = first16;
        #pragma unroll 1
        for (u32 c = lane + 32; c < nch; c += 32) stage[c] = __ldcs(src + c);   // streaming: the frontier must not evict the graph from L1
        __syncwarp();
        const u64 Phs = ((const u64*)stage)[1], Phv = ((const u64*)stage)[2], Pbig = ((const u64*)stage)[3];
        const i64* flux = (const i64*)(gs + kHdr);
        const u64* vis = (const u64*)(flux + ns);
        const i64* ef = (const i64*)(vis + nv);
        const u16* arc = (const u16*)(ef + nu);
        const u16* efmet = arc + ns;

        // ---- support bitset, EF index table, PROC0: lowest unbalanced metabolite i* (reading G12)
        #pragma unroll 1
        for (int t = lane; t < ns; t += 32) { const u32 a = arc[t]; atomicOr(&sbits[a >> 5], 1u << (a & 31)); }
        u32 best = 0xffffffffu;
        #pragma unroll 1
        for (int t = lane; t < nu; t += 32) {
            const u32 i = efmet[t];
            upos[i] = (u16)(t + 1);
            best = min(best, (i << 16) | (u32)t);
        }
        best = __reduce_min_sync(FULL, best);
        if (lane == 0) { sst[SS_KC] = 0; sst[SS_KC + 2] = 0; }
        __syncwarp();
        const int istar = (int)(best >> 16);
        const i64 E = ef[best & 0xffffu];
        const bool fwd = E > 0;
        const u64 absE = abs64(E);
        auto ef_of = [&](int met) -> i64 { const u32 u = upos[met]; return u ? ef[u - 1] : 0; };
        if (MODE != MODE_WRITE && lane == 0) { sst[SS_EXPANDED]++; sst[SS_BYTES] += algo_entry_bytes((u32)ns, (u32)nv); }
        if (MODE == MODE_WRITE && lane == 0) sst[SS_WRITE_PARENTS]++;
        u64 kmin = ~0ULL;   // smallest key among the active children of p (count pass)
        // visited?
        int vk = -1;
        #pragma unroll 1
        for (int base = 0; base < nv && vk < 0; base += 32) {
            const int u = base + lane;
            const u32 hit = __ballot_sync(FULL, u < nv && (int)((vis[u] >> 32) & 0xffffu) == istar);
            if (hit) vk = base + __ffs(hit) - 1;
        }
        const bool firstv = vk < 0;
        if (MODE != MODE_WRITE && lane == 0) { sst[SS_FIRST] += firstv; sst[SS_SATURATED] += ns >= A.D; }
        const int in0 = __ldg(&A.g.in_ptr[istar]), nI = __ldg(&A.g.in_ptr[istar + 1]) - in0;
        const int out0 = __ldg(&A.g.out_ptr[istar]), nO = __ldg(&A.g.out_ptr[istar + 1]) - out0;

        // ---- what to branch over: the OR-alternatives of i* (first visit) or the single Eq 4 / Eq 5 bump (revisit)
        const int2* alist = nullptr;
        int alen = 0, prim = -1;
        int r_a = 0, r_c = 1, r_sign = +1;
        u64 rec = 0, r_newrec = 0;
        if (firstv) {
            // PROC1 / PROC1' (Eq 3; readings G1, G13, G14, G15, G22)
            if (nv >= A.V) {
                if (MODE != MODE_WRITE && lane == 0) sst[SS_VISITED]++;
            } else {
                // primary on the side the flux arrives from: lowest arc of that side in the support (G13)
                const int2* plist = fwd ? A.g.in_e + in0 : A.g.out_e + out0;
                const int plen = fwd ? nI : nO;
                #pragma unroll 1
                for (int base = 0; base < plen && prim < 0; base += 32) {
                    const int q = base + lane;
                    const int pa = q < plen ? __ldg(&plist[q]).x : -1;
                    const u32 bal = __ballot_sync(FULL, pa >= 0 && sbit(sbits, pa));
                    if (bal) prim = __shfl_sync(FULL, pa, __ffs(bal) - 1);
                }
                alist = fwd ? A.g.out_e + out0 : A.g.in_e + in0;
                alen = fwd ? nO : nI;
            }
        } else {
            // PROC2-4 (readings G2-G5)
            rec = vis[vk];
            const int cntv = (int)(rec >> 48) + 1;
            if (cntv > A.max_loop) {
                if (MODE != MODE_WRITE && lane == 0) sst[SS_NOTEFM]++;
            } else {
                const int PI = (int)((rec >> 16) & 0xffffu), PO = (int)(rec & 0xffffu);
                int lPI = -1, lPO = -1, cPI = 0, cPO = 0;
                #pragma unroll 1
                for (int q = lane; q < nI; q += 32) { const int2 e = __ldg(&A.g.in_e[in0 + q]); if (e.x == PI) { lPI = q; cPI = e.y; } }
                #pragma unroll 1
                for (int q = lane; q < nO; q += 32) { const int2 e = __ldg(&A.g.out_e[out0 + q]); if (e.x == PO) { lPO = q; cPO = e.y; } }
                lPI = __reduce_max_sync(FULL, lPI); cPI = __reduce_max_sync(FULL, cPI);
                lPO = __reduce_max_sync(FULL, lPO); cPO = __reduce_max_sync(FULL, cPO);
                // Def 11: forward PO ~ SI, backward PI ~ SO, secondary = any arc of that side in the support (G5)
                bool dep = false;
                const i64 doff = __ldg(&A.g.dep_off[istar]);
                if (fwd) {
                    #pragma unroll 1
                    for (int q = lane; q < nI; q += 32) {
                        const i64 b = doff + (i64)lPO * nI + q;
                        dep = dep || (sbit(sbits, __ldg(&A.g.in_e[in0 + q]).x) && ((__ldg(&A.g.dep_bits[b >> 5]) >> (b & 31)) & 1u));
                    }
                } else {
                    #pragma unroll 1
                    for (int q = lane; q < nO; q += 32) {
                        const i64 b = doff + (i64)q * nI + lPI;
                        dep = dep || (sbit(sbits, __ldg(&A.g.out_e[out0 + q]).x) && ((__ldg(&A.g.dep_bits[b >> 5]) >> (b & 31)) & 1u));
                    }
                }
                dep = __any_sync(FULL, dep);
                if (fwd) { if (!dep) { r_a = PO; r_c = cPO; r_sign = +1; } else { r_a = PI; r_c = cPI; r_sign = -1; } }   // Eq 4 / Eq 5
                else     { if (!dep) { r_a = PI; r_c = cPI; r_sign = +1; } else { r_a = PO; r_c = cPO; r_sign = -1; } }
                r_newrec = vis_pack((u32)istar, (u32)PI, (u32)PO, (u32)cntv);
                alen = 1;
            }
        }
        const bool fastP = firstv && fast_graph && Pbig < kSmall;
        int n_adm = 0;
        #pragma unroll 1
        for (int base = 0; base < alen; base += 32) {
            const int q = base + lane;
            int a = -1, c = 1;
            bool adm = false, insup = false;
            if (firstv) {
                if (q < alen) {
                    const int2 e = __ldg(&alist[q]);
                    a = e.x; c = e.y;
                    const int tw = __ldg(&A.g.twin[a]);
                    insup = sbit(sbits, a);
                    adm = !(tw >= 0 && sbit(sbits, tw)) && (insup || ns < A.D);
                }
            } else if (lane == 0) {
                a = r_a; c = r_c; adm = true; insup = true;   // PI / PO are arcs of the support
            }
            if (MODE != MODE_WRITE && lane == 0) sst[SS_ROUNDS]++;
            const u32 adm_m = __ballot_sync(FULL, adm);
            if (adm_m == 0) continue;
            n_adm += __popc(adm_m);
            // ---- lane-parallel evaluation: new arc, small integers => no overflow, no common factor
            const bool fast = adm && !insup && fastP;
            const u32 fast_m = __ballot_sync(FULL, fast);
            u32 k = 1; u64 d = absE;
            int nu2 = nu;
            u64 hs2 = 0, hv2 = 0, key = 0;
            if (fast_m) {
                if (fast) {
                    if (c != 1) scale_small(absE, (u32)c, k, d);
                    const int q1 = __ldg(&A.g.col_ptr[a + 1]);
                    #pragma unroll 1
                    for (int qq = __ldg(&A.g.col_ptr[a]); qq < q1; ++qq) {
                        const int2 e = __ldg(&A.g.col[qq]);
                        const i64 efp = ef_of(e.x);
                        const i64 x = (i64)k * efp + (i64)d * (i64)e.y;   // |.| < 2^60 + 2^60
                        nu2 += (int)(x != 0) - (int)(efp != 0);
                    }
                }
                u64 hsb = Phs;
                u32 need = __ballot_sync(FULL, fast && k > 1);
                #pragma unroll 1
                while (need) {
                    const u32 kk = __shfl_sync(FULL, k, __ffs(need) - 1);
                    u64 s;
                    if ((u64)kk == sst[SS_KC]) s = sst[SS_KC + 1];
                    else if ((u64)kk == sst[SS_KC + 2]) s = sst[SS_KC + 3];
                    else {
                        s = 0;
                        #pragma unroll 1
                        for (int t = lane; t < ns; t += 32) s += arc_term_t(A.g, (u32)arc[t], (u64)kk * (u64)flux[t]);
                        s = w_sum(s);
                        __syncwarp();
                        if (lane == 0) { sst[SS_KC + 2] = sst[SS_KC]; sst[SS_KC + 3] = sst[SS_KC + 1]; sst[SS_KC] = kk; sst[SS_KC + 1] = s; }
                        __syncwarp();
                    }
                    const bool same = fast && k == kk;
                    if (same) hsb = s;
                    need &= ~__ballot_sync(FULL, same);
                }
                if (fast) {
                    const u64 newrec = vis_pack((u32)istar, (u32)(fwd ? prim : a), (u32)(fwd ? a : prim), 0u);
                    hs2 = hsb + arc_term_t(A.g, (u32)a, d);
                    hv2 = Phv + vis_term(newrec);
                    key = beam_key((u32)nu2, mix64(hs2 + hv2));
                }
            }
            const u32 done_m = __ballot_sync(FULL, fast && nu2 == 0);
            if (MODE != MODE_WRITE && lane == 0) {
                const int nf = __popc(fast_m);
                sst[SS_CHILDREN] += nf; sst[SS_BYTES] += 8 * nf; sst[SS_DONE] += __popc(done_m);
            }
            u32 keep_m;
            if (MODE == MODE_COUNT) {
                const bool act = fast && nu2 != 0;
                if (lane == 0) sst[SS_ACTIVE] += __popc(fast_m & ~done_m);
                ko.push(A, lane, act, key);
                if (act) kmin = min(kmin, key);
                keep_m = done_m;
            } else if (MODE == MODE_WRITE) {
                keep_m = __ballot_sync(FULL, fast && nu2 != 0 && (notrunc || key < X));
            } else {
                keep_m = fast_m;
            }
            // ---- one child at a time: general evaluation (arc of the support, large integers) and / or materialisation
            const u32 slow_m = adm_m & ~fast_m;
            u32 work_m = keep_m | slow_m;
            #pragma unroll 1
            while (work_m) {
                const int l = __ffs(work_m) - 1;
                work_m &= work_m - 1;
                const bool general = (slow_m >> l) & 1u;
                // warp-uniform description of the child relative to its parent
                const int ca = __shfl_sync(FULL, a, l);
                u64 ck = __shfl_sync(FULL, k, l);        // scale
                u64 cd = w_bcast(d, l);                  // |E| / gcd(|E|, c)
                u64 cT = cd;                             // un-normalised new flux of arc ca
                u64 cg = 1;                              // common divisor of the un-normalised child
                u64 chs = w_bcast(hs2, l), chv = w_bcast(hv2, l);
                int cnu = __shfl_sync(FULL, nu2, l);
                int csign = +1, cia = -1;
                bool cin = false, keep = true;
                u64 newrec = firstv ? vis_pack((u32)istar, (u32)(fwd ? prim : ca), (u32)(fwd ? ca : prim), 0u) : r_newrec;
                const int qa0 = __ldg(&A.g.col_ptr[ca]), qa1 = __ldg(&A.g.col_ptr[ca + 1]);
                if (general) {
                    // bump(f, a, sign*|E|/c) of SURVEY.md 8(c) O6 with the whole warp
                    const int cc = __shfl_sync(FULL, c, l);
                    csign = firstv ? +1 : r_sign;
                    const u64 gg = cc == 1 ? 1ULL : gcd64(absE, (u64)cc);
                    ck = gg == 1 ? (u64)cc : (u64)cc / gg;
                    cd = gg == 1 ? absE : absE / gg;
                    cin = sbit(sbits, ca);
                    if (cin) {   // position of the arc in the sorted support
                        #pragma unroll 1
                        for (int b2 = 0; b2 < ns && cia < 0; b2 += 32) {
                            const int t = b2 + lane;
                            const u32 hit = __ballot_sync(FULL, t < ns && arc[t] == ca);
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
                    if (bigk) {   // exact: the largest flux among t != ia (a new arc carries d <= |E| <= 2^62)
                        u64 mx = 0;
                        #pragma unroll 1
                        for (int t = lane; t < ns; t += 32) if (t != cia) mx = max(mx, (u64)flux[t]);
                        mx = w_max(mx);
                        ovf = ovf || umul_gt_guard(ck, mx);
                    }
                    int status = ovf ? CH_OVERFLOW : (nonpos ? CH_NONPOS : CH_OK);   // Prop 3, G11
                    if (status == CH_OK) {
                        // extra fluxes of the un-normalised child: EF'_i = k EF_i + sign d s_ia (Eq 2 on the scaled fluxes)
                        bool ovf2 = false;
                        if (bigk) {   // exact sweep over the unbalanced metabolites outside col(a)
                            #pragma unroll 1
                            for (int t = lane; t < nu; t += 32) {
                                const int i = efmet[t];
                                bool in_a = false;
                                #pragma unroll 1
                                for (int r = qa0; r < qa1; ++r) in_a = in_a || __ldg(&A.g.col[r]).x == i;
                                if (!in_a) ovf2 = ovf2 || abs_gt_guard(mul_s((i64)ck, ef[t]));
                            }
                        }
                        int delta = 0;
                        #pragma unroll 1
                        for (int qq = qa0 + lane; qq < qa1; qq += 32) {
                            const int2 e = __ldg(&A.g.col[qq]);
                            const i64 efp = ef_of(e.x);
                            const S128 x = add_s(mul_s((i64)ck, efp), mul_s(csign > 0 ? (i64)cd : -(i64)cd, (i64)e.y));
                            ovf2 = ovf2 || abs_gt_guard(x);
                            delta += (int)((x.lo | (u64)x.hi) != 0) - (int)(efp != 0);
                        }
                        if (__any_sync(FULL, ovf2)) status = CH_OVERFLOW;
                        else cnu = nu + __reduce_add_sync(FULL, delta);
                    }
                    if (status != CH_OK) {
                        if (MODE != MODE_WRITE && lane == 0) sst[status == CH_OVERFLOW ? SS_OVF : SS_NONPOS]++;
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
                        for (int t = lane; t < ns; t += 32) {
                            if (t == cia) continue;
                            const u64 x = ck * (u64)flux[t];   // <= 2^62 (no overflow was found above)
                            if (narrow) {
                                const u32 r32 = (u32)r;
                                r = gcd32(r32, (x >> 32) == 0 ? (u32)x % r32 : (u32)(x % (u64)r32));
                            } else r = gcd64(r, x);
                        }
                        if (!__any_sync(FULL, r == 1)) cg = w_gcd(r, narrow);
                    }
                    if (ck == 1 && cg == 1) {
                        chs = Phs + arc_term_t(A.g, (u32)ca, cT) - (cin ? arc_term_t(A.g, (u32)ca, (u64)flux[cia]) : 0ULL);
                    } else {
                        chs = 0;
                        #pragma unroll 1
                        for (int t = lane; t < ns; t += 32) {
                            u64 F = t == cia ? cT : ck * (u64)flux[t];
                            if (cg > 1) F /= cg;
                            chs += arc_term_t(A.g, (u32)arc[t], F);
                        }
                        chs = w_sum(chs);
                        if (!cin) chs += arc_term_t(A.g, (u32)ca, cT);
                    }
                    chv = Phv + vis_term(newrec) - (firstv ? 0ULL : vis_term(rec));
                    // account for the child, classify it, decide whether it is materialised in this pass
                    const bool cdone = cnu == 0;
                    if (MODE != MODE_WRITE && lane == 0) { sst[SS_CHILDREN]++; sst[SS_GENERAL]++; sst[SS_BYTES] += 8; if (cdone) sst[SS_DONE]++; }
                    if (cdone) keep = MODE != MODE_WRITE;   // balanced children are written where they are first seen
                    else {
                        const u64 ckey = beam_key((u32)cnu, mix64(chs + chv));
                        if (MODE == MODE_COUNT) {
                            if (lane == 0) sst[SS_ACTIVE]++;
                            ko.push(A, lane, lane == 0, ckey);
                            kmin = min(kmin, ckey);
                            keep = false;
                        } else keep = MODE == MODE_DIRECT || notrunc || ckey < X;
                    }
                }
                if (!keep) continue;
                // ---- place: a candidate slot (balanced) or a packed entry of the next frontier
                const bool to_cand = cnu == 0;
                const int n2 = ns + (cin ? 0 : 1);
                const int nv2 = to_cand ? 0 : nv + (firstv ? 1 : 0);
                const int nu2c = to_cand ? 0 : cnu;
                if (lane == 0) sst[SS_BYTES] += algo_entry_bytes((u32)n2, (u32)(nv + (firstv ? 1 : 0)));
                unsigned char* dst;
                if (to_cand) {
                    u64 slot = 0;
                    if (lane == 0) slot = atomicAdd(&ctl->n_cand, 1ULL);
                    slot = w_bcast(slot, 0);
                    if (slot >= A.max_cand) { if (lane == 0) atomicOr(&ctl->error, (u32)ERR_CAND); continue; }
                    dst = A.cand + slot * A.cand_stride;
                } else {
                    const u64 units = entry_bytes((u32)n2, (u32)nv2, (u32)nu2c) >> 4;
                    u64 old = 0;
                    if (lane == 0) old = atomicAdd(&ctl->n_next, (1ULL << kAllocShift) | units);
                    old = w_bcast(old, 0);
                    const u64 slot = old >> kAllocShift, off = old & kAllocUnitMask;
                    if (slot >= A.max_frontier || off + units > A.frontier_units) {
                        if (lane == 0) atomicOr(&ctl->error, (u32)ERR_FRONTIER);
                        continue;
                    }
                    if (lane == 0) A.nxt_off[slot] = off;
                    dst = A.nxt + (off << 4);
                }
                // ---- write
                int ins = 0;   // a new arc goes where the ascending order puts it
                if (!cin)
                    #pragma unroll 1
                    for (int b2 = 0; b2 < ns; b2 += 32) {
                        const int t = b2 + lane;
                        ins += __popc(__ballot_sync(FULL, t < ns && (int)arc[t] < ca));
                    }
                // The child is assembled in shared memory and leaves the SM as whole 16-byte chunks, so HBM sees full
                // sectors (element-wise stores into fresh lines make the L2 fill every sector from DRAM first).  An
                // entry larger than the assembly buffer is written in place.
                const u32 cbytes = entry_bytes((u32)n2, (u32)nv2, (u32)nu2c);
                const bool via_smem = cbytes <= A.sm_out_bytes;
                unsigned char* wb = via_smem ? gs + A.sm_out : dst;
                i64* flux2 = (i64*)(wb + kHdr);
                u64* vis2 = (u64*)(flux2 + n2);
                i64* ef2 = (i64*)(vis2 + nv2);
                u16* arc2 = (u16*)(ef2 + nu2c);
                u16* efmet2 = arc2 + n2;
                u64 mx = cin ? 0ULL : cT;   // a new arc never comes with a common divisor
                #pragma unroll 1
                for (int t = lane; t < ns; t += 32) {
                    u64 F = t == cia ? cT : ck * (u64)flux[t];
                    if (cg > 1) F /= cg;
                    const int pos = t + ((!cin && t >= ins) ? 1 : 0);
                    flux2[pos] = (i64)F;
                    arc2[pos] = arc[t];
                    mx = max(mx, F);
                }
                if (!cin && lane == 0) { flux2[ins] = (i64)cT; arc2[ins] = (u16)ca; }
                if (!to_cand) {
                    #pragma unroll 1
                    for (int u = lane; u < nv; u += 32) vis2[u] = (!firstv && u == vk) ? newrec : vis[u];
                    if (firstv && lane == 0) vis2[nv] = newrec;
                    // EF list of the child: EF' = (k EF + sign d s_.a) / g over the parent's list, then the metabolites
                    // of col(a) that were balanced in the parent.  The evaluation above (or the bounds of the fast path)
                    // established that nothing exceeds 2^62, so the wrapping 64-bit arithmetic is exact.
                    const u64 sd = csign > 0 ? cd : (u64)0 - cd;
                    int wbase = 0;
                    #pragma unroll 1
                    for (int t0 = 0; t0 < nu; t0 += 32) {
                        const int t = t0 + lane;
                        const bool valid = t < nu;
                        i64 x = 0;
                        int met = 0;
                        if (valid) {
                            met = efmet[t];
                            i64 s = 0;
                            #pragma unroll 1
                            for (int qq = qa0; qq < qa1; ++qq) { const int2 e = __ldg(&A.g.col[qq]); if (e.x == met) s = e.y; }
                            x = (i64)(ck * (u64)ef[t] + sd * (u64)s);
                            if (cg > 1) x /= (i64)cg;
                        }
                        const u32 nz = __ballot_sync(FULL, valid && x != 0);
                        if (valid && x != 0) {
                            const int pos = wbase + __popc(nz & lt);
                            ef2[pos] = x; efmet2[pos] = (u16)met;
                            mx = max(mx, abs64(x));
                        }
                        wbase += __popc(nz);
                    }
                    #pragma unroll 1
                    for (int q0 = qa0; q0 < qa1; q0 += 32) {
                        const int qq = q0 + lane;
                        int2 e = make_int2(0, 0);
                        bool only = false;
                        if (qq < qa1) { e = __ldg(&A.g.col[qq]); only = upos[e.x] == 0; }
                        const u32 m = __ballot_sync(FULL, only);
                        if (only) {
                            i64 x = (i64)(sd * (u64)(i64)e.y);
                            if (cg > 1) x /= (i64)cg;
                            const int pos = wbase + __popc(m & lt);
                            ef2[pos] = x; efmet2[pos] = (u16)e.x;
                            mx = max(mx, abs64(x));
                        }
                        wbase += __popc(m);
                    }
                    mx = w_max(mx);
                }
                if (lane == 0) {
                    uint4* h4 = (uint4*)wb;
                    h4[0] = make_uint4((u32)n2 | ((u32)nv2 << 16), (u32)nu2c, (u32)chs, (u32)(chs >> 32));
                    h4[1] = make_uint4((u32)chv, (u32)(chv >> 32), (u32)mx, (u32)(mx >> 32));
                }
                if (via_smem) {
                    __syncwarp();
                    const uint4* o4 = (const uint4*)(gs + A.sm_out);
                    #pragma unroll 1
                    for (u32 c = lane; c < cbytes / 16; c += 32) __stcs((uint4*)dst + c, o4[c]);
                    __syncwarp();
                }
            }
        }
        if (MODE != MODE_WRITE && firstv && nv < A.V && n_adm == 0 && lane == 0) sst[SS_DEAD]++;   // no admissible alternative
        if (MODE == MODE_COUNT) {
            kmin = w_min(kmin);
            if (lane == 0) A.pmin[p] = kmin;
        }
        // ---- restore the shared tables to zero for the next parent
        __syncwarp();
        #pragma unroll 1
        for (int t = lane; t < ns; t += 32) sbits[arc[t] >> 5] = 0;
        #pragma unroll 1
        for (int t = lane; t < nu; t += 32) upos[efmet[t]] = 0;
        __syncwarp();
    }
    if (MODE == MODE_COUNT) ko.finish(A, lane);
    __syncwarp();
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
        if (sst[SS_WRITE_PARENTS]) atomicAdd(&st[ST_WRITE_PARENTS], sst[SS_WRITE_PARENTS]);
    }
}

__global__ void k_level_begin(Ctl* ctl) {
    ctl->n_next = 0; ctl->n_keys = 0; ctl->n_slots = 0; ctl->lvl_done = 0; ctl->lvl_children = 0; ctl->lvl_expanded = 0;
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
    size_t off = align16(a.max_entry);   // staging holds the largest entry
    a.sm_sbits = (u32)off; off = align16(off + (size_t)a.g.W32 * 4);
    a.sm_upos = (u32)off;  off = align16(off + (size_t)a.g.M * 2 + 16);   // zeroed in 16-byte chunks
    a.sm_misc = (u32)off;  off = align16(off + (size_t)SS_WORDS * 8);
    a.sm_out_bytes = a.max_entry < 2048u ? a.max_entry : 2048u;   // child assembly buffer (larger children: in place)
    a.sm_out = (u32)off;   off = align16(off + a.sm_out_bytes);
    a.sm_group = (u32)off;
}

// key slots the count pass can leave unused: every warp of the largest grid may strand one chunk
// every warp may strand one chunk of key slots; a warp covers kParentsPerWarp parents
u64 expand_key_slack(u64 max_parents) { return (max_parents / kParentsPerWarp + 16384) * kKeyChunk; }

template <int MODE>
static cudaError_t launch_t(const ExpandArgs& a, int sm_count, cudaStream_t s) {
    // warps per block: as many as fit beside the per-warp staging (huge networks fall back to fewer warps)
    int warps = kWarps;
    while (warps > 1 && (size_t)a.sm_group * warps > 200 * 1024) warps >>= 1;
    const size_t smem = (size_t)a.sm_group * warps;
    if (smem > 227 * 1024) return cudaErrorInvalidValue;
    static int bps_cache[kWarps + 1] = {0};
    static size_t smem_cache[kWarps + 1] = {0};
    if (bps_cache[warps] == 0 || smem_cache[warps] != smem) {
        cudaError_t e = cudaFuncSetAttribute(k_expand<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
        if (e != cudaSuccess) return e;
        int bps = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, k_expand<MODE>, warps * 32, smem);
        if (e != cudaSuccess) return e;
        bps_cache[warps] = bps < 1 ? 1 : bps;
        smem_cache[warps] = smem;
    }
    // small levels: fewer parents per warp so that every SM still gets its share of warps
    u64 ppw = a.n_cur / ((u64)sm_count * 32);
    ppw = ppw < 1 ? 1 : (ppw > (u64)kParentsPerWarp ? (u64)kParentsPerWarp : ppw);
    ExpandArgs a2 = a;
    a2.ppw = (u32)ppw;
    const u64 per_block = (u64)warps * ppw;
    const u64 need = (a.n_cur + per_block - 1) / per_block;
    if (need > 0x7fffffffULL) return cudaErrorInvalidValue;
    unsigned grid = (unsigned)(need ? need : 1);
    k_expand<MODE><<<grid, warps * 32, smem, s>>>(a2);
    return cudaGetLastError();
}

cudaError_t launch_expand(int mode, const ExpandArgs& a, int sm_count, cudaStream_t s) {
    if (mode == MODE_COUNT) return launch_t<MODE_COUNT>(a, sm_count, s);
    if (mode == MODE_WRITE) return launch_t<MODE_WRITE>(a, sm_count, s);
    return launch_t<MODE_DIRECT>(a, sm_count, s);
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
