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
constexpr int kBlock = 128;
constexpr int kWarps = kBlock / 32;
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

// ------------------------------------------------------------------ per-parent context (warp-uniform)
struct Parent {
    int n_supp, n_vis, n_unb;
    const i64* flux; const u64* vis; const i64* ef; const u16* arc; const u16* efmet;   // shared-memory staging
    u32* sbits;   // support bitset over arcs
    u32* ubits;   // bitset over metabolites: member of the EF list
    u64 hs, hv, big;
    int istar;
    i64 E;
};
struct Child {          // warp-uniform description of one child relative to its parent
    int status; bool done;
    int a; bool in_supp; int ia; int sign;
    u64 k, g2, T, d;    // scale, common divisor, un-normalised new flux of arc a, |E| / gcd(|E|, c)
    u64 hs, hv;         // hash sums of the child state
    int n_unb;
};

__device__ __forceinline__ bool sbit(const u32* bits, int a) { return (bits[a >> 5] >> (a & 31)) & 1u; }

// EF_met of the parent: zero unless met is in the list
__device__ __forceinline__ i64 ef_lookup(const Parent& P, int met) {
    if (met == P.istar) return P.E;
    if (!sbit(P.ubits, met)) return 0;
    for (int t = 0; t < P.n_unb; ++t) if ((int)P.efmet[t] == met) return P.ef[t];
    return 0;
}

// General routine: evaluate the child bump(f, a, sign*|E|/c) with the whole warp.
//   first: new visited record newrec; otherwise record oldrec is replaced by newrec
__device__ __noinline__ void eval_child(const DevGraph& g, const Parent& P, int lane, int a, int c, int sign,
                                        bool first, u64 oldrec, u64 newrec, Child& ch) {
    const u64 absE = abs64(P.E);
    const u64 gg = c == 1 ? 1ULL : gcd64(absE, (u64)c);
    const u64 k = gg == 1 ? (u64)c : (u64)c / gg;
    const u64 d = gg == 1 ? absE : absE / gg;
    ch.a = a; ch.k = k; ch.g2 = 1; ch.d = d; ch.sign = sign;
    ch.in_supp = sbit(P.sbits, a);
    int ia = -1;
    if (ch.in_supp) {   // position of a in the sorted support
        for (int base = 0; base < P.n_supp && ia < 0; base += 32) {
            const int t = base + lane;
            const u32 hit = __ballot_sync(FULL, t < P.n_supp && P.arc[t] == a);
            if (hit) ia = base + __ffs(hit) - 1;
        }
    }
    ch.ia = ia;
    // scaled fluxes F_t = k f_t, F_a = k f_a +- d: overflow first, then non-positive (order of the definition, O6).
    // P.big >= every flux and every |EF| of the parent: products below the guard with it need no exact sweep.
    const bool bigk = k > 1 && umul_gt_guard(k, P.big);
    bool ovf = false, nonpos = false;
    u64 T = d;
    if (ch.in_supp) {
        const u64 fa = (u64)P.flux[ia];
        const u64 lo = k * fa, hi = __umul64hi(k, fa);
        if (sign > 0) {
            T = lo + d;
            const u64 hi2 = hi + (T < lo);
            ovf = hi2 != 0 || T > EFM_GUARD;
        } else {
            if (hi == 0 && lo <= d) { nonpos = true; T = 0; }           // k f_a - d <= 0
            else { T = lo - d; const u64 hi2 = hi - (lo < d); ovf = hi2 != 0 || T > EFM_GUARD; }
        }
    }
    if (bigk) {   // exact: the largest flux among t != ia (the new arc carries d <= |E| <= 2^62)
        u64 mx = 0;
        for (int t = lane; t < P.n_supp; t += 32) if (t != ia) mx = max(mx, (u64)P.flux[t]);
        mx = w_max(mx);
        ovf = ovf || umul_gt_guard(k, mx);
    }
    ch.T = T;
    if (ovf) { ch.status = CH_OVERFLOW; return; }
    if (nonpos) { ch.status = CH_NONPOS; return; }   // Prop 3, reading G11
    // extra fluxes of the un-normalised child: EF'_i = k EF_i + sign d s_ia  (Eq 2 on the scaled fluxes)
    const int qa0 = __ldg(&g.col_ptr[a]), qa1 = __ldg(&g.col_ptr[a + 1]);
    bool ovf2 = false;
    if (bigk) {   // exact sweep over the unbalanced metabolites outside col(a)
        for (int t = lane; t < P.n_unb; t += 32) {
            const int i = P.efmet[t];
            bool in_a = false;
            for (int r = qa0; r < qa1; ++r) in_a = in_a || __ldg(&g.col[r]).x == i;
            if (!in_a) ovf2 = ovf2 || abs_gt_guard(mul_s((i64)k, P.ef[t]));
        }
    }
    int delta = 0;
    for (int q = qa0 + lane; q < qa1; q += 32) {
        const int2 e = __ldg(&g.col[q]);
        const i64 efp = ef_lookup(P, e.x);
        S128 x = add_s(mul_s((i64)k, efp), mul_s(sign > 0 ? (i64)d : -(i64)d, (i64)e.y));
        ovf2 = ovf2 || abs_gt_guard(x);
        delta += (int)((x.lo | (u64)x.hi) != 0) - (int)(efp != 0);
    }
    if (__any_sync(FULL, ovf2)) { ch.status = CH_OVERFLOW; return; }
    delta = __reduce_add_sync(FULL, delta);
    ch.status = CH_OK;
    ch.n_unb = P.n_unb + delta;
    ch.done = ch.n_unb == 0;
    // gcd normalisation (reading G10).  A new arc cannot introduce a common factor: gcd_t(k f_t) = k and gcd(k, d) = 1.
    // An arc of the support: g = gcd(k G, T) with G the gcd of the other fluxes; another flux equal to 1 gives G = 1
    // and g = gcd(k, k f_a +- d) = gcd(k, d) = 1 without any gcd.
    if (ch.in_supp && T != 1) {
        bool one = false;
        for (int t = lane; t < P.n_supp; t += 32) one = one || (t != ia && P.flux[t] == 1);
        if (!__any_sync(FULL, one)) {
            const bool narrow = P.big < (1ULL << 32);
            u64 G = 0;
            for (int t = lane; t < P.n_supp; t += 32)
                if (t != ia) G = narrow ? (u64)gcd32((u32)G, (u32)P.flux[t]) : gcd64(G, (u64)P.flux[t]);
            G = w_gcd(G, narrow);
            ch.g2 = gcd64(k * G, T);   // k G <= k fmax <= 2^62
        }
    }
    u64 hs;
    if (k == 1 && ch.g2 == 1) {
        hs = P.hs + arc_term_t(g, (u32)a, T) - (ch.in_supp ? arc_term_t(g, (u32)a, (u64)P.flux[ia]) : 0ULL);
    } else {
        hs = 0;
        for (int t = lane; t < P.n_supp; t += 32) {
            u64 F = t == ia ? T : k * (u64)P.flux[t];
            if (ch.g2 > 1) F /= ch.g2;
            hs += arc_term_t(g, (u32)P.arc[t], F);
        }
        hs = w_sum(hs);
        if (!ch.in_supp) hs += arc_term_t(g, (u32)a, T);
    }
    ch.hs = hs;
    ch.hv = P.hv + vis_term(newrec) - (first ? 0ULL : vis_term(oldrec));
}

// Write the child into a packed frontier entry (or a candidate slot: no visited records, no EF list).
__device__ __forceinline__ void write_child(const DevGraph& g, unsigned char* dst, const Parent& P, const Child& ch,
                                            int lane, bool first, int vk, u64 newrec, bool to_cand) {
    const int n2 = P.n_supp + (ch.in_supp ? 0 : 1);
    const int nv2 = to_cand ? 0 : P.n_vis + (first ? 1 : 0);
    const int nu2 = to_cand ? 0 : ch.n_unb;
    const u32 lt = (1u << lane) - 1u;
    int ins = 0;   // a new arc goes where the ascending order puts it
    if (!ch.in_supp)
        for (int base = 0; base < P.n_supp; base += 32) {
            const int t = base + lane;
            ins += __popc(__ballot_sync(FULL, t < P.n_supp && (int)P.arc[t] < ch.a));
        }
    i64* flux2 = (i64*)(dst + kHdr);
    u64* vis2 = (u64*)(flux2 + n2);
    i64* ef2 = (i64*)(vis2 + nv2);
    u16* arc2 = (u16*)(ef2 + nu2);
    u16* efmet2 = arc2 + n2;
    u64 mx = ch.in_supp ? 0ULL : (ch.g2 > 1 ? ch.T / ch.g2 : ch.T);
    for (int t = lane; t < P.n_supp; t += 32) {
        u64 F = t == ch.ia ? ch.T : ch.k * (u64)P.flux[t];
        if (ch.g2 > 1) F /= ch.g2;
        const int pos = t + ((!ch.in_supp && t >= ins) ? 1 : 0);
        flux2[pos] = (i64)F;
        arc2[pos] = P.arc[t];
        mx = max(mx, F);
    }
    if (!ch.in_supp && lane == 0) { flux2[ins] = (i64)ch.T; arc2[ins] = (u16)ch.a; }
    if (!to_cand) {
        for (int u = lane; u < P.n_vis; u += 32) vis2[u] = (!first && u == vk) ? newrec : P.vis[u];
        if (first && lane == 0) vis2[P.n_vis] = newrec;
        // EF list of the child: EF' = (k EF + sign d s_.a) / g over the parent's list, then the metabolites of col(a)
        // that were balanced in the parent.  eval_child / the fast path established that nothing exceeds 2^62, so
        // the wrapping 64-bit arithmetic below is exact.
        const int qa0 = __ldg(&g.col_ptr[ch.a]), qa1 = __ldg(&g.col_ptr[ch.a + 1]);
        const u64 sd = ch.sign > 0 ? ch.d : (u64)0 - ch.d;
        int base = 0;
        for (int t0 = 0; t0 < P.n_unb; t0 += 32) {
            const int t = t0 + lane;
            const bool valid = t < P.n_unb;
            i64 x = 0;
            int met = 0;
            if (valid) {
                met = P.efmet[t];
                i64 s = 0;
                for (int q = qa0; q < qa1; ++q) { const int2 e = __ldg(&g.col[q]); if (e.x == met) s = e.y; }
                x = (i64)(ch.k * (u64)P.ef[t] + sd * (u64)s);
                if (ch.g2 > 1) x /= (i64)ch.g2;
            }
            const u32 nz = __ballot_sync(FULL, valid && x != 0);
            if (valid && x != 0) {
                const int pos = base + __popc(nz & lt);
                ef2[pos] = x; efmet2[pos] = (u16)met;
                mx = max(mx, abs64(x));
            }
            base += __popc(nz);
        }
        for (int q0 = qa0; q0 < qa1; q0 += 32) {
            const int q = q0 + lane;
            int2 e = make_int2(0, 0);
            bool only = false;
            if (q < qa1) { e = __ldg(&g.col[q]); only = !sbit(P.ubits, e.x); }
            const u32 m = __ballot_sync(FULL, only);
            if (only) {
                i64 x = (i64)(sd * (u64)(i64)e.y);
                if (ch.g2 > 1) x /= (i64)ch.g2;
                const int pos = base + __popc(m & lt);
                ef2[pos] = x; efmet2[pos] = (u16)e.x;
                mx = max(mx, abs64(x));
            }
            base += __popc(m);
        }
        mx = w_max(mx);
    }
    if (lane == 0) {
        uint4* h4 = (uint4*)dst;
        h4[0] = make_uint4((u32)n2 | ((u32)nv2 << 16), (u32)nu2, (u32)ch.hs, (u32)(ch.hs >> 32));
        h4[1] = make_uint4((u32)ch.hv, (u32)(ch.hv >> 32), (u32)mx, (u32)(mx >> 32));
    }
}

// Per-warp chunked reservation of beam-key slots: one atomic per kKeyChunk keys instead of one per child.
struct KeyOut {
    u64 base; u32 left;
    __device__ __forceinline__ void push(const ExpandArgs& A, int lane, bool want, u64 key) {
        const u32 m = __ballot_sync(FULL, want);
        const u32 cnt = (u32)__popc(m);
        if (cnt == 0) return;
        if (cnt > left) {
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
        if (want) A.keys[base + __popc(m & ((1u << lane) - 1u))] = key;
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

template <int MODE>
__global__ void __launch_bounds__(kBlock) k_expand(const ExpandArgs A) {
    extern __shared__ __align__(16) unsigned char smem[];
    const DevGraph& g = A.g;
    const int lane = threadIdx.x & 31;
    const int wib = threadIdx.x >> 5;
    const u32 lt = (1u << lane) - 1u;
    unsigned char* gs = smem + (size_t)wib * A.sm_group;
    uint4* stage = (uint4*)gs;
    Parent P;
    P.sbits = (u32*)(gs + A.sm_sbits);
    P.ubits = (u32*)(gs + A.sm_ubits);
    for (int i = lane; i < g.W32; i += 32) P.sbits[i] = 0;
    for (int i = lane; i < g.M32; i += 32) P.ubits[i] = 0;
    __syncwarp();

    Ctl* ctl = A.ctl;
    const bool notrunc = MODE == MODE_WRITE ? ctl->notrunc != 0 : true;
    const u64 X = MODE == MODE_WRITE ? ctl->X : 0;
    const bool fast_graph = !A.no_fast && g.max_coef < kSmallCoef;

    // warp-uniform counters, flushed once per warp
    u64 s_expanded = 0, s_children = 0, s_done = 0, s_active = 0, s_dead = 0, s_notefm = 0, s_nonpos = 0, s_ovf = 0,
        s_visited = 0, s_bytes = 0;
    KeyOut ko; ko.base = 0; ko.left = 0;

    for (u64 p = (u64)blockIdx.x * kWarps + wib; p < A.n_cur; p += (u64)gridDim.x * kWarps) {
        if (MODE == MODE_WRITE && !notrunc && __ldg(&A.pmin[p]) >= X) continue;   // no child of p survives the beam
        // ---- stage the parent: the first 32 16-byte chunks speculatively, the rest once the header is known
        const uint4* src = (const uint4*)(A.cur + (__ldg(&A.cur_off[p]) << 4));
        const uint4 first = __ldg(src + lane);   // the buffers end in 512 spare bytes
        const u32 hdr = __shfl_sync(FULL, first.x, 0);
        P.n_supp = (int)(hdr & 0xffffu);
        P.n_vis = (int)(hdr >> 16);
        P.n_unb = (int)__shfl_sync(FULL, first.y, 0);
        const u32 nch = entry_bytes((u32)P.n_supp, (u32)P.n_vis, (u32)P.n_unb) / 16;
        if ((u32)lane < nch) stage[lane] = first;
        for (u32 c = lane + 32; c < nch; c += 32) stage[c] = __ldg(src + c);
        __syncwarp();
        P.hs = ((const u64*)stage)[1];
        P.hv = ((const u64*)stage)[2];
        P.big = ((const u64*)stage)[3];
        P.flux = (const i64*)(gs + kHdr);
        P.vis = (const u64*)(P.flux + P.n_supp);
        P.ef = (const i64*)(P.vis + P.n_vis);
        P.arc = (const u16*)(P.ef + P.n_unb);
        P.efmet = P.arc + P.n_supp;

        // ---- support bitset, unbalanced-metabolite bitset, PROC0: lowest unbalanced metabolite i* (reading G12)
        for (int t = lane; t < P.n_supp; t += 32) { const u32 a = P.arc[t]; atomicOr(&P.sbits[a >> 5], 1u << (a & 31)); }
        u32 best = 0xffffffffu;
        for (int t = lane; t < P.n_unb; t += 32) {
            const u32 i = P.efmet[t];
            atomicOr(&P.ubits[i >> 5], 1u << (i & 31));
            best = min(best, (i << 16) | (u32)t);
        }
        best = __reduce_min_sync(FULL, best);
        __syncwarp();
        const int cnt = P.n_unb;
        const int istar = (int)(best >> 16);
        P.istar = istar;
        P.E = P.ef[best & 0xffffu];
        {
            const bool fwd = P.E > 0;
            const u64 absE = abs64(P.E);
            if (MODE != MODE_WRITE) { s_expanded++; s_bytes += algo_entry_bytes((u32)P.n_supp, (u32)P.n_vis); }
            u64 kmin = ~0ULL;   // smallest key among the active children of p (count pass)
            // visited?
            int vk = -1;
            for (int base = 0; base < P.n_vis && vk < 0; base += 32) {
                const int u = base + lane;
                const u32 hit = __ballot_sync(FULL, u < P.n_vis && (int)((P.vis[u] >> 32) & 0xffffu) == istar);
                if (hit) vk = base + __ffs(hit) - 1;
            }
            const int in0 = __ldg(&g.in_ptr[istar]), nI = __ldg(&g.in_ptr[istar + 1]) - in0;
            const int out0 = __ldg(&g.out_ptr[istar]), nO = __ldg(&g.out_ptr[istar + 1]) - out0;

            // materialise one kept child (warp-uniform description)
            auto place = [&](const Child& ch, bool first, u64 newrec) {
                const int n2 = P.n_supp + (ch.in_supp ? 0 : 1), nv2 = P.n_vis + (first ? 1 : 0);
                s_bytes += algo_entry_bytes((u32)n2, (u32)nv2);
                unsigned char* dst;
                if (ch.done) {
                    u64 slot = 0;
                    if (lane == 0) slot = atomicAdd(&ctl->n_cand, 1ULL);
                    slot = w_bcast(slot, 0);
                    if (slot >= A.max_cand) { if (lane == 0) atomicOr(&ctl->error, (u32)ERR_CAND); return; }
                    dst = A.cand + slot * A.cand_stride;
                } else {
                    const u64 units = entry_bytes((u32)n2, (u32)nv2, (u32)ch.n_unb) >> 4;
                    u64 old = 0;
                    if (lane == 0) old = atomicAdd(&ctl->n_next, (1ULL << kAllocShift) | units);
                    old = w_bcast(old, 0);
                    const u64 slot = old >> kAllocShift, off = old & kAllocUnitMask;
                    if (slot >= A.max_frontier || off + units > A.frontier_units) {
                        if (lane == 0) atomicOr(&ctl->error, (u32)ERR_FRONTIER);
                        return;
                    }
                    if (lane == 0) A.nxt_off[slot] = off;
                    dst = A.nxt + (off << 4);
                }
                write_child(g, dst, P, ch, lane, first, vk, newrec, ch.done);
            };
            // account for / emit one child evaluated by the general routine
            auto emit = [&](const Child& ch, bool first, u64 newrec) {
                if (ch.status != CH_OK) {
                    if (MODE != MODE_WRITE) { if (ch.status == CH_OVERFLOW) s_ovf++; else s_nonpos++; }
                    return;
                }
                if (MODE != MODE_WRITE) { s_children++; s_bytes += 8; if (ch.done) s_done++; }
                if (ch.done) {   // balanced children are written where they are first seen
                    if (MODE != MODE_WRITE) place(ch, first, newrec);
                    return;
                }
                const u64 key = beam_key((u32)ch.n_unb, mix64(ch.hs + ch.hv));
                if (MODE == MODE_COUNT) {
                    s_active++; ko.push(A, lane, lane == 0, key); kmin = min(kmin, key);
                    return;
                }
                if (MODE == MODE_DIRECT || notrunc || key < X) place(ch, first, newrec);
            };

            if (vk < 0) {
                // ---- first visit: PROC1 / PROC1' (Eq 3; readings G1, G13, G14, G15, G22)
                if (P.n_vis >= A.V) {
                    if (MODE != MODE_WRITE) s_visited++;
                } else {
                    // primary on the side the flux arrives from: lowest arc of that side in the support (G13)
                    const int2* plist = fwd ? g.in_e + in0 : g.out_e + out0;
                    const int plen = fwd ? nI : nO;
                    int prim = -1;
                    for (int base = 0; base < plen && prim < 0; base += 32) {
                        const int q = base + lane;
                        const int pa = q < plen ? __ldg(&plist[q]).x : -1;
                        const u32 bal = __ballot_sync(FULL, pa >= 0 && sbit(P.sbits, pa));
                        if (bal) prim = __shfl_sync(FULL, pa, __ffs(bal) - 1);
                    }
                    const int2* alist = fwd ? g.out_e + out0 : g.in_e + in0;
                    const int alen = fwd ? nO : nI;
                    const bool fastP = fast_graph && P.big < kSmall;
                    u64 kc_k0 = 0, kc_s0 = 0, kc_k1 = 0, kc_s1 = 0;   // hash sums of the k-scaled support, last two k
                    int n_adm = 0;
                    for (int base = 0; base < alen; base += 32) {
                        const int q = base + lane;
                        int a = -1, c = 1;
                        bool adm = false, insup = false;
                        if (q < alen) {
                            const int2 e = __ldg(&alist[q]);
                            a = e.x; c = e.y;
                            const int tw = __ldg(&g.twin[a]);
                            insup = sbit(P.sbits, a);
                            adm = !(tw >= 0 && sbit(P.sbits, tw)) && (insup || P.n_supp < A.D);
                        }
                        const u32 adm_m = __ballot_sync(FULL, adm);
                        if (adm_m == 0) continue;
                        n_adm += __popc(adm_m);
                        // ---- lane-parallel evaluation: new arc, small integers => no overflow, no common factor
                        const bool fast = adm && !insup && fastP;
                        const u32 fast_m = __ballot_sync(FULL, fast);
                        u32 k = 1; u64 d = absE;
                        int nu2 = cnt;
                        if (fast) {
                            if (c != 1) scale_small(absE, (u32)c, k, d);
                            const int q1 = __ldg(&g.col_ptr[a + 1]);
                            for (int qq = __ldg(&g.col_ptr[a]); qq < q1; ++qq) {
                                const int2 e = __ldg(&g.col[qq]);
                                const i64 efp = ef_lookup(P, e.x);
                                const i64 x = (i64)k * efp + (i64)d * (i64)e.y;   // |.| < 2^60 + 2^60
                                nu2 += (int)(x != 0) - (int)(efp != 0);
                            }
                        }
                        u64 hsb = P.hs;
                        u32 need = __ballot_sync(FULL, fast && k > 1);
                        while (need) {
                            const u32 kk = __shfl_sync(FULL, k, __ffs(need) - 1);
                            u64 s;
                            if ((u64)kk == kc_k0) s = kc_s0;
                            else if ((u64)kk == kc_k1) s = kc_s1;
                            else {
                                s = 0;
                                for (int t = lane; t < P.n_supp; t += 32) s += arc_term_t(g, (u32)P.arc[t], (u64)kk * (u64)P.flux[t]);
                                s = w_sum(s);
                                kc_k1 = kc_k0; kc_s1 = kc_s0; kc_k0 = kk; kc_s0 = s;
                            }
                            const bool same = fast && k == kk;
                            if (same) hsb = s;
                            need &= ~__ballot_sync(FULL, same);
                        }
                        u64 hs2 = 0, hv2 = 0, key = 0;
                        bool done = false;
                        if (fast) {
                            const u64 newrec = vis_pack((u32)istar, (u32)(fwd ? prim : a), (u32)(fwd ? a : prim), 0u);
                            hs2 = hsb + arc_term_t(g, (u32)a, d);
                            hv2 = P.hv + vis_term(newrec);
                            key = beam_key((u32)nu2, mix64(hs2 + hv2));
                            done = nu2 == 0;
                        }
                        const u32 done_m = __ballot_sync(FULL, done);
                        if (MODE != MODE_WRITE) {
                            const int nf = __popc(fast_m);
                            s_children += nf; s_bytes += 8 * nf; s_done += __popc(done_m);
                        }
                        u32 keep_m;
                        if (MODE == MODE_COUNT) {
                            s_active += __popc(fast_m & ~done_m);
                            ko.push(A, lane, fast && !done, key);
                            if (fast && !done) kmin = min(kmin, key);
                            keep_m = done_m;
                        } else if (MODE == MODE_WRITE) {
                            keep_m = __ballot_sync(FULL, fast && !done && (notrunc || key < X));
                        } else {
                            keep_m = fast_m;
                        }
                        while (keep_m) {
                            const int l = __ffs(keep_m) - 1;
                            keep_m &= keep_m - 1;
                            Child ch;
                            ch.status = CH_OK; ch.in_supp = false; ch.ia = -1; ch.g2 = 1; ch.sign = +1;
                            ch.a = __shfl_sync(FULL, a, l);
                            ch.k = __shfl_sync(FULL, k, l);
                            ch.T = w_bcast(d, l);
                            ch.d = ch.T;
                            ch.hs = w_bcast(hs2, l);
                            ch.hv = w_bcast(hv2, l);
                            ch.n_unb = __shfl_sync(FULL, nu2, l);
                            ch.done = ch.n_unb == 0;
                            const u64 newrec = vis_pack((u32)istar, (u32)(fwd ? prim : ch.a), (u32)(fwd ? ch.a : prim), 0u);
                            place(ch, true, newrec);
                        }
                        // ---- everything else through the general routine
                        u32 slow_m = adm_m & ~fast_m;
                        while (slow_m) {
                            const int l = __ffs(slow_m) - 1;
                            slow_m &= slow_m - 1;
                            const int sa = __shfl_sync(FULL, a, l);
                            const int sc = __shfl_sync(FULL, c, l);
                            const u64 newrec = vis_pack((u32)istar, (u32)(fwd ? prim : sa), (u32)(fwd ? sa : prim), 0u);
                            Child ch;
                            eval_child(g, P, lane, sa, sc, +1, true, 0ULL, newrec, ch);
                            emit(ch, true, newrec);
                        }
                    }
                    if (n_adm == 0 && MODE != MODE_WRITE) s_dead++;
                }
            } else {
                // ---- revisit: PROC2-4 (readings G2-G5)
                const u64 rec = P.vis[vk];
                const int cntv = (int)(rec >> 48) + 1;
                if (cntv > A.max_loop) {
                    if (MODE != MODE_WRITE) s_notefm++;
                } else {
                    const int PI = (int)((rec >> 16) & 0xffffu), PO = (int)(rec & 0xffffu);
                    int lPI = -1, lPO = -1, cPI = 0, cPO = 0;
                    for (int q = lane; q < nI; q += 32) { const int2 e = __ldg(&g.in_e[in0 + q]); if (e.x == PI) { lPI = q; cPI = e.y; } }
                    for (int q = lane; q < nO; q += 32) { const int2 e = __ldg(&g.out_e[out0 + q]); if (e.x == PO) { lPO = q; cPO = e.y; } }
                    lPI = __reduce_max_sync(FULL, lPI); cPI = __reduce_max_sync(FULL, cPI);
                    lPO = __reduce_max_sync(FULL, lPO); cPO = __reduce_max_sync(FULL, cPO);
                    // Def 11: forward PO ~ SI, backward PI ~ SO, secondary = any arc of that side in the support (G5)
                    bool dep = false;
                    const i64 doff = __ldg(&g.dep_off[istar]);
                    if (fwd) {
                        for (int q = lane; q < nI; q += 32) {
                            const i64 b = doff + (i64)lPO * nI + q;
                            dep = dep || (sbit(P.sbits, __ldg(&g.in_e[in0 + q]).x) && ((__ldg(&g.dep_bits[b >> 5]) >> (b & 31)) & 1u));
                        }
                    } else {
                        for (int q = lane; q < nO; q += 32) {
                            const i64 b = doff + (i64)q * nI + lPI;
                            dep = dep || (sbit(P.sbits, __ldg(&g.out_e[out0 + q]).x) && ((__ldg(&g.dep_bits[b >> 5]) >> (b & 31)) & 1u));
                        }
                    }
                    dep = __any_sync(FULL, dep);
                    int a, c, sign;
                    if (fwd) { if (!dep) { a = PO; c = cPO; sign = +1; } else { a = PI; c = cPI; sign = -1; } }   // Eq 4 / Eq 5
                    else     { if (!dep) { a = PI; c = cPI; sign = +1; } else { a = PO; c = cPO; sign = -1; } }
                    const u64 newrec = vis_pack((u32)istar, (u32)PI, (u32)PO, (u32)cntv);
                    Child ch;
                    eval_child(g, P, lane, a, c, sign, false, rec, newrec, ch);
                    emit(ch, false, newrec);
                }
            }
            if (MODE == MODE_COUNT) {
                kmin = w_min(kmin);
                if (lane == 0) A.pmin[p] = kmin;
            }
        }
        // ---- restore the shared bitsets to zero for the next parent
        __syncwarp();
        for (int t = lane; t < P.n_supp; t += 32) P.sbits[P.arc[t] >> 5] = 0;
        for (int t = lane; t < P.n_unb; t += 32) P.ubits[P.efmet[t] >> 5] = 0;
        __syncwarp();
    }
    if (MODE == MODE_COUNT) ko.finish(A, lane);
    if (lane == 0) {
        u64* st = ctl->st;
        if (s_expanded) { atomicAdd(&st[ST_EXPANDED], s_expanded); atomicAdd(&ctl->lvl_expanded, s_expanded); }
        if (s_children) { atomicAdd(&st[ST_CHILDREN], s_children); atomicAdd(&ctl->lvl_children, s_children); }
        if (s_done) atomicAdd(&ctl->lvl_done, s_done);
        if (s_active) atomicAdd(&ctl->n_keys, s_active);
        if (s_dead) atomicAdd(&st[ST_DEAD_END], s_dead);
        if (s_notefm) atomicAdd(&st[ST_NOT_EFM], s_notefm);
        if (s_nonpos) atomicAdd(&st[ST_NONPOS], s_nonpos);
        if (s_ovf) atomicAdd(&st[ST_OVERFLOW], s_ovf);
        if (s_visited) atomicAdd(&st[ST_VISITED], s_visited);
        if (s_bytes) atomicAdd(&st[ST_ALGO_BYTES], s_bytes);
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
    a.sm_ubits = (u32)off; off = align16(off + (size_t)a.g.M32 * 4);
    a.sm_group = (u32)off;
}

// key slots the count pass can leave unused: every warp of the largest grid may strand one chunk
constexpr u64 kMaxGrid = 16384;
u64 expand_key_slack() { return kMaxGrid * kWarps * kKeyChunk; }

template <int MODE>
static cudaError_t launch_t(const ExpandArgs& a, int sm_count, cudaStream_t s) {
    const size_t smem = (size_t)a.sm_group * kWarps;
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(k_expand<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    if (smem > 227 * 1024) return cudaErrorInvalidValue;
    u64 need = (a.n_cur + kWarps - 1) / kWarps;
    int bps = (int)((227 * 1024) / (smem + 1024));
    if (bps > 16) bps = 16;
    if (bps < 1) bps = 1;
    u64 cap = (u64)sm_count * bps * 4;
    if (cap > kMaxGrid) cap = kMaxGrid;
    unsigned grid = (unsigned)(need < cap ? need : cap);
    if (grid == 0) grid = 1;
    k_expand<MODE><<<grid, kBlock, smem, s>>>(a);
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
