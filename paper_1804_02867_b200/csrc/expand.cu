// Frontier expansion kernels: one lane group ("group", GW lanes of a warp)
// owns one partial pathway.  The group stages the parent entry in shared memory, scatters its extra fluxes
// EF_i (Eq 2) into a dense per-group shared array, picks the lowest unbalanced metabolite i*
// (reading G12), fans out over the OR-alternatives of i* (first visit, PROC1/1', Eq 3) or applies
// Eq 4 / Eq 5 (revisit, PROC2-4), rescales to integers with gcd normalisation (reading G10) and
// classifies every child (balanced -> candidate; otherwise beam key).  Three modes:
//   COUNT  : count children, write only their 8-byte beam keys           (pass 1 of a level the beam may cut)
//   WRITE  : regenerate the children and materialise those with key < X  (pass 2)
//   DIRECT : single pass, every child is materialised                     (beam cannot bind)
#include <climits>

#include "device_common.cuh"
#include "launch.hpp"

namespace efm {

enum { MODE_COUNT = 0, MODE_WRITE = 1, MODE_DIRECT = 2 };
enum { CH_OK = 0, CH_NONPOS = 1, CH_OVERFLOW = 2 };
constexpr int kBlock = 128;

// ------------------------------------------------------------------ group collectives (GW lanes of one warp)
template <int GW> __device__ __forceinline__ u64 g_sum(u64 v, u32 m) {
#pragma unroll
    for (int o = GW / 2; o; o >>= 1) v += __shfl_xor_sync(m, v, o, GW);
    return v;
}
template <int GW> __device__ __forceinline__ int g_sum(int v, u32 m) {
#pragma unroll
    for (int o = GW / 2; o; o >>= 1) v += __shfl_xor_sync(m, v, o, GW);
    return v;
}
template <int GW> __device__ __forceinline__ u64 g_max(u64 v, u32 m) {
#pragma unroll
    for (int o = GW / 2; o; o >>= 1) { u64 w = __shfl_xor_sync(m, v, o, GW); v = w > v ? w : v; }
    return v;
}
template <int GW> __device__ __forceinline__ int g_max(int v, u32 m) {
#pragma unroll
    for (int o = GW / 2; o; o >>= 1) v = max(v, __shfl_xor_sync(m, v, o, GW));
    return v;
}
template <int GW> __device__ __forceinline__ int g_min(int v, u32 m) {
#pragma unroll
    for (int o = GW / 2; o; o >>= 1) v = min(v, __shfl_xor_sync(m, v, o, GW));
    return v;
}
// ballot restricted to the group, bit l = lane l of the group
template <int GW> __device__ __forceinline__ u32 g_ballot(bool p, u32 m, int shift) {
    return (__ballot_sync(m, p) & m) >> shift;
}

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
template <int GW> __device__ __forceinline__ u64 g_gcd(u64 v, u32 m) {
#pragma unroll
    for (int o = GW / 2; o; o >>= 1) { u64 w = __shfl_xor_sync(m, v, o, GW); v = gcd64(v, w); }
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

// ------------------------------------------------------------------ per-parent context (group-uniform)
struct Parent {
    int n_supp, n_vis;
    const i64* flux; const u64* vis; const u16* arc;   // shared-memory staging
    i64* EF; u32* sbits; u32* mseen;
    u64 hs, hv, fmax, maxabsEF;
    int n_unb, istar;
    i64 E;
};
struct Child {          // group-uniform description of one child relative to its parent
    int status; bool done; u64 key;
    int a; bool in_supp; int ia, ins;
    u64 k, d, g2, T;    // scale, increment, common divisor, un-normalised new flux of arc a
    int n_unb;
};

__device__ __forceinline__ bool sbit(const u32* sbits, int a) { return (sbits[a >> 5] >> (a & 31)) & 1u; }

// Evaluate the child bump(f, a, sign*|E|/c) cooperatively.
//   first: new visited record (istar, PI, PO, 0); otherwise record index vk is replaced by newrec
template <int GW, bool NEED_KEY>
__device__ __forceinline__ void eval_child(const DevGraph& g, const Parent& P, int lane, u32 gmask, int a, int c, int sign,
                                           bool first, u64 oldrec, u64 newrec, Child& ch) {
    const u64 absE = (u64)(P.E < 0 ? -P.E : P.E);
    const u64 gg = gcd64(absE, (u64)c);
    const u64 k = gg == 1 ? (u64)c : (u64)c / gg;
    const u64 d = gg == 1 ? absE : absE / gg;
    ch.a = a; ch.k = k; ch.d = d; ch.g2 = 1;
    ch.in_supp = sbit(P.sbits, a);
    // position of a in the sorted support
    int ia = -1, ins = 0;
    for (int t = lane; t < P.n_supp; t += GW) { int at = P.arc[t]; ia = at == a ? t : ia; ins += at < a; }
    ia = g_max<GW>(ia, gmask); ins = g_sum<GW>(ins, gmask);
    ch.ia = ia; ch.ins = ins;
    // scaled fluxes F_t = k f_t, F_a = k f_a +- d: overflow first, then non-positive (order of the definition, O6)
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
        if (k > 1 && umul_gt_guard(k, P.fmax)) {
            // exact: the largest flux among t != ia
            u64 mx = 0;
            for (int t = lane; t < P.n_supp; t += GW) if (t != ia) mx = max(mx, (u64)P.flux[t]);
            mx = g_max<GW>(mx, gmask);
            ovf = ovf || umul_gt_guard(k, mx);
        }
    } else {
        ovf = k > 1 && umul_gt_guard(k, P.fmax);   // the new arc carries d <= |E| <= 2^62
    }
    ch.T = T;
    if (ovf) { ch.status = CH_OVERFLOW; return; }
    if (nonpos) { ch.status = CH_NONPOS; return; }   // Prop 3, reading G11
    // extra fluxes of the un-normalised child: EF'_i = k EF_i + sign d s_ia  (Eq 2 on the scaled fluxes)
    bool ovf2 = false;
    if (k > 1 && umul_gt_guard(k, P.maxabsEF)) {
        // exact sweep over every touched metabolite outside col(a)
        const int qa0 = g.col_ptr[a], qa1 = g.col_ptr[a + 1];
        for (int t = lane; t < P.n_supp; t += GW) {
            const int at = P.arc[t];
            for (int q = g.col_ptr[at]; q < g.col_ptr[at + 1]; ++q) {
                const int i = g.col[q].x;
                bool in_a = false;
                for (int r = qa0; r < qa1; ++r) in_a = in_a || g.col[r].x == i;
                if (!in_a) ovf2 = ovf2 || abs_gt_guard(mul_s((i64)k, P.EF[i]));
            }
        }
    }
    int delta = 0;
    for (int q = g.col_ptr[a] + lane; q < g.col_ptr[a + 1]; q += GW) {
        const int2 e = g.col[q];
        const i64 efp = P.EF[e.x];
        S128 x = add_s(mul_s((i64)k, efp), mul_s(sign > 0 ? (i64)d : -(i64)d, (i64)e.y));
        ovf2 = ovf2 || abs_gt_guard(x);
        delta += (int)((x.lo | (u64)x.hi) != 0) - (int)(efp != 0);
    }
    ovf2 = g_ballot<GW>(ovf2, gmask, 0) != 0;   // any lane of the group (shift irrelevant for a zero test)
    if (ovf2) { ch.status = CH_OVERFLOW; return; }
    delta = g_sum<GW>(delta, gmask);
    ch.status = CH_OK;
    ch.n_unb = P.n_unb + delta;
    ch.done = ch.n_unb == 0;
    // gcd normalisation (reading G10).  A new arc cannot introduce a common factor: gcd_t(k f_t) = k and gcd(k, d) = 1.
    if (ch.in_supp) {
        u64 G = 0;
        for (int t = lane; t < P.n_supp; t += GW) if (t != ia) G = gcd64(G, (u64)P.flux[t]);
        G = g_gcd<GW>(G, gmask);
        ch.g2 = gcd64(k * G, T);   // k G <= k fmax <= 2^62
    }
    if (NEED_KEY) {
        u64 hs;
        if (k == 1 && ch.g2 == 1) {
            hs = P.hs + arc_term((u32)a, T) - (ch.in_supp ? arc_term((u32)a, (u64)P.flux[ia]) : 0ULL);
        } else {
            hs = 0;
            for (int t = lane; t < P.n_supp; t += GW) {
                u64 F = t == ia ? T : k * (u64)P.flux[t];
                if (ch.g2 > 1) F /= ch.g2;
                hs += arc_term((u32)P.arc[t], F);
            }
            hs = g_sum<GW>(hs, gmask);
            if (!ch.in_supp) hs += arc_term((u32)a, T);
        }
        const u64 hv = P.hv + vis_term(newrec) - (first ? 0ULL : vis_term(oldrec));
        ch.key = beam_key((u32)ch.n_unb, mix64(hs + hv));
    }
}

// Write the child into a frontier slot (or a candidate slot: no visited records).
template <int GW>
__device__ __forceinline__ void write_child(unsigned char* dst, const Parent& P, const Child& ch, int lane, bool first,
                                            int vk, u64 newrec, bool to_cand) {
    const int n2 = P.n_supp + (ch.in_supp ? 0 : 1);
    const int nv2 = to_cand ? 0 : P.n_vis + (first ? 1 : 0);
    if (lane == 0) *(uint4*)dst = make_uint4((u32)n2 | ((u32)nv2 << 16), 0u, 0u, 0u);
    i64* flux2 = (i64*)(dst + 16);
    u64* vis2 = (u64*)(flux2 + n2);
    u16* arc2 = (u16*)(vis2 + nv2);
    for (int t = lane; t < P.n_supp; t += GW) {
        u64 F = t == ch.ia ? ch.T : ch.k * (u64)P.flux[t];
        if (ch.g2 > 1) F /= ch.g2;
        const int pos = t + ((!ch.in_supp && t >= ch.ins) ? 1 : 0);
        flux2[pos] = (i64)F;
        arc2[pos] = P.arc[t];
    }
    if (!ch.in_supp && lane == 0) { flux2[ch.ins] = (i64)ch.T; arc2[ch.ins] = (u16)ch.a; }
    if (!to_cand) {
        for (int u = lane; u < P.n_vis; u += GW) vis2[u] = (!first && u == vk) ? newrec : P.vis[u];
        if (first && lane == 0) vis2[P.n_vis] = newrec;
    }
}

template <int GW, int MODE, bool ROOTS>
__global__ void __launch_bounds__(kBlock) k_expand(const ExpandArgs A) {
    extern __shared__ __align__(16) unsigned char smem[];
    const DevGraph& g = A.g;
    const int lane = threadIdx.x % GW;
    const int gib = threadIdx.x / GW;
    constexpr int GPB = kBlock / GW;
    const int shift = (threadIdx.x & 31) / GW * GW;
    const u32 gmask = GW == 32 ? 0xffffffffu : (((1u << GW) - 1u) << shift);
    unsigned char* gs = smem + (size_t)gib * A.sm_group;
    uint4* stage = (uint4*)gs;
    Parent P;
    P.EF = (i64*)(gs + A.sm_EF);
    P.sbits = (u32*)(gs + A.sm_sbits);
    P.mseen = (u32*)(gs + A.sm_mseen);
    for (int i = lane; i < g.M; i += GW) P.EF[i] = 0;
    for (int i = lane; i < g.W32; i += GW) P.sbits[i] = 0;
    for (int i = lane; i < g.M32; i += GW) P.mseen[i] = 0;
    __syncwarp(gmask);

    Ctl* ctl = A.ctl;
    const bool notrunc = MODE == MODE_WRITE ? ctl->notrunc != 0 : true;
    const u64 X = MODE == MODE_WRITE ? ctl->X : 0;

    u64 st[ST_COUNT];
#pragma unroll
    for (int i = 0; i < ST_COUNT; ++i) st[i] = 0;
    u64 l_done = 0, l_children = 0, l_expanded = 0;
    const u32 slot_chunks = A.stride / 16;

    for (u64 p = (u64)blockIdx.x * GPB + gib; p < A.n_cur; p += (u64)gridDim.x * GPB) {
        // ---- stage the parent: the first GW 16-byte chunks speculatively, the rest once the header is known
        const uint4* src = (const uint4*)(A.cur + p * A.stride);
        uint4 first = make_uint4(0, 0, 0, 0);
        if ((u32)lane < slot_chunks) first = __ldg(src + lane);
        const u32 hdr = __shfl_sync(gmask, first.x, 0, GW);
        P.n_supp = (int)(hdr & 0xffffu);
        P.n_vis = (int)(hdr >> 16);
        const u32 nch = entry_bytes((u32)P.n_supp, (u32)P.n_vis) / 16;
        if ((u32)lane < nch) stage[lane] = first;
        for (u32 c = lane + GW; c < nch; c += GW) stage[c] = __ldg(src + c);
        __syncwarp(gmask);
        P.flux = (const i64*)(stage + 1);
        P.vis = (const u64*)(P.flux + P.n_supp);
        P.arc = (const u16*)(P.vis + P.n_vis);

        // ---- Eq 2: scatter s_ia f_a into the dense EF array; support bitset; hash sums; largest flux
        u64 hs = 0, hv = 0, fmax = 0;
        for (int t = lane; t < P.n_supp; t += GW) {
            const u32 a = P.arc[t];
            const i64 f = P.flux[t];
            atomicOr(&P.sbits[a >> 5], 1u << (a & 31));
            const int q1 = g.col_ptr[a + 1];
            for (int q = g.col_ptr[a]; q < q1; ++q) {
                const int2 e = __ldg(&g.col[q]);
                atomicAdd((u64*)&P.EF[e.x], (u64)((i64)e.y * f));
            }
            if (MODE != MODE_DIRECT) hs += arc_term(a, (u64)f);
            fmax = max(fmax, (u64)f);
        }
        if (MODE != MODE_DIRECT) {
            for (int u = lane; u < P.n_vis; u += GW) hv += vis_term(P.vis[u]);
            hs = g_sum<GW>(hs, gmask);
            hv = g_sum<GW>(hv, gmask);
        }
        fmax = g_max<GW>(fmax, gmask);
        __syncwarp(gmask);
        // ---- PROC0: lowest unbalanced metabolite i*, number of unbalanced metabolites, largest |EF|
        int imin = INT_MAX, cnt = 0;
        u64 maxabs = 0;
        for (int t = lane; t < P.n_supp; t += GW) {
            const u32 a = P.arc[t];
            const int q1 = g.col_ptr[a + 1];
            for (int q = g.col_ptr[a]; q < q1; ++q) {
                const int i = __ldg(&g.col[q]).x;
                const i64 v = P.EF[i];
                if (v != 0) {
                    imin = min(imin, i);
                    maxabs = max(maxabs, (u64)(v < 0 ? -v : v));
                    const u32 bit = 1u << (i & 31);
                    const u32 old = atomicOr(&P.mseen[i >> 5], bit);
                    cnt += (old & bit) ? 0 : 1;
                }
            }
        }
        imin = g_min<GW>(imin, gmask);
        cnt = g_sum<GW>(cnt, gmask);
        maxabs = g_max<GW>(maxabs, gmask);
        P.hs = hs; P.hv = hv; P.fmax = fmax; P.maxabsEF = maxabs; P.n_unb = cnt; P.istar = imin;

        if (ROOTS) {
            // level 0: classify the root itself (arbiter "Done")
            const bool done = cnt == 0;
            const u64 key = beam_key((u32)cnt, mix64(hs + hv));
            if (MODE == MODE_COUNT) {
                if (done) l_done++;
                else {
                    u64 ks = 0;
                    if (lane == 0) ks = atomicAdd(&ctl->n_keys, 1ULL);
                    ks = __shfl_sync(gmask, ks, 0, GW);
                    if (ks < A.max_keys) { if (lane == 0) A.keys[ks] = key; }
                    else if (lane == 0) atomicOr(&ctl->error, (u32)ERR_KEYS);
                }
            } else if (done || notrunc || key < X) {
                u64 slot = 0;
                if (lane == 0) slot = atomicAdd(done ? &ctl->n_cand : &ctl->n_next, 1ULL);
                slot = __shfl_sync(gmask, slot, 0, GW);
                if (slot >= (done ? A.max_cand : A.max_frontier)) {
                    if (lane == 0) atomicOr(&ctl->error, (u32)(done ? ERR_CAND : ERR_FRONTIER));
                } else {
                    unsigned char* dst = done ? A.cand + slot * A.cand_stride : A.nxt + slot * A.stride;
                    if (lane == 0) *(uint4*)dst = make_uint4((u32)P.n_supp | ((u32)(done ? 0 : P.n_vis) << 16), 0u, 0u, 0u);
                    i64* flux2 = (i64*)(dst + 16);
                    u64* vis2 = (u64*)(flux2 + P.n_supp);
                    u16* arc2 = (u16*)(vis2 + (done ? 0 : P.n_vis));
                    for (int t = lane; t < P.n_supp; t += GW) { flux2[t] = P.flux[t]; arc2[t] = P.arc[t]; }
                    if (!done) for (int u = lane; u < P.n_vis; u += GW) vis2[u] = P.vis[u];
                }
            }
        } else {
            P.E = P.EF[imin];
            const int istar = imin;
            const bool fwd = P.E > 0;
            if (MODE != MODE_WRITE) { l_expanded++; st[ST_EXPANDED]++; st[ST_ALGO_BYTES] += algo_entry_bytes((u32)P.n_supp, (u32)P.n_vis); }
            // visited?
            int vk = -1;
            for (int u = lane; u < P.n_vis; u += GW) if ((int)((P.vis[u] >> 32) & 0xffffu) == istar) vk = u;
            vk = g_max<GW>(vk, gmask);
            const int in0 = g.in_ptr[istar], nI = g.in_ptr[istar + 1] - in0;
            const int out0 = g.out_ptr[istar], nO = g.out_ptr[istar + 1] - out0;

            // shared tail: account for / emit one evaluated child
            auto emit = [&](const Child& ch, bool first, u64 newrec) {
                if (ch.status != CH_OK) {
                    if (MODE != MODE_WRITE) st[ch.status == CH_OVERFLOW ? ST_OVERFLOW : ST_NONPOS]++;
                    return;
                }
                if (MODE != MODE_WRITE) { st[ST_CHILDREN]++; l_children++; st[ST_ALGO_BYTES] += 8; if (ch.done) l_done++; }
                if (MODE == MODE_COUNT) {
                    if (!ch.done) {
                        u64 ks = 0;
                        if (lane == 0) ks = atomicAdd(&ctl->n_keys, 1ULL);
                        ks = __shfl_sync(gmask, ks, 0, GW);
                        if (ks < A.max_keys) { if (lane == 0) A.keys[ks] = ch.key; }
                        else if (lane == 0) atomicOr(&ctl->error, (u32)ERR_KEYS);
                    }
                    return;
                }
                const bool keep = ch.done || MODE == MODE_DIRECT || notrunc || ch.key < X;
                if (!keep) return;
                const int n2 = P.n_supp + (ch.in_supp ? 0 : 1), nv2 = P.n_vis + (first ? 1 : 0);
                st[ST_ALGO_BYTES] += algo_entry_bytes((u32)n2, (u32)nv2);
                u64 slot = 0;
                if (lane == 0) slot = atomicAdd(ch.done ? &ctl->n_cand : &ctl->n_next, 1ULL);
                slot = __shfl_sync(gmask, slot, 0, GW);
                if (slot >= (ch.done ? A.max_cand : A.max_frontier)) {
                    if (lane == 0) atomicOr(&ctl->error, (u32)(ch.done ? ERR_CAND : ERR_FRONTIER));
                    return;
                }
                unsigned char* dst = ch.done ? A.cand + slot * A.cand_stride : A.nxt + slot * A.stride;
                write_child<GW>(dst, P, ch, lane, first, vk, newrec, ch.done);
            };

            if (vk < 0) {
                // ---- first visit: PROC1 / PROC1' (Eq 3; readings G1, G13, G14, G15, G22)
                if (P.n_vis >= A.V) {
                    if (MODE != MODE_WRITE) st[ST_VISITED]++;
                } else {
                    // primary on the side the flux arrives from: lowest arc of that side in the support (G13)
                    const int2* plist = fwd ? g.in_e + in0 : g.out_e + out0;
                    const int plen = fwd ? nI : nO;
                    int prim = -1;
                    for (int base = 0; base < plen && prim < 0; base += GW) {
                        const int q = base + lane;
                        const int pa = q < plen ? __ldg(&plist[q]).x : -1;
                        const u32 bal = g_ballot<GW>(pa >= 0 && sbit(P.sbits, pa), gmask, shift);
                        if (bal) prim = __shfl_sync(gmask, pa, __ffs(bal) - 1, GW);
                    }
                    const int2* alist = fwd ? g.out_e + out0 : g.in_e + in0;
                    const int alen = fwd ? nO : nI;
                    int n_adm = 0;
                    for (int base = 0; base < alen; base += GW) {
                        const int q = base + lane;
                        int2 e = make_int2(-1, 0);
                        bool adm = false;
                        if (q < alen) {
                            e = __ldg(&alist[q]);
                            const int tw = __ldg(&g.twin[e.x]);
                            adm = !(tw >= 0 && sbit(P.sbits, tw)) && (sbit(P.sbits, e.x) || P.n_supp < A.D);
                        }
                        u32 bal = g_ballot<GW>(adm, gmask, shift);
                        n_adm += __popc(bal);
                        while (bal) {
                            const int l = __ffs(bal) - 1;
                            bal &= bal - 1;
                            const int a = __shfl_sync(gmask, e.x, l, GW);
                            const int c = __shfl_sync(gmask, e.y, l, GW);
                            const u64 newrec = vis_pack((u32)istar, (u32)(fwd ? prim : a), (u32)(fwd ? a : prim), 0u);
                            Child ch;
                            eval_child<GW, MODE != MODE_DIRECT>(g, P, lane, gmask, a, c, +1, true, 0ULL, newrec, ch);
                            emit(ch, true, newrec);
                        }
                    }
                    if (n_adm == 0 && MODE != MODE_WRITE) st[ST_DEAD_END]++;
                }
            } else {
                // ---- revisit: PROC2-4 (readings G2-G5)
                const u64 rec = P.vis[vk];
                const int cntv = (int)(rec >> 48) + 1;
                if (cntv > A.max_loop) {
                    if (MODE != MODE_WRITE) st[ST_NOT_EFM]++;
                } else {
                    const int PI = (int)((rec >> 16) & 0xffffu), PO = (int)(rec & 0xffffu);
                    int lPI = -1, lPO = -1, cPI = 0, cPO = 0;
                    for (int q = lane; q < nI; q += GW) { const int2 e = __ldg(&g.in_e[in0 + q]); if (e.x == PI) { lPI = q; cPI = e.y; } }
                    for (int q = lane; q < nO; q += GW) { const int2 e = __ldg(&g.out_e[out0 + q]); if (e.x == PO) { lPO = q; cPO = e.y; } }
                    lPI = g_max<GW>(lPI, gmask); cPI = g_max<GW>(cPI, gmask);
                    lPO = g_max<GW>(lPO, gmask); cPO = g_max<GW>(cPO, gmask);
                    // Def 11: forward PO ~ SI, backward PI ~ SO, secondary = any arc of that side in the support (G5)
                    bool dep = false;
                    const i64 doff = g.dep_off[istar];
                    if (fwd) {
                        for (int q = lane; q < nI; q += GW) {
                            const i64 b = doff + (i64)lPO * nI + q;
                            dep = dep || (sbit(P.sbits, __ldg(&g.in_e[in0 + q]).x) && ((__ldg(&g.dep_bits[b >> 5]) >> (b & 31)) & 1u));
                        }
                    } else {
                        for (int q = lane; q < nO; q += GW) {
                            const i64 b = doff + (i64)q * nI + lPI;
                            dep = dep || (sbit(P.sbits, __ldg(&g.out_e[out0 + q]).x) && ((__ldg(&g.dep_bits[b >> 5]) >> (b & 31)) & 1u));
                        }
                    }
                    dep = g_ballot<GW>(dep, gmask, 0) != 0;
                    int a, c, sign;
                    if (fwd) { if (!dep) { a = PO; c = cPO; sign = +1; } else { a = PI; c = cPI; sign = -1; } }   // Eq 4 / Eq 5
                    else     { if (!dep) { a = PI; c = cPI; sign = +1; } else { a = PO; c = cPO; sign = -1; } }
                    const u64 newrec = vis_pack((u32)istar, (u32)PI, (u32)PO, (u32)cntv);
                    Child ch;
                    eval_child<GW, MODE != MODE_DIRECT>(g, P, lane, gmask, a, c, sign, false, rec, newrec, ch);
                    emit(ch, false, newrec);
                }
            }
        }
        // ---- restore the shared scratch to zero for the next parent
        __syncwarp(gmask);
        for (int t = lane; t < P.n_supp; t += GW) {
            const u32 a = P.arc[t];
            P.sbits[a >> 5] = 0;
            const int q1 = g.col_ptr[a + 1];
            for (int q = g.col_ptr[a]; q < q1; ++q) { const int i = __ldg(&g.col[q]).x; P.EF[i] = 0; P.mseen[i >> 5] = 0; }
        }
        __syncwarp(gmask);
    }
    if (lane == 0) {
#pragma unroll
        for (int i = 0; i < ST_COUNT; ++i) if (st[i]) atomicAdd(&ctl->st[i], st[i]);
        if (l_done) atomicAdd(&ctl->lvl_done, l_done);
        if (l_children) atomicAdd(&ctl->lvl_children, l_children);
        if (l_expanded) atomicAdd(&ctl->lvl_expanded, l_expanded);
    }
}

__global__ void k_level_begin(Ctl* ctl) {
    ctl->n_next = 0; ctl->n_keys = 0; ctl->lvl_done = 0; ctl->lvl_children = 0; ctl->lvl_expanded = 0;
}

// ------------------------------------------------------------------ host launchers
static size_t align16(size_t x) { return (x + 15) & ~(size_t)15; }

void expand_smem_layout(ExpandArgs& a) {
    size_t off = align16(a.stride);   // staging holds the largest entry
    a.sm_EF = (u32)off;    off = align16(off + (size_t)a.g.M * 8);
    a.sm_sbits = (u32)off; off = align16(off + (size_t)a.g.W32 * 4);
    a.sm_mseen = (u32)off; off = align16(off + (size_t)a.g.M32 * 4);
    a.sm_group = (u32)off;
}

template <int GW, int MODE, bool ROOTS>
static cudaError_t launch_t(const ExpandArgs& a, int sm_count, cudaStream_t s) {
    const int gpb = kBlock / GW;
    const size_t smem = (size_t)a.sm_group * gpb;
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(k_expand<GW, MODE, ROOTS>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    if (smem > 227 * 1024) return cudaErrorInvalidValue;
    u64 need = (a.n_cur + gpb - 1) / gpb;
    int bps = (int)((227 * 1024) / (smem + 1024));
    if (bps > 16) bps = 16;
    if (bps < 1) bps = 1;
    u64 cap = (u64)sm_count * bps * 4;
    unsigned grid = (unsigned)(need < cap ? need : cap);
    if (grid == 0) grid = 1;
    k_expand<GW, MODE, ROOTS><<<grid, kBlock, smem, s>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_expand(int mode, bool roots, const ExpandArgs& a, int sm_count, cudaStream_t s) {
    if (roots) {
        if (mode == MODE_COUNT) return launch_t<32, MODE_COUNT, true>(a, sm_count, s);
        return launch_t<32, MODE_WRITE, true>(a, sm_count, s);
    }
    if (mode == MODE_COUNT) return launch_t<32, MODE_COUNT, false>(a, sm_count, s);
    if (mode == MODE_WRITE) return launch_t<32, MODE_WRITE, false>(a, sm_count, s);
    return launch_t<32, MODE_DIRECT, false>(a, sm_count, s);
}

cudaError_t launch_level_begin(Ctl* ctl, cudaStream_t s) {
    k_level_begin<<<1, 1, 0, s>>>(ctl);
    return cudaGetLastError();
}

}  // namespace efm
