// Beam threshold selection (a-4), candidate support dedup (a-6), minimality filter (a-7) and canonical output (a-8).
#include "device_common.cuh"
#include "launch.hpp"

namespace efm {

// =================================================================================================================
// a-4  Beam select: X = the key at sorted position `cap`; the level keeps exactly {key < X}.
// MSD radix select over the 64-bit keys without a host round trip:
//   k_select_hist x2  histograms of the top 11 bits, then of the next 11 bits inside the selected bin (the top byte of a
//                     key is n_unb, so the first level alone leaves an eighth of an n_unb class); the last block
//                     (ticket) finds the bin holding rank cap
//   k_select_narrow   copies the keys with the selected 22-bit prefix to a compact buffer; the last block finishes the
//                     remaining 42 bits on the compact buffer alone (11/11/10/10-bit rounds in shared memory)
// =================================================================================================================
constexpr int kSelThreads = 256;
constexpr int kTopBits = 11;

// Whole block: the bin b with cum(b) <= rank < cum(b) + h[b]; returns through shared memory.
__device__ void block_find_bin(const u32* h, int nb, u64 rank, u32* s_bin, u64* s_cum, u64* scratch) {
    const int T = blockDim.x, per = (nb + T - 1) / T, b0 = threadIdx.x * per;
    u64 sum = 0;
    for (int j = 0; j < per; ++j) if (b0 + j < nb) sum += h[b0 + j];
    scratch[threadIdx.x] = sum;
    if (threadIdx.x == 0) { *s_bin = (u32)(nb - 1); *s_cum = 0; }   // rank beyond the total: unreachable while n_keys > cap
    __syncthreads();
    for (int off = 1; off < T; off <<= 1) {
        const u64 v = threadIdx.x >= off ? scratch[threadIdx.x - off] : 0;
        __syncthreads();
        scratch[threadIdx.x] += v;
        __syncthreads();
    }
    const u64 incl = scratch[threadIdx.x];
    u64 cum = incl - sum;
    if (cum <= rank && rank < incl)
        for (int j = 0; j < per; ++j) {
            const u64 c = h[b0 + j];
            if (rank < cum + c) { *s_bin = (u32)(b0 + j); *s_cum = cum; break; }
            cum += c;
        }
    __syncthreads();
}

// level 0: histogram of the top 11 bits of every key; level 1: of the next 11 bits of the keys inside the bin level 0
// selected.  The last block (ticket) finds the bin that holds the wanted rank and extends the selected prefix.
__global__ void __launch_bounds__(kSelThreads) k_select_hist(const u64* __restrict__ keys, Ctl* ctl, int par, u64 cap, u64 max_keys, int level) {
    const LevelCtl* lv = &ctl->lv[par];
    if (cap == 0 || lv->n_keys <= cap) return;   // the beam does not bind on this level
    __shared__ u32 h[SEL_BINS];
    __shared__ u64 scratch[kSelThreads];
    __shared__ u32 s_bin; __shared__ u64 s_cum; __shared__ bool is_last;
    for (int b = threadIdx.x; b < SEL_BINS; b += kSelThreads) h[b] = 0;
    __syncthreads();
    const u64 n = min(lv->n_slots, max_keys);   // an overflowed key array is reported by the host (ERR_KEYS)
    const u64 top = level == 0 ? 0ULL : ctl->sel_prefix;
    const int shift = 64 - kTopBits * (level + 1);
    // keys of one parent are neighbours and share their top bits: aggregate runs of equal bins per thread
    constexpr int RUN = 4;
    for (u64 i0 = ((u64)blockIdx.x * kSelThreads + threadIdx.x) * RUN; i0 < n; i0 += (u64)gridDim.x * kSelThreads * RUN) {
        u32 cur = 0xffffffffu, cnt = 0;
#pragma unroll
        for (int j = 0; j < RUN; ++j) {
            if (i0 + j >= n) break;
            const u64 key = keys[i0 + j];
            if (key >= kKeyDone) continue;   // filler of a reserved, unused slot / balanced child
            if (level == 1 && (key >> (64 - kTopBits)) != top) continue;
            const u32 b = (u32)(key >> shift) & (u32)(SEL_BINS - 1);
            if (b != cur) { if (cnt) atomicAdd(&h[cur], cnt); cur = b; cnt = 0; }
            ++cnt;
        }
        if (cnt) atomicAdd(&h[cur], cnt);
    }
    __syncthreads();
    for (int b = threadIdx.x; b < SEL_BINS; b += kSelThreads) if (h[b]) atomicAdd(&ctl->hist[b], h[b]);
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) is_last = atomicAdd(&ctl->sel_ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    for (int b = threadIdx.x; b < SEL_BINS; b += kSelThreads) { h[b] = ((volatile u32*)ctl->hist)[b]; ctl->hist[b] = 0; }
    __syncthreads();
    const u64 rank = level == 0 ? cap : ctl->sel_rank;   // level 0 starts the selection: X = the key at sorted position cap
    block_find_bin(h, SEL_BINS, rank, &s_bin, &s_cum, scratch);
    if (threadIdx.x == 0) {
        ctl->sel_prefix = (level == 0 ? 0ULL : top << kTopBits) | s_bin; ctl->sel_rank = rank - s_cum; ctl->sel_ticket = 0;
        ctl->n_compact = 0;
    }
}

// copies the keys that carry the selected 22-bit prefix to a compact buffer; the last block finishes the remaining
// 42 bits on that buffer alone
__global__ void __launch_bounds__(kSelThreads) k_select_narrow(const u64* __restrict__ keys, u64* __restrict__ ckeys, u64 max_ckeys, Ctl* ctl,
                                                               int par, u64 cap, u64 max_keys) {
    const LevelCtl* lv = &ctl->lv[par];
    if (cap == 0 || lv->n_keys <= cap) return;
    __shared__ u32 h[SEL_BINS];
    __shared__ u64 scratch[kSelThreads];
    __shared__ u32 s_bin; __shared__ u64 s_cum; __shared__ bool is_last;
    const u64 n = min(lv->n_slots, max_keys);
    const u64 top = ctl->sel_prefix;
    constexpr int kLow = 64 - 2 * kTopBits;   // bits still open
    const int lane = threadIdx.x & 31;
    const u64 span = (u64)gridDim.x * kSelThreads;
    for (u64 base = (u64)blockIdx.x * kSelThreads; base < n; base += span) {   // warp-uniform trip count
        const u64 i = base + threadIdx.x;
        const u64 key = i < n ? keys[i] : kKeySentinel;
        const bool hit = key < kKeyDone && (key >> kLow) == top;
        const u32 m = __ballot_sync(0xffffffffu, hit);
        if (m) {
            u64 pos = 0;
            if (lane == 0) pos = atomicAdd(&ctl->n_compact, (u64)__popc(m));
            pos = __shfl_sync(0xffffffffu, pos, 0);
            if (pos + __popc(m) > max_ckeys) { if (lane == 0) atomicOr(&ctl->error, (u32)ERR_KEYS); }   // loud, never a wrong threshold
            else if (hit) ckeys[pos + __popc(m & ((1u << lane) - 1u))] = key;
        }
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) is_last = atomicAdd(&ctl->sel_ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    const u64 nc = min(*(volatile u64*)&ctl->n_compact, max_ckeys);
    u64 rank = ctl->sel_rank, prefix = 0;
    const int bits[4] = {11, 11, 10, 10};
    int shift = kLow;
    for (int r = 0; r < 4; ++r) {
        shift -= bits[r];
        const int nb = 1 << bits[r];
        for (int b = threadIdx.x; b < nb; b += kSelThreads) h[b] = 0;
        __syncthreads();
        const u64 low = (1ULL << kLow) - 1ULL;
        for (u64 i = threadIdx.x; i < nc; i += kSelThreads) {
            const u64 key = __ldcg(&ckeys[i]) & low;
            if (r == 0 || (key >> (shift + bits[r])) == prefix) atomicAdd(&h[(key >> shift) & (u64)(nb - 1)], 1u);
        }
        __syncthreads();
        block_find_bin(h, nb, rank, &s_bin, &s_cum, scratch);
        prefix = (prefix << bits[r]) | (u64)s_bin;
        rank -= s_cum;
        __syncthreads();
    }
    if (threadIdx.x == 0) { ctl->X = (top << kLow) | prefix; ctl->sel_ticket = 0; }
}

cudaError_t launch_select(const u64* keys, u64* ckeys, u64 max_ckeys, Ctl* ctl, int par, u64 cap, u64 max_keys, int sm_count, cudaStream_t s,
                          int* n_launches) {
    if (cap == 0) return cudaSuccess;
    u64 blocks = (max_keys + kSelThreads * 8 - 1) / (kSelThreads * 8);
    if (blocks > (u64)sm_count * 8) blocks = (u64)sm_count * 8;
    if (blocks < 1) blocks = 1;
    k_select_hist<<<(unsigned)blocks, kSelThreads, 0, s>>>(keys, ctl, par, cap, max_keys, 0);
    k_select_hist<<<(unsigned)blocks, kSelThreads, 0, s>>>(keys, ctl, par, cap, max_keys, 1);
    k_select_narrow<<<(unsigned)blocks, kSelThreads, 0, s>>>(keys, ckeys, max_ckeys, ctl, par, cap, max_keys);
    *n_launches += 3;
    return cudaGetLastError();
}

// =================================================================================================================
// a-6  Candidate dedup: open-addressing hash keyed on the arc-space support (the sorted arc list is the bitset in
// sparse form).  The first candidate to claim a slot represents its support; a later candidate with the same support
// and a different coprime flux vector poisons it (reading G18) -- order-independent.
// =================================================================================================================
__device__ __forceinline__ const i64* cand_flux(const unsigned char* e) { return (const i64*)(e + kHdr); }
__device__ __forceinline__ int cand_n(const unsigned char* e) { return (int)(*(const u32*)e & 0xffffu); }
__device__ __forceinline__ const u16* cand_arc(const unsigned char* e, int n) { return (const u16*)(e + kHdr + 8 * (size_t)n); }

__global__ void __launch_bounds__(256) k_dedup_insert(const PostArgs a, u64 n_cand) {
    const u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_cand) return;
    const unsigned char* e = a.cand + i * a.cand_stride;
    const int n = cand_n(e);
    const u16* arc = cand_arc(e, n);
    const i64* f = cand_flux(e);
    const u32 own_steps = ((const u32*)e)[11];
    atomicMin(&a.c_steps[i], own_steps);
    u64 h = 0;
    for (int t = 0; t < n; ++t) h += mix64(0x0300000000000000ULL | (u64)arc[t]);
    u64 slot = mix64(h) & (a.table_size - 1);
    for (;;) {
        const u32 prev = atomicCAS(&a.table[slot], 0xFFFFFFFFu, (u32)i);
        if (prev == 0xFFFFFFFFu) { a.isrep[i] = 1; return; }
        const unsigned char* o = a.cand + (u64)prev * a.cand_stride;
        const int no = cand_n(o);
        if (no == n) {
            const u16* oarc = cand_arc(o, no);
            bool same = true;
            for (int t = 0; t < n && same; ++t) same = arc[t] == oarc[t];
            if (same) {
                const i64* of = cand_flux(o);
                bool eq = true;
                for (int t = 0; t < n && eq; ++t) eq = f[t] == of[t];
                if (!eq) a.poison[prev] = 1;
                else atomicMin(&a.c_steps[prev], own_steps);   // equal duplicates are one pathway: its quickest construction counts
                return;
            }
        }
        slot = (slot + 1) & (a.table_size - 1);
    }
}

__global__ void __launch_bounds__(256) k_dedup_collect(const PostArgs a, u64 n_cand) {
    const u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_cand || !a.isrep[i]) return;
    atomicAdd(&a.ctl->n_unique, 1ULL);
    if (a.poison[i]) { atomicAdd(&a.ctl->n_poisoned, 1ULL); return; }
    const u64 pos = atomicAdd(&a.ctl->n_uniq_ok, 1ULL);
    a.uniq[pos] = (u32)i;
}

cudaError_t launch_dedup(const PostArgs& a, u64 n_cand, cudaStream_t s, int* n_launches) {
    cudaError_t e;
    if ((e = cudaMemsetAsync(a.table, 0xFF, a.table_size * sizeof(u32), s)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(a.isrep, 0, n_cand + 1, s)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(a.poison, 0, n_cand + 1, s)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(a.c_steps, 0xFF, (n_cand + 1) * sizeof(u32), s)) != cudaSuccess) return e;
    if (n_cand == 0) return cudaSuccess;
    const unsigned blocks = (unsigned)((n_cand + 255) / 256);
    k_dedup_insert<<<blocks, 256, 0, s>>>(a, n_cand);
    k_dedup_collect<<<blocks, 256, 0, s>>>(a, n_cand);
    *n_launches += 2;
    return cudaGetLastError();
}

// =================================================================================================================
// a-7  Minimality filter (Def 3; reading G17): drop v if some other unique support w
// is a strict subset.  supp(w) inside supp(v) needs EVERY arc of w in v, in particular the arc of w that is rarest
// among all candidates.  So rows are grouped by their rarest arc (counting sort over arcs) and a row v is tested
// only against the groups of its own arcs: sum over a in supp(v) of |group(a)| pair tests instead of K.  A pair test
// is the 128-bit signature test (exact bitsets when A <= 128, a 128-bucket image of the arc set otherwise; coalesced
// 16-byte loads, one lane per w), signature hits are verified on the sorted arc lists.
// =================================================================================================================
// 112-bit signature of a support (exact bitset when A <= 112, otherwise arc -> one of 112 buckets); the remaining 16
// bits of the 128-bit record hold |supp| so that one 16-byte load serves the whole pair test
constexpr int kSigBits = 112;
__device__ __forceinline__ u32 sig_bit(int arc, bool exact) { return exact ? (u32)arc : (((u32)arc * 0x9E3779B1u) >> 16) % (u32)kSigBits; }
__device__ __forceinline__ uint4 sig_of(const u16* arc, int n, bool exact) {   // whole signature by one thread
    u32 w[4] = {0, 0, 0, 0};
    for (int t = 0; t < n; ++t) { const u32 b = sig_bit(arc[t], exact); w[b >> 5] |= 1u << (b & 31); }
    return make_uint4(w[0], w[1], w[2], w[3] | ((u32)n << 16));
}

// first-stage signature: arc -> one of 64 buckets.  A support of 45 arcs sets about 32 of the bits, one of 50 arcs about 35:
// a pair passes with probability around 0.54^32, so a warp almost never leaves the straight-line loop, and two of these
// tests cost one 16-byte shared-memory load and four LOP3.
__device__ __forceinline__ uint2 sig64_of(const u16* arc, int n) {
    u32 w0 = 0, w1 = 0;
    for (int t = 0; t < n; ++t) {
        const u32 b = ((u32)arc[t] * 0x9E3779B1u) >> 26;
        if (b < 32) w0 |= 1u << b; else w1 |= 1u << (b - 32);
    }
    return make_uint2(w0, w1);
}

__global__ void __launch_bounds__(256) k_filter_freq(const PostArgs a, u64 K, int use_smem) {
    // per-block histogram in shared memory when the arcs fit (popular arcs would otherwise serialise in L2)
    extern __shared__ u32 hist[];
    if (use_smem) {
        for (int i = threadIdx.x; i < a.g.A; i += blockDim.x) hist[i] = 0;
        __syncthreads();
    }
    for (u64 u = (u64)blockIdx.x * blockDim.x + threadIdx.x; u < K; u += (u64)gridDim.x * blockDim.x) {
        const unsigned char* e = a.cand + (u64)a.uniq[u] * a.cand_stride;
        const int n = cand_n(e);
        const u16* arc = cand_arc(e, n);
        for (int t = 0; t < n; ++t) atomicAdd(use_smem ? &hist[arc[t]] : &a.freq[arc[t]], 1u);
    }
    if (use_smem) {
        __syncthreads();
        for (int i = threadIdx.x; i < a.g.A; i += blockDim.x) if (hist[i]) atomicAdd(&a.freq[i], hist[i]);
    }
}
__device__ __forceinline__ int rarest_arc(const PostArgs& a, const u16* arc, int n) {   // ties: lowest arc id
    u32 best = 0xffffffffu; int key = 0;
    for (int t = 0; t < n; ++t) { const u32 f = a.freq[arc[t]]; if (f < best) { best = f; key = arc[t]; } }
    return key;
}
__global__ void __launch_bounds__(256) k_filter_count(const PostArgs a, u64 K) {
    const u64 u = (u64)blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= K) return;
    const unsigned char* e = a.cand + (u64)a.uniq[u] * a.cand_stride;
    const int n = cand_n(e);
    if (n == 0) return;   // the empty support belongs to no group (it has no strict subset and nothing tests against it)
    atomicAdd(&a.gcount[(size_t)rarest_arc(a, cand_arc(e, n), n) * a.n_sizes + n], 1u);   // group key: (rarest arc, |supp|)
}
// exclusive scan of `len` counters by one block: start[i] and fill[i] get the prefix, start[len] the total
__global__ void __launch_bounds__(1024) k_filter_scan(const u32* __restrict__ count, u32* __restrict__ start, u32* __restrict__ fill, int len) {
    __shared__ u32 part[1024];
    const int T = blockDim.x, per = (len + T - 1) / T, b0 = threadIdx.x * per;
    u32 sum = 0;
    for (int j = 0; j < per; ++j) if (b0 + j < len) sum += count[b0 + j];
    part[threadIdx.x] = sum;
    __syncthreads();
    for (int off = 1; off < T; off <<= 1) {
        const u32 v = threadIdx.x >= off ? part[threadIdx.x - off] : 0;
        __syncthreads();
        part[threadIdx.x] += v;
        __syncthreads();
    }
    u32 acc = part[threadIdx.x] - sum;
    for (int j = 0; j < per; ++j)
        if (b0 + j < len) { const u32 c = count[b0 + j]; start[b0 + j] = acc; fill[b0 + j] = acc; acc += c; }
    if (threadIdx.x == T - 1) start[len] = part[T - 1];
}
__global__ void __launch_bounds__(256) k_filter_scatter(const PostArgs a, u64 K) {
    const u64 u = (u64)blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= K) return;
    const u32 id = a.uniq[u];
    const unsigned char* e = a.cand + (u64)id * a.cand_stride;
    const int n = cand_n(e);
    if (n == 0) return;
    const u16* arc = cand_arc(e, n);
    const u32 pos = atomicAdd(&a.gfill[(size_t)rarest_arc(a, arc, n) * a.n_sizes + n], 1u);
    const uint4 sg = sig_of(arc, n, a.g.A <= kSigBits);
    const uint2 s64 = sig64_of(arc, n);
    a.g_row[pos] = id;
    a.g_sig[pos] = sg;
    a.g_sig64[pos] = s64;
    a.r_sig[u] = sg;   // the same records in row order, for the v side of the join
    a.r_sig64[u] = s64;
}
__device__ bool arcs_subset(const unsigned char* w, const unsigned char* v) {   // supp(w) subset of supp(v), sorted lists
    const int nw = cand_n(w), nv = cand_n(v);
    const u16* aw = cand_arc(w, nw);
    const u16* av = cand_arc(v, nv);
    int j = 0;
    for (int t = 0; t < nw; ++t) {
        while (j < nv && av[j] < aw[t]) ++j;
        if (j == nv || av[j] != aw[t]) return false;
        ++j;
    }
    return true;
}
// ---- the join, tiled.  For every arc a: V(a) = the rows that contain a, W(a) = the group of a (rows whose rarest arc
// is a, ordered by size).  A block takes 256 rows of V(a) -- one per thread, signature in registers -- and streams
// W(a) through shared memory in tiles of 256 records: every 16-byte record is read from L2 / HBM once per block instead
// of once per row.  k_filter_vprep sizes V(a) (only for arcs with a non-empty group) and numbers the tiles,
// k_filter_vscatter fills the lists, k_filter_join maps a block to (arc, tile) by binary search over the tile prefix.
#ifndef EFM_JOIN_THREADS
#define EFM_JOIN_THREADS 128   // rows of V(a) per block: four warps share every tile of W(a)
#endif
constexpr int kJoinThreads = EFM_JOIN_THREADS;
constexpr int kWTile = 1024;   // rows of W(a) per shared-memory tile (first-stage signatures: 8 KB)
// V lists are ordered by (arc, size) too: the rows of a tile have about the same size, hence the same range of W
__global__ void __launch_bounds__(256) k_filter_vcount(const PostArgs a, u64 K, int fill) {
    const u64 u = (u64)blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= K) return;
    if (fill) a.keep[u] = 1;
    const unsigned char* e = a.cand + (u64)a.uniq[u] * a.cand_stride;
    const int n = cand_n(e);
    const u16* arc = cand_arc(e, n);
    for (int t = 0; t < n; ++t) {
        const size_t gb = (size_t)arc[t] * a.n_sizes;
        if (a.gstart[gb + n] > a.gstart[gb]) {   // the group of this arc has rows strictly smaller than this one
            if (fill) a.v_row[atomicAdd(&a.vfill[gb + n], 1u)] = (u32)u;
            else atomicAdd(&a.vcount[gb + n], 1u);
        }
    }
}
__global__ void __launch_bounds__(1024) k_filter_tiles(const PostArgs a) {   // tiles of kJoinThreads rows per arc, prefix over the arcs
    __shared__ u32 part[1024];
    const int A = a.g.A, T = blockDim.x, per = (A + T - 1) / T, b0 = threadIdx.x * per;
    u32 st = 0;
    for (int j = 0; j < per; ++j) {
        const int x = b0 + j;
        if (x < A) st += (a.vstart[(size_t)(x + 1) * a.n_sizes] - a.vstart[(size_t)x * a.n_sizes] + kJoinThreads - 1) / kJoinThreads;
    }
    part[threadIdx.x] = st;
    __syncthreads();
    for (int off = 1; off < T; off <<= 1) {
        const u32 v = threadIdx.x >= off ? part[threadIdx.x - off] : 0;
        __syncthreads();
        part[threadIdx.x] += v;
        __syncthreads();
    }
    u32 at = part[threadIdx.x] - st;
    for (int j = 0; j < per; ++j) {
        const int x = b0 + j;
        if (x >= A) break;
        a.tstart[x] = at;
        at += (a.vstart[(size_t)(x + 1) * a.n_sizes] - a.vstart[(size_t)x * a.n_sizes] + kJoinThreads - 1) / kJoinThreads;
    }
    if (threadIdx.x == T - 1) a.tstart[A] = part[T - 1];
}
// Two stages per pair (w, v): the 64-bit bucket signatures (two rows of W per 16-byte shared-memory load), then, for the
// few pairs that pass, the 112-bit signature + size record and the exact test on the sorted arc lists.
__global__ void __launch_bounds__(kJoinThreads) k_filter_join(const PostArgs a) {
    __shared__ uint4 wt4[kWTile / 2];
    __shared__ u32 s_gend;
    __shared__ unsigned long long s_pairs;
    uint2* wt = (uint2*)wt4;
    const int A = a.g.A;
    const u32 n_tiles = a.tstart[A];
    const bool exact = A <= kSigBits;
    for (u32 tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {   // block-uniform
        // arc of this tile: the last x with tstart[x] <= tile
        int lo = 0, hi = A;
        while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (a.tstart[mid] <= tile) lo = mid; else hi = mid; }
        const int x = lo;
        const size_t gb = (size_t)x * a.n_sizes;
        const u32 vi = a.vstart[gb] + (tile - a.tstart[x]) * kJoinThreads + threadIdx.x;
        const bool live = vi < a.vstart[gb + a.n_sizes];
        u32 u = 0, gend = 0, vn0 = 0, vn1 = 0;
        uint4 sv = make_uint4(0, 0, 0, 0);
        const u32 g0 = a.gstart[gb];
        if (live) {
            u = a.v_row[vi];
            sv = a.r_sig[u];
            { const uint2 t = a.r_sig64[u]; vn0 = ~t.x; vn1 = ~t.y; }
            gend = a.gstart[gb + (sv.w >> 16)];   // group rows of size < |supp(v)|
        }
        if (threadIdx.x == 0) { s_gend = 0; s_pairs = 0; }
        __syncthreads();
        if (live) atomicMax(&s_gend, gend);
        __syncthreads();
        const u32 bend = s_gend;
        const u32 n0 = ~sv.x, n1 = ~sv.y, n2 = ~sv.z, n3 = ~sv.w & 0xffffu;
        bool found = false;
        u32 tested = 0;   // first-stage pair tests this row really made (a hit ends its scan)
        for (u32 base = g0; base < bend; base += kWTile) {
            for (u32 i = threadIdx.x; i < (u32)kWTile; i += kJoinThreads) wt[i] = base + i < bend ? a.g_sig64[base + i] : make_uint2(0xffffffffu, 0xffffffffu);
            __syncthreads();
            if (live && !found && base < gend) {
                // eight rows of W per step, one branch: rows behind gend (or behind the tile) are filtered in the closer look
                const u32 jn = (min((u32)kWTile, gend - base) + 7u) / 8u;
                u32 jstop = jn;
#pragma unroll 1
                for (u32 j = 0; j < jn; ++j) {
                    const uint4 ra = wt4[4 * j], rb = wt4[4 * j + 1], rc = wt4[4 * j + 2], rd = wt4[4 * j + 3];
                    u32 z = min((ra.x & vn0) | (ra.y & vn1), (ra.z & vn0) | (ra.w & vn1));
                    z = min(z, min((rb.x & vn0) | (rb.y & vn1), (rb.z & vn0) | (rb.w & vn1)));
                    z = min(z, min((rc.x & vn0) | (rc.y & vn1), (rc.z & vn0) | (rc.w & vn1)));
                    z = min(z, min((rd.x & vn0) | (rd.y & vn1), (rd.z & vn0) | (rd.w & vn1)));
                    if (__builtin_expect(z == 0, 0)) {   // rare: some row of the eight passes the first stage, look closer
#pragma unroll 1
                        for (u32 c = 0; c < 8 && !found; ++c) {
                            const u32 row = base + 8 * j + c;
                            const uint2 w = wt[8 * j + c];
                            if (((w.x & vn0) | (w.y & vn1)) != 0 || row >= gend) continue;
                            const uint4 sg = a.g_sig[row];
                            if (((sg.x & n0) | (sg.y & n1) | (sg.z & n2) | (sg.w & n3)) == 0)
                                found = exact || arcs_subset(a.cand + (u64)a.g_row[row] * a.cand_stride, a.cand + (u64)a.uniq[u] * a.cand_stride);
                        }
                        if (found) { jstop = j + 1; break; }
                    }
                }
                tested += min(8u * jstop, min((u32)kWTile, gend - base));
            }
            __syncthreads();
        }
        if (found) a.keep[u] = 0;
        if (tested) atomicAdd(&s_pairs, (unsigned long long)tested);
        __syncthreads();
        if (threadIdx.x == 0 && s_pairs) atomicAdd(&a.ctl->filter_pairs, (u64)s_pairs);
        __syncthreads();
    }
}

// =================================================================================================================
// SURVEY.md 8(f)-3  Exact elementarity (Def 3; "recognizing the elementarity through rank
// test"): a unique, unpoisoned support stays iff the internal rows of S restricted to its arcs have rank |supp| - 1 over
// GF(p), p = 2^31 - 1 (reading G24).  One warp per support.  The rows (metabolites touched by the support) are
// never materialised as a matrix: a row is gathered from the columns of the arcs (lane = arc), reduced against the basis
// kept in shared memory (one vector per pivot column, fraction-free: v <- piv v - v_c b_c) and either vanishes or joins
// the basis.  The rank of a matrix does not depend on the elimination order, so the result is bit-exact with any other
// elimination over the same field.
// =================================================================================================================
constexpr u32 kRankP = 2147483647u;
__device__ __forceinline__ u32 mulmod_p(u32 x, u32 y) {
    u64 t = (u64)x * y;
    t = (t & kRankP) + (t >> 31);
    t = (t & kRankP) + (t >> 31);
    return t >= kRankP ? (u32)(t - kRankP) : (u32)t;
}
template <int CH>   // CH chunks of 32 arcs: supports of up to 32 CH arcs
__global__ void __launch_bounds__(128) k_rank_test(const PostArgs a, u64 K, int warps_per_block) {
    extern __shared__ u32 rk_smem[];
    constexpr int N = 32 * CH;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    if (wib >= warps_per_block) return;
    u32* basis = rk_smem + (size_t)wib * N * N;   // basis[c * N + k]: the vector whose pivot column is c
    for (u64 u = (u64)blockIdx.x * warps_per_block + wib; u < K; u += (u64)gridDim.x * warps_per_block) {
        const unsigned char* e = a.cand + (u64)a.uniq[u] * a.cand_stride;
        const int n = cand_n(e);
        const u16* arc = cand_arc(e, n);
        int my_arc[CH];
#pragma unroll
        for (int ch = 0; ch < CH; ++ch) my_arc[ch] = lane + 32 * ch < n ? (int)arc[lane + 32 * ch] : -1;
        u32 has_piv[CH];
#pragma unroll
        for (int ch = 0; ch < CH; ++ch) has_piv[ch] = 0;
        int rank = 0;
#pragma unroll 1
        for (int t = 0; t < n && rank < n - 1; ++t) {
            const int at = arc[t];
            const int q0 = a.g.col_ptr[at], q1 = a.g.col_ptr[at + 1];
#pragma unroll 1
            for (int q = q0; q < q1 && rank < n - 1; ++q) {
                const int met = col_met(a.g.col[q]);
                // the row of `met` over the arcs of the support
                u32 v[CH];
                bool earlier = false;
#pragma unroll
                for (int ch = 0; ch < CH; ++ch) {
                    v[ch] = 0;
                    const int am = my_arc[ch];
                    if (am >= 0 && (((a.g.colsig[2 * am] | a.g.colsig[2 * am + 1]) >> (met & 63)) & 1ULL)) {
                        for (int r = a.g.col_ptr[am]; r < a.g.col_ptr[am + 1]; ++r) {
                            const int2 ce = a.g.col[r];
                            if (col_met(ce) == met) { const long long sv = (long long)ce.y % (long long)kRankP; v[ch] = (u32)(sv < 0 ? sv + kRankP : sv); }
                        }
                    }
                    if (v[ch] != 0 && lane + 32 * ch < t) earlier = true;
                }
                if (__any_sync(0xffffffffu, earlier)) continue;   // an arc before t holds this metabolite: its row was taken then
                // reduce against the basis
#pragma unroll 1
                for (;;) {
                    int c = -1;
#pragma unroll
                    for (int ch = CH - 1; ch >= 0; --ch) { const u32 m = __ballot_sync(0xffffffffu, v[ch] != 0); if (m) c = 32 * ch + __ffs(m) - 1; }
                    if (c < 0) break;   // the row depends on the basis
                    const bool have = (has_piv[c >> 5] >> (c & 31)) & 1u;
                    if (!have) {   // a new pivot
#pragma unroll
                        for (int ch = 0; ch < CH; ++ch) basis[(size_t)c * N + lane + 32 * ch] = v[ch];
                        has_piv[c >> 5] |= 1u << (c & 31);
                        ++rank;
                        __syncwarp();
                        break;
                    }
                    const u32 piv = basis[(size_t)c * N + c];
                    u32 vc = 0;
#pragma unroll
                    for (int ch = 0; ch < CH; ++ch) { const u32 x = __shfl_sync(0xffffffffu, v[ch], c & 31); if ((c >> 5) == ch) vc = x; }
#pragma unroll
                    for (int ch = 0; ch < CH; ++ch) {
                        const u32 x = mulmod_p(piv, v[ch]), y = mulmod_p(vc, basis[(size_t)c * N + lane + 32 * ch]);
                        v[ch] = x >= y ? x - y : x + kRankP - y;
                    }
                }
            }
        }
        if (lane == 0) a.keep[u] = rank == n - 1 ? 1 : 0;
        __syncwarp();
    }
}
cudaError_t launch_rank_test(const PostArgs& a, u64 K, int sm_count, cudaStream_t s, int* n_launches) {
    if (K == 0) return cudaSuccess;
    const int ch = (a.D + 31) / 32;
    if (ch > 4) return cudaErrorInvalidValue;   // efm_create refuses the flag for D > 128
    const size_t per_warp = (size_t)(32 * ch) * (32 * ch) * 4;
    int wpb = (int)((96 * 1024) / per_warp);
    wpb = wpb > 4 ? 4 : (wpb < 1 ? 1 : wpb);
    const size_t smem = per_warp * wpb;
    u64 blocks = (K + wpb - 1) / wpb;
    if (blocks > (u64)sm_count * 8) blocks = (u64)sm_count * 8;
    cudaError_t e = cudaSuccess;
#define EFM_RANK_LAUNCH(CHN)                                                                                                      \
    do {                                                                                                                          \
        e = cudaFuncSetAttribute(k_rank_test<CHN>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);                      \
        if (e == cudaSuccess) k_rank_test<CHN><<<(unsigned)blocks, 128, smem, s>>>(a, K, wpb);                                    \
    } while (0)
    if (ch <= 1) EFM_RANK_LAUNCH(1);
    else if (ch == 2) EFM_RANK_LAUNCH(2);
    else if (ch == 3) EFM_RANK_LAUNCH(3);
    else EFM_RANK_LAUNCH(4);
#undef EFM_RANK_LAUNCH
    if (e != cudaSuccess) return e;
    ++*n_launches;
    return cudaGetLastError();
}

cudaError_t launch_filter(const PostArgs& a, u64 K, int sm_count, cudaStream_t s, int* n_launches) {
    cudaError_t e;
    if ((e = cudaMemsetAsync(a.freq, 0, sizeof(u32) * (a.g.A + 2), s)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(a.gcount, 0, sizeof(u32) * ((size_t)a.g.A * a.n_sizes + 2), s)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(a.vcount, 0, sizeof(u32) * ((size_t)a.g.A * a.n_sizes + 2), s)) != cudaSuccess) return e;
    if (K == 0) return cudaSuccess;
    const unsigned blocks = (unsigned)((K + 255) / 256);
    {
        const int use_smem = (size_t)a.g.A * 4 <= 40 * 1024;
        unsigned fb = blocks < (unsigned)sm_count * 8 ? blocks : (unsigned)sm_count * 8;
        k_filter_freq<<<fb, 256, use_smem ? (size_t)a.g.A * 4 : 0, s>>>(a, K, use_smem);
    }
    k_filter_count<<<blocks, 256, 0, s>>>(a, K);
    k_filter_scan<<<1, 1024, 0, s>>>(a.gcount, a.gstart, a.gfill, a.g.A * a.n_sizes);
    k_filter_scatter<<<blocks, 256, 0, s>>>(a, K);
    k_filter_vcount<<<blocks, 256, 0, s>>>(a, K, 0);
    k_filter_scan<<<1, 1024, 0, s>>>(a.vcount, a.vstart, a.vfill, a.g.A * a.n_sizes);
    k_filter_tiles<<<1, 1024, 0, s>>>(a);
    k_filter_vcount<<<blocks, 256, 0, s>>>(a, K, 1);
    k_filter_join<<<(unsigned)(sm_count * 16), kJoinThreads, 0, s>>>(a);
    *n_launches += 9;
    return cudaGetLastError();
}

// =================================================================================================================
// a-8  Canonical output: arc space -> reaction space (v_j = f_j+ - f_j-), lexicographic order of the dense signed
// vectors, computed on the sparse rows with a bitonic sort of row indices.
// =================================================================================================================
// Order-preserving 64-bit code of "the next non-zero entry is value v at reaction j" (all earlier reactions equal):
// a negative entry at a smaller reaction makes the row smaller, a positive one makes it larger, and a row without
// further entries sits between the two classes.  Values are clamped to 32 bits; codes at the clamp (and the "no entry"
// code) decide nothing on a tie.  Two such codes (first and second entry) settle almost every comparison of the sort
// without touching the rows.
__device__ __forceinline__ u64 order_code(bool has, int j, i64 v) {
    if (!has) return 1ULL << 63;
    const i64 L = (1LL << 31) - 1;
    const u32 c = (u32)((v < -L ? -L : (v > L ? L : v)) + (1LL << 31));   // [1, 2^32 - 1]
    return v < 0 ? ((u64)(u32)j << 32) | c : (1ULL << 63) | ((u64)(0x7fffffffu - (u32)j) << 32) | c;
}
__device__ __forceinline__ int key_cmp(const ulonglong2 kx, const ulonglong2 ky) {   // -1: x < y, +1: x > y, 0: look at the rows
    if (kx.x != ky.x) return kx.x < ky.x ? -1 : 1;
    const u32 low = (u32)kx.x;
    if (low <= 1u || low == 0xffffffffu) return 0;
    if (kx.y != ky.y) return kx.y < ky.y ? -1 : 1;
    return 0;
}
__global__ void __launch_bounds__(256) k_out_rows(const PostArgs a, u64 K) {   // one warp per kept row
    const u64 p = (u64)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (p >= K || !a.keep[p]) return;
    const int lane = threadIdx.x & 31;
    u64 r = 0;
    if (lane == 0) r = atomicAdd(&a.ctl->n_keep, 1ULL);
    r = __shfl_sync(0xffffffffu, r, 0);
    const unsigned char* e = a.cand + (u64)a.uniq[p] * a.cand_stride;
    const int n = cand_n(e);
    const u16* arc = cand_arc(e, n);
    const i64* f = cand_flux(e);
    if (lane == 0) { a.u_nnz[r] = n; a.u_steps[r] = (int)a.c_steps[a.uniq[p]]; }
    int j01 = 0; i64 v01 = 0;   // lanes 0 and 1 keep the first two entries for the order codes
    for (int t = lane; t < n; t += 32) {   // arcs ascend => reactions ascend (twins never share a support)
        const int j = a.g.arc_rxn[arc[t]];
        const i64 v = a.g.arc_dir[arc[t]] < 0 ? -f[t] : f[t];
        a.u_rxn[r * a.D + t] = j;
        a.u_val[r * a.D + t] = v;
        if (t < 2) { j01 = j; v01 = v; }
    }
    const int j1 = __shfl_sync(0xffffffffu, j01, 1);
    const i64 v1 = __shfl_sync(0xffffffffu, v01, 1);
    if (lane == 0) a.u_key[r] = make_ulonglong2(order_code(n > 0, j01, v01), order_code(n > 1, j1, v1));
}

// strict lexicographic "row x < row y" on the dense vectors, evaluated on the sparse rows
__device__ bool row_less(const PostArgs& a, u32 x, u32 y) {
    if (x == 0xFFFFFFFFu) return false;   // padding sorts last
    if (y == 0xFFFFFFFFu) return true;
    const int nx = a.u_nnz[x], ny = a.u_nnz[y];
    const int* jx = a.u_rxn + (u64)x * a.D; const int* jy = a.u_rxn + (u64)y * a.D;
    const i64* vx = a.u_val + (u64)x * a.D; const i64* vy = a.u_val + (u64)y * a.D;
    int tx = 0, ty = 0;
    for (;;) {
        if (tx == nx && ty == ny) return false;
        const int cx = tx < nx ? jx[tx] : 0x7fffffff, cy = ty < ny ? jy[ty] : 0x7fffffff;
        if (cx == cy) { if (vx[tx] != vy[ty]) return vx[tx] < vy[ty]; ++tx; ++ty; }
        else if (cx < cy) return vx[tx] < 0;   // y is 0 at reaction cx
        else return 0 < vy[ty];                // x is 0 at reaction cy
    }
}
__global__ void __launch_bounds__(256) k_sort_init(const PostArgs a, u64 n_keep) {
    const u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < a.n_pad) a.sort_idx[i] = i < n_keep ? (u32)i : 0xFFFFFFFFu;
}
__global__ void __launch_bounds__(256) k_bitonic_global(const PostArgs a, u64 j, u64 k) {
    const u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.n_pad) return;
    const u64 ixj = i ^ j;
    if (ixj <= i) return;
    const bool asc = (i & k) == 0;
    const u32 x = a.sort_idx[i], y = a.sort_idx[ixj];
    bool swap;
    if (x == 0xFFFFFFFFu || y == 0xFFFFFFFFu) swap = asc ? row_less(a, y, x) : row_less(a, x, y);
    else {
        const int c = key_cmp(a.u_key[x], a.u_key[y]);   // sign of x - y when the keys decide
        swap = c ? (asc ? c > 0 : c < 0) : (asc ? row_less(a, y, x) : row_less(a, x, y));
    }
    if (swap) { a.sort_idx[i] = y; a.sort_idx[ixj] = x; }
}
constexpr int kSortChunk = 1024;
// all compare-exchange steps with j < kSortChunk of the stages k in [k_lo, k_hi] on one shared-memory chunk
__global__ void __launch_bounds__(kSortChunk / 2) k_bitonic_local(const PostArgs a, u64 k_lo, u64 k_hi) {
    __shared__ u32 s[kSortChunk];
    __shared__ ulonglong2 sk[kSortChunk];   // the order keys travel with the indices
    const u64 base = (u64)blockIdx.x * kSortChunk;
    for (int t = threadIdx.x; t < kSortChunk; t += blockDim.x) {
        s[t] = base + t < a.n_pad ? a.sort_idx[base + t] : 0xFFFFFFFFu;
        sk[t] = s[t] == 0xFFFFFFFFu ? make_ulonglong2(~0ULL, ~0ULL) : a.u_key[s[t]];
    }
    __syncthreads();
    for (u64 k = k_lo; k <= k_hi; k <<= 1) {
        for (u64 j = min(k >> 1, (u64)kSortChunk >> 1); j > 0; j >>= 1) {
            const int t = threadIdx.x;
            const int i = (int)(((t & ~((int)j - 1)) << 1) | (t & ((int)j - 1)));   // lower index of the pair
            const int ixj = i | (int)j;
            const bool asc = ((base + i) & k) == 0;
            const u32 x = s[i], y = s[ixj];
            const ulonglong2 kx = sk[i], ky = sk[ixj];
            bool swap;
            if (x == 0xFFFFFFFFu || y == 0xFFFFFFFFu) swap = asc ? row_less(a, y, x) : row_less(a, x, y);
            else {
                const int c = key_cmp(kx, ky);
                swap = c ? (asc ? c > 0 : c < 0) : (asc ? row_less(a, y, x) : row_less(a, x, y));
            }
            if (swap) { s[i] = y; s[ixj] = x; sk[i] = ky; sk[ixj] = kx; }
            __syncthreads();
        }
    }
    for (int t = threadIdx.x; t < kSortChunk; t += blockDim.x) if (base + t < a.n_pad) a.sort_idx[base + t] = s[t];
}
__global__ void __launch_bounds__(256) k_out_gather(const PostArgs a, u64 n_keep) {   // one warp per row
    const u64 r = (u64)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (r >= n_keep) return;
    const int lane = threadIdx.x & 31;
    const u32 src = a.sort_idx[r];
    const int n = a.u_nnz[src];
    if (lane == 0) { a.r_nnz[r] = n; a.r_steps[r] = a.u_steps[src]; }
    for (int t = lane; t < n; t += 32) { a.r_rxn[r * a.D + t] = a.u_rxn[(u64)src * a.D + t]; a.r_val[r * a.D + t] = a.u_val[(u64)src * a.D + t]; }
}

// Compressed rows (CSR) of the final result: row pointer by a three-step scan (1024-row blocks, their totals, the sum),
// then one warp per row.
__global__ void __launch_bounds__(1024) k_csr_scan_blocks(const int* __restrict__ r_nnz, u64 K, i64* __restrict__ row_ptr, i64* __restrict__ totals) {
    __shared__ i64 part[1024];
    const u64 r = (u64)blockIdx.x * 1024 + threadIdx.x;
    const i64 v = r < K ? r_nnz[r] : 0;
    part[threadIdx.x] = v;
    __syncthreads();
    for (int off = 1; off < 1024; off <<= 1) {
        const i64 x = threadIdx.x >= off ? part[threadIdx.x - off] : 0;
        __syncthreads();
        part[threadIdx.x] += x;
        __syncthreads();
    }
    if (r < K) row_ptr[r] = part[threadIdx.x] - v;   // exclusive, block-local
    if (threadIdx.x == 1023) totals[blockIdx.x] = part[1023];
}
__global__ void __launch_bounds__(1024) k_csr_scan_totals(i64* __restrict__ totals, u64 n_blocks, u64 K, i64* __restrict__ row_ptr, Ctl* ctl) {
    __shared__ i64 part[1024];
    __shared__ i64 carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (u64 base = 0; base < n_blocks; base += 1024) {
        const u64 b = base + threadIdx.x;
        const i64 v = b < n_blocks ? totals[b] : 0;
        part[threadIdx.x] = v;
        __syncthreads();
        for (int off = 1; off < 1024; off <<= 1) {
            const i64 x = threadIdx.x >= off ? part[threadIdx.x - off] : 0;
            __syncthreads();
            part[threadIdx.x] += x;
            __syncthreads();
        }
        if (b < n_blocks) totals[b] = carry + part[threadIdx.x] - v;   // exclusive offset of block b
        __syncthreads();
        if (threadIdx.x == 1023) carry += part[1023];
        __syncthreads();
    }
    if (threadIdx.x == 0) { row_ptr[K] = carry; ctl->csr_nnz = (u64)carry; }
}
__global__ void __launch_bounds__(256) k_csr_pack(const PostArgs a, u64 K, i64* __restrict__ row_ptr, const i64* __restrict__ totals,
                                                  int* __restrict__ c_rxn, i64* __restrict__ c_val) {
    const u64 r = (u64)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (r >= K) return;
    const int lane = threadIdx.x & 31, n = a.r_nnz[r];
    const i64 o = row_ptr[r] + totals[r >> 10];
    __syncwarp();
    if (lane == 0) row_ptr[r] = o;
    for (int t = lane; t < n; t += 32) { c_rxn[o + t] = a.r_rxn[r * a.D + t]; c_val[o + t] = a.r_val[r * a.D + t]; }
}
cudaError_t launch_output_csr(const PostArgs& a, u64 K, i64* row_ptr, int* c_rxn, i64* c_val, cudaStream_t s, int* n_launches) {
    // block totals live behind the row pointer (the region holds capacity + 1 + capacity / 1024 + 2 entries)
    i64* totals = row_ptr + a.max_cand + 1;
    const u64 nb = (K + 1023) / 1024;
    if (nb) { k_csr_scan_blocks<<<(unsigned)nb, 1024, 0, s>>>(a.r_nnz, K, row_ptr, totals); ++*n_launches; }
    k_csr_scan_totals<<<1, 1024, 0, s>>>(totals, nb, K, row_ptr, a.ctl);
    ++*n_launches;
    if (K) { k_csr_pack<<<(unsigned)((K + 7) / 8), 256, 0, s>>>(a, K, row_ptr, totals, c_rxn, c_val); ++*n_launches; }
    return cudaGetLastError();
}

cudaError_t launch_output_rows(const PostArgs& a, u64 K, cudaStream_t s, int* n_launches) {
    if (K == 0) return cudaSuccess;
    k_out_rows<<<(unsigned)((K + 7) / 8), 256, 0, s>>>(a, K);
    ++*n_launches;
    return cudaGetLastError();
}
cudaError_t launch_output_sort(const PostArgs& a, u64 n_keep, cudaStream_t s, int* n_launches) {
    if (n_keep == 0) return cudaSuccess;
    const unsigned blocks = (unsigned)((a.n_pad + 255) / 256);
    k_sort_init<<<blocks, 256, 0, s>>>(a, n_keep);
    ++*n_launches;
    const unsigned chunks = (unsigned)((a.n_pad + kSortChunk - 1) / kSortChunk);
    const u64 k_local_hi = a.n_pad < (u64)kSortChunk ? a.n_pad : (u64)kSortChunk;
    k_bitonic_local<<<chunks, kSortChunk / 2, 0, s>>>(a, 2, k_local_hi);
    ++*n_launches;
    for (u64 k = (u64)kSortChunk * 2; k <= a.n_pad; k <<= 1) {
        for (u64 j = k >> 1; j >= (u64)kSortChunk; j >>= 1) { k_bitonic_global<<<blocks, 256, 0, s>>>(a, j, k); ++*n_launches; }
        k_bitonic_local<<<chunks, kSortChunk / 2, 0, s>>>(a, k, k);
        ++*n_launches;
    }
    k_out_gather<<<(unsigned)((n_keep + 7) / 8), 256, 0, s>>>(a, n_keep);
    ++*n_launches;
    return cudaGetLastError();
}

__global__ void __launch_bounds__(256) k_densify(const int* r_nnz, const int* r_rxn, const i64* r_val, int D, int n_rxn,
                                                 i64 row0, i64 n_rows, i64* out) {
    const i64 r = (i64)blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32;
    if (r >= n_rows) return;
    const int lane = threadIdx.x & 31;
    const i64 src = row0 + r;
    const int n = r_nnz[src];
    for (int t = lane; t < n; t += 32) out[r * n_rxn + r_rxn[src * D + t]] = r_val[src * D + t];
}
cudaError_t launch_densify(const int* r_nnz, const int* r_rxn, const i64* r_val, int D, int n_rxn, i64 row0, i64 n_rows,
                           i64* d_out, cudaStream_t s) {
    if (n_rows <= 0) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(d_out, 0, (size_t)n_rows * n_rxn * sizeof(i64), s);
    if (e != cudaSuccess) return e;
    k_densify<<<(unsigned)((n_rows + 7) / 8), 256, 0, s>>>(r_nnz, r_rxn, r_val, D, n_rxn, row0, n_rows, d_out);
    return cudaGetLastError();
}

__global__ void k_debug_hash(int n_supp, const int* arc, const i64* flux, int n_vis, const int* vis4, u64* out) {
    u64 s = 0;
    for (int t = 0; t < n_supp; ++t) s += arc_term((u32)arc[t], (u64)flux[t]);
    for (int u = 0; u < n_vis; ++u) s += vis_term(vis_pack((u32)vis4[4 * u], (u32)vis4[4 * u + 1], (u32)vis4[4 * u + 2], (u32)vis4[4 * u + 3]));
    *out = mix64(s);
}
cudaError_t launch_debug_hash(int n_supp, const int* arc, const i64* flux, int n_vis, const int* vis4, u64* out, cudaStream_t s) {
    k_debug_hash<<<1, 1, 0, s>>>(n_supp, arc, flux, n_vis, vis4, out);
    return cudaGetLastError();
}

}  // namespace efm
