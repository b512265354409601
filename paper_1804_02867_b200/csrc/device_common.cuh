// Types shared by the kernels and the host driver.  Notation follows the paper: M internal metabolites (nodes),
// I / O input / output reaction arrays of a node, c coefficient, f flux, EF extra flux (Eq 2),
// PI / PO primary input / output (Def 10).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace efm {

typedef unsigned long long u64;
typedef long long i64;
typedef unsigned int u32;
typedef unsigned short u16;

// ---------------------------------------------------------------------------------------------------------------
// Entry format in HBM.  Frontier entries are PACKED back to back (16-byte aligned); entry
// indices and 16-byte units come from ONE packed atomic, so entries with consecutive indices are contiguous and the
// size of entry p is off[p + 1] - off[p].  An entry is
//   [ 0,48)  header: u32 n_supp | n_vis << 16; u32 n_unb | ones << 16 (ones = number of fluxes equal to 1);
//            u64 hs = sum of the arc terms of the state hash;
//            u64 hv = sum of its visited terms; u64 big = max(largest flux, largest |EF|);
//            i64 E = EF of i*; u32 i* | (vk + 1) << 16 (i* = lowest unbalanced metabolite, reading G12; vk = index of
//            its visited record, vk + 1 = 0: first visit); u32 root / sampled candidate the pathway descends from
//            (candidate slots: the number of expansions that built the pathway)
//   i64  flux[n_supp]   fluxes of the support arcs, > 0, gcd 1
//   u64  vis[n_vis]     visited records: cnt << 48 | met << 32 | PI << 16 | PO   (unordered)
//   i64  ef[n_unb]      the non-zero extra fluxes EF_i (Eq 2) of the state   (unordered)
//   u16  arc[n_supp]    support arcs, ascending arc id
//   u16  efmet[n_unb]   metabolite of each ef[] element
// hs / hv / big / ef[] / E / i* / vk are derived data the producer has in registers anyway: carrying them saves the
// consumer the re-hash of the parent, the Eq 2 scatter over the support, the search for i* and the scan of the visited
// list (children update the EF list incrementally: EF' = (k EF + sign d s_.a) / g).  A candidate slot (fixed stride)
// holds the same with n_vis = n_unb = 0.
// ---------------------------------------------------------------------------------------------------------------
constexpr u32 kHdr = 48;   // header bytes of a frontier / candidate entry
__host__ __device__ inline u32 entry_bytes(u32 n_supp, u32 n_vis, u32 n_unb) {
    return (kHdr + 10u * n_supp + 8u * n_vis + 10u * n_unb + 15u) & ~15u;
}
// irreducible content of an entry, the unit of the algorithmic-byte count
__host__ __device__ inline u32 algo_entry_bytes(u32 n_supp, u32 n_vis) { return n_supp * 10u + n_vis * 7u + 16u; }
// packed allocation counter of a frontier: entry count in the high 30 bits, 16-byte units in the low 34
// (2^34 units = 256 GB, more than a B200 holds)
constexpr int kAllocShift = 34;
constexpr u64 kAllocUnitMask = (1ULL << kAllocShift) - 1ULL;
// parent list word (k_order): 16-byte unit offset of the entry in the low 40 bits, its size in units above
constexpr int kListShift = 40;
constexpr u64 kListOffMask = (1ULL << kListShift) - 1ULL;

struct DevGraph {
    int M, A, W32, M32;
    const int* col_ptr;   const int2* col;    // column of an arc: {met | pos << 16, s}; pos = index of the arc in I[met] (s > 0) / O[met] (s < 0)
    const int4* node;                          // per metabolite {in0, |I|, out0, |O|}: its slices of in_e / out_e
    const int2* in_e;                          // I[i]: {arc, c}, ascending arc id
    const int2* out_e;                         // O[i]
    // per entry of in_e / out_e one 32-byte record with everything the lane-parallel evaluation of that OR-alternative
    // needs: {arc | c << 16, twin | ncol << 16 | generic << 24, 6 x (met | s << 16)}; generic = 1: the column has more
    // than 6 entries or a number does not fit 16 bits, take the general routine
    const uint4* in_alt;  const uint4* out_alt;
    const u64* colsig;    // per arc two words: bit (met & 63) set for every metabolite the arc produces / consumes (filter of the column scans)
    const int* twin;
    const i64* dep_off;   const u32* dep_bits;
    const int* arc_rxn;   const int* arc_dir;
    const u64* arc_mix;   // m_a = mix64(0x01 << 56 | a): the multiplier of arc a in the state hash
    int max_coef;         // largest |s_ia| of the network (bounds the lane-parallel fast path)
};
__host__ __device__ inline int col_met(const int2& e) { return e.x & 0xffff; }
__host__ __device__ inline int col_pos(const int2& e) { return (int)((unsigned)e.x >> 16); }

// Device-resident control block: per-level counters (two sets, alternating with the level parity, so that a whole batch
// of levels runs without the host), beam-select state, cumulative statistics.
enum { ST_CHILDREN = 0, ST_DEAD_END, ST_NOT_EFM, ST_NONPOS, ST_OVERFLOW, ST_VISITED, ST_ALGO_BYTES, ST_EXPANDED,
       // work profile (not part of the oracle parity): first-visit parents, children through the general routine
       ST_FIRST, ST_GENERAL, ST_COUNT };
enum { ERR_FRONTIER = 1, ERR_CAND = 2, ERR_KEYS = 4, ERR_LEVELS = 8 };
enum { SEL_BINS = 2048 };

struct LevelCtl {
    u64 alloc;         // packed allocator of the entries OF this level (count << 34 | 16-byte units); its children
                       // allocate in the other set
    u64 nF, nR;        // first-visit / revisit parents listed by k_order
    u64 work;          // next work item of k_expand (dynamic distribution)
    u64 n_slots;       // key slots reserved (chunked per warp; unused slots hold kKeySentinel)
    u64 n_tasks;       // task slots reserved (children of the general routine)
    u64 n_keys;        // active children generated
    u64 n_done;        // balanced children generated
    u64 n_surv;        // children of the level that are materialised (k_compact)
    u64 pad[7];
};
// per-level record kept for the host (efm_get_level_stats), written by k_materialise of the level
struct LevelStats { u64 parents, active_children, done_children, kept, surv, pad[3]; };

struct Ctl {
    LevelCtl lv[2];
    u64 n_cand;        // candidates emitted so far
    u32 error, pad0;
    u64 X;             // beam threshold: keep key < X
    u64 sel_prefix, sel_rank, n_compact;
    u32 sel_ticket, pad1;
    u64 st[ST_COUNT];
    // post-processing counters
    u64 n_unique, n_poisoned, n_uniq_ok, n_keep, filter_pairs, csr_nnz;
    // everything above is read back by the host; the histogram stays on the device
    u32 hist[SEL_BINS];
};

struct ExpandArgs {
    DevGraph g;
    const unsigned char* cur;   // parents (packed)
    const u64* cur_off;         // 16-byte-unit offset of entry p of the current level, allocation order
    u64* plist;                 // parent list of the level (k_order): first-visit parents from the front, revisit parents from
                                // the back (index max_frontier - 1 - j); word = offset | size << 40 (16-byte units)
    u32* pprim;                 // per parent-list index: primary arc chosen at a first visit (reading G13), set by k_expand
    unsigned char* nxt;         // children that stay active (packed)
    u64* nxt_off;
    unsigned char* cand;        // balanced children (fixed stride)
    u64* keys;                  // per child slot: beam key (kKeyDone: balanced child; kKeySentinel: unused slot)
    u64* tags;                  // per child slot: parent-list index << 34 | kind << 32 | payload (see k_expand)
    uint4* tasks;               // 4 x 16 bytes per child of the general routine (see k_expand / k_materialise)
    ulonglong2* surv;           // children that are materialised: {slot, offset of the parent entry in 16-byte units}
    u64* surv_dst;              // ... and where they go: bit 63 set: candidate slot, else 16-byte unit offset in the next
                                // frontier (its entry index was written to nxt_off by k_compact); ~0: capacity exceeded
    LevelStats* lvl;            // per-level records
    Ctl* ctl;
    u32 level, par;             // level of the parents, its parity
    u32 max_entry, cand_stride; // largest entry in bytes, candidate slot stride
    u64 max_frontier, frontier_units, max_cand, max_keys, max_tasks, max_surv, max_levels;
    u64 cap;                    // beam: entries kept per level, 0 = unbounded
    int D, V, max_loop;
    // SURVEY.md 8(f)-1 literal sampling (one alternative per first visit, chosen by sample_pick) and 8(f)-2 reaction mask
    u64 sample_seed; u32 sample; // sample != 0: sampling mode
    const u32* amask;           // bit per arc: its reaction is in the allowed subset (nullptr: all)
    u64* cand_end;              // sampling mode: per candidate how and when it ended (END_* | steps << 8)
    int force_inplace;          // EFM_F_NO_STAGING: read every parent in place
    int no_fast;                // EFM_F_NO_FASTPATH: every child through the warp-cooperative general routine
    // shared-memory carve-up per warp (bytes)
    u32 sm_group, sm_stage_bytes, sm_sbits, sm_upos, sm_misc;
};

// roots (INIT): seed sets uploaded by the host, entries built and classified on the device
struct RootArgs {
    DevGraph g;
    const int* seed_ptr; const int* seed_arc;   // CSR of arc ids, ascending inside a set
    const u64* stage_off;                       // 16-byte-unit offset of root r in the staging buffer
    unsigned char* stage;                       // root entries (packed), built by the count pass
    unsigned char* nxt; u64* nxt_off;           // surviving active roots
    unsigned char* cand;
    u64* keys;                                  // one key per root (kKeySentinel for balanced roots)
    LevelStats* lvl;                            // record 0: the roots as children of a level "-1"
    Ctl* ctl;
    u64 n_roots;
    u32 cand_stride;
    u64 max_frontier, frontier_units, max_cand, cap;
    u64* cand_end;
};

// ---------------------------------------------------------------------------------------------------------------
// SURVEY.md 8(c)-B state hash: written here from the formula, independently of oracle/.
//   mix = SplitMix64 finaliser
//   h = mix( sum_{a in supp} mix(0x01<<56 | a) * f_a + sum_{i visited} mix(0x02<<56 | cnt<<48 | i<<32 | PI<<16 | PO) )
//   key = min(n_unb, 255) << 56 | h >> 8
// (sums and products modulo 2^64).  The arc part is linear in the flux vector: the sum of a child whose fluxes are
// k f + d e_a is k hs + m_a d, no pass over the support (only a common divisor g > 1 needs one).
// ---------------------------------------------------------------------------------------------------------------
__host__ __device__ inline u64 mix64(u64 x) {
    x ^= x >> 30; x *= 0xBF58476D1CE4E5B9ULL;
    x ^= x >> 27; x *= 0x94D049BB133111EBULL;
    x ^= x >> 31; return x;
}
__host__ __device__ inline u64 arc_term(u32 a, u64 f) { return mix64(0x0100000000000000ULL | (u64)a) * f; }
__host__ __device__ inline u64 vis_term(u64 rec) { return mix64(0x0200000000000000ULL | rec); }
__host__ __device__ inline u64 vis_pack(u32 met, u32 PI, u32 PO, u32 cnt) {
    return ((u64)cnt << 48) | ((u64)met << 32) | ((u64)PI << 16) | (u64)PO;
}
__host__ __device__ inline u64 beam_key(u32 n_unb, u64 h) { return ((u64)(n_unb > 255u ? 255u : n_unb) << 56) | (h >> 8); }

// how a sampled candidate ended, code | steps << 8
enum { END_NONE = 0, END_DONE = 1, END_NOTEFM = 2, END_DEAD = 3, END_VISITED = 4, END_NONPOS = 5, END_OVERFLOW = 6 };
// alternative candidate c takes at the first visit of metabolite i (reading G23, written here independently of oracle/):
//   pick(seed, c, i) = mix( mix(seed + 0x9E3779B97F4A7C15 * (c + 1)) ^ (0x04 << 56 | i) ), index = pick mod (admissible alternatives)
__host__ __device__ inline u64 sample_pick(u64 seed, u32 cand, u32 met) {
    return mix64(mix64(seed + 0x9E3779B97F4A7C15ULL * ((u64)cand + 1ULL)) ^ (0x0400000000000000ULL | (u64)met));
}
constexpr u64 kKeyDone = ~0ULL - 1ULL;   // key slot of a balanced child: always materialised, outside the beam ranking
enum { TF_NEG = 1, TF_FIRST = 2, TF_INSUPP = 4 };   // task flags: bump subtracts (Eq 5); first visit; arc already in the support
// child tag: [63:34] parent-list index, [33:32] kind, [31:0] payload
//   kind 0: first-visit child on a new arc, evaluated lane-parallel: payload = alternative index q << 16 | n_unb of the child
//           (k_materialise rebuilds it from the parent, the OR-alternative record q and pprim[parent])
//   kind 1: child of the general routine: payload = index of its 64-byte task
constexpr int kTagParentShift = 34;
enum { TK_FAST = 0, TK_TASK = 1 };
constexpr u64 kKeySentinel = ~0ULL;   // filler of reserved but unused key slots: never < X, skipped by the select
#ifndef EFM_KEYCHUNK
#define EFM_KEYCHUNK 64
#endif
constexpr u32 kKeyChunk = EFM_KEYCHUNK;   // key slots a warp reserves per atomic

#define EFM_GUARD (1ULL << 62)   // reading G21: any state integer above 2^62 discards the pathway

}  // namespace efm
