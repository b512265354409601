/*
 * efm_b200.h -- C ABI of the B200 (sm_100a) library for the data-parallel hot path of
 * arXiv 1804.02867 ("A system architecture for parallel analysis of flux-balanced metabolic
 * pathways"): the AND/OR-graph pathway traversal (Alg 1 + Alg 3 METAx).
 *
 * Problem statement the interface follows (Alg 1): "Input: the stoichiometric
 * matrix of a given metabolic network.  Output: a set of minimal flux-balanced pathways"; the
 * reversibility flags and the internal/external split are properties of the input network
 * and the set of initial reactions is a user choice.
 *
 * Conventions
 *   - every function returns EFM_OK (0) or a negative EFM_E_* code; nothing throws;
 *   - "host" / "device" is stated for every pointer; host inputs are caller-owned and copied;
 *   - the library never allocates device memory: the caller (PyTorch in this repo) owns one
 *     workspace allocation and the CUDA stream, both passed to efm_enumerate();
 *   - results live inside the workspace and are invalidated by the next efm_enumerate() on
 *     the handle, by freeing the workspace, or by efm_destroy();
 *   - a handle is not thread-safe;
 *   - the work is done by CUDA kernels only: there is no CPU fallback.  Without a usable
 *     CUDA device efm_enumerate() fails with EFM_E_CUDA.
 */
#ifndef EFM_B200_H
#define EFM_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define EFM_OK 0
#define EFM_E_INVAL (-1)    /* bad pointer / shape / parameter / seed set                         */
#define EFM_E_NOMEM (-2)    /* workspace smaller than efm_workspace_bytes() reports               */
#define EFM_E_CAPACITY (-3) /* a frontier / candidate / key buffer overflowed: results undefined, */
                            /* never silently truncated                                           */
#define EFM_E_CUDA (-4)     /* CUDA runtime error (text retained for efm_last_error())            */
#define EFM_E_STATE (-5)    /* result accessor called before a successful efm_enumerate()         */

/* flags */
#define EFM_F_TIMING 0x1u       /* record CUDA events around every kernel phase (efm_stats.ms_*)   */
#define EFM_F_NO_FASTPATH 0x4u  /* evaluate every child with the warp-cooperative general routine  */
#define EFM_F_NO_STAGING 0x8u   /* read every parent in place (the route of entries larger than the   */
                                /* shared-memory staging buffer)                                      */

#define EFM_F_EXACT_ELEMENTARITY 0x10u /* replace "minimal among the candidates found" by the rank test    */
                                /* of Def 3: a support stays iff the internal rows of S restricted */
                                /* to it have rank |supp| - 1 over GF(2^31 - 1); needs max_support <= 128               */

#define EFM_F_COMPRESS 0x20u    /* SURVEY.md 8(f)-4 compression pre-pass: efm_create() leaves the reactions    */
                                /* out of the graph that efm_blocked_reactions() reports; results stay in the caller's     */
                                /* reaction space; a seed on such a reaction is EFM_E_INVAL                                 */

typedef struct efm_handle efm_handle; /* opaque: host copy of the graph + pointers INTO the workspace */

/* Traversal parameters.  Alg 1's #defines M, R are taken from S; C (number of
 * candidate blocks) is replaced by the beam `frontier_cap`; r_max / m_max / #B / #T are thread-index
 * artefacts of the paper's mapping and do not exist here. */
typedef struct {
    int32_t max_support;    /* D: max arcs in a pathway; 0 = number of arcs                          */
    int32_t max_loop;       /* MAX_LOOP; 0 = 8                          */
    int32_t dep_depth;      /* L: chain length of the dependent-reaction search; 0 = 4 */
    int32_t max_visited;    /* V: max visited metabolites per pathway; 0 = 2*D                       */
    int64_t frontier_cap;   /* beam: entries expanded per level; 0 = unbounded                       */
    int64_t max_frontier;   /* entries per frontier buffer; 0 = max(frontier_cap, 4096), 2^20 when cap == 0 */
    int64_t max_candidates; /* capacity of the candidate buffer / support hash; 0 = 2^20             */
    int64_t max_child_keys; /* child slots per level (8-byte beam key + 8-byte tag each, < 2^32);    */
                            /* 0 = max(frontier_cap * the largest fan-out of a node, sample_count,   */
                            /* 65536): never overflows with a beam or in sampling mode; an unbounded */
                            /* run (frontier_cap 0) with more children in a level, or a smaller      */
                            /* explicit value, reports EFM_E_CAPACITY when exceeded                  */
    int32_t device;         /* CUDA device ordinal the workspace lives on                            */
    uint32_t flags;         /* EFM_F_*                                                               */
    int64_t max_frontier_bytes; /* bytes of one frontier buffer (entries are packed, variable size);         */
                            /* 0 = max_frontier * the largest possible entry, which can never overflow;      */
                            /* a smaller value saves HBM and reports EFM_E_CAPACITY if a level outgrows it   */
    int64_t max_child_tasks; /* 64-byte tasks per level (children on arcs of the support: every revisit, some     */
                            /* alternatives of a first visit); 0 = 4 * max_frontier + 65536 (max_child_keys with     */
                            /* EFM_F_NO_FASTPATH); EFM_E_CAPACITY when exceeded                                      */
    int64_t sample_count;   /* SURVEY.md 8(f)-1 literal sampling mode ("each pathway is created using randomly */
                            /* selected output/input"; "after attempting 48 EFM candidates"): C > 0 runs C     */
                            /* candidate pathways; candidate c starts from seed set c mod n_sets and takes ONE admissible   */
                            /* alternative per first visit (counter-based generator keyed on (sample_seed, c, metabolite),  */
                            /* DESIGN.md reading G23); no fan-out, frontier_cap is ignored; needs C <= max_frontier         */
    uint64_t sample_seed;
} efm_params;

typedef struct {
    int64_t levels, expanded, children, done, dead_end, not_efm_maxloop, discarded_nonpos,
        discarded_overflow, discarded_visited, truncated_beam, unique_supports, poisoned, output;
    int64_t peak_frontier;  /* largest number of active entries in a level, before the beam          */
    int64_t algo_bytes;     /* algorithmic bytes of all expansions            */
    int64_t n_roots;
    int64_t launches;       /* kernels launched by the last efm_enumerate()                          */
    int64_t two_pass_levels, direct_levels; /* levels enqueued with / without the threshold selection (frontier_cap > 0 / = 0) */
    int64_t h2d_bytes;      /* bytes efm_enumerate() copied host -> device (graph on first use, seed sets)          */
    int64_t host_syncs;     /* stream synchronisations inside efm_enumerate(): one per batch of levels + post stages */
    /* milliseconds; ms_total is always measured (CUDA events on the caller's stream), the per-phase
     * figures only with EFM_F_TIMING */
    double ms_build, ms_total, ms_order, ms_expand_count, ms_beam, ms_expand_write, ms_hash, ms_filter, ms_output;
    /* ms_order: k_order (parents by kind); ms_expand_count: k_expand (evaluates every child: beam key + tag);
     * ms_beam: threshold selection; ms_expand_write: k_compact + k_materialise (survivors -> next frontier / candidates) */
    int64_t n_expand_count; /* levels enqueued (levels behind the end of the traversal return at once)                 */
    int64_t filter_pairs;   /* signature pair tests done by the minimality filter                    */
    /* work profile of the expansion: first-visit parents, children through the general routine, children materialised */
    int64_t first_visits, general_children, materialised;
    int64_t non_elementary; /* EFM_F_EXACT_ELEMENTARITY: unique, unpoisoned supports the rank test rejected          */
    int64_t blocked_reactions; /* EFM_F_COMPRESS: reactions left out of the graph                                    */
} efm_stats;

/* Build the modified AND/OR graph MG (Defs 4-6; "Convert the given matrix to the MG
 * graph structure") and the static flux-dependency table (Def 11, PAPER.md:130;
 * Alg 2 DEPTHy).
 *   S          host, int32, m x n, element (i, j) at S[i*row_stride + j]; > 0 produced, < 0 consumed
 *
 *   reversible host, uint8[n]; nonzero = reaction j may run backwards (split into two arcs)
 *   internal   host, uint8[m]; nonzero = metabolite i is internal (balanced); others are external
 *   p          host; NULL = all defaults
 *   out        host; receives the handle (free with efm_destroy)
 * Errors: EFM_E_INVAL for NULL pointers, m/n <= 0, more than 65535 arcs or internal metabolites,
 * negative parameters. */
int efm_create(const int32_t* S, int32_t m, int32_t n, int64_t row_stride, const uint8_t* reversible,
               const uint8_t* internal, const efm_params* p, efm_handle** out);

/* Compression pre-pass ("partitioning and compression preprocessing methods"): the reactions
 * that cannot carry flux in any steady state (Def 2) for a topological reason.  An internal metabolite whose
 * remaining reactions offer no pair (one that can produce it, another one that can consume it) forces all of them to
 * zero; they are removed and the rule is iterated to its fixed point.  Host only, no handle needed.
 *   S, m, n, row_stride, reversible, internal   as for efm_create()
 *   blocked    host, uint8[n] out: 1 = blocked
 *   n_blocked  host out (may be NULL) */
int efm_blocked_reactions(const int32_t* S, int32_t m, int32_t n, int64_t row_stride, const uint8_t* reversible,
                          const uint8_t* internal, uint8_t* blocked, int32_t* n_blocked);

/* Sizes of the graph: internal metabolites M, arcs A, 64-bit bitset words W = ceil(A/64), nonzeros of the
 * internal arc columns, entries of the dependency table (sum over nodes of |O| * |I|).  All host. */
int efm_graph_info(const efm_handle* h, int32_t* n_internal, int32_t* n_arcs, int32_t* bitset_words,
                   int64_t* nnz, int64_t* dep_entries);

/* Copy the host-side graph out (builder tests).  Every pointer is host memory sized from
 * efm_graph_info(): arc_rxn/arc_dir/twin [A]; in_ptr/out_ptr [M+1]; in_arc/in_c and out_arc/out_c
 * [in_ptr[M]] / [out_ptr[M]]; col_ptr [A+1]; col_met/col_s [nnz]; dep_off [M+1]; dep [dep_entries]
 * with dep[dep_off[i] + lo*|I_i| + le] = 1 iff (O_i[lo], I_i[le]) are flux-dependent.  NULLs are skipped. */
int efm_graph_export(const efm_handle* h, int32_t* arc_rxn, int32_t* arc_dir, int32_t* twin, int32_t* in_ptr,
                     int32_t* in_arc, int64_t* in_c, int32_t* out_ptr, int32_t* out_arc, int64_t* out_c,
                     int32_t* col_ptr, int32_t* col_met, int64_t* col_s, int64_t* dep_off, uint8_t* dep);

/* Bytes of device workspace efm_enumerate() needs for this handle's parameters (host out). */
int efm_workspace_bytes(const efm_handle* h, size_t* bytes);

/* Run the traversal (INIT + METAx), the support dedup, the minimality filter
 * (Def 3) and the canonical output stage, all on the device.
 *   seed_ptr      host, int32[n_sets+1], CSR offsets into seed_arc_code
 *   seed_arc_code host, int32: 2*j + (direction < 0) for reaction j; each set becomes one root pathway
 *                 with those arcs at flux 1
 *   n_sets        0 = default seeds: one root per boundary arc (Def 8)
 *   d_workspace   DEVICE memory, >= efm_workspace_bytes(), 256-byte aligned, caller-owned
 *   cuda_stream   a cudaStream_t (NULL = default stream); all work is enqueued there and the call
 *                 returns after the stream has been synchronised
 * Errors: EFM_E_INVAL (bad seed: unknown code, duplicate, both twins, backward arc of an irreversible
 * reaction, empty or larger than D), EFM_E_NOMEM, EFM_E_CAPACITY, EFM_E_CUDA. */
int efm_enumerate(efm_handle* h, const int32_t* seed_ptr, const int32_t* seed_arc_code, int32_t n_sets,
                  void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/* SURVEY.md 8(f)-2 targeted observability ("contributing reactions of each EFM were selected intentionally",
 * PAPER.md:392-396): restrict the OR-alternatives to a subset of the reactions for the following efm_enumerate() calls.
 *   allowed  host, uint8[n]; allowed[j] = 0 makes every alternative of reaction j (both directions) inadmissible;
 *            NULL lifts the restriction.  Seed sets are the caller's choice and are not checked against the subset.
 * Together with efm_result_steps() this answers whether, and in how many expansions, a known pathway is constructed. */
int efm_set_reaction_mask(efm_handle* h, const uint8_t* allowed);

/* The graph arrays are uploaded into the workspace by the first efm_enumerate() that sees a given workspace
 * pointer and are assumed resident afterwards (the network is an input that stays in HBM across calls).  A caller
 * that overwrites the workspace, or frees it and gets the same address back, must call this before the next run. */
int efm_workspace_invalidate(efm_handle* h);

/* Number of pathways found (host out). */
int efm_result_count(const efm_handle* h, int64_t* n_pathways);

/* Dense result: flux is HOST memory, capacity_rows x n int64 row-major; row r = coprime integer flux
 * vector in reaction space (v_j = f_j+ - f_j-), rows in strict lexicographic order.  Rows are densified
 * on the device in chunks and copied back.  EFM_E_INVAL if capacity_rows < count. */
int efm_result_copy(const efm_handle* h, int64_t* flux, int64_t capacity_rows);

/* Sparse result to HOST memory: nnz[count]; rxn and val are count x row_capacity (row_capacity from
 * efm_result_sparse_stride()), entries beyond nnz[r] are unspecified; rxn ascending within a row. */
int efm_result_sparse_stride(const efm_handle* h, int32_t* row_capacity);
int efm_result_copy_sparse(const efm_handle* h, int32_t* nnz, int32_t* rxn, int64_t* val, int64_t capacity_rows);

/* Steps of every pathway to HOST memory (int32[count], same order as the rows): the number of expansions that built it,
 * the smallest over its equal duplicates (the "steps" of PAPER.md:376-388, one metabolite per step, reading G12). */
int efm_result_steps(const efm_handle* h, int32_t* steps, int64_t capacity_rows);

/* Sampling mode: how every candidate ended, HOST int64[capacity]: code | steps << 8 with code 1 = balanced (Done),
 * 2 = notEFM (MAX_LOOP), 3 = no admissible alternative, 4 = visited cap, 5 = non-positive flux (Prop 3),
 * 6 = above the 2^62 guard; steps = expansions made.  *n_candidates receives C (0 outside sampling mode). */
int efm_sample_ends(const efm_handle* h, int64_t* code_steps, int64_t capacity, int64_t* n_candidates);

/* Compressed sparse rows to HOST memory (pinned memory makes the copies fast): row_ptr[count+1], then rxn / val with
 * efm_result_nnz() entries; row r occupies [row_ptr[r], row_ptr[r+1]), reactions ascending.  The copies are enqueued
 * on `cuda_stream` and the call returns after they completed. */
int efm_result_nnz(const efm_handle* h, int64_t* total_nnz);
int efm_result_copy_csr(const efm_handle* h, int64_t* row_ptr, int32_t* rxn, int64_t* val, void* cuda_stream);

/* DEVICE pointers to the sparse result inside the workspace (same layout as above). */
int efm_result_device(const efm_handle* h, const int32_t** d_nnz, const int32_t** d_rxn, const int64_t** d_val);

/* Densify rows [row0, row0+n_rows) into caller-owned DEVICE memory d_out (n_rows x n int64) on `cuda_stream`. */
int efm_result_densify(const efm_handle* h, int64_t row0, int64_t n_rows, int64_t* d_out, void* cuda_stream);

int efm_get_stats(const efm_handle* h, efm_stats* st);

/* Per-level counters of the last run (host out, each `capacity` long; returns the number of levels through
 * *n_levels): active entries before the beam, balanced (Done) entries, entries expanded, children generated. */
int efm_get_level_stats(const efm_handle* h, int64_t* active, int64_t* done, int64_t* expanded, int64_t* children,
                        int64_t capacity, int64_t* n_levels);

/* Beam key of an explicit state, computed by a one-thread kernel on `device`; test hook
 * for the device copy of the state hash.  All pointers host. vis4 rows are (met, PI, PO, cnt). */
int efm_debug_state_hash(int32_t device, int32_t n_supp, const int32_t* arc, const int64_t* flux, int32_t n_vis,
                         const int32_t* vis4, uint64_t* hash_out);

/* ---- The beam threshold selection as a call of its own (a-4; "X = the key at sorted position
 * frontier_cap; the level keeps exactly the children with key < X").  Keys are the 64-bit beam keys of one level's
 * child slots; the two largest values (0xFF..FE: balanced child, 0xFF..FF: unused slot) stand outside the ranking.
 *
 * efm_beam_threshold(): the selection exactly as efm_enumerate() runs it (same kernels, same launcher), with its
 * control block and compact key buffer in caller-provided scratch instead of the traversal's workspace.
 *   d_keys       DEVICE, uint64[n_slots]
 *   n_active     number of selectable keys among them (the traversal counts them while it writes them); must be > cap,
 *                since the traversal skips the selection when the beam does not bind (EFM_E_INVAL otherwise)
 *   d_scratch    DEVICE, 256-byte aligned, >= efm_beam_threshold_scratch_bytes(n_slots), caller-owned, contents lost
 *   d_threshold  DEVICE, uint64[1] out
 * Enqueued on `cuda_stream`; returns after the stream has been synchronised. */
int efm_beam_threshold_scratch_bytes(int64_t n_slots, size_t* bytes);
int efm_beam_threshold(const uint64_t* d_keys, int64_t n_slots, int64_t n_active, int64_t cap, void* d_scratch, size_t scratch_bytes,
                       uint64_t* d_threshold, int32_t device, void* cuda_stream);

/* efm_beam_threshold_static(): the same selection for a caller that can hand over its keys and a result slot but has
 * nowhere to get scratch from -- code that runs as a guest inside another program's GPU process (a plug-in of a host
 * application or a serving engine whose own allocator holds all of HBM, a job under a hard memory cap), or a
 * latency-critical loop in which cudaMalloc / cudaFree are off limits because they can stall the whole device.  This
 * call, and everything it calls, allocates no memory of any kind, device or pinned host: the histogram, the rank /
 * prefix words and the compact key buffer sit in ONE array compiled into the library, EFM_STATIC_SELECT_BYTES on every
 * GPU that loads the library, held until the process exits.  That fixes the limit below.
 *   d_keys       DEVICE, uint64[n_keys], read only
 *   n_keys       key slots, 0 .. EFM_STATIC_SELECT_MAX_KEYS; more is refused with EFM_E_CAPACITY before any CUDA call
 *   cap          > 0: sorted position of the threshold (frontier_cap)
 *   d_threshold  DEVICE, uint64[1] out: the key at sorted position cap among the selectable keys; 0xFF..FF (keeps
 *                every selectable key) when there are no more than cap of them -- the call counts them itself
 *   device       ordinal of the GPU that holds d_keys / d_threshold; made current by the call
 *   cuda_stream  the three kernels and one memset are enqueued there; the call does NOT synchronise, the result is
 *                valid once the stream has reached that point
 * Shared state, read this: all calls on one device use the same array.  (1) It keeps whatever the last call left; the
 * call clears the part that must start at zero itself, nothing to do for the caller.  (2) Two calls whose kernels can
 * overlap on the GPU (different streams, or different host threads without ordering between their streams) race on it
 * and both results are garbage: order them on one stream or with events.  (3) The first call on each device looks up
 * where the array lives on that device (once, under a lock); make that first call during start-up, before any stream
 * capture begins.
 * Errors: EFM_E_INVAL (NULL pointer, n_keys < 0, cap <= 0, device outside 0..63), EFM_E_CAPACITY (n_keys above the
 * limit), EFM_E_CUDA; efm_beam_threshold_static_error() gives the text of this thread's last failure ("" after success). */
#define EFM_STATIC_SELECT_MAX_KEYS (1u << 20)
#define EFM_STATIC_SELECT_BYTES (8448u + 8u * EFM_STATIC_SELECT_MAX_KEYS) /* 8 MiB + 8.25 KiB of device memory per GPU */
int efm_beam_threshold_static(const uint64_t* d_keys, int64_t n_keys, int64_t cap, uint64_t* d_threshold, int32_t device,
                              void* cuda_stream);
const char* efm_beam_threshold_static_error(void);

void efm_destroy(efm_handle* h);
const char* efm_strerror(int code);
const char* efm_last_error(const efm_handle* h); /* text of the last CUDA error, "" if none */

#ifdef __cplusplus
}
#endif
#endif /* EFM_B200_H */
