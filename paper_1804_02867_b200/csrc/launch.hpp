// Host-callable launchers of the kernels in expand.cu and post.cu.
#pragma once
#include "device_common.cuh"

namespace efm {

// expand.cu
void expand_smem_layout(ExpandArgs& a);
u64 expand_key_slack(int sm_count);    // key slots the evaluation can strand (one chunk per resident warp)
u64 expand_task_slack(int sm_count);
cudaError_t launch_order(const ExpandArgs& a, int sm_count, cudaStream_t s);
cudaError_t launch_expand(const ExpandArgs& a, int sm_count, cudaStream_t s);
cudaError_t launch_compact(const ExpandArgs& a, int sm_count, cudaStream_t s);
cudaError_t launch_materialise(const ExpandArgs& a, int sm_count, cudaStream_t s);
cudaError_t launch_roots(bool write /*false: build + classify, true: keep the survivors*/, const RootArgs& r, cudaStream_t s);

// post.cu
struct PostArgs {
    DevGraph g;
    Ctl* ctl;
    const unsigned char* cand; u32 cand_stride; u64 max_cand;
    u32* table; u64 table_size;        // open-addressing support hash (a-6), power of two
    unsigned char* isrep; unsigned char* poison;
    u32* c_steps;                      // per candidate: expansions that built it; a representative ends with the minimum over its equal duplicates
    u32* uniq;                         // candidate ids of the unique, unpoisoned supports
    // minimality filter (a-7)
    u32* freq; u32* gcount; u32* gstart; u32* gfill;      // per arc: candidates using it, group size / start / fill
    uint4* r_sig; u32* v_row; u32* vcount; u32* vstart; u32* vfill; u32* tstart;   // join: row-order signatures, rows per (arc, size), tile prefix per arc
    uint2* g_sig64; uint2* r_sig64;                       // first-stage 64-bit bucket signatures, grouped order / row order
    u32* g_row; uint4* g_sig;                             // rows grouped by their rarest arc: candidate id, 112-bit signature + |supp|
    int n_sizes;                                          // D + 1: the (arc, |supp|) bins of gcount / gstart / gfill
    unsigned char* keep;                                  // per unique support (uniq order)
    // canonical output (a-8)
    int D; int n_rxn;
    int* u_nnz; int* u_rxn; i64* u_val;   // unsorted reaction-space rows
    int* u_steps; int* r_steps;            // step count of every row (unsorted / final order)
    ulonglong2* u_key;                     // order codes of the first two entries of every unsorted row
    u32* sort_idx; u64 n_pad;
    int* r_nnz; int* r_rxn; i64* r_val;   // final, lexicographic order
};
cudaError_t launch_select(const u64* keys, u64* ckeys /*compact buffer*/, u64 max_ckeys, Ctl* ctl, int par /*level set holding n_keys / n_slots*/, u64 cap, u64 max_keys, int sm_count, cudaStream_t s, int* n_launches);
cudaError_t launch_dedup(const PostArgs& a, u64 n_cand, cudaStream_t s, int* n_launches);
cudaError_t launch_rank_test(const PostArgs& a, u64 n_uniq, int sm_count, cudaStream_t s, int* n_launches);
cudaError_t launch_filter(const PostArgs& a, u64 n_uniq, int sm_count, cudaStream_t s, int* n_launches);
cudaError_t launch_output_rows(const PostArgs& a, u64 n_uniq, cudaStream_t s, int* n_launches);
cudaError_t launch_output_sort(const PostArgs& a, u64 n_keep, cudaStream_t s, int* n_launches);
cudaError_t launch_output_csr(const PostArgs& a, u64 n_keep, i64* row_ptr, int* c_rxn, i64* c_val, cudaStream_t s, int* n_launches);
cudaError_t launch_densify(const int* r_nnz, const int* r_rxn, const i64* r_val, int D, int n_rxn, i64 row0, i64 n_rows,
                           i64* d_out, cudaStream_t s);
cudaError_t launch_debug_hash(int n_supp, const int* arc, const i64* flux, int n_vis, const int* vis4, u64* out, cudaStream_t s);

}  // namespace efm
