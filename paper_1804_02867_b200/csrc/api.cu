// C ABI of the library (include/efm_b200.h) and the host driver of the level loop (Alg 1 main body).
// The driver only sequences kernels and reads back one small control block per level; every step of the path
// (roots, classify, beam select, expand, dedup, minimality filter, canonical output) runs in the kernels.
#include <algorithm>
#include <cstdio>
#include <chrono>
#include <cstddef>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/efm_b200.h"
#include "device_common.cuh"
#include "graph.hpp"
#include "launch.hpp"

using namespace efm;

namespace {

struct Region { size_t off = 0, bytes = 0; };

struct Layout {
    Region col_ptr, col, colsig, node, in_e, out_e, in_alt, out_alt, twin, dep_off, dep_bits, arc_rxn, arc_dir, arc_mix;
    Region amask, cand_end, c_steps, u_steps, r_steps, g_sig64, r_sig64;
    Region ctl, lvl, buf[2], off[2], plist, pprim, keys, tags, ckeys, tasks, surv, surv_dst, cand, table, isrep, poison, uniq, freq, gcount, gstart, gfill, vcount, vstart, vfill, tstart;
    Region g_row, g_sig, g_size, keep, u_nnz, u_rxn, u_val, u_key, sort_idx, r_nnz, r_rxn, r_val, csr_ptr, dense;
    size_t total = 0;
};

size_t pow2_at_least(size_t x) { size_t p = 1; while (p < x) p <<= 1; return p; }

}  // namespace

struct efm_handle {
    HostGraph G;
    int32_t D = 0, V = 0, max_loop = 8, L = 4;
    int64_t sample_count = 0; uint64_t sample_seed = 0;
    int32_t n_blocked = 0;   // EFM_F_COMPRESS: reactions left out of the graph
    std::vector<uint32_t> amask;   // bit per arc, empty = no restriction (efm_set_reaction_mask)
    int64_t cap = 0, max_frontier = 0, max_cand = 0, max_keys = 0, max_tasks = 0, max_ckeys = 0, max_surv = 0, max_levels = 0;
    int32_t device = 0;
    uint32_t flags = 0;
    uint32_t max_entry = 0, cand_stride = 0;   // largest frontier entry in bytes; candidate slot stride
    int64_t frontier_bytes = 0;                // bytes of one packed frontier buffer
    size_t table_size = 0, dense_bytes = 0;
    Layout lay;
    double ms_build = 0;
    // run state
    unsigned char* ws = nullptr;
    unsigned char* graph_ws = nullptr;   // workspace the graph arrays were last uploaded to
    bool have_result = false;
    int64_t n_out = 0, csr_nnz = 0;
    efm_stats stats;
    std::vector<int64_t> lvl_active, lvl_done, lvl_expanded, lvl_children;
    std::string last_error;
    Ctl* h_ctl = nullptr;   // pinned host mirror of the control block
    int sm_count = 148;
    cudaStream_t stream = nullptr;   // stream of the last efm_enumerate(): the result accessors without a stream argument use it
    std::vector<cudaEvent_t> events;
};

namespace {

void add_region(Layout& L, Region& r, size_t bytes) {
    L.total = (L.total + 255) & ~(size_t)255;
    r.off = L.total;
    r.bytes = bytes;
    L.total += bytes;
}

void make_layout(efm_handle* h) {
    const HostGraph& G = h->G;
    Layout L;
    add_region(L, L.col_ptr, sizeof(int) * (G.A + 1));
    add_region(L, L.col, sizeof(int2) * (G.col.size() + 1));
    add_region(L, L.colsig, sizeof(u64) * 2 * (G.A + 1));
    add_region(L, L.node, sizeof(int4) * (G.M + 1));
    add_region(L, L.in_e, sizeof(int2) * (G.in.size() + 1));
    add_region(L, L.out_e, sizeof(int2) * (G.out.size() + 1));
    add_region(L, L.in_alt, 32 * (G.in.size() + 1));
    add_region(L, L.out_alt, 32 * (G.out.size() + 1));
    add_region(L, L.twin, sizeof(int) * (G.A + 1));
    add_region(L, L.dep_off, sizeof(i64) * (G.M + 1));
    add_region(L, L.dep_bits, sizeof(u32) * G.dep_bits.size());
    add_region(L, L.arc_rxn, sizeof(int) * (G.A + 1));
    add_region(L, L.arc_dir, sizeof(int) * (G.A + 1));
    add_region(L, L.arc_mix, sizeof(u64) * (G.A + 1));
    add_region(L, L.amask, sizeof(u32) * ((G.A + 31) / 32 + 1));
    add_region(L, L.cand_end, sizeof(u64) * (size_t)(h->sample_count + 1));
    add_region(L, L.ctl, sizeof(Ctl));
    add_region(L, L.lvl, sizeof(LevelStats) * (size_t)(h->max_levels + 2));
    add_region(L, L.buf[0], (size_t)h->frontier_bytes + 256);
    add_region(L, L.buf[1], (size_t)h->frontier_bytes + 256);
    add_region(L, L.off[0], (size_t)(h->max_frontier + 1) * 8);
    add_region(L, L.off[1], (size_t)(h->max_frontier + 1) * 8);
    add_region(L, L.plist, (size_t)(h->max_frontier + 1) * 8);
    add_region(L, L.pprim, (size_t)(h->max_frontier + 1) * 4);
    add_region(L, L.keys, (size_t)h->max_keys * 8);
    add_region(L, L.tags, (size_t)h->max_keys * 8);
    add_region(L, L.ckeys, (size_t)h->max_ckeys * 8);
    add_region(L, L.tasks, (size_t)h->max_tasks * 64);
    add_region(L, L.surv, (size_t)h->max_surv * 16);
    add_region(L, L.surv_dst, (size_t)h->max_surv * 8);
    const size_t C = (size_t)h->max_cand;
    add_region(L, L.cand, C * h->cand_stride);
    add_region(L, L.table, h->table_size * 4);
    add_region(L, L.isrep, C + 1);
    add_region(L, L.poison, C + 1);
    add_region(L, L.uniq, C * 4);
    add_region(L, L.c_steps, (C + 1) * 4);
    add_region(L, L.u_steps, C * 4);
    add_region(L, L.r_steps, C * 4);
    const size_t bins = (size_t)h->G.A + 2;   // per-arc and per-(arc, size) tables of the minimality filter
    const size_t gbins = (size_t)h->G.A * ((size_t)h->D + 1) + 2;
    add_region(L, L.freq, bins * 4);
    add_region(L, L.gcount, gbins * 4);
    add_region(L, L.gstart, gbins * 4);
    add_region(L, L.gfill, gbins * 4);
    add_region(L, L.vcount, gbins * 4);
    add_region(L, L.vstart, gbins * 4);
    add_region(L, L.vfill, gbins * 4);
    add_region(L, L.tstart, bins * 4);
    add_region(L, L.g_row, C * 4);
    add_region(L, L.g_sig, C * 16);
    add_region(L, L.g_sig64, C * 8 + 16);
    add_region(L, L.r_sig64, C * 8 + 16);
    add_region(L, L.g_size, C * 2);
    add_region(L, L.keep, C);
    add_region(L, L.u_nnz, C * 4);
    add_region(L, L.u_rxn, C * h->D * 4);
    add_region(L, L.u_val, C * h->D * 8);
    add_region(L, L.u_key, C * 16);
    add_region(L, L.sort_idx, pow2_at_least(C) * 4);
    add_region(L, L.r_nnz, C * 4);
    add_region(L, L.r_rxn, C * h->D * 4);
    add_region(L, L.r_val, C * h->D * 8);
    add_region(L, L.csr_ptr, (C + 1 + C / 1024 + 2) * 8);   // row pointer + totals of its 1024-row scan blocks
    add_region(L, L.dense, h->dense_bytes);
    L.total = (L.total + 255) & ~(size_t)255;
    h->lay = L;
}

int fail_cuda(efm_handle* h, cudaError_t e, const char* what) {
    char buf[256];
    snprintf(buf, sizeof buf, "%s: %s", what, cudaGetErrorString(e));
    h->last_error = buf;
    cudaGetLastError();
    return EFM_E_CUDA;
}
#define CK(call)                                                       \
    do {                                                               \
        cudaError_t e__ = (call);                                      \
        if (e__ != cudaSuccess) return fail_cuda(h, e__, #call);       \
    } while (0)

DevGraph dev_graph(const efm_handle* h, unsigned char* ws) {
    const Layout& L = h->lay;
    DevGraph g;
    g.M = h->G.M; g.A = h->G.A; g.W32 = (h->G.A + 31) / 32; g.M32 = (h->G.M + 31) / 32;
    g.col_ptr = (const int*)(ws + L.col_ptr.off);   g.col = (const int2*)(ws + L.col.off);
    g.node = (const int4*)(ws + L.node.off);        g.colsig = (const u64*)(ws + L.colsig.off);
    g.in_e = (const int2*)(ws + L.in_e.off);        g.out_e = (const int2*)(ws + L.out_e.off);
    g.in_alt = (const uint4*)(ws + L.in_alt.off);   g.out_alt = (const uint4*)(ws + L.out_alt.off);
    g.twin = (const int*)(ws + L.twin.off);
    g.dep_off = (const i64*)(ws + L.dep_off.off);   g.dep_bits = (const u32*)(ws + L.dep_bits.off);
    g.arc_rxn = (const int*)(ws + L.arc_rxn.off);   g.arc_dir = (const int*)(ws + L.arc_dir.off);
    g.arc_mix = (const u64*)(ws + L.arc_mix.off);
    g.max_coef = 0;
    for (const ColRef& c : h->G.col) g.max_coef = std::max(g.max_coef, c.s < 0 ? -c.s : c.s);
    return g;
}

// 32-byte records of the OR-alternatives (DevGraph::in_alt / out_alt): 8 words per entry of `list`.
std::vector<uint32_t> alt_records(const HostGraph& G, const std::vector<ArcRef>& list) {
    std::vector<uint32_t> out(list.size() * 8, 0u);
    for (size_t q = 0; q < list.size(); ++q) {
        const int a = list[q].arc, c = list[q].c;
        const int n = G.col_ptr[a + 1] - G.col_ptr[a];
        bool generic = n > 6 || c > 0xffff;
        uint32_t* w = &out[q * 8];
        for (int t = 0; t < n && t < 6; ++t) {
            const ColRef& e = G.col[G.col_ptr[a] + t];
            if (e.s > 32767 || e.s < -32767) generic = true;
            w[2 + t] = (uint32_t)e.met | ((uint32_t)(uint16_t)(int16_t)e.s << 16);
        }
        w[0] = (uint32_t)a | ((uint32_t)(c & 0xffff) << 16);
        w[1] = (uint32_t)(G.twin[a] < 0 ? 0xffff : G.twin[a]) | ((uint32_t)(n > 6 ? 0 : n) << 16) | ((generic ? 1u : 0u) << 24);
    }
    return out;
}

// The API calls run on the handle's device and leave the caller's current device as they found it.
struct DeviceGuard {
    int prev = -1; bool ok = true;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; cudaGetLastError(); }
        if (prev != dev && cudaSetDevice(dev) != cudaSuccess) { ok = false; }
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};
#define ON_DEVICE(h) DeviceGuard dg__((h)->device); if (!dg__.ok) return fail_cuda((h), cudaGetLastError(), "cudaSetDevice")

// Events for the optional per-phase timers.
struct Timer {
    efm_handle* h; cudaStream_t s; bool on; size_t used = 0;
    struct Span { size_t a, b; int phase; };
    std::vector<Span> spans;
    cudaEvent_t get() {
        if (used == h->events.size()) { cudaEvent_t e; cudaEventCreate(&e); h->events.push_back(e); }
        return h->events[used++];
    }
    size_t mark() { if (!on) return 0; cudaEvent_t e = get(); cudaEventRecord(e, s); return used - 1; }
    void span(size_t a, size_t b, int phase) { if (on) spans.push_back(Span{a, b, phase}); }
};
enum { PH_ORDER = 0, PH_COUNT, PH_BEAM, PH_WRITE, PH_HASH, PH_FILTER, PH_OUTPUT, PH_N };

}  // namespace

extern "C" {

const char* efm_strerror(int code) {
    switch (code) {
        case EFM_OK: return "ok";
        case EFM_E_INVAL: return "invalid argument";
        case EFM_E_NOMEM: return "workspace too small";
        case EFM_E_CAPACITY: return "frontier / candidate / key capacity exceeded (results undefined)";
        case EFM_E_CUDA: return "CUDA error (see efm_last_error)";
        case EFM_E_STATE: return "no result available";
        default: return "unknown error";
    }
}
const char* efm_last_error(const efm_handle* h) { return h ? h->last_error.c_str() : ""; }

int efm_create(const int32_t* S, int32_t m, int32_t n, int64_t row_stride, const uint8_t* reversible,
               const uint8_t* internal, const efm_params* p, efm_handle** out) {
    if (!out) return EFM_E_INVAL;
    *out = nullptr;
    efm_params P;
    memset(&P, 0, sizeof P);
    if (p) P = *p;
    if (P.max_support < 0 || P.max_loop < 0 || P.dep_depth < 0 || P.max_visited < 0 || P.frontier_cap < 0 ||
        P.max_frontier < 0 || P.max_candidates < 0 || P.max_child_keys < 0 || P.device < 0 || P.max_frontier_bytes < 0 ||
        P.max_child_tasks < 0 || P.sample_count < 0)
        return EFM_E_INVAL;
    efm_handle* h = new (std::nothrow) efm_handle();
    if (!h) return EFM_E_NOMEM;
    memset(&h->stats, 0, sizeof h->stats);
    const auto c0 = std::chrono::steady_clock::now();
    h->L = P.dep_depth ? P.dep_depth : 4;
    if (!S || !reversible || !internal || m <= 0 || n <= 0 || row_stride < n) { delete h; return EFM_E_INVAL; }
    std::vector<uint8_t> skip;
    if (P.flags & EFM_F_COMPRESS) {   // blocked reactions get no arcs
        skip.assign((size_t)n, 0);
        h->n_blocked = blocked_reactions(S, m, n, row_stride, reversible, internal, skip.data());
    }
    int rc = build_graph(h->G, S, m, n, row_stride, reversible, internal, h->L, skip.empty() ? nullptr : skip.data());
    if (rc != EFM_OK) { delete h; return rc; }
    h->ms_build = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - c0).count();   // wall time
    const HostGraph& G = h->G;
    h->D = P.max_support ? P.max_support : G.A;
    if (h->D > G.A) h->D = std::max(G.A, 1);
    h->V = P.max_visited ? P.max_visited : 2 * h->D;
    h->max_loop = P.max_loop ? P.max_loop : 8;
    if (h->D > 4096 || h->max_loop > 65535) { delete h; return EFM_E_INVAL; }
    if ((P.flags & EFM_F_EXACT_ELEMENTARITY) && h->D > 128) { delete h; return EFM_E_INVAL; }   // the basis of the rank test lives in shared memory
    h->cap = P.sample_count ? 0 : P.frontier_cap;   // a sampled candidate has one descendant at most: nothing to cut
    h->sample_count = P.sample_count; h->sample_seed = P.sample_seed;
    h->device = P.device;
    h->flags = P.flags;
    const int Veff = std::min(h->V, std::max(G.M, 1));   // a pathway cannot visit more nodes than exist
    int max_col = 0;
    for (int a = 0; a < G.A; ++a) max_col = std::max(max_col, G.col_ptr[a + 1] - G.col_ptr[a]);
    const int64_t Ueff = std::min<int64_t>(G.M, (int64_t)h->D * max_col);   // unbalanced metabolites a pathway can have
    h->max_entry = entry_bytes((u32)h->D, (u32)Veff, (u32)Ueff);
    h->cand_stride = entry_bytes((u32)h->D, 0, 0);
    h->max_frontier = P.max_frontier ? P.max_frontier : (h->cap ? std::max<int64_t>(h->cap, 4096) : (int64_t)1 << 20);
    if (h->sample_count > h->max_frontier) { if (P.max_frontier) { delete h; return EFM_E_INVAL; } h->max_frontier = h->sample_count; }
    if (h->max_frontier >= ((int64_t)1 << (64 - kAllocShift))) { delete h; return EFM_E_INVAL; }
    h->frontier_bytes = P.max_frontier_bytes ? ((P.max_frontier_bytes + 15) & ~(int64_t)15) : h->max_frontier * (int64_t)h->max_entry;
    if (h->frontier_bytes < (int64_t)h->max_entry) h->frontier_bytes = h->max_entry;
    if ((uint64_t)h->frontier_bytes >> 4 > kAllocUnitMask) {
        if (P.max_frontier_bytes) { delete h; return EFM_E_INVAL; }
        h->frontier_bytes = (int64_t)(kAllocUnitMask << 4);   // the default never needs more than the allocator can address
    }
    h->max_cand = P.max_candidates ? P.max_candidates : (int64_t)1 << 20;
    if (h->max_cand > 0xFFFFFFF0LL) { delete h; return EFM_E_INVAL; }
    // child slots of a level (8-byte key + 8-byte tag each).  The evaluation strands at most one chunk per resident warp
    // (kSlackSMs bounds the SM count of the device the handle will run on).
    int kSlackSMs = 256;
    {
        int smc = 0;
        if (cudaDeviceGetAttribute(&smc, cudaDevAttrMultiProcessorCount, P.device) == cudaSuccess && smc > 0) kSlackSMs = smc;
        else cudaGetLastError();
    }
    // default: a capped level has at most cap * fan-out children; a sampled candidate has one child at most; an unbounded
    // run (cap == 0) gets 65536 slots and reports EFM_E_CAPACITY beyond (the caller sizes max_child_keys for its network)
    const int64_t dflt_keys = std::max<int64_t>(std::max<int64_t>(h->cap * (int64_t)G.max_fanout, h->sample_count), 65536);
    h->max_keys = (P.max_child_keys ? P.max_child_keys : dflt_keys) + (int64_t)expand_key_slack(kSlackSMs);
    if (h->max_keys > 0xFFFFFFF0LL) {   // slots are addressed with 32 bits; the default is clamped, an explicit request is refused
        if (P.max_child_keys) { delete h; return EFM_E_INVAL; }
        h->max_keys = 0xFFFFFFF0LL;
    }
    // 64-byte tasks of the children of the general routine: one per revisit parent plus the alternatives of a first visit
    // that are arcs of the support; every child when EFM_F_NO_FASTPATH sends all of them there
    h->max_tasks = P.max_child_tasks ? P.max_child_tasks
                   : ((P.flags & EFM_F_NO_FASTPATH) ? h->max_keys : std::min<int64_t>(h->max_keys, 4 * h->max_frontier + 65536));
    h->max_tasks += (int64_t)expand_task_slack(kSlackSMs);
    // keys sharing the selected 22-bit prefix (8 bits of n_unb + 14 bits of the state hash): 1 / 16384 of a class on average
    h->max_ckeys = std::max<int64_t>(h->max_keys / 64, std::min<int64_t>(h->max_keys, (int64_t)1 << 20));
    h->max_surv = h->max_frontier + h->max_cand + 1024;
    // a pathway gains a visited node or a revisit count with every level
    h->max_levels = std::min<int64_t>((int64_t)std::min(h->V, std::max(G.M, 1)) * ((int64_t)h->max_loop + 1) + 2, (int64_t)1 << 20);
    h->table_size = pow2_at_least((size_t)h->max_cand * 2);
    h->dense_bytes = std::max<size_t>((size_t)64 << 20, (size_t)n * 8 * 64);
    make_layout(h);
    *out = h;
    return EFM_OK;
}

int efm_blocked_reactions(const int32_t* S, int32_t m, int32_t n, int64_t row_stride, const uint8_t* reversible,
                          const uint8_t* internal, uint8_t* blocked, int32_t* n_blocked) {
    if (!S || !reversible || !internal || !blocked || m <= 0 || n <= 0 || row_stride < n) return EFM_E_INVAL;
    const int32_t nb = blocked_reactions(S, m, n, row_stride, reversible, internal, blocked);
    if (n_blocked) *n_blocked = nb;
    return EFM_OK;
}

int efm_graph_info(const efm_handle* h, int32_t* n_internal, int32_t* n_arcs, int32_t* bitset_words, int64_t* nnz,
                   int64_t* dep_entries) {
    if (!h) return EFM_E_INVAL;
    if (n_internal) *n_internal = h->G.M;
    if (n_arcs) *n_arcs = h->G.A;
    if (bitset_words) *bitset_words = (h->G.A + 63) / 64;
    if (nnz) *nnz = (int64_t)h->G.col.size();
    if (dep_entries) *dep_entries = h->G.dep_off[h->G.M];
    return EFM_OK;
}

int efm_graph_export(const efm_handle* h, int32_t* arc_rxn, int32_t* arc_dir, int32_t* twin, int32_t* in_ptr,
                     int32_t* in_arc, int64_t* in_c, int32_t* out_ptr, int32_t* out_arc, int64_t* out_c,
                     int32_t* col_ptr, int32_t* col_met, int64_t* col_s, int64_t* dep_off, uint8_t* dep) {
    if (!h) return EFM_E_INVAL;
    const HostGraph& G = h->G;
    for (int a = 0; a < G.A; ++a) {
        if (arc_rxn) arc_rxn[a] = G.arc_rxn[a];
        if (arc_dir) arc_dir[a] = G.arc_dir[a];
        if (twin) twin[a] = G.twin[a];
    }
    for (int i = 0; i <= G.M; ++i) {
        if (in_ptr) in_ptr[i] = G.in_ptr[i];
        if (out_ptr) out_ptr[i] = G.out_ptr[i];
        if (dep_off) dep_off[i] = G.dep_off[i];
    }
    for (size_t q = 0; q < G.in.size(); ++q) { if (in_arc) in_arc[q] = G.in[q].arc; if (in_c) in_c[q] = G.in[q].c; }
    for (size_t q = 0; q < G.out.size(); ++q) { if (out_arc) out_arc[q] = G.out[q].arc; if (out_c) out_c[q] = G.out[q].c; }
    for (int a = 0; a <= G.A; ++a) if (col_ptr) col_ptr[a] = G.col_ptr[a];
    for (size_t q = 0; q < G.col.size(); ++q) { if (col_met) col_met[q] = G.col[q].met; if (col_s) col_s[q] = G.col[q].s; }
    if (dep)
        for (int64_t b = 0; b < G.dep_off[G.M]; ++b) dep[b] = (uint8_t)((G.dep_bits[b >> 5] >> (b & 31)) & 1u);
    return EFM_OK;
}

int efm_workspace_bytes(const efm_handle* h, size_t* bytes) {
    if (!h || !bytes) return EFM_E_INVAL;
    *bytes = h->lay.total;
    return EFM_OK;
}

int efm_enumerate(efm_handle* h, const int32_t* seed_ptr, const int32_t* seed_arc_code, int32_t n_sets,
                  void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
    if (!h || !d_workspace || n_sets < 0 || (n_sets > 0 && (!seed_ptr || !seed_arc_code))) return EFM_E_INVAL;
    if (((uintptr_t)d_workspace & 255) != 0) return EFM_E_INVAL;
    if (workspace_bytes < h->lay.total) return EFM_E_NOMEM;
    h->have_result = false;
    h->last_error.clear();
    const HostGraph& G = h->G;
    const Layout& L = h->lay;
    cudaStream_t s = (cudaStream_t)cuda_stream;

    // ---- O2 roots (INIT kernel of the paper): host packs the seed sets, the device classifies them
    std::vector<std::vector<int>> roots;
    if (n_sets == 0) {
        // default: one root per boundary arc = non-empty, single-signed internal column (Def 8)
        for (int a = 0; a < G.A; ++a) {
            int pos = 0, neg = 0;
            for (int q = G.col_ptr[a]; q < G.col_ptr[a + 1]; ++q) (G.col[q].s > 0 ? pos : neg)++;
            if ((pos > 0) != (neg > 0)) roots.push_back(std::vector<int>(1, a));
        }
    } else {
        std::vector<char> mark((size_t)G.A, 0);
        for (int t = 0; t < n_sets; ++t) {
            const int cnt = seed_ptr[t + 1] - seed_ptr[t];
            if (cnt <= 0 || cnt > h->D) return EFM_E_INVAL;
            std::vector<int> arcs;
            bool bad = false;
            for (int k = 0; k < cnt && !bad; ++k) {
                const int code = seed_arc_code[seed_ptr[t] + k];
                const int a = (code >= 0 && code < 2 * G.n) ? G.code2arc[code] : -1;
                if (a < 0 || mark[a] || (G.twin[a] >= 0 && mark[G.twin[a]])) bad = true;
                else { mark[a] = 1; arcs.push_back(a); }
            }
            for (int a : arcs) mark[a] = 0;
            if (bad) return EFM_E_INVAL;
            std::sort(arcs.begin(), arcs.end());
            roots.push_back(arcs);
        }
    }
    if (h->sample_count > 0 && !roots.empty()) {   // 8(f)-1: candidate c is a copy of seed set c mod (number of sets)
        std::vector<std::vector<int>> cands((size_t)h->sample_count);
        for (size_t c = 0; c < cands.size(); ++c) cands[c] = roots[c % roots.size()];
        roots.swap(cands);
    }
    const u64 n_roots = roots.size();
    if ((int64_t)n_roots > h->max_frontier || (int64_t)n_roots > h->max_keys) {
        h->last_error = "more roots than max_frontier / max_child_keys hold";
        return EFM_E_CAPACITY;
    }
    // seed sets as CSR of arc ids + the offset of every root entry in the staging buffer (16-byte units); the
    // entries themselves are built on the device (k_roots)
    std::vector<int> h_seed_ptr(n_roots + 1, 0), h_seed_arc;
    std::vector<u64> stage_off(n_roots, 0);
    u64 stage_units = 0;
    for (size_t r = 0; r < roots.size(); ++r) {
        int64_t touched = 0;
        for (int a : roots[r]) { h_seed_arc.push_back(a); touched += G.col_ptr[a + 1] - G.col_ptr[a]; }
        h_seed_ptr[r + 1] = (int)h_seed_arc.size();
        stage_off[r] = stage_units;
        stage_units += entry_bytes((u32)roots[r].size(), 0, (u32)std::min<int64_t>(touched, G.M)) >> 4;
    }
    if ((int64_t)(stage_units << 4) > h->frontier_bytes || h_seed_arc.size() * sizeof(int) > (size_t)h->max_keys * 8) {
        h->last_error = "the root entries / seed arcs do not fit max_frontier_bytes / max_child_keys";
        return EFM_E_CAPACITY;
    }

    ON_DEVICE(h);
    if (!h->h_ctl) {
        CK(cudaMallocHost((void**)&h->h_ctl, sizeof(Ctl)));
        int smc = 0;
        CK(cudaDeviceGetAttribute(&smc, cudaDevAttrMultiProcessorCount, h->device));
        if (smc > 0) h->sm_count = smc;
    }
    memset(h->h_ctl, 0, sizeof(Ctl));   // a run without roots reads no control block: its counters are zero, not stale
    h->stream = (cudaStream_t)cuda_stream;
    unsigned char* ws = (unsigned char*)d_workspace;
    h->ws = ws;
    Timer tm{h, s, (h->flags & EFM_F_TIMING) != 0};
    cudaEvent_t ev_start = tm.get(), ev_end = tm.get();
    CK(cudaEventRecord(ev_start, s));

    // ---- upload the graph (~0.5 MB) and the roots; clear the control block
    int64_t h2d = 0;
    auto up = [&](unsigned char* dst, const void* src, size_t bytes) -> cudaError_t {
        if (bytes == 0) return cudaSuccess;
        h2d += (int64_t)bytes;
        return cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, s);
    };
    std::vector<u64> arc_mix, colsig;
    std::vector<uint32_t> alt_in, alt_out;
    std::vector<int> node, colp;
    if (h->graph_ws != ws) {   // the network is an input: it stays resident in the workspace across calls
        h->graph_ws = nullptr;
        // columns with the position of the arc in I[met] / O[met] next to the metabolite: {met | pos << 16, s}
        colp.resize(2 * G.col.size());
        colsig.assign(2 * (size_t)G.A, 0ULL);
        {
            std::vector<int> fin(G.in_ptr.begin(), G.in_ptr.end() - 1), fout(G.out_ptr.begin(), G.out_ptr.end() - 1);
            for (int a = 0; a < G.A; ++a)
                for (int q = G.col_ptr[a]; q < G.col_ptr[a + 1]; ++q) {
                    const ColRef& e = G.col[q];
                    const int pos = e.s > 0 ? fin[e.met]++ - G.in_ptr[e.met] : fout[e.met]++ - G.out_ptr[e.met];
                    colp[2 * (size_t)q] = (int)((uint32_t)e.met | ((uint32_t)pos << 16));
                    colp[2 * (size_t)q + 1] = e.s;
                    colsig[2 * (size_t)a + (e.s > 0 ? 0 : 1)] |= 1ULL << (e.met & 63);
                }
        }
        node.resize(4 * (size_t)G.M);
        for (int i = 0; i < G.M; ++i) {
            node[4 * (size_t)i] = G.in_ptr[i]; node[4 * (size_t)i + 1] = G.in_ptr[i + 1] - G.in_ptr[i];
            node[4 * (size_t)i + 2] = G.out_ptr[i]; node[4 * (size_t)i + 3] = G.out_ptr[i + 1] - G.out_ptr[i];
        }
        CK(up(ws + L.col_ptr.off, G.col_ptr.data(), sizeof(int) * G.col_ptr.size()));
        CK(up(ws + L.col.off, colp.data(), sizeof(int) * colp.size()));
        CK(up(ws + L.colsig.off, colsig.data(), sizeof(u64) * colsig.size()));
        CK(up(ws + L.node.off, node.data(), sizeof(int) * node.size()));
        CK(up(ws + L.in_e.off, G.in.data(), sizeof(ArcRef) * G.in.size()));
        CK(up(ws + L.out_e.off, G.out.data(), sizeof(ArcRef) * G.out.size()));
        alt_in = alt_records(G, G.in); alt_out = alt_records(G, G.out);
        CK(up(ws + L.in_alt.off, alt_in.data(), sizeof(uint32_t) * alt_in.size()));
        CK(up(ws + L.out_alt.off, alt_out.data(), sizeof(uint32_t) * alt_out.size()));
        CK(up(ws + L.twin.off, G.twin.data(), sizeof(int) * G.twin.size()));
        CK(up(ws + L.dep_off.off, G.dep_off.data(), sizeof(i64) * G.dep_off.size()));
        CK(up(ws + L.dep_bits.off, G.dep_bits.data(), sizeof(u32) * G.dep_bits.size()));
        CK(up(ws + L.arc_rxn.off, G.arc_rxn.data(), sizeof(int) * G.arc_rxn.size()));
        CK(up(ws + L.arc_dir.off, G.arc_dir.data(), sizeof(int) * G.arc_dir.size()));
        arc_mix.resize((size_t)G.A);
        for (int a = 0; a < G.A; ++a) arc_mix[a] = mix64(0x0100000000000000ULL | (u64)a);   // multiplier of arc a in the state hash
        CK(up(ws + L.arc_mix.off, arc_mix.data(), sizeof(u64) * arc_mix.size()));
        h->graph_ws = ws;
    }
    if (!h->amask.empty()) CK(up(ws + L.amask.off, h->amask.data(), sizeof(uint32_t) * h->amask.size()));   // a few hundred bytes
    // the seed sets travel in regions that are unused until the first level is ordered / expanded
    CK(up(ws + L.plist.off, h_seed_ptr.data(), sizeof(int) * h_seed_ptr.size()));
    CK(up(ws + L.tags.off, h_seed_arc.data(), sizeof(int) * h_seed_arc.size()));
    CK(up(ws + L.off[1].off, stage_off.data(), sizeof(u64) * stage_off.size()));
    CK(cudaMemsetAsync(ws + L.ctl.off, 0, sizeof(Ctl), s));
    // every record the host may walk: k_materialise skips record level + 1 at the last level, which must then read as empty
    CK(cudaMemsetAsync(ws + L.lvl.off, 0, sizeof(LevelStats) * (size_t)(h->max_levels + 2), s));
    if (h->sample_count > 0) CK(cudaMemsetAsync(ws + L.cand_end.off, 0, sizeof(u64) * (size_t)(h->sample_count + 1), s));
    CK(cudaStreamSynchronize(s));   // the host staging vectors above go out of scope later; keep it simple
    int host_syncs = 1;

    Ctl* d_ctl = (Ctl*)(ws + L.ctl.off);
    Ctl* hc = h->h_ctl;
    const size_t ctl_read = offsetof(Ctl, hist);
    int launches = 0;
    ExpandArgs ea;
    memset(&ea, 0, sizeof ea);
    ea.g = dev_graph(h, ws);
    ea.cand = ws + L.cand.off;
    ea.keys = (u64*)(ws + L.keys.off);
    ea.tags = (u64*)(ws + L.tags.off);
    ea.tasks = (uint4*)(ws + L.tasks.off);
    ea.plist = (u64*)(ws + L.plist.off);
    ea.pprim = (u32*)(ws + L.pprim.off);
    ea.lvl = (LevelStats*)(ws + L.lvl.off);
    ea.ctl = d_ctl;
    ea.surv = (ulonglong2*)(ws + L.surv.off); ea.surv_dst = (u64*)(ws + L.surv_dst.off);
    ea.max_entry = h->max_entry; ea.cand_stride = h->cand_stride;
    ea.frontier_units = (u64)h->frontier_bytes >> 4;
    ea.max_frontier = (u64)h->max_frontier; ea.max_cand = (u64)h->max_cand; ea.max_keys = (u64)h->max_keys;
    ea.max_tasks = (u64)h->max_tasks; ea.max_surv = (u64)h->max_surv; ea.max_levels = (u64)h->max_levels;
    ea.cap = (u64)h->cap;
    ea.D = h->D; ea.V = h->V; ea.max_loop = h->max_loop;
    ea.no_fast = (h->flags & EFM_F_NO_FASTPATH) ? 1 : 0;
    ea.sample = h->sample_count > 0 ? 1u : 0u; ea.sample_seed = h->sample_seed;
    ea.amask = h->amask.empty() ? nullptr : (const u32*)(ws + L.amask.off);
    ea.cand_end = h->sample_count > 0 ? (u64*)(ws + L.cand_end.off) : nullptr;
    expand_smem_layout(ea);
    ea.force_inplace = (h->flags & EFM_F_NO_STAGING) ? 1 : 0;

    auto read_ctl = [&]() -> cudaError_t {
        cudaError_t e = cudaMemcpyAsync(hc, d_ctl, ctl_read, cudaMemcpyDeviceToHost, s);
        if (e != cudaSuccess) return e;
        ++host_syncs;
        return cudaStreamSynchronize(s);
    };

    efm_stats& st = h->stats;
    memset(&st, 0, sizeof st);
    st.ms_build = h->ms_build;
    st.n_roots = (int64_t)n_roots;
    h->lvl_active.clear(); h->lvl_done.clear(); h->lvl_expanded.clear(); h->lvl_children.clear();
    int64_t truncated = 0, done_total = 0, materialised = 0;

    if (n_roots > 0) {
        // ---- level 0: classify the roots, beam-select, keep the survivors
        RootArgs ra;
        memset(&ra, 0, sizeof ra);
        ra.g = ea.g; ra.ctl = d_ctl; ra.lvl = ea.lvl; ra.n_roots = n_roots;
        ra.seed_ptr = (const int*)(ws + L.plist.off); ra.seed_arc = (const int*)(ws + L.tags.off);
        ra.stage_off = (const u64*)(ws + L.off[1].off); ra.stage = ws + L.buf[1].off;
        ra.nxt = ws + L.buf[0].off; ra.nxt_off = (u64*)(ws + L.off[0].off);
        ra.cand = ea.cand; ra.cand_stride = h->cand_stride; ra.keys = ea.keys;
        ra.cand_end = ea.cand_end;
        ra.max_frontier = ea.max_frontier; ra.frontier_units = ea.frontier_units; ra.max_cand = ea.max_cand; ra.cap = ea.cap;
        size_t t0 = tm.mark();
        CK(launch_roots(false, ra, s)); ++launches;
        size_t t1 = tm.mark();
        CK(launch_select(ea.keys, (u64*)(ws + L.ckeys.off), (u64)h->max_ckeys, d_ctl, 1, (u64)h->cap, ea.max_keys, h->sm_count, s, &launches));
        size_t t2 = tm.mark();
        CK(launch_roots(true, ra, s)); ++launches;
        size_t t3 = tm.mark();
        tm.span(t0, t1, PH_COUNT); tm.span(t1, t2, PH_BEAM); tm.span(t2, t3, PH_WRITE);

        // ---- level loop (Alg 3 while(true), as level-synchronous frontier expansion).  The kernels find
        // their work through the control block, so a whole batch of levels is enqueued before the host looks again; the
        // levels behind the end of the traversal see an empty frontier and return at once.
        std::vector<LevelStats> recs;
        const int kBatch = 8;
        u64 level = 0;
        bool more = true;
        while (more) {
            const u64 l0 = level;
            for (int bi = 0; bi < kBatch && level < (u64)h->max_levels; ++bi, ++level) {
                const int par = (int)(level & 1);
                ea.level = (u32)level; ea.par = (u32)par;
                ea.cur = ws + L.buf[par].off; ea.nxt = ws + L.buf[par ^ 1].off;
                ea.cur_off = (const u64*)(ws + L.off[par].off); ea.nxt_off = (u64*)(ws + L.off[par ^ 1].off);
                // order the parents -> evaluate every child (keys + tags) -> beam threshold -> survivors -> materialise them
                size_t a0 = tm.mark();
                CK(launch_order(ea, h->sm_count, s)); ++launches;
                size_t a1 = tm.mark();
                CK(launch_expand(ea, h->sm_count, s)); ++launches;
                size_t a2 = tm.mark();
                CK(launch_select(ea.keys, (u64*)(ws + L.ckeys.off), (u64)h->max_ckeys, d_ctl, par, (u64)h->cap, ea.max_keys, h->sm_count, s, &launches));
                size_t a3 = tm.mark();
                CK(launch_compact(ea, h->sm_count, s)); ++launches;
                CK(launch_materialise(ea, h->sm_count, s)); ++launches;
                size_t a4 = tm.mark();
                tm.span(a0, a1, PH_ORDER); tm.span(a1, a2, PH_COUNT); tm.span(a2, a3, PH_BEAM); tm.span(a3, a4, PH_WRITE);
                st.n_expand_count++;
                if (h->cap > 0) st.two_pass_levels++; else st.direct_levels++;
            }
            // records 0 .. level (record 0: the roots; record L + 1: the children of level L)
            recs.resize((size_t)level + 1);
            CK(cudaMemcpyAsync(recs.data() + l0, ws + L.lvl.off + sizeof(LevelStats) * l0, sizeof(LevelStats) * (size_t)(level + 1 - l0),
                               cudaMemcpyDeviceToHost, s));
            CK(read_ctl());
            if (hc->error) {
                char buf[160];
                snprintf(buf, sizeof buf, "capacity exceeded near level %llu:%s%s%s%s", (unsigned long long)level,
                         (hc->error & ERR_FRONTIER) ? " frontier (max_frontier / max_frontier_bytes)" : "",
                         (hc->error & ERR_CAND) ? " candidates (max_candidates)" : "",
                         (hc->error & ERR_KEYS) ? " child keys / tasks (max_child_keys / max_child_tasks)" : "",
                         (hc->error & ERR_LEVELS) ? " levels" : "");
                h->last_error = buf;
                return EFM_E_CAPACITY;
            }
            more = (hc->lv[level & 1].alloc >> kAllocShift) != 0;
            if (more && level >= (u64)h->max_levels) { h->last_error = "active entries left after max_levels levels"; return EFM_E_CAPACITY; }
        }
        // per-level figures: record r holds the children of level r - 1 = the entries of level r
        for (size_t r = 0; r < recs.size(); ++r) {
            const int64_t active = (int64_t)recs[r].active_children, done = (int64_t)recs[r].done_children;
            if (active + done == 0) break;
            const bool have_next = r + 1 < recs.size();
            h->lvl_active.push_back(active);
            h->lvl_done.push_back(done);
            h->lvl_expanded.push_back(have_next ? (int64_t)recs[r + 1].parents : 0);
            h->lvl_children.push_back(have_next ? (int64_t)(recs[r + 1].active_children + recs[r + 1].done_children) : 0);
            done_total += done;
            truncated += active - (have_next ? (int64_t)recs[r + 1].parents : 0);
            materialised += (int64_t)recs[r].surv;
        }
    }

    // ---- O8: support dedup + poison (a-6), minimality filter (a-7), canonical output (a-8)
    const u64 n_cand = n_roots ? hc->n_cand : 0;
    PostArgs pa;
    memset(&pa, 0, sizeof pa);
    pa.g = ea.g; pa.ctl = d_ctl;
    pa.cand = ws + L.cand.off; pa.cand_stride = h->cand_stride; pa.max_cand = (u64)h->max_cand;
    pa.table = (u32*)(ws + L.table.off); pa.table_size = h->table_size;
    pa.isrep = ws + L.isrep.off; pa.poison = ws + L.poison.off; pa.uniq = (u32*)(ws + L.uniq.off);
    pa.c_steps = (u32*)(ws + L.c_steps.off); pa.u_steps = (int*)(ws + L.u_steps.off); pa.r_steps = (int*)(ws + L.r_steps.off);
    pa.freq = (u32*)(ws + L.freq.off); pa.gcount = (u32*)(ws + L.gcount.off);
    pa.gstart = (u32*)(ws + L.gstart.off); pa.gfill = (u32*)(ws + L.gfill.off);
    // the join's row lists and row-order signatures live in regions the output stage fills only afterwards
    pa.v_row = (u32*)(ws + L.u_rxn.off); pa.r_sig = (uint4*)(ws + L.u_key.off);
    pa.vcount = (u32*)(ws + L.vcount.off); pa.vstart = (u32*)(ws + L.vstart.off); pa.vfill = (u32*)(ws + L.vfill.off); pa.tstart = (u32*)(ws + L.tstart.off);
    pa.g_row = (u32*)(ws + L.g_row.off); pa.g_sig = (uint4*)(ws + L.g_sig.off);
    pa.g_sig64 = (uint2*)(ws + L.g_sig64.off); pa.r_sig64 = (uint2*)(ws + L.r_sig64.off);
    pa.keep = ws + L.keep.off;
    pa.D = h->D; pa.n_rxn = G.n; pa.n_sizes = h->D + 1;
    pa.u_nnz = (int*)(ws + L.u_nnz.off); pa.u_rxn = (int*)(ws + L.u_rxn.off); pa.u_val = (i64*)(ws + L.u_val.off);
    pa.u_key = (ulonglong2*)(ws + L.u_key.off);
    pa.sort_idx = (u32*)(ws + L.sort_idx.off);
    pa.r_nnz = (int*)(ws + L.r_nnz.off); pa.r_rxn = (int*)(ws + L.r_rxn.off); pa.r_val = (i64*)(ws + L.r_val.off);
    u64 n_uniq_ok = 0, n_keep = 0;
    if (n_cand > 0) {
        size_t t0 = tm.mark();
        CK(launch_dedup(pa, n_cand, s, &launches));
        size_t t1 = tm.mark();
        tm.span(t0, t1, PH_HASH);
        CK(read_ctl());
        n_uniq_ok = hc->n_uniq_ok;
        st.unique_supports = (int64_t)hc->n_unique;
        st.poisoned = (int64_t)hc->n_poisoned;
        if (n_uniq_ok > 0) {
            size_t t2 = tm.mark();
            if (h->flags & EFM_F_EXACT_ELEMENTARITY) CK(launch_rank_test(pa, n_uniq_ok, h->sm_count, s, &launches));   // 8(f)-3
            else CK(launch_filter(pa, n_uniq_ok, h->sm_count, s, &launches));
            size_t t3 = tm.mark();
            CK(launch_output_rows(pa, n_uniq_ok, s, &launches));
            CK(read_ctl());
            n_keep = hc->n_keep;
            st.filter_pairs = (int64_t)hc->filter_pairs;
            pa.n_pad = pow2_at_least((size_t)std::max<u64>(n_keep, 2));
            CK(launch_output_sort(pa, n_keep, s, &launches));
            // compressed rows for efm_result_copy_csr (the unsorted row arrays are dead by now and hold the packed rows)
            CK(launch_output_csr(pa, n_keep, (i64*)(ws + L.csr_ptr.off), pa.u_rxn, pa.u_val, s, &launches));
            CK(read_ctl());
            size_t t4 = tm.mark();
            tm.span(t2, t3, PH_FILTER); tm.span(t3, t4, PH_OUTPUT);
        }
    }
    CK(cudaEventRecord(ev_end, s));
    CK(cudaStreamSynchronize(s));

    st.levels = (int64_t)h->lvl_active.size();
    st.expanded = (int64_t)hc->st[ST_EXPANDED];
    st.children = (int64_t)hc->st[ST_CHILDREN];
    st.done = done_total;
    st.dead_end = (int64_t)hc->st[ST_DEAD_END];
    st.not_efm_maxloop = (int64_t)hc->st[ST_NOT_EFM];
    st.discarded_nonpos = (int64_t)hc->st[ST_NONPOS];
    st.discarded_overflow = (int64_t)hc->st[ST_OVERFLOW];
    st.discarded_visited = (int64_t)hc->st[ST_VISITED];
    st.truncated_beam = truncated;
    st.output = (int64_t)n_keep;
    st.blocked_reactions = h->n_blocked;
    st.non_elementary = (h->flags & EFM_F_EXACT_ELEMENTARITY) ? (int64_t)n_uniq_ok - (int64_t)n_keep : 0;
    st.algo_bytes = (int64_t)hc->st[ST_ALGO_BYTES];
    st.general_children = (int64_t)hc->st[ST_GENERAL]; st.first_visits = (int64_t)hc->st[ST_FIRST];
    st.materialised = materialised;
    st.h2d_bytes = h2d; st.host_syncs = host_syncs;
    st.peak_frontier = 0;
    for (int64_t a : h->lvl_active) st.peak_frontier = std::max(st.peak_frontier, a);
    st.launches = launches;
    float ms = 0;
    CK(cudaEventElapsedTime(&ms, ev_start, ev_end));
    st.ms_total = ms;
    if (tm.on) {
        double acc[PH_N] = {0};
        for (const Timer::Span& sp : tm.spans) {
            float t = 0;
            CK(cudaEventElapsedTime(&t, h->events[sp.a], h->events[sp.b]));
            acc[sp.phase] += t;
        }
        st.ms_order = acc[PH_ORDER]; st.ms_expand_count = acc[PH_COUNT]; st.ms_beam = acc[PH_BEAM]; st.ms_expand_write = acc[PH_WRITE];
        st.ms_hash = acc[PH_HASH]; st.ms_filter = acc[PH_FILTER]; st.ms_output = acc[PH_OUTPUT];
    }
    h->n_out = (int64_t)n_keep;
    h->csr_nnz = n_keep ? (int64_t)hc->csr_nnz : 0;
    h->have_result = true;
    return EFM_OK;
}

int efm_set_reaction_mask(efm_handle* h, const uint8_t* allowed) {
    if (!h) return EFM_E_INVAL;
    h->amask.clear();
    if (allowed) {
        h->amask.assign((size_t)(h->G.A + 31) / 32 + 1, 0u);
        for (int a = 0; a < h->G.A; ++a)
            if (allowed[h->G.arc_rxn[a]]) h->amask[(size_t)a >> 5] |= 1u << (a & 31);
    }
    return EFM_OK;
}

int efm_result_steps(const efm_handle* hc, int32_t* steps, int64_t capacity_rows) {
    efm_handle* h = const_cast<efm_handle*>(hc);
    if (!h || (!steps && capacity_rows > 0)) return EFM_E_INVAL;
    if (!h->have_result) return EFM_E_STATE;
    if (capacity_rows < h->n_out) return EFM_E_INVAL;
    if (h->n_out == 0) return EFM_OK;
    ON_DEVICE(h);
    CK(cudaMemcpyAsync(steps, h->ws + h->lay.r_steps.off, (size_t)h->n_out * 4, cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    return EFM_OK;
}

int efm_sample_ends(const efm_handle* hc, int64_t* code_steps, int64_t capacity, int64_t* n_candidates) {
    efm_handle* h = const_cast<efm_handle*>(hc);
    if (!h || !n_candidates || capacity < 0 || (capacity > 0 && !code_steps)) return EFM_E_INVAL;
    if (!h->have_result) return EFM_E_STATE;
    const int64_t n = h->sample_count > 0 ? (int64_t)h->stats.n_roots : 0;
    *n_candidates = n;
    const int64_t c = std::min(n, capacity);
    if (c == 0) return EFM_OK;
    ON_DEVICE(h);
    CK(cudaMemcpyAsync(code_steps, h->ws + h->lay.cand_end.off, (size_t)c * 8, cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    return EFM_OK;
}

int efm_workspace_invalidate(efm_handle* h) {
    if (!h) return EFM_E_INVAL;
    h->graph_ws = nullptr;
    h->have_result = false;
    return EFM_OK;
}

int efm_result_count(const efm_handle* h, int64_t* n_pathways) {
    if (!h || !n_pathways) return EFM_E_INVAL;
    if (!h->have_result) return EFM_E_STATE;
    *n_pathways = h->n_out;
    return EFM_OK;
}

int efm_result_device(const efm_handle* h, const int32_t** d_nnz, const int32_t** d_rxn, const int64_t** d_val) {
    if (!h) return EFM_E_INVAL;
    if (!h->have_result) return EFM_E_STATE;
    if (d_nnz) *d_nnz = (const int32_t*)(h->ws + h->lay.r_nnz.off);
    if (d_rxn) *d_rxn = (const int32_t*)(h->ws + h->lay.r_rxn.off);
    if (d_val) *d_val = (const int64_t*)(h->ws + h->lay.r_val.off);
    return EFM_OK;
}

int efm_result_sparse_stride(const efm_handle* h, int32_t* row_capacity) {
    if (!h || !row_capacity) return EFM_E_INVAL;
    *row_capacity = h->D;
    return EFM_OK;
}

int efm_result_densify(const efm_handle* hc, int64_t row0, int64_t n_rows, int64_t* d_out, void* cuda_stream) {
    efm_handle* h = const_cast<efm_handle*>(hc);
    if (!h || !d_out || row0 < 0 || n_rows < 0) return EFM_E_INVAL;
    if (!h->have_result) return EFM_E_STATE;
    if (row0 + n_rows > h->n_out) return EFM_E_INVAL;
    ON_DEVICE(h);
    CK(launch_densify((const int*)(h->ws + h->lay.r_nnz.off), (const int*)(h->ws + h->lay.r_rxn.off),
                      (const i64*)(h->ws + h->lay.r_val.off), h->D, h->G.n, row0, n_rows, (i64*)d_out, (cudaStream_t)cuda_stream));
    return EFM_OK;
}

int efm_result_copy(const efm_handle* hc, int64_t* flux, int64_t capacity_rows) {
    efm_handle* h = const_cast<efm_handle*>(hc);
    if (!h || (!flux && capacity_rows > 0)) return EFM_E_INVAL;
    if (!h->have_result) return EFM_E_STATE;
    if (capacity_rows < h->n_out) return EFM_E_INVAL;
    if (h->n_out == 0) return EFM_OK;
    ON_DEVICE(h);
    const int64_t n = h->G.n;
    const int64_t chunk = std::max<int64_t>(1, (int64_t)(h->lay.dense.bytes / ((size_t)n * 8)));
    i64* d_dense = (i64*)(h->ws + h->lay.dense.off);
    for (int64_t r0 = 0; r0 < h->n_out; r0 += chunk) {
        const int64_t nr = std::min(chunk, h->n_out - r0);
        CK(launch_densify((const int*)(h->ws + h->lay.r_nnz.off), (const int*)(h->ws + h->lay.r_rxn.off),
                          (const i64*)(h->ws + h->lay.r_val.off), h->D, (int)n, r0, nr, d_dense, h->stream));
        CK(cudaMemcpyAsync(flux + r0 * n, d_dense, (size_t)nr * n * 8, cudaMemcpyDeviceToHost, h->stream));
        CK(cudaStreamSynchronize(h->stream));
    }
    return EFM_OK;
}

int efm_result_nnz(const efm_handle* h, int64_t* total_nnz) {
    if (!h || !total_nnz) return EFM_E_INVAL;
    if (!h->have_result) return EFM_E_STATE;
    *total_nnz = h->csr_nnz;
    return EFM_OK;
}

int efm_result_copy_csr(const efm_handle* hc, int64_t* row_ptr, int32_t* rxn, int64_t* val, void* cuda_stream) {
    efm_handle* h = const_cast<efm_handle*>(hc);
    if (!h || !row_ptr) return EFM_E_INVAL;
    if (!h->have_result) return EFM_E_STATE;
    if (h->n_out == 0) { row_ptr[0] = 0; return EFM_OK; }
    if (!rxn || !val) return EFM_E_INVAL;
    ON_DEVICE(h);
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const size_t K = (size_t)h->n_out, Z = (size_t)h->csr_nnz;
    CK(cudaMemcpyAsync(row_ptr, h->ws + h->lay.csr_ptr.off, (K + 1) * 8, cudaMemcpyDeviceToHost, s));
    CK(cudaMemcpyAsync(rxn, h->ws + h->lay.u_rxn.off, Z * 4, cudaMemcpyDeviceToHost, s));
    CK(cudaMemcpyAsync(val, h->ws + h->lay.u_val.off, Z * 8, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    return EFM_OK;
}

int efm_result_copy_sparse(const efm_handle* hc, int32_t* nnz, int32_t* rxn, int64_t* val, int64_t capacity_rows) {
    efm_handle* h = const_cast<efm_handle*>(hc);
    if (!h) return EFM_E_INVAL;
    if (!h->have_result) return EFM_E_STATE;
    if (capacity_rows < h->n_out) return EFM_E_INVAL;
    if (h->n_out == 0) return EFM_OK;
    ON_DEVICE(h);
    const size_t K = (size_t)h->n_out;
    if (nnz) CK(cudaMemcpyAsync(nnz, h->ws + h->lay.r_nnz.off, K * 4, cudaMemcpyDeviceToHost, h->stream));
    if (rxn) CK(cudaMemcpyAsync(rxn, h->ws + h->lay.r_rxn.off, K * h->D * 4, cudaMemcpyDeviceToHost, h->stream));
    if (val) CK(cudaMemcpyAsync(val, h->ws + h->lay.r_val.off, K * h->D * 8, cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    return EFM_OK;
}

int efm_get_stats(const efm_handle* h, efm_stats* st) {
    if (!h || !st) return EFM_E_INVAL;
    *st = h->stats;
    return EFM_OK;
}

int efm_get_level_stats(const efm_handle* h, int64_t* active, int64_t* done, int64_t* expanded, int64_t* children,
                        int64_t capacity, int64_t* n_levels) {
    if (!h || !n_levels) return EFM_E_INVAL;
    const int64_t nl = (int64_t)h->lvl_active.size();
    *n_levels = nl;
    for (int64_t i = 0; i < std::min(nl, capacity); ++i) {
        if (active) active[i] = h->lvl_active[i];
        if (done) done[i] = h->lvl_done[i];
        if (expanded) expanded[i] = h->lvl_expanded[i];
        if (children) children[i] = h->lvl_children[i];
    }
    return EFM_OK;
}

int efm_debug_state_hash(int32_t device, int32_t n_supp, const int32_t* arc, const int64_t* flux, int32_t n_vis,
                         const int32_t* vis4, uint64_t* hash_out) {
    if (n_supp < 0 || n_vis < 0 || !hash_out || (n_supp && (!arc || !flux)) || (n_vis && !vis4)) return EFM_E_INVAL;
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return EFM_E_CUDA; }
    // pinned, device-mapped host staging: the library never allocates device memory
    const size_t bytes = 16 + (size_t)n_supp * 12 + (size_t)n_vis * 16 + 64;
    unsigned char* p = nullptr;
    if (cudaHostAlloc((void**)&p, bytes, cudaHostAllocMapped) != cudaSuccess) { cudaGetLastError(); return EFM_E_CUDA; }
    u64* out = (u64*)p;
    i64* f = (i64*)(p + 16);
    int* a = (int*)(f + n_supp);
    int* v = a + n_supp;
    for (int t = 0; t < n_supp; ++t) { f[t] = flux[t]; a[t] = arc[t]; }
    for (int t = 0; t < 4 * n_vis; ++t) v[t] = vis4[t];
    cudaError_t e = launch_debug_hash(n_supp, a, f, n_vis, v, out, 0);
    if (e == cudaSuccess) e = cudaStreamSynchronize(0);
    if (e == cudaSuccess) *hash_out = *out;
    cudaFreeHost(p);
    if (e != cudaSuccess) { cudaGetLastError(); return EFM_E_CUDA; }
    return EFM_OK;
}

int efm_beam_threshold_scratch_bytes(int64_t n_slots, size_t* bytes) {
    if (n_slots < 0 || !bytes) return EFM_E_INVAL;
    *bytes = ((sizeof(Ctl) + 255) & ~(size_t)255) + 8 * (size_t)std::max<int64_t>(n_slots, 1);
    return EFM_OK;
}

int efm_beam_threshold(const uint64_t* d_keys, int64_t n_slots, int64_t n_active, int64_t cap, void* d_scratch, size_t scratch_bytes,
                       uint64_t* d_threshold, int32_t device, void* cuda_stream) {
    size_t need = 0;
    if (n_slots <= 0 || cap <= 0 || n_active <= cap || n_active > n_slots || !d_keys || !d_scratch || !d_threshold ||
        ((uintptr_t)d_scratch & 255)) return EFM_E_INVAL;
    efm_beam_threshold_scratch_bytes(n_slots, &need);
    if (scratch_bytes < need) return EFM_E_NOMEM;
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return EFM_E_CUDA; }
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess || sms <= 0) { cudaGetLastError(); return EFM_E_CUDA; }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    Ctl* ctl = (Ctl*)d_scratch;
    u64* ckeys = (u64*)((unsigned char*)d_scratch + ((sizeof(Ctl) + 255) & ~(size_t)255));
    // the control block as the traversal leaves it before launch_select(): level set 0 knows its slots and its active children
    LevelCtl lv;
    memset(&lv, 0, sizeof lv);
    lv.n_slots = (u64)n_slots; lv.n_keys = (u64)n_active;
    int launches = 0;
    u32 err = 0;
    cudaError_t e = cudaMemsetAsync(ctl, 0, sizeof(Ctl), s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(&ctl->lv[0], &lv, sizeof lv, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = launch_select((const u64*)d_keys, ckeys, (u64)n_slots, ctl, 0, (u64)cap, (u64)n_slots, sms, s, &launches);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_threshold, &ctl->X, sizeof(u64), cudaMemcpyDeviceToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(&err, &ctl->error, sizeof err, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { cudaGetLastError(); return EFM_E_CUDA; }
    return err ? EFM_E_CAPACITY : EFM_OK;
}

void efm_destroy(efm_handle* h) {
    if (!h) return;
    for (cudaEvent_t e : h->events) cudaEventDestroy(e);
    if (h->h_ctl) cudaFreeHost(h->h_ctl);
    delete h;
}

}  // extern "C"
