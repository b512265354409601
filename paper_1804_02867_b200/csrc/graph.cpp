// Stoichiometry -> AND/OR graph builder.  Host C++, runs once per efm_create().
#include "graph.hpp"

#include <algorithm>
#include <thread>

#include "../../include/efm_b200.h"

namespace efm {

int32_t blocked_reactions(const int32_t* S, int32_t m, int32_t n, int64_t row_stride, const uint8_t* reversible,
                          const uint8_t* internal, uint8_t* blocked) {
    // sparse rows of the internal metabolites; a work list of the metabolites whose reactions changed
    std::vector<std::vector<int32_t>> row((size_t)m);
    std::vector<std::vector<int32_t>> col((size_t)n);
    for (int32_t i = 0; i < m; ++i) {
        if (!internal[i]) continue;
        const int32_t* r = S + (int64_t)i * row_stride;
        for (int32_t j = 0; j < n; ++j)
            if (r[j] != 0) { row[i].push_back(j); col[j].push_back(i); }
    }
    std::fill(blocked, blocked + n, (uint8_t)0);
    std::vector<int32_t> work;
    std::vector<char> queued((size_t)m, 0);
    for (int32_t i = 0; i < m; ++i) if (internal[i] && !row[i].empty()) { work.push_back(i); queued[i] = 1; }
    int32_t n_blocked = 0;
    while (!work.empty()) {
        const int32_t i = work.back();
        work.pop_back();
        queued[i] = 0;
        // first two distinct reactions that can produce / consume i: a pair of different reactions exists iff
        // both sides are non-empty and they are not one and the same single reaction
        int32_t p0 = -1, p1 = -1, c0 = -1, c1 = -1, touching = 0;
        const int32_t* r = S + (int64_t)i * row_stride;
        for (int32_t j : row[i]) {
            if (blocked[j]) continue;
            ++touching;
            if (r[j] > 0 || reversible[j]) { if (p0 < 0) p0 = j; else if (p1 < 0) p1 = j; }
            if (r[j] < 0 || reversible[j]) { if (c0 < 0) c0 = j; else if (c1 < 0) c1 = j; }
        }
        if (touching == 0) continue;
        const bool ok = p0 >= 0 && c0 >= 0 && (p1 >= 0 || c1 >= 0 || p0 != c0);
        if (ok) continue;
        for (int32_t j : row[i]) {
            if (blocked[j]) continue;
            blocked[j] = 1;
            ++n_blocked;
            for (int32_t i2 : col[j]) if (i2 != i && !queued[i2]) { work.push_back(i2); queued[i2] = 1; }
        }
    }
    return n_blocked;
}

int build_graph(HostGraph& G, const int32_t* S, int32_t m, int32_t n, int64_t row_stride,
                const uint8_t* reversible, const uint8_t* internal, int32_t dep_depth, const uint8_t* skip_rxn) {
    if (!S || !reversible || !internal || m <= 0 || n <= 0 || row_stride < n || dep_depth < 1) return EFM_E_INVAL;
    G = HostGraph();
    G.m = m;
    G.n = n;
    // Nodes exist only for internal metabolites, in row order (Def 4).
    for (int32_t r = 0; r < m; ++r)
        if (internal[r]) G.met_row.push_back(r);
    G.M = (int32_t)G.met_row.size();
    // Arcs: reaction j's forward arc, directly followed by its backward arc iff reversible (the "direction of the
    // reaction for reversible reactions").
    G.code2arc.assign((size_t)2 * n, -1);
    for (int32_t j = 0; j < n; ++j) {
        if (skip_rxn && skip_rxn[j]) continue;   // compression pre-pass: a blocked reaction gets no arcs
        int32_t fwd = (int32_t)G.arc_rxn.size();
        G.arc_rxn.push_back(j);
        G.arc_dir.push_back(+1);
        G.twin.push_back(reversible[j] ? fwd + 1 : -1);
        G.code2arc[2 * (size_t)j] = fwd;
        if (reversible[j]) {
            G.arc_rxn.push_back(j);
            G.arc_dir.push_back(-1);
            G.twin.push_back(fwd);
            G.code2arc[2 * (size_t)j + 1] = fwd + 1;
        }
    }
    G.A = (int32_t)G.arc_rxn.size();
    if (G.A > 65535 || G.M > 65535) return EFM_E_INVAL;  // 16-bit arc / metabolite ids in the entry format

    // Sparse transpose of S restricted to internal rows: per reaction the list of (node, coefficient).
    std::vector<std::vector<ColRef>> rxn_col((size_t)n);
    for (int32_t i = 0; i < G.M; ++i) {
        const int32_t* row = S + (int64_t)G.met_row[i] * row_stride;
        for (int32_t j = 0; j < n; ++j)
            if (row[j] != 0) rxn_col[j].push_back(ColRef{i, row[j]});
    }
    G.col_ptr.assign((size_t)G.A + 1, 0);
    for (int32_t a = 0; a < G.A; ++a) {
        G.col_ptr[a] = (int32_t)G.col.size();
        for (const ColRef& e : rxn_col[G.arc_rxn[a]]) G.col.push_back(ColRef{e.met, e.s * G.arc_dir[a]});
        G.max_col = std::max(G.max_col, (int32_t)G.col.size() - G.col_ptr[a]);
    }
    G.col_ptr[G.A] = (int32_t)G.col.size();

    // I[i] / O[i] by counting sort over the arc columns; visiting arcs in ascending id keeps each list sorted.
    std::vector<int32_t> n_in((size_t)G.M, 0), n_out((size_t)G.M, 0);
    for (const ColRef& e : G.col) (e.s > 0 ? n_in : n_out)[e.met]++;
    G.in_ptr.assign((size_t)G.M + 1, 0);
    G.out_ptr.assign((size_t)G.M + 1, 0);
    for (int32_t i = 0; i < G.M; ++i) {
        G.in_ptr[i + 1] = G.in_ptr[i] + n_in[i];
        G.out_ptr[i + 1] = G.out_ptr[i] + n_out[i];
        G.max_fanout = std::max(G.max_fanout, std::max(n_in[i], n_out[i]));
    }
    G.in.resize((size_t)G.in_ptr[G.M]);
    G.out.resize((size_t)G.out_ptr[G.M]);
    std::vector<int32_t> fill_in(G.in_ptr.begin(), G.in_ptr.end() - 1), fill_out(G.out_ptr.begin(), G.out_ptr.end() - 1);
    for (int32_t a = 0; a < G.A; ++a)
        for (int32_t q = G.col_ptr[a]; q < G.col_ptr[a + 1]; ++q) {
            const ColRef& e = G.col[q];
            if (e.s > 0) G.in[fill_in[e.met]++] = ArcRef{a, e.s};
            else G.out[fill_out[e.met]++] = ArcRef{a, -e.s};
        }

    // Flux-dependency table (Def 11; Alg 2, readings G6/G7): for node i, output arc o and input
    // arc e != o are dependent iff e is reachable from o in at most L-1 hops of the relation
    //   x -> y  :  y consumes an internal product q != i of x, and y is not the twin of x.
    // The hop relation depends on the current arc only, so a breadth-first sweep with hop stamps is exact.
    G.dep_off.assign((size_t)G.M + 1, 0);
    for (int32_t i = 0; i < G.M; ++i)
        G.dep_off[i + 1] = G.dep_off[i] + (int64_t)(G.out_ptr[i + 1] - G.out_ptr[i]) * (G.in_ptr[i + 1] - G.in_ptr[i]);
    G.dep_bits.assign((size_t)((G.dep_off[G.M] + 31) / 32) + 1, 0u);
    // 64 searches run at once, one bit each (bit s of R[y]: arc y is reachable from the start arc of search s).  A hop
    // goes through the metabolites: ANY[q] = OR of R over the producers of q, MULTI[q] = bits set in at least two of
    // them, both without the searches whose own node is q (the chain must not pass through N_i).  A consumer y of q
    // whose twin also produces q must not be entered from that twin: it takes MULTI[q] | (ANY[q] & ~R[twin(y)]),
    // every other consumer takes ANY[q].  The relation x -> y is a property of the pair, so reachability within
    // L-1 hops is R_{h+1} = R_h | step(R_h).
    struct Src { int32_t node, lo, arc; };
    std::vector<Src> srcs;
    for (int32_t i = 0; i < G.M; ++i) {
        if (G.in_ptr[i + 1] == G.in_ptr[i]) continue;
        for (int32_t lo = 0; lo < G.out_ptr[i + 1] - G.out_ptr[i]; ++lo) srcs.push_back(Src{i, lo, G.out[G.out_ptr[i] + lo].arc});
    }
    const int64_t n_batches = ((int64_t)srcs.size() + 63) / 64;
    auto worker = [&G, &srcs, n_batches, dep_depth](int32_t tid, int32_t nthreads) {
        std::vector<uint64_t> R((size_t)G.A), Rn((size_t)G.A), any((size_t)G.M), multi((size_t)G.M), ex((size_t)G.M, 0);
        for (int64_t b = tid; b < n_batches; b += nthreads) {
            const size_t s0 = (size_t)b * 64, s1 = std::min(srcs.size(), s0 + 64);
            std::fill(R.begin(), R.end(), 0ULL);
            for (size_t s = s0; s < s1; ++s) { R[srcs[s].arc] |= 1ULL << (s - s0); ex[srcs[s].node] |= 1ULL << (s - s0); }
            for (int32_t hop = 1; hop < dep_depth; ++hop) {
                for (int32_t q = 0; q < G.M; ++q) {
                    uint64_t an = 0, mu = 0;
                    for (int32_t r = G.in_ptr[q]; r < G.in_ptr[q + 1]; ++r) { const uint64_t v = R[G.in[r].arc]; mu |= an & v; an |= v; }
                    any[q] = an & ~ex[q]; multi[q] = mu & ~ex[q];
                }
                for (int32_t y = 0; y < G.A; ++y) {
                    uint64_t acc = 0;
                    const int32_t t = G.twin[y];
                    const uint64_t not_t = t >= 0 ? ~R[t] : ~0ULL;   // twin(y) produces exactly what y consumes
                    for (int32_t q = G.col_ptr[y]; q < G.col_ptr[y + 1]; ++q)
                        if (G.col[q].s < 0) acc |= multi[G.col[q].met] | (any[G.col[q].met] & not_t);
                    Rn[y] = R[y] | acc;
                }
                R.swap(Rn);
            }
            for (size_t s = s0; s < s1; ++s) {
                const int32_t i = srcs[s].node, nI = G.in_ptr[i + 1] - G.in_ptr[i];
                for (int32_t le = 0; le < nI; ++le) {
                    const int32_t e = G.in[G.in_ptr[i] + le].arc;
                    if (e != srcs[s].arc && ((R[e] >> (s - s0)) & 1ULL)) {
                        const int64_t bit = G.dep_off[i] + (int64_t)srcs[s].lo * nI + le;
                        __atomic_fetch_or(&G.dep_bits[bit >> 5], 1u << (bit & 31), __ATOMIC_RELAXED);
                    }
                }
                ex[srcs[s].node] = 0;
            }
        }
    };
    int32_t nthreads = (int32_t)std::thread::hardware_concurrency();
    nthreads = std::max(1, std::min(nthreads, 32));
    nthreads = (int32_t)std::max<int64_t>(1, std::min<int64_t>(nthreads, n_batches));
    if (nthreads == 1) worker(0, 1);
    else {
        std::vector<std::thread> pool;
        for (int32_t t = 0; t < nthreads; ++t) pool.emplace_back(worker, t, nthreads);
        for (std::thread& t : pool) t.join();
    }
    return EFM_OK;
}

}  // namespace efm
