// Stoichiometry -> AND/OR graph builder.  Host C++, runs once per efm_create().
#include "graph.hpp"

#include <algorithm>
#include <thread>

#include "../../include/efm_b200.h"

namespace efm {

int build_graph(HostGraph& G, const int32_t* S, int32_t m, int32_t n, int64_t row_stride,
                const uint8_t* reversible, const uint8_t* internal, int32_t dep_depth) {
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
    // A metabolite's consumer list is swept once per search: the first arc x that reaches q stamps every consumer but
    // twin(x); a second, different arc reaching q can only add that one twin.  Nodes are independent, so the searches
    // are spread over host threads (bits of neighbouring nodes can share a word: atomic OR).
    auto worker = [&G, dep_depth](int32_t tid, int32_t nthreads) {
        std::vector<int32_t> stamp((size_t)G.A, -1), frontier, next;
        std::vector<int32_t> q_epoch((size_t)G.M, -1), q_first((size_t)G.M, -1);
        std::vector<char> q_full((size_t)G.M, 0);
        int32_t epoch = 0;
        for (int32_t i = tid; i < G.M; i += nthreads) {
            const int32_t nI = G.in_ptr[i + 1] - G.in_ptr[i];
            if (nI == 0) continue;
            for (int32_t lo = 0; lo < G.out_ptr[i + 1] - G.out_ptr[i]; ++lo) {
                const int32_t o = G.out[G.out_ptr[i] + lo].arc;
                ++epoch;
                frontier.assign(1, o);
                stamp[o] = epoch;
                for (int32_t hop = 1; hop < dep_depth && !frontier.empty(); ++hop) {
                    next.clear();
                    for (int32_t x : frontier)
                        for (int32_t q = G.col_ptr[x]; q < G.col_ptr[x + 1]; ++q) {
                            if (G.col[q].s <= 0 || G.col[q].met == i) continue;
                            const int32_t via = G.col[q].met;
                            if (q_epoch[via] != epoch) {
                                q_epoch[via] = epoch; q_first[via] = x; q_full[via] = 0;
                                for (int32_t r = G.out_ptr[via]; r < G.out_ptr[via + 1]; ++r) {
                                    const int32_t y = G.out[r].arc;
                                    if (y == G.twin[x] || stamp[y] == epoch) continue;
                                    stamp[y] = epoch;
                                    next.push_back(y);
                                }
                            } else if (!q_full[via] && q_first[via] != x) {
                                q_full[via] = 1;
                                const int32_t y = G.twin[q_first[via]];   // consumes `via` because its twin produces it
                                if (y >= 0 && stamp[y] != epoch) { stamp[y] = epoch; next.push_back(y); }
                            }
                        }
                    frontier.swap(next);
                }
                for (int32_t le = 0; le < nI; ++le) {
                    const int32_t e = G.in[G.in_ptr[i] + le].arc;
                    if (e != o && stamp[e] == epoch) {
                        const int64_t b = G.dep_off[i] + (int64_t)lo * nI + le;
                        __atomic_fetch_or(&G.dep_bits[b >> 5], 1u << (b & 31), __ATOMIC_RELAXED);
                    }
                }
            }
        }
    };
    int32_t nthreads = (int32_t)std::thread::hardware_concurrency();
    nthreads = std::max(1, std::min(nthreads, 32));
    if (G.dep_off[G.M] < 4096) nthreads = 1;
    if (nthreads == 1) worker(0, 1);
    else {
        std::vector<std::thread> pool;
        for (int32_t t = 0; t < nthreads; ++t) pool.emplace_back(worker, t, nthreads);
        for (std::thread& t : pool) t.join();
    }
    return EFM_OK;
}

}  // namespace efm
