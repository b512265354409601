// Host-side builder of the modified AND/OR graph MG (Defs 4-6) and of the static
// flux-dependency table (Def 11; Alg 2 DEPTHy) -- SURVEY.md 8(a) row a-1.
// Part of the product library; shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <vector>

namespace efm {

struct ArcRef {   // one entry of a node's I or O array (Def 5): reaction arc + coefficient c_ij
    int32_t arc;
    int32_t c;    // |stoichiometric coefficient| (Def 6)
};
struct ColRef {   // one nonzero of an arc's column over the internal metabolites
    int32_t met;
    int32_t s;    // signed: > 0 the arc produces met, < 0 it consumes met
};

struct HostGraph {
    int32_t m = 0, n = 0;   // rows / columns of S
    int32_t M = 0, A = 0;   // internal metabolites (nodes of MG), arcs
    std::vector<int32_t> met_row;            // node -> row of S
    std::vector<int32_t> arc_rxn, arc_dir, twin;   // arc -> reaction, +1/-1, twin arc or -1
    std::vector<int32_t> code2arc;           // 2*j + (dir<0) -> arc or -1
    std::vector<int32_t> col_ptr;            // [A+1]
    std::vector<ColRef> col;                 // internal column of every arc, ascending metabolite
    std::vector<int32_t> in_ptr, out_ptr;    // [M+1]
    std::vector<ArcRef> in, out;             // I[i] producers, O[i] consumers, ascending arc id
    std::vector<int64_t> dep_off;            // [M+1], entry index of (lo = 0, le = 0) of node i
    std::vector<uint32_t> dep_bits;          // bit (dep_off[i] + lo*|I_i| + le)
    int32_t max_fanout = 1;                  // max over nodes of max(|I_i|, |O_i|)
    int32_t max_col = 0;                     // longest internal column

    bool dep(int32_t i, int32_t lo, int32_t le) const {
        int64_t b = dep_off[i] + (int64_t)lo * (in_ptr[i + 1] - in_ptr[i]) + le;
        return (dep_bits[b >> 5] >> (b & 31)) & 1u;
    }
};

// Returns 0 or a negative EFM_E_* code.  skip_rxn (may be null): reactions left out of the graph (no arcs are made for them;
// the arcs of the others keep the ORIGINAL reaction index in arc_rxn, so results stay in the caller's reaction space).
int build_graph(HostGraph& G, const int32_t* S, int32_t m, int32_t n, int64_t row_stride,
                const uint8_t* reversible, const uint8_t* internal, int32_t dep_depth, const uint8_t* skip_rxn = nullptr);

// SURVEY.md 8(f)-4 compression pre-pass: reactions that cannot carry flux in any steady state for a
// topological reason.  An internal metabolite whose remaining reactions offer no pair (producer, consumer) of two different
// reactions forces all of them to zero; iterated to the fixed point.  blocked[n] out; returns the number blocked.
int32_t blocked_reactions(const int32_t* S, int32_t m, int32_t n, int64_t row_stride, const uint8_t* reversible,
                          const uint8_t* internal, uint8_t* blocked);

}  // namespace efm
