/*
 * efm_oracle.c -- TEST INFRASTRUCTURE.  Plain, slow, CPU-only oracle for the AND/OR-graph
 * pathway traversal of arXiv 1804.02867, following the algorithm
 * step by step in the reading fixed by SURVEY.md 8(c) (steps O1-O9, beam B) and DESIGN.md
 * ("Readings").  It shares NO code with the CUDA library: only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 *
 * What is pinned (tests/test_oracle_pins.py, -m "not gpu"; every rule below dies under a one-line mutation):
 *   - hand-derived mini networks P1-P6 and H1-H8 (tests/golden/hand_pins.json) with the state of every partial pathway
 *     on every level: Eq 3 scaling, Eq 4 / Eq 5 forward and backward, the Def 11 lookup per (output, input) pair,
 *     PI / PO = lowest arc (G13), lowest metabolite first (G12), first visit over arcs of the support (G22), gcd
 *     normalisation (G10), MAX_LOOP / V / D exactly reached and exceeded, the poison rule and the minimality filter;
 *   - closed forms: linear chains (P6), the 2^62 guard on coefficient chains (3^39 < 2^62 < 3^40, 2^62 vs 2^63, the
 *     extra-flux guard);
 *   - the mirror symmetry S -> -S (forward and backward halves of the procedure must agree);
 *   - unimolecular networks = textbook path / cycle enumeration (P7), brute-force EFM enumeration on toy (P9),
 *     invariants (P8), order independence (P10), default seeds = boundary arcs;
 *   - beam B against its sort-based definition restated on the level contents (test hook `trace`), ties;
 *   - O8(ii)/(iii) restated on the oracle's own balanced entries with multi-arc seed sets (poison and drops occur);
 *   - the state hash against published SplitMix64 vectors and its written composition; the DEP table against
 *     exhaustive chain enumeration.
 *   - the extra modes (tests/test_oracle_modes.py, tests/test_compress.py): the sampled choice against the generator
 *     restated in Python, states reached by sampling against the exhaustive fan-out (Theorem 1), hand-derived reaction
 *     masks and step counts, the exact mode against rational rank by fraction elimination and brute force, the
 *     compression pre-pass (oracle/compress.py) against brute-force EFMs and the unchanged exhaustive result.
 * Parity unpinned: the exact output sets of the configs "small".."genome" as a whole (no external truth exists; they
 * are held by the pins above, which cover every rule that produces them, and by GPU<->oracle parity).
 *
 * Arithmetic: fluxes and extra fluxes are exact integers (reading G10); every product is formed
 * in __int128 so the 2^62 guard (reading G21) can never itself overflow.
 *
 * Notation follows the paper: M internal metabolites N_i (Def 4), I / O input and
 * output reaction arrays (Def 5), coefficient c (Def 6), flux f,
 * EF extra flux (Eq 2), PI / PO primary input / output (Def 10).
 */
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef __int128 i128;
#define GUARD ((i128)1 << 62) /* reading G21: any state integer above 2^62 discards the pathway */

/* ------------------------------------------------------------------ parameters / results */
typedef struct {
    int32_t max_support;   /* D  : max arcs in a pathway (reading G15)                     */
    int32_t max_loop;      /* MAX_LOOP (reading G9)                     */
    int32_t dep_depth;     /* L  : chain length of the dependency search    */
    int32_t max_visited;   /* V  : max visited metabolites per pathway                     */
    int64_t frontier_cap;  /* beam B: entries expanded per level, 0 = unbounded            */
    int32_t threads;       /* OpenMP threads used over the entries of a level              */
    int32_t trace;         /* 1: record every entry of every level, 2: only the balanced ones (test hook) */
    uint64_t shuffle_seed; /* != 0: permute every level before processing (pin P10)        */
    /* SURVEY.md 8(f)-1 literal sampling mode ("each pathway is created using randomly selected output/input",
     * PAPER.md:360 "after attempting 48 EFM candidates"): sample_count = C > 0 runs C candidate pathways, candidate c starts
     * from seed set c mod n_sets and takes ONE admissible alternative per first visit, chosen by the counter-based
     * generator pick(sample_seed, c, i*) below; no fan-out, no beam. */
    int32_t sample_count;
    /* SURVEY.md 8(f)-3 exact elementarity (Def 3; "recognizing the elementarity through rank
     * test"): exact != 0 replaces step O8(iii) "minimal among the candidates found" by the rank test on every unique,
     * unpoisoned support: it stays iff the internal rows of S restricted to its arcs have rank |supp| - 1 (nullity 1).
     * The rank is taken over GF(p), p = 2^31 - 1: a well-defined number (any elimination order gives it), never above the
     * rational rank, and the candidate's own flux vector bounds the rational rank by |supp| - 1 from above -- so every
     * "elementary" verdict is exact; a "not elementary" verdict errs only if p divides a minor (reading G24). */
    int32_t exact;
    uint64_t sample_seed;
    /* SURVEY.md 8(f)-2 targeted observability ("contributing reactions of each EFM were selected intentionally",
     * PAPER.md:392-396): allowed[j] = 0 makes every OR-alternative of reaction j inadmissible; NULL = all allowed */
    const uint8_t *allowed;
} oracle_params;

typedef struct {
    int64_t levels, expanded, children, done, dead_end, not_efm_maxloop, discarded_nonpos,
        discarded_overflow, discarded_visited, truncated_beam, unique_supports, poisoned, output;
    int64_t peak_frontier; /* largest number of active entries in a level (before the beam) */
    int64_t algo_bytes;    /* SURVEY.md 8(d) algorithmic bytes summed over all expansions   */
    int64_t non_elementary; /* exact mode: unique, unpoisoned supports the rank test rejected */
} oracle_stats;

/* ------------------------------------------------------------------ O1: the MG graph */
typedef struct {
    int m, n;  /* rows (metabolites), columns (reactions) of S                               */
    int M, A;  /* internal metabolites, arcs                                                 */
    int *met_row;                    /* internal index -> row of S                           */
    int *arc_rxn, *arc_dir, *twin;   /* arc -> reaction, +1/-1, twin arc or -1               */
    /* column of arc a over internal metabolites: signed arc coefficient s_ia               */
    int *col_ptr, *col_met;
    int64_t *col_s;
    /* I[i]: arcs producing i (s_ia > 0), O[i]: arcs consuming i (s_ia < 0); ascending arc id */
    int *in_ptr, *in_arc, *out_ptr, *out_arc;
    int64_t *in_c, *out_c;
    /* O7: dep[dep_off[i] + lo * |I[i]| + le] = 1 iff (O[i][lo], I[i][le]) is flux-dependent */
    int64_t *dep_off;
    uint8_t *dep;
    int W; /* bitset words of 64 arcs */
} graph;

static void graph_free(graph *G) {
    free(G->met_row); free(G->arc_rxn); free(G->arc_dir); free(G->twin);
    free(G->col_ptr); free(G->col_met); free(G->col_s);
    free(G->in_ptr); free(G->in_arc); free(G->in_c);
    free(G->out_ptr); free(G->out_arc); free(G->out_c);
    free(G->dep_off); free(G->dep);
    memset(G, 0, sizeof *G);
}

/* O1 (Defs 4-6): nodes = internal metabolites in row order; arcs in reaction order,
 * forward arc then (iff reversible) backward arc whose column is -S_j. */
static int graph_build(graph *G, const int32_t *S, int m, int n, const uint8_t *rev,
                       const uint8_t *internal, int L) {
    memset(G, 0, sizeof *G);
    G->m = m; G->n = n;
    G->met_row = malloc(sizeof(int) * (m + 1));
    for (int r = 0; r < m; r++) if (internal[r]) G->met_row[G->M++] = r;
    int A = 0;
    for (int j = 0; j < n; j++) A += rev[j] ? 2 : 1;
    G->A = A; G->W = (A + 63) / 64;
    G->arc_rxn = malloc(sizeof(int) * (A + 1));
    G->arc_dir = malloc(sizeof(int) * (A + 1));
    G->twin = malloc(sizeof(int) * (A + 1));
    int a = 0;
    for (int j = 0; j < n; j++) {
        G->arc_rxn[a] = j; G->arc_dir[a] = +1; G->twin[a] = rev[j] ? a + 1 : -1; a++;
        if (rev[j]) { G->arc_rxn[a] = j; G->arc_dir[a] = -1; G->twin[a] = a - 1; a++; }
    }
    int M = G->M;
    /* columns */
    G->col_ptr = calloc(A + 1, sizeof(int));
    int64_t nnz = 0;
    for (a = 0; a < A; a++)
        for (int i = 0; i < M; i++)
            if (S[(int64_t)G->met_row[i] * n + G->arc_rxn[a]] != 0) nnz++;
    G->col_met = malloc(sizeof(int) * (nnz + 1));
    G->col_s = malloc(sizeof(int64_t) * (nnz + 1));
    int64_t p = 0;
    for (a = 0; a < A; a++) {
        G->col_ptr[a] = (int)p;
        for (int i = 0; i < M; i++) {
            int64_t s = (int64_t)S[(int64_t)G->met_row[i] * n + G->arc_rxn[a]] * G->arc_dir[a];
            if (s != 0) { G->col_met[p] = i; G->col_s[p] = s; p++; }
        }
    }
    G->col_ptr[A] = (int)p;
    /* I / O arrays per node, ascending arc id, c = |s| (Def 6) */
    G->in_ptr = calloc(M + 1, sizeof(int)); G->out_ptr = calloc(M + 1, sizeof(int));
    G->in_arc = malloc(sizeof(int) * (nnz + 1)); G->out_arc = malloc(sizeof(int) * (nnz + 1));
    G->in_c = malloc(sizeof(int64_t) * (nnz + 1)); G->out_c = malloc(sizeof(int64_t) * (nnz + 1));
    int pi = 0, po = 0;
    for (int i = 0; i < M; i++) {
        G->in_ptr[i] = pi; G->out_ptr[i] = po;
        for (a = 0; a < A; a++) {
            int64_t s = (int64_t)S[(int64_t)G->met_row[i] * n + G->arc_rxn[a]] * G->arc_dir[a];
            if (s > 0) { G->in_arc[pi] = a; G->in_c[pi] = s; pi++; }
            if (s < 0) { G->out_arc[po] = a; G->out_c[po] = -s; po++; }
        }
    }
    G->in_ptr[M] = pi; G->out_ptr[M] = po;
    /* O7 (Def 11; Alg 2; readings G6, G7): (o, e) in DEP[i] iff a
     * chain of arcs x_1 = o, ..., x_k = e with k <= L exists in which x_{t+1} consumes an internal
     * product q != i of x_t and x_{t+1} != twin(x_t).  Breadth-first over arcs, L-1 steps. */
    G->dep_off = malloc(sizeof(int64_t) * (M + 1));
    int64_t tot = 0;
    for (int i = 0; i < M; i++) {
        G->dep_off[i] = tot;
        tot += (int64_t)(G->out_ptr[i + 1] - G->out_ptr[i]) * (G->in_ptr[i + 1] - G->in_ptr[i]);
    }
    G->dep_off[M] = tot;
    G->dep = calloc(tot + 1, 1);
    uint8_t *seen = malloc(A + 1);
    int *cur = malloc(sizeof(int) * (A + 1)), *nxt = malloc(sizeof(int) * (A + 1));
    for (int i = 0; i < M; i++) {
        int nI = G->in_ptr[i + 1] - G->in_ptr[i];
        for (int lo = 0; lo < G->out_ptr[i + 1] - G->out_ptr[i]; lo++) {
            int o = G->out_arc[G->out_ptr[i] + lo];
            memset(seen, 0, A);
            int ncur = 0, nnxt;
            seen[o] = 1; cur[ncur++] = o;
            for (int step = 1; step < L && ncur > 0; step++) {
                nnxt = 0;
                for (int t = 0; t < ncur; t++) {
                    int x = cur[t];
                    for (int q0 = G->col_ptr[x]; q0 < G->col_ptr[x + 1]; q0++) {
                        if (G->col_s[q0] <= 0) continue; /* products of x only */
                        int q = G->col_met[q0];
                        if (q == i) continue;            /* do not continue through N_i */
                        for (int y0 = G->out_ptr[q]; y0 < G->out_ptr[q + 1]; y0++) {
                            int y = G->out_arc[y0];
                            if (y == G->twin[x]) continue;
                            if (!seen[y]) { seen[y] = 1; nxt[nnxt++] = y; }
                        }
                    }
                }
                int *tmp = cur; cur = nxt; nxt = tmp; ncur = nnxt;
            }
            for (int le = 0; le < nI; le++) {
                int e = G->in_arc[G->in_ptr[i] + le];
                if (e != o && seen[e]) G->dep[G->dep_off[i] + (int64_t)lo * nI + le] = 1;
            }
        }
    }
    free(seen); free(cur); free(nxt);
    return 0;
}

/* ------------------------------------------------------------------ O3: state of a partial pathway */
typedef struct { int32_t met, PI, PO, cnt; } visit;
typedef struct {
    int32_t n_supp, n_vis;
    int32_t cand;  /* root (seed set / sampled candidate) the pathway descends from */
    int32_t level; /* number of expansions that built it (its "steps") */
    int32_t *arc;  /* support arcs, ascending arc id       */
    int64_t *f;    /* their fluxes, > 0, gcd = 1           */
    visit *vis;    /* visited metabolites, ascending index */
} entry;

static entry *entry_new(int n_supp, int n_vis) {
    size_t sz = sizeof(entry) + sizeof(int64_t) * n_supp + sizeof(visit) * n_vis + sizeof(int32_t) * n_supp + 16;
    char *p = malloc(sz);
    if (!p) { fprintf(stderr, "oracle: out of memory\n"); abort(); }
    entry *e = (entry *)p;
    e->n_supp = n_supp; e->n_vis = n_vis; e->cand = 0; e->level = 0;
    e->f = (int64_t *)(p + sizeof(entry));
    e->vis = (visit *)(e->f + n_supp);
    e->arc = (int32_t *)(e->vis + n_vis);
    return e;
}

typedef struct { entry **v; int64_t n, cap; } evec;
static void evec_push(evec *V, entry *e) {
    if (V->n == V->cap) { V->cap = V->cap ? V->cap * 2 : 64; V->v = realloc(V->v, sizeof(entry *) * V->cap); }
    V->v[V->n++] = e;
}

static int find_arc(const entry *e, int a) {
    for (int k = 0; k < e->n_supp; k++) if (e->arc[k] == a) return k;
    return -1;
}
static int find_vis(const entry *e, int i) {
    for (int k = 0; k < e->n_vis; k++) if (e->vis[k].met == i) return k;
    return -1;
}

static uint64_t ugcd(uint64_t a, uint64_t b) { while (b) { uint64_t t = a % b; a = b; b = t; } return a; }

/* Eq 2: EF_i = sum over support arcs of s_ia * f_a, internal metabolites only (G20) */
static void extra_flux(const graph *G, const entry *e, i128 *EF /* [M], zero on entry */, int *touched, int *ntouched) {
    *ntouched = 0;
    for (int k = 0; k < e->n_supp; k++) {
        int a = e->arc[k];
        for (int q = G->col_ptr[a]; q < G->col_ptr[a + 1]; q++) {
            int i = G->col_met[q];
            touched[(*ntouched)++] = i;
            EF[i] += (i128)G->col_s[q] * e->f[k];
        }
    }
}

/* ------------------------------------------------------------------ beam B: key of an entry */
static uint64_t mix64(uint64_t x) { /* splitmix64 finaliser */
    x ^= x >> 30; x *= 0xBF58476D1CE4E5B9ULL;
    x ^= x >> 27; x *= 0x94D049BB133111EBULL;
    x ^= x >> 31; return x;
}
/* State hash h of beam B ("a 64-bit hash of the complete state ... The builder may change h,
 * but it must be written down once and implemented twice, independently"; reading G16 writes it down):
 *   h = mix( sum_{a in supp} mix(0x01<<56 | a) * f_a  +  sum_{i visited} mix(0x02<<56 | cnt<<48 | i<<32 | PI<<16 | PO) )
 * all sums and products modulo 2^64.  The arc part is a multiply-add (universal) hash with one fixed
 * pseudo-random multiplier per arc, so it is linear in the flux vector. */
static uint64_t state_hash(const entry *e) {
    uint64_t s = 0;
    for (int k = 0; k < e->n_supp; k++)
        s += mix64(0x0100000000000000ULL | (uint64_t)e->arc[k]) * (uint64_t)e->f[k];
    for (int k = 0; k < e->n_vis; k++) {
        const visit *v = &e->vis[k];
        s += mix64(0x0200000000000000ULL | ((uint64_t)v->cnt << 48) | ((uint64_t)v->met << 32) |
                   ((uint64_t)v->PI << 16) | (uint64_t)v->PO);
    }
    return mix64(s);
}
static uint64_t beam_key(const entry *e, int n_unb) {
    uint64_t nu = n_unb > 255 ? 255 : (uint64_t)n_unb;
    return (nu << 56) | (state_hash(e) >> 8);
}
static int cmp_u64(const void *a, const void *b) {
    uint64_t x = *(const uint64_t *)a, y = *(const uint64_t *)b;
    return x < y ? -1 : (x > y ? 1 : 0);
}

/* irreducible content of an entry */
static int64_t algo_entry_bytes(const entry *e) { return (int64_t)e->n_supp * 10 + (int64_t)e->n_vis * 7 + 16; }

/* ------------------------------------------------------------------ O6: bump */
enum { BUMP_OK = 0, BUMP_NONPOS = 1, BUMP_OVERFLOW = 2 };

/* bump(f, a, sign * |E| / c): g = gcd(|E|, c); k = c/g; every flux * k; f_a <- f_a +- |E|/g; discard
 * if any scaled flux or any extra flux of the un-normalised child exceeds 2^62 (overflow, G21), or if
 * f_a <= 0 (Prop 3; G11); then divide all fluxes by their gcd (G10).
 * Returns the child (support sorted by arc id; visited list copied unchanged) or NULL. */
static entry *bump(const graph *G, const entry *e, int a, int sign, i128 absE, int64_t c, int extra_vis,
                   i128 *EFs /* scratch [M], zero */, int *touched, int *status) {
    uint64_t g = ugcd((uint64_t)absE, (uint64_t)c);
    i128 k = (i128)(c / (int64_t)g);
    i128 d = absE / (i128)g;
    int pos = find_arc(e, a);
    int n_supp = e->n_supp + (pos < 0 ? 1 : 0);
    entry *ch = entry_new(n_supp, e->n_vis + extra_vis);
    i128 *F = malloc(sizeof(i128) * n_supp);
    int w = 0, placed = (pos >= 0);
    for (int t = 0; t < e->n_supp; t++) {
        if (!placed && a < e->arc[t]) { ch->arc[w] = a; F[w] = 0; w++; placed = 1; }
        ch->arc[w] = e->arc[t]; F[w] = k * (i128)e->f[t]; w++;
    }
    if (!placed) { ch->arc[w] = a; F[w] = 0; w++; }
    int ia = -1;
    for (int t = 0; t < n_supp; t++) if (ch->arc[t] == a) ia = t;
    F[ia] += sign > 0 ? d : -d;
    *status = BUMP_OK;
    for (int t = 0; t < n_supp; t++) if (F[t] > GUARD) *status = BUMP_OVERFLOW;
    if (*status == BUMP_OK && F[ia] <= 0) *status = BUMP_NONPOS;
    if (*status == BUMP_OK) {
        /* extra fluxes of the un-normalised child, from scratch (Eq 2) */
        int nt = 0;
        for (int t = 0; t < n_supp; t++)
            for (int q = G->col_ptr[ch->arc[t]]; q < G->col_ptr[ch->arc[t] + 1]; q++) {
                touched[nt++] = G->col_met[q];
                EFs[G->col_met[q]] += (i128)G->col_s[q] * F[t];
            }
        for (int t = 0; t < nt; t++) {
            i128 v = EFs[touched[t]];
            if (v > GUARD || v < -GUARD) *status = BUMP_OVERFLOW;
        }
        for (int t = 0; t < nt; t++) EFs[touched[t]] = 0;
    }
    if (*status != BUMP_OK) { free(F); free(ch); return NULL; }
    uint64_t g2 = 0;
    for (int t = 0; t < n_supp; t++) g2 = ugcd(g2, (uint64_t)F[t]);
    for (int t = 0; t < n_supp; t++) ch->f[t] = (int64_t)(F[t] / (i128)g2);
    free(F);
    for (int t = 0; t < e->n_vis; t++) ch->vis[t] = e->vis[t];
    return ch;
}

/* insert / update the visited record of metabolite i, keeping the list sorted by metabolite */
static void set_visit(entry *ch, int n_old, int i, int PI, int PO, int cnt) {
    int k = -1;
    for (int t = 0; t < n_old; t++) if (ch->vis[t].met == i) k = t;
    if (k < 0) {
        k = n_old;
        while (k > 0 && ch->vis[k - 1].met > i) { ch->vis[k] = ch->vis[k - 1]; k--; }
    }
    ch->vis[k].met = i; ch->vis[k].PI = PI; ch->vis[k].PO = PO; ch->vis[k].cnt = cnt;
}

/* ------------------------------------------------------------------ O5: pick and branch */
typedef struct {
    oracle_stats st;
    evec children;
    i128 *EF, *EFs;
    int *touched, *touched2;
    uint8_t *insupp;
    int64_t *cand_end;   /* sampling mode: how and when candidate c ended (shared array, one writer per candidate) */
} worker;

/* how a sampled candidate ended: code | steps << 8 (steps = expansions made before the end) */
enum { END_NONE = 0, END_DONE = 1, END_NOTEFM = 2, END_DEAD = 3, END_VISITED = 4, END_NONPOS = 5, END_OVERFLOW = 6 };

/* 8(f)-1: the alternative candidate c takes at the first visit of metabolite i among n admissible ones is number
 * pick mod n in ascending arc order; a counter-based generator (no state, no order dependence), reading G23:
 *   pick(seed, c, i) = mix( mix(seed + 0x9E3779B97F4A7C15 * (c + 1)) ^ (0x04 << 56 | i) ) */
static uint64_t sample_pick(uint64_t seed, int32_t cand, int32_t met) {
    return mix64(mix64(seed + 0x9E3779B97F4A7C15ULL * ((uint64_t)cand + 1ULL)) ^ (0x0400000000000000ULL | (uint64_t)met));
}

static void expand(const graph *G, const oracle_params *P, const entry *e, int istar, i128 E, worker *wk) {
    oracle_stats *st = &wk->st;
    int D = P->max_support, V = P->max_visited;
    uint8_t *in = wk->insupp;
    for (int k = 0; k < e->n_supp; k++) in[e->arc[k]] = 1;
    int fwd = E > 0;
    i128 absE = fwd ? E : -E;
    int vk = find_vis(e, istar);
    st->expanded++;
    int64_t bytes = algo_entry_bytes(e);
    if (vk < 0) {
        /* first visit: PROC1 / PROC1' (Eq 3; readings G1, G13, G14, G15, G22) */
        if (e->n_vis >= V) { st->discarded_visited++; if (wk->cand_end) wk->cand_end[e->cand] = END_VISITED | ((int64_t)e->level << 8); goto out; }
        int prim = -1; /* forward: PI = lowest producer in the support; backward: PO = lowest consumer */
        if (fwd) { for (int q = G->in_ptr[istar]; q < G->in_ptr[istar + 1] && prim < 0; q++) if (in[G->in_arc[q]]) prim = G->in_arc[q]; }
        else     { for (int q = G->out_ptr[istar]; q < G->out_ptr[istar + 1] && prim < 0; q++) if (in[G->out_arc[q]]) prim = G->out_arc[q]; }
        int lo = fwd ? G->out_ptr[istar] : G->in_ptr[istar];
        int hi = fwd ? G->out_ptr[istar + 1] : G->in_ptr[istar + 1];
        int n_adm = 0, pick = -1;
        if (P->sample_count > 0) {   /* sampling: count the admissible alternatives first, then take exactly one of them */
            for (int q = lo; q < hi; q++) {
                int a = fwd ? G->out_arc[q] : G->in_arc[q];
                if (G->twin[a] >= 0 && in[G->twin[a]]) continue;
                if (!in[a] && e->n_supp >= D) continue;
                if (P->allowed && !P->allowed[G->arc_rxn[a]]) continue;
                n_adm++;
            }
            if (n_adm > 0) pick = (int)(sample_pick(P->sample_seed, e->cand, istar) % (uint64_t)n_adm);
            n_adm = 0;
        }
        for (int q = lo; q < hi; q++) {
            int a = fwd ? G->out_arc[q] : G->in_arc[q];
            int64_t c = fwd ? G->out_c[q] : G->in_c[q];
            if (G->twin[a] >= 0 && in[G->twin[a]]) continue;     /* G14 twin exclusion */
            if (!in[a] && e->n_supp >= D) continue;              /* G15 support cap    */
            if (P->allowed && !P->allowed[G->arc_rxn[a]]) continue;   /* 8(f)-2: reaction outside the given subset */
            n_adm++;
            if (pick >= 0 && n_adm - 1 != pick) continue;        /* 8(f)-1: only the sampled alternative */
            int status;
            entry *ch = bump(G, e, a, +1, absE, c, 1, wk->EFs, wk->touched2, &status);
            if (!ch) {
                if (status == BUMP_OVERFLOW) st->discarded_overflow++; else st->discarded_nonpos++;
                if (wk->cand_end) wk->cand_end[e->cand] = (status == BUMP_OVERFLOW ? END_OVERFLOW : END_NONPOS) | ((int64_t)e->level << 8);
                continue;
            }
            ch->cand = e->cand; ch->level = e->level + 1;
            set_visit(ch, e->n_vis, istar, fwd ? prim : a, fwd ? a : prim, 0);
            evec_push(&wk->children, ch);
            st->children++;
            bytes += 8;
        }
        if (n_adm == 0) { st->dead_end++; if (wk->cand_end) wk->cand_end[e->cand] = END_DEAD | ((int64_t)e->level << 8); }
    } else {
        /* revisit: PROC2-4 (readings G2-G5) */
        int cnt = e->vis[vk].cnt + 1;
        if (cnt > P->max_loop) { st->not_efm_maxloop++; if (wk->cand_end) wk->cand_end[e->cand] = END_NOTEFM | ((int64_t)e->level << 8); goto out; }
        int PI = e->vis[vk].PI, PO = e->vis[vk].PO;
        int nI = G->in_ptr[istar + 1] - G->in_ptr[istar];
        int lPI = -1, lPO = -1;
        for (int q = 0; q < nI; q++) if (G->in_arc[G->in_ptr[istar] + q] == PI) lPI = q;
        for (int q = 0; q < G->out_ptr[istar + 1] - G->out_ptr[istar]; q++) if (G->out_arc[G->out_ptr[istar] + q] == PO) lPO = q;
        if (lPI < 0 || lPO < 0) { fprintf(stderr, "oracle: primary reaction not adjacent to its node\n"); abort(); }
        int dep = 0;
        if (fwd) { /* PO ~ SI: some producer of i* in the support is reachable from PO */
            for (int q = 0; q < nI; q++)
                if (in[G->in_arc[G->in_ptr[istar] + q]] && G->dep[G->dep_off[istar] + (int64_t)lPO * nI + q]) dep = 1;
        } else {   /* PI ~ SO: PI is reachable from some consumer of i* in the support */
            for (int q = 0; q < G->out_ptr[istar + 1] - G->out_ptr[istar]; q++)
                if (in[G->out_arc[G->out_ptr[istar] + q]] && G->dep[G->dep_off[istar] + (int64_t)q * nI + lPI]) dep = 1;
        }
        int a, sign; int64_t c;
        int64_t cPI = G->in_c[G->in_ptr[istar] + lPI], cPO = G->out_c[G->out_ptr[istar] + lPO];
        if (fwd) { if (!dep) { a = PO; c = cPO; sign = +1; } else { a = PI; c = cPI; sign = -1; } }   /* Eq 4 / Eq 5 */
        else     { if (!dep) { a = PI; c = cPI; sign = +1; } else { a = PO; c = cPO; sign = -1; } }
        int status;
        entry *ch = bump(G, e, a, sign, absE, c, 0, wk->EFs, wk->touched2, &status);
        if (!ch) {
            if (status == BUMP_OVERFLOW) st->discarded_overflow++; else st->discarded_nonpos++;
            if (wk->cand_end) wk->cand_end[e->cand] = (status == BUMP_OVERFLOW ? END_OVERFLOW : END_NONPOS) | ((int64_t)e->level << 8);
            goto out;
        }
        ch->cand = e->cand; ch->level = e->level + 1;
        set_visit(ch, e->n_vis, istar, PI, PO, cnt);
        evec_push(&wk->children, ch);
        st->children++;
        bytes += 8;
    }
out:
    st->algo_bytes += bytes;
    for (int k = 0; k < e->n_supp; k++) in[e->arc[k]] = 0;
}

/* ------------------------------------------------------------------ results */
typedef struct {
    int n;               /* reactions */
    int64_t n_out;
    int64_t *flux;       /* n_out x n, canonical order */
    oracle_stats st;
    int64_t *steps;      /* per output row: expansions that built the pathway (smallest over equal duplicates) */
    int64_t n_cand_end;  /* sampling mode: candidates */
    int64_t *cand_end;   /* code | steps << 8 per candidate */
    int64_t n_levels_rec;
    int64_t *lvl_active, *lvl_done, *lvl_expanded, *lvl_children;
    graph G;
    int n_roots;
    int have_graph;
    /* test hook: one record per entry of every level, in the order the level was processed:
     * level, n_supp, n_vis, n_unb, i* (-1 = balanced), beam key (bit pattern), kept (1 = expanded or balanced),
     * then n_supp x (arc, flux), then n_vis x (met, PI, PO, cnt) */
    int64_t *trace; int64_t trace_n, trace_cap;
} oracle_result;

static void trace_push(oracle_result *R, int64_t v) {
    if (R->trace_n == R->trace_cap) { R->trace_cap = R->trace_cap ? R->trace_cap * 2 : 1024; R->trace = realloc(R->trace, sizeof(int64_t) * R->trace_cap); }
    R->trace[R->trace_n++] = v;
}

static int g_sort_n;
static int cmp_rows(const void *a, const void *b) {
    const int64_t *x = a, *y = b;
    for (int j = 0; j < g_sort_n; j++) { if (x[j] < y[j]) return -1; if (x[j] > y[j]) return 1; }
    return 0;
}
static int cmp_cand(const void *a, const void *b) { /* by support (arc list), then flux */
    const entry *x = *(entry *const *)a, *y = *(entry *const *)b;
    int n = x->n_supp < y->n_supp ? x->n_supp : y->n_supp;
    for (int k = 0; k < n; k++) { if (x->arc[k] != y->arc[k]) return x->arc[k] < y->arc[k] ? -1 : 1; }
    if (x->n_supp != y->n_supp) return x->n_supp < y->n_supp ? -1 : 1;
    for (int k = 0; k < n; k++) { if (x->f[k] != y->f[k]) return x->f[k] < y->f[k] ? -1 : 1; }
    return 0;
}
static int same_support(const entry *x, const entry *y) {
    if (x->n_supp != y->n_supp) return 0;
    for (int k = 0; k < x->n_supp; k++) if (x->arc[k] != y->arc[k]) return 0;
    return 1;
}

static uint64_t rng_next(uint64_t *s) {
    *s += 0x9E3779B97F4A7C15ULL; uint64_t z = *s;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL; z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL; return z ^ (z >> 31);
}

/* ------------------------------------------------------------------ the whole procedure, O2 + O4 + O8 */
#define E_INVAL (-1)

/* 8(f)-3: rank over GF(2^31 - 1) of the internal rows of S restricted to the arcs of e, by plain Gaussian elimination on the
 * dense (touched metabolites) x (arcs) matrix. */
#define RANK_P 2147483647LL
static int64_t inv_mod_p(int64_t a) { /* a^(p-2) mod p */
    int64_t r = 1, b = a % RANK_P, e = RANK_P - 2;
    while (e) { if (e & 1) r = r * b % RANK_P; b = b * b % RANK_P; e >>= 1; }
    return r;
}
static int support_rank(const graph *G, const entry *e) {
    int n = e->n_supp, M = G->M;
    int *row_of = malloc(sizeof(int) * (M + 1));
    for (int i = 0; i < M; i++) row_of[i] = -1;
    int R = 0;
    for (int k = 0; k < n; k++)
        for (int q = G->col_ptr[e->arc[k]]; q < G->col_ptr[e->arc[k] + 1]; q++)
            if (row_of[G->col_met[q]] < 0) row_of[G->col_met[q]] = R++;
    int64_t *Mx = calloc((size_t)(R + 1) * (n + 1), sizeof(int64_t));
    for (int k = 0; k < n; k++)
        for (int q = G->col_ptr[e->arc[k]]; q < G->col_ptr[e->arc[k] + 1]; q++) {
            int64_t v = G->col_s[q] % RANK_P;
            if (v < 0) v += RANK_P;
            Mx[(size_t)row_of[G->col_met[q]] * n + k] = v;
        }
    int rank = 0;
    for (int c = 0; c < n && rank < R; c++) {
        int piv = -1;
        for (int r = rank; r < R; r++) if (Mx[(size_t)r * n + c]) { piv = r; break; }
        if (piv < 0) continue;
        for (int k = 0; k < n; k++) { int64_t t = Mx[(size_t)piv * n + k]; Mx[(size_t)piv * n + k] = Mx[(size_t)rank * n + k]; Mx[(size_t)rank * n + k] = t; }
        int64_t inv = inv_mod_p(Mx[(size_t)rank * n + c]);
        for (int r = rank + 1; r < R; r++) {
            int64_t f = Mx[(size_t)r * n + c] * inv % RANK_P;
            if (!f) continue;
            for (int k = c; k < n; k++) Mx[(size_t)r * n + k] = ((Mx[(size_t)r * n + k] - f * Mx[(size_t)rank * n + k]) % RANK_P + RANK_P) % RANK_P;
        }
        rank++;
    }
    free(Mx); free(row_of);
    return rank;
}

int oracle_enumerate(const int32_t *S, int32_t m, int32_t n, const uint8_t *rev, const uint8_t *internal,
                     const oracle_params *P0, const int32_t *seed_ptr, const int32_t *seed_code, int32_t n_sets,
                     oracle_result **out) {
    oracle_params P = *P0;
    oracle_result *R = calloc(1, sizeof *R);
    graph *G = &R->G;
    graph_build(G, S, m, n, rev, internal, P.dep_depth);
    R->have_graph = 1; R->n = n;
    int M = G->M, A = G->A;
    if (P.max_support <= 0) P.max_support = A;
    if (P.max_visited <= 0) P.max_visited = 2 * P.max_support;
    int nthreads = P.threads > 0 ? P.threads : 1;

    /* arc code 2*j + (dir<0) -> arc id */
    int *code2arc = malloc(sizeof(int) * (2 * n + 2));
    for (int j = 0; j < 2 * n; j++) code2arc[j] = -1;
    for (int a = 0; a < A; a++) code2arc[2 * G->arc_rxn[a] + (G->arc_dir[a] < 0)] = a;

    /* O2 roots: seed arcs <- flux 1; default = one root per boundary arc */
    evec level = {0};
    if (n_sets == 0) {
        for (int a = 0; a < A; a++) {
            int pos = 0, neg = 0;
            for (int q = G->col_ptr[a]; q < G->col_ptr[a + 1]; q++) { if (G->col_s[q] > 0) pos++; else neg++; }
            if ((pos > 0) != (neg > 0)) {
                entry *e = entry_new(1, 0); e->arc[0] = a; e->f[0] = 1; evec_push(&level, e);
            }
        }
    } else {
        uint8_t *mark = calloc(A + 1, 1);
        for (int s = 0; s < n_sets; s++) {
            int cnt = seed_ptr[s + 1] - seed_ptr[s];
            if (cnt <= 0 || cnt > P.max_support) { free(mark); free(code2arc); *out = R; return E_INVAL; }
            entry *e = entry_new(cnt, 0);
            int bad = 0;
            for (int t = 0; t < cnt; t++) {
                int code = seed_code[seed_ptr[s] + t];
                int a = (code >= 0 && code < 2 * n) ? code2arc[code] : -1;
                if (a < 0 || mark[a] || (G->twin[a] >= 0 && mark[G->twin[a]])) { bad = 1; break; }
                mark[a] = 1; e->arc[t] = a; e->f[t] = 1;
            }
            for (int t = 0; t < cnt; t++) { int code = seed_code[seed_ptr[s] + t]; if (code >= 0 && code < 2 * n && code2arc[code] >= 0) mark[code2arc[code]] = 0; }
            if (bad) { free(e); free(mark); free(code2arc); *out = R; return E_INVAL; }
            for (int x = 1; x < cnt; x++) /* keep the support sorted by arc id */
                for (int y = x; y > 0 && e->arc[y - 1] > e->arc[y]; y--) { int t = e->arc[y]; e->arc[y] = e->arc[y - 1]; e->arc[y - 1] = t; }
            evec_push(&level, e);
        }
        free(mark);
    }
    free(code2arc);
    if (P.sample_count > 0) {   /* 8(f)-1: candidate c is a copy of root c mod (number of seed sets) */
        evec sets = level;
        evec cl = {0};
        for (int c = 0; c < P.sample_count && sets.n > 0; c++) {
            const entry *src = sets.v[c % sets.n];
            entry *e = entry_new(src->n_supp, 0);
            for (int t = 0; t < src->n_supp; t++) { e->arc[t] = src->arc[t]; e->f[t] = 1; }
            evec_push(&cl, e);
        }
        for (int64_t x = 0; x < sets.n; x++) free(sets.v[x]);
        free(sets.v);
        level = cl;
        P.frontier_cap = 0;     /* a candidate has one descendant at most: nothing to cut */
    }
    for (int64_t x = 0; x < level.n; x++) { level.v[x]->cand = (int32_t)x; level.v[x]->level = 0; }
    R->n_roots = (int)level.n;
    if (P.sample_count > 0) { R->n_cand_end = level.n; R->cand_end = calloc(level.n + 1, sizeof(int64_t)); }

    worker *wk = calloc(nthreads, sizeof(worker));
    for (int t = 0; t < nthreads; t++) {
        wk[t].EF = calloc(M + 1, sizeof(i128)); wk[t].EFs = calloc(M + 1, sizeof(i128));
        int maxnnz = G->col_ptr[A] + 16;
        wk[t].touched = malloc(sizeof(int) * maxnnz); wk[t].touched2 = malloc(sizeof(int) * maxnnz);
        wk[t].insupp = calloc(A + 1, 1);
        wk[t].cand_end = R->cand_end;
    }
    evec cands = {0};
    oracle_stats *st = &R->st;
    int64_t lrec_cap = 0;
    uint64_t shuf = P.shuffle_seed;

    /* O4 level loop */
    while (level.n > 0) {
        if (shuf) for (int64_t x = level.n - 1; x > 0; x--) {
            int64_t y = (int64_t)(rng_next(&shuf) % (uint64_t)(x + 1));
            entry *t = level.v[x]; level.v[x] = level.v[y]; level.v[y] = t;
        }
        st->levels++;
        int64_t N = level.n;
        int32_t *istar = malloc(sizeof(int32_t) * N);
        int32_t *nunb = malloc(sizeof(int32_t) * N);
        i128 *Estar = malloc(sizeof(i128) * N);
        /* classify: PROC0 + arbiter */
#pragma omp parallel for schedule(dynamic, 64) num_threads(nthreads)
        for (int64_t x = 0; x < N; x++) {
#ifdef _OPENMP
            worker *w = &wk[omp_get_thread_num()];
#else
            worker *w = &wk[0];
#endif
            int nt;
            extra_flux(G, level.v[x], w->EF, w->touched, &nt);
            int lowest = -1, cnt = 0;
            for (int t = 0; t < nt; t++) {
                int i = w->touched[t];
                if (w->EF[i] != 0) {
                    if (w->EF[i] > GUARD || w->EF[i] < -GUARD) { fprintf(stderr, "oracle: extra flux above guard\n"); abort(); }
                    if (lowest < 0 || i < lowest) lowest = i;
                }
            }
            /* count distinct unbalanced metabolites: scan all nodes (plain, M is small) */
            for (int i = 0; i < M; i++) if (w->EF[i] != 0) cnt++;
            istar[x] = lowest; nunb[x] = cnt; Estar[x] = lowest >= 0 ? w->EF[lowest] : 0;
            for (int t = 0; t < nt; t++) w->EF[w->touched[t]] = 0;
        }
        int64_t n_done = 0, n_active = 0;
        for (int64_t x = 0; x < N; x++) if (istar[x] < 0) n_done++; else n_active++;
        st->done += n_done;
        if (n_active > st->peak_frontier) st->peak_frontier = n_active;
        /* beam B: keep key < X where X is the (cap)-th smallest key, i.e. key <= T* with T* the largest
         * value such that #{key <= T*} <= cap */
        uint8_t *keep = malloc(N);
        for (int64_t x = 0; x < N; x++) keep[x] = istar[x] >= 0;
        if (P.frontier_cap > 0 && n_active > P.frontier_cap) {
            uint64_t *keys = malloc(sizeof(uint64_t) * N), *sorted = malloc(sizeof(uint64_t) * n_active);
            int64_t w = 0;
#pragma omp parallel for schedule(static) num_threads(nthreads)
            for (int64_t x = 0; x < N; x++) keys[x] = istar[x] >= 0 ? beam_key(level.v[x], nunb[x]) : 0;
            for (int64_t x = 0; x < N; x++) if (istar[x] >= 0) sorted[w++] = keys[x];
            qsort(sorted, n_active, sizeof(uint64_t), cmp_u64);
            uint64_t X = sorted[P.frontier_cap];
            for (int64_t x = 0; x < N; x++) if (istar[x] >= 0 && !(keys[x] < X)) { keep[x] = 0; st->truncated_beam++; }
            free(keys); free(sorted);
        }
        if (P.trace)
            for (int64_t x = 0; x < N; x++) {
                const entry *e = level.v[x];
                if (P.trace == 2 && istar[x] >= 0) continue;   /* 2: balanced entries only */
                trace_push(R, st->levels - 1); trace_push(R, e->n_supp); trace_push(R, e->n_vis); trace_push(R, nunb[x]);
                trace_push(R, istar[x]); trace_push(R, (int64_t)beam_key(e, nunb[x])); trace_push(R, keep[x] || istar[x] < 0);
                for (int k = 0; k < e->n_supp; k++) { trace_push(R, e->arc[k]); trace_push(R, e->f[k]); }
                for (int k = 0; k < e->n_vis; k++) { trace_push(R, e->vis[k].met); trace_push(R, e->vis[k].PI); trace_push(R, e->vis[k].PO); trace_push(R, e->vis[k].cnt); }
            }
        /* an expansion reads its parent, writes one 8-byte key per generated child and
         * writes the children that survive (balanced ones and those the beam keeps); roots are not written
         * by an expansion */
        if (st->levels > 1)
            for (int64_t x = 0; x < N; x++) if (istar[x] < 0 || keep[x]) st->algo_bytes += algo_entry_bytes(level.v[x]);
        /* expand the survivors */
        for (int t = 0; t < nthreads; t++) { wk[t].children.n = 0; memset(&wk[t].st, 0, sizeof(oracle_stats)); }
#pragma omp parallel for schedule(dynamic, 64) num_threads(nthreads)
        for (int64_t x = 0; x < N; x++) {
            if (!keep[x]) continue;
#ifdef _OPENMP
            worker *w = &wk[omp_get_thread_num()];
#else
            worker *w = &wk[0];
#endif
            expand(G, &P, level.v[x], istar[x], Estar[x], w);
        }
        evec next = {0};
        int64_t lvl_exp = 0, lvl_ch = 0;
        for (int t = 0; t < nthreads; t++) {
            oracle_stats *s = &wk[t].st;
            st->expanded += s->expanded; st->children += s->children; st->dead_end += s->dead_end;
            st->not_efm_maxloop += s->not_efm_maxloop; st->discarded_nonpos += s->discarded_nonpos;
            st->discarded_overflow += s->discarded_overflow; st->discarded_visited += s->discarded_visited;
            st->algo_bytes += s->algo_bytes;
            lvl_exp += s->expanded; lvl_ch += s->children;
            for (int64_t x = 0; x < wk[t].children.n; x++) evec_push(&next, wk[t].children.v[x]);
        }
        if (R->n_levels_rec == lrec_cap) {
            lrec_cap = lrec_cap ? lrec_cap * 2 : 64;
            R->lvl_active = realloc(R->lvl_active, sizeof(int64_t) * lrec_cap);
            R->lvl_done = realloc(R->lvl_done, sizeof(int64_t) * lrec_cap);
            R->lvl_expanded = realloc(R->lvl_expanded, sizeof(int64_t) * lrec_cap);
            R->lvl_children = realloc(R->lvl_children, sizeof(int64_t) * lrec_cap);
        }
        R->lvl_active[R->n_levels_rec] = n_active; R->lvl_done[R->n_levels_rec] = n_done;
        R->lvl_expanded[R->n_levels_rec] = lvl_exp; R->lvl_children[R->n_levels_rec] = lvl_ch;
        R->n_levels_rec++;
        for (int64_t x = 0; x < N; x++) {
            if (istar[x] < 0) {
                if (R->cand_end) R->cand_end[level.v[x]->cand] = END_DONE | ((int64_t)level.v[x]->level << 8);
                evec_push(&cands, level.v[x]);
            } else free(level.v[x]);
        }
        free(istar); free(nunb); free(Estar); free(keep); free(level.v);
        level = next;
    }
    free(level.v);

    /* O8 candidates -> output */
    /* (i) steady-state guard: S_int . f = 0 */
    for (int64_t x = 0; x < cands.n; x++) {
        int nt; extra_flux(G, cands.v[x], wk[0].EF, wk[0].touched, &nt);
        for (int t = 0; t < nt; t++) {
            if (wk[0].EF[wk[0].touched[t]] != 0) { fprintf(stderr, "oracle: unbalanced candidate\n"); abort(); }
        }
    }
    /* (ii) group by support; two different flux vectors on one support poison it (G18) */
    qsort(cands.v, cands.n, sizeof(entry *), cmp_cand);
    evec uniq = {0};
    for (int64_t x = 0; x < cands.n;) {
        int64_t y = x; int poisoned = 0;
        while (y < cands.n && same_support(cands.v[x], cands.v[y])) {
            if (cmp_cand(&cands.v[x], &cands.v[y]) != 0) poisoned = 1;
            if (cands.v[y]->level < cands.v[x]->level) cands.v[x]->level = cands.v[y]->level;   /* steps of the support: its quickest construction */
            y++;
        }
        st->unique_supports++;
        if (poisoned) st->poisoned++; else evec_push(&uniq, cands.v[x]);
        x = y;
    }
    /* (iii) support-minimality among the survivors (Def 3; G17) */
    int W = G->W;
    uint64_t *bits = calloc((size_t)(uniq.n + 1) * W, sizeof(uint64_t));
    for (int64_t x = 0; x < uniq.n; x++)
        for (int k = 0; k < uniq.v[x]->n_supp; k++) bits[x * W + uniq.v[x]->arc[k] / 64] |= 1ULL << (uniq.v[x]->arc[k] % 64);
    uint8_t *minimal = malloc(uniq.n + 1);
#pragma omp parallel for schedule(dynamic, 16) num_threads(nthreads)
    for (int64_t x = 0; x < uniq.n; x++) {
        if (P.exact) {   /* 8(f)-3: the rank test instead of the comparison with the other candidates */
            minimal[x] = (uint8_t)(support_rank(G, uniq.v[x]) == uniq.v[x]->n_supp - 1);
            continue;
        }
        int ok = 1;
        for (int64_t y = 0; y < uniq.n && ok; y++) {
            if (y == x) continue;
            int sub = 1, eq = 1;
            for (int w = 0; w < W; w++) {
                uint64_t bw = bits[y * W + w], bv = bits[x * W + w];
                if (bw & ~bv) { sub = 0; break; }
                if (bw != bv) eq = 0;
            }
            if (sub && !eq) ok = 0; /* supp(w) strictly inside supp(v) */
        }
        minimal[x] = (uint8_t)ok;
    }
    /* (iv) reaction space v_j = f_j+ - f_j-, (v) lexicographic order */
    int64_t n_out = 0;
    for (int64_t x = 0; x < uniq.n; x++) n_out += minimal[x];
    if (P.exact) st->non_elementary = uniq.n - n_out;
    /* rows carry their step count behind the n flux columns while they are sorted */
    int64_t *rows = calloc((size_t)(n_out + 1) * (n + 1), sizeof(int64_t));
    int64_t r = 0;
    for (int64_t x = 0; x < uniq.n; x++) {
        if (!minimal[x]) continue;
        for (int k = 0; k < uniq.v[x]->n_supp; k++) {
            int a = uniq.v[x]->arc[k];
            rows[r * (n + 1) + G->arc_rxn[a]] += (int64_t)G->arc_dir[a] * uniq.v[x]->f[k];
        }
        rows[r * (n + 1) + n] = uniq.v[x]->level;
        r++;
    }
    g_sort_n = n;   /* the comparison looks at the n flux columns only (they are distinct) */
    qsort(rows, n_out, sizeof(int64_t) * (n + 1), cmp_rows);
    R->flux = calloc((size_t)(n_out + 1) * n, sizeof(int64_t));
    R->steps = calloc((size_t)n_out + 1, sizeof(int64_t));
    for (int64_t x = 0; x < n_out; x++) {
        memcpy(R->flux + x * n, rows + x * (n + 1), sizeof(int64_t) * n);
        R->steps[x] = rows[x * (n + 1) + n];
    }
    free(rows);
    R->n_out = n_out; st->output = n_out;

    free(bits); free(minimal); free(uniq.v);
    for (int64_t x = 0; x < cands.n; x++) free(cands.v[x]);
    free(cands.v);
    for (int t = 0; t < nthreads; t++) { free(wk[t].EF); free(wk[t].EFs); free(wk[t].touched); free(wk[t].touched2); free(wk[t].insupp); free(wk[t].children.v); }
    free(wk);
    *out = R;
    return 0;
}

/* ------------------------------------------------------------------ accessors (ctypes) */
int64_t oracle_result_count(const oracle_result *R) { return R->n_out; }
void oracle_result_copy(const oracle_result *R, int64_t *dst) { memcpy(dst, R->flux, sizeof(int64_t) * R->n_out * R->n); }
void oracle_result_stats(const oracle_result *R, oracle_stats *st) { *st = R->st; }
void oracle_result_steps(const oracle_result *R, int64_t *dst) { memcpy(dst, R->steps, sizeof(int64_t) * R->n_out); }
int64_t oracle_result_cand_end(const oracle_result *R, int64_t *dst, int64_t cap) {
    for (int64_t x = 0; x < R->n_cand_end && x < cap; x++) dst[x] = R->cand_end[x];
    return R->n_cand_end;
}
int64_t oracle_result_levels(const oracle_result *R, int64_t *active, int64_t *done, int64_t *expanded, int64_t *children, int64_t cap) {
    int64_t k = R->n_levels_rec < cap ? R->n_levels_rec : cap;
    for (int64_t x = 0; x < k; x++) { active[x] = R->lvl_active[x]; done[x] = R->lvl_done[x]; expanded[x] = R->lvl_expanded[x]; children[x] = R->lvl_children[x]; }
    return R->n_levels_rec;
}
int32_t oracle_result_roots(const oracle_result *R) { return R->n_roots; }
void oracle_graph_info(const oracle_result *R, int32_t *M, int32_t *A, int32_t *W, int64_t *nnz, int64_t *dep_bits) {
    *M = R->G.M; *A = R->G.A; *W = R->G.W; *nnz = R->G.col_ptr[R->G.A]; *dep_bits = R->G.dep_off[R->G.M];
}
/* graph arrays, widened to int64 where needed, for the builder-parity test */
void oracle_graph_export(const oracle_result *R, int32_t *arc_rxn, int32_t *arc_dir, int32_t *twin,
                         int32_t *in_ptr, int32_t *in_arc, int64_t *in_c,
                         int32_t *out_ptr, int32_t *out_arc, int64_t *out_c,
                         int32_t *col_ptr, int32_t *col_met, int64_t *col_s,
                         int64_t *dep_off, uint8_t *dep) {
    const graph *G = &R->G;
    for (int a = 0; a < G->A; a++) { arc_rxn[a] = G->arc_rxn[a]; arc_dir[a] = G->arc_dir[a]; twin[a] = G->twin[a]; }
    for (int i = 0; i <= G->M; i++) { in_ptr[i] = G->in_ptr[i]; out_ptr[i] = G->out_ptr[i]; dep_off[i] = G->dep_off[i]; }
    for (int q = 0; q < G->in_ptr[G->M]; q++) { in_arc[q] = G->in_arc[q]; in_c[q] = G->in_c[q]; }
    for (int q = 0; q < G->out_ptr[G->M]; q++) { out_arc[q] = G->out_arc[q]; out_c[q] = G->out_c[q]; }
    for (int a = 0; a <= G->A; a++) col_ptr[a] = G->col_ptr[a];
    for (int q = 0; q < G->col_ptr[G->A]; q++) { col_met[q] = G->col_met[q]; col_s[q] = G->col_s[q]; }
    memcpy(dep, G->dep, G->dep_off[G->M]);
}
int64_t oracle_result_trace(const oracle_result *R, int64_t *dst, int64_t cap) {
    for (int64_t x = 0; x < R->trace_n && x < cap; x++) dst[x] = R->trace[x];
    return R->trace_n;
}
void oracle_result_free(oracle_result *R) {
    if (!R) return;
    if (R->have_graph) graph_free(&R->G);
    free(R->trace);
    free(R->steps); free(R->cand_end);
    free(R->flux); free(R->lvl_active); free(R->lvl_done); free(R->lvl_expanded); free(R->lvl_children);
    free(R);
}
/* the state hash / beam key of an explicitly given state, for the hash pins */
uint64_t oracle_state_hash(int32_t n_supp, const int32_t *arc, const int64_t *f, int32_t n_vis, const int32_t *vis4 /* met,PI,PO,cnt */) {
    entry *e = entry_new(n_supp, n_vis);
    for (int k = 0; k < n_supp; k++) { e->arc[k] = arc[k]; e->f[k] = f[k]; }
    for (int k = 0; k < n_vis; k++) { e->vis[k].met = vis4[4 * k]; e->vis[k].PI = vis4[4 * k + 1]; e->vis[k].PO = vis4[4 * k + 2]; e->vis[k].cnt = vis4[4 * k + 3]; }
    uint64_t h = state_hash(e);
    free(e);
    return h;
}
int32_t oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
/* the mixing primitive alone, for the SplitMix64 test-vector pin */
uint64_t oracle_mix64(uint64_t x) { return mix64(x); }
