"""Seeded synthetic metabolic networks shaped like the paper's workloads.

The paper evaluates on a CHO core model (12 x 18) and E. coli
iAF1260 (1668 x 2382).  Neither model is available offline, so the
five ``BASELINE.json`` configs are *synthetic stand-ins* with the same shapes;
no item of either model is reproduced.  Everything here is integer-only
(SplitMix64 + Python ints) so a given (config, seed) is bit-reproducible on any
machine.  This module contains input generation ONLY - no part of the traversal,
balancing, hashing or filtering arithmetic lives here.

Recipe:
  rows       : m_int internal + m_ext external metabolites, interleaved by a seeded shuffle
  exchanges  : n_exch reactions "1 external <-> 1 internal" (even = import, odd = export)
  routes     : planted unimolecular chains import -> ... -> export (guaranteed balanced routes)
  random     : reactions with 1..side_max substrates and products; first slot of each side
               walks a seeded permutation (every metabolite gets used), remaining slots are
               drawn with power-law weights rank^(-1/(gamma-1)), gamma = 2.2 (configs 3-5)
  hubs       : the n_hubs top-ranked metabolites are forced into hub_deg[0]..hub_deg[1] reactions
  links      : unimolecular reactions added until the internal graph is strongly connected
  reversible : exactly n_rev reactions, seeded sample
  coefficients: drawn from coef_dist (percent weights)
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

MASK64 = (1 << 64) - 1


class SplitMix64:
    """Counter-based 64-bit PRNG (Steele/Lea/Flood SplitMix64), integer-only."""

    def __init__(self, seed: int):
        self.s = seed & MASK64

    def next(self) -> int:
        self.s = (self.s + 0x9E3779B97F4A7C15) & MASK64
        z = self.s
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & MASK64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & MASK64
        return z ^ (z >> 31)

    def below(self, n: int) -> int:
        """Uniform integer in [0, n) by multiply-shift."""
        return (self.next() * n) >> 64

    def between(self, lo: int, hi: int) -> int:
        return lo + self.below(hi - lo + 1)

    def shuffle(self, xs: list) -> None:
        for i in range(len(xs) - 1, 0, -1):
            j = self.below(i + 1)
            xs[i], xs[j] = xs[j], xs[i]

    def sample(self, population: Sequence[int], k: int) -> List[int]:
        xs = list(population)
        k = min(k, len(xs))
        for i in range(k):
            j = i + self.below(len(xs) - i)
            xs[i], xs[j] = xs[j], xs[i]
        return xs[:k]

    def pick_cum(self, cum: Sequence[int]) -> int:
        """Index drawn with integer weights given as a cumulative list."""
        x = self.below(cum[-1])
        lo, hi = 0, len(cum) - 1
        while lo < hi:
            mid = (lo + hi) // 2
            if cum[mid] > x:
                hi = mid
            else:
                lo = mid + 1
        return lo


def _iroot6(x: int) -> int:
    """floor(x ** (1/6)) for a non-negative Python int."""
    lo, hi = 0, 1
    while hi ** 6 <= x:
        hi *= 2
    while lo + 1 < hi:
        mid = (lo + hi) // 2
        if mid ** 6 <= x:
            lo = mid
        else:
            hi = mid
    return lo


def _powerlaw_weight(rank: int) -> int:
    """Integer weight ~ 2^24 * rank^(-1/(gamma-1)) with gamma = 2.2, i.e. rank^(-5/6)."""
    return max(1, _iroot6((1 << 144) // (rank ** 5)))


@dataclass
class Spec:
    name: str
    m_int: int
    m_ext: int
    n_rxn: int
    n_rev: int
    side_max: int
    coef_dist: Tuple[Tuple[int, int], ...]
    power_law: bool
    n_hubs: int
    hub_deg: Tuple[int, int]
    n_exch: int
    n_routes: int
    route_len: Tuple[int, int]  # number of internal chain reactions per planted route
    strongly_connected: bool
    # traversal parameters (identical for oracle and GPU; printed with every result)
    max_support: int  # D, 0 = number of arcs
    max_loop: int
    dep_depth: int
    max_visited: int  # V, 0 = 2 * D
    frontier_cap: int  # 0 = none
    seed_mode: str  # "default" | "targets"
    n_targets: int = 0


COEF_12 = ((1, 80), (2, 20))
COEF_123 = ((1, 80), (2, 15), (3, 5))

CONFIGS: Dict[str, Spec] = {
    # BASELINE.json configs[0]
    "toy": Spec("toy", 6, 3, 10, 3, 2, COEF_12, False, 0, (0, 0), 4, 2, (1, 2), False,
                0, 8, 4, 0, 0, "default"),
    # BASELINE.json configs[1]
    "small": Spec("small", 20, 6, 32, 6, 3, COEF_123, False, 0, (0, 0), 6, 4, (2, 3), False,
                  0, 8, 4, 0, 0, "default"),
    # BASELINE.json configs[2]
    "core": Spec("core", 72, 20, 95, 24, 3, COEF_123, True, 5, (25, 40), 20, 4, (3, 5), True,
                 24, 8, 4, 48, 1 << 20, "default"),
    # BASELINE.json configs[3]
    "mid": Spec("mid", 250, 40, 350, 88, 3, COEF_123, True, 10, (30, 60), 40, 8, (4, 8), True,
                40, 8, 4, 80, 1 << 24, "default"),
    # BASELINE.json configs[4]; frontier_cap is the nominal bound of BASELINE.json (2^28);
    # bench/tests pass the cap they actually run with.
    "genome": Spec("genome", 1000, 150, 2000, 600, 3, COEF_123, True, 20, (100, 300), 150, 16,
                   (6, 28), True, 60, 8, 4, 120, 1 << 28, "targets", 8),
}


def config_names() -> List[str]:
    return list(CONFIGS.keys())


@dataclass
class Network:
    name: str
    seed: int
    S: np.ndarray  # int32 [m, n], C-contiguous; S[i, j] > 0 produced, < 0 consumed
    reversible: np.ndarray  # uint8 [n]
    internal: np.ndarray  # uint8 [m]
    params: Dict[str, int]
    # explicit seed sets as arc codes 2*j + (dir < 0), or None for the default (boundary arcs)
    seed_sets: Optional[List[List[int]]] = None
    info: Dict[str, object] = field(default_factory=dict)

    @property
    def m(self) -> int:
        return int(self.S.shape[0])

    @property
    def n(self) -> int:
        return int(self.S.shape[1])

    @property
    def n_arcs(self) -> int:
        return self.n + int(self.reversible.sum())


def _draw_coef(rng: SplitMix64, dist) -> int:
    total = sum(w for _, w in dist)
    x = rng.below(total)
    for c, w in dist:
        if x < w:
            return c
        x -= w
    return dist[-1][0]


def _scc(n: int, adj: List[List[int]]) -> List[int]:
    """Iterative Tarjan; returns component id per node."""
    index = [-1] * n
    low = [0] * n
    on = [False] * n
    comp = [-1] * n
    stack: List[int] = []
    idx = 0
    ncomp = 0
    for root in range(n):
        if index[root] != -1:
            continue
        work = [(root, 0)]
        while work:
            v, pi = work[-1]
            if pi == 0:
                index[v] = low[v] = idx
                idx += 1
                stack.append(v)
                on[v] = True
            recurse = False
            while pi < len(adj[v]):
                w = adj[v][pi]
                pi += 1
                if index[w] == -1:
                    work[-1] = (v, pi)
                    work.append((w, 0))
                    recurse = True
                    break
                if on[w]:
                    low[v] = min(low[v], index[w])
            if recurse:
                continue
            work.pop()
            if work:
                u = work[-1][0]
                low[u] = min(low[u], low[v])
            if low[v] == index[v]:
                while True:
                    w = stack.pop()
                    on[w] = False
                    comp[w] = ncomp
                    if w == v:
                        break
                ncomp += 1
    return comp


class _Rxn:
    __slots__ = ("subs", "prods", "kind")

    def __init__(self, subs, prods, kind):
        self.subs = subs  # list of (metabolite label, coef); label = ("i", k) or ("e", k)
        self.prods = prods
        self.kind = kind

    def has(self, lab) -> bool:
        return any(m == lab for m, _ in self.subs) or any(m == lab for m, _ in self.prods)


def _internal_graph(m_int: int, rxns: List[_Rxn], rev: Sequence[bool]) -> List[List[int]]:
    adj: List[List[int]] = [[] for _ in range(m_int)]
    for r, is_rev in zip(rxns, rev):
        si = [m[1] for m, _ in r.subs if m[0] == "i"]
        pi = [m[1] for m, _ in r.prods if m[0] == "i"]
        for u in si:
            for v in pi:
                adj[u].append(v)
                if is_rev:
                    adj[v].append(u)
    return adj


def make_network(name: str, seed: int = 0) -> Network:
    """Build the synthetic network of one BASELINE.json config."""
    sp = CONFIGS[name]
    tag = sum((ord(ch) << (8 * i)) for i, ch in enumerate(name[:8]))
    rng = SplitMix64((seed * 0x9E3779B97F4A7C15 + tag) & MASK64)
    M, X, n = sp.m_int, sp.m_ext, sp.n_rxn

    # popularity ranking over a seeded permutation of the internal metabolites
    order = list(range(M))
    rng.shuffle(order)
    hubs = order[: sp.n_hubs]
    hubset = set(hubs)
    nonhub = [k for k in order if k not in hubset]
    weights = []
    for r, _k in enumerate(nonhub):
        weights.append(_powerlaw_weight(r + 1) if sp.power_law else 1)
    # external metabolites share ~10 % of the draw mass in random reactions
    w_int_total = sum(weights)
    w_ext_each = max(1, w_int_total // (9 * max(1, X)))
    pool = [("i", k) for k in nonhub] + [("e", k) for k in range(X)]
    cum = []
    acc = 0
    for w in weights + [w_ext_each] * X:
        acc += w
        cum.append(acc)

    def coef():
        return _draw_coef(rng, sp.coef_dist)

    # exchanges: external e (round-robin) <-> a distinct internal metabolite
    exch_mets = rng.sample(nonhub, sp.n_exch)
    exchanges: List[_Rxn] = []
    for e in range(sp.n_exch):
        ext = ("e", e % X)
        met = ("i", exch_mets[e % len(exch_mets)])
        if e % 2 == 0:
            exchanges.append(_Rxn([(ext, 1)], [(met, 1)], "import"))
        else:
            exchanges.append(_Rxn([(met, 1)], [(ext, 1)], "export"))
    imports = [e for e in range(sp.n_exch) if e % 2 == 0]
    exports = [e for e in range(sp.n_exch) if e % 2 == 1]

    # planted routes: import exchange -> unimolecular chain -> export exchange
    planted: List[_Rxn] = []
    for r in range(sp.n_routes):
        if sp.seed_mode == "targets" and sp.n_targets:
            t = r % sp.n_targets
            if t % 2 == 0:
                e_in, e_out = t, exports[rng.below(len(exports))]
            else:
                e_in, e_out = imports[rng.below(len(imports))], t
        else:
            e_in = imports[r % len(imports)]
            e_out = exports[r % len(exports)]
        a = exchanges[e_in].prods[0][0][1]
        b = exchanges[e_out].subs[0][0][1]
        L = rng.between(sp.route_len[0], sp.route_len[1])
        mids = rng.sample([k for k in nonhub if k != a and k != b], L - 1)
        chain = [a] + mids + [b]
        for u, v in zip(chain[:-1], chain[1:]):
            if u == v:
                continue
            subs = [(("i", u), coef())]
            prods = [(("i", v), coef())]
            if X and rng.below(4) == 0:  # an external co-substrate or co-product
                ext = ("e", rng.below(X))
                (subs if rng.below(2) == 0 else prods).append((ext, coef()))
            planted.append(_Rxn(subs, prods, "planted"))

    def side_size() -> int:
        # 1..side_max, larger sides favoured (20/40/40 %) so that columns carry ~3.5 nonzeros
        if sp.side_max == 2:
            return 1 if rng.below(5) < 2 else 2
        x = rng.below(5)
        return 1 if x == 0 else (2 if x < 3 else 3)

    def random_reaction(t: int, back: List[int]) -> _Rxn:
        # slot 0 of each side follows a backbone chain back[t] -> back[t+1] through every
        # non-hub metabolite; the remaining slots are drawn from the weighted pool
        first_sub = ("i", back[t % len(back)])
        first_prod = ("i", back[(t + 1) % len(back)])
        ns, npd = side_size(), side_size()
        subs_l = [first_sub]
        prods_l = [first_prod]
        tries = 0
        while (len(subs_l) < ns or len(prods_l) < npd) and tries < 64:
            tries += 1
            cand = pool[rng.pick_cum(cum)]
            if cand in subs_l or cand in prods_l:
                continue
            (subs_l if len(subs_l) < ns else prods_l).append(cand)
        return _Rxn([(m, coef()) for m in subs_l], [(m, coef()) for m in prods_l], "random")

    def force_hubs(rxns: List[_Rxn]) -> None:
        hub_labs = {("i", h) for h in hubs}
        for h in hubs:
            lab = ("i", h)
            target = min(rng.between(sp.hub_deg[0], sp.hub_deg[1]), len(rxns))
            deg = 0
            cand = list(range(len(rxns)))
            rng.shuffle(cand)
            for ridx in cand:
                if deg >= target:
                    break
                r = rxns[ridx]
                if r.has(lab):
                    continue
                side = r.subs if rng.below(2) == 0 else r.prods
                if len(side) < sp.side_max:
                    side.append((lab, coef()))
                    deg += 1
                    continue
                # never the backbone slot 0, never another hub
                slots = [k for k in range(1, len(side)) if side[k][0] not in hub_labs]
                if slots:
                    side[slots[rng.below(len(slots))]] = (lab, coef())
                    deg += 1

    n_fixed = len(exchanges) + len(planted)
    if n_fixed >= n:
        raise ValueError(f"{name}: exchanges + planted routes already use {n_fixed} of {n} reactions")
    used = set(exch_mets)
    for r in planted:
        for lab, _c in r.subs + r.prods:
            if lab[0] == "i":
                used.add(lab[1])
    # reversibility is drawn over generation indices up front (the total is always n)
    rev_gen = [False] * n
    for j in rng.sample(range(n), sp.n_rev):
        rev_gen[j] = True
    budget = max(2, M // 16) if sp.strongly_connected else 0
    for _attempt in range(64):
        R = n - n_fixed - budget
        if R < 0:
            raise ValueError(f"{name}: cannot fit connectivity links into {n} reactions")
        fresh = [k for k in nonhub if k not in used]
        stale = [k for k in nonhub if k in used]
        rng.shuffle(fresh)
        rng.shuffle(stale)
        back = fresh + stale
        randoms = [random_reaction(t, back) for t in range(R)]
        force_hubs(randoms)
        rxns = exchanges + planted + randoms
        links: List[_Rxn] = []
        if sp.strongly_connected:
            # link sink components to source components of the condensation until one component is left
            for _round in range(64):
                adj = _internal_graph(M, rxns + links, rev_gen[: len(rxns)] + [False] * len(links))
                comp = _scc(M, adj)
                ncomp = max(comp) + 1
                if ncomp == 1:
                    break
                rep = [-1] * ncomp
                indeg = [0] * ncomp
                outdeg = [0] * ncomp
                for u in range(M):
                    if rep[comp[u]] == -1:
                        rep[comp[u]] = u
                    for v in adj[u]:
                        if comp[u] != comp[v]:
                            outdeg[comp[u]] += 1
                            indeg[comp[v]] += 1
                sources = [c for c in range(ncomp) if indeg[c] == 0]
                sinks = [c for c in range(ncomp) if outdeg[c] == 0]
                for t in range(max(len(sources), len(sinks))):
                    u = rep[sinks[t % len(sinks)]]
                    v = rep[sources[(t + 1) % len(sources)]]
                    if u != v:
                        links.append(_Rxn([(("i", u), coef())], [(("i", v), coef())], "link"))
            if len(links) > budget:
                budget = len(links)
                continue
        # unused link budget becomes extra random reactions (cannot break connectivity)
        extra = [random_reaction(R + t, back) for t in range(budget - len(links))]
        gen_order = exchanges + planted + randoms + links + extra
        break
    else:
        raise ValueError(f"{name}: connectivity loop did not converge")

    assert len(gen_order) == n
    rev_of = {id(r): rev_gen[g] for g, r in enumerate(gen_order)}
    others = gen_order[len(exchanges):]
    # final reaction order: exchanges keep their relative order at seeded positions
    exch_pos = sorted(rng.sample(range(n), len(exchanges)))
    rng.shuffle(others)
    slots: List[Optional[_Rxn]] = [None] * n
    for p, r in zip(exch_pos, exchanges):
        slots[p] = r
    it = iter(others)
    for p in range(n):
        if slots[p] is None:
            slots[p] = next(it)
    rxn_list: List[_Rxn] = [r for r in slots if r is not None]

    # rows: internal/external interleaved by a seeded shuffle; internal k -> k-th internal row
    row_kind = [1] * M + [0] * X
    rng.shuffle(row_kind)
    int_rows = [i for i, k in enumerate(row_kind) if k == 1]
    ext_rows = [i for i, k in enumerate(row_kind) if k == 0]

    def row_of(lab) -> int:
        return int_rows[lab[1]] if lab[0] == "i" else ext_rows[lab[1]]

    S = np.zeros((M + X, n), dtype=np.int32)
    for j, r in enumerate(rxn_list):
        for lab, c in r.subs:
            S[row_of(lab), j] -= c
        for lab, c in r.prods:
            S[row_of(lab), j] += c
    reversible = np.array([1 if rev_of[id(r)] else 0 for r in rxn_list], dtype=np.uint8)
    internal = np.array(row_kind, dtype=np.uint8)

    seed_sets: Optional[List[List[int]]] = None
    if sp.seed_mode == "targets":
        seed_sets = []
        for p in exch_pos[: sp.n_targets]:
            seed_sets.append([2 * p])
            if reversible[p]:
                seed_sets.append([2 * p + 1])

    n_arcs = n + int(reversible.sum())
    D = sp.max_support if sp.max_support else n_arcs
    params = dict(
        max_support=D,
        max_loop=sp.max_loop,
        dep_depth=sp.dep_depth,
        max_visited=sp.max_visited if sp.max_visited else 2 * D,
        frontier_cap=sp.frontier_cap,
    )
    kinds: Dict[str, int] = {}
    for r in rxn_list:
        kinds[r.kind] = kinds.get(r.kind, 0) + 1
    info = dict(kinds=kinds, exchange_positions=exch_pos, hubs=[int_rows[h] for h in hubs],
                nnz_per_column=float((S != 0).sum()) / n)
    return Network(name, seed, np.ascontiguousarray(S), reversible, internal, params, seed_sets, info)


def hand_network(reactions: Sequence[Tuple[Dict[str, int], Dict[str, int], bool]],
                 internal_names: Sequence[str], name: str = "hand",
                 **params: int) -> Network:
    """Network from explicit reactions ``(substrates, products, reversible)``.

    Metabolite names not listed in ``internal_names`` become external rows (appended after
    the internal ones).  Used by the pin tests."""
    names = list(internal_names)
    ext: List[str] = []
    for subs, prods, _ in reactions:
        for k in list(subs) + list(prods):
            if k not in names and k not in ext:
                ext.append(k)
    rows = names + ext
    S = np.zeros((len(rows), len(reactions)), dtype=np.int32)
    rev = np.zeros(len(reactions), dtype=np.uint8)
    for j, (subs, prods, r) in enumerate(reactions):
        for k, c in subs.items():
            S[rows.index(k), j] -= c
        for k, c in prods.items():
            S[rows.index(k), j] += c
        rev[j] = 1 if r else 0
    internal = np.array([1] * len(names) + [0] * len(ext), dtype=np.uint8)
    A = len(reactions) + int(rev.sum())
    D = params.get("max_support", 0) or A
    p = dict(max_support=D, max_loop=params.get("max_loop", 8), dep_depth=params.get("dep_depth", 4),
             max_visited=params.get("max_visited", 0) or 2 * D, frontier_cap=params.get("frontier_cap", 0))
    return Network(name, 0, S, rev, internal, p, None, {})


def wide_fan_network(n_p: int = 300, n_q: int = 200, **params) -> Network:
    """r0 -> P_0 .. P_{n_p-1} and r1 -> Q_0 .. Q_{n_q-1}, every product with two consumers: a pathway grown from r0 has
    n_p - k unbalanced metabolites after k steps (with n_p = 300: more than the 255 the top byte of a beam key can hold), one
    grown from r1 has n_q - k, and both families double their number of entries with every level."""
    mets = [f"P{i}" for i in range(n_p)] + [f"Q{i}" for i in range(n_q)]
    rx = [({}, {f"P{i}": 1 for i in range(n_p)}, False), ({}, {f"Q{i}": 1 for i in range(n_q)}, False)]
    for m in mets:
        rx += [({m: 1}, {}, False), ({m: 1}, {}, False)]
    return hand_network(rx, mets, **params)


def chain_pair_network(len_a: int, len_b: int, **params) -> Network:
    """Two disjoint linear chains a0: -> A_0, a_i: A_{i-1} -> A_i, a_len: A_{len-1} -> (and the same with B); every tenth step
    produces two molecules so that the fluxes are not all 1.  Each chain is one EFM with len + 1 reactions; a pathway seeded on
    both a0 and b0 balances to their sum (len_a + len_b + 2 reactions), which is not elementary."""
    rx, mets = [], []
    for tag, ln in (("A", len_a), ("B", len_b)):
        names = [f"{tag}{i}" for i in range(ln)]
        mets += names
        rx.append(({}, {names[0]: 1}, False))
        for i in range(1, ln):
            rx.append(({names[i - 1]: 1}, {names[i]: 2 if i % 10 == 0 else 1}, False))
        rx.append(({names[-1]: 1}, {}, False))
    return hand_network(rx, mets, **params)


def unimolecular_network(seed: int, m_int: int, n_rxn: int, n_rev: int = 0) -> Network:
    """Unit-coefficient network with at most one internal substrate and one internal product per
    reaction (sources, sinks and internal A->B links).  On such networks the EFM set is exactly
    {simple source->sink paths} U {simple directed cycles} (SURVEY.md 8(c) pin P7)."""
    rng = SplitMix64((seed * 0x9E3779B97F4A7C15 + 0x756E696D6F6C) & MASK64)
    S = np.zeros((m_int, n_rxn), dtype=np.int32)
    seen = set()
    j = 0
    guard = 0
    while j < n_rxn and guard < 100000:
        guard += 1
        kind = rng.below(6)
        u = rng.below(m_int)
        v = rng.below(m_int)
        if kind == 0:
            key = ("src", v)
        elif kind == 1:
            key = ("snk", u)
        else:
            if u == v:
                continue
            key = ("lnk", u, v)
        if key in seen:
            continue
        seen.add(key)
        if key[0] == "src":
            S[v, j] = 1
        elif key[0] == "snk":
            S[u, j] = -1
        else:
            S[u, j] = -1
            S[v, j] = 1
        j += 1
    S = np.ascontiguousarray(S[:, :j])
    rev = np.zeros(j, dtype=np.uint8)
    for r in rng.sample(range(j), min(n_rev, j)):
        rev[r] = 1
    A = j + int(rev.sum())
    p = dict(max_support=A, max_loop=8, dep_depth=4, max_visited=2 * A, frontier_cap=0)
    return Network(f"unimolecular-{seed}", seed, S, rev, np.ones(m_int, dtype=np.uint8), p, None, {})


def random_seed_sets(net: Network, count: int, size: int, seed: int = 0) -> List[List[int]]:
    """``count`` seeded random seed sets of ``size`` distinct arcs each (arc codes 2*j + (dir < 0)), never both
    directions of one reaction.  Multi-arc seed sets reach one support along several routes, which is what exercises
    the poison rule and the minimality filter."""
    rng = SplitMix64((seed * 0x9E3779B97F4A7C15 + 0x73656564) & MASK64)
    codes = []
    for j in range(net.n):
        codes.append(2 * j)
        if net.reversible[j]:
            codes.append(2 * j + 1)
    out: List[List[int]] = []
    while len(out) < count:
        pick = rng.sample(codes, size)
        if len({c // 2 for c in pick}) == size:
            out.append(sorted(pick))
    return out


def mirrored(net: Network) -> Network:
    """The same network with every reaction reversed (S -> -S); reversibility, masks, parameters and seed sets kept."""
    return Network(net.name + "-mirrored", net.seed, np.ascontiguousarray(-net.S), net.reversible.copy(),
                   net.internal.copy(), dict(net.params), None if net.seed_sets is None else [list(s) for s in net.seed_sets],
                   dict(net.info))


def with_dead_ends(net: Network, count: int, seed: int = 0) -> Network:
    """``net`` plus ``count`` dead-end branches: an internal metabolite X feeds a chain X -> D1 -> D2 whose last metabolite
    nothing consumes (every second branch has a reversible first step).  No steady state can use these reactions; the
    compression pre-pass removes them by cascade, the traversal without it wastes expansions on them."""
    rng = SplitMix64((seed * 0x9E3779B97F4A7C15 + 0x64656164) & MASK64)
    m, n = net.S.shape
    internal_rows = [i for i in range(m) if net.internal[i]]
    S = np.zeros((m + 2 * count, n + 2 * count), dtype=np.int32)
    S[:m, :n] = net.S
    rev = np.concatenate([net.reversible, np.zeros(2 * count, dtype=np.uint8)])
    internal = np.concatenate([net.internal, np.ones(2 * count, dtype=np.uint8)])
    for b in range(count):
        x = internal_rows[rng.below(len(internal_rows))]
        d1, d2 = m + 2 * b, m + 2 * b + 1
        j1, j2 = n + 2 * b, n + 2 * b + 1
        S[x, j1] = -1; S[d1, j1] = 1 + b % 2
        S[d1, j2] = -1; S[d2, j2] = 1
        rev[j1] = b % 2
    A = int(S.shape[1] + rev.sum())
    p = dict(net.params)
    if net.params.get("max_support", 0) >= net.n_arcs:
        p["max_support"] = A
        p["max_visited"] = 2 * A
    return Network(net.name + f"-deadends{count}", net.seed, S, rev, internal, p,
                   None if net.seed_sets is None else [list(s) for s in net.seed_sets], dict(net.info))
