"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these compares the oracle with itself: expected values are hand-derived fixtures
(tests/golden/hand_pins.json), closed forms, textbook enumerations written here independently,
brute-force subset enumeration, published SplitMix64 test vectors, or invariants.
"""
import json
import os
from fractions import Fraction
from math import gcd

import numpy as np
import pytest

from netgen import (SplitMix64, chain_pair_network, hand_network, make_network, mirrored, random_seed_sets, unimolecular_network,
                    wide_fan_network)

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "hand_pins.json")


def _cases():
    with open(GOLDEN) as fh:
        return json.load(fh)["cases"]


def _norm_trace_level(states):
    return sorted((tuple(st["f"]), tuple(sorted(tuple(v) for v in st["vis"]))) for st in states)


@pytest.mark.parametrize("case", _cases(), ids=lambda c: c["name"])
def test_hand_pins(oracle_mod, case):
    rx = [(s, p, r) for s, p, r in case["reactions"]]
    net = hand_network(rx, case["internal"], **case.get("params", {}))
    res = oracle_mod.enumerate_pathways(net.S, net.reversible, net.internal, net.params, case["seeds"],
                                        trace="trace" in case)
    assert res.flux.tolist() == case["flux"]
    for k in ("expanded", "levels", "discarded_nonpos"):
        if k in case:
            assert res.stats[k] == case[k], k
    for k, v in case.get("stats", {}).items():
        assert res.stats[k] == v, (k, res.stats[k], v)
    if "trace" in case:
        A = net.n_arcs
        assert len(res.trace) == len(case["trace"])
        for lvl, (got, want) in enumerate(zip(res.trace, case["trace"])):
            got_n = sorted((tuple(e["flux"].get(a, 0) for a in range(A)),
                            tuple(sorted((m,) + v for m, v in e["visited"].items()))) for e in got)
            assert got_n == _norm_trace_level(want), f"level {lvl}"


def test_linear_chain_closed_form(oracle_mod):
    """P6 in general: ->A0, c0 A0 -> p0 A1, ..., A_k ->  has the single EFM given by ratio products."""
    rng = SplitMix64(7)
    for _trial in range(40):
        k = rng.between(1, 6)
        cons = [rng.between(1, 5) for _ in range(k)]
        prod = [rng.between(1, 5) for _ in range(k)]
        names = [f"A{t}" for t in range(k + 1)]
        rx = [({}, {names[0]: 1}, False)]
        for t in range(k):
            rx.append(({names[t]: cons[t]}, {names[t + 1]: prod[t]}, False))
        rx.append(({names[k]: 1}, {}, False))
        net = hand_network(rx, names)
        # closed form with rationals: v0 = 1; flux of chain reaction t = (amount of A_t) / cons[t]
        v = [Fraction(1)]
        amount = Fraction(1)
        for t in range(k):
            v.append(amount / cons[t])
            amount = v[-1] * prod[t]
        v.append(amount)
        den = 1
        for x in v:
            den = den * x.denominator // gcd(den, x.denominator)
        iv = [int(x * den) for x in v]
        g = 0
        for x in iv:
            g = gcd(g, x)
        expect = [x // g for x in iv]
        res = oracle_mod.enumerate_pathways(net.S, net.reversible, net.internal, net.params, [[0]])
        assert res.flux.tolist() == [expect]


def _paths_and_cycles(S, rev):
    """Textbook enumeration on a unimolecular unit network: simple source->sink paths and simple directed
    cycles over arcs (a reversible reaction contributes two arcs that exclude each other)."""
    m, n = S.shape
    arcs = []  # (rxn, dir, tail or None, head or None)
    for j in range(n):
        col = S[:, j]
        tail = [i for i in range(m) if col[i] < 0]
        head = [i for i in range(m) if col[i] > 0]
        t = tail[0] if tail else None
        h = head[0] if head else None
        arcs.append((j, +1, t, h))
        if rev[j]:
            arcs.append((j, -1, h, t))
    out = set()

    def emit(used):
        v = [0] * n
        for a in used:
            v[arcs[a][0]] += arcs[a][1]
        out.add(tuple(v))

    by_tail = {}
    for a, (_j, _d, t, _h) in enumerate(arcs):
        by_tail.setdefault(t, []).append(a)

    def rxns(used):
        return {arcs[a][0] for a in used}

    # source -> sink simple paths
    def dfs(node, used, seen):
        for a in by_tail.get(node, []):
            j, _d, _t, h = arcs[a]
            if j in rxns(used):
                continue
            if h is None:
                emit(used + [a])
            elif h not in seen:
                dfs(h, used + [a], seen | {h})

    for a in by_tail.get(None, []):
        h = arcs[a][3]
        if h is None:
            continue
        dfs(h, [a], {h})
    # simple directed cycles (rooted at their lowest node)
    def cyc(start, node, used, seen):
        for a in by_tail.get(node, []):
            j, _d, _t, h = arcs[a]
            if h is None or j in rxns(used):
                continue
            if h == start:
                emit(used + [a])
            elif h not in seen and h > start:
                cyc(start, h, used + [a], seen | {h})

    for s in range(m):
        cyc(s, s, [], {s})
    return out


def test_unimolecular_equals_paths_and_cycles(oracle_mod):
    """P7 (Lemma 2 type I, Theorem 1): with every arc seeded the output is
    exactly {simple source->sink paths} U {simple directed cycles}."""
    total = 0
    for seed in range(24):
        net = unimolecular_network(seed, m_int=4 + seed % 4, n_rxn=7 + seed % 6, n_rev=seed % 3)
        seeds = oracle_mod.all_arc_seed_sets(net.reversible)
        res = oracle_mod.enumerate_pathways(net.S, net.reversible, net.internal, net.params, seeds)
        got = set(map(tuple, res.flux.tolist()))
        expect = _paths_and_cycles(net.S, net.reversible)
        assert got == expect, f"seed {seed}"
        total += len(expect)
    assert total > 50


def test_toy_against_brute_force(oracle_mod, capsys):
    """P9: recall/precision of the (approximate) method against Definition 3 written out."""
    from oracle.brute_force import brute_force_efms
    net = make_network("toy", 0)
    truth = brute_force_efms(net.S, net.reversible, net.internal)
    assert len(truth) >= 2  # the planted routes
    for label, seeds in (("boundary", None), ("all-arcs", oracle_mod.all_arc_seed_sets(net.reversible))):
        res = oracle_mod.enumerate_pathways(net.S, net.reversible, net.internal, net.params, seeds)
        got = set(map(tuple, res.flux.tolist()))
        recall = len(got & truth) / len(truth)
        precision = len(got & truth) / max(1, len(got))
        with capsys.disabled():
            print(f"\n[toy/{label}] EFMs {len(truth)}, found {len(got)}, recall {recall:.2f}, precision {precision:.2f}")
        assert recall >= 0.5 and precision >= 0.5
    # small brute-forceable random networks: every balanced output must be a true EFM or be reported
    rng = SplitMix64(3)
    hits = tot = 0
    for t in range(12):
        net = unimolecular_network(100 + t, 4, 8, 1)
        # make it non-unimolecular: add a hyperarc reaction A+B -> C
        S = np.concatenate([net.S, np.zeros((net.S.shape[0], 1), np.int32)], axis=1)
        a, b, c = rng.sample(range(4), 3)
        S[a, -1], S[b, -1], S[c, -1] = -1, -rng.between(1, 2), rng.between(1, 2)
        rev = np.concatenate([net.reversible, [0]]).astype(np.uint8)
        truth = brute_force_efms(S, rev, net.internal)
        params = dict(max_support=0, max_loop=8, dep_depth=4, max_visited=0, frontier_cap=0)
        res = oracle_mod.enumerate_pathways(S, rev, net.internal, params, oracle_mod.all_arc_seed_sets(rev))
        got = set(map(tuple, res.flux.tolist()))
        hits += len(got & truth)
        tot += len(truth)
    assert tot > 0 and hits / tot >= 0.6


def test_invariants_and_precision(oracle_mod, capsys):
    """P8: Def 2 / Def 3 invariants hold on every output; precision by exact rank test is reported."""
    from oracle.check import check_outputs
    for name, over in (("toy", {}), ("small", {}), ("core", dict(frontier_cap=2048)),
                       ("mid", dict(frontier_cap=512)), ("genome", dict(frontier_cap=256))):
        net = make_network(name, 0)
        res = oracle_mod.enumerate_network(net, threads=2, self_check=False, **over)
        rep = check_outputs(net.S, net.reversible, net.internal, res.flux)
        with capsys.disabled():
            print(f"\n[{name}] outputs {len(res.flux)}, precision {rep['precision']:.3f}, stats {res.stats}")
        assert res.stats["output"] == len(res.flux)
        assert res.stats["unique_supports"] >= res.stats["output"] + res.stats["poisoned"]
        assert res.stats["children"] + res.n_roots == res.stats["done"] + res.stats["expanded"] + res.stats["truncated_beam"]


def test_order_independence(oracle_mod):
    """P10: shuffling every level and changing the thread count changes nothing, beam active."""
    for name, cap in (("small", 300), ("core", 1024), ("genome", 128)):
        net = make_network(name, 0)
        base = oracle_mod.enumerate_network(net, threads=1, self_check=False, frontier_cap=cap)
        assert base.stats["truncated_beam"] > 0
        for threads, shuf in ((1, 12345), (3, 0), (4, 999)):
            other = oracle_mod.enumerate_network(net, threads=threads, shuffle_seed=shuf, self_check=False,
                                                 frontier_cap=cap)
            assert other.stats == base.stats
            assert np.array_equal(other.flux, base.flux)
            assert all(np.array_equal(other.levels[k], base.levels[k]) for k in base.levels)


def test_beam_is_inactive_above_peak(oracle_mod):
    """A cap at or above the peak frontier must reproduce the uncapped run exactly."""
    net = make_network("small", 0)
    free = oracle_mod.enumerate_network(net, self_check=False)
    peak = free.stats["peak_frontier"]
    capped = oracle_mod.enumerate_network(net, self_check=False, frontier_cap=peak)
    assert capped.stats == free.stats and np.array_equal(capped.flux, free.flux)
    tight = oracle_mod.enumerate_network(net, self_check=False, frontier_cap=peak - 1)
    assert tight.stats["truncated_beam"] > 0
    assert all(a <= peak for a in tight.levels["expanded"])
    assert all(e <= peak - 1 for e in tight.levels["expanded"])


def test_mix64_matches_published_splitmix64_vectors(oracle_mod):
    """SplitMix64 (Steele, Lea, Flood 2014) seeded with 0 emits 0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4,
    0x06C45D188009454F; output t is the finaliser applied to t * 0x9E3779B97F4A7C15."""
    gamma = 0x9E3779B97F4A7C15
    expect = [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]
    for t, e in enumerate(expect, start=1):
        assert oracle_mod.mix64((t * gamma) & ((1 << 64) - 1)) == e


def test_state_hash_structure(oracle_mod):
    """h is a function of the complete state and of nothing else (beam B): order-free, field-sensitive,
    and composed as mix(sum of element terms) - checked through the exported primitive."""
    h = oracle_mod.state_hash
    base = h([3, 9, 4], [2, 5, 1], [(1, 3, 9, 0), (7, 4, 9, 2)])
    assert base == h([4, 3, 9], [1, 2, 5], [(7, 4, 9, 2), (1, 3, 9, 0)])
    variants = [
        h([3, 9, 5], [2, 5, 1], [(1, 3, 9, 0), (7, 4, 9, 2)]),
        h([3, 9, 4], [2, 5, 2], [(1, 3, 9, 0), (7, 4, 9, 2)]),
        h([3, 9, 4], [2, 5, 1], [(1, 3, 9, 1), (7, 4, 9, 2)]),
        h([3, 9, 4], [2, 5, 1], [(1, 9, 3, 0), (7, 4, 9, 2)]),
        h([3, 9, 4], [2, 5, 1], [(2, 3, 9, 0), (7, 4, 9, 2)]),
        h([3, 9, 4], [2, 5, 1], [(1, 3, 9, 0)]),
        h([3, 9], [2, 5], [(1, 3, 9, 0), (7, 4, 9, 2)]),
    ]
    assert len(set(variants + [base])) == len(variants) + 1
    m = oracle_mod.mix64
    mask = (1 << 64) - 1
    one_arc = (m((1 << 56) | 11) * 6) & mask   # multiply-add arc term (reading G16)
    one_vis = m((2 << 56) | (3 << 48) | (5 << 32) | (11 << 16) | 12)
    assert h([11], [6], []) == m(one_arc)
    assert h([11], [6], [(5, 11, 12, 3)]) == m((one_arc + one_vis) & mask)


def _walk_dep(g, L):
    """Def 11 / Alg 2 by exhaustive enumeration of arc chains (no breadth-first shortcut)."""
    M, A = g["M"], g["A"]
    prods = [[] for _ in range(A)]
    for a in range(A):
        for q in range(g["col_ptr"][a], g["col_ptr"][a + 1]):
            if g["col_s"][q] > 0:
                prods[a].append(int(g["col_met"][q]))
    consumers = [[int(x) for x in g["out_arc"][g["out_ptr"][i]:g["out_ptr"][i + 1]]] for i in range(M)]
    dep = set()
    for i in range(M):
        ins = [int(x) for x in g["in_arc"][g["in_ptr"][i]:g["in_ptr"][i + 1]]]

        def walk(o, x, length):
            if x in ins and x != o:
                dep.add((i, o, x))
            if length == L:
                return
            for q in prods[x]:
                if q == i:
                    continue
                for y in consumers[q]:
                    if y != g["twin"][x]:
                        walk(o, y, length + 1)

        for o in consumers[i]:
            walk(o, o, 1)
    return dep


def test_graph_and_dep_table(oracle_mod):
    """O1 against S itself (sign convention PAPER.md:45) and O7 against exhaustive chain enumeration."""
    for name in ("toy", "small"):
        net = make_network(name, 0)
        res = oracle_mod.enumerate_network(net, export_graph=True, self_check=False)
        g = res.graph
        Sint = net.S[net.internal.astype(bool)].astype(np.int64)
        assert g["M"] == Sint.shape[0] and g["A"] == net.n_arcs
        dense = np.zeros((g["M"], g["A"]), np.int64)
        for a in range(g["A"]):
            for q in range(g["col_ptr"][a], g["col_ptr"][a + 1]):
                dense[g["col_met"][q], a] = g["col_s"][q]
        for a in range(g["A"]):
            assert np.array_equal(dense[:, a], Sint[:, g["arc_rxn"][a]] * g["arc_dir"][a])
            t = g["twin"][a]
            if t >= 0:
                assert g["arc_rxn"][t] == g["arc_rxn"][a] and g["arc_dir"][t] == -g["arc_dir"][a]
                assert net.reversible[g["arc_rxn"][a]]
        for i in range(g["M"]):
            ins = g["in_arc"][g["in_ptr"][i]:g["in_ptr"][i + 1]]
            outs = g["out_arc"][g["out_ptr"][i]:g["out_ptr"][i + 1]]
            assert list(ins) == [a for a in range(g["A"]) if dense[i, a] > 0]
            assert list(outs) == [a for a in range(g["A"]) if dense[i, a] < 0]
            assert list(g["in_c"][g["in_ptr"][i]:g["in_ptr"][i + 1]]) == [dense[i, a] for a in ins]
            assert list(g["out_c"][g["out_ptr"][i]:g["out_ptr"][i + 1]]) == [-dense[i, a] for a in outs]
        truth = _walk_dep(g, net.params["dep_depth"])
        got = set()
        for i in range(g["M"]):
            ins = g["in_arc"][g["in_ptr"][i]:g["in_ptr"][i + 1]]
            outs = g["out_arc"][g["out_ptr"][i]:g["out_ptr"][i + 1]]
            for lo, o in enumerate(outs):
                for le, e in enumerate(ins):
                    if g["dep"][g["dep_off"][i] + lo * len(ins) + le]:
                        got.add((i, int(o), int(e)))
        assert got == truth
        assert len(truth) > 0


def test_seed_validation(oracle_mod):
    net = make_network("toy", 0)
    j_rev = int(np.nonzero(net.reversible)[0][0])
    j_irr = int(np.nonzero(net.reversible == 0)[0][0])
    for bad in ([[2 * j_rev, 2 * j_rev + 1]], [[2 * j_irr + 1]], [[2 * net.n]], [[0, 0]], [[]]):
        with pytest.raises(ValueError):
            oracle_mod.enumerate_pathways(net.S, net.reversible, net.internal, net.params, bad)


def _chain(coef_cons, length, tail=None):
    """->A0, c A_t -> A_{t+1} (t < length), A_length ->; optional extra product (name, coefficient) of the source."""
    names = [f"A{t}" for t in range(length + 1)]
    src = {names[0]: 1}
    internal = list(names)
    if tail:
        src[tail[0]] = tail[1]
        internal.append(tail[0])   # highest node index: it is visited last (reading G12)
    rx = [({}, src, False)]
    for t in range(length):
        rx.append(({names[t]: coef_cons}, {names[t + 1]: 1}, False))
    rx.append(({names[length]: 1}, {}, False))
    if tail:
        rx.append(({tail[0]: 1}, {}, False))
    return hand_network(rx, internal)


def test_overflow_guard_closed_form(oracle_mod):
    """Reading G21 (any state integer above 2^62 discards the pathway) on chains whose fluxes are known in closed form:
    c A_t -> A_{t+1} multiplies the scale by c per step (Eq 3 with the integer rescaling of reading G10), so the source
    flux is c^length.  3^39 < 2^62 < 3^40; 2^62 itself is allowed, 2^63 is not; and the guard also covers extra fluxes:
    a source that makes 3 Z per unit has EF_Z = 3 * 2^k, above 2^62 from k = 61 on while every flux is still below."""
    def run(net):
        return oracle_mod.enumerate_pathways(net.S, net.reversible, net.internal, net.params, [[0]])
    r = run(_chain(3, 30))
    assert r.stats["output"] == 1 and int(r.flux.max()) == 3 ** 30 and r.stats["discarded_overflow"] == 0
    r = run(_chain(3, 39))
    assert r.stats["output"] == 1 and int(r.flux.max()) == 3 ** 39 and r.stats["discarded_overflow"] == 0
    assert r.flux.tolist()[0] == [3 ** 39] + [3 ** (38 - t) for t in range(39)] + [1]
    r = run(_chain(3, 40))
    assert r.stats["output"] == 0 and r.stats["discarded_overflow"] == 1 and r.stats["expanded"] == 40
    r = run(_chain(2, 62))
    assert r.stats["output"] == 1 and int(r.flux.max()) == 2 ** 62 and r.stats["discarded_overflow"] == 0
    r = run(_chain(2, 63))
    assert r.stats["output"] == 0 and r.stats["discarded_overflow"] == 1
    r = run(_chain(2, 60, tail=("Z", 3)))
    assert r.stats["output"] == 1 and int(r.flux.max()) == 3 * 2 ** 60 and r.stats["discarded_overflow"] == 0
    r = run(_chain(2, 61, tail=("Z", 3)))
    assert r.stats["output"] == 0 and r.stats["discarded_overflow"] == 1


def test_mirror_symmetry(oracle_mod):
    """Def 9 treats surplus and deficit symmetrically: forward flow pushes through O, backward flow pulls
    through I; PROC1/PROC1' and Eq 3-5 come in mirrored pairs (Table 1) and Def 11 reads PO~SI one way
    and PI~SO the other.  Reversing every reaction (S -> -S) therefore swaps the two halves of the procedure and must
    reproduce the same flux vectors and the same counters.  With the forward half pinned by the hand cases this pins
    the backward half (Eq 4 / Eq 5 backward, the PI~SO lookup, PO = lowest consumer)."""
    cases = [(make_network("toy", 0), None, {}), (make_network("small", 0), None, {}), (make_network("small", 3), None, {}),
             (make_network("core", 0), None, dict(max_support=12))]
    net = make_network("toy", 0)
    cases.append((net, oracle_mod.all_arc_seed_sets(net.reversible), {}))
    net = make_network("small", 0)
    cases.append((net, random_seed_sets(net, 60, 2, 5), {}))
    for seed in range(6):
        net = unimolecular_network(seed, 5, 9, 2)
        cases.append((net, oracle_mod.all_arc_seed_sets(net.reversible), {}))
    n_rev = 0
    for net, seeds, over in cases:
        kw = dict(seed_sets=seeds) if seeds is not None else {}
        a = oracle_mod.enumerate_network(net, self_check=False, **kw, **over)
        b = oracle_mod.enumerate_network(mirrored(net), self_check=False, **kw, **over)
        assert np.array_equal(a.flux, b.flux), net.name
        assert a.stats == b.stats, net.name
        n_rev += a.stats["expanded"] - a.stats["children"] > 0
    assert n_rev > 0


def _python_state_hash(oracle_mod, e):
    arcs = sorted(e["flux"])
    return oracle_mod.state_hash(arcs, [e["flux"][a] for a in arcs], [(m,) + v for m, v in sorted(e["visited"].items())])


@pytest.mark.parametrize("name,cap", [("small", 300), ("small", 37), ("core", 512)])
def test_beam_against_sorted_definition(oracle_mod, name, cap):
    """Beam B restated on the oracle's own level contents (test hook): key = min(n_unb, 255) << 56 |
    h >> 8 with n_unb counted here from S_int . v; the level keeps exactly the entries with key <= T*, T* the largest
    value such that #{key <= T*} <= cap (sort-based, ties stand or fall together)."""
    net = make_network(name, 0)
    _beam_restatement(oracle_mod, net, cap, object)


def test_beam_key_clamps_the_unbalanced_count_at_255(oracle_mod):
    """key = min(n_unb, 255) << 56 | h >> 8.  On netgen.wide_fan_network (r0 -> P_0 .. P_299, r1 -> Q_0 .. Q_199,
    two consumers per product) with seeds {r0}, {r1} level k holds 2^k
    entries with n_unb = 300 - k (clamped: top byte 0xff) and 2^k with n_unb = 200 - k (top byte 200 - k < 0xff).  cap 40 binds
    from level 5 on (32 + 32 entries): every entry of the r1 family ranks before every entry of the r0 family, which are ranked
    among themselves by the hash bits alone.  A clamp at 127 would mix the families, no clamp would wrap 295 to 39 and put the r0
    family first; the restatement (n_unb recounted from S . v) fails on either."""
    net = wide_fan_network()
    levels = _beam_restatement(oracle_mod, net, 40, np.int64, seed_sets=[[0], [2]], max_visited=7)
    lvl5 = levels[5]
    big = [e for e in lvl5 if e["n_unb"] == 295]
    small = [e for e in lvl5 if e["n_unb"] == 195]
    assert len(big) == 32 and len(small) == 32
    assert all(e["key"] >> 56 == 0xff for e in big) and all(e["key"] >> 56 == 195 for e in small)
    assert all(e["kept"] for e in small) and sum(e["kept"] for e in big) == 8
    kept_big = sorted(e["key"] for e in big if e["kept"])
    assert kept_big == sorted(e["key"] for e in big)[:8]          # ... by the 56 hash bits


def _beam_restatement(oracle_mod, net, cap, dtype, **over):
    res = oracle_mod.enumerate_network(net, self_check=False, trace=True, frontier_cap=cap, **over)
    assert res.stats["truncated_beam"] > 0
    Sint = net.S[net.internal.astype(bool)].astype(dtype)
    arc_col = []
    for j in range(net.n):
        arc_col.append((j, 1))
        if net.reversible[j]:
            arc_col.append((j, -1))
    cut_levels = 0
    truncated = 0
    for lvl in res.trace:
        keys = []
        for e in lvl:
            v = np.zeros(net.n, dtype=dtype)
            for a, f in e["flux"].items():
                v[arc_col[a][0]] += arc_col[a][1] * f
            n_unb = int(np.count_nonzero(Sint.dot(v)))
            assert n_unb == e["n_unb"]
            if n_unb == 0:
                assert e["kept"] and e["istar"] < 0
                continue
            key = (min(n_unb, 255) << 56) | (_python_state_hash(oracle_mod, e) >> 8)
            assert key == e["key"]
            keys.append((key, e["kept"]))
        if len(keys) <= cap:
            assert all(k for _, k in keys)
            continue
        cut_levels += 1
        srt = sorted(k for k, _ in keys)
        # T* = largest value with #{key <= T*} <= cap: walk the distinct keys
        tstar = -1
        count = 0
        i = 0
        while i < len(srt):
            j = i
            while j < len(srt) and srt[j] == srt[i]:
                j += 1
            if j > cap:
                break
            tstar, count, i = srt[i], j, j
        assert [kept for _, kept in keys] == [k <= tstar for k, _ in keys]
        assert count <= cap
        truncated += len(keys) - count
    assert cut_levels > 0 and truncated == res.stats["truncated_beam"]
    return res.trace


def test_beam_ties_stand_or_fall_together(oracle_mod):
    """Two identical seed sets give identical states, hence equal keys: with cap = 1 neither may be kept (SURVEY.md
    8(c)-B: 'entries with equal keys stand or fall together ... if even the smallest key bucket exceeds cap, the level
    empties')."""
    rx = [({}, {"A": 1}, False), ({"A": 1}, {}, False)]
    net = hand_network(rx, ["A"], frontier_cap=1)
    res = oracle_mod.enumerate_pathways(net.S, net.reversible, net.internal, net.params, [[0], [0]])
    assert res.stats["truncated_beam"] == 2 and res.stats["output"] == 0 and res.stats["expanded"] == 0
    net2 = hand_network(rx, ["A"], frontier_cap=2)
    res = oracle_mod.enumerate_pathways(net2.S, net2.reversible, net2.internal, net2.params, [[0], [0]])
    assert res.stats["truncated_beam"] == 0 and res.flux.tolist() == [[1, 1]]


@pytest.mark.parametrize("name,over,count,size", [("small", {}, 200, 2), ("core", dict(frontier_cap=4096), 200, 2),
                                                  ("small", {}, 120, 3)])
def test_poison_and_minimality_at_scale(oracle_mod, name, over, count, size):
    """O8(ii)/(iii) restated on the oracle's own balanced entries (test hook): group the Done states by support; a support
    with two different vectors is poisoned; among the rest, drop every support that strictly contains another
    (Def 3).  Multi-arc seed sets make both rules fire."""
    net = make_network(name, 0)
    seeds = random_seed_sets(net, count, size, 11)
    res = oracle_mod.enumerate_network(net, self_check=True, seed_sets=seeds, trace=2, threads=2, **over)
    groups = {}
    n_done = 0
    for lvl in res.trace:
        for e in lvl:
            if e["n_unb"] == 0:
                n_done += 1
                groups.setdefault(frozenset(e["flux"]), set()).add(tuple(sorted(e["flux"].items())))
    assert n_done == res.stats["done"]
    ok = {s: next(iter(v)) for s, v in groups.items() if len(v) == 1}
    poisoned = len(groups) - len(ok)
    minimal = [s for s in ok if not any(o < s for o in ok)]
    arc_col = []
    for j in range(net.n):
        arc_col.append((j, 1))
        if net.reversible[j]:
            arc_col.append((j, -1))
    rows = []
    for s in minimal:
        v = [0] * net.n
        for a, f in ok[s]:
            v[arc_col[a][0]] += arc_col[a][1] * f
        rows.append(v)
    rows.sort()
    assert res.stats["unique_supports"] == len(groups) and res.stats["poisoned"] == poisoned
    assert res.flux.tolist() == rows
    assert poisoned > 0 and len(ok) - len(minimal) > 0   # both rules did something


def test_default_seeds_are_the_boundary_arcs(oracle_mod):
    """O2 / Def 8 'starting from a boundary reaction': without explicit seeds there is one root per arc whose
    internal column is non-empty and single-signed.  P5 network: r0 ->A, r1 A<=>B, r2 B->, r3 ->B, r4 A->: the boundary
    arcs are r0, r2, r3, r4 (codes 0, 4, 6, 8); neither direction of r1 is one; an all-external reaction is none either."""
    rx = [({}, {"A": 1}, False), ({"A": 1}, {"B": 1}, True), ({"B": 1}, {}, False), ({}, {"B": 1}, False), ({"A": 1}, {}, False),
          ({"X": 1}, {"Y": 1}, False)]
    net = hand_network(rx, ["A", "B"])
    dflt = oracle_mod.enumerate_pathways(net.S, net.reversible, net.internal, net.params, None)
    expl = oracle_mod.enumerate_pathways(net.S, net.reversible, net.internal, net.params, [[0], [4], [6], [8]])
    assert dflt.n_roots == 4 and dflt.stats == expl.stats and np.array_equal(dflt.flux, expl.flux)
    assert dflt.flux.tolist() == [[0, -1, 0, 1, 1, 0], [0, 0, 1, 1, 0, 0], [1, 0, 0, 0, 1, 0], [1, 1, 1, 0, 0, 0]]
