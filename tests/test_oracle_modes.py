"""Pins of the oracle's two extra modes (SURVEY.md 8(f)-1 literal sampling, 8(f)-2 targeted observability) and of the
step count it reports per pathway.  Nothing here compares the oracle with itself only: the sampled choice is restated in
Python from the formula in DESIGN.md (reading G23), the reachable states are compared with the exhaustive fan-out
(Theorem 1: "by selecting all outputs/inputs ... all pathways are produced"), the mask and the step
counts are derived by hand on the P1 / P2 / P5 networks of SURVEY.md 8(c)."""
import numpy as np
import pytest

from netgen import chain_pair_network, hand_network, make_network

M64 = (1 << 64) - 1


def mix(x):   # SplitMix64 finaliser, written out (published constants; pinned against vectors in test_oracle_pins.py)
    x &= M64
    x ^= x >> 30; x = (x * 0xBF58476D1CE4E5B9) & M64
    x ^= x >> 27; x = (x * 0x94D049BB133111EB) & M64
    x ^= x >> 31
    return x


def pick(seed, cand, met):   # DESIGN.md reading G23
    return mix(mix((seed + 0x9E3779B97F4A7C15 * (cand + 1)) & M64) ^ ((0x04 << 56) | met))


P1 = ([({}, {"A": 1}, False), ({"A": 1}, {"B": 1, "C": 1}, False), ({"B": 1}, {}, False), ({"C": 1}, {}, False)], ["A", "B", "C"])
P2 = ([({}, {"A": 1}, False), ({"A": 1}, {"B": 1, "C": 1}, False), ({"C": 2}, {"A": 1}, False), ({"B": 1}, {}, False)], ["A", "B", "C"])
P5 = ([({}, {"A": 1}, False), ({"A": 1}, {"B": 1}, True), ({"B": 1}, {}, False), ({}, {"B": 1}, False), ({"A": 1}, {}, False)], ["A", "B"])


def run(oracle_mod, net, seeds, **kw):
    return oracle_mod.enumerate_pathways(net.S, net.reversible, net.internal, net.params, seeds, **kw)


def test_steps_of_hand_traces(oracle_mod):
    """P1: three expansions (A, B, C) build (1,1,1,1); P2: four (A, B, C, A again) build (1,2,1,2) -- SURVEY.md 8(c) P1 / P2
    traces.  P5 with seeds {r0}, {r2}: (1,0,0,0,1) and (1,1,1,0,0) take 1 and 2 expansions from r0, (0,0,1,1,0) takes one
    backward expansion from r2."""
    r = run(oracle_mod, hand_network(*P1), [[0]])
    assert r.flux.tolist() == [[1, 1, 1, 1]] and r.steps.tolist() == [3]
    r = run(oracle_mod, hand_network(*P2), [[0]])
    assert r.flux.tolist() == [[1, 2, 1, 2]] and r.steps.tolist() == [4]
    r = run(oracle_mod, hand_network(*P5), [[0], [4]])
    assert r.flux.tolist() == [[0, 0, 1, 1, 0], [1, 0, 0, 0, 1], [1, 1, 1, 0, 0]]
    assert r.steps.tolist() == [1, 1, 2]


def test_steps_take_the_quickest_construction(oracle_mod):
    """Seeds {r0} and {r0, r4} of P5 both reach (1,0,0,0,1): in one expansion and in none (the seed set is balanced at
    once); equal duplicates are one pathway and its step count is the smallest."""
    r = run(oracle_mod, hand_network(*P5), [[0], [0, 8]])
    rows = {tuple(v): s for v, s in zip(r.flux.tolist(), r.steps.tolist())}
    assert rows[(1, 0, 0, 0, 1)] == 0 and rows[(1, 1, 1, 0, 0)] == 2


def test_reaction_mask_by_hand(oracle_mod):
    """8(f)-2 on P5 (r0: ->A, r1: A<=>B, r2: B->, r3: ->B, r4: A->), seed r0.  All reactions allowed: A first visited,
    alternatives r1+ and r4 => (1,1,1,0,0) and (1,0,0,0,1).  Without r4: only the route through r1, r2.  Without r1:
    only r4.  Without r1 and r4: A has no admissible alternative, a dead end.  The mask of exactly the reactions of
    (1,1,1,0,0) constructs it in 2 expansions (the 'observability' question of PAPER.md:392-396)."""
    net = hand_network(*P5)
    full = run(oracle_mod, net, [[0]])
    assert full.flux.tolist() == [[1, 0, 0, 0, 1], [1, 1, 1, 0, 0]]
    same = run(oracle_mod, net, [[0]], allowed=np.ones(5, np.uint8))
    assert same.flux.tolist() == full.flux.tolist() and same.stats == full.stats
    r = run(oracle_mod, net, [[0]], allowed=np.array([1, 1, 1, 1, 0], np.uint8))
    assert r.flux.tolist() == [[1, 1, 1, 0, 0]] and r.steps.tolist() == [2]
    r = run(oracle_mod, net, [[0]], allowed=np.array([1, 0, 1, 1, 1], np.uint8))
    assert r.flux.tolist() == [[1, 0, 0, 0, 1]] and r.steps.tolist() == [1]
    r = run(oracle_mod, net, [[0]], allowed=np.array([1, 0, 1, 1, 0], np.uint8))
    assert r.flux.tolist() == [] and r.stats["dead_end"] == 1 and r.stats["expanded"] == 1
    r = run(oracle_mod, net, [[0]], allowed=np.array([1, 1, 1, 0, 0], np.uint8))
    assert r.flux.tolist() == [[1, 1, 1, 0, 0]] and r.steps.tolist() == [2]
    # the mask does not touch the seeds: a seed outside the subset still starts its pathway
    r = run(oracle_mod, net, [[8]], allowed=np.array([1, 1, 1, 1, 0], np.uint8))
    assert r.flux.tolist() == [[0, -1, 0, 1, 1], [1, 0, 0, 0, 1]]


def test_mask_removes_exactly_the_pathways_through_masked_reactions_when_no_choice_depends_on_them(oracle_mod):
    """Unimolecular networks (every node balances by choosing ONE alternative, no AND): masking reaction j can only
    remove alternatives, so the result is the unmasked result minus the rows that use j."""
    from netgen import unimolecular_network
    for seed in range(6):
        net = unimolecular_network(seed, m_int=5, n_rxn=9, n_rev=seed % 2)
        seeds = oracle_mod.all_arc_seed_sets(net.reversible)
        full = run(oracle_mod, net, seeds)
        for j in range(net.S.shape[1]):
            al = np.ones(net.S.shape[1], np.uint8); al[j] = 0
            r = run(oracle_mod, net, [s for s in seeds if s[0] // 2 != j], allowed=al)
            want = [row for row in full.flux.tolist() if row[j] == 0]
            assert r.flux.tolist() == want, (seed, j)


def test_sampled_choice_follows_the_written_generator(oracle_mod):
    """One node with five outputs: candidate c must take alternative pick(seed, c, 0) mod 5 in ascending arc order."""
    rx = [({}, {"A": 1}, False)] + [({"A": 1}, {}, False) for _ in range(5)]
    net = hand_network(rx, ["A"])
    for seed in (0, 1, 12345, M64):
        r = run(oracle_mod, net, [[0]], sample_count=40, sample_seed=seed)
        assert r.cand_end[:, 0].tolist() == [1] * 40 and r.cand_end[:, 1].tolist() == [1] * 40
        used = sorted({1 + pick(seed, c, 0) % 5 for c in range(40)})
        assert [int(np.nonzero(row[1:])[0][0]) + 1 for row in r.flux.tolist()] == sorted(used, reverse=True)
    # the choice skips inadmissible alternatives: with r2 and r4 masked three remain, in arc order r1, r3, r5
    al = np.array([1, 1, 0, 1, 0, 1], np.uint8)
    r = run(oracle_mod, net, [[0]], sample_count=40, sample_seed=7, allowed=al)
    used = {[1, 3, 5][pick(7, c, 0) % 3] for c in range(40)}
    assert {int(np.nonzero(row[1:])[0][0]) + 1 for row in r.flux.tolist()} == used


def _done_states(res):
    return {tuple(sorted(e["flux"].items())) for lvl in res.trace for e in lvl if e["n_unb"] == 0}


@pytest.mark.parametrize("name", ["toy", "P5"])
def test_sampling_reaches_only_and_eventually_all_states_of_the_fan_out(oracle_mod, name):
    """Theorem 1: every balanced state a sampled candidate reaches is a balanced state of the exhaustive
    fan-out, and over enough generator seeds the union is the whole set (the lineage of a state fixes one choice per
    visited metabolite, which some seed realises)."""
    if name == "toy":
        net = make_network("toy", 0)
        seeds = None
    else:
        net = hand_network(*P5)
        seeds = [[0], [4], [6]]
    full = _done_states(run(oracle_mod, net, seeds, trace=2))
    n_roots = run(oracle_mod, net, seeds).n_roots
    got = set()
    for s in range(400):
        r = run(oracle_mod, net, seeds, trace=2, sample_count=n_roots, sample_seed=s)
        st = _done_states(r)
        assert st <= full
        assert r.stats["children"] <= r.stats["expanded"]          # no fan-out: one child per expansion at most
        got |= st
        if got == full:
            break
    assert got == full


def test_sampling_bookkeeping_and_order_independence(oracle_mod):
    """Every candidate ends exactly once, the per-candidate records add up to the counters, and neither the thread count
    nor the processing order changes anything (the generator is keyed on (candidate, metabolite), not on order)."""
    net = make_network("small", 0)
    a = oracle_mod.enumerate_network(net, sample_count=300, sample_seed=5)
    codes = a.cand_end[:, 0]
    assert a.n_roots == 300 and np.all(codes > 0)
    st = a.stats
    assert (codes == 1).sum() == st["done"] and (codes == 2).sum() == st["not_efm_maxloop"]
    assert (codes == 3).sum() == st["dead_end"] and (codes == 4).sum() == st["discarded_visited"]
    assert (codes == 5).sum() == st["discarded_nonpos"] and (codes == 6).sum() == st["discarded_overflow"]
    assert st["peak_frontier"] <= 300 and st["truncated_beam"] == 0
    # a candidate that ended Done after s expansions sits on level s
    assert int(a.cand_end[codes == 1, 1].max()) < st["levels"]
    b = oracle_mod.enumerate_network(net, sample_count=300, sample_seed=5, threads=3, shuffle_seed=99, frontier_cap=7)
    assert np.array_equal(a.flux, b.flux) and a.stats == b.stats and np.array_equal(a.cand_end, b.cand_end)
    c = oracle_mod.enumerate_network(net, sample_count=300, sample_seed=6)
    assert not np.array_equal(a.cand_end, c.cand_end)
    # candidate c starts from seed set c mod n_sets: with 8 default roots, candidates 3 and 11 share their seed arc
    full = oracle_mod.enumerate_network(net)
    assert full.n_roots >= 2


# ---------------------------------------------------------------------------------------------------------------------
# SURVEY.md 8(f)-3 exact elementarity (rank test instead of "minimal among the candidates found")
# ---------------------------------------------------------------------------------------------------------------------
def _rational_rank(rows):
    """Rank over the rationals by fraction elimination (independent of the oracle's modular elimination)."""
    from fractions import Fraction
    Mx = [[Fraction(int(v)) for v in r] for r in rows]
    rank, ncol = 0, len(Mx[0]) if Mx else 0
    for c in range(ncol):
        piv = next((r for r in range(rank, len(Mx)) if Mx[r][c] != 0), None)
        if piv is None:
            continue
        Mx[rank], Mx[piv] = Mx[piv], Mx[rank]
        for r in range(rank + 1, len(Mx)):
            if Mx[r][c] != 0:
                f = Mx[r][c] / Mx[rank][c]
                Mx[r] = [x - f * y for x, y in zip(Mx[r], Mx[rank])]
        rank += 1
    return rank


def test_exact_mode_by_hand(oracle_mod):
    """H7 network r0: ->A, r1: A->, r2: ->B, r3: 2B->, seed {r0, r2}: the balanced pathway (2,2,2,1) uses all four reactions.
    Its internal rows are A: (1,-1,0,0), B: (0,0,1,-2): rank 2 = |supp| - 2, nullity 2 -- it is the sum of the two EFMs
    (1,1,0,0) and (0,0,2,1), not elementary (Def 3).  Alone among the candidates it passes the pairwise
    filter; the rank test rejects it.  Seed {r0}: (1,1,0,0), one row, rank 1 = |supp| - 1: elementary."""
    net = hand_network([({}, {"A": 1}, False), ({"A": 1}, {}, False), ({}, {"B": 1}, False), ({"B": 2}, {}, False)], ["A", "B"])
    assert run(oracle_mod, net, [[0, 4]]).flux.tolist() == [[2, 2, 2, 1]]
    r = run(oracle_mod, net, [[0, 4]], exact=True)
    assert r.flux.tolist() == [] and r.stats["non_elementary"] == 1 and r.stats["unique_supports"] == 1
    r = run(oracle_mod, net, [[0, 4], [0], [4]], exact=True)
    assert r.flux.tolist() == [[0, 0, 2, 1], [1, 1, 0, 0]] and r.stats["non_elementary"] == 1
    # P2 (recycle): (1,2,1,2) on r0..r3; rows A: (1,-1,1,0), B: (0,1,0,-1), C: (0,1,-2,0): rank 3 = 4 - 1
    r = run(oracle_mod, hand_network(*P2), [[0]], exact=True)
    assert r.flux.tolist() == [[1, 2, 1, 2]] and r.stats["non_elementary"] == 0


@pytest.mark.parametrize("name,over,count", [("toy", {}, 0), ("small", {}, 150), ("core", dict(frontier_cap=4096), 150),
                                             ("mid", dict(frontier_cap=2048), 200)])
def test_exact_mode_against_rational_rank(oracle_mod, name, over, count):
    """Every balanced state the traversal reaches (test hook), grouped by support: a support with one flux vector whose
    internal rows have RATIONAL rank |supp| - 1 (fraction elimination, written here) must be an output of the exact
    mode, every other one must not."""
    from netgen import random_seed_sets
    net = make_network(name, 0)
    seeds = random_seed_sets(net, count, 2, 11) if count else oracle_mod.all_arc_seed_sets(net.reversible)
    res = oracle_mod.enumerate_network(net, seed_sets=seeds, exact=True, trace=2, self_check=False, **over)
    groups = {}
    for lvl in res.trace:
        for e in lvl:
            if e["n_unb"] == 0:
                groups.setdefault(frozenset(e["flux"]), set()).add(tuple(sorted(e["flux"].items())))
    arcs = []
    for j in range(net.n):
        arcs.append((j, 1))
        if net.reversible[j]:
            arcs.append((j, -1))
    Sint = net.S[net.internal.astype(bool)].astype(np.int64)
    want, rejected = [], 0
    for supp, vecs in groups.items():
        if len(vecs) != 1:
            continue
        cols = sorted(supp)
        sub = np.stack([Sint[:, arcs[a][0]] * arcs[a][1] for a in cols], axis=1)
        sub = sub[np.any(sub != 0, axis=1)]
        if _rational_rank(sub.tolist()) == len(cols) - 1:
            v = [0] * net.n
            for a, f in next(iter(vecs)):
                v[arcs[a][0]] += arcs[a][1] * f
            want.append(v)
        else:
            rejected += 1
    want.sort()
    assert res.flux.tolist() == want
    assert res.stats["non_elementary"] == rejected and res.stats["output"] == len(want)
    if count:
        assert rejected > 0   # the rank test did something the data could show


def chain_flux(length):
    """Closed form of netgen.chain_pair_network's single chain: step i (1 <= i < length) turns one A_{i-1} into 2 A_i when
    i % 10 == 0, else into one; balancing node by node, reaction i + 1 runs at the rate A_i is produced."""
    f = [1, 1]
    for i in range(1, length):
        f.append(f[-1] * (2 if i % 10 == 0 else 1))
    return f


@pytest.mark.parametrize("len_a,len_b,D", [(70, 20, 96), (100, 24, 128)])
def test_exact_mode_on_supports_wider_than_64_arcs(oracle_mod, len_a, len_b, D):
    """Def 3 on supports of 71 / 101 arcs: each chain alone is elementary (closed-form fluxes above), the
    pathway seeded on both chain heads balances to their sum over len_a + len_b + 2 arcs and has nullity 2."""
    net = chain_pair_network(len_a, len_b, max_support=D)
    na = len_a + 1
    fa, fb = chain_flux(len_a), chain_flux(len_b)
    r = run(oracle_mod, net, [[0], [2 * na], [0, 2 * na]], exact=True)
    assert r.flux.tolist() == sorted([fa + [0] * (len_b + 1), [0] * na + fb])
    assert (r.stats["unique_supports"], r.stats["non_elementary"], r.stats["output"]) == (3, 1, 2)
    plain = run(oracle_mod, net, [[0, 2 * na]])          # the pairwise filter alone cannot see it: nothing smaller was found
    assert plain.flux.tolist() == [fa + fb]


def test_exact_mode_outputs_are_true_efms_of_the_toy_network(oracle_mod):
    """Brute force (every arc subset without a twin pair whose nullspace is one strictly positive ray) fixes the EFM set of
    toy; the exact mode returns exactly the found candidates that are in it."""
    from oracle.brute_force import brute_force_efms
    net = make_network("toy", 0)
    truth = {tuple(int(x) for x in r) for r in brute_force_efms(net.S, net.reversible, net.internal)}
    seeds = oracle_mod.all_arc_seed_sets(net.reversible)
    ex = oracle_mod.enumerate_network(net, seed_sets=seeds, exact=True)
    assert {tuple(r) for r in ex.flux.tolist()} <= truth
    assert ex.stats["output"] + ex.stats["non_elementary"] + ex.stats["poisoned"] == ex.stats["unique_supports"]


# ---------------------------------------------------------------------------------------------------------------------
# sharper pins of the sampling rule: one candidate at a time, so that nothing is averaged away
# ---------------------------------------------------------------------------------------------------------------------
def test_each_candidate_takes_exactly_its_own_pick(oracle_mod):
    """Node B (metabolite index 1) with five outputs behind A -> B: with C candidates the alternatives in use are exactly
    {pick(seed, c, 1) mod 5 : c < C} -- checked for C = 1, 2, 3 and twenty generator seeds, so the candidate number, the
    metabolite index and the modulus all matter.  With r3 and r5 masked the count runs over the three admissible ones only."""
    rx = [({}, {"A": 1}, False), ({"A": 1}, {"B": 1}, False)] + [({"B": 1}, {}, False) for _ in range(5)]
    net = hand_network(rx, ["A", "B"])
    for seed in range(20):
        for C in (1, 2, 3):
            r = run(oracle_mod, net, [[0]], sample_count=C, sample_seed=seed)
            got = {int(np.nonzero(row[2:])[0][0]) for row in r.flux.tolist()}
            assert got == {pick(seed, c, 1) % 5 for c in range(C)}, (seed, C)
            al = np.array([1, 1, 1, 0, 1, 0, 1], np.uint8)     # alternatives r2, r4, r6 remain (positions 0, 2, 4)
            r = run(oracle_mod, net, [[0]], sample_count=C, sample_seed=seed, allowed=al)
            got = {int(np.nonzero(row[2:])[0][0]) for row in r.flux.tolist()}
            assert got == {[0, 2, 4][pick(seed, c, 1) % 3] for c in range(C)}, (seed, C)
            assert r.cand_end[:, 0].tolist() == [1] * C


def test_sampled_choice_counts_only_what_the_support_cap_admits(oracle_mod):
    """Reading G23 with a binding D (reading G15): r0 -> A, r1 A -> 3 B, r2 .. r6 B ->; one candidate from the seed set
    {r0, r3, r5} with max_support = 4.  A (first visit) adds r1: the support {r0, r1, r3, r5} is full.  B: EF = 3 - 2 = +1,
    first visit; of its five outputs only r3 and r5 (already in the support) are admissible, so the candidate takes
    [r3, r5][pick(seed, 0, 1) mod 2] -- not mod 5 -- bumps it to 2 and is balanced after two expansions."""
    rx = [({}, {"A": 1}, False), ({"A": 1}, {"B": 3}, False)] + [({"B": 1}, {}, False) for _ in range(5)]
    net = hand_network(rx, ["A", "B"], max_support=4)
    free = hand_network(rx, ["A", "B"])
    seen = set()
    differs = 0
    for seed in range(24):
        r = run(oracle_mod, net, [[0, 6, 10]], sample_count=1, sample_seed=seed)
        k = pick(seed, 0, 1) % 2
        seen.add(k)
        differs += [3, 5][k] != 2 + pick(seed, 0, 1) % 5
        want = [1, 1, 0, 1, 0, 1, 0]
        want[[3, 5][k]] = 2
        assert r.flux.tolist() == [want], seed
        assert r.cand_end.tolist() == [[1, 2]] and r.steps.tolist() == [2]
    assert seen == {0, 1} and differs >= 12
    # without the cap all five are admissible again and the modulus is 5
    for seed in range(24):
        r = run(oracle_mod, free, [[0, 6, 10]], sample_count=1, sample_seed=seed)
        j = 2 + pick(seed, 0, 1) % 5
        want = [1, 1, 0, 1, 0, 1, 0]
        want[j] += 1
        assert r.flux.tolist() == [want], seed


def test_candidate_c_starts_from_seed_set_c_mod_n(oracle_mod):
    """P5 with two seed sets (arcs: r0 -> 0, r2 -> 3): the roots of level 0 (test hook) show which set every candidate took."""
    net = hand_network(*P5)

    def roots(seed_sets, C, seed):
        r = run(oracle_mod, net, seed_sets, sample_count=C, sample_seed=seed, trace=1)
        assert r.n_roots == C
        return sorted(tuple(sorted(e["flux"])) for e in r.trace[0])

    for seed in range(4):
        assert roots([[0], [4]], 1, seed) == [(0,)]
        assert roots([[4], [0]], 1, seed) == [(3,)]
        assert roots([[4], [0]], 2, seed) == [(0,), (3,)]
        assert roots([[4], [0]], 3, seed) == [(0,), (3,), (3,)]      # candidates 0 and 2 start from {r2}, candidate 1 from {r0}
        assert roots([[0], [4], [0, 4]], 5, seed) == [(0,), (0,), (0, 3), (3,), (3,)]


def test_step_count_is_the_minimum_over_all_equal_duplicates(oracle_mod):
    """P5: (1,1,1,0,0) is reached from {r0} in 2 expansions, from {r0, r1+} in 1 and from {r0, r1+, r2} in 0; (1,0,0,0,1) from
    {r0} in 1 and from {r0, r4} in 0.  Whatever order the duplicates are grouped in, the smallest count is reported."""
    net = hand_network(*P5)
    sets = [[0], [0, 2], [0, 2, 4], [0, 8]]
    import itertools
    for perm in itertools.permutations(sets):
        r = run(oracle_mod, net, list(perm))
        rows = {tuple(v): s for v, s in zip(r.flux.tolist(), r.steps.tolist())}
        assert rows[(1, 1, 1, 0, 0)] == 0 and rows[(1, 0, 0, 0, 1)] == 0
    r = run(oracle_mod, net, [[0], [0, 2]])
    rows = {tuple(v): s for v, s in zip(r.flux.tolist(), r.steps.tolist())}
    assert rows[(1, 1, 1, 0, 0)] == 1 and rows[(1, 0, 0, 0, 1)] == 1
    r = run(oracle_mod, net, [[0, 2], [0]])
    rows = {tuple(v): s for v, s in zip(r.flux.tolist(), r.steps.tolist())}
    assert rows[(1, 1, 1, 0, 0)] == 1 and rows[(1, 0, 0, 0, 1)] == 1
