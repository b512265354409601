"""GPU <-> oracle parity (bit-exact): the CUDA path, called through the C ABI, must return the same set of pathways
as the CPU oracle -- same coprime integer flux vectors in the same canonical order -- and the same counters
(every discard reason, per-level frontier sizes, beam truncation, unique supports, algorithmic bytes)."""
import json
import os

import numpy as np
import pytest

from netgen import (chain_pair_network, hand_network, make_network, random_seed_sets, unimolecular_network, wide_fan_network,
                    with_dead_ends)

pytestmark = pytest.mark.gpu

STAT_KEYS = ["levels", "expanded", "children", "done", "dead_end", "not_efm_maxloop", "discarded_nonpos",
             "discarded_overflow", "discarded_visited", "truncated_beam", "unique_supports", "poisoned", "output",
             "peak_frontier", "algo_bytes"]
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "hand_pins.json")


@pytest.fixture(scope="module")
def efm():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_1804_02867_b200 import build
    build.build()
    import paper_1804_02867_b200 as mod
    mod.load()
    return mod


def _threads(oracle_mod):
    return max(1, min(oracle_mod.max_threads(), os.cpu_count() or 1, 64))


def assert_parity(efm, oracle_mod, net, seeds="net", flags=0, check_levels=True, allowed=None, **over):
    got = efm.enumerate_network(net, seed_sets=seeds, flags=flags, allowed=allowed, **over)
    okeys = {k: v for k, v in over.items() if k in ("max_support", "max_loop", "dep_depth", "max_visited", "frontier_cap",
                                                    "sample_count", "sample_seed")}
    exact = bool(flags & efm.EFM_F_EXACT_ELEMENTARITY)
    if flags & efm.EFM_F_COMPRESS:   # 8(f)-4: the oracle runs on the network its own pre-pass reduced
        params = dict(net.params)
        params.update(okeys)
        ref = oracle_mod.enumerate_compressed(net.S, net.reversible, net.internal, params,
                                              net.seed_sets if isinstance(seeds, str) else seeds, threads=_threads(oracle_mod),
                                              self_check=False, exact=exact)
        assert int(got.stats["blocked_reactions"]) == int(ref.blocked.sum())
    else:
        ref = oracle_mod.enumerate_network(net, threads=_threads(oracle_mod), seed_sets=seeds, self_check=False, allowed=allowed,
                                           exact=exact, **okeys)
    assert int(got.stats["non_elementary"]) == int(ref.stats["non_elementary"])
    for k in STAT_KEYS:
        assert int(got.stats[k]) == int(ref.stats[k]), (k, got.stats[k], ref.stats[k])
    if check_levels:
        for k in ("active", "done", "expanded", "children"):
            assert np.array_equal(got.levels[k], ref.levels[k]), k
    assert got.flux.shape == ref.flux.shape
    assert np.array_equal(got.flux, ref.flux)
    assert np.array_equal(got.steps, ref.steps)          # expansions that built every pathway
    assert int(got.stats["n_roots"]) == ref.n_roots
    if over.get("sample_count"):
        assert np.array_equal(got.cand_end, ref.cand_end)   # how and when every sampled candidate ended
    return got, ref


def test_hash_matches_oracle_hash(efm, oracle_mod):
    cases = [([11], [6], []), ([11], [6], [(5, 11, 12, 3)]), ([3, 9, 4], [2, 5, 1], [(1, 3, 9, 0), (7, 4, 9, 2)]),
             ([0, 65535], [1 << 61, 1], [(65535, 65535, 0, 8)])]
    for arcs, flux, vis in cases:
        assert efm.debug_state_hash(arcs, flux, vis) == oracle_mod.state_hash(arcs, flux, vis)


def _golden_cases():
    with open(GOLDEN) as fh:
        return json.load(fh)["cases"]


@pytest.mark.parametrize("case", _golden_cases(), ids=lambda c: c["name"])
def test_hand_pins_on_gpu(efm, case):
    """The hand-derived fixtures of tests/golden pin the CUDA path directly (no oracle involved)."""
    net = hand_network([(s, p, r) for s, p, r in case["reactions"]], case["internal"], **case.get("params", {}))
    got = efm.enumerate_network(net, seed_sets=case["seeds"])
    assert got.flux.tolist() == case["flux"]
    for k in ("expanded", "levels", "discarded_nonpos"):
        if k in case:
            assert int(got.stats[k]) == case[k], k
    for k, v in case.get("stats", {}).items():
        assert int(got.stats[k]) == v, (k, got.stats[k], v)


def _h7_shifted(n_pad):
    """The H7 network of tests/golden (r0: ->A, r1: A->, r2: ->B, r3: 2B->) behind n_pad reversible reactions between
    external metabolites: the arc ids move past 2 * n_pad, so with n_pad >= 56 the supports no longer fit the exact
    112-bit signature of the minimality filter and the hashed signature + sorted-list verification decides."""
    rx = [({"X%d" % t: 1}, {"Y%d" % t: 1}, True) for t in range(n_pad)]
    rx += [({}, {"A": 1}, False), ({"A": 1}, {}, False), ({}, {"B": 1}, False), ({"B": 2}, {}, False)]
    return hand_network(rx, ["A", "B"]), 2 * n_pad


@pytest.mark.parametrize("n_pad", [0, 60, 700])
def test_filter_drop_and_poison_by_hand(efm, n_pad):
    """Def 3 / PAPER.md:456 and SURVEY.md 8(c) O8(ii), derived by hand (tests/golden H7): seeds {r0, r2} and
    {r0} balance to supports {r0,r1,r2,r3} and {r0,r1}: the superset is dropped.  Seeds {r0, r2} and {r0, r3} reach the
    support {r0,r1,r2,r3} with fluxes (2,2,2,1) and (1,1,2,1): poisoned, nothing is left.  No oracle involved."""
    net, c0 = _h7_shifted(n_pad)
    z = [0] * n_pad
    got = efm.enumerate_network(net, seed_sets=[[c0, c0 + 4], [c0]])
    assert got.flux.tolist() == [z + [1, 1, 0, 0]]
    assert (got.stats["unique_supports"], got.stats["poisoned"], got.stats["output"]) == (2, 0, 1)
    got = efm.enumerate_network(net, seed_sets=[[c0, c0 + 4], [c0, c0 + 6]])
    assert got.flux.tolist() == []
    assert (got.stats["done"], got.stats["unique_supports"], got.stats["poisoned"], got.stats["output"]) == (2, 1, 1, 0)
    # three nested supports plus an unrelated one: only the minimal ones stay, in canonical order
    got = efm.enumerate_network(net, seed_sets=[[c0, c0 + 4], [c0], [c0 + 4]])
    assert got.flux.tolist() == [z + [0, 0, 2, 1], z + [1, 1, 0, 0]]
    assert (got.stats["unique_supports"], got.stats["poisoned"], got.stats["output"]) == (3, 0, 2)


@pytest.mark.parametrize("name,over,count,size", [("small", {}, 200, 2), ("small", {}, 120, 3),
                                                  ("core", dict(frontier_cap=4096), 200, 2),
                                                  ("mid", dict(frontier_cap=4096), 300, 2),
                                                  ("genome", dict(frontier_cap=4096), 300, 2)])
def test_poison_and_minimality_at_scale(efm, oracle_mod, name, over, count, size):
    """Multi-arc seed sets reach one support along several routes: the poison rule (a-6) and the drop branch of the
    minimality filter (a-7) both fire, on both sides, and the results stay bit-exact.  core / mid / genome have more
    than 112 arcs: the hashed-signature route with its sorted-list verification runs with true positives."""
    net = make_network(name, 0)
    seeds = random_seed_sets(net, count, size, 11)
    got, ref = assert_parity(efm, oracle_mod, net, seeds=seeds, **over)
    for st in (got.stats, ref.stats):
        assert int(st["poisoned"]) > 0
        if name != "mid":
            assert int(st["unique_supports"]) - int(st["poisoned"]) - int(st["output"]) > 0


@pytest.mark.parametrize("two_pass", [False, True])
def test_toy(efm, oracle_mod, two_pass):
    net = make_network("toy", 0)
    over = dict(frontier_cap=1 << 20) if two_pass else {}   # with a cap the threshold selection is enqueued on every level
    assert_parity(efm, oracle_mod, net, **over)
    assert_parity(efm, oracle_mod, net, seeds=oracle_mod.all_arc_seed_sets(net.reversible), **over)


def test_small(efm, oracle_mod):
    net = make_network("small", 0)
    got, _ = assert_parity(efm, oracle_mod, net)
    assert got.stats["direct_levels"] > 0 and got.stats["two_pass_levels"] == 0
    got, _ = assert_parity(efm, oracle_mod, net, frontier_cap=1 << 20)
    assert got.stats["two_pass_levels"] > 0 and got.stats["truncated_beam"] == 0


@pytest.mark.parametrize("cap", [300, 1000, 3918, 3919])
def test_small_beam(efm, oracle_mod, cap):
    """The beam binds (or just does not, at the peak frontier 3919): threshold selection must agree exactly."""
    net = make_network("small", 0)
    got, ref = assert_parity(efm, oracle_mod, net, frontier_cap=cap)
    assert (got.stats["truncated_beam"] > 0) == (cap < 3919)


def test_unimolecular_networks(efm, oracle_mod):
    for seed in range(12):
        net = unimolecular_network(seed, m_int=4 + seed % 4, n_rxn=7 + seed % 6, n_rev=seed % 3)
        assert_parity(efm, oracle_mod, net, seeds=oracle_mod.all_arc_seed_sets(net.reversible))


def test_core_full(efm, oracle_mod):
    net = make_network("core", 0)
    assert_parity(efm, oracle_mod, net)


@pytest.mark.parametrize("cap", [2048, 65536])
def test_core_beam(efm, oracle_mod, cap):
    net = make_network("core", 0)
    got, _ = assert_parity(efm, oracle_mod, net, frontier_cap=cap)
    assert got.stats["truncated_beam"] > 0


@pytest.mark.parametrize("cap", [512, 16384, 65536, 262144])
def test_mid(efm, oracle_mod, cap):
    net = make_network("mid", 0)
    got, _ = assert_parity(efm, oracle_mod, net, frontier_cap=cap)
    assert got.stats["truncated_beam"] > 0


@pytest.mark.parametrize("cap", [256, 4096, 16384])
def test_genome(efm, oracle_mod, cap):
    net = make_network("genome", 0)
    got, _ = assert_parity(efm, oracle_mod, net, frontier_cap=cap)
    assert got.stats["truncated_beam"] > 0 and got.stats["output"] > 1000


def test_genome_at_the_bench_configuration(efm, oracle_mod):
    """Element-by-element parity of the bench workload (genome seed 0) at the sweep point bench.PARITY_CAP, sized as the
    bench sizes it: the largest beam the oracle finishes in minutes on the box's host cores (about 2 ms per unit of cap)."""
    import bench
    net = make_network("genome", 0)
    sized = bench.sized_params(net.params, bench.PARITY_CAP)
    got, _ = assert_parity(efm, oracle_mod, net, **{k: v for k, v in sized.items() if k not in net.params or k == "frontier_cap"})
    assert got.stats["truncated_beam"] > 0 and got.stats["output"] > 100000


def _digest_cases():
    path = os.path.join(os.path.dirname(GOLDEN), "digests.json")
    with open(path) as fh:
        return json.load(fh)["cases"]


@pytest.mark.parametrize("case", _digest_cases(), ids=lambda c: f"{c['workload']}-{c['frontier_cap']}")
def test_digests_at_large_beams(efm, case):
    """The CUDA path against what the oracle returned at beams the oracle needs tens of minutes for (tests/golden/digests.json,
    written by tests/golden/make_digests.py from oracle/ alone): every counter, the per-level series, and SHA-256 of the
    canonical output rows (CSR, strict lexicographic order) and of their step counts."""
    import importlib.util
    import bench
    spec = importlib.util.spec_from_file_location("make_digests", os.path.join(os.path.dirname(GOLDEN), "make_digests.py"))
    md = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(md)
    net = make_network(case["workload"], case["generator_seed"])
    cap = case["frontier_cap"]
    assert dict(net.params, frontier_cap=cap) == case["params"]
    if case["workload"] == "genome":
        params = bench.sized_params(net.params, cap)
    else:   # capacity only (an overflow would be a loud EFM_E_CAPACITY): room for twice the balanced pathways the oracle counted
        params = dict(net.params, frontier_cap=cap, max_candidates=max(1 << 20, 2 * case["counters"]["done"]))
    en = efm.Enumerator(net.S, net.reversible, net.internal, params)
    res = en.enumerate(net.seed_sets, dense=False)
    for k, v in case["counters"].items():
        assert int(res.stats[k]) == v, (k, res.stats[k], v)
    assert int(res.stats["n_roots"]) == case["n_roots"]
    for k, v in case["levels"].items():
        assert res.levels[k].tolist() == v, k
    row_ptr, rxn, val = (t.numpy() for t in en.result_csr(pinned=False))
    got = md.digest_csr(row_ptr, rxn, val, res.steps)
    for k in ("rows", "nnz", "steps_sha256", "rows_sha256"):
        assert got[k] == case[k], k
    en.close()


def test_general_routine_only(efm, oracle_mod):
    """EFM_F_NO_FASTPATH sends every child through the warp-cooperative general routine: both routes must agree
    with the oracle (and hence with each other)."""
    for name, over in (("small", {}), ("core", dict(frontier_cap=2048)), ("genome", dict(frontier_cap=256))):
        assert_parity(efm, oracle_mod, make_network(name, 0), flags=efm.EFM_F_NO_FASTPATH, **over)
    assert_parity(efm, oracle_mod, make_network("small", 0), flags=efm.EFM_F_NO_FASTPATH, frontier_cap=1 << 20)


def test_parents_read_in_place(efm, oracle_mod):
    """EFM_F_NO_STAGING: every parent takes the route of entries larger than the staging buffer (read from HBM in
    place instead of from shared memory)."""
    for name, over in (("small", {}), ("core", dict(frontier_cap=2048)), ("genome", dict(frontier_cap=256))):
        assert_parity(efm, oracle_mod, make_network(name, 0), flags=efm.EFM_F_NO_STAGING, **over)


def test_other_seeds_of_the_generator(efm, oracle_mod):
    for name, seed, over in (("small", 1, {}), ("small", 2, dict(frontier_cap=500)), ("core", 1, dict(frontier_cap=4096)),
                             ("mid", 3, dict(frontier_cap=1024))):
        assert_parity(efm, oracle_mod, make_network(name, seed), **over)


def test_parameter_edges(efm, oracle_mod):
    net = make_network("small", 0)
    assert_parity(efm, oracle_mod, net, max_loop=1)
    assert_parity(efm, oracle_mod, net, max_support=6)
    assert_parity(efm, oracle_mod, net, max_visited=3)
    assert_parity(efm, oracle_mod, net, dep_depth=1)
    assert_parity(efm, oracle_mod, net, frontier_cap=1)
    assert_parity(efm, oracle_mod, net, frontier_cap=2, seeds=oracle_mod.all_arc_seed_sets(net.reversible))


def test_wide_columns_and_large_coefficients(efm, oracle_mod):
    """Reactions whose column has more than 6 internal metabolites, or a coefficient beyond 16 bits, do not fit the
    32-byte record of an OR-alternative: they are evaluated by the general routine."""
    prods = {f"P{t}": 1 + t % 3 for t in range(8)}
    rx = [({}, {"A": 1}, False), ({"A": 1}, prods, False), ({"A": 70000}, {"B": 3}, False), ({"B": 1}, {}, False),
          ({"A": 2}, {"B": 70001}, True)]
    rx += [({f"P{t}": 1}, {}, False) for t in range(8)]
    net = hand_network(rx, ["A", "B"] + [f"P{t}" for t in range(8)])
    got, ref = assert_parity(efm, oracle_mod, net, seeds=[[0]])
    assert ref.stats["output"] >= 2
    assert_parity(efm, oracle_mod, net, seeds=oracle_mod.all_arc_seed_sets(net.reversible))


def test_columns_longer_than_a_warp(efm, oracle_mod):
    """A reaction with 40 internal products: the column of its arc is longer than 32 entries (the route of
    k_materialise that scans the parent's list again) and every product becomes unbalanced at once."""
    names = ["A"] + [f"P{t}" for t in range(40)]
    rx = [({}, {"A": 1}, False), ({"A": 2}, {f"P{t}": 1 + t % 3 for t in range(40)}, False)]
    rx += [({f"P{t}": 1}, {}, False) for t in range(40)]
    rx += [({f"P{t}": 2, f"P{t + 1}": 1}, {"A": 1}, False) for t in range(0, 40, 8)]
    net = hand_network(rx, names)
    got, ref = assert_parity(efm, oracle_mod, net, seeds=[[0]])
    assert ref.stats["output"] >= 1 and ref.stats["expanded"] > 40
    assert_parity(efm, oracle_mod, net, seeds=[[0], [2], [2 * 41 + 2]])


def test_key_capacity_error(efm):
    """max_child_keys too small for a level: EFM_E_CAPACITY, never a silently truncated result."""
    net = make_network("genome", 0)
    with pytest.raises(efm.EfmError) as ei:   # a level of 32768 parents evaluates about half a million children
        efm.enumerate_network(net, frontier_cap=32768, max_child_keys=64)
    assert ei.value.code == efm.EFM_E_CAPACITY
    with pytest.raises(efm.EfmError) as ei:   # ... and sends thousands of them through the general routine
        efm.enumerate_network(net, frontier_cap=32768, max_child_tasks=16, flags=efm.EFM_F_NO_FASTPATH)
    assert ei.value.code == efm.EFM_E_CAPACITY


def test_overflow_guard(efm, oracle_mod):
    """Coefficient chains that multiply the scale past 2^62 (reading G21): both sides must discard identically."""
    names = [f"A{t}" for t in range(48)]
    rx = [({}, {names[0]: 1}, False)]
    for t in range(47):
        rx.append(({names[t]: 3}, {names[t + 1]: 1}, False))
    rx.append(({names[47]: 1}, {}, False))
    net = hand_network(rx, names)
    got, ref = assert_parity(efm, oracle_mod, net, seeds=[[0]])
    assert ref.stats["discarded_overflow"] > 0
    rx2 = [({}, {names[0]: 1}, False)]
    for t in range(30):
        rx2.append(({names[t]: 3}, {names[t + 1]: 2}, False))
    rx2.append(({names[30]: 1}, {}, False))
    got, ref = assert_parity(efm, oracle_mod, hand_network(rx2, names[:31]), seeds=[[0]])
    assert ref.stats["output"] == 1 and int(abs(ref.flux).max()) == 3 ** 30


def test_degenerate_inputs(efm, oracle_mod):
    # a seed that is balanced at once (all-external reaction) and a network without any internal metabolite
    net = hand_network([({"X": 1}, {"Y": 1}, False), ({}, {"A": 1}, False), ({"A": 1}, {}, False)], ["A"])
    assert_parity(efm, oracle_mod, net, seeds=[[0], [2]])
    net0 = hand_network([({"X": 1}, {"Y": 2}, True)], [])
    got = efm.enumerate_network(net0)
    assert got.n_out == 0 and got.stats["levels"] == 0
    for k in ("expanded", "children", "done", "dead_end", "algo_bytes", "unique_supports", "launches"):
        assert int(got.stats[k]) == 0, k          # no roots: nothing ran, nothing stale is reported
    got = efm.enumerate_network(net0, seed_sets=[[0], [1]])
    assert got.flux.tolist() == [[-1], [1]]
    # capacity errors are reported, never silently truncated
    net = make_network("small", 0)
    with pytest.raises(efm.EfmError) as ei:
        efm.enumerate_network(net, max_frontier=64)
    assert ei.value.code == efm.EFM_E_CAPACITY
    with pytest.raises(efm.EfmError) as ei:
        efm.enumerate_network(net, max_candidates=4)
    assert ei.value.code == efm.EFM_E_CAPACITY
    # the packed frontier buffer can be sized in bytes: too few bytes for the peak level is a capacity error as well,
    # enough bytes (far below entries x worst case) gives the same result
    with pytest.raises(efm.EfmError) as ei:
        efm.enumerate_network(net, max_frontier_bytes=64 * 1024)
    assert ei.value.code == efm.EFM_E_CAPACITY
    ref = efm.enumerate_network(net)
    got = efm.enumerate_network(net, max_frontier_bytes=4 << 20)
    assert np.array_equal(got.flux, ref.flux)


def test_sparse_and_dense_results_agree(efm):
    net = make_network("small", 0)
    en = efm.Enumerator(net.S, net.reversible, net.internal, net.params)
    res = en.enumerate()
    nnz, rxn, val = en.result_sparse()
    dense = np.zeros_like(res.flux)
    for r in range(res.n_out):
        dense[r, rxn[r, : nnz[r]]] = val[r, : nnz[r]]
    assert np.array_equal(dense, res.flux)
    row_ptr, crxn, cval = (t.numpy() for t in en.result_csr())
    assert row_ptr[0] == 0 and np.array_equal(np.diff(row_ptr), nnz)
    for r in range(res.n_out):
        assert np.array_equal(crxn[row_ptr[r]: row_ptr[r + 1]], rxn[r, : nnz[r]])
        assert np.array_equal(cval[row_ptr[r]: row_ptr[r + 1]], val[r, : nnz[r]])
    again = en.enumerate()   # the handle and the workspace are reusable
    assert np.array_equal(again.flux, res.flux)
    en.close()


def test_bench_configuration_properties(efm):
    """The bench workload at the sweep point bench.PROPERTY_CAP is too large for the oracle (about 2 ms per unit of cap),
    so it is held by what is true at any size: Def 2 on every output, canonical form, support-minimality and
    lexicographic order on samples, counter identities, and run-to-run determinism (the kernels allocate with atomics,
    the result must not depend on their order)."""
    import scipy.sparse as sp
    import bench
    cap = bench.PROPERTY_CAP
    net = make_network("genome", 0)
    params = bench.sized_params(net.params, cap)
    en = efm.Enumerator(net.S, net.reversible, net.internal, params)
    res = en.enumerate(net.seed_sets, dense=False)
    nnz, rxn, val = en.result_sparse()
    st, lv = res.stats, res.levels
    K, n = res.n_out, net.S.shape[1]
    assert K == int(st["output"]) > 100000 and st["truncated_beam"] > 0
    mask = np.arange(rxn.shape[1])[None, :] < nnz[:, None]
    rows = np.repeat(np.arange(K), nnz)
    V = sp.csr_matrix((val[mask], (rows, rxn[mask])), shape=(K, n), dtype=np.int64)
    # Def 2: S_int . v = 0, v >= 0 on irreversible reactions; gcd 1 (reading G10)
    Sint = sp.csr_matrix(net.S[net.internal.astype(bool)].astype(np.int64))
    assert (Sint @ V.T).count_nonzero() == 0
    assert np.all(val[mask][~net.reversible.astype(bool)[rxn[mask]]] > 0)
    assert np.all(val[mask] != 0) and np.all(np.diff(np.where(mask, rxn, n + np.arange(rxn.shape[1])[None, :]), axis=1) > 0)
    assert np.all(np.gcd.reduce(np.where(mask, np.abs(val), 0), axis=1) == 1)
    # strict lexicographic order on sampled neighbours
    rng = np.random.default_rng(0)
    for r in rng.choice(K - 1, 1000, replace=False):
        a, b = V[r].toarray()[0], V[r + 1].toarray()[0]
        d = np.nonzero(a != b)[0]
        assert d.size and a[d[0]] < b[d[0]], r
    # Def 3 on sampled outputs: no other output support strictly inside (arc space: sign matters)
    arcs = np.where(val[mask] > 0, rxn[mask], rxn[mask] + n)
    B = sp.csr_matrix((np.ones(arcs.size, np.int32), (rows, arcs)), shape=(K, 2 * n))
    size = np.asarray(B.sum(axis=1)).ravel()
    for r in rng.choice(K, 150, replace=False):
        shared = np.asarray((B @ B[r].T).todense()).ravel()
        inside = (shared == size) & (size < size[r])
        assert not inside.any(), (r, int(np.nonzero(inside)[0][0]))
    # counters
    assert int(st["expanded"]) == int(lv["expanded"].sum()) and int(st["children"]) == int(lv["children"].sum())
    assert int(st["done"]) == int(lv["done"].sum()) >= int(st["unique_supports"])
    assert int(st["unique_supports"]) - int(st["poisoned"]) >= K
    assert int(st["peak_frontier"]) == int(lv["active"].max()) and int(st["levels"]) == len(lv["active"])
    assert np.all(lv["expanded"] <= cap) and int(lv["expanded"].max()) > 0.9 * cap
    assert int(st["truncated_beam"]) == int(lv["active"].sum() - lv["expanded"].sum())
    # determinism
    again = en.enumerate(net.seed_sets, dense=False)
    nnz2, rxn2, val2 = en.result_sparse()
    assert again.n_out == K and np.array_equal(nnz, nnz2)
    assert np.array_equal(np.where(mask, rxn, 0), np.where(mask, rxn2, 0)) and np.array_equal(np.where(mask, val, 0), np.where(mask, val2, 0))
    for k in STAT_KEYS:
        assert int(again.stats[k]) == int(st[k]), k
    en.close()


# ---------------------------------------------------------------------------------------------------------------------
# SURVEY.md 8(f)-1 literal sampling mode and 8(f)-2 reaction mask
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,count,seed,over", [("toy", 48, 1, {}), ("small", 300, 5, {}), ("small", 7, 0, {}), ("core", 5000, 2, {}),
                                                  ("mid", 20000, 3, {}), ("genome", 30000, 4, {}),
                                                  ("genome", 2000, 9, dict(max_loop=2, max_visited=30))])
def test_sampling_mode(efm, oracle_mod, name, count, seed, over):
    """C candidate pathways, one sampled alternative per first visit: same pathways, same counters, and
    the same end (code, steps) of every single candidate as the oracle."""
    net = make_network(name, 0)
    got, ref = assert_parity(efm, oracle_mod, net, sample_count=count, sample_seed=seed, **over)
    assert got.cand_end.shape == (count, 2) and np.all(got.cand_end[:, 0] > 0)
    assert int(got.stats["children"]) <= int(got.stats["expanded"]) and int(got.stats["truncated_beam"]) == 0
    if name != "toy":
        assert len(set(got.cand_end[:, 0].tolist())) >= 3   # several kinds of ends occur


def test_sampling_mode_with_multi_arc_seed_sets_and_the_general_routine(efm, oracle_mod):
    net = make_network("core", 0)
    seeds = random_seed_sets(net, 64, 2, 3)
    assert_parity(efm, oracle_mod, net, seeds=seeds, sample_count=4000, sample_seed=11)
    assert_parity(efm, oracle_mod, net, seeds=seeds, sample_count=4000, sample_seed=11, flags=efm.EFM_F_NO_FASTPATH)


def test_reaction_mask_by_hand(efm):
    """P5 network (r0: ->A, r1: A<=>B, r2: B->, r3: ->B, r4: A->), seed r0, derived by hand (tests/test_oracle_modes.py has the
    derivation): no oracle involved."""
    net = hand_network([({}, {"A": 1}, False), ({"A": 1}, {"B": 1}, True), ({"B": 1}, {}, False), ({}, {"B": 1}, False),
                        ({"A": 1}, {}, False)], ["A", "B"])
    en = efm.Enumerator(net.S, net.reversible, net.internal, net.params)
    r = en.enumerate([[0]])
    assert r.flux.tolist() == [[1, 0, 0, 0, 1], [1, 1, 1, 0, 0]] and r.steps.tolist() == [1, 2]
    en.set_reaction_mask(np.array([1, 1, 1, 1, 0], np.uint8))
    r = en.enumerate([[0]])
    assert r.flux.tolist() == [[1, 1, 1, 0, 0]] and r.steps.tolist() == [2]
    en.set_reaction_mask(np.array([1, 0, 1, 1, 0], np.uint8))
    r = en.enumerate([[0]])
    assert r.flux.tolist() == [] and r.stats["dead_end"] == 1
    en.set_reaction_mask(None)
    r = en.enumerate([[0], [0, 8]])
    assert r.flux.tolist() == [[1, 0, 0, 0, 1], [1, 1, 1, 0, 0]] and r.steps.tolist() == [0, 2]   # quickest construction counts
    en.close()


@pytest.mark.parametrize("name,over", [("small", {}), ("core", dict(frontier_cap=4096)), ("genome", dict(frontier_cap=2048))])
def test_reaction_mask(efm, oracle_mod, name, over):
    """Random subsets of the reactions (8(f)-2): the restricted traversal agrees with the oracle, and the subset made of
    the reactions of one known output reconstructs that pathway."""
    net = make_network(name, 0)
    rng = np.random.default_rng(7)
    n = net.S.shape[1]
    for keep in (0.9, 0.6):
        allowed = (rng.random(n) < keep).astype(np.uint8)
        assert_parity(efm, oracle_mod, net, allowed=allowed, **over)
    full = efm.enumerate_network(net, **over)
    row = full.flux[len(full.flux) // 2]
    allowed = (row != 0).astype(np.uint8)
    got, ref = assert_parity(efm, oracle_mod, net, allowed=allowed, **over)
    assert any(np.array_equal(row, r) for r in got.flux)


def test_bench_headline_configuration_sampled(efm):
    """The configuration bench.py times by default (genome seed 0, frontier_cap bench.DEFAULT_CAP, 153 GB of workspace, or
    the next smaller power of two this GPU can hold): Def 2, gcd 1 and strict order on sampled outputs, counter identities."""
    import torch
    import bench
    net = make_network("genome", 0)
    cap = bench.DEFAULT_CAP
    while True:
        en = efm.Enumerator(net.S, net.reversible, net.internal, bench.sized_params(net.params, cap))
        try:
            res = en.enumerate(net.seed_sets, dense=False)
            break
        except (torch.cuda.OutOfMemoryError, efm.EfmError) as exc:
            en.close()
            # only "this GPU cannot hold the workspace" is a reason to go down a size (the rule of bench.py); a capacity
            # overflow of bench.sized_params or a kernel fault at the headline size must fail the test
            if isinstance(exc, efm.EfmError) and exc.code != efm.EFM_E_NOMEM:
                raise
            torch.cuda.empty_cache()
            assert cap > (1 << 20)
            cap //= 2
    free, total = torch.cuda.mem_get_info()
    if total > 170e9:
        assert cap == bench.DEFAULT_CAP, f"a full B200 holds the headline workspace; only cap {cap} ran"
    print(f"headline configuration verified at frontier_cap {cap}")
    st, lv = res.stats, res.levels
    K = res.n_out
    assert K == int(st["output"]) > cap // 2 and st["truncated_beam"] > 0
    row_ptr, rxn, val = (t.numpy() for t in en.result_csr(pinned=False))
    assert row_ptr[0] == 0 and row_ptr[-1] == len(rxn) and np.all(np.diff(row_ptr) > 0)
    Sint = net.S[net.internal.astype(bool)].astype(np.int64)
    irrev = ~net.reversible.astype(bool)
    rng = np.random.default_rng(1)
    prev = None
    for r in np.sort(rng.choice(K - 1, 4000, replace=False)):
        rows = []
        for q in (r, r + 1):
            j, v = rxn[row_ptr[q]: row_ptr[q + 1]], val[row_ptr[q]: row_ptr[q + 1]]
            assert np.all(np.diff(j) > 0) and np.all(v != 0) and np.gcd.reduce(np.abs(v)) == 1
            assert np.all(v[irrev[j]] > 0)                                  # Def 2: sign on irreversible reactions
            assert not np.any(Sint[:, j] @ v)                               # Def 2: S_int . v = 0
            d = np.zeros(net.S.shape[1], np.int64); d[j] = v
            rows.append(d)
        nz = np.nonzero(rows[0] != rows[1])[0]
        assert nz.size and rows[0][nz[0]] < rows[1][nz[0]], r               # strict lexicographic order
    assert int(st["expanded"]) == int(lv["expanded"].sum()) and int(st["children"]) == int(lv["children"].sum())
    assert int(st["done"]) == int(lv["done"].sum()) >= int(st["unique_supports"]) >= K
    assert np.all(lv["expanded"] <= cap) and int(lv["expanded"].max()) > 0.9 * cap
    assert int(st["truncated_beam"]) == int(lv["active"].sum() - lv["expanded"].sum())
    en.close()


# ---------------------------------------------------------------------------------------------------------------------
# SURVEY.md 8(f)-3 exact elementarity on the device
# ---------------------------------------------------------------------------------------------------------------------
def test_exact_elementarity_by_hand(efm):
    """H7 network, derived by hand in tests/test_oracle_modes.py: the balanced pathway (2,2,2,1) over all four reactions has
    nullity 2 (it is the sum of two EFMs) and goes; (1,1,0,0) and (0,0,2,1) stay.  No oracle involved."""
    net = hand_network([({}, {"A": 1}, False), ({"A": 1}, {}, False), ({}, {"B": 1}, False), ({"B": 2}, {}, False)], ["A", "B"])
    assert efm.enumerate_network(net, seed_sets=[[0, 4]]).flux.tolist() == [[2, 2, 2, 1]]
    r = efm.enumerate_network(net, seed_sets=[[0, 4]], flags=efm.EFM_F_EXACT_ELEMENTARITY)
    assert r.flux.tolist() == [] and r.stats["non_elementary"] == 1
    r = efm.enumerate_network(net, seed_sets=[[0, 4], [0], [4]], flags=efm.EFM_F_EXACT_ELEMENTARITY)
    assert r.flux.tolist() == [[0, 0, 2, 1], [1, 1, 0, 0]] and r.stats["non_elementary"] == 1


@pytest.mark.parametrize("name,over,count", [("toy", {}, 0), ("small", {}, 150), ("core", dict(frontier_cap=4096), 150),
                                             ("mid", dict(frontier_cap=4096), 300), ("genome", dict(frontier_cap=4096), 300),
                                             ("genome", dict(frontier_cap=16384), 0)])
def test_exact_elementarity(efm, oracle_mod, name, over, count):
    """Rank test instead of the pairwise filter: same pathways as the oracle's plain Gaussian elimination over the same
    field (supports of 1 to 60 arcs, one to two chunks of 32 lanes); with multi-arc seed sets the test rejects candidates."""
    net = make_network(name, 0)
    seeds = random_seed_sets(net, count, 2, 11) if count else "net"
    got, ref = assert_parity(efm, oracle_mod, net, seeds=seeds, flags=efm.EFM_F_EXACT_ELEMENTARITY, **over)
    if count:
        assert int(got.stats["non_elementary"]) > 0
    if net.n_arcs > 129:   # the basis of the rank test lives in shared memory: supports of at most 128 arcs
        with pytest.raises(efm.EfmError):
            efm.Enumerator(net.S, net.reversible, net.internal, dict(net.params, max_support=129), flags=efm.EFM_F_EXACT_ELEMENTARITY)


@pytest.mark.parametrize("len_a,len_b,D", [(70, 20, 96), (100, 24, 128)])
def test_exact_elementarity_three_and_four_chunks_by_hand(efm, oracle_mod, len_a, len_b, D):
    """k_rank_test<3> (D 65..96) and <4> (D 97..128) on supports that really are that wide: two disjoint chains of 71 / 101 and
    21 / 25 reactions.  Each chain is elementary; the pathway seeded on both heads is their sum (92 / 126 arcs, nullity 2) and
    goes.  Expected values are the closed form of the chain (tests/test_oracle_modes.py), then parity with the oracle."""
    from test_oracle_modes import chain_flux
    net = chain_pair_network(len_a, len_b, max_support=D)
    na = len_a + 1
    seeds = [[0], [2 * na], [0, 2 * na]]
    got = efm.enumerate_network(net, seed_sets=seeds, flags=efm.EFM_F_EXACT_ELEMENTARITY)
    assert got.flux.tolist() == sorted([chain_flux(len_a) + [0] * (len_b + 1), [0] * na + chain_flux(len_b)])
    assert (got.stats["unique_supports"], got.stats["non_elementary"], got.stats["output"]) == (3, 1, 2)
    assert_parity(efm, oracle_mod, net, seeds=seeds, flags=efm.EFM_F_EXACT_ELEMENTARITY)


@pytest.mark.parametrize("over", [dict(frontier_cap=2048, max_support=96), dict(frontier_cap=1024, max_support=128, max_visited=200)])
def test_exact_elementarity_three_and_four_chunks_on_genome(efm, oracle_mod, over):
    """The same two instantiations on the genome-scale network with multi-arc seed sets: thousands of candidate supports of
    up to D arcs, most of them rejected, on both sides."""
    net = make_network("genome", 0)
    seeds = random_seed_sets(net, 300, 2, 11)
    got, ref = assert_parity(efm, oracle_mod, net, seeds=seeds, flags=efm.EFM_F_EXACT_ELEMENTARITY, **over)
    assert int(got.stats["non_elementary"]) > 1000 and int(got.stats["output"]) > 100
    assert int((got.flux != 0).sum(axis=1).max()) > 64


# ---------------------------------------------------------------------------------------------------------------------
# SURVEY.md 8(c)-B key clamp and reading G23 under a binding support cap, on the device
# ---------------------------------------------------------------------------------------------------------------------
def test_more_than_255_unbalanced_metabolites(efm, oracle_mod):
    """netgen.wide_fan_network: entries with 300 - k unbalanced metabolites (key top byte clamped to 0xff) next to entries with
    200 - k, a beam of 40 that binds from level 5 on (tests/test_oracle_pins.py restates which entries stay)."""
    net = wide_fan_network()
    got, ref = assert_parity(efm, oracle_mod, net, seeds=[[0], [2]], frontier_cap=40, max_visited=7)
    assert int(got.stats["truncated_beam"]) > 0 and int(got.stats["discarded_visited"]) > 0
    assert_parity(efm, oracle_mod, net, seeds=[[0]], frontier_cap=16, max_visited=12)   # every key of every level has the top byte 0xff


def test_sampled_choice_under_a_binding_support_cap(efm, oracle_mod):
    """Reading G23 with D binding (hand-derived in tests/test_oracle_modes.py): r0 -> A, r1 A -> 3 B, r2 .. r6 B ->; seed set
    {r0, r3, r5}, max_support 4: the candidate chooses among r3 and r5 only.  No oracle needed for the expected row."""
    from test_oracle_modes import pick
    rx = [({}, {"A": 1}, False), ({"A": 1}, {"B": 3}, False)] + [({"B": 1}, {}, False) for _ in range(5)]
    net = hand_network(rx, ["A", "B"], max_support=4)
    for seed in range(24):
        got = efm.enumerate_network(net, seed_sets=[[0, 6, 10]], sample_count=1, sample_seed=seed)
        want = [1, 1, 0, 1, 0, 1, 0]
        want[[3, 5][pick(seed, 0, 1) % 2]] = 2
        assert got.flux.tolist() == [want], seed
        assert got.cand_end.tolist() == [[1, 2]]
    assert_parity(efm, oracle_mod, net, seeds=[[0, 6, 10], [0, 8]], sample_count=7, sample_seed=5)


# ---------------------------------------------------------------------------------------------------------------------
# SURVEY.md 8(f)-4 compression pre-pass
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,branches,over", [("toy", 3, {}), ("small", 4, {}), ("core", 12, dict(frontier_cap=4096)),
                                                ("genome", 200, dict(frontier_cap=4096))])
def test_compression_prepass(efm, oracle_mod, name, branches, over):
    """Networks with dead-end branches: with EFM_F_COMPRESS the library leaves the blocked reactions out of the graph and
    agrees with the oracle run on the network its own pre-pass reduced; results stay in the caller's reaction space."""
    net = with_dead_ends(make_network(name, 0), branches, 5)
    got, ref = assert_parity(efm, oracle_mod, net, flags=efm.EFM_F_COMPRESS, **over)
    assert int(got.stats["blocked_reactions"]) >= 2 * branches
    assert got.flux.shape[1] == net.S.shape[1] and not got.flux[:, -2 * branches:].any()
    plain = efm.enumerate_network(net, **over)
    assert int(plain.stats["blocked_reactions"]) == 0
    if not over:   # no beam: the pathways found do not depend on the pre-pass, the work does
        assert np.array_equal(plain.flux, got.flux) and int(got.stats["expanded"]) < int(plain.stats["expanded"])
    with pytest.raises(efm.EfmError):   # a seed on a removed reaction is refused
        efm.enumerate_network(net, flags=efm.EFM_F_COMPRESS, seed_sets=[[2 * (net.S.shape[1] - 1)]], **over)


# ---------------------------------------------------------------------------------------------------------------------
# differential test on random small networks: every mode, random parameters
# ---------------------------------------------------------------------------------------------------------------------
def _random_network(rng):
    m_int, m_ext, n = int(rng.integers(2, 9)), int(rng.integers(1, 4)), int(rng.integers(4, 15))
    m = m_int + m_ext
    S = np.zeros((m, n), dtype=np.int32)
    for j in range(n):
        rows = rng.choice(m, size=int(rng.integers(1, min(m, 4) + 1)), replace=False)
        for i in rows:
            S[i, j] = int(rng.choice([-3, -2, -1, -1, -1, 1, 1, 1, 2, 3]))
    rev = (rng.random(n) < 0.3).astype(np.uint8)
    internal = np.array([1] * m_int + [0] * m_ext, dtype=np.uint8)
    perm = rng.permutation(m)
    return S[perm], rev, internal[perm]


def test_random_small_networks_in_every_mode(efm, oracle_mod):
    """150 random networks (2-8 internal metabolites, 4-14 reactions, coefficients up to 3, random reversibility) with random
    parameters, seeds and modes (beam, sampling, reaction mask, exact elementarity, general routine only, no staging):
    the CUDA path and the oracle agree on pathways, steps and every counter."""
    from netgen.networks import Network
    rng = np.random.default_rng(2024)
    ran = {"beam": 0, "sample": 0, "mask": 0, "exact": 0, "outputs": 0}
    for t in range(150):
        S, rev, internal = _random_network(rng)
        A = int(S.shape[1] + rev.sum())
        D = int(rng.integers(2, A + 1))
        params = dict(max_support=D, max_loop=int(rng.integers(1, 9)), dep_depth=int(rng.integers(1, 6)),
                      max_visited=int(rng.integers(1, 2 * D + 1)), frontier_cap=0)
        net = Network(f"random-{t}", t, S, rev, internal, params, None, {})
        mode = t % 5
        over, flags, allowed = {}, 0, None
        seeds = oracle_mod.all_arc_seed_sets(rev) if t % 2 else "net"
        if mode == 1:
            over["frontier_cap"] = int(rng.integers(1, 40)); ran["beam"] += 1
        elif mode == 2:
            over.update(sample_count=int(rng.integers(1, 60)), sample_seed=int(rng.integers(0, 1 << 30))); ran["sample"] += 1
        elif mode == 3:
            allowed = (rng.random(S.shape[1]) < 0.8).astype(np.uint8); ran["mask"] += 1
        elif mode == 4:
            flags |= efm.EFM_F_EXACT_ELEMENTARITY; ran["exact"] += 1
        if t % 7 == 0:
            flags |= efm.EFM_F_NO_FASTPATH
        if t % 11 == 0:
            flags |= efm.EFM_F_NO_STAGING
        got, ref = assert_parity(efm, oracle_mod, net, seeds=seeds, flags=flags, allowed=allowed, **over)
        ran["outputs"] += got.n_out
    assert min(ran["beam"], ran["sample"], ran["mask"], ran["exact"]) >= 30 and ran["outputs"] > 300
