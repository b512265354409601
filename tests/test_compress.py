"""SURVEY.md 8(f)-4, compression pre-pass: the library's host routine against the oracle-side restatement,
and the restatement against what the mathematics fixes (a blocked reaction has zero flux in every EFM; removing blocked
reactions does not change what the exhaustive traversal finds)."""
import numpy as np
import pytest

from netgen import hand_network, make_network, with_dead_ends
from oracle.compress import blocked_reactions as oracle_blocked


@pytest.fixture(scope="module")
def lib_mod():
    from paper_1804_02867_b200 import build
    build.build()
    import paper_1804_02867_b200 as efm
    efm.load()
    return efm


def test_blocked_by_hand():
    """r0: ->A, r1: A->B, r2: B->, r3: A->C, r4: C->D (nothing consumes D): D has only a producer, so r4 is blocked; then C
    has only the producer r3: blocked by cascade.  r5: A<=>E is the only reaction at E: blocked although reversible."""
    rx = [({}, {"A": 1}, False), ({"A": 1}, {"B": 1}, False), ({"B": 1}, {}, False), ({"A": 1}, {"C": 1}, False),
          ({"C": 1}, {"D": 1}, False), ({"A": 1}, {"E": 1}, True)]
    net = hand_network(rx, ["A", "B", "C", "D", "E"])
    assert oracle_blocked(net.S, net.reversible, net.internal).tolist() == [False, False, False, True, True, True]
    # two reversible reactions at a metabolite can balance each other: nothing is blocked
    net = hand_network([({"X": 1}, {"A": 1}, True), ({"A": 1}, {"Y": 1}, True)], ["A"])
    assert not oracle_blocked(net.S, net.reversible, net.internal).any()
    # two producers and no consumer
    net = hand_network([({}, {"A": 1}, False), ({"X": 1}, {"A": 2}, False)], ["A"])
    assert oracle_blocked(net.S, net.reversible, net.internal).all()


def test_blocked_reactions_carry_no_flux_in_any_efm():
    """Brute-force EFM enumeration on random small networks: every reaction the pre-pass removes is zero in every EFM."""
    from oracle.brute_force import brute_force_efms
    rng = np.random.default_rng(3)
    seen_blocked = 0
    for _ in range(60):
        m, n = int(rng.integers(2, 6)), int(rng.integers(3, 9))
        S = rng.choice([-2, -1, 0, 0, 0, 1, 1], size=(m, n)).astype(np.int32)
        rev = (rng.random(n) < 0.3).astype(np.uint8)
        internal = np.ones(m, np.uint8)
        b = oracle_blocked(S, rev, internal)
        seen_blocked += int(b.sum())
        for v in brute_force_efms(S, rev, internal):
            assert all(v[j] == 0 for j in np.nonzero(b)[0])
    assert seen_blocked > 20


def test_library_routine_equals_the_restatement(lib_mod):
    rng = np.random.default_rng(0)
    for _ in range(300):
        m, n = int(rng.integers(2, 9)), int(rng.integers(2, 12))
        S = rng.choice([-2, -1, 0, 0, 0, 1, 1, 3], size=(m, n)).astype(np.int32)
        rev = (rng.random(n) < 0.3).astype(np.uint8)
        internal = (rng.random(m) < 0.8).astype(np.uint8)
        assert np.array_equal(lib_mod.blocked_reactions(S, rev, internal), oracle_blocked(S, rev, internal))
    for name in ("toy", "small", "core", "mid"):
        net = with_dead_ends(make_network(name, 0), 7, 1)
        b = lib_mod.blocked_reactions(net.S, net.reversible, net.internal)
        assert np.array_equal(b, oracle_blocked(net.S, net.reversible, net.internal))
        assert b[-14:].all()          # both reactions of every dead-end branch


def test_compression_does_not_change_the_exhaustive_result(oracle_mod):
    """Without a beam the traversal through a blocked reaction can only end in dead ends and discards: the pathways found on
    the compressed network are the pathways found on the full one."""
    for name, cnt in (("toy", 3), ("small", 4)):
        net = with_dead_ends(make_network(name, 0), cnt, 2)
        full = oracle_mod.enumerate_pathways(net.S, net.reversible, net.internal, net.params, net.seed_sets)
        comp = oracle_mod.enumerate_compressed(net.S, net.reversible, net.internal, net.params, net.seed_sets)
        assert comp.blocked.sum() >= 2 * cnt
        assert np.array_equal(full.flux, comp.flux)
        assert comp.stats["expanded"] < full.stats["expanded"]
