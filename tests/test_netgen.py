"""The seeded generator reproduces the shapes BASELINE.json names and is deterministic."""
import numpy as np
import pytest

from netgen import CONFIGS, make_network

SHAPES = {"toy": (6, 3, 10, 3), "small": (20, 6, 32, 6), "core": (72, 20, 95, 24),
          "mid": (250, 40, 350, 88), "genome": (1000, 150, 2000, 600)}


@pytest.mark.parametrize("name", list(CONFIGS))
def test_shapes(name):
    net = make_network(name, 0)
    mi, me, n, nrev = SHAPES[name]
    assert net.S.shape == (mi + me, n) and net.S.dtype == np.int32
    assert int(net.internal.sum()) == mi and int(net.reversible.sum()) == nrev
    assert not np.any((net.S != 0).sum(axis=0) == 0)
    coefs = np.abs(net.S[net.S != 0])
    assert coefs.max() <= (2 if name == "toy" else 3)
    side_max = CONFIGS[name].side_max
    assert ((net.S < 0).sum(axis=0) <= side_max + 1).all() and ((net.S > 0).sum(axis=0) <= side_max + 1).all()
    again = make_network(name, 0)
    assert np.array_equal(net.S, again.S) and np.array_equal(net.reversible, again.reversible)
    assert not np.array_equal(net.S, make_network(name, 1).S)


def test_hubs_and_targets():
    net = make_network("genome", 0)
    deg = (net.S[net.internal.astype(bool)] != 0).sum(axis=1)
    top = np.sort(deg)[-20:]
    assert top.min() >= 100 and top.max() <= 320
    assert net.seed_sets is not None and 8 <= len(net.seed_sets) <= 16
    core = make_network("core", 0)
    deg = (core.S[core.internal.astype(bool)] != 0).sum(axis=1)
    assert np.sort(deg)[-5:].min() >= 25
