"""CPU-side checks of the CUDA library: it builds, loads, exports the C ABI of include/efm_b200.h, its host-side
graph builder agrees with the oracle's graph, seeds are validated, and without a GPU the
product path fails loudly instead of falling back to anything."""
import ctypes
import os

import numpy as np
import pytest

from netgen import hand_network, make_network


@pytest.fixture(scope="module")
def lib_mod():
    from paper_1804_02867_b200 import build
    build.build()
    import paper_1804_02867_b200 as efm
    efm.load()
    return efm


def test_exports_every_declared_symbol(lib_mod):
    lib = lib_mod.load()
    names = lib_mod.exported_symbols()
    assert len(names) >= 15
    for name in names:
        assert hasattr(lib, name), name
    assert lib.efm_strerror(0) == b"ok"
    assert b"capacity" in lib.efm_strerror(lib_mod.EFM_E_CAPACITY)


def test_struct_sizes_match_header(lib_mod, tmp_path):
    """The ctypes mirrors of efm_params / efm_stats have the sizes a C compiler gives the header's structs."""
    import subprocess
    src = tmp_path / "sz.c"
    src.write_text('#include <stdio.h>\n#include "efm_b200.h"\nint main(void) { printf("%zu %zu\\n", sizeof(efm_params), sizeof(efm_stats)); return 0; }\n')
    exe = tmp_path / "sz"
    subprocess.run(["gcc", "-I", os.path.dirname(lib_mod.HEADER_PATH), str(src), "-o", str(exe)], check=True)
    c_params, c_stats = (int(x) for x in subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split())
    assert ctypes.sizeof(lib_mod.efm_params) == c_params == 88
    assert ctypes.sizeof(lib_mod.efm_stats) == c_stats


@pytest.mark.parametrize("name", ["toy", "small", "core", "mid", "genome"])
def test_graph_builder_matches_oracle_graph(lib_mod, oracle_mod, name):
    """Two independent builders (library: counting sort + 64-way bit-parallel reachability; oracle: dense scans + seen array) must
    produce the same MG graph and the same dependency table."""
    net = make_network(name, 0)
    en = lib_mod.Enumerator(net.S, net.reversible, net.internal, net.params)
    g = en.graph_export()
    en.close()
    ref = oracle_mod.enumerate_network(net, export_graph=True, self_check=False, frontier_cap=4, max_support=2).graph
    for k in ("M", "A", "W"):
        assert g[k] == ref[k], k
    for k in ("arc_rxn", "arc_dir", "twin", "in_ptr", "in_arc", "in_c", "out_ptr", "out_arc", "out_c", "col_ptr",
              "col_met", "col_s", "dep_off", "dep"):
        assert np.array_equal(g[k], ref[k]), k
    assert g["dep"].sum() > 0


def test_dep_depth_is_respected(lib_mod, oracle_mod):
    net = make_network("small", 0)
    sums = []
    for L in (1, 2, 3, 5):
        params = dict(net.params, dep_depth=L)
        en = lib_mod.Enumerator(net.S, net.reversible, net.internal, params)
        g = en.graph_export()
        en.close()
        ref = oracle_mod.enumerate_pathways(net.S, net.reversible, net.internal, dict(params, frontier_cap=2, max_support=2),
                                            export_graph=True, self_check=False).graph
        assert np.array_equal(g["dep"], ref["dep"])
        sums.append(int(g["dep"].sum()))
    assert sums[0] == 0 and sums == sorted(sums) and sums[-1] > sums[1]


def test_create_rejects_bad_input(lib_mod):
    net = make_network("toy", 0)
    lib = lib_mod.load()
    h = ctypes.c_void_p()
    S = np.ascontiguousarray(net.S)
    rev, internal = net.reversible, net.internal
    ptr = lambda a: a.ctypes.data_as(ctypes.c_void_p)
    assert lib.efm_create(None, net.m, net.n, net.n, ptr(rev), ptr(internal), None, ctypes.byref(h)) == lib_mod.EFM_E_INVAL
    assert lib.efm_create(ptr(S), 0, net.n, net.n, ptr(rev), ptr(internal), None, ctypes.byref(h)) == lib_mod.EFM_E_INVAL
    assert lib.efm_create(ptr(S), net.m, net.n, net.n - 1, ptr(rev), ptr(internal), None, ctypes.byref(h)) == lib_mod.EFM_E_INVAL
    p = lib_mod.efm_params(max_support=-1)
    assert lib.efm_create(ptr(S), net.m, net.n, net.n, ptr(rev), ptr(internal), ctypes.byref(p), ctypes.byref(h)) == lib_mod.EFM_E_INVAL
    assert lib.efm_create(ptr(S), net.m, net.n, net.n, ptr(rev), ptr(internal), None, ctypes.byref(h)) == 0
    k = ctypes.c_int64()
    assert lib.efm_result_count(h, ctypes.byref(k)) == lib_mod.EFM_E_STATE
    lib.efm_destroy(h)


def test_seed_validation_and_no_cpu_fallback(lib_mod):
    """Bad seed sets are rejected before any CUDA call; a valid call on a box without a GPU fails with EFM_E_CUDA
    (nothing in the product path computes on the CPU)."""
    import torch
    net = make_network("toy", 0)
    en = lib_mod.Enumerator(net.S, net.reversible, net.internal, net.params)
    j_rev = int(np.nonzero(net.reversible)[0][0])
    j_irr = int(np.nonzero(net.reversible == 0)[0][0])
    need = en.workspace_bytes()
    assert need > 0
    fake = 1 << 20  # never dereferenced on the failing paths
    for bad in ([[2 * j_rev, 2 * j_rev + 1]], [[2 * j_irr + 1]], [[2 * net.n]], [[0, 0]], [[-1]]):
        with pytest.raises(lib_mod.EfmError) as ei:
            en.enumerate_raw(bad, fake, need)
        assert ei.value.code == lib_mod.EFM_E_INVAL
    with pytest.raises(lib_mod.EfmError) as ei:
        en.enumerate_raw(None, fake, need - 1)
    assert ei.value.code == lib_mod.EFM_E_NOMEM
    if not torch.cuda.is_available():
        with pytest.raises(lib_mod.EfmError) as ei:
            en.enumerate_raw(None, fake, need)
        assert ei.value.code == lib_mod.EFM_E_CUDA
        with pytest.raises(lib_mod.EfmError):
            en.enumerate()
    en.close()


def test_workspace_scales_with_capacity(lib_mod):
    net = make_network("core", 0)
    sizes = []
    for cap in (1 << 10, 1 << 14, 1 << 18):
        en = lib_mod.Enumerator(net.S, net.reversible, net.internal, dict(net.params, frontier_cap=cap, max_candidates=1 << 12))
        sizes.append(en.workspace_bytes())
        en.close()
    assert sizes[0] < sizes[1] < sizes[2]
