"""CPU oracle for the AND/OR-graph pathway traversal of arXiv 1804.02867 -- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It shares no code with ``paper_1804_02867_b200`` (the CUDA library) and
never imports it.  ``efm_oracle.c`` is the plain-C step-by-step procedure (SURVEY.md 8(c) O1-O9 + beam B);
``check.py`` is the O9 self-check run on every output; ``brute_force.py`` enumerates all EFMs of tiny
networks by subset enumeration (pin P9).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import Dict, List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "efm_oracle.c")
_LIB = os.path.join(_HERE, "liboracle_efm.so")


def build(force: bool = False) -> str:
    """Compile efm_oracle.c with gcc (OpenMP over the entries of a level)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


END_CODES = {0: "none", 1: "done", 2: "not_efm_maxloop", 3: "dead_end", 4: "visited_cap", 5: "nonpos", 6: "overflow"}


class _Params(ctypes.Structure):
    _fields_ = [("max_support", ctypes.c_int32), ("max_loop", ctypes.c_int32), ("dep_depth", ctypes.c_int32),
                ("max_visited", ctypes.c_int32), ("frontier_cap", ctypes.c_int64), ("threads", ctypes.c_int32),
                ("trace", ctypes.c_int32), ("shuffle_seed", ctypes.c_uint64), ("sample_count", ctypes.c_int32),
                ("exact", ctypes.c_int32), ("sample_seed", ctypes.c_uint64), ("allowed", ctypes.c_void_p)]


STAT_FIELDS = ["levels", "expanded", "children", "done", "dead_end", "not_efm_maxloop", "discarded_nonpos",
               "discarded_overflow", "discarded_visited", "truncated_beam", "unique_supports", "poisoned",
               "output", "peak_frontier", "algo_bytes", "non_elementary"]


class _Stats(ctypes.Structure):
    _fields_ = [(k, ctypes.c_int64) for k in STAT_FIELDS]


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.oracle_enumerate.restype = ctypes.c_int
        lib.oracle_enumerate.argtypes = [ctypes.c_void_p, ctypes.c_int32, ctypes.c_int32, ctypes.c_void_p,
                                         ctypes.c_void_p, ctypes.POINTER(_Params), ctypes.c_void_p,
                                         ctypes.c_void_p, ctypes.c_int32, ctypes.POINTER(ctypes.c_void_p)]
        lib.oracle_result_count.restype = ctypes.c_int64
        lib.oracle_result_count.argtypes = [ctypes.c_void_p]
        lib.oracle_result_copy.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
        lib.oracle_result_stats.argtypes = [ctypes.c_void_p, ctypes.POINTER(_Stats)]
        lib.oracle_result_levels.restype = ctypes.c_int64
        lib.oracle_result_levels.argtypes = [ctypes.c_void_p] + [ctypes.c_void_p] * 4 + [ctypes.c_int64]
        lib.oracle_result_roots.restype = ctypes.c_int32
        lib.oracle_result_roots.argtypes = [ctypes.c_void_p]
        lib.oracle_graph_info.argtypes = [ctypes.c_void_p] + [ctypes.c_void_p] * 5
        lib.oracle_graph_export.argtypes = [ctypes.c_void_p] + [ctypes.c_void_p] * 14
        lib.oracle_result_free.argtypes = [ctypes.c_void_p]
        lib.oracle_result_steps.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
        lib.oracle_result_cand_end.restype = ctypes.c_int64
        lib.oracle_result_cand_end.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64]
        lib.oracle_result_trace.restype = ctypes.c_int64
        lib.oracle_result_trace.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64]
        lib.oracle_state_hash.restype = ctypes.c_uint64
        lib.oracle_state_hash.argtypes = [ctypes.c_int32, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int32,
                                          ctypes.c_void_p]
        lib.oracle_max_threads.restype = ctypes.c_int32
        lib.oracle_mix64.restype = ctypes.c_uint64
        lib.oracle_mix64.argtypes = [ctypes.c_uint64]
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(_load().oracle_max_threads())


@dataclass
class OracleResult:
    flux: np.ndarray  # int64 [n_out, n], reaction space, coprime, lexicographic order
    stats: Dict[str, int]
    levels: Dict[str, np.ndarray]  # per level: active, done, expanded, children
    n_roots: int
    graph: Optional[Dict[str, np.ndarray]] = None
    # test hook (trace=True): per level the list of entries as dicts
    # {flux: {arc: f}, visited: {met: (PI, PO, cnt)}, n_unb, istar, key, kept}
    trace: Optional[List[List[dict]]] = None
    steps: Optional[np.ndarray] = None      # per output row: expansions that built the pathway
    cand_end: Optional[np.ndarray] = None   # sampling mode (8(f)-1): per candidate (code, steps); codes in END_CODES
    blocked: Optional[np.ndarray] = None    # enumerate_compressed: reactions the pre-pass removed


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def enumerate_pathways(S: np.ndarray, reversible: np.ndarray, internal: np.ndarray, params: Dict[str, int],
                       seed_sets: Optional[Sequence[Sequence[int]]] = None, threads: int = 1,
                       shuffle_seed: int = 0, export_graph: bool = False,
                       self_check: bool = True, trace: bool = False, sample_count: int = 0, sample_seed: int = 0,
                       allowed: Optional[np.ndarray] = None, exact: bool = False) -> OracleResult:
    """Run the oracle.  ``seed_sets`` holds arc codes 2*j + (dir < 0); None = default boundary arcs (O2)."""
    lib = _load()
    S = np.ascontiguousarray(S, dtype=np.int32)
    rev = np.ascontiguousarray(reversible, dtype=np.uint8)
    internal = np.ascontiguousarray(internal, dtype=np.uint8)
    m, n = S.shape
    p = _Params(int(params.get("max_support", 0)), int(params.get("max_loop", 8)), int(params.get("dep_depth", 4)),
                int(params.get("max_visited", 0)), int(params.get("frontier_cap", 0)), int(threads), int(trace),
                int(shuffle_seed), int(sample_count), int(bool(exact)), int(sample_seed) & ((1 << 64) - 1), None)
    if allowed is not None:
        allowed = np.ascontiguousarray(allowed, dtype=np.uint8)
        assert allowed.shape == (n,)
        p.allowed = allowed.ctypes.data
    if seed_sets:
        ptr = np.zeros(len(seed_sets) + 1, dtype=np.int32)
        ptr[1:] = np.cumsum([len(s) for s in seed_sets])
        codes = np.array([c for s in seed_sets for c in s], dtype=np.int32)
        n_sets = len(seed_sets)
    else:
        ptr = np.zeros(1, dtype=np.int32)
        codes = np.zeros(1, dtype=np.int32)
        n_sets = 0
    handle = ctypes.c_void_p()
    rc = lib.oracle_enumerate(_ptr(S), m, n, _ptr(rev), _ptr(internal), ctypes.byref(p), _ptr(ptr), _ptr(codes),
                              n_sets, ctypes.byref(handle))
    try:
        if rc != 0:
            raise ValueError(f"oracle_enumerate: invalid input (code {rc})")
        k = lib.oracle_result_count(handle)
        flux = np.zeros((k, n), dtype=np.int64)
        if k:
            lib.oracle_result_copy(handle, _ptr(flux))
        st = _Stats()
        lib.oracle_result_stats(handle, ctypes.byref(st))
        stats = {f: int(getattr(st, f)) for f in STAT_FIELDS}
        nl = int(stats["levels"])
        arrs = [np.zeros(max(nl, 1), dtype=np.int64) for _ in range(4)]
        lib.oracle_result_levels(handle, *[_ptr(a) for a in arrs], nl)
        levels = dict(active=arrs[0][:nl], done=arrs[1][:nl], expanded=arrs[2][:nl], children=arrs[3][:nl])
        graph = None
        if export_graph:
            M, A, W = ctypes.c_int32(), ctypes.c_int32(), ctypes.c_int32()
            nnz, depb = ctypes.c_int64(), ctypes.c_int64()
            lib.oracle_graph_info(handle, ctypes.byref(M), ctypes.byref(A), ctypes.byref(W), ctypes.byref(nnz),
                                  ctypes.byref(depb))
            M, A, W, nnz, depb = M.value, A.value, W.value, nnz.value, depb.value
            g = dict(
                arc_rxn=np.zeros(A, np.int32), arc_dir=np.zeros(A, np.int32), twin=np.zeros(A, np.int32),
                in_ptr=np.zeros(M + 1, np.int32), in_arc=np.zeros(nnz, np.int32), in_c=np.zeros(nnz, np.int64),
                out_ptr=np.zeros(M + 1, np.int32), out_arc=np.zeros(nnz, np.int32), out_c=np.zeros(nnz, np.int64),
                col_ptr=np.zeros(A + 1, np.int32), col_met=np.zeros(nnz, np.int32), col_s=np.zeros(nnz, np.int64),
                dep_off=np.zeros(M + 1, np.int64), dep=np.zeros(max(depb, 1), np.uint8))
            order = ["arc_rxn", "arc_dir", "twin", "in_ptr", "in_arc", "in_c", "out_ptr", "out_arc", "out_c",
                     "col_ptr", "col_met", "col_s", "dep_off", "dep"]
            lib.oracle_graph_export(handle, *[_ptr(g[k2]) for k2 in order])
            g["in_arc"] = g["in_arc"][: g["in_ptr"][-1]]
            g["in_c"] = g["in_c"][: g["in_ptr"][-1]]
            g["out_arc"] = g["out_arc"][: g["out_ptr"][-1]]
            g["out_c"] = g["out_c"][: g["out_ptr"][-1]]
            g["dep"] = g["dep"][:depb]
            g.update(M=M, A=A, W=W)
            graph = g
        n_roots = int(lib.oracle_result_roots(handle))
        steps = np.zeros(k, dtype=np.int64)
        if k:
            lib.oracle_result_steps(handle, _ptr(steps))
        cand_end = None
        if sample_count > 0:
            raw = np.zeros(max(n_roots, 1), dtype=np.int64)
            lib.oracle_result_cand_end(handle, _ptr(raw), n_roots)
            cand_end = np.stack([raw[:n_roots] & 0xff, raw[:n_roots] >> 8], axis=1)
        tr = None
        if trace:
            nt = int(lib.oracle_result_trace(handle, None, 0))
            buf = np.zeros(max(nt, 1), dtype=np.int64)
            lib.oracle_result_trace(handle, _ptr(buf), nt)
            tr = [[] for _ in range(nl)]
            x = 0
            while x < nt:
                lvl, ns, nv, nu, istar, key, kept = (int(v) for v in buf[x:x + 7])
                x += 7
                fl = {int(buf[x + 2 * k]): int(buf[x + 2 * k + 1]) for k in range(ns)}
                x += 2 * ns
                vis = {int(buf[x + 4 * k]): tuple(int(v) for v in buf[x + 4 * k + 1:x + 4 * k + 4]) for k in range(nv)}
                x += 4 * nv
                tr[lvl].append(dict(flux=fl, visited=vis, n_unb=nu, istar=istar, key=key & ((1 << 64) - 1), kept=bool(kept)))
    finally:
        lib.oracle_result_free(handle)
    res = OracleResult(flux, stats, levels, n_roots, graph, tr, steps, cand_end)
    if self_check:
        from .check import check_outputs
        check_outputs(S, rev, internal, flux)
    return res


def enumerate_network(net, threads: int = 1, shuffle_seed: int = 0, export_graph: bool = False,
                      self_check: bool = True, seed_sets="net", trace: bool = False, sample_count: int = 0,
                      sample_seed: int = 0, allowed: Optional[np.ndarray] = None, exact: bool = False,
                      **param_overrides) -> OracleResult:
    """Run the oracle on a ``netgen.Network`` with its own parameters (optionally overridden).

    ``seed_sets="net"`` uses the network's own seed sets (None there = default boundary arcs)."""
    params = dict(net.params)
    params.update(param_overrides)
    seeds = net.seed_sets if isinstance(seed_sets, str) else seed_sets
    return enumerate_pathways(net.S, net.reversible, net.internal, params, seeds, threads, shuffle_seed,
                              export_graph, self_check, trace, sample_count, sample_seed, allowed, exact)


def enumerate_compressed(S: np.ndarray, reversible: np.ndarray, internal: np.ndarray, params: Dict[str, int],
                         seed_sets: Optional[Sequence[Sequence[int]]] = None, **kw) -> OracleResult:
    """the traversal after the compression pre-pass of oracle/compress.py.  The blocked reactions are
    removed from S (the arcs of the others are numbered consecutively, as always), seed codes are renumbered, and the
    pathways are returned in the caller's reaction space (zero on the removed reactions)."""
    from .compress import blocked_reactions
    S = np.asarray(S)
    blocked = blocked_reactions(S, reversible, internal)
    keep = np.nonzero(~blocked)[0]
    new_id = -np.ones(S.shape[1], dtype=np.int64)
    new_id[keep] = np.arange(len(keep))
    seeds = None
    if seed_sets:
        seeds = []
        for st in seed_sets:
            if any(blocked[c // 2] for c in st):
                raise ValueError("seed on a blocked reaction")
            seeds.append([int(2 * new_id[c // 2] + (c & 1)) for c in st])
    res = enumerate_pathways(np.ascontiguousarray(S[:, keep]), np.asarray(reversible)[keep], internal, params, seeds, **kw)
    full = np.zeros((res.flux.shape[0], S.shape[1]), dtype=np.int64)
    full[:, keep] = res.flux
    res.flux = full
    res.blocked = blocked
    return res


def state_hash(arcs: Sequence[int], fluxes: Sequence[int], visited: Sequence[Sequence[int]]) -> int:
    """h of beam B for an explicit state; visited rows are (met, PI, PO, cnt)."""
    lib = _load()
    a = np.array(list(arcs), dtype=np.int32)
    f = np.array(list(fluxes), dtype=np.int64)
    v = np.array([x for row in visited for x in row], dtype=np.int32)
    if v.size == 0:
        v = np.zeros(4, dtype=np.int32)
    return int(lib.oracle_state_hash(len(a), _ptr(a), _ptr(f), len(visited), _ptr(v)))


def mix64(x: int) -> int:
    return int(_load().oracle_mix64(ctypes.c_uint64(x & ((1 << 64) - 1))))


def all_arc_seed_sets(reversible: np.ndarray) -> List[List[int]]:
    """One seed set per arc (pins P7, P9)."""
    out: List[List[int]] = []
    for j, r in enumerate(reversible):
        out.append([2 * j])
        if r:
            out.append([2 * j + 1])
    return out
