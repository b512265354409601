"""B200-native AND/OR-graph pathway traversal (arXiv 1804.02867) -- thin Python binding of ``libefm_b200.so``.

Argument marshalling only: every step of the path (roots, classify, beam select, expand, support dedup,
minimality filter, canonical output) runs in the CUDA kernels behind the C ABI declared in
``include/efm_b200.h``.  PyTorch is used for device memory (the workspace tensor) and the stream.
There is no CPU fallback: without the built library ``load()`` raises, without a CUDA device
``Enumerator.enumerate`` raises.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Dict, List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libefm_b200.so")
HEADER_PATH = os.path.join(os.path.dirname(_HERE), "include", "efm_b200.h")

EFM_OK, EFM_E_INVAL, EFM_E_NOMEM, EFM_E_CAPACITY, EFM_E_CUDA, EFM_E_STATE = 0, -1, -2, -3, -4, -5
EFM_F_TIMING, EFM_F_NO_FASTPATH, EFM_F_NO_STAGING, EFM_F_EXACT_ELEMENTARITY, EFM_F_COMPRESS = 0x1, 0x4, 0x8, 0x10, 0x20


class efm_params(ctypes.Structure):
    _fields_ = [("max_support", ctypes.c_int32), ("max_loop", ctypes.c_int32), ("dep_depth", ctypes.c_int32),
                ("max_visited", ctypes.c_int32), ("frontier_cap", ctypes.c_int64), ("max_frontier", ctypes.c_int64),
                ("max_candidates", ctypes.c_int64), ("max_child_keys", ctypes.c_int64), ("device", ctypes.c_int32),
                ("flags", ctypes.c_uint32), ("max_frontier_bytes", ctypes.c_int64), ("max_child_tasks", ctypes.c_int64),
                ("sample_count", ctypes.c_int64), ("sample_seed", ctypes.c_uint64)]


_STAT_INT = ["levels", "expanded", "children", "done", "dead_end", "not_efm_maxloop", "discarded_nonpos",
             "discarded_overflow", "discarded_visited", "truncated_beam", "unique_supports", "poisoned", "output",
             "peak_frontier", "algo_bytes", "n_roots", "launches", "two_pass_levels", "direct_levels", "h2d_bytes",
             "host_syncs"]
_STAT_MS = ["ms_build", "ms_total", "ms_order", "ms_expand_count", "ms_beam", "ms_expand_write", "ms_hash",
            "ms_filter", "ms_output"]
_STAT_INT2 = ["n_expand_count", "filter_pairs", "first_visits", "general_children", "materialised", "non_elementary", "blocked_reactions"]


class efm_stats(ctypes.Structure):
    _fields_ = ([(k, ctypes.c_int64) for k in _STAT_INT] + [(k, ctypes.c_double) for k in _STAT_MS] +
                [(k, ctypes.c_int64) for k in _STAT_INT2])


class EfmError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"efm error {code}: {text}")
        self.code = code


_lib = None


def load() -> ctypes.CDLL:
    """Load the CUDA library; raise if it has not been built (``python -m paper_1804_02867_b200.build``)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1804_02867_b200.build` "
                          "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i32, i64, sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_size_t
    P = ctypes.POINTER
    lib.efm_create.argtypes = [vp, i32, i32, i64, vp, vp, P(efm_params), P(vp)]
    lib.efm_blocked_reactions.argtypes = [vp, i32, i32, i64, vp, vp, vp, P(i32)]
    lib.efm_graph_info.argtypes = [vp, P(i32), P(i32), P(i32), P(i64), P(i64)]
    lib.efm_graph_export.argtypes = [vp] + [vp] * 14
    lib.efm_workspace_bytes.argtypes = [vp, P(sz)]
    lib.efm_enumerate.argtypes = [vp, vp, vp, i32, vp, sz, vp]
    lib.efm_workspace_invalidate.argtypes = [vp]
    lib.efm_set_reaction_mask.argtypes = [vp, vp]
    lib.efm_result_steps.argtypes = [vp, vp, i64]
    lib.efm_sample_ends.argtypes = [vp, vp, i64, P(i64)]
    lib.efm_result_count.argtypes = [vp, P(i64)]
    lib.efm_result_copy.argtypes = [vp, vp, i64]
    lib.efm_result_sparse_stride.argtypes = [vp, P(i32)]
    lib.efm_result_copy_sparse.argtypes = [vp, vp, vp, vp, i64]
    lib.efm_result_nnz.argtypes = [vp, P(i64)]
    lib.efm_result_copy_csr.argtypes = [vp, vp, vp, vp, vp]
    lib.efm_result_device.argtypes = [vp, P(vp), P(vp), P(vp)]
    lib.efm_result_densify.argtypes = [vp, i64, i64, vp, vp]
    lib.efm_get_stats.argtypes = [vp, P(efm_stats)]
    lib.efm_get_level_stats.argtypes = [vp, vp, vp, vp, vp, i64, P(i64)]
    lib.efm_debug_state_hash.argtypes = [i32, i32, vp, vp, i32, vp, P(ctypes.c_uint64)]
    lib.efm_beam_threshold_scratch_bytes.argtypes = [i64, P(sz)]
    lib.efm_beam_threshold.argtypes = [vp, i64, i64, i64, vp, sz, vp, i32, vp]
    lib.efm_beam_threshold_static.argtypes = [vp, i64, i64, vp, i32, vp]
    lib.efm_beam_threshold_static_error.argtypes = []
    lib.efm_beam_threshold_static_error.restype = ctypes.c_char_p
    lib.efm_destroy.argtypes = [vp]
    lib.efm_destroy.restype = None
    lib.efm_strerror.argtypes = [ctypes.c_int]
    lib.efm_strerror.restype = ctypes.c_char_p
    lib.efm_last_error.argtypes = [vp]
    lib.efm_last_error.restype = ctypes.c_char_p
    _lib = lib
    return lib


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


@dataclass
class Result:
    flux: Optional[np.ndarray]  # int64 [n_out, n], reaction space, coprime, strict lexicographic order
    steps: Optional[np.ndarray] = None      # int32 [n_out]: expansions that built each pathway
    cand_end: Optional[np.ndarray] = None   # sampling mode: int64 [C, 2] (code, steps) per candidate
    stats: Dict[str, float] = None
    levels: Dict[str, np.ndarray] = None
    n_out: int = 0


class Enumerator:
    """One network + one parameter set (``efm_create`` ... ``efm_destroy``)."""

    def __init__(self, S: np.ndarray, reversible: np.ndarray, internal: np.ndarray, params: Optional[Dict[str, int]] = None,
                 device: int = 0, flags: int = 0):
        self._lib = load()
        self._h = ctypes.c_void_p()
        S = np.ascontiguousarray(S, dtype=np.int32)
        self.S = S
        self.m, self.n = S.shape
        rev = np.ascontiguousarray(reversible, dtype=np.uint8)
        internal = np.ascontiguousarray(internal, dtype=np.uint8)
        if rev.shape != (self.n,) or internal.shape != (self.m,):
            raise ValueError("reversible must have n entries and internal m entries")
        params = dict(params or {})
        p = efm_params(int(params.get("max_support", 0)), int(params.get("max_loop", 0)), int(params.get("dep_depth", 0)),
                       int(params.get("max_visited", 0)), int(params.get("frontier_cap", 0)),
                       int(params.get("max_frontier", 0)), int(params.get("max_candidates", 0)),
                       int(params.get("max_child_keys", 0)), int(device), int(flags),
                       int(params.get("max_frontier_bytes", 0)), int(params.get("max_child_tasks", 0)),
                       int(params.get("sample_count", 0)), int(params.get("sample_seed", 0)) & ((1 << 64) - 1))
        self.device = int(device)
        self._check(self._lib.efm_create(_ptr(S), self.m, self.n, self.n, _ptr(rev), _ptr(internal), ctypes.byref(p),
                                         ctypes.byref(self._h)))
        self._workspace = None

    # -- plumbing ----------------------------------------------------------------------------------------------
    def _check(self, rc: int):
        if rc != EFM_OK:
            text = self._lib.efm_strerror(rc).decode()
            if rc in (EFM_E_CUDA, EFM_E_CAPACITY) and self._h and self._lib.efm_last_error(self._h):
                text += ": " + self._lib.efm_last_error(self._h).decode()
            raise EfmError(rc, text)

    def close(self):
        if getattr(self, "_h", None):
            self._lib.efm_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- graph -------------------------------------------------------------------------------------------------
    def graph_info(self) -> Dict[str, int]:
        M, A, W = ctypes.c_int32(), ctypes.c_int32(), ctypes.c_int32()
        nnz, dep = ctypes.c_int64(), ctypes.c_int64()
        self._check(self._lib.efm_graph_info(self._h, ctypes.byref(M), ctypes.byref(A), ctypes.byref(W),
                                             ctypes.byref(nnz), ctypes.byref(dep)))
        return dict(M=M.value, A=A.value, W=W.value, nnz=nnz.value, dep_entries=dep.value)

    def graph_export(self) -> Dict[str, np.ndarray]:
        gi = self.graph_info()
        M, A, nnz, depn = gi["M"], gi["A"], gi["nnz"], gi["dep_entries"]
        g = dict(arc_rxn=np.zeros(A, np.int32), arc_dir=np.zeros(A, np.int32), twin=np.zeros(A, np.int32),
                 in_ptr=np.zeros(M + 1, np.int32), in_arc=np.zeros(nnz, np.int32), in_c=np.zeros(nnz, np.int64),
                 out_ptr=np.zeros(M + 1, np.int32), out_arc=np.zeros(nnz, np.int32), out_c=np.zeros(nnz, np.int64),
                 col_ptr=np.zeros(A + 1, np.int32), col_met=np.zeros(nnz, np.int32), col_s=np.zeros(nnz, np.int64),
                 dep_off=np.zeros(M + 1, np.int64), dep=np.zeros(max(depn, 1), np.uint8))
        order = ["arc_rxn", "arc_dir", "twin", "in_ptr", "in_arc", "in_c", "out_ptr", "out_arc", "out_c", "col_ptr",
                 "col_met", "col_s", "dep_off", "dep"]
        self._check(self._lib.efm_graph_export(self._h, *[_ptr(g[k]) for k in order]))
        for k in ("in_arc", "in_c"):
            g[k] = g[k][: g["in_ptr"][-1]]
        for k in ("out_arc", "out_c"):
            g[k] = g[k][: g["out_ptr"][-1]]
        g["dep"] = g["dep"][:depn]
        g.update(M=M, A=A, W=gi["W"])
        return g

    # -- run ---------------------------------------------------------------------------------------------------
    def workspace_bytes(self) -> int:
        b = ctypes.c_size_t()
        self._check(self._lib.efm_workspace_bytes(self._h, ctypes.byref(b)))
        return int(b.value)

    def enumerate_raw(self, seed_sets: Optional[Sequence[Sequence[int]]], d_workspace: int, workspace_bytes: int,
                      stream: int = 0) -> None:
        """``efm_enumerate`` with a raw device pointer (the caller owns the memory and the stream)."""
        if seed_sets:
            ptr = np.zeros(len(seed_sets) + 1, dtype=np.int32)
            ptr[1:] = np.cumsum([len(s) for s in seed_sets])
            codes = np.array([c for s in seed_sets for c in s] + [0], dtype=np.int32)
            n_sets = len(seed_sets)
        else:
            ptr, codes, n_sets = np.zeros(1, np.int32), np.zeros(1, np.int32), 0
        self._check(self._lib.efm_enumerate(self._h, _ptr(ptr), _ptr(codes), n_sets, ctypes.c_void_p(d_workspace),
                                            ctypes.c_size_t(workspace_bytes), ctypes.c_void_p(stream)))

    def set_reaction_mask(self, allowed: Optional[np.ndarray]) -> None:
        """Restrict the OR-alternatives to the reactions with allowed[j] != 0 (None lifts the restriction)."""
        if allowed is not None:
            allowed = np.ascontiguousarray(allowed, dtype=np.uint8)
            if allowed.shape != (self.n,):
                raise ValueError("allowed must have n entries")
        self._check(self._lib.efm_set_reaction_mask(self._h, _ptr(allowed)))

    def enumerate(self, seed_sets: Optional[Sequence[Sequence[int]]] = None, dense: bool = True) -> Result:
        """Allocate (once) the workspace with torch on ``cuda:device`` and run on torch's current stream."""
        import torch
        if not torch.cuda.is_available():
            raise EfmError(EFM_E_CUDA, "no CUDA device: the traversal runs in CUDA kernels only (no CPU fallback)")
        need = self.workspace_bytes()
        if self._workspace is None or self._workspace.numel() < need:
            self._workspace = torch.empty(need, dtype=torch.uint8, device=f"cuda:{self.device}")
            self._check(self._lib.efm_workspace_invalidate(self._h))
        with torch.cuda.device(self.device):
            stream = torch.cuda.current_stream().cuda_stream
            self.enumerate_raw(seed_sets, self._workspace.data_ptr(), self._workspace.numel(), stream)
        return self.result(dense=dense)

    def result(self, dense: bool = True) -> Result:
        k = ctypes.c_int64()
        self._check(self._lib.efm_result_count(self._h, ctypes.byref(k)))
        flux = None
        if dense:
            flux = np.zeros((k.value, self.n), dtype=np.int64)
            self._check(self._lib.efm_result_copy(self._h, _ptr(flux), k.value))
        steps = np.zeros(k.value, dtype=np.int32)
        self._check(self._lib.efm_result_steps(self._h, _ptr(steps), k.value))
        nc = ctypes.c_int64()
        self._check(self._lib.efm_sample_ends(self._h, None, 0, ctypes.byref(nc)))
        cand_end = None
        if nc.value:
            raw = np.zeros(nc.value, dtype=np.int64)
            self._check(self._lib.efm_sample_ends(self._h, _ptr(raw), nc.value, ctypes.byref(nc)))
            cand_end = np.stack([raw & 0xff, raw >> 8], axis=1)
        return Result(flux, steps, cand_end, self.stats(), self.level_stats(), int(k.value))

    def result_sparse(self):
        k = ctypes.c_int64()
        self._check(self._lib.efm_result_count(self._h, ctypes.byref(k)))
        cap = ctypes.c_int32()
        self._check(self._lib.efm_result_sparse_stride(self._h, ctypes.byref(cap)))
        nnz = np.zeros(k.value, np.int32)
        rxn = np.zeros((k.value, cap.value), np.int32)
        val = np.zeros((k.value, cap.value), np.int64)
        self._check(self._lib.efm_result_copy_sparse(self._h, _ptr(nnz), _ptr(rxn), _ptr(val), k.value))
        return nnz, rxn, val

    def result_csr(self, pinned: bool = True):
        """Compressed rows (row_ptr int64[K+1], rxn int32[nnz], val int64[nnz]) as torch CPU tensors; pinned host
        memory by default so that the device-to-host copies run at link speed."""
        import torch
        k, z = ctypes.c_int64(), ctypes.c_int64()
        self._check(self._lib.efm_result_count(self._h, ctypes.byref(k)))
        self._check(self._lib.efm_result_nnz(self._h, ctypes.byref(z)))
        pin = bool(pinned) and torch.cuda.is_available()
        row_ptr = torch.empty(k.value + 1, dtype=torch.int64, pin_memory=pin)
        rxn = torch.empty(max(z.value, 1), dtype=torch.int32, pin_memory=pin)
        val = torch.empty(max(z.value, 1), dtype=torch.int64, pin_memory=pin)
        with torch.cuda.device(self.device):
            stream = torch.cuda.current_stream().cuda_stream
            self._check(self._lib.efm_result_copy_csr(self._h, ctypes.c_void_p(row_ptr.data_ptr()), ctypes.c_void_p(rxn.data_ptr()),
                                                      ctypes.c_void_p(val.data_ptr()), ctypes.c_void_p(stream)))
        return row_ptr, rxn[: z.value], val[: z.value]

    def stats(self) -> Dict[str, float]:
        st = efm_stats()
        self._check(self._lib.efm_get_stats(self._h, ctypes.byref(st)))
        return {f: getattr(st, f) for f, _ in efm_stats._fields_}

    def level_stats(self) -> Dict[str, np.ndarray]:
        n = ctypes.c_int64()
        self._check(self._lib.efm_get_level_stats(self._h, None, None, None, None, 0, ctypes.byref(n)))
        arrs = [np.zeros(max(n.value, 1), np.int64) for _ in range(4)]
        self._check(self._lib.efm_get_level_stats(self._h, *[_ptr(a) for a in arrs], n.value, ctypes.byref(n)))
        return dict(active=arrs[0][: n.value], done=arrs[1][: n.value], expanded=arrs[2][: n.value],
                    children=arrs[3][: n.value])


def enumerate_network(net, device: int = 0, flags: int = 0, seed_sets="net", dense: bool = True, allowed=None, **overrides) -> Result:
    """Run the CUDA path on a ``netgen.Network`` with its own parameters (optionally overridden)."""
    params = dict(net.params)
    params.update(overrides)
    en = Enumerator(net.S, net.reversible, net.internal, params, device=device, flags=flags)
    try:
        seeds = net.seed_sets if isinstance(seed_sets, str) else seed_sets
        if allowed is not None:
            en.set_reaction_mask(allowed)
        return en.enumerate(seeds, dense=dense)
    finally:
        en.close()


def blocked_reactions(S: np.ndarray, reversible: np.ndarray, internal: np.ndarray) -> np.ndarray:
    """Compression pre-pass (``efm_blocked_reactions``): boolean mask of the reactions that cannot carry steady-state flux."""
    lib = load()
    S = np.ascontiguousarray(S, dtype=np.int32)
    m, n = S.shape
    rev = np.ascontiguousarray(reversible, dtype=np.uint8)
    internal = np.ascontiguousarray(internal, dtype=np.uint8)
    out = np.zeros(n, dtype=np.uint8)
    nb = ctypes.c_int32()
    rc = lib.efm_blocked_reactions(_ptr(S), m, n, n, _ptr(rev), _ptr(internal), _ptr(out), ctypes.byref(nb))
    if rc != EFM_OK:
        raise EfmError(rc, lib.efm_strerror(rc).decode())
    return out.astype(bool)


def debug_state_hash(arcs: Sequence[int], fluxes: Sequence[int], visited: Sequence[Sequence[int]], device: int = 0) -> int:
    """State hash of beam B computed by the device code (test hook)."""
    lib = load()
    a = np.array(list(arcs) + [0], dtype=np.int32)
    f = np.array(list(fluxes) + [0], dtype=np.int64)
    v = np.array([x for row in visited for x in row] + [0, 0, 0, 0], dtype=np.int32)
    out = ctypes.c_uint64()
    rc = lib.efm_debug_state_hash(device, len(arcs), _ptr(a), _ptr(f), len(visited), _ptr(v), ctypes.byref(out))
    if rc != EFM_OK:
        raise EfmError(rc, lib.efm_strerror(rc).decode())
    return int(out.value)


STATIC_SELECT_MAX_KEYS = 1 << 20   # EFM_STATIC_SELECT_MAX_KEYS of include/efm_b200.h


def beam_threshold_scratch_bytes(n_slots: int) -> int:
    b = ctypes.c_size_t()
    rc = load().efm_beam_threshold_scratch_bytes(int(n_slots), ctypes.byref(b))
    if rc != EFM_OK:
        raise EfmError(rc, load().efm_strerror(rc).decode())
    return int(b.value)


def beam_threshold(d_keys: int, n_slots: int, n_active: int, cap: int, d_scratch: int, scratch_bytes: int, d_threshold: int,
                   device: int = 0, stream: int = 0) -> None:
    """``efm_beam_threshold``: the traversal's own beam selection on raw device pointers, scratch from the caller."""
    lib = load()
    rc = lib.efm_beam_threshold(ctypes.c_void_p(d_keys), int(n_slots), int(n_active), int(cap), ctypes.c_void_p(d_scratch),
                                ctypes.c_size_t(scratch_bytes), ctypes.c_void_p(d_threshold), int(device), ctypes.c_void_p(stream))
    if rc != EFM_OK:
        raise EfmError(rc, lib.efm_strerror(rc).decode())


def beam_threshold_static(d_keys: int, n_keys: int, cap: int, d_threshold: int, device: int = 0, stream: int = 0) -> None:
    """``efm_beam_threshold_static``: the beam selection for a caller that cannot allocate scratch (a guest in another
    program's GPU process, a loop where cudaMalloc is banned).  Raw device pointers in, nothing allocated here or in the
    library; at most ``STATIC_SELECT_MAX_KEYS`` keys; enqueued on ``stream`` WITHOUT a synchronisation.  All calls on a
    device share one built-in scratch array: keep them ordered on the GPU."""
    lib = load()
    rc = lib.efm_beam_threshold_static(ctypes.c_void_p(d_keys), int(n_keys), int(cap), ctypes.c_void_p(d_threshold), int(device),
                                       ctypes.c_void_p(stream))
    if rc != EFM_OK:
        raise EfmError(rc, lib.efm_strerror(rc).decode() + ": " + lib.efm_beam_threshold_static_error().decode())


def exported_symbols() -> List[str]:
    """Function names declared in include/efm_b200.h (for the symbol-export test)."""
    import re
    with open(HEADER_PATH) as fh:
        text = fh.read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(efm_[a-z_0-9]+)\s*\(", text)))
