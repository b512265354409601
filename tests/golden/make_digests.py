"""Writes tests/golden/digests.json: what the CPU oracle returns at beams too large for the oracle to be re-run inside
the test suite (the configs of BASELINE.json at the frontier caps they name).

    python tests/golden/make_digests.py [--out tests/golden/digests.json] [--threads N] [name:frontier_cap ...]

Imports ``oracle`` and ``netgen`` only -- never the CUDA library: a stored value is the oracle's.  The `-m gpu` test
test_parity_gpu.py::test_digests_at_large_beams runs the CUDA path on the same seeded network and compares

  * every counter of the traversal (levels, expanded, children, every discard reason, beam truncation, unique supports,
    poisoned, outputs, peak frontier, algorithmic bytes) and the four per-level series, stored in clear;
  * SHA-256 of the canonical output: the pathways as compressed sparse rows in their strict lexicographic order
    (row_ptr int64, reaction index int32 ascending within a row, coprime flux int64) and the step count of every row (int32).

Cost on the GPU box's 16 host cores: mid at frontier_cap 2^22 (the beam binds: 19.5 M active entries at the peak, 229 M
expansions) took the oracle 176 s and tens of GB of host memory (it keeps every child of a level until the beam has been
cut), which is why this is a stored digest and not a test.  genome at 2^20 did not finish within 40 minutes: the
oracle's O8 stage compares the ~2 M unique supports pairwise; it is left out of the default cases (genome stays compared
element by element up to 2^18 and by invariants above).
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

COUNTERS = ["levels", "expanded", "children", "done", "dead_end", "not_efm_maxloop", "discarded_nonpos", "discarded_overflow",
            "discarded_visited", "truncated_beam", "unique_supports", "poisoned", "output", "peak_frontier", "algo_bytes"]
LEVEL_SERIES = ["active", "done", "expanded", "children"]
DEFAULT_CASES = ["small:300", "genome:4096", "mid:4194304"]


def digest_csr(row_ptr: np.ndarray, rxn: np.ndarray, val: np.ndarray, steps: np.ndarray) -> dict:
    """SHA-256 of the canonical output in a fixed binary form (little-endian, C order)."""
    row_ptr = np.ascontiguousarray(row_ptr, dtype="<i8")
    rxn = np.ascontiguousarray(rxn, dtype="<i4")
    val = np.ascontiguousarray(val, dtype="<i8")
    steps = np.ascontiguousarray(steps, dtype="<i4")
    h = hashlib.sha256()
    for a in (row_ptr, rxn, val):
        h.update(np.int64(a.size).tobytes())
        h.update(a.tobytes())
    return dict(rows=int(row_ptr.size - 1), nnz=int(rxn.size), rows_sha256=h.hexdigest(),
                steps_sha256=hashlib.sha256(steps.tobytes()).hexdigest())


def dense_to_csr(flux: np.ndarray, chunk: int = 1 << 16):
    """Rows of a dense int64 matrix as (row_ptr, column indices ascending within a row, values), a chunk of rows at a time."""
    K = flux.shape[0]
    row_ptr = np.zeros(K + 1, dtype=np.int64)
    cols, vals = [], []
    for r0 in range(0, K, chunk):
        blk = flux[r0:r0 + chunk]
        rr, cc = np.nonzero(blk)              # row-major: columns ascend within a row
        row_ptr[r0 + 1:r0 + 1 + blk.shape[0]] = np.bincount(rr, minlength=blk.shape[0])
        cols.append(cc.astype(np.int32))
        vals.append(blk[rr, cc])
    np.cumsum(row_ptr, out=row_ptr)
    cat = lambda parts, dt: np.concatenate(parts) if parts else np.zeros(0, dt)   # noqa: E731
    return row_ptr, cat(cols, np.int32), cat(vals, np.int64)


def oracle_digest(name: str, cap: int, threads: int) -> dict:
    import oracle
    from netgen import make_network
    net = make_network(name, 0)
    t = time.time()
    res = oracle.enumerate_network(net, threads=threads, self_check=False, frontier_cap=cap)
    secs = time.time() - t
    row_ptr, rxn, val = dense_to_csr(res.flux)
    d = dict(workload=name, generator_seed=0, frontier_cap=int(cap), params=dict(net.params, frontier_cap=int(cap)))
    d.update(digest_csr(row_ptr, rxn, val, res.steps))
    d["counters"] = {k: int(res.stats[k]) for k in COUNTERS}
    d["levels"] = {k: [int(x) for x in res.levels[k]] for k in LEVEL_SERIES}
    d["n_roots"] = int(res.n_roots)
    d["oracle_seconds"] = round(secs, 1)
    d["oracle_threads"] = int(threads)
    return d


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("cases", nargs="*", default=DEFAULT_CASES, help="name:frontier_cap")
    ap.add_argument("--out", default=os.path.join(os.path.dirname(os.path.abspath(__file__)), "digests.json"))
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--min-free-gb", type=float, default=0.0, help="refuse a case when less host memory than this is available")
    args = ap.parse_args()
    import oracle
    oracle.build()
    threads = args.threads or max(1, min(oracle.max_threads(), os.cpu_count() or 1))
    out = {"_about": "Written by tests/golden/make_digests.py from oracle/ alone (see its docstring).", "cases": []}
    if os.path.exists(args.out):
        with open(args.out) as fh:
            out = json.load(fh)
    for case in args.cases:
        name, cap = case.split(":")
        if args.min_free_gb:
            with open("/proc/meminfo") as fh:
                avail = [int(line.split()[1]) for line in fh if line.startswith("MemAvailable")][0] / 1e6
            if avail < args.min_free_gb:
                print(f"{case}: only {avail:.0f} GB of host memory available, skipped", flush=True)
                continue
        d = oracle_digest(name, int(cap), threads)
        out["cases"] = [c for c in out["cases"] if (c["workload"], c["frontier_cap"]) != (name, int(cap))] + [d]
        out["cases"].sort(key=lambda c: (c["workload"], c["frontier_cap"]))
        with open(args.out, "w") as fh:   # after every case: a run cut short keeps what it finished
            json.dump(out, fh, indent=1)
            fh.write("\n")
        print(f"{case}: {d['rows']} rows, {d['oracle_seconds']} s on {threads} threads", flush=True)
    return 0


if __name__ == "__main__":
    sys.exit(main())
