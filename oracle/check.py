"""O9 self-check of every oracle (or library) output -- TEST INFRASTRUCTURE.

Checks the definitions the paper fixes, in exact integer arithmetic:
  Def 2: S_int . v = 0 and v_j >= 0 on irreversible reactions;
  canonical form (reading G10): gcd(|v|) = 1, no zero vector, rows strictly increasing lexicographically;
  Def 3 among the outputs (reading G17): no output support strictly contains another;
and reports *precision*: the fraction of outputs that are true EFMs by the rank test
(nullity of S_int restricted to the arc support = 1), which the method does not guarantee.
"""
from __future__ import annotations

from math import gcd
from typing import Dict

import numpy as np

_P = 2147483647  # Mersenne prime 2^31 - 1 for the modular rank test


def _rank_mod_p(Mx: np.ndarray) -> int:
    A = (Mx.astype(object) % _P).astype(np.int64)
    rows, cols = A.shape
    r = 0
    for c in range(cols):
        piv = -1
        for i in range(r, rows):
            if A[i, c] % _P:
                piv = i
                break
        if piv < 0:
            continue
        if piv != r:
            A[[r, piv]] = A[[piv, r]]
        inv = pow(int(A[r, c]), _P - 2, _P)
        A[r] = (A[r] * inv) % _P
        for i in range(rows):
            if i != r and A[i, c]:
                A[i] = (A[i] - A[i, c] * A[r]) % _P
        r += 1
        if r == rows:
            break
    return r


def check_outputs(S: np.ndarray, reversible: np.ndarray, internal: np.ndarray, flux: np.ndarray,
                  rank_test: bool = True, max_pairwise: int = 6000, max_rank_rows: int = 2000) -> Dict[str, float]:
    S = np.asarray(S)
    rev = np.asarray(reversible).astype(bool)
    Sint = S[np.asarray(internal).astype(bool)]
    flux = np.asarray(flux, dtype=np.int64).reshape(-1, S.shape[1])
    K, n = flux.shape
    out = dict(n=float(K), precision=float("nan"))
    if K == 0:
        return out
    # Def 2, exact: Python integers so that 2^62-scale fluxes cannot wrap
    big = int(np.abs(flux).max()) >= (1 << 40)
    if big:
        So = Sint.astype(object)
        for r in range(K):
            assert not np.any(So.dot(flux[r].astype(object))), f"row {r}: S_int . v != 0"
    else:
        assert not np.any(Sint.astype(np.int64) @ flux.T), "S_int . v != 0"
    assert np.all(flux[:, ~rev] >= 0), "negative flux on an irreversible reaction"
    for r in range(K):
        g = 0
        for x in flux[r][flux[r] != 0]:
            g = gcd(g, abs(int(x)))
        assert g == 1, f"row {r}: gcd = {g}"
    for r in range(1, K):
        d = np.nonzero(flux[r - 1] != flux[r])[0]
        assert d.size and flux[r - 1, d[0]] < flux[r, d[0]], f"rows {r-1},{r} not in strict lexicographic order"
    # Def 3 among the outputs: arc-space supports (sign matters for reversible reactions)
    bits = np.concatenate([flux > 0, flux < 0], axis=1)
    packed = np.packbits(bits, axis=1)
    rows = range(K) if K <= max_pairwise else np.random.default_rng(0).choice(K, max_pairwise, replace=False)
    for r in rows:
        inside = ~np.any(packed & ~packed[r], axis=1)  # supp(w) subset of supp(r)
        inside[r] = False
        assert not inside.any(), f"output {r} strictly contains output {int(np.nonzero(inside)[0][0])}"
    if rank_test:
        ok = 0
        rr = list(range(K)) if K <= max_rank_rows else list(np.random.default_rng(1).choice(K, max_rank_rows, replace=False))
        for r in rr:
            cols = np.nonzero(flux[r])[0]
            sub = Sint[:, cols].astype(np.int64) * np.sign(flux[r, cols])
            sub = sub[np.any(sub != 0, axis=1)]
            rank = _rank_mod_p(sub) if sub.size else 0
            ok += (len(cols) - rank) == 1
        out["precision"] = ok / len(rr)
    return out
