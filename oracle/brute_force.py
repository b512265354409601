"""Brute-force EFM enumeration for tiny networks -- TEST INFRASTRUCTURE (pin P9).

Definition 3 written out: for every arc subset T that holds no twin pair, T is the
support of an EFM iff the null space of S_int restricted to the columns T has dimension 1 and is
spanned by a strictly positive vector.  Exact rational arithmetic (fractions); exponential in the
number of arcs, so only for networks with <= ~20 arcs.  Shares no code with efm_oracle.c.
"""
from __future__ import annotations

from fractions import Fraction
from itertools import combinations
from math import gcd
from typing import List, Set, Tuple

import numpy as np


def _nullspace(cols: List[List[int]]) -> List[List[Fraction]]:
    """Null-space basis of the matrix whose columns are ``cols`` (reduced row echelon form)."""
    k = len(cols)
    rows = len(cols[0]) if k else 0
    A = [[Fraction(cols[c][r]) for c in range(k)] for r in range(rows)]
    piv_cols: List[int] = []
    r = 0
    for c in range(k):
        p = next((i for i in range(r, rows) if A[i][c] != 0), None)
        if p is None:
            continue
        A[r], A[p] = A[p], A[r]
        inv = 1 / A[r][c]
        A[r] = [x * inv for x in A[r]]
        for i in range(rows):
            if i != r and A[i][c] != 0:
                f = A[i][c]
                A[i] = [x - f * y for x, y in zip(A[i], A[r])]
        piv_cols.append(c)
        r += 1
        if r == rows:
            break
    free = [c for c in range(k) if c not in piv_cols]
    basis = []
    for fc in free:
        v = [Fraction(0)] * k
        v[fc] = Fraction(1)
        for i, pc in enumerate(piv_cols):
            v[pc] = -A[i][fc]
        basis.append(v)
    return basis


def brute_force_efms(S: np.ndarray, reversible: np.ndarray, internal: np.ndarray,
                     max_arcs: int = 22) -> Set[Tuple[int, ...]]:
    """All EFMs as coprime integer reaction-space vectors (v and -v of a reversible cycle are distinct)."""
    S = np.asarray(S)
    n = S.shape[1]
    Sint = S[np.asarray(internal).astype(bool)]
    arcs: List[Tuple[int, int]] = []
    for j in range(n):
        arcs.append((j, +1))
        if reversible[j]:
            arcs.append((j, -1))
    A = len(arcs)
    if A > max_arcs:
        raise ValueError(f"{A} arcs is too many for subset enumeration")
    col = [[int(d * x) for x in Sint[:, j]] for j, d in arcs]
    twin = {}
    for a, (j, d) in enumerate(arcs):
        if d < 0:
            twin[a] = a - 1
            twin[a - 1] = a
    efms: Set[Tuple[int, ...]] = set()
    for size in range(1, A + 1):
        for T in combinations(range(A), size):
            Ts = set(T)
            if any(twin.get(a, -1) in Ts for a in T):
                continue
            ns = _nullspace([col[a] for a in T])
            if len(ns) != 1:
                continue
            v = ns[0]
            if all(x < 0 for x in v):
                v = [-x for x in v]
            if not all(x > 0 for x in v):
                continue
            den = 1
            for x in v:
                den = den * x.denominator // gcd(den, x.denominator)
            iv = [int(x * den) for x in v]
            g = 0
            for x in iv:
                g = gcd(g, x)
            iv = [x // g for x in iv]
            out = [0] * n
            for a, x in zip(T, iv):
                out[arcs[a][0]] += arcs[a][1] * x
            efms.add(tuple(out))
    return efms
