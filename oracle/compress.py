"""SURVEY.md 8(f)-4, compression pre-pass ("partitioning and compression preprocessing methods can be used
further to overcome the limitation of the hardware platforms"), oracle side: reactions that cannot carry flux in ANY
steady state (Def 2) for a purely topological reason are removed before the traversal.

Rule, iterated to a fixed point: an internal metabolite i is balanced by S_i . v = 0.  Among the reactions still present
let P_i be those that can produce i (s_ij > 0, or reversible with s_ij != 0) and C_i those that can consume it.  If no
pair (p in P_i, c in C_i) of two DIFFERENT reactions exists, every term of the sum has one sign (or there is a single
term), so every reaction touching i has flux 0: it is blocked and removed.  Test infrastructure: plain Python loops."""
from typing import List

import numpy as np


def blocked_reactions(S: np.ndarray, reversible: np.ndarray, internal: np.ndarray) -> np.ndarray:
    S = np.asarray(S)
    m, n = S.shape
    blocked = np.zeros(n, dtype=bool)
    changed = True
    while changed:
        changed = False
        for i in range(m):
            if not internal[i]:
                continue
            prod: List[int] = []
            cons: List[int] = []
            touch: List[int] = []
            for j in range(n):
                if blocked[j] or S[i, j] == 0:
                    continue
                touch.append(j)
                if S[i, j] > 0 or reversible[j]:
                    prod.append(j)
                if S[i, j] < 0 or reversible[j]:
                    cons.append(j)
            if not touch:
                continue
            ok = any(p != c for p in prod for c in cons)
            if not ok:
                for j in touch:
                    blocked[j] = True
                changed = True
    return blocked
