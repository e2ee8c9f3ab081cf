"""ORACLE -- TEST INFRASTRUCTURE ONLY.  Structures (sets of base pairs) of the Nussinov problem.

  check_structure -- the DEFINITION of a feasible solution: pairs are complementary (A-U, C-G;
                     DESIGN.md reading g1: no other pair, no minimum loop length), every base is in at most
                     one pair, and no two pairs cross.
  traceback       -- a plain sequential traceback of eq. (1) (PAPER.md:49-52; the paper's D*, PAPER.md:54, :87,
                     stores the same choices as arg-max indices) over the oracle's own table.  Pure Python:
                     small n only.  Pinned in tests/test_traceback.py: its output is feasible and has D(1,n)
                     pairs, and D(1,n) is pinned to brute force (tests/test_oracle_pins.py), so it is optimal.
Several optimal structures may exist; the CUDA traceback is compared on what is unique (the number of pairs)
and checked for feasibility with check_structure.
"""
from __future__ import annotations

import numpy as np

_COMP = {("A", "U"), ("U", "A"), ("C", "G"), ("G", "C")}


def _norm(seq) -> str:
    s = seq.decode() if isinstance(seq, (bytes, bytearray)) else str(seq)
    return s.upper().replace("T", "U")


def check_structure(seq, partner) -> int:
    """partner[i] = index (0-based) of the base paired with i, or -1.  Returns the number of pairs;
    raises AssertionError if the structure is not feasible."""
    s = _norm(seq)
    partner = np.asarray(partner)
    n = len(s)
    assert partner.shape == (n,), "one entry per base"
    stack = []
    npairs = 0
    for i in range(n):
        j = int(partner[i])
        if j == -1:
            continue
        assert 0 <= j < n and j != i, f"partner of {i} out of range"
        assert int(partner[j]) == i, f"pair ({i},{j}) is not symmetric"
        assert (s[i], s[j]) in _COMP, f"bases {s[i]}{s[j]} at ({i},{j}) are not complementary"
        if j > i:
            stack.append(j)           # opens: must close before anything opened earlier closes
            npairs += 1
        else:
            assert stack and stack[-1] == i, f"pair closing at {i} crosses another pair"
            stack.pop()
    assert not stack
    return npairs


def traceback(seq, table) -> np.ndarray:
    """table[i-1][j-1] = D(i,j), i <= j (as oracle.nussinov returns it).  Returns partner[0..n-1]."""
    s = _norm(seq)
    n = len(s)
    partner = np.full(n, -1, dtype=np.int32)

    def D(i, j):                       # 1-based; D(i,i-1) = D(i,i) = 0
        return 0 if j <= i else int(table[i - 1][j - 1])

    todo = [(1, n)] if n >= 2 else []
    while todo:
        i, j = todo.pop()
        if j <= i or D(i, j) == 0:
            continue
        if (s[i - 1], s[j - 1]) in _COMP and D(i, j) == 1 + D(i + 1, j - 1):       # first term of eq. (1)
            partner[i - 1], partner[j - 1] = j - 1, i - 1
            todo.append((i + 1, j - 1))
            continue
        for k in range(i + 1, j + 1):                                              # second term of eq. (1)
            if D(i, j) == D(i, k - 1) + D(k, j):
                todo.append((i, k - 1))
                todo.append((k, j))
                break
        else:
            raise AssertionError("table is not a table of eq. (1)")
    return partner
