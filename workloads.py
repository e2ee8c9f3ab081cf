"""Seeded synthetic input generators shared by tests, bench.py and smoke().

This module holds NONE of the method's arithmetic: it only draws sequences.  It is the
one module both the oracle-side tests and the CUDA-side harness may import (the oracle
and the CUDA path never import each other).

Recipe (restated in DESIGN.md "Input recipe"): the paper measured
on mouse non-coding RNA, random substrings of real RNA and random strings over A,C,G,U
(PAPER.md:301).  The real sequences are not available and are not reconstructed; i.i.d.
random strings -- the paper's own third workload -- stand in for all of them, with the
lengths BASELINE.json's five configs name.  The legacy `numpy.random.RandomState` stream is
used so the draws are frozen across numpy versions.
"""
from __future__ import annotations

import numpy as np

ALPHABET = "ACGU"

# name -> (seed, n, q list, table dtype) for the single-sequence configs of BASELINE.json
SINGLE_CONFIGS = {
    "cfg1": {"seed": 0, "n": 256, "q": (4,), "table_dtype": "int32"},
    "cfg2": {"seed": 1, "n": 2000, "q": (8,), "table_dtype": "int16"},
    "cfg3": {"seed": 2, "n": 6000, "q": (8,), "table_dtype": "int16"},
    "cfg5": {"seed": 4, "n": 16384, "q": (8, 10), "table_dtype": "int16"},
    # beyond BASELINE.json's five configs ("n > 16384"): the same recipe at twice the length
    "cfg6": {"seed": 6, "n": 32768, "q": (8,), "table_dtype": "int16"},
}
BATCH_CONFIG = {"seed": 3, "count": 1024, "lo": 300, "hi": 700, "q": (8,)}


def uniform_sequence(seed: int, n: int) -> bytes:
    """n bases i.i.d. uniform over {A,C,G,U}: codes = RandomState(seed).randint(0,4,n)."""
    rs = np.random.RandomState(seed)
    codes = rs.randint(0, 4, size=n)
    return np.frombuffer(ALPHABET.encode(), dtype=np.uint8)[codes].tobytes()


def single_config(name: str) -> bytes:
    c = SINGLE_CONFIGS[name]
    return uniform_sequence(c["seed"], c["n"])


def gc_rich_batch(seed: int = 3, count: int = 1024, lo: int = 300, hi: int = 700):
    """Config 4: `count` sequences, lengths uniform in [lo,hi], P(A)=P(U)=0.2, P(C)=P(G)=0.3.

    lens = rs.randint(lo, hi+1, count); then, sequence by sequence in order,
    u = rs.random_sample(len); base = A if u<0.2, C if u<0.5, G if u<0.8, else U.
    Returns (list of bytes, int32 array of lengths).
    """
    rs = np.random.RandomState(seed)
    lens = rs.randint(lo, hi + 1, size=count).astype(np.int32)
    lut = np.frombuffer(ALPHABET.encode(), dtype=np.uint8)
    seqs = []
    for ln in lens:
        u = rs.random_sample(int(ln))
        codes = np.where(u < 0.2, 0, np.where(u < 0.5, 1, np.where(u < 0.8, 2, 3)))
        seqs.append(lut[codes].tobytes())
    return seqs, lens


def random_sequences(seed: int, count: int, lo: int, hi: int, alphabet: str = ALPHABET):
    """Generic helper for parity sweeps: `count` uniform sequences with lengths in [lo,hi]."""
    rs = np.random.RandomState(seed)
    lens = rs.randint(lo, hi + 1, size=count).astype(np.int32)
    lut = np.frombuffer(alphabet.encode(), dtype=np.uint8)
    return [lut[rs.randint(0, len(alphabet), size=int(ln))].tobytes() for ln in lens], lens


def pack_batch(seqs):
    """Concatenate sequences -> (uint8 array, int64 offsets[count+1], int32 lens[count])."""
    lens = np.array([len(s) for s in seqs], dtype=np.int32)
    offsets = np.zeros(len(seqs) + 1, dtype=np.int64)
    np.cumsum(lens, out=offsets[1:])
    flat = np.frombuffer(b"".join(seqs), dtype=np.uint8).copy() if len(seqs) else np.zeros(0, np.uint8)
    return flat, offsets, lens


def sample_cells(n: int, q: int, count: int, seed: int = 12345):
    """Sampled (i,j) cells, 1-based, i<=j, for large-n parity: all of the last
    three diagonals, row 1, column n (strided), cells with (j-i) mod q in {0,1,q-1}, plus
    uniform random cells.  Pure index selection, no method arithmetic."""
    rs = np.random.RandomState(seed)
    cells = set()
    for d in (n - 1, n - 2, n - 3):
        if d >= 0:
            for i in range(1, n - d + 1):
                cells.add((i, i + d))
    stride = max(1, n // 512)
    for j in range(1, n + 1, stride):
        cells.add((1, j))
    for i in range(1, n + 1, stride):
        cells.add((i, n))
    while len(cells) < count:
        i = int(rs.randint(1, n + 1))
        j = int(rs.randint(i, n + 1))
        r = int(rs.randint(0, 4))
        if r < 3 and n > q:
            want = (0, 1, q - 1)[r]
            d = j - i
            d = d - (d % q) + want
            j = i + d
            if j > n or j < i:
                continue
        cells.add((i, j))
    out = np.array(sorted(cells), dtype=np.int32)
    return out
