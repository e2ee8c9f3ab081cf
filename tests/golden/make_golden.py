"""Writes the stored expected values under tests/golden/ for the large configs.

Calls ONLY oracle/ (plus the seeded input generators in workloads.py).  No value here ever comes
from the CUDA path.  Usage:  python tests/golden/make_golden.py [cfg1 cfg2 cfg3 cfg4 cfg5]

Files written (text):
  <cfg>_expected.txt : "n", "score" = D(1,n), "table_sum" = sum_{i<=j} D(i,j), first 24 bases
  <cfg>_cells.txt    : one line "i j D(i,j)" per sampled cell (workloads.sample_cells)
  cfg4_scores.txt    : one line "t len score" per sequence of the batch config
cfg1/cfg2 use the plain oracle (oracle.nussinov); cfg3/cfg4/cfg5 use its fast-plain storage mode
(oracle.nussinov_fast, validated cell by cell against the plain mode in tests/test_oracle_pins.py).
"""
from __future__ import annotations

import os
import sys
import time

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "..", ".."))

import numpy as np  # noqa: E402

import oracle  # noqa: E402
import workloads  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
THREADS = os.cpu_count() or 1


def single(name: str):
    cfg = workloads.SINGLE_CONFIGS[name]
    seq = workloads.single_config(name)
    n = cfg["n"]
    cells = workloads.sample_cells(n, cfg["q"][0], 10000)
    t0 = time.time()
    if n <= 2000:
        score, tab = oracle.nussinov(seq, want_table=True)
        vals = tab[cells[:, 0] - 1, cells[:, 1] - 1]
        tsum = int(tab.astype(np.int64).sum())
    else:
        r = oracle.nussinov_fast(seq, threads=THREADS, cells=cells, want_sum=True)
        score, vals, tsum = r["score"], r["cells"], r["table_sum"]
    dt = time.time() - t0
    with open(os.path.join(HERE, f"{name}_expected.txt"), "w") as f:
        f.write(f"# written by tests/golden/make_golden.py from oracle/ (eq. (1), PAPER.md:49-52); {dt:.1f} s, {THREADS} threads\n")
        f.write(f"n {n}\nseed {cfg['seed']}\nscore {score}\ntable_sum {tsum}\nfirst24 {seq[:24].decode()}\n")
    with open(os.path.join(HERE, f"{name}_cells.txt"), "w") as f:
        f.write("# i j D(i,j)  (1-based, oracle/ eq. (1)); cells = workloads.sample_cells(n, q, 10000)\n")
        for (i, j), v in zip(cells, vals):
            f.write(f"{i} {j} {int(v)}\n")
    print(name, "score", score, "sum", tsum, f"{dt:.1f}s")


def batch():
    seqs, lens = workloads.gc_rich_batch()
    t0 = time.time()
    with open(os.path.join(HERE, "cfg4_scores.txt"), "w") as f:
        f.write("# t len score ; oracle/ eq. (1) on workloads.gc_rich_batch() (seed 3)\n")
        total = 0
        for t, s in enumerate(seqs):
            sc = oracle.nussinov_fast(s, threads=1)["score"]
            total += sc
            f.write(f"{t} {len(s)} {sc}\n")
    print("cfg4 sum of scores", total, "total bases", int(lens.sum()), f"{time.time() - t0:.1f}s")


if __name__ == "__main__":
    which = sys.argv[1:] or ["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"]
    for w in which:
        if w == "cfg4":
            batch()
        else:
            single(w)
