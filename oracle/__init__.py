"""ORACLE -- TEST INFRASTRUCTURE ONLY (see the headers of the .c files).

Thin ctypes access to oracle/liboracle.so.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package; the product path
(paper_1307_7820_b200) never does and shares no code with it.

Functions and the passages they follow:
  nussinov / nussinov_fourterm / nussinov_fast  -- eq. (1), PAPER.md:45-54         (pinned)
  brute_force_matchings / brute_force_structural -- the definition, PAPER.md:45     (the pins)
  blackbox / rtable                             -- listing PAPER.md:91-113          (pinned)
  two_vector_serial                             -- Algorithm 1, PAPER.md:125-187    (baseline, pinned to eq. (1))
  serial_variant                                -- partially / completely memoised and Frid-Gusfield variants,
                                                   PAPER.md:199-219                 (baselines, pinned to eq. (1))
  structure.check_structure / structure.traceback -- feasibility by the definition; plain
                                                   traceback of eq. (1), PAPER.md:54, :87 (pinned)
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build.build())
        L = _lib
        u8p, i32p, i16p, i64p = (ctypes.POINTER(t) for t in (ctypes.c_uint8, ctypes.c_int32, ctypes.c_int16, ctypes.c_int64))
        L.oracle_nussinov.argtypes = [ctypes.c_char_p, ctypes.c_int, i32p]
        L.oracle_nussinov_fourterm.argtypes = [ctypes.c_char_p, ctypes.c_int, i32p]
        L.oracle_nussinov_fast.argtypes = [ctypes.c_char_p, ctypes.c_int, ctypes.c_int, i32p, ctypes.c_int, i32p, i16p, i64p]
        L.oracle_brute_force_matchings.argtypes = [ctypes.c_char_p, ctypes.c_int]
        L.oracle_brute_force_structural.argtypes = [ctypes.c_char_p, ctypes.c_int]
        L.oracle_blackbox.argtypes = [ctypes.c_int, ctypes.c_uint32, ctypes.c_uint32, ctypes.POINTER(ctypes.c_int)]
        L.oracle_rtable.argtypes = [ctypes.c_int, u8p]
        L.oracle_two_vector_serial.argtypes = [ctypes.c_char_p, ctypes.c_int, ctypes.c_int, i32p, i64p]
        L.oracle_serial_variant.argtypes = [ctypes.c_char_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, i32p, i64p]
        L.oracle_validate.argtypes = [ctypes.c_char_p, ctypes.c_int]
    return _lib


def _as_bytes(seq) -> bytes:
    if isinstance(seq, str):
        return seq.encode()
    return bytes(seq)


def _p(arr, ctype):
    return arr.ctypes.data_as(ctypes.POINTER(ctype))


def nussinov(seq, want_table: bool = False):
    """Plain eq. (1).  Returns score, or (score, n x n int32 table) if want_table."""
    s = _as_bytes(seq)
    n = len(s)
    tab = np.zeros((n, n), dtype=np.int32) if want_table else None
    r = lib().oracle_nussinov(s, n, _p(tab, ctypes.c_int32) if want_table and n else None)
    return (r, tab) if want_table else r


def nussinov_fourterm(seq, want_table: bool = False):
    s = _as_bytes(seq)
    n = len(s)
    tab = np.zeros((n, n), dtype=np.int32) if want_table else None
    r = lib().oracle_nussinov_fourterm(s, n, _p(tab, ctypes.c_int32) if want_table and n else None)
    return (r, tab) if want_table else r


def nussinov_fast(seq, threads: int = 1, cells=None, want_table: bool = False, want_sum: bool = False):
    """fast-plain mode (same recurrence, mirrored storage).  cells: int32 array [m,2] of 1-based (i,j).
    Returns dict(score=, cells=, table=, table_sum=)."""
    s = _as_bytes(seq)
    n = len(s)
    if cells is None:
        cells = np.zeros((0, 2), dtype=np.int32)
    cells = np.ascontiguousarray(cells, dtype=np.int32)
    vals = np.zeros(len(cells), dtype=np.int32)
    tab = np.zeros((n, n), dtype=np.int16) if want_table else None
    tsum = ctypes.c_int64(0)
    r = lib().oracle_nussinov_fast(
        s, n, int(threads),
        _p(cells, ctypes.c_int32) if len(cells) else None, len(cells),
        _p(vals, ctypes.c_int32) if len(cells) else None,
        _p(tab, ctypes.c_int16) if want_table and n else None,
        ctypes.byref(tsum) if want_sum else None)
    return {"score": r, "cells": vals, "table": tab, "table_sum": tsum.value if want_sum else None}


def brute_force_matchings(seq) -> int:
    s = _as_bytes(seq)
    return lib().oracle_brute_force_matchings(s, len(s))


def brute_force_structural(seq) -> int:
    s = _as_bytes(seq)
    return lib().oracle_brute_force_structural(s, len(s))


def blackbox(q: int, v: int, vbar: int):
    """(max-val, max-index) of the listing PAPER.md:94-111."""
    idx = ctypes.c_int(0)
    val = lib().oracle_blackbox(q, v, vbar, ctypes.byref(idx))
    return val, idx.value


def rtable(q: int) -> np.ndarray:
    N = 1 << q
    R = np.zeros((N, N), dtype=np.uint8)
    rc = lib().oracle_rtable(q, _p(R, ctypes.c_uint8))
    if rc != 0:
        raise ValueError("bad q")
    return R


def two_vector_serial(seq, q: int, want_table: bool = False):
    """Algorithm 1 (serial two-vector).  Returns dict(score=, table=, lookups=)."""
    s = _as_bytes(seq)
    n = len(s)
    tab = np.zeros((n, n), dtype=np.int32) if want_table else None
    lk = ctypes.c_int64(0)
    r = lib().oracle_two_vector_serial(s, n, q, _p(tab, ctypes.c_int32) if want_table and n else None, ctypes.byref(lk))
    return {"score": r, "table": tab, "lookups": lk.value}


SERIAL_VARIANTS = {"partially_memoized": 1, "completely_memoized": 2, "frid_gusfield": 3}


def serial_variant(seq, q: int, variant: str, want_table: bool = False):
    """The paper's other serial variants: 'partially_memoized', 'completely_memoized',
    'frid_gusfield'.  Returns dict(score=, table=, lookups=, blackbox_evals=, table_bytes=)."""
    s = _as_bytes(seq)
    n = len(s)
    tab = np.zeros((n, n), dtype=np.int32) if want_table else None
    st = (ctypes.c_int64 * 3)()
    r = lib().oracle_serial_variant(s, n, q, SERIAL_VARIANTS[variant], _p(tab, ctypes.c_int32) if want_table and n else None, st)
    if r == -2:
        raise MemoryError("serial_variant: out of memory")
    return {"score": r, "table": tab, "lookups": st[0], "blackbox_evals": st[1], "table_bytes": st[2]}
