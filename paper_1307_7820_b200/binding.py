"""Thin Python binding of the C ABI in include/rna4r.h (argument marshalling only).

Every step of the fold runs inside librna4r.so's CUDA kernels; torch is used here only for
device memory and streams.  There is no CPU fallback: if the library is missing or no sm_100
device exists, calls raise.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import build as _build

TABLE_NONE, TABLE_INT16, TABLE_INT32 = 0, 1, 2
ENGINE_AUTO, ENGINE_TILED, ENGINE_DIAG, ENGINE_SMEM, ENGINE_PAPER_TILE, ENGINE_MAXPLUS = 0, 1, 2, 3, 4, 5

_lib = None


class Rna4rError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        msg = load().rna4r_strerror(code).decode()
        super().__init__(f"{where}: {msg} (code {code})")


def load():
    """Loads librna4r.so (building it in-tree if the sources are newer)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if _build.is_stale():
        path = _build.build()
    L = ctypes.CDLL(path)
    vp, i32p, u8p, i64p = ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p
    L.rna4r_version.restype = ctypes.c_char_p
    L.rna4r_strerror.restype = ctypes.c_char_p
    L.rna4r_strerror.argtypes = [ctypes.c_int]
    L.rna4r_prepare.argtypes = [ctypes.c_int, ctypes.c_int, vp, ctypes.POINTER(vp)]
    L.rna4r_destroy.argtypes = [vp]
    L.rna4r_q.argtypes = [vp]
    L.rna4r_table.argtypes = [vp]
    L.rna4r_table.restype = vp
    L.rna4r_table_compact.argtypes = [vp]
    L.rna4r_table_compact.restype = vp
    L.rna4r_table_to_host.argtypes = [vp, vp, ctypes.c_int]
    L.rna4r_set_engine.argtypes = [vp, ctypes.c_int]
    L.rna4r_engine.argtypes = [vp]
    L.rna4r_smem_max_n.argtypes = [vp]
    L.rna4r_workspace_bytes.argtypes = [vp, ctypes.c_int, ctypes.c_int, ctypes.c_int]
    L.rna4r_set_max_blocks_per_sm.argtypes = [vp, ctypes.c_int]
    L.rna4r_set_max_blocks.argtypes = [vp, ctypes.c_int]
    L.rna4r_microbench_lookups.argtypes = [vp, ctypes.c_int, ctypes.c_int, ctypes.c_int, vp, vp,
                                           ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_double)]
    L.rna4r_fold_batch_status.argtypes = [vp, u8p, i64p, i32p, ctypes.c_int, i32p, i32p, vp, ctypes.c_size_t, vp]
    L.rna4r_workspace_bytes.restype = ctypes.c_size_t
    L.rna4r_workspace_bytes_batch.argtypes = [vp, i32p, ctypes.c_int]
    L.rna4r_workspace_bytes_batch.restype = ctypes.c_size_t
    L.rna4r_workspace_bytes_host.argtypes = [vp, i32p, ctypes.c_int, ctypes.c_int]
    L.rna4r_workspace_bytes_host.restype = ctypes.c_size_t
    L.rna4r_fold.argtypes = [vp, u8p, ctypes.c_int, i32p, vp, ctypes.c_int, vp, ctypes.c_size_t, vp]
    L.rna4r_fold_batch.argtypes = [vp, u8p, i64p, i32p, ctypes.c_int, i32p, vp, ctypes.c_size_t, vp]
    L.rna4r_fold_host.argtypes = [vp, u8p, ctypes.c_int, i32p, vp, ctypes.c_int, vp, ctypes.c_size_t, vp]
    L.rna4r_fold_batch_host.argtypes = [vp, u8p, i32p, ctypes.c_int, i32p, vp, ctypes.c_size_t, vp]
    L.rna4r_enable_kernel_timing.argtypes = [vp, ctypes.c_int]
    L.rna4r_last_fill_kernel_ms.argtypes = [vp, ctypes.POINTER(ctypes.c_float)]
    L.rna4r_traceback_workspace_bytes.argtypes = [vp, ctypes.c_int]
    L.rna4r_traceback_workspace_bytes.restype = ctypes.c_size_t
    L.rna4r_traceback.argtypes = [vp, vp, ctypes.c_int, vp, ctypes.c_int, vp, vp, vp, ctypes.c_size_t, vp]
    L.rna4r_set_trace.argtypes = [vp, ctypes.c_int]
    L.rna4r_trace_to_host.argtypes = [vp, vp, ctypes.c_int]
    L.rna4r_last_launch_count.argtypes = [vp]
    L.rna4r_last_cuda_error.argtypes = [vp]
    L.rna4r_fold_static_setup.argtypes = [vp, vp]
    L.rna4r_fold_static_max_n.argtypes = [vp]
    L.rna4r_fold_static.argtypes = [vp, vp, ctypes.c_int, vp, vp]
    _lib = L
    return L


def _check(code: int, where: str):
    if code != 0:
        raise Rna4rError(code, where)


def _stream_ptr(stream) -> int:
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


class Rna4r:
    """One prepared context (rna4r_prepare) on one device for one q."""

    def __init__(self, q: int, device: int = 0, engine: int = ENGINE_AUTO, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("rna4r needs a CUDA (sm_100) device; there is no CPU fallback")
        self.lib = load()
        self.device = device
        self.q = q
        self._ws = None
        torch.cuda.set_device(device)
        h = ctypes.c_void_p()
        _check(self.lib.rna4r_prepare(q, device, _stream_ptr(stream), ctypes.byref(h)), "rna4r_prepare")
        self.h = h
        if engine != ENGINE_AUTO:
            self.set_engine(engine)

    # -- context -----------------------------------------------------------------------------
    def close(self):
        if getattr(self, "h", None):
            self.lib.rna4r_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_engine(self, engine: int):
        _check(self.lib.rna4r_set_engine(self.h, engine), "rna4r_set_engine")

    @property
    def engine(self) -> int:
        return self.lib.rna4r_engine(self.h)

    def smem_max_n(self) -> int:
        """rna4r_smem_max_n: longest sequence ENGINE_SMEM folds at this q (-1: q not supported)."""
        return self.lib.rna4r_smem_max_n(self.h)

    def table(self) -> np.ndarray:
        """R as a numpy uint8 array [2^q, 2^q] (host copy via rna4r_table_to_host)."""
        return self._table_host(0)

    def table_compact(self) -> np.ndarray:
        return self._table_host(1)

    def table_ternary(self) -> np.ndarray:
        """Rt, 3^(q-1) bytes indexed by sum (v_k + vbar_k + 1) 3^(k-1); q = 9..11 only (rna4r.h)."""
        out = np.empty(3 ** (self.q - 1), dtype=np.uint8)
        _check(self.lib.rna4r_table_to_host(self.h, out.ctypes.data, 2), "rna4r_table_to_host")
        return out

    def _table_host(self, compact: int) -> np.ndarray:
        side = 1 << (self.q - 1 if compact else self.q)
        out = np.empty((side, side), dtype=np.uint8)
        _check(self.lib.rna4r_table_to_host(self.h, out.ctypes.data, compact), "rna4r_table_to_host")
        return out

    def enable_kernel_timing(self, on: bool = True):
        _check(self.lib.rna4r_enable_kernel_timing(self.h, int(on)), "rna4r_enable_kernel_timing")

    def last_fill_kernel_ms(self) -> float:
        ms = ctypes.c_float(0)
        _check(self.lib.rna4r_last_fill_kernel_ms(self.h, ctypes.byref(ms)), "rna4r_last_fill_kernel_ms")
        return float(ms.value)

    def set_max_blocks(self, blocks: int):
        _check(self.lib.rna4r_set_max_blocks(self.h, int(blocks)), "rna4r_set_max_blocks")

    def microbench_lookups(self, variant: int, iters: int = 4000, blocks_per_sm: int = 0, stream=None):
        """rna4r_microbench_lookups: (milliseconds, lookups executed) of the bare lookup sequence on every SM."""
        ms, n = ctypes.c_float(0), ctypes.c_double(0)
        ws = self.workspace(256)
        _check(self.lib.rna4r_microbench_lookups(self.h, variant, iters, blocks_per_sm, ws.data_ptr(), _stream_ptr(stream),
                                                 ctypes.byref(ms), ctypes.byref(n)), "rna4r_microbench_lookups")
        return float(ms.value), float(n.value)

    def set_trace(self, max_tiles: int):
        _check(self.lib.rna4r_set_trace(self.h, int(max_tiles)), "rna4r_set_trace")

    def trace(self, tiles: int) -> np.ndarray:
        out = np.zeros((tiles, int(os.environ.get("RNA4R_TRACE_WORDS", "8"))), dtype=np.uint64)
        _check(self.lib.rna4r_trace_to_host(self.h, out.ctypes.data, tiles), "rna4r_trace_to_host")
        return out

    def last_launch_count(self) -> int:
        return self.lib.rna4r_last_launch_count(self.h)

    # -- workspace ---------------------------------------------------------------------------
    def workspace(self, nbytes: int):
        """A cached torch uint8 device buffer of at least nbytes (caller-owned memory of the ABI)."""
        import torch
        if self._ws is None or self._ws.numel() < nbytes:
            self._ws = None
            self._ws = torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=f"cuda:{self.device}")
        return self._ws

    def workspace_bytes(self, n_max: int, count: int = 1, flags: int = 0) -> int:
        return self.lib.rna4r_workspace_bytes(self.h, n_max, count, flags)

    def set_max_blocks_per_sm(self, blocks_per_sm: int):
        _check(self.lib.rna4r_set_max_blocks_per_sm(self.h, int(blocks_per_sm)), "rna4r_set_max_blocks_per_sm")

    def workspace_bytes_batch(self, lens: np.ndarray) -> int:
        lens = np.ascontiguousarray(lens, dtype=np.int32)
        return self.lib.rna4r_workspace_bytes_batch(self.h, lens.ctypes.data, len(lens))

    def workspace_bytes_host(self, lens: np.ndarray, table_dtype: int = TABLE_NONE) -> int:
        lens = np.ascontiguousarray(lens, dtype=np.int32)
        return self.lib.rna4r_workspace_bytes_host(self.h, lens.ctypes.data, len(lens), table_dtype)

    # -- folds (device buffers) ----------------------------------------------------------------
    def fold(self, seq_dev, n: int | None = None, score_out=None, table_dtype: int = TABLE_NONE, table_out=None,
             workspace=None, stream=None):
        """rna4r_fold.  seq_dev: torch uint8 CUDA tensor of ASCII bases.  Enqueues only; returns
        (score tensor int32[1], table tensor or None)."""
        import torch
        n = int(seq_dev.numel()) if n is None else n
        dev = f"cuda:{self.device}"
        if score_out is None:
            score_out = torch.empty(1, dtype=torch.int32, device=dev)
        if table_dtype != TABLE_NONE and table_out is None:
            table_out = torch.empty((n, n), dtype=torch.int16 if table_dtype == TABLE_INT16 else torch.int32, device=dev)
        if workspace is None:
            workspace = self.workspace(self.workspace_bytes(n, 1))
        _check(self.lib.rna4r_fold(self.h, seq_dev.data_ptr() if n else None, n, score_out.data_ptr(),
                                   table_out.data_ptr() if table_out is not None else None, table_dtype,
                                   workspace.data_ptr(), workspace.numel(), _stream_ptr(stream)), "rna4r_fold")
        return score_out, table_out

    def fold_static_setup(self, stream=None):
        """rna4r_fold_static_setup: once per device (and per q), before fold_static."""
        _check(self.lib.rna4r_fold_static_setup(self.h, _stream_ptr(stream)), "rna4r_fold_static_setup")

    def fold_static_max_n(self) -> int:
        n = self.lib.rna4r_fold_static_max_n(self.h)
        _check(min(n, 0), "rna4r_fold_static_max_n")
        return n

    def fold_static(self, seq_dev, score_out, n: int | None = None, stream=None):
        """rna4r_fold_static: score-only fold out of the library's static scratch array; allocates nothing (the caller
        passes the int32[1] CUDA tensor score_out).  Enqueues only."""
        n = int(seq_dev.numel()) if n is None else n
        _check(self.lib.rna4r_fold_static(self.h, seq_dev.data_ptr() if n else None, n, score_out.data_ptr(),
                                          _stream_ptr(stream)), "rna4r_fold_static")
        return score_out

    def fold_batch(self, seqs_dev, offsets_dev, lens_host: np.ndarray, scores_out=None, workspace=None, stream=None,
                   status_out=None):
        """rna4r_fold_batch (rna4r_fold_batch_status when status_out, an int32[count] CUDA tensor, is given).
        Enqueues only; returns the int32[count] score tensor."""
        import torch
        lens_host = np.ascontiguousarray(lens_host, dtype=np.int32)
        count = len(lens_host)
        if scores_out is None:
            scores_out = torch.empty(max(count, 1), dtype=torch.int32, device=f"cuda:{self.device}")
        if workspace is None:
            workspace = self.workspace(self.workspace_bytes_batch(lens_host))
        if status_out is not None:
            _check(self.lib.rna4r_fold_batch_status(self.h, seqs_dev.data_ptr(), offsets_dev.data_ptr(), lens_host.ctypes.data,
                                                    count, scores_out.data_ptr(), status_out.data_ptr(), workspace.data_ptr(),
                                                    workspace.numel(), _stream_ptr(stream)), "rna4r_fold_batch_status")
        else:
            _check(self.lib.rna4r_fold_batch(self.h, seqs_dev.data_ptr(), offsets_dev.data_ptr(), lens_host.ctypes.data, count,
                                             scores_out.data_ptr(), workspace.data_ptr(), workspace.numel(),
                                             _stream_ptr(stream)), "rna4r_fold_batch")
        return scores_out[:count]

    # -- traceback --------------------------------------------------------------------------------
    def traceback(self, seq_dev, table, n: int | None = None, stream=None):
        """rna4r_traceback.  seq_dev: torch uint8 CUDA tensor; table: the (n, n) int16/int32 CUDA tensor
        rna4r_fold wrote.  Enqueues only; returns (pairs int32[n] with -1 = unpaired, npairs int32[1])."""
        import torch
        n = int(seq_dev.numel()) if n is None else n
        dev = f"cuda:{self.device}"
        dt = TABLE_INT16 if table.dtype == torch.int16 else TABLE_INT32
        pairs = torch.empty(max(n, 1), dtype=torch.int32, device=dev)
        npairs = torch.empty(1, dtype=torch.int32, device=dev)
        ws = torch.empty(self.lib.rna4r_traceback_workspace_bytes(self.h, n), dtype=torch.uint8, device=dev)
        _check(self.lib.rna4r_traceback(self.h, seq_dev.data_ptr() if n else None, n, table.data_ptr() if n else None, dt,
                                        pairs.data_ptr(), npairs.data_ptr(), ws.data_ptr(), ws.numel(), _stream_ptr(stream)),
               "rna4r_traceback")
        self._tb_ws = ws          # keep the scratch alive until the stream has run
        return pairs[:n], npairs

    # -- folds (host buffers; copies inside, synchronises) ---------------------------------------
    def fold_host(self, seq_host, table_dtype: int = TABLE_NONE, workspace=None, stream=None, score_host=None, table_host=None):
        """rna4r_fold_host.  seq_host: bytes / numpy uint8 / pinned torch uint8 CPU tensor.
        Returns (int score, numpy table or None)."""
        import torch
        if isinstance(seq_host, (bytes, bytearray, str)):
            seq_host = np.frombuffer(seq_host.encode() if isinstance(seq_host, str) else bytes(seq_host), dtype=np.uint8)
        if isinstance(seq_host, np.ndarray):
            seq_ptr, n = seq_host.ctypes.data, int(seq_host.size)
        else:
            seq_ptr, n = seq_host.data_ptr(), int(seq_host.numel())
        lens = np.array([n], dtype=np.int32)
        if workspace is None:
            workspace = self.workspace(self.workspace_bytes_host(lens, table_dtype))
        if score_host is None:
            score_host = torch.empty(1, dtype=torch.int32).pin_memory()
        if table_dtype != TABLE_NONE and table_host is None:
            table_host = torch.empty((n, n), dtype=torch.int16 if table_dtype == TABLE_INT16 else torch.int32).pin_memory()
        _check(self.lib.rna4r_fold_host(self.h, seq_ptr if n else None, n, score_host.data_ptr(),
                                        table_host.data_ptr() if table_host is not None else None, table_dtype,
                                        workspace.data_ptr(), workspace.numel(), _stream_ptr(stream)), "rna4r_fold_host")
        return int(score_host[0]), (table_host.numpy() if table_host is not None else None)

    def fold_batch_host(self, seqs_host, lens_host: np.ndarray, workspace=None, stream=None, scores_host=None):
        """rna4r_fold_batch_host.  seqs_host: concatenated bases (numpy uint8 or pinned torch tensor)."""
        import torch
        lens_host = np.ascontiguousarray(lens_host, dtype=np.int32)
        count = len(lens_host)
        seq_ptr = seqs_host.ctypes.data if isinstance(seqs_host, np.ndarray) else seqs_host.data_ptr()
        if workspace is None:
            workspace = self.workspace(self.workspace_bytes_host(lens_host, TABLE_NONE))
        if scores_host is None:
            scores_host = torch.empty(max(count, 1), dtype=torch.int32).pin_memory()
        _check(self.lib.rna4r_fold_batch_host(self.h, seq_ptr, lens_host.ctypes.data, count, scores_host.data_ptr(),
                                              workspace.data_ptr(), workspace.numel(), _stream_ptr(stream)),
               "rna4r_fold_batch_host")
        return scores_host[:count].numpy().copy()


def rna4r_prepare(q: int, device: int = 0, engine: int = ENGINE_AUTO) -> Rna4r:
    return Rna4r(q, device, engine)
