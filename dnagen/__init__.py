"""Seeded synthetic inputs for the five BASELINE.json configs (inputs only).

The generators live in ``dnagen.c`` (xoshiro256** per record, seeded from
(seed, config, record index)); this module compiles that file with gcc on first
use, lays out record offsets and fans the per-record fill out over threads.

Nothing here computes a token: neither ``oracle/`` nor the CUDA library imports
this package, and it imports neither of them.  Tests and ``bench.py`` hand the
same generated buffers to both sides.

Recipes (readings Q18-Q24) are restated in DESIGN.md.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dnagen.c")
_LIB = os.path.join(_HERE, "libdnagen.so")
_lock = threading.Lock()
_lib = None

_u8p = ctypes.POINTER(ctypes.c_uint8)
_i64p = ctypes.POINTER(ctypes.c_int64)
_i32p = ctypes.POINTER(ctypes.c_int32)
_f64p = ctypes.POINTER(ctypes.c_double)


def build(force: bool = False) -> str:
    """Compile dnagen.c -> libdnagen.so (gcc -O2) if missing or stale."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fPIC", "-shared", "-std=c11", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    with _lock:
        if _lib is None:
            lib = ctypes.CDLL(build())
            lib.dnagen_markov_table.argtypes = [ctypes.c_uint64, _f64p]
            lib.dnagen_markov_table.restype = None
            lib.dnagen_record.restype = ctypes.c_int64
            lib.dnagen_record.argtypes = [_u8p, ctypes.c_int64, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint64,
                                          ctypes.c_int, _f64p, ctypes.c_double, ctypes.c_double,
                                          ctypes.c_int, ctypes.c_int, ctypes.c_int]
            lib.dnagen_fill_records.restype = None
            lib.dnagen_fill_records.argtypes = [_u8p, _i64p, _i64p, ctypes.c_int64, ctypes.c_int64,
                                                ctypes.c_uint64, ctypes.c_uint64, ctypes.c_int, _f64p,
                                                ctypes.c_double, ctypes.c_double,
                                                ctypes.c_int, ctypes.c_int, ctypes.c_int]
            lib.dnagen_n_runs.restype = ctypes.c_int64
            lib.dnagen_n_runs.argtypes = [_u8p, ctypes.c_int64, ctypes.c_uint64, ctypes.c_double, ctypes.c_int]
            lib.dnagen_lengths_uniform.restype = None
            lib.dnagen_lengths_uniform.argtypes = [_i64p, ctypes.c_int64, ctypes.c_int64, ctypes.c_int64,
                                                   ctypes.c_uint64, ctypes.c_uint64]
            lib.dnagen_lengths_loguniform.restype = ctypes.c_int64
            lib.dnagen_lengths_loguniform.argtypes = [_i64p, ctypes.c_int64, ctypes.c_int64, ctypes.c_int64,
                                                      ctypes.c_int64, ctypes.c_uint64, ctypes.c_uint64]
            lib.dnagen_merge_table.restype = ctypes.c_int
            lib.dnagen_merge_table.argtypes = [_i32p, ctypes.c_int, ctypes.c_int64, ctypes.c_uint64, _f64p]
            _lib = lib
    return _lib


def _p(a: np.ndarray, t):
    return a.ctypes.data_as(t)


@dataclass
class Workload:
    """bytes: uint8[n_bytes] flat buffer; offsets: int64[n_records+1] record starts."""
    name: str
    data: np.ndarray
    offsets: np.ndarray
    n_bases: np.ndarray                      # kept bases per record (what the generator wrote)
    meta: dict = field(default_factory=dict)
    merges: np.ndarray | None = None         # config 4 only: int32[n_merges, 2]

    @property
    def n_records(self) -> int:
        return int(self.offsets.shape[0] - 1)

    @property
    def n_bytes(self) -> int:
        return int(self.offsets[-1])


def markov_table(seed: int = 0) -> np.ndarray:
    cum = np.empty(64, dtype=np.float64)
    _load().dnagen_markov_table(seed, _p(cum, _f64p))
    return cum


def _record_bytes(n_bases: np.ndarray, header: bool, line_width: int, term_newline: bool) -> np.ndarray:
    nb = n_bases.astype(np.int64)
    out = nb.copy()
    if line_width > 0:
        out += (nb + line_width - 1) // line_width
    elif term_newline:
        out += 1
    if header:
        idx = np.arange(nb.shape[0])
        # len(">r%d len=%d\n") = 2 + digits(idx) + 5 + digits(len) + 1
        dig = lambda v: np.where(v > 0, np.floor(np.log10(np.maximum(v, 1))).astype(np.int64) + 1, 1)
        out += 8 + dig(idx) + dig(nb)
    return out


def _fill(data: np.ndarray, offsets: np.ndarray, n_bases: np.ndarray, seed: int, cfg: int, model: int,
          cum, p_n: float, p_lower: float, header: bool, line_width: int, term_newline: bool,
          threads: int | None = None) -> None:
    lib = _load()
    n = int(n_bases.shape[0])
    threads = threads or min(32, os.cpu_count() or 1)
    cump = _p(cum, _f64p) if cum is not None else None
    # split by bytes, not by record count, so threads get equal work
    targets = np.linspace(0, int(offsets[-1]), threads * 4 + 1)
    cuts = np.unique(np.searchsorted(offsets[:-1], targets, side="left"))
    cuts = np.unique(np.concatenate([[0], cuts, [n]]))
    dp, op, nbp = _p(data, _u8p), _p(offsets, _i64p), _p(n_bases, _i64p)

    def job(i):
        lib.dnagen_fill_records(dp, op, nbp, int(cuts[i]), int(cuts[i + 1]), seed, cfg, model, cump,
                                p_n, p_lower, int(header), line_width, int(term_newline))

    with ThreadPoolExecutor(max_workers=threads) as ex:
        list(ex.map(job, range(len(cuts) - 1)))


def _make(name: str, n_bases: np.ndarray, seed: int, cfg: int, model: int, cum, p_n: float, p_lower: float,
          header: bool, line_width: int, term_newline: bool, out: np.ndarray | None = None,
          threads: int | None = None) -> Workload:
    n_bases = np.ascontiguousarray(n_bases, dtype=np.int64)
    rb = _record_bytes(n_bases, header, line_width, term_newline)
    offsets = np.zeros(n_bases.shape[0] + 1, dtype=np.int64)
    np.cumsum(rb, out=offsets[1:])
    total = int(offsets[-1])
    if out is None:
        data = np.empty(total, dtype=np.uint8)
    else:
        assert out.dtype == np.uint8 and out.size >= total
        data = out[:total]
    _fill(data, offsets, n_bases, seed, cfg, model, cum, p_n, p_lower, header, line_width, term_newline, threads)
    return Workload(name, data, offsets, n_bases, meta={"seed": seed, "config": cfg})


# --------------------------------------------------------------------------- configs
def config1(seed: int = 0, n_records: int = 16, bases: int = 65536) -> Workload:
    """BJ config 1 (Q24): i.i.d. ACGT, 1 % N, 5 % lowercase, '\\n' every 60 bases and after the last line."""
    nb = np.full(n_records, bases, dtype=np.int64)
    return _make("config1", nb, seed, 1, 0, None, 0.01, 0.05, False, 60, False)


def config2(seed: int = 0, n_records: int = 4096, bases: int = 65536, n_frac: float = 0.005,
            out: np.ndarray | None = None) -> Workload:
    """BJ config 2 (Q22, Q23): order-2 Markov, GC 0.41, N runs 1..500 covering 0.5 %, no newlines."""
    nb = np.full(n_records, bases, dtype=np.int64)
    w = _make("config2", nb, seed, 2, 1, markov_table(seed), 0.0, 0.0, False, 0, False, out=out)
    if n_frac > 0:
        w.meta["n_runs"] = int(_load().dnagen_n_runs(_p(w.data, _u8p), w.n_bytes, seed, n_frac, 500))
    return w


def config3(seed: int = 0, total_bases: int = 1 << 30, lo: int = 1000, hi: int = 131072) -> Workload:
    """BJ config 3 (Q19): uniform ACGT, lengths log-uniform [1000, 131072] until total_bases, FASTA layout
    ('>r<i> len=<L>' header line, 80-column lines)."""
    max_n = total_bases // lo + 2
    buf = np.empty(max_n, dtype=np.int64)
    n = int(_load().dnagen_lengths_loguniform(_p(buf, _i64p), max_n, total_bases, lo, hi, seed, 3))
    return _make("config3", buf[:n].copy(), seed, 3, 0, None, 0.0, 0.0, True, 80, False)


def merge_table(seed: int = 0, n_merges: int = 4092, corpus_bases: int = 256 * 1024) -> np.ndarray:
    """Config 4 merge table (Q21): int32[n_merges, 2]; rule r merges (left, right) into token 4 + r."""
    m = np.zeros((n_merges, 2), dtype=np.int32)
    cum = markov_table(seed)
    got = _load().dnagen_merge_table(_p(m, _i32p), n_merges, corpus_bases, seed, _p(cum, _f64p))
    assert got == n_merges, f"corpus too small: only {got} merges"
    return m


def config4(seed: int = 0, n_reads: int = 65536, lo: int = 500, hi: int = 1500, n_merges: int = 4092,
            corpus_bases: int = 256 * 1024) -> Workload:
    """BJ config 4 (Q20-Q23): reads uniform [500, 1500], order-2 Markov + 2 % N i.i.d., no newlines."""
    nb = np.empty(n_reads, dtype=np.int64)
    _load().dnagen_lengths_uniform(_p(nb, _i64p), n_reads, lo, hi, seed, 4)
    w = _make("config4", nb, seed, 4, 1, markov_table(seed), 0.02, 0.0, False, 0, False)
    w.merges = merge_table(seed, n_merges, corpus_bases)
    return w


def config5(seed: int = 0, total_bytes: int = 8 << 30, bases: int = 32768, out: np.ndarray | None = None,
            threads: int | None = None) -> Workload:
    """BJ config 5 (Q18): records of `bases` uniform ACGT + '\\n'; the last record takes what is left of
    total_bytes and has no terminator."""
    full = total_bytes // (bases + 1)
    rest = total_bytes - full * (bases + 1)
    data = out[:total_bytes] if out is not None else np.empty(total_bytes, dtype=np.uint8)
    assert data.dtype == np.uint8 and data.size == total_bytes
    nb = np.full(full, bases, dtype=np.int64)
    w = _make("config5", nb, seed, 5, 0, None, 0.0, 0.0, False, 0, True, out=data, threads=threads)
    if rest:    # ragged last record: `rest` bases, no terminator
        tail_off = int(w.offsets[-1])
        _load().dnagen_record(_p(data[tail_off:], _u8p), rest, seed, 5, full, 0, None, 0.0, 0.0, 0, 0, 0)
        w.offsets = np.concatenate([w.offsets, [total_bytes]]).astype(np.int64)
        w.n_bases = np.concatenate([nb, [rest]]).astype(np.int64)
        w.data = data
    return w
