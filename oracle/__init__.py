"""ctypes front end of the CPU oracle (``dnatok_oracle.c``).  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from the
CUDA package and the CUDA package imports nothing from here.

All arithmetic lives in the C file; this module only marshals numpy arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dnatok_oracle.c")
_SRC_EXT = os.path.join(_HERE, "dnatok_oracle_ext.c")      # SURVEY.md 8(f) operations
_LIB = os.path.join(_HERE, "liboracle.so")
_lock = threading.Lock()
_lib = None

SINGLE_NT, KMER, BPE = 0, 1, 2
TAIL_PER_BASE, TAIL_DROP, TAIL_UNK = 0, 1, 2
PAD_LEFT, PAD_RIGHT = 0, 1
CLS_N, CLS_UNK, CLS_SKIP = 4, 5, 255

_u8p = ctypes.POINTER(ctypes.c_uint8)
_i64p = ctypes.POINTER(ctypes.c_int64)
_i32p = ctypes.POINTER(ctypes.c_int32)


def build(force: bool = False) -> str:
    """Compile dnatok_oracle.c -> liboracle.so (gcc -O2) if missing or stale."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_EXT)):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fPIC", "-shared", "-std=c11", "-Wall", "-o", tmp, _SRC, _SRC_EXT])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    with _lock:
        if _lib is None:
            lib = ctypes.CDLL(build())
            lib.oracle_default_lut.argtypes = [_u8p]
            lib.oracle_default_lut.restype = None
            lib.oracle_strip.argtypes = [_u8p, ctypes.c_int64, _u8p, ctypes.c_int, _u8p]
            lib.oracle_strip.restype = ctypes.c_int64
            lib.oracle_single_nt.argtypes = [_u8p, ctypes.c_int64, _i32p, ctypes.c_int32, _i32p]
            lib.oracle_single_nt.restype = ctypes.c_int64
            lib.oracle_kmer.argtypes = [_u8p, ctypes.c_int64, ctypes.c_int, ctypes.c_int32, ctypes.c_int32,
                                        ctypes.c_int, _i32p]
            lib.oracle_kmer.restype = ctypes.c_int64
            lib.oracle_bpe_table_create.argtypes = [_i32p, ctypes.c_int32]
            lib.oracle_bpe_table_create.restype = ctypes.c_void_p
            lib.oracle_bpe_table_destroy.argtypes = [ctypes.c_void_p]
            lib.oracle_bpe_table_destroy.restype = None
            lib.oracle_bpe.argtypes = [_u8p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int32,
                                       ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, _i32p]
            lib.oracle_bpe.restype = ctypes.c_int64
            lib.oracle_encode.argtypes = [_u8p, _i64p, ctypes.c_int64, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                          ctypes.c_int, _u8p, _i32p, ctypes.c_int32, ctypes.c_int32,
                                          ctypes.c_int32, ctypes.c_void_p, ctypes.c_int32, _i32p, _i64p]
            lib.oracle_encode.restype = ctypes.c_int64
            lib.oracle_pad.argtypes = [_i32p, _i64p, ctypes.c_int64, ctypes.c_int32, ctypes.c_int, ctypes.c_int32,
                                       _i32p, _u8p]
            lib.oracle_pad.restype = None
            lib.oracle_kmer_table.argtypes = [_u8p, ctypes.c_int64, ctypes.c_int, _i32p, _i32p, ctypes.c_int32,
                                              ctypes.c_int, _i32p]
            lib.oracle_kmer_table.restype = ctypes.c_int64
            lib.oracle_microbatch_rows.argtypes = [ctypes.c_int64] * 3
            lib.oracle_microbatch_rows.restype = ctypes.c_int64
            lib.oracle_embed.argtypes = [_i32p, ctypes.c_int64, _u8p, ctypes.c_int64, ctypes.c_int64, _u8p]
            lib.oracle_embed.restype = None
            lib.oracle_revcomp.argtypes = [_u8p, _i64p, ctypes.c_int64, _u8p]
            lib.oracle_revcomp.restype = None
            lib.oracle_decode.argtypes = [_i32p, _i64p, ctypes.c_int64, ctypes.c_int, ctypes.c_int, _i32p, ctypes.c_int32,
                                          ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, _i32p, ctypes.c_int32, _u8p,
                                          ctypes.c_int64, _i64p]
            lib.oracle_decode.restype = ctypes.c_int64
            lib.oracle_widen.argtypes = [_i32p, ctypes.c_int64, _i64p]
            lib.oracle_widen.restype = None
            _lib = lib
    return _lib


def _p(a: np.ndarray, t):
    return a.ctypes.data_as(t)


def default_lut() -> np.ndarray:
    lut = np.empty(256, dtype=np.uint8)
    _load().oracle_default_lut(_p(lut, _u8p))
    return lut


@dataclass
class Config:
    """Mirror of the create-time spec; defaults are the BASELINE.json vocabulary (Q1)."""
    mode: int = SINGLE_NT
    k: int = 1
    tail_policy: int = TAIL_PER_BASE
    strip_headers: bool = True
    class_lut: np.ndarray = field(default_factory=default_lut)
    pad_id: int = 0
    unk_id: int = 1
    nt_ids: tuple = (2, 3, 4, 5, 6)
    base_id: int = 3
    n_id: int = 2
    merges: np.ndarray | None = None
    seq_len: int = 0
    pad_side: int = PAD_LEFT


class _RuleTable:
    def __init__(self, merges):
        m = np.ascontiguousarray(merges, dtype=np.int32).reshape(-1, 2)
        self.n = int(m.shape[0])
        self.ptr = _load().oracle_bpe_table_create(_p(m, _i32p), self.n)
        if not self.ptr:
            raise ValueError("invalid merge table (Q12: parts must be earlier tokens, pairs unique)")

    def __del__(self):
        if getattr(self, "ptr", None):
            _load().oracle_bpe_table_destroy(self.ptr)
            self.ptr = None


def strip(rec: bytes | np.ndarray, cfg: Config | None = None) -> np.ndarray:
    """Step 1 on one record -> kept class codes (uint8)."""
    cfg = cfg or Config()
    rec = np.frombuffer(bytes(rec), dtype=np.uint8) if not isinstance(rec, np.ndarray) else np.ascontiguousarray(rec)
    cls = np.empty(max(rec.size, 1), dtype=np.uint8)
    lut = np.ascontiguousarray(cfg.class_lut, dtype=np.uint8)
    n = _load().oracle_strip(_p(rec, _u8p), rec.size, _p(lut, _u8p), int(cfg.strip_headers), _p(cls, _u8p))
    return cls[:n].copy()


def encode(data: np.ndarray | bytes, offsets, cfg: Config) -> tuple[np.ndarray, np.ndarray]:
    """Steps 1-5 on a batch -> (ids int32[total], out_offsets int64[n_records+1])."""
    if not isinstance(data, np.ndarray):
        data = np.frombuffer(bytes(data), dtype=np.uint8)
    data = np.ascontiguousarray(data, dtype=np.uint8)
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    n_records = offsets.size - 1
    cap = max(int(offsets[-1] - offsets[0]), 1)
    ids = np.empty(cap, dtype=np.int32)
    out_offsets = np.empty(n_records + 1, dtype=np.int64)
    lut = np.ascontiguousarray(cfg.class_lut, dtype=np.uint8)
    nt = np.asarray(cfg.nt_ids, dtype=np.int32)
    table = _RuleTable(cfg.merges) if cfg.mode == BPE else None
    if data.size == 0:
        data = np.zeros(1, dtype=np.uint8)
    total = _load().oracle_encode(_p(data, _u8p), _p(offsets, _i64p), n_records, cfg.mode, cfg.k, cfg.tail_policy,
                                  int(cfg.strip_headers), _p(lut, _u8p), _p(nt, _i32p), cfg.base_id, cfg.n_id,
                                  cfg.unk_id, table.ptr if table else None, table.n if table else 0,
                                  _p(ids, _i32p), _p(out_offsets, _i64p))
    if total < 0:
        raise MemoryError
    return ids[:total].copy(), out_offsets


def encode_one(rec: bytes, cfg: Config) -> np.ndarray:
    """Steps 1-4 on a single record."""
    b = np.frombuffer(bytes(rec), dtype=np.uint8)
    return encode(b, np.array([0, b.size], dtype=np.int64), cfg)[0]


def pad(ids: np.ndarray, out_offsets: np.ndarray, cfg: Config) -> tuple[np.ndarray, np.ndarray]:
    """Step 6 -> (batch_ids int32[n_records, seq_len], mask uint8[n_records, seq_len])."""
    ids = np.ascontiguousarray(ids, dtype=np.int32)
    out_offsets = np.ascontiguousarray(out_offsets, dtype=np.int64)
    n = out_offsets.size - 1
    batch = np.empty((n, cfg.seq_len), dtype=np.int32)
    mask = np.empty((n, cfg.seq_len), dtype=np.uint8)
    if ids.size == 0:
        ids = np.zeros(1, dtype=np.int32)
    _load().oracle_pad(_p(ids, _i32p), _p(out_offsets, _i64p), n, cfg.seq_len, cfg.pad_side, cfg.pad_id,
                       _p(batch, _i32p), _p(mask, _u8p))
    return batch, mask


# ------------------------------------------------------------------------------------------- SURVEY.md 8(f)
def encode_kmer_table(data, offsets, cfg: Config, kmer_lut: np.ndarray) -> tuple[np.ndarray, np.ndarray]:
    """f1: steps 1, 5 as encode(); step 3 through the base-5 table kmer_lut[5^k] (one record at a time)."""
    if not isinstance(data, np.ndarray):
        data = np.frombuffer(bytes(data), dtype=np.uint8)
    data = np.ascontiguousarray(data, dtype=np.uint8)
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    kl = np.ascontiguousarray(kmer_lut, dtype=np.int32)
    assert kl.size == 5 ** cfg.k
    nt = np.asarray(cfg.nt_ids, dtype=np.int32)
    lut = np.ascontiguousarray(cfg.class_lut, dtype=np.uint8)
    lib = _load()
    parts, out = [], np.zeros(offsets.size, dtype=np.int64)
    for r in range(offsets.size - 1):
        rec = np.ascontiguousarray(data[int(offsets[r]): int(offsets[r + 1])])
        cls = np.empty(max(rec.size, 1), dtype=np.uint8)
        n = lib.oracle_strip(_p(rec if rec.size else cls, _u8p), rec.size, _p(lut, _u8p), int(cfg.strip_headers), _p(cls, _u8p))
        ids = np.empty(max(n, 1), dtype=np.int32)
        t = lib.oracle_kmer_table(_p(cls, _u8p), n, cfg.k, _p(kl, _i32p), _p(nt, _i32p), cfg.unk_id, cfg.tail_policy,
                                  _p(ids, _i32p))
        parts.append(ids[:t].copy())
        out[r + 1] = out[r] + t
    return (np.concatenate(parts) if parts else np.zeros(0, np.int32)), out


def microbatch_rows(b_emb: int, m_tokens: int, t_len: int) -> int:
    """f2: rows per embedding call, b = min(B_emb, max(1, floor(M / T')))."""
    return int(_load().oracle_microbatch_rows(int(b_emb), int(m_tokens), int(t_len)))


def embed(ids: np.ndarray, table: np.ndarray) -> np.ndarray:
    """f2: out[..., :] = table[ids[...], :] (rows copied bit for bit; an ID outside the table gives a zero row)."""
    ids32 = np.ascontiguousarray(ids, dtype=np.int32)
    table = np.ascontiguousarray(table)
    row_bytes = table.shape[1] * table.itemsize
    out = np.empty(ids32.shape + (table.shape[1],), dtype=table.dtype)
    if ids32.size:
        _load().oracle_embed(_p(ids32, _i32p), ids32.size, _p(table.view(np.uint8).reshape(-1), _u8p), table.shape[0],
                             row_bytes, _p(out.view(np.uint8).reshape(-1), _u8p))
    return out


def revcomp(data, offsets) -> np.ndarray:
    """f3: every record reversed and complemented (same layout as the input)."""
    if not isinstance(data, np.ndarray):
        data = np.frombuffer(bytes(data), dtype=np.uint8)
    data = np.ascontiguousarray(data, dtype=np.uint8)
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    out = data.copy()
    if data.size:
        _load().oracle_revcomp(_p(data, _u8p), _p(offsets, _i64p), offsets.size - 1, _p(out, _u8p))
    return out


def decode(ids: np.ndarray, out_offsets: np.ndarray, cfg: Config) -> tuple[np.ndarray, np.ndarray]:
    """f3: token IDs -> upper-case bases (uint8[total], byte_offsets int64[n_records + 1])."""
    ids = np.ascontiguousarray(ids, dtype=np.int32)
    out_offsets = np.ascontiguousarray(out_offsets, dtype=np.int64)
    n = out_offsets.size - 1
    nt = np.asarray(cfg.nt_ids, dtype=np.int32)
    merges = np.ascontiguousarray(cfg.merges if cfg.merges is not None else np.zeros((0, 2)), dtype=np.int32).reshape(-1, 2)
    boff = np.zeros(n + 1, dtype=np.int64)
    cap = 1 << 16
    idp = ids if ids.size else np.zeros(1, np.int32)
    mp = merges if merges.size else np.zeros((1, 2), np.int32)
    while True:
        out = np.empty(cap, dtype=np.uint8)
        tot = _load().oracle_decode(_p(idp, _i32p), _p(out_offsets, _i64p), n, cfg.mode, cfg.k, _p(nt, _i32p), cfg.base_id,
                                    cfg.n_id, cfg.unk_id, cfg.pad_id, _p(mp, _i32p), merges.shape[0], _p(out, _u8p), cap,
                                    _p(boff, _i64p))
        if tot >= 0:
            return out[:tot].copy(), boff
        cap *= 4


def widen(ids: np.ndarray) -> np.ndarray:
    """f4: int32 IDs -> int64."""
    ids = np.ascontiguousarray(ids, dtype=np.int32)
    out = np.empty(ids.shape, dtype=np.int64)
    if ids.size:
        _load().oracle_widen(_p(ids.reshape(-1), _i32p), ids.size, _p(out.reshape(-1), _i64p))
    return out
