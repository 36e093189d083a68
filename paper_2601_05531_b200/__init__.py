"""paper_2601_05531_b200 -- B200-native DNATok hot path (raw ASCII DNA bytes -> token-ID streams).

Thin Python binding over the C-ABI in ``include/dnatok.h`` (``libdnatok.so``, hand-written CUDA for
sm_100a).  Argument marshalling only: every step of the path runs in the library's kernels.  PyTorch is
used for device memory and streams, nothing else.  There is no CPU fallback: if the library cannot be
loaded, importing the binding's entry points raises.

    import torch, paper_2601_05531_b200 as dn
    tok = dn.DNATok(mode="kmer", k=6)
    ids, out_offsets = tok.encode(d_bytes, d_rec_offsets)          # enqueue only, no sync
    batch, mask = dn.DNATok(mode="kmer", k=6, seq_len=8192).encode_padded(d_bytes, d_rec_offsets)
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass, field
from typing import Callable, Optional, Sequence

import numpy as np

from . import _build

__all__ = [
    "DNATok", "Config", "Batch", "DNATokError", "lib", "library_path",
    "SINGLE_NT", "KMER", "BPE", "I16", "I32", "TAIL_PER_BASE", "TAIL_DROP", "TAIL_UNK", "PAD_LEFT", "PAD_RIGHT",
    "dnatok_create", "dnatok_destroy", "dnatok_encode", "dnatok_pad", "dnatok_encode_pad", "dnatok_stream_encode", "dnatok_check",
    "dnatok_last_error", "dnatok_launch_count", "dnatok_version", "dnatok_config_default", "dnatok_set_super_tile", "dnatok_set_grid_cap", "dnatok_set_fast_path", "dnatok_fast_path_taken",
    "dnatok_stream_encode_from", "dnatok_revcomp", "dnatok_decode", "dnatok_decode_static", "DECODE_STATIC_MAX_RECORDS", "dnatok_microbatch_rows", "dnatok_embed", "dnatok_widen_ids",
]

SINGLE_NT, KMER, BPE = 0, 1, 2
I16, I32 = 2, 4
DECODE_STATIC_MAX_RECORDS = 1 << 20     # dnatok.h DNATOK_DECODE_STATIC_MAX_RECORDS
TAIL_PER_BASE, TAIL_DROP, TAIL_UNK = 0, 1, 2
PAD_LEFT, PAD_RIGHT = 0, 1
OK, EINVAL, ENOMEM, ECUDA, ECAPACITY, ESTATE = range(6)
_STATUS_NAMES = {0: "OK", 1: "EINVAL", 2: "ENOMEM", 3: "ECUDA", 4: "ECAPACITY", 5: "ESTATE"}
_MODES = {"single_nt": SINGLE_NT, "single": SINGLE_NT, "kmer": KMER, "bpe": BPE}


class DNATokError(RuntimeError):
    def __init__(self, code: int, msg: str = ""):
        self.code = code
        super().__init__(f"dnatok: {_STATUS_NAMES.get(code, code)}{': ' + msg if msg else ''}")


class _CConfig(ctypes.Structure):
    _fields_ = [
        ("struct_size", ctypes.c_uint32), ("mode", ctypes.c_int32), ("k", ctypes.c_int32),
        ("id_dtype", ctypes.c_int32), ("class_lut", ctypes.c_uint8 * 256), ("strip_headers", ctypes.c_int32),
        ("pad_id", ctypes.c_int32), ("unk_id", ctypes.c_int32), ("nt_ids", ctypes.c_int32 * 5),
        ("base_id", ctypes.c_int32), ("n_id", ctypes.c_int32), ("tail_policy", ctypes.c_int32),
        ("merges", ctypes.POINTER(ctypes.c_int32)), ("n_merges", ctypes.c_int32),
        ("seq_len", ctypes.c_int32), ("pad_side", ctypes.c_int32), ("max_record_bytes", ctypes.c_int64),
        ("kmer_lut", ctypes.POINTER(ctypes.c_int32)), ("kmer_lut_len", ctypes.c_int64),
    ]


class _CBatch(ctypes.Structure):
    _fields_ = [
        ("first_record", ctypes.c_int64), ("n_records", ctypes.c_int64), ("d_ids", ctypes.c_void_p),
        ("d_out_offsets", ctypes.c_void_p), ("d_batch_ids", ctypes.c_void_p), ("d_mask", ctypes.c_void_p),
        ("chunk_index", ctypes.c_int64), ("stream", ctypes.c_void_p),
    ]


_BATCH_FN = ctypes.CFUNCTYPE(None, ctypes.c_void_p, ctypes.POINTER(_CBatch))
_FILL_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_int64, ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p)
_MICROBATCH_FN = ctypes.CFUNCTYPE(None, ctypes.c_void_p, ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p)
_lib = None
SUPER_TILE = 0      # sub-tiles per super-tile applied to new DNATok handles (0 = automatic); a tuning knob, see dnatok.h
FAST_PATH = 1       # dnatok_set_fast_path value applied to new DNATok handles (1 = library default; a test knob, see dnatok.h)
GRID_CAP = 0        # cap on persistent CTAs per launch applied to new DNATok handles (0 = none); a test knob, see dnatok.h


def library_path() -> str:
    return _build.LIB


def lib() -> ctypes.CDLL:
    """Load libdnatok.so (building it with nvcc if the sources are newer).  Raises if that fails: there is
    no fallback path."""
    global _lib
    if _lib is None:
        try:
            path = _build.build()
        except Exception as e:  # no nvcc on this box: the prebuilt library must be present
            if not os.path.exists(_build.LIB):
                raise ImportError(f"libdnatok.so is missing and could not be built: {e}") from e
            path = _build.LIB
        L = ctypes.CDLL(path)
        vp, i64, i32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32
        L.dnatok_version.restype = ctypes.c_char_p
        L.dnatok_version.argtypes = []
        L.dnatok_config_default.restype = None
        L.dnatok_config_default.argtypes = [ctypes.POINTER(_CConfig), i32, i32]
        L.dnatok_create.restype = ctypes.c_int
        L.dnatok_create.argtypes = [ctypes.POINTER(_CConfig), ctypes.c_int, ctypes.POINTER(vp)]
        L.dnatok_destroy.restype = ctypes.c_int
        L.dnatok_destroy.argtypes = [vp]
        L.dnatok_encode.restype = ctypes.c_int
        L.dnatok_encode.argtypes = [vp, vp, i64, vp, i64, vp, i64, vp, vp]
        L.dnatok_pad.restype = ctypes.c_int
        L.dnatok_pad.argtypes = [vp, vp, vp, i64, vp, vp, vp]
        L.dnatok_encode_pad.restype = ctypes.c_int
        L.dnatok_encode_pad.argtypes = [vp, vp, i64, vp, i64, vp, i64, vp, vp, vp, vp]
        L.dnatok_stream_encode.restype = ctypes.c_int
        L.dnatok_stream_encode.argtypes = [vp, vp, i64, vp, i64, i64, ctypes.c_int, i64, _BATCH_FN, vp]
        L.dnatok_stream_encode_from.restype = ctypes.c_int
        L.dnatok_stream_encode_from.argtypes = [vp, _FILL_FN, vp, i64, vp, i64, i64, ctypes.c_int, i64, _BATCH_FN, vp]
        L.dnatok_check.restype = ctypes.c_int
        L.dnatok_check.argtypes = [vp, vp]
        L.dnatok_last_error.restype = ctypes.c_char_p
        L.dnatok_last_error.argtypes = [vp]
        L.dnatok_set_super_tile.restype = ctypes.c_int
        L.dnatok_set_super_tile.argtypes = [vp, i32]
        L.dnatok_set_grid_cap.restype = ctypes.c_int
        L.dnatok_set_grid_cap.argtypes = [vp, i32]
        L.dnatok_set_fast_path.restype = ctypes.c_int
        L.dnatok_set_fast_path.argtypes = [vp, i32]
        L.dnatok_fast_path_taken.restype = ctypes.c_int
        L.dnatok_fast_path_taken.argtypes = [vp, vp]
        L.dnatok_launch_count.restype = i64
        L.dnatok_launch_count.argtypes = [vp]
        L.dnatok_revcomp.restype = ctypes.c_int
        L.dnatok_revcomp.argtypes = [vp, vp, i64, vp, i64, vp, vp]
        L.dnatok_decode.restype = ctypes.c_int
        L.dnatok_decode.argtypes = [vp, vp, vp, i64, vp, i64, vp, vp]
        L.dnatok_decode_static.restype = ctypes.c_int
        L.dnatok_decode_static.argtypes = [vp, vp, vp, i64, vp, i64, vp, vp]
        L.dnatok_microbatch_rows.restype = i64
        L.dnatok_microbatch_rows.argtypes = [i64, i64, i64]
        L.dnatok_embed.restype = ctypes.c_int
        L.dnatok_embed.argtypes = [vp, vp, i64, i64, vp, i64, i64, vp, i64, i64, _MICROBATCH_FN, vp, vp]
        L.dnatok_widen_ids.restype = ctypes.c_int
        L.dnatok_widen_ids.argtypes = [vp, vp, i64, vp, vp]
        _lib = L
    return _lib


# ------------------------------------------------------------------ same-name thin wrappers (C-ABI 1:1)
def dnatok_version() -> str:
    return lib().dnatok_version().decode()


def dnatok_config_default(mode: int, k: int) -> _CConfig:
    c = _CConfig()
    lib().dnatok_config_default(ctypes.byref(c), mode, k)
    return c


def dnatok_create(cfg: _CConfig, device: int = 0) -> int:
    h = ctypes.c_void_p()
    rc = lib().dnatok_create(ctypes.byref(cfg), device, ctypes.byref(h))
    if rc != OK:
        raise DNATokError(rc, "dnatok_create rejected the configuration")
    return h.value


def dnatok_destroy(h: int) -> None:
    lib().dnatok_destroy(h)


def _chk(h: int, rc: int) -> None:
    if rc != OK:
        raise DNATokError(rc, lib().dnatok_last_error(h).decode())


def dnatok_encode(h: int, d_bytes: int, n_bytes: int, d_rec_offsets: int, n_records: int, d_ids_out: int,
                  ids_capacity: int, d_out_offsets: int, stream: int = 0) -> None:
    _chk(h, lib().dnatok_encode(h, d_bytes, n_bytes, d_rec_offsets, n_records, d_ids_out, ids_capacity,
                                d_out_offsets, stream))


def dnatok_pad(h: int, d_ids: int, d_out_offsets: int, n_records: int, d_batch_ids: int, d_mask: int,
               stream: int = 0) -> None:
    _chk(h, lib().dnatok_pad(h, d_ids, d_out_offsets, n_records, d_batch_ids, d_mask, stream))


def dnatok_encode_pad(h: int, d_bytes: int, n_bytes: int, d_rec_offsets: int, n_records: int, d_ids_out: int,
                      ids_capacity: int, d_out_offsets: int, d_batch_ids: int, d_mask: int, stream: int = 0) -> None:
    _chk(h, lib().dnatok_encode_pad(h, d_bytes, n_bytes, d_rec_offsets, n_records, d_ids_out, ids_capacity,
                                    d_out_offsets, d_batch_ids, d_mask, stream))


def dnatok_stream_encode(h: int, h_pinned: int, n_bytes: int, h_rec_offsets: int, n_records: int,
                         chunk_bytes: int, n_streams: int, max_rows_per_chunk: int, on_batch, user: int = 0) -> None:
    _chk(h, lib().dnatok_stream_encode(h, h_pinned, n_bytes, h_rec_offsets, n_records, chunk_bytes, n_streams,
                                       max_rows_per_chunk, on_batch, user))


def dnatok_stream_encode_from(h: int, fill, fill_user: int, n_bytes: int, h_rec_offsets: int, n_records: int,
                              chunk_bytes: int, n_streams: int, max_rows_per_chunk: int, on_batch, user: int = 0) -> None:
    _chk(h, lib().dnatok_stream_encode_from(h, fill, fill_user, n_bytes, h_rec_offsets, n_records, chunk_bytes, n_streams,
                                            max_rows_per_chunk, on_batch, user))


def dnatok_check(h: int, stream: int = 0) -> None:
    _chk(h, lib().dnatok_check(h, stream))


def dnatok_last_error(h: int) -> str:
    return lib().dnatok_last_error(h).decode()


def dnatok_set_super_tile(h: int, sub_tiles: int) -> None:
    _chk(h, lib().dnatok_set_super_tile(h, int(sub_tiles)))


def dnatok_set_grid_cap(h: int, max_ctas: int) -> None:
    _chk(h, lib().dnatok_set_grid_cap(h, int(max_ctas)))


def dnatok_set_fast_path(h: int, enable: int) -> None:
    _chk(h, lib().dnatok_set_fast_path(h, int(enable)))


def dnatok_fast_path_taken(h: int, stream: int = 0) -> bool:
    rc = lib().dnatok_fast_path_taken(h, stream)
    if rc < 0:
        _chk(h, rc)
    return rc == 1


def dnatok_launch_count(h: int) -> int:
    return int(lib().dnatok_launch_count(h))


def dnatok_revcomp(h: int, d_bytes: int, n_bytes: int, d_rec_offsets: int, n_records: int, d_out: int, stream: int = 0) -> None:
    _chk(h, lib().dnatok_revcomp(h, d_bytes, n_bytes, d_rec_offsets, n_records, d_out, stream))


def dnatok_decode(h: int, d_ids: int, d_out_offsets: int, n_records: int, d_bytes_out: int, bytes_capacity: int,
                  d_byte_offsets: int, stream: int = 0) -> None:
    _chk(h, lib().dnatok_decode(h, d_ids, d_out_offsets, n_records, d_bytes_out, bytes_capacity, d_byte_offsets, stream))


def dnatok_decode_static(h: int, d_ids: int, d_out_offsets: int, n_records: int, d_bytes_out: int, bytes_capacity: int,
                         d_byte_offsets: int, stream: int = 0) -> None:
    _chk(h, lib().dnatok_decode_static(h, d_ids, d_out_offsets, n_records, d_bytes_out, bytes_capacity, d_byte_offsets, stream))


def dnatok_microbatch_rows(b_emb: int, m_tokens: int, t_len: int) -> int:
    return int(lib().dnatok_microbatch_rows(int(b_emb), int(m_tokens), int(t_len)))


def dnatok_embed(h: int, d_ids: int, n_rows: int, t_len: int, d_table: int, vocab: int, row_bytes: int, d_out: int,
                 b_emb: int, m_tokens: int, on_microbatch=None, user: int = 0, stream: int = 0) -> None:
    cb = on_microbatch if on_microbatch is not None else _MICROBATCH_FN()
    _chk(h, lib().dnatok_embed(h, d_ids, n_rows, t_len, d_table, vocab, row_bytes, d_out, b_emb, m_tokens, cb, user, stream))


def dnatok_widen_ids(h: int, d_ids: int, n: int, d_out: int, stream: int = 0) -> None:
    _chk(h, lib().dnatok_widen_ids(h, d_ids, n, d_out, stream))


# ------------------------------------------------------------------ convenience layer
@dataclass
class Config:
    mode: int | str = KMER
    k: int = 6
    id_dtype: int = I32
    class_lut: Optional[Sequence[int]] = None      # None => library default
    strip_headers: bool = True
    pad_id: int = 0
    unk_id: int = 1
    nt_ids: Sequence[int] = (2, 3, 4, 5, 6)
    base_id: int = 3
    n_id: int = 2
    tail_policy: int = TAIL_PER_BASE
    merges: Optional[np.ndarray] = None            # BPE: int32[n_merges, 2]
    seq_len: int = 0
    pad_side: int = PAD_LEFT
    max_record_bytes: int = 1 << 20
    kmer_lut: Optional[np.ndarray] = None          # KMER: int32[5^k] id table (None: base-4 closed form)

    def to_c(self) -> tuple[_CConfig, object]:
        mode = _MODES[self.mode] if isinstance(self.mode, str) else int(self.mode)
        c = dnatok_config_default(mode, int(self.k))
        c.id_dtype = int(self.id_dtype)
        if self.class_lut is not None:
            lut = np.asarray(self.class_lut, dtype=np.uint8)
            assert lut.shape == (256,)
            ctypes.memmove(c.class_lut, lut.ctypes.data, 256)
        c.strip_headers = int(bool(self.strip_headers))
        c.pad_id, c.unk_id, c.base_id, c.n_id = int(self.pad_id), int(self.unk_id), int(self.base_id), int(self.n_id)
        for i, v in enumerate(self.nt_ids):
            c.nt_ids[i] = int(v)
        c.tail_policy = int(self.tail_policy)
        keep = None
        if self.merges is not None:
            keep = np.ascontiguousarray(self.merges, dtype=np.int32).reshape(-1, 2)
            c.merges = keep.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))
            c.n_merges = int(keep.shape[0])
        c.seq_len, c.pad_side = int(self.seq_len), int(self.pad_side)
        c.max_record_bytes = int(self.max_record_bytes)
        if self.kmer_lut is not None:
            kl = np.ascontiguousarray(self.kmer_lut, dtype=np.int32).reshape(-1)
            c.kmer_lut = kl.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))
            c.kmer_lut_len = int(kl.size)
            keep = (keep, kl)
        return c, keep


@dataclass
class Batch:
    """One delivered batch of stream_encode; tensors alias the slot's device buffers and are valid until the
    work enqueued on `stream` inside the callback has run."""
    first_record: int
    n_records: int
    chunk_index: int
    stream: int
    ids_ptr: int
    out_offsets_ptr: int
    batch_ids_ptr: int
    mask_ptr: int
    seq_len: int
    id_dtype: int
    _keep: list = field(default_factory=list)

    def _view(self, ptr: int, shape, typestr: str):
        import torch

        class _Arr:
            pass
        a = _Arr()
        a.__cuda_array_interface__ = {"shape": tuple(shape), "typestr": typestr, "data": (ptr, False), "version": 2}
        return torch.as_tensor(a, device="cuda")

    def out_offsets(self):
        return self._view(self.out_offsets_ptr, (self.n_records + 1,), "<i8")

    def batch_ids(self):
        return self._view(self.batch_ids_ptr, (self.n_records, self.seq_len), "<i4")

    def mask(self):
        return self._view(self.mask_ptr, (self.n_records, self.seq_len), "|u1")

    def ids(self, n_tokens: int):
        return self._view(self.ids_ptr, (n_tokens,), "<i2" if self.id_dtype == I16 else "<i4")


class DNATok:
    """Handle + torch-tensor marshalling around the C-ABI."""

    def __init__(self, cfg: Config | None = None, device: int = 0, **kw):
        import torch
        self._torch = torch
        self.cfg = cfg if cfg is not None else Config(**kw)
        c, self._keep = self.cfg.to_c()
        self.device = device
        self.h = dnatok_create(c, device)
        if SUPER_TILE:
            dnatok_set_super_tile(self.h, SUPER_TILE)
        if GRID_CAP:
            dnatok_set_grid_cap(self.h, GRID_CAP)
        if FAST_PATH != 1:
            dnatok_set_fast_path(self.h, FAST_PATH)
        self.id_torch_dtype = torch.int16 if self.cfg.id_dtype == I16 else torch.int32

    def close(self) -> None:
        if getattr(self, "h", None):
            dnatok_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _stream(self, stream) -> int:
        if stream is None:
            return int(self._torch.cuda.current_stream(self.device).cuda_stream)
        return int(getattr(stream, "cuda_stream", stream))

    def encode(self, d_bytes, d_rec_offsets, ids_out=None, out_offsets=None, stream=None):
        """Steps 1-5.  d_bytes: cuda uint8[n_bytes]; d_rec_offsets: cuda int64[n_records+1].
        Returns (ids_out, out_offsets): ids_out has capacity n_bytes unless given; the first
        out_offsets[-1] entries are valid.  Enqueue only."""
        t = self._torch
        assert d_bytes.is_cuda and d_bytes.dtype == t.uint8 and d_bytes.is_contiguous()
        assert d_rec_offsets.is_cuda and d_rec_offsets.dtype == t.int64 and d_rec_offsets.is_contiguous()
        n_bytes, n_rec = d_bytes.numel(), d_rec_offsets.numel() - 1
        if ids_out is None:
            ids_out = t.empty(max(n_bytes, 1), dtype=self.id_torch_dtype, device=d_bytes.device)
        if out_offsets is None:
            out_offsets = t.empty(n_rec + 1, dtype=t.int64, device=d_bytes.device)
        assert ids_out.dtype == self.id_torch_dtype and out_offsets.dtype == t.int64
        dnatok_encode(self.h, d_bytes.data_ptr(), n_bytes, d_rec_offsets.data_ptr(), n_rec, ids_out.data_ptr(),
                      ids_out.numel(), out_offsets.data_ptr(), self._stream(stream))
        return ids_out, out_offsets

    def pad(self, ids, out_offsets, batch_ids=None, mask=None, stream=None):
        """Step 6 -> (batch_ids int32[n_records, seq_len], mask uint8[n_records, seq_len]).  Enqueue only."""
        t = self._torch
        n_rec = out_offsets.numel() - 1
        L = self.cfg.seq_len
        if batch_ids is None:
            batch_ids = t.empty((n_rec, L), dtype=t.int32, device=ids.device)
        if mask is None:
            mask = t.empty((n_rec, L), dtype=t.uint8, device=ids.device)
        dnatok_pad(self.h, ids.data_ptr(), out_offsets.data_ptr(), n_rec, batch_ids.data_ptr(), mask.data_ptr(),
                   self._stream(stream))
        return batch_ids, mask

    def encode_padded(self, d_bytes, d_rec_offsets, ids_out=None, out_offsets=None, batch_ids=None, mask=None, stream=None):
        """Steps 1-6 in one call -> (batch_ids, mask, out_offsets); the same results as encode() + pad().  ids_out is
        workspace: regular-layout inputs are written straight into the batch and leave it untouched (dnatok.h)."""
        t = self._torch
        assert d_bytes.is_cuda and d_bytes.dtype == t.uint8 and d_bytes.is_contiguous()
        assert d_rec_offsets.is_cuda and d_rec_offsets.dtype == t.int64 and d_rec_offsets.is_contiguous()
        n_bytes, n_rec = d_bytes.numel(), d_rec_offsets.numel() - 1
        L = self.cfg.seq_len
        if ids_out is None:
            ids_out = t.empty(max(n_bytes, 1), dtype=self.id_torch_dtype, device=d_bytes.device)
        if out_offsets is None:
            out_offsets = t.empty(n_rec + 1, dtype=t.int64, device=d_bytes.device)
        if batch_ids is None:
            batch_ids = t.empty((n_rec, L), dtype=t.int32, device=d_bytes.device)
        if mask is None:
            mask = t.empty((n_rec, L), dtype=t.uint8, device=d_bytes.device)
        assert ids_out.dtype == self.id_torch_dtype and out_offsets.dtype == t.int64
        dnatok_encode_pad(self.h, d_bytes.data_ptr(), n_bytes, d_rec_offsets.data_ptr(), n_rec, ids_out.data_ptr(),
                          ids_out.numel(), out_offsets.data_ptr(), batch_ids.data_ptr(), mask.data_ptr(), self._stream(stream))
        return batch_ids, mask, out_offsets

    def _batch_cb(self, on_batch):
        cfg = self.cfg

        def _cb(_user, bp):
            b = bp.contents
            if on_batch is not None:
                on_batch(Batch(b.first_record, b.n_records, b.chunk_index, b.stream or 0, b.d_ids or 0,
                               b.d_out_offsets or 0, b.d_batch_ids or 0, b.d_mask or 0, cfg.seq_len, cfg.id_dtype))
        return _BATCH_FN(_cb)

    def stream_encode_from(self, fill: Callable[[int, int, np.ndarray], None], n_bytes: int, h_rec_offsets, chunk_bytes: int,
                           n_streams: int = 4, max_rows_per_chunk: int = 0, on_batch: Callable[[Batch], None] | None = None) -> None:
        """Step 7 with a producer: fill(chunk_index, offset, dst) writes input bytes [offset, offset + dst.size) into dst, a
        numpy view of one of the handle's pinned staging slots (e.g. f.readinto(dst))."""
        offs = np.ascontiguousarray(np.asarray(h_rec_offsets), dtype=np.int64)

        def _fill(_user, i, off, n, dst):
            try:
                fill(int(i), int(off), np.ctypeslib.as_array(ctypes.cast(dst, ctypes.POINTER(ctypes.c_uint8)), shape=(int(n),)))
                return 0
            except Exception:
                return 1

        dnatok_stream_encode_from(self.h, _FILL_FN(_fill), 0, int(n_bytes), offs.ctypes.data, offs.size - 1, int(chunk_bytes),
                                  int(n_streams), int(max_rows_per_chunk), self._batch_cb(on_batch), 0)

    def stream_encode(self, h_pinned, h_rec_offsets, chunk_bytes: int, n_streams: int = 4,
                      max_rows_per_chunk: int = 0, on_batch: Callable[[Batch], None] | None = None) -> None:
        """Step 7.  h_pinned: CPU uint8 tensor or numpy array, pinned (read in place) or pageable (staged through the handle's
        pinned ring); h_rec_offsets: CPU int64 tensor / numpy array.  on_batch(Batch) runs on this thread per chunk."""
        t = self._torch
        if isinstance(h_pinned, t.Tensor):
            assert h_pinned.dtype == t.uint8 and not h_pinned.is_cuda and h_pinned.is_contiguous()
            ptr, n_bytes = h_pinned.data_ptr(), h_pinned.numel()
        else:
            ptr, n_bytes = h_pinned.ctypes.data, h_pinned.size
        offs = h_rec_offsets.numpy() if isinstance(h_rec_offsets, t.Tensor) else np.asarray(h_rec_offsets)
        offs = np.ascontiguousarray(offs, dtype=np.int64)
        cfg = self.cfg

        def _cb(_user, bp):
            b = bp.contents
            if on_batch is not None:
                on_batch(Batch(b.first_record, b.n_records, b.chunk_index, b.stream or 0, b.d_ids or 0,
                               b.d_out_offsets or 0, b.d_batch_ids or 0, b.d_mask or 0, cfg.seq_len, cfg.id_dtype))

        cb = _BATCH_FN(_cb)
        dnatok_stream_encode(self.h, ptr, n_bytes, offs.ctypes.data, offs.size - 1, int(chunk_bytes), int(n_streams),
                             int(max_rows_per_chunk), cb, 0)

    # ---- SURVEY.md 8(f) ------------------------------------------------------------------------------
    def revcomp(self, d_bytes, d_rec_offsets, out=None, stream=None):
        """Reverse complement of every record (cuda uint8, same layout).  Enqueue only."""
        t = self._torch
        if out is None:
            out = t.empty_like(d_bytes)
        dnatok_revcomp(self.h, d_bytes.data_ptr(), d_bytes.numel(), d_rec_offsets.data_ptr(), d_rec_offsets.numel() - 1,
                       out.data_ptr(), self._stream(stream))
        return out

    def decode(self, ids, out_offsets, bytes_capacity: int, stream=None):
        """Token ids -> upper-case bases: (cuda uint8[bytes_capacity], byte_offsets int64[n_records + 1]).  Enqueue only."""
        t = self._torch
        n_rec = out_offsets.numel() - 1
        out = t.empty(max(int(bytes_capacity), 1), dtype=t.uint8, device=ids.device)
        boff = t.empty(n_rec + 1, dtype=t.int64, device=ids.device)
        dnatok_decode(self.h, ids.data_ptr(), out_offsets.data_ptr(), n_rec, out.data_ptr(), int(bytes_capacity), boff.data_ptr(),
                      self._stream(stream))
        return out, boff

    def decode_static(self, ids, out_offsets, out, byte_offsets, stream=None):
        """decode() into caller-owned buffers with no device allocation anywhere in the call (dnatok_decode_static): out is
        cuda uint8[bytes_capacity], byte_offsets cuda int64[n_records + 1].  At most DECODE_STATIC_MAX_RECORDS records; calls
        that overlap on the GPU race on the library's static scratch.  Enqueue only."""
        t = self._torch
        assert out.is_cuda and out.dtype == t.uint8 and out.is_contiguous()
        assert byte_offsets.is_cuda and byte_offsets.dtype == t.int64 and byte_offsets.numel() == out_offsets.numel()
        dnatok_decode_static(self.h, ids.data_ptr(), out_offsets.data_ptr(), out_offsets.numel() - 1, out.data_ptr(), out.numel(),
                             byte_offsets.data_ptr(), self._stream(stream))
        return out, byte_offsets

    def embed(self, ids2d, table, b_emb: int = 4096, m_tokens: int = 1 << 20, on_microbatch=None, stream=None):
        """out[r, t, :] = table[ids2d[r, t], :], dnatok_microbatch_rows(b_emb, m_tokens, T) rows per launch.
        on_microbatch(first_row, n_rows) is called once per launch.  Enqueue only."""
        t = self._torch
        assert ids2d.dtype == t.int32 and ids2d.is_contiguous() and table.is_contiguous() and ids2d.dim() == 2
        n_rows, T = ids2d.shape
        out = t.empty((n_rows, T, table.shape[1]), dtype=table.dtype, device=ids2d.device)
        cb = _MICROBATCH_FN((lambda _u, r0, n, _p, _s: on_microbatch(int(r0), int(n))) if on_microbatch else (lambda *_: None))
        dnatok_embed(self.h, ids2d.data_ptr(), n_rows, T, table.data_ptr(), table.shape[0], table.shape[1] * table.element_size(),
                     out.data_ptr(), int(b_emb), int(m_tokens), cb, 0, self._stream(stream))
        return out

    def widen(self, ids32, stream=None):
        """int32 ids -> int64 (the paper's "32-bit + on-device cast").  Enqueue only."""
        t = self._torch
        out = t.empty(ids32.shape, dtype=t.int64, device=ids32.device)
        dnatok_widen_ids(self.h, ids32.data_ptr(), ids32.numel(), out.data_ptr(), self._stream(stream))
        return out

    def check(self, stream=None) -> None:
        """Synchronise the stream and raise DNATokError if the device status word reports a failure."""
        dnatok_check(self.h, self._stream(stream))

    def fast_path_taken(self, stream=None) -> bool:
        """Synchronise the stream; True if the last encode() was served by the regular-layout encoder alone."""
        return dnatok_fast_path_taken(self.h, self._stream(stream))

    @property
    def launch_count(self) -> int:
        return dnatok_launch_count(self.h)
