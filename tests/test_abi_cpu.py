"""CPU-side checks of the boundary: the C-ABI library builds/loads without a GPU and exports every symbol
include/dnatok.h declares; the ctypes mirror of dnatok_config matches the C layout.  No compute calls."""
import ctypes
import os
import re

import pytest

import paper_2601_05531_b200 as dn

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "dnatok.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(dnatok_[a-z_]+)\s*\(", src)) - {"dnatok_batch_fn"})


def test_library_loads_and_exports_every_declared_symbol():
    L = dn.lib()
    syms = declared_symbols()
    assert {"dnatok_create", "dnatok_destroy", "dnatok_encode", "dnatok_pad", "dnatok_stream_encode"} <= set(syms)
    for s in syms:
        assert hasattr(L, s), s
    assert "sm_100a" in dn.dnatok_version()


def test_python_binding_has_the_same_names():
    for s in declared_symbols():
        assert hasattr(dn, s), s


def test_config_default_and_struct_layout():
    c = dn.dnatok_config_default(dn.KMER, 6)
    assert c.struct_size == ctypes.sizeof(dn._CConfig)          # C sizeof == ctypes mirror
    assert (c.mode, c.k, c.id_dtype, c.strip_headers) == (dn.KMER, 6, dn.I32, 1)
    assert (c.pad_id, c.unk_id, c.base_id, c.n_id) == (0, 1, 3, 2)  # BASELINE.json vocabulary (Q1)
    assert list(c.nt_ids) == [2, 3, 4, 5, 6]
    lut = bytes(c.class_lut)
    for up, lo, v in zip(b"ACGTN", b"acgtn", range(5)):
        assert lut[up] == v and lut[lo] == v
    assert lut[10] == 255 and lut[13] == 255 and sum(1 for b in lut if b == 5) == 244


def test_sources_are_sm100a_only_and_have_no_cpu_fallback():
    from paper_2601_05531_b200 import _build
    assert "arch=compute_100a,code=sm_100a" in " ".join(_build.FLAGS)
    pkg = os.path.join(ROOT, "paper_2601_05531_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "dnagen" not in text, f
