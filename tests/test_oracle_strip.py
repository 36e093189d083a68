"""Pins for oracle steps 1-2 (classify, strip, single-nt).  None of these re-types the oracle's loops:
they use the paper's printed self-test, hand-worked cases, and an independent
restatement of stripping with Python string operations (SURVEY.md 8(c) "What pins each part")."""
import json
import os
import random

import numpy as np
import pytest

import oracle

ACGT = "ACGT"


def nt(s, **kw):
    return oracle.encode_one(s.encode() if isinstance(s, str) else s, oracle.Config(mode=oracle.SINGLE_NT, **kw)).tolist()


def test_selftest_string_paper_and_baseline_vocab(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "selftest_acgtn.json")))
    for key in ("paper_fallback_lut", "baseline_vocab"):
        v = g[key]
        assert nt(g["string"], nt_ids=tuple(v["nt_ids"]), unk_id=v["unk_id"]) == v["ids"]


def test_lut_enumerates_256_bytes():
    # PAPER.md:88 Alg. 1 l.9-12: exactly the 10 letters map to base classes; Q2/Q3: '\n','\r' SKIP, rest UNK
    lut = oracle.default_lut()
    base = {b for b in range(256) if lut[b] <= 4}
    assert base == {ord(c) for c in "ACGTNacgtn"}
    assert {b for b in range(256) if lut[b] == oracle.CLS_SKIP} == {10, 13}
    assert sum(1 for b in range(256) if lut[b] == oracle.CLS_UNK) == 244
    for up, lo, c in zip("ACGTN", "acgtn", range(5)):
        assert lut[ord(up)] == c and lut[ord(lo)] == c


def test_every_other_byte_is_unk_and_emits_a_token():
    # Q2: IUPAC codes, U, '-', '*', space, tab, digits, bytes >= 0x80 are UNK and each emits unk_id
    for b in list(b"RYKMSWBDHVU-* \t0123456789") + [0x00, 0x7F, 0x80, 0xFF]:
        assert nt(bytes([65, b, 67]), strip_headers=False) == [2, 1, 3], b


def test_case_invariance():
    rng = random.Random(1)
    for _ in range(50):
        s = "".join(rng.choice("ACGTNacgtnRy-") for _ in range(rng.randrange(0, 200)))
        assert nt(s) == nt(s.upper())


def strip_by_string_ops(rec: bytes, strip_headers=True) -> bytes:
    """Independent restatement (Q3-Q5): split on '\\n'; a line is a header if, after removing leading
    '\\r' bytes (SKIP bytes leave line_start unchanged), it starts with '>'; drop those lines; remove the
    remaining '\\r'; join."""
    out = []
    for line in rec.split(b"\n"):
        if strip_headers and line.lstrip(b"\r").startswith(b">"):
            continue
        out.append(line.replace(b"\r", b""))
    return b"".join(out)


@pytest.mark.parametrize("seed", range(30))
def test_strip_equals_string_restatement(seed):
    rng = random.Random(seed)
    alphabet = "ACGTNacgtn" * 3 + "\n\n\n>>\r Rx1"
    rec = "".join(rng.choice(alphabet) for _ in range(rng.randrange(0, 400))).encode()
    for sh in (True, False):
        clean = strip_by_string_ops(rec, sh)
        assert nt(rec, strip_headers=sh) == nt(clean, strip_headers=False), (rec, sh)
        assert len(nt(rec, strip_headers=sh)) == len(clean)


def test_line_width_invariance():
    rng = random.Random(7)
    seq = "".join(rng.choice("ACGTN") for _ in range(1000))
    want = nt(seq)
    for w in (1, 60, 80):
        wrapped = "\n".join(seq[i:i + w] for i in range(0, len(seq), w))
        assert nt(wrapped) == want
        assert nt(wrapped + "\n") == want
        assert nt(">hdr\n" + wrapped + "\n") == want


def test_hand_cases():
    assert nt("") == []
    assert nt(">only a header\n") == []
    assert nt(">header without newline ACGT") == []          # Q4: runs to the record's end
    assert nt("\n\nAC\n\n\nGT\n\n") == [2, 3, 4, 5]           # blank lines
    assert nt("AC>GT\n") == [2, 3, 1, 4, 5]                   # '>' in mid-line is an ordinary UNK byte
    assert nt("AC\r\nGT\r\n") == [2, 3, 4, 5]                 # CRLF (Q3)
    assert nt(">h\r\nAC\r\n>h2\r\nGT") == [2, 3, 4, 5]        # CRLF with headers
    assert nt("A\r>C\n") == [2, 1, 3]                         # '\r' does not start a line (Q3)
    assert nt("\r>hdr\nAC") == [2, 3]                         # SKIP at line start leaves line_start set
    assert nt(">h1\n>h2\nAC\n>h3\nGT") == [2, 3, 4, 5]        # consecutive headers
    assert nt(">h\nAC", strip_headers=False) == [1, 1, 2, 3]  # headers kept as UNK bytes when stripping is off
    assert nt("ACGT" * 3) == [2, 3, 4, 5] * 3


def test_header_state_does_not_leak_across_records():
    # Q4/Q5: record boundaries come only from rec_offsets; a header with no '\n' ends at the record's end
    data = b">hdr no newlineACGT"
    offs = np.array([0, 15, 19], dtype=np.int64)
    ids, out = oracle.encode(data, offs, oracle.Config(mode=oracle.SINGLE_NT))
    assert ids.tolist() == [2, 3, 4, 5] and out.tolist() == [0, 0, 4]


def test_decode_round_trip_and_length():
    rng = random.Random(3)
    inv = {2: "A", 3: "C", 4: "G", 5: "T", 6: "N"}
    for _ in range(20):
        seq = "".join(rng.choice("ACGTNacgtn") for _ in range(rng.randrange(1, 300)))
        fasta = ">x\n" + "\n".join(seq[i:i + 13] for i in range(0, len(seq), 13)) + "\n"
        ids = nt(fasta)
        assert len(ids) == len(seq)
        assert "".join(inv[i] for i in ids) == seq.upper()


def test_handworked_example_kept_classes_and_single_nt(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "handworked_example.json")))
    data = (g["record0"] + g["record1"]).encode()
    assert len(data) == 23
    for r, rec in enumerate((g["record0"], g["record1"])):
        assert oracle.strip(rec.encode()).tolist() == g["kept_classes"][r]
    ids, out = oracle.encode(data, g["rec_offsets"], oracle.Config(mode=oracle.SINGLE_NT))
    assert ids.tolist() == g["single_nt"]["ids"] and out.tolist() == g["single_nt"]["out_offsets"]


def test_custom_lut_skip_byte():
    # a custom LUT may mark any byte SKIP; only '\n' sets line_start (8(c) step 1)
    lut = oracle.default_lut()
    lut[ord("-")] = oracle.CLS_SKIP
    assert nt("A-C-\n->x\nG", class_lut=lut) == [2, 3, 4]     # '-' after '\n' leaves line_start: '>x' is a header
    assert nt("A->C", class_lut=lut) == [2, 1, 3]             # '-' mid-line does not create a line start
