"""Pins of the SURVEY.md 8(f) oracle functions (oracle/dnatok_oracle_ext.c) against what the paper and the mathematics
fix: hand-worked values, Python string operations, numpy closed forms and library routines, involutions, round trips.
None of them re-types the oracle's loops."""
import random

import numpy as np
import pytest

import oracle

COMP = bytes.maketrans(b"ACGTURYKMBVDHSWNacgturykmbvdhswn", b"TGCAAYRMKVBHDSWNtgcaayrmkvbhdswn")


# ------------------------------------------------------------------------------------------- f3 reverse complement
def test_revcomp_handworked():
    # PAPER.md:325-327 (reverse complement); worked by hand: reverse, then A<->T, C<->G, N stays
    assert oracle.revcomp(b"ACGTN", [0, 5]).tobytes() == b"NACGT"
    assert oracle.revcomp(b"AAACGATTACA", [0, 4, 11]).tobytes() == b"GTTT" + b"TGTAATC"
    assert oracle.revcomp(b"acgRYkmBVdhSWnU", [0, 15]).tobytes() == b"AnWSdhBVkmRYcgt"
    assert oracle.revcomp(b"", [0, 0]).tobytes() == b""
    assert oracle.revcomp(b"AC", [0, 0, 2, 2]).tobytes() == b"GT"


@pytest.mark.parametrize("seed", range(8))
def test_revcomp_equals_python_string_ops_and_is_an_involution(seed):
    rng = random.Random(seed)
    alphabet = b"ACGTNacgtnRYKMBVDHSWU-*\n>x"
    recs = [bytes(rng.choice(alphabet) for _ in range(rng.choice([0, 1, 2, 7, rng.randrange(0, 300)]))) for _ in range(40)]
    data = b"".join(recs)
    offs = np.cumsum([0] + [len(r) for r in recs])
    got = oracle.revcomp(data, offs).tobytes()
    assert got == b"".join(r.translate(COMP)[::-1] for r in recs)
    assert oracle.revcomp(got, offs).tobytes() == data.replace(b"U", b"T").replace(b"u", b"t")   # U -> A -> T: the only non-involutive byte


# ------------------------------------------------------------------------------------------- f3 decode
def test_decode_handworked_example():
    # the ids of the SURVEY.md 8(c) hand-worked example, spelled back (PAPER.md:315-317 inverse vocabulary table)
    cfg = oracle.Config(mode=oracle.SINGLE_NT)
    b, o = oracle.decode([2, 3, 4, 5, 6, 2, 3, 4, 4, 2, 5, 5, 2, 3, 2], [0, 8, 15], cfg)
    assert b.tobytes() == b"ACGTNACG" + b"GATTACA" and o.tolist() == [0, 8, 15]
    cfg = oracle.Config(mode=oracle.KMER, k=3)
    b, o = oracle.decode([9, 1, 68, 69, 38, 52, 67], [0, 4, 7], cfg)       # ACG, (TNa) -> NNN, c, g | GAT, TAC, A
    assert b.tobytes() == b"ACGNNNCG" + b"GATTACA" and o.tolist() == [0, 8, 15]
    merges = np.array([[0, 1], [4, 2], [2, 3]], dtype=np.int32)              # (A,C)->4, (AC,G)->5, (G,T)->6
    cfg = oracle.Config(mode=oracle.BPE, merges=merges)
    b, o = oracle.decode([8, 6, 2, 8, 5, 3, 6, 6, 7, 3], [0, 4, 10], cfg)
    assert b.tobytes() == b"ACGTNACG" + b"GATTACA" and o.tolist() == [0, 8, 15]


def test_decode_skips_pad_and_spells_unknown_ids_as_n():
    cfg = oracle.Config(mode=oracle.KMER, k=2)
    b, o = oracle.decode([0, 0, 3, 18, 19 + 4, 1, 9999], [0, 7], cfg)        # pad pad AA TT tail-N UNK unknown
    assert b.tobytes() == b"AATTN" + b"NN" + b"NN" and o.tolist() == [0, 9]
    cfg = oracle.Config(mode=oracle.SINGLE_NT)
    assert oracle.decode([1, 0, 77, 5], [0, 4], cfg)[0].tobytes() == b"NNT"
    cfg = oracle.Config(mode=oracle.BPE, merges=np.array([[0, 0], [4, 4]], dtype=np.int32))
    assert oracle.decode([8, 2, 1, 7, 3 + 6], [0, 5], cfg)[0].tobytes() == b"AAAA" + b"N" + b"N" + b"AA" + b"N"


@pytest.mark.parametrize("mode,k", [(oracle.SINGLE_NT, 1), (oracle.KMER, 1), (oracle.KMER, 4), (oracle.KMER, 6), (oracle.KMER, 8),
                                    (oracle.BPE, 1)])
def test_decode_round_trip_on_n_free_fasta(mode, k):
    rng = random.Random(100 + k + mode)
    import dnagen
    merges = dnagen.merge_table(seed=2, n_merges=300, corpus_bases=8192) if mode == oracle.BPE else None
    recs, clean = [], []
    for i in range(30):
        n = rng.choice([0, 1, 5, rng.randrange(0, 400)])
        seq = "".join(rng.choice("ACGTacgt") for _ in range(n))
        clean.append(seq.upper().encode())
        recs.append((f">r{i}\n" + "\n".join(seq[j: j + 60] for j in range(0, n, 60)) + "\n").encode())
    data = b"".join(recs)
    offs = np.cumsum([0] + [len(r) for r in recs])
    cfg = oracle.Config(mode=mode, k=k, merges=merges)
    ids, out = oracle.encode(data, offs, cfg)
    b, bo = oracle.decode(ids, out, cfg)
    assert b.tobytes() == b"".join(clean)
    assert bo.tolist() == np.cumsum([0] + [len(c) for c in clean]).tolist()


# ------------------------------------------------------------------------------------------- f1 table-driven k-mers
def closed_form_table(k, base_id=3, unk_id=1):
    """kmer_lut[5^k] that reproduces the base-4 closed form: a window without digit 4 -> base_id + base-4 code, else unk."""
    lut = np.empty(5 ** k, dtype=np.int32)
    for code in range(5 ** k):
        d = [(code // 5 ** (k - 1 - i)) % 5 for i in range(k)]
        lut[code] = unk_id if 4 in d else base_id + sum(x * 4 ** (k - 1 - i) for i, x in enumerate(d))
    return lut


def test_kmer_table_handworked():
    # PAPER.md:88 Alg. 1 l.18-22: base-5 window code, first base most significant: AC -> 0*5+1 = 1, NT -> 4*5+3 = 23, xG -> 4*5+2 = 22
    lut = np.arange(1000, 1025, dtype=np.int32)
    cfg = oracle.Config(mode=oracle.KMER, k=2)
    ids, out = oracle.encode_kmer_table(b"ACNT-Gt", [0, 7], cfg, lut)
    assert ids.tolist() == [1001, 1023, 1022, 5] and out.tolist() == [0, 4]           # tail 't' -> nt_ids[T] = 5
    ids, out = oracle.encode_kmer_table(b">h\nAC\nGT\n", [0, 9], cfg, lut)
    assert ids.tolist() == [1001, 1000 + 2 * 5 + 3] and out.tolist() == [0, 2]


@pytest.mark.parametrize("k", [1, 2, 3, 6])
def test_kmer_table_with_the_closed_form_table_equals_the_base4_encoder(k):
    import dnagen
    w = dnagen.config3(total_bases=30_000, lo=50, hi=3000, seed=k)
    data = w.data.copy()
    rng = np.random.default_rng(k)
    pos = rng.integers(0, data.size, size=300)
    data[pos[data[pos] != 10]] = ord("N")                                              # sprinkle N (not over line breaks)
    cfg4 = oracle.Config(mode=oracle.KMER, k=k)
    want_ids, want_off = oracle.encode(data, w.offsets, cfg4)
    cfg5 = oracle.Config(mode=oracle.KMER, k=k, nt_ids=tuple(3 + 4 ** k + c for c in range(5)))
    ids, out = oracle.encode_kmer_table(data, w.offsets, cfg5, closed_form_table(k))
    assert np.array_equal(ids, want_ids) and np.array_equal(out, want_off)


def test_kmer_table_equals_numpy_base5_gather():
    rng = np.random.default_rng(3)
    k = 4
    n = 4000
    digits = rng.integers(0, 5, size=n)
    seq = np.frombuffer(b"ACGTN", dtype=np.uint8)[digits]
    lut = rng.integers(0, 100000, size=5 ** k).astype(np.int32)
    cfg = oracle.Config(mode=oracle.KMER, k=k)
    ids, _ = oracle.encode_kmer_table(seq, [0, n], cfg, lut)
    codes = digits.reshape(-1, k) @ (5 ** np.arange(k - 1, -1, -1))
    assert np.array_equal(ids, lut[codes])


# ------------------------------------------------------------------------------------------- f2 embedding gather
def test_microbatch_rule_values():
    # PAPER.md:181 / Alg. 2 l.17: b = min(B_emb, max(1, floor(M / T'))), M = 1,048,576; evaluated by hand
    M = 1_048_576
    assert oracle.microbatch_rows(4096, M, 512) == 2048
    assert oracle.microbatch_rows(8192, M, 512) == 2048
    assert oracle.microbatch_rows(2048, M, 2048) == 512
    assert oracle.microbatch_rows(64, M, 512) == 64
    assert oracle.microbatch_rows(4096, M, 8192) == 128
    assert oracle.microbatch_rows(4096, M, 3_000_000) == 1
    assert oracle.microbatch_rows(4096, M, 1000) == 1048


@pytest.mark.parametrize("dtype", [np.float32, np.float16, np.uint16])
def test_embed_equals_numpy_take(dtype):
    rng = np.random.default_rng(0)
    table = rng.standard_normal((11, 128)).astype(np.float32)
    table = table.astype(dtype) if dtype != np.uint16 else (table.view(np.uint32) >> 16).astype(np.uint16)   # bf16 bit patterns
    ids = rng.integers(0, 11, size=(7, 33)).astype(np.int32)
    got = oracle.embed(ids, table)
    assert got.shape == (7, 33, 128) and np.array_equal(got, table[ids])
    bad = np.array([[-1, 11, 3]], dtype=np.int32)
    got = oracle.embed(bad, table)
    assert not got[0, 0].any() and not got[0, 1].any() and np.array_equal(got[0, 2], table[3])


# ------------------------------------------------------------------------------------------- f4 widening
def test_widen_equals_astype():
    rng = np.random.default_rng(1)
    ids = rng.integers(-2 ** 31, 2 ** 31 - 1, size=(5, 77)).astype(np.int32)
    assert np.array_equal(oracle.widen(ids), ids.astype(np.int64)) and oracle.widen(ids).dtype == np.int64
