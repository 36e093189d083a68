"""Pins for oracle step 3 (non-overlapping k-mer pack): worked closed-form values (Q7), the numpy
reshape-matmul reduction, count identity, decode round trip, brute-force N rule, k=1 vs single-nt,
exhaustive 4^6 (SURVEY.md 8(c) "What pins each part"; BASELINE.json north_star closed form)."""
import itertools
import json
import os
import random

import numpy as np
import pytest

import oracle

CODE = {"A": 0, "C": 1, "G": 2, "T": 3}


def kmer(s, k, **kw):
    return oracle.encode_one(s.encode(), oracle.Config(mode=oracle.KMER, k=k, **kw)).tolist()


def test_worked_values(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "kmer_closed_form.json")))
    for c in g["cases"]:
        assert kmer(c["seq"], c["k"]) == [c["id"]], c
    for c in g["tails"]:
        assert kmer(c["seq"], c["k"]) == c["ids"], c


@pytest.mark.parametrize("k", [1, 2, 3, 4, 5, 6, 8, 11, 15])
def test_numpy_closed_form_reduction(k):
    # library reduction on N-free input whose length is a multiple of k
    rng = np.random.default_rng(k)
    codes = rng.integers(0, 4, size=k * 257)
    seq = "".join("ACGT"[c] for c in codes)
    want = codes.reshape(-1, k) @ (4 ** np.arange(k - 1, -1, -1, dtype=np.int64)) + 3
    assert kmer(seq, k) == want.tolist()


@pytest.mark.parametrize("k", [1, 2, 3, 6, 8])
def test_count_identity_and_tail_policies(k):
    rng = random.Random(k)
    for _ in range(20):
        n = rng.randrange(0, 100)
        seq = "".join(rng.choice("ACGTN") for _ in range(n))
        per_base = kmer(seq, k)
        assert len(per_base) == n // k + n % k
        drop = kmer(seq, k, tail_policy=oracle.TAIL_DROP)
        unk = kmer(seq, k, tail_policy=oracle.TAIL_UNK)
        assert drop == per_base[: n // k]
        assert unk == per_base[: n // k] + ([1] if n % k else [])


@pytest.mark.parametrize("k", [1, 3, 6, 8])
def test_decode_round_trip(k):
    rng = random.Random(100 + k)
    for _ in range(20):
        n = rng.randrange(1, 200)
        seq = "".join(rng.choice("ACGT") for _ in range(n))
        ids = kmer(seq, k)
        out = []
        for t in ids:
            v = t - 3
            if v < 4 ** k:
                out.append("".join("ACGT"[(v >> (2 * (k - 1 - i))) & 3] for i in range(k)))
            else:
                out.append("ACGTN"[v - 4 ** k])
        assert "".join(out) == seq


@pytest.mark.parametrize("k", [2, 6])
def test_n_rule_brute_force(k):
    # token j is UNK iff any of bases [jk, jk+k) has class >= 4; tail N -> 3 + 4^k + 4, tail UNK byte -> 1
    rng = random.Random(k)
    for _ in range(30):
        n = rng.randrange(0, 120)
        seq = "".join(rng.choice("ACGT" * 4 + "NR") for _ in range(n))
        ids = kmer(seq, k)
        for j in range(n // k):
            bad = any(ch in "NR" for ch in seq[j * k:(j + 1) * k])
            assert (ids[j] == 1) == bad
        for i, ch in enumerate(seq[(n // k) * k:]):
            want = 1 if ch == "R" else 3 + 4 ** k + "ACGTN".index(ch)
            assert ids[n // k + i] == want


def test_k1_equals_single_nt_plus_one_on_n_free_input():
    rng = random.Random(5)
    seq = "".join(rng.choice("ACGTacgt") for _ in range(500))
    single = oracle.encode_one(seq.encode(), oracle.Config(mode=oracle.SINGLE_NT)).tolist()
    assert kmer(seq, 1) == [i + 1 for i in single]


def test_exhaustive_six_mers_in_order():
    seq = "".join("".join(p) for p in itertools.product("ACGT", repeat=6))
    assert kmer(seq, 6) == list(range(3, 3 + 4 ** 6))


def test_windows_span_line_breaks_and_headers(golden_dir):
    # Q10: windows are counted from the record's first kept base, after stripping
    assert kmer(">h\nAC\nGTA\nC\n", 6) == [436]
    g = json.load(open(os.path.join(golden_dir, "handworked_example.json")))
    data = (g["record0"] + g["record1"]).encode()
    ids, out = oracle.encode(data, g["rec_offsets"], oracle.Config(mode=oracle.KMER, k=3))
    assert ids.tolist() == g["kmer3"]["ids"] and out.tolist() == g["kmer3"]["out_offsets"]


def test_record_shorter_than_k_is_all_tail():
    assert kmer("AC", 6) == [3 + 4096 + 0, 3 + 4096 + 1]
    assert kmer("", 6) == []
