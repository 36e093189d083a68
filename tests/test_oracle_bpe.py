"""Pins for oracle step 4 (BPE, lowest rank first): hand-worked cases, termination invariant, decode
round trip, and a brute force in a DIFFERENT formulation (rules applied in rank order, one full
left-to-right sweep per rule) on random strings of <= 20 bases (pins (i)-(v))."""
import json
import os
import random

import numpy as np
import pytest

import oracle


def bpe(s, merges, **kw):
    return oracle.encode_one(s.encode(), oracle.Config(mode=oracle.BPE, merges=np.array(merges, dtype=np.int32).reshape(-1, 2), **kw)).tolist()


def random_table(rng, n_merges):
    """valid table: rule r's parts are tokens < 4 + r, pairs unique"""
    seen, merges = set(), []
    while len(merges) < n_merges:
        r = len(merges)
        p = (rng.randrange(0, 4 + r), rng.randrange(0, 4 + r))
        if p in seen:
            continue
        seen.add(p)
        merges.append(p)
    return merges


def spellings(merges):
    sp = ["A", "C", "G", "T"]
    for l, r in merges:
        sp.append(sp[l] + sp[r])
    return sp


def brute_rank_order(seq, merges):
    """for r = 0..M-1 in order, sweep left to right replacing every occurrence of rule r (Q11: equivalent
    to lowest-rank-first for valid tables; shares no logic with the min-pair loop)"""
    toks = ["ACGT".index(c) for c in seq]
    for r, (l, rr) in enumerate(merges):
        out, i = [], 0
        while i < len(toks):
            if i + 1 < len(toks) and toks[i] == l and toks[i + 1] == rr:
                out.append(4 + r)
                i += 2
            else:
                out.append(toks[i])
                i += 1
        toks = out
    return [3 + t for t in toks]


def test_hand_worked(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "bpe_handworked.json")))
    for c in g["cases"]:
        assert bpe(c["seq"], c["merges"]) == c["ids"], c["why"]


def test_handworked_example_batch(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "handworked_example.json")))
    data = (g["record0"] + g["record1"]).encode()
    cfg = oracle.Config(mode=oracle.BPE, merges=np.array(g["bpe"]["merges"], dtype=np.int32), n_id=g["bpe"]["n_id"])
    ids, out = oracle.encode(data, g["rec_offsets"], cfg)
    assert ids.tolist() == g["bpe"]["ids"] and out.tolist() == g["bpe"]["out_offsets"]


@pytest.mark.parametrize("seed", range(40))
def test_brute_force_small_strings(seed):
    rng = random.Random(seed)
    merges = random_table(rng, rng.randrange(1, 12))
    for _ in range(25):
        seq = "".join(rng.choice("ACGT") for _ in range(rng.randrange(0, 21)))
        assert bpe(seq, merges) == brute_rank_order(seq, merges), (seq, merges)


@pytest.mark.parametrize("seed", range(10))
def test_termination_invariant_and_decode_round_trip(seed):
    rng = random.Random(1000 + seed)
    merges = random_table(rng, 40)
    rules = set(merges)
    sp = spellings(merges)
    for _ in range(10):
        seq = "".join(rng.choice("ACGT" * 8 + "N") for _ in range(rng.randrange(0, 300)))
        ids = bpe(seq, merges)
        # (ii) no adjacent output pair inside a segment has a rule; N (id 2) separates segments
        for a, b in zip(ids, ids[1:]):
            if a != 2 and b != 2:
                assert (a - 3, b - 3) not in rules
        # (iii) concatenated spellings give back the input
        assert "".join("N" if t == 2 else sp[t - 3] for t in ids) == seq


def test_n_runs_and_unk_boundaries():
    # Q13: a run of N gives one token each; UNK bytes likewise with id 1
    assert bpe("NNNN", [(0, 1)]) == [2, 2, 2, 2]
    assert bpe("ACNNRAC", [(0, 1)]) == [7, 2, 2, 1, 7]
    assert bpe("", [(0, 1)]) == []


def test_invalid_tables_rejected():
    # Q12: parts must be earlier tokens; pairs must be unique
    with pytest.raises(ValueError):
        bpe("ACGT", [(0, 4)])
    with pytest.raises(ValueError):
        bpe("ACGT", [(0, 1), (0, 1)])


def test_against_hf_tokenizers_bpe_optional():
    """(v) optional, non-gating: the same vocabulary and rules in the Hugging Face `tokenizers` BPE model."""
    tokenizers = pytest.importorskip("tokenizers")
    rng = random.Random(99)
    merges = random_table(rng, 30)
    sp = spellings(merges)
    if len(set(sp)) != len(sp):          # two rules may spell the same string (Q12); HF vocab needs unique strings
        pytest.skip("table spells a string twice")
    vocab = {s: i for i, s in enumerate(sp)}
    try:
        model = tokenizers.models.BPE(vocab=vocab, merges=[(sp[l], sp[r]) for l, r in merges])
    except Exception as e:                # pragma: no cover
        pytest.skip(f"tokenizers BPE construction failed: {e}")
    tok = tokenizers.Tokenizer(model)
    for _ in range(30):
        seq = "".join(rng.choice("ACGT") for _ in range(rng.randrange(1, 60)))
        assert [3 + i for i in tok.encode(seq).ids] == bpe(seq, merges), seq
