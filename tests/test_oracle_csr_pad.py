"""Pins for oracle steps 5-6 (CSR offsets; pad + mask): structural invariants and the hand-worked rows
(PAPER.md:124-129 left padding, right-aligned)."""
import json
import os
import random

import numpy as np
import pytest

import dnagen
import oracle


def random_batch(rng, n_records):
    recs = []
    for _ in range(n_records):
        n = rng.choice([0, 0, 1, 5, 6, 7, rng.randrange(0, 200)])
        body = "".join(rng.choice("ACGTNacgt") for _ in range(n))
        if rng.random() < 0.5:
            body = ">h%d\n" % n + "\n".join(body[i:i + 17] for i in range(0, n, 17)) + "\n"
        recs.append(body.encode())
    data = b"".join(recs)
    offs = np.cumsum([0] + [len(r) for r in recs]).astype(np.int64)
    return recs, np.frombuffer(data, dtype=np.uint8), offs


@pytest.mark.parametrize("mode,k", [(oracle.SINGLE_NT, 1), (oracle.KMER, 3), (oracle.KMER, 6), (oracle.BPE, 0)])
def test_csr_offsets_and_concatenation(mode, k):
    rng = random.Random(11 + k)
    merges = dnagen.merge_table(seed=3, n_merges=50, corpus_bases=4096) if mode == oracle.BPE else None
    cfg = oracle.Config(mode=mode, k=max(k, 1), merges=merges)
    recs, data, offs = random_batch(rng, 40)
    ids, out = oracle.encode(data, offs, cfg)
    assert out[0] == 0 and np.all(np.diff(out) >= 0) and out[-1] == ids.size
    alone = [oracle.encode_one(r, cfg) for r in recs]
    assert np.array_equal(np.concatenate(alone), ids)
    assert [a.size for a in alone] == np.diff(out).tolist()


def test_offsets_need_not_start_at_zero_or_cover_the_buffer():
    data = np.frombuffer(b"TTTTACGTACGGGGG", dtype=np.uint8)
    ids, out = oracle.encode(data, np.array([4, 8, 10], dtype=np.int64), oracle.Config(mode=oracle.SINGLE_NT))
    assert ids.tolist() == [2, 3, 4, 5, 2, 3] and out.tolist() == [0, 4, 6]


@pytest.mark.parametrize("side", [oracle.PAD_LEFT, oracle.PAD_RIGHT])
@pytest.mark.parametrize("seq_len", [1, 5, 8, 64])
def test_pad_mask_properties(side, seq_len):
    rng = random.Random(seq_len)
    cfg = oracle.Config(mode=oracle.KMER, k=3, seq_len=seq_len, pad_side=side)
    _, data, offs = random_batch(rng, 30)
    ids, out = oracle.encode(data, offs, cfg)
    batch, mask = oracle.pad(ids, out, cfg)
    tok = np.diff(out)
    m = np.minimum(tok, seq_len)
    assert mask.sum(axis=1).tolist() == m.tolist()
    assert np.all(batch[mask == 0] == cfg.pad_id)
    for r in range(tok.size):
        kept = batch[r][mask[r] == 1]
        assert kept.tolist() == ids[out[r]:out[r] + m[r]].tolist()      # Q15: first seq_len tokens
        cols = np.flatnonzero(mask[r])
        if m[r]:
            want0 = seq_len - m[r] if side == oracle.PAD_LEFT else 0   # PAPER.md:127 right-aligned
            assert cols[0] == want0 and cols[-1] == want0 + m[r] - 1


def test_left_and_right_are_mirror_placements():
    rng = random.Random(2)
    _, data, offs = random_batch(rng, 20)
    cl = oracle.Config(mode=oracle.KMER, k=2, seq_len=16, pad_side=oracle.PAD_LEFT)
    cr = oracle.Config(mode=oracle.KMER, k=2, seq_len=16, pad_side=oracle.PAD_RIGHT)
    ids, out = oracle.encode(data, offs, cl)
    bl, ml = oracle.pad(ids, out, cl)
    br, mr = oracle.pad(ids, out, cr)
    for r in range(bl.shape[0]):
        m = int(ml[r].sum())
        assert np.array_equal(bl[r, 16 - m:], br[r, :m]) and np.array_equal(ml[r][::-1], mr[r])


def test_handworked_pad_rows(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "handworked_example.json")))
    data = (g["record0"] + g["record1"]).encode()
    for side, key in ((oracle.PAD_LEFT, "kmer3_pad5_left"), (oracle.PAD_RIGHT, "kmer3_pad5_right")):
        cfg = oracle.Config(mode=oracle.KMER, k=3, seq_len=5, pad_side=side)
        ids, out = oracle.encode(data, g["rec_offsets"], cfg)
        batch, mask = oracle.pad(ids, out, cfg)
        assert batch.tolist() == g[key]["ids"] and mask.tolist() == g[key]["mask"]
