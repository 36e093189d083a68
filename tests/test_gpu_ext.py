"""GPU parity of the SURVEY.md 8(f) operations against the oracle (oracle/dnatok_oracle_ext.c), through the C-ABI:
reverse complement, decode, embedding gather with the micro-batch rule, int32 -> int64 widening.  Bit-exact."""
import random

import numpy as np
import pytest
import torch

import dnagen
import oracle
import paper_2601_05531_b200 as dn

pytestmark = pytest.mark.gpu


def cuda(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


# ------------------------------------------------------------------------------------------- reverse complement
@pytest.mark.parametrize("seed", range(4))
def test_revcomp_fuzz(seed):
    rng = random.Random(seed)
    alphabet = b"ACGTNacgtnRYKMBVDHSWU-*\n>x\x00\xff"
    recs = [bytes(rng.choice(alphabet) for _ in range(rng.choice([0, 1, 2, 15, 16, 17, rng.randrange(0, 5000)]))) for _ in range(60)]
    pre, post = bytes(rng.choice(alphabet) for _ in range(7)), bytes(rng.choice(alphabet) for _ in range(21))
    data = np.frombuffer(pre + b"".join(recs) + post, dtype=np.uint8)
    offs = (np.cumsum([0] + [len(r) for r in recs]) + len(pre)).astype(np.int64)
    tok = dn.DNATok(mode="kmer", k=6)
    for shift in (0, 1, 5):                                       # output pointers of every alignment
        buf = torch.empty(data.size + shift, dtype=torch.uint8, device="cuda")
        out = tok.revcomp(cuda(data), cuda(offs), out=buf[shift:])
        tok.check()
        assert np.array_equal(out.cpu().numpy(), oracle.revcomp(data, offs))


def test_revcomp_config3_slice_and_no_records():
    w = dnagen.config2(n_records=40)
    tok = dn.DNATok(mode="kmer", k=6)
    out = tok.revcomp(cuda(w.data), cuda(w.offsets))
    tok.check()
    assert np.array_equal(out.cpu().numpy(), oracle.revcomp(w.data, w.offsets))
    d = cuda(np.frombuffer(b"ACGT", dtype=np.uint8))
    assert tok.revcomp(d, cuda(np.array([0], dtype=np.int64))).cpu().numpy().tobytes() == b"ACGT"


def test_revcomp_then_encode_equals_oracle_of_the_reversed_records():
    w = dnagen.config2(n_records=8)
    tok = dn.DNATok(mode="kmer", k=6)
    d, o = cuda(w.data), cuda(w.offsets)
    ids, out = tok.encode(tok.revcomp(d, o), o)
    tok.check()
    want_ids, want_off = oracle.encode(oracle.revcomp(w.data, w.offsets), w.offsets, oracle.Config(mode=oracle.KMER, k=6))
    out = out.cpu().numpy()
    assert np.array_equal(out, want_off) and np.array_equal(ids[: out[-1]].cpu().numpy(), want_ids)


# ------------------------------------------------------------------------------------------- decode
def decode_case(data, offs, ocfg, **kw):
    data = np.frombuffer(data, dtype=np.uint8) if isinstance(data, (bytes, bytearray)) else data
    offs = np.asarray(offs, dtype=np.int64)
    tok = dn.DNATok(**kw)
    ids, out = tok.encode(cuda(data), cuda(offs))
    want_ids, want_off = oracle.encode(data, offs, ocfg)
    want_b, want_bo = oracle.decode(want_ids, want_off, ocfg)
    got_b, got_bo = tok.decode(ids, out, bytes_capacity=max(int(want_bo[-1]), 1))
    tok.check()
    assert np.array_equal(got_bo.cpu().numpy(), want_bo)
    assert np.array_equal(got_b[: int(want_bo[-1])].cpu().numpy(), want_b)
    return tok, ids, out, want_bo


@pytest.mark.parametrize("k,dt", [(1, 4), (3, 2), (6, 2), (6, 4), (8, 4)])
def test_decode_kmer_fasta_with_n(k, dt):
    w = dnagen.config3(total_bases=150_000, lo=10, hi=9000, seed=k)
    data = w.data.copy()
    rng = np.random.default_rng(k)
    pos = rng.integers(0, data.size, size=500)
    data[pos[data[pos] != 10]] = ord("N")
    decode_case(data, w.offsets, oracle.Config(mode=oracle.KMER, k=k), mode="kmer", k=k, id_dtype=dt)


def test_decode_single_nt_config1_and_custom_vocabulary():
    w = dnagen.config1()
    decode_case(w.data, w.offsets, oracle.Config(mode=oracle.SINGLE_NT), mode="single_nt")
    # the paper's fallback vocabulary (PAPER.md:88 l.10): A..T -> 1..4, N -> 0, pad id -1 so that N is not skipped
    ocfg = oracle.Config(mode=oracle.SINGLE_NT, nt_ids=(1, 2, 3, 4, 0), unk_id=0, pad_id=-1)
    decode_case(b"ACGTNacgtn-x\nACG", [0, 13, 16], ocfg, mode="single_nt", nt_ids=(1, 2, 3, 4, 0), unk_id=0, pad_id=-1)


def test_decode_bpe_config4_and_round_trip():
    w = dnagen.config4(n_reads=300, n_merges=4092)
    decode_case(w.data, w.offsets, oracle.Config(mode=oracle.BPE, merges=w.merges), mode="bpe", merges=w.merges, max_record_bytes=2048)
    # N-free reads: decode(encode(x)) == x
    clean = np.frombuffer(bytes(w.data).replace(b"N", b"A"), dtype=np.uint8)
    tok, ids, out, bo = decode_case(clean, w.offsets, oracle.Config(mode=oracle.BPE, merges=w.merges), mode="bpe", merges=w.merges,
                                    max_record_bytes=2048)
    got, _ = tok.decode(ids, out, bytes_capacity=clean.size)
    tok.check()
    assert np.array_equal(got.cpu().numpy(), clean) and np.array_equal(bo, w.offsets)


def test_decode_padded_rows_skip_pad_and_capacity_overflow_is_reported():
    w = dnagen.config3(total_bases=40_000, lo=10, hi=3000)
    tok = dn.DNATok(mode="kmer", k=6, seq_len=300)
    d, o = cuda(w.data), cuda(w.offsets)
    ids, out = tok.encode(d, o)
    batch, mask = tok.pad(ids, out)
    n = batch.shape[0]
    row_off = torch.arange(0, (n + 1) * 300, 300, dtype=torch.int64, device="cuda")
    got_b, got_bo = tok.decode(batch.reshape(-1), row_off, bytes_capacity=n * 300 * 6)
    tok.check()
    ocfg = oracle.Config(mode=oracle.KMER, k=6, seq_len=300)
    want_ids, want_off = oracle.encode(w.data, w.offsets, ocfg)
    wb, _ = oracle.pad(want_ids, want_off, ocfg)
    want_b, want_bo = oracle.decode(wb.reshape(-1), np.arange(0, (n + 1) * 300, 300), ocfg)
    assert np.array_equal(got_bo.cpu().numpy(), want_bo) and np.array_equal(got_b[: int(want_bo[-1])].cpu().numpy(), want_b)
    tok.decode(batch.reshape(-1), row_off, bytes_capacity=100)
    with pytest.raises(dn.DNATokError) as e:
        tok.check()
    assert e.value.code == dn.ECAPACITY


# ------------------------------------------------------------------------------------------- embedding gather
def test_microbatch_rows_matches_the_oracle():
    for args in [(4096, 1 << 20, 512), (8192, 1 << 20, 512), (2048, 1 << 20, 2048), (64, 1 << 20, 512), (4096, 1 << 20, 8192),
                 (4096, 1 << 20, 3_000_000), (4096, 1 << 20, 1000), (1, 1, 1)]:
        assert dn.dnatok_microbatch_rows(*args) == oracle.microbatch_rows(*args)


@pytest.mark.parametrize("dtype,D", [(torch.bfloat16, 128), (torch.float32, 128), (torch.float16, 6), (torch.float32, 3)])
def test_embed_gather_and_microbatch_launches(dtype, D):
    torch.manual_seed(0)
    V, B, T = 11, 37, 512
    table = torch.randn(V, D, device="cuda").to(dtype)
    ids = torch.randint(0, V, (B, T), dtype=torch.int32, device="cuda")
    ids[3, 7] = -1
    ids[5, 0] = V
    tok = dn.DNATok(mode="single_nt")
    calls = []
    out = tok.embed(ids, table, b_emb=16, m_tokens=4096, on_microbatch=lambda r0, n: calls.append((r0, n)))
    tok.check()
    b = oracle.microbatch_rows(16, 4096, T)                       # min(16, 4096 / 512) = 8 rows per call
    assert b == 8 and calls == [(r, min(8, B - r)) for r in range(0, B, 8)]
    raw = table.view(torch.int16 if table.element_size() == 2 else torch.int32).cpu().numpy()
    want = oracle.embed(ids.cpu().numpy(), raw)
    got = out.view(torch.int16 if table.element_size() == 2 else torch.int32).cpu().numpy()
    assert np.array_equal(got, want)


def test_embed_after_encode_and_pad_paper_shape():
    # vocabulary of 11, D = 128; ids straight from encode + pad
    w = dnagen.config1()
    tok = dn.DNATok(mode="single_nt", seq_len=2048)
    ids, out = tok.encode(cuda(w.data), cuda(w.offsets))
    batch, mask = tok.pad(ids, out)
    table = torch.randn(11, 128, device="cuda").to(torch.bfloat16)
    emb = tok.embed(batch, table)
    tok.check()
    ocfg = oracle.Config(mode=oracle.SINGLE_NT, seq_len=2048)
    wi, wo = oracle.encode(w.data, w.offsets, ocfg)
    wb, _ = oracle.pad(wi, wo, ocfg)
    want = oracle.embed(wb, table.view(torch.int16).cpu().numpy())
    assert np.array_equal(emb.view(torch.int16).cpu().numpy(), want)


# ------------------------------------------------------------------------------------------- widening
@pytest.mark.parametrize("n,shift", [(0, 0), (1, 0), (5, 0), (4096, 0), (100_003, 0), (100_003, 1)])
def test_widen(n, shift):
    rng = np.random.default_rng(n)
    a = rng.integers(-2 ** 31, 2 ** 31 - 1, size=n + shift).astype(np.int32)
    tok = dn.DNATok(mode="single_nt")
    got = tok.widen(cuda(a)[shift:])
    tok.check()
    assert np.array_equal(got.cpu().numpy(), oracle.widen(a[shift:]))


# ------------------------------------------------------------------------------------------- table-driven k-mer ids (f1)
def dense_lut():
    lut = np.full(256, 5, dtype=np.uint8)
    for i, (u, l) in enumerate(zip(b"ACGTN", b"acgtn")):
        lut[u] = lut[l] = i
    return lut


@pytest.mark.parametrize("k,dt", [(1, 4), (2, 2), (3, 4), (6, 2), (6, 4), (8, 4)])
@pytest.mark.parametrize("layout", ["fasta", "dense"])
def test_kmer_table_ids(k, dt, layout):
    """PAPER.md:88 Alg. 1 l.18-22: ids through kmer_lut[5^k]; windows holding N / other bytes take digit 4; both encoders"""
    rng = np.random.default_rng(10 * k + dt)
    lut5 = rng.integers(0, 30000, size=5 ** k).astype(np.int32)
    nt = (30001, 30002, 30003, 30004, 30005)
    if layout == "fasta":
        w = dnagen.config3(total_bases=120_000, lo=10, hi=9000, seed=k)
        data = w.data.copy()
        pos = rng.integers(0, data.size, size=600)
        data[pos[data[pos] != 10]] = rng.choice(np.frombuffer(b"NNNnRY-", dtype=np.uint8), size=int((data[pos] != 10).sum()))
        kw, okw = {}, {}
    else:
        w = dnagen.config2(n_records=3)
        data = w.data.copy()
        data[rng.integers(0, data.size, size=300)] = ord("x")
        kw = dict(class_lut=dense_lut(), strip_headers=False)
        okw = dict(class_lut=dense_lut(), strip_headers=False)
    ocfg = oracle.Config(mode=oracle.KMER, k=k, nt_ids=nt, **okw)
    want_ids, want_off = oracle.encode_kmer_table(data, w.offsets, ocfg, lut5)
    for S in (0, 1):
        dn.SUPER_TILE = S
        try:
            tok = dn.DNATok(mode="kmer", k=k, id_dtype=dt, nt_ids=nt, kmer_lut=lut5, **kw)
        finally:
            dn.SUPER_TILE = 0
        ids, out = tok.encode(cuda(data), cuda(w.offsets))
        tok.check()
        out = out.cpu().numpy()
        assert np.array_equal(out, want_off)
        assert np.array_equal(ids[: out[-1]].cpu().numpy().astype(np.int32), want_ids)


def test_kmer_table_closed_form_table_reproduces_the_default_ids_and_bad_tables_are_rejected():
    k = 4
    lut5 = np.empty(5 ** k, dtype=np.int32)
    for code in range(5 ** k):
        d = [(code // 5 ** (k - 1 - i)) % 5 for i in range(k)]
        lut5[code] = 1 if 4 in d else 3 + sum(x * 4 ** (k - 1 - i) for i, x in enumerate(d))
    w = dnagen.config1()
    d, o = cuda(w.data), cuda(w.offsets)
    a = dn.DNATok(mode="kmer", k=k)
    b = dn.DNATok(mode="kmer", k=k, kmer_lut=lut5, nt_ids=tuple(3 + 4 ** k + c for c in range(5)))
    ia, oa = a.encode(d, o)
    ib, ob = b.encode(d, o)
    a.check(); b.check()
    n = int(oa[-1])
    assert torch.equal(oa, ob) and torch.equal(ia[:n], ib[:n])
    for bad in (dict(mode="kmer", k=4, kmer_lut=lut5[:-1]), dict(mode="kmer", k=9, kmer_lut=np.zeros(5 ** 9, np.int32)),
                dict(mode="single_nt", kmer_lut=lut5), dict(mode="kmer", k=4, id_dtype=dn.I16, kmer_lut=lut5 + 40000)):
        with pytest.raises(dn.DNATokError) as e:
            dn.DNATok(**bad)
        assert e.value.code == dn.EINVAL
    with pytest.raises(dn.DNATokError):
        b.decode(ib, ob, bytes_capacity=10)
