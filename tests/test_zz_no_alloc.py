"""dnatok_decode_static: the decode entry point that allocates no device memory (its scratch is a static device array inside
the library, see include/dnatok.h).  Checked bit for bit against the existing dnatok_decode on the same inputs, on two calls
in a row that share the static array (the second smaller, so that it runs over the first call's left-over contents), and against
the oracle; sizes beyond the stated maximum are rejected before anything is launched.  Collected last on purpose (file name)."""
import numpy as np
import pytest

import dnagen
import oracle

torch = pytest.importorskip("torch")
pytestmark = [pytest.mark.gpu]

if torch.cuda.is_available():
    import paper_2601_05531_b200 as dn


def encode_on_gpu(tok, w_data, w_offsets):
    d = torch.from_numpy(np.ascontiguousarray(w_data)).cuda()
    o = torch.from_numpy(np.ascontiguousarray(w_offsets, dtype=np.int64)).cuda()
    ids, out = tok.encode(d, o)
    tok.check()
    return ids, out


def both_paths(tok, ids, out, cap):
    """(bytes, byte_offsets) from dnatok_decode and from dnatok_decode_static, as numpy"""
    n_rec = out.numel() - 1
    ref_b, ref_bo = tok.decode(ids, out, bytes_capacity=cap)
    tok.check()
    got_b = torch.full((max(cap, 1),), 0x7A, dtype=torch.uint8, device="cuda")
    got_bo = torch.full((n_rec + 1,), -1, dtype=torch.int64, device="cuda")
    free0 = torch.cuda.mem_get_info()[0]
    tok.decode_static(ids, out, got_b, got_bo)
    tok.check()
    assert torch.cuda.mem_get_info()[0] >= free0, "device memory was taken during a call that must not allocate"
    ref_bo, got_bo = ref_bo.cpu().numpy(), got_bo.cpu().numpy()
    n = int(ref_bo[-1])
    return ref_b[:n].cpu().numpy(), ref_bo, got_b[:n].cpu().numpy(), got_bo


@pytest.mark.parametrize("kw", [dict(mode="kmer", k=6), dict(mode="kmer", k=6, id_dtype=2), dict(mode="single_nt")],
                         ids=["kmer6-int32", "kmer6-int16", "single-nt"])
def test_two_calls_in_a_row_equal_the_allocating_path_and_the_oracle(kw):
    tok = dn.DNATok(**kw)
    okw = dict(kw)
    okw["mode"] = {"single_nt": oracle.SINGLE_NT, "kmer": oracle.KMER}[okw["mode"]]
    okw.pop("id_dtype", None)
    ocfg = oracle.Config(**okw)
    # first call: ~2,000 records; second call: ~60 records of other lengths over the same static scratch
    for total, lo, hi, seed in ((600_000, 10, 900, 1), (150_000, 200, 9000, 2)):
        w = dnagen.config3(total_bases=total, lo=lo, hi=hi, seed=seed)
        data = w.data.copy()
        rng = np.random.default_rng(seed)
        pos = rng.integers(0, data.size, size=400)
        data[pos[data[pos] != 10]] = ord("N")
        ids, out = encode_on_gpu(tok, data, w.offsets)
        ref_b, ref_bo, got_b, got_bo = both_paths(tok, ids, out, cap=data.size)
        assert np.array_equal(got_bo, ref_bo)
        assert np.array_equal(got_b, ref_b)
        want_ids, want_off = oracle.encode(data, w.offsets, ocfg)
        want_b, want_bo = oracle.decode(want_ids, want_off, ocfg)
        assert np.array_equal(got_bo, want_bo) and np.array_equal(got_b, want_b)


def test_bpe_and_an_empty_call():
    w = dnagen.config4(n_reads=300, n_merges=500, corpus_bases=16384)
    tok = dn.DNATok(mode="bpe", merges=w.merges, max_record_bytes=2048)
    ids, out = encode_on_gpu(tok, w.data, w.offsets)
    for _ in range(2):
        ref_b, ref_bo, got_b, got_bo = both_paths(tok, ids, out, cap=w.data.size)
        assert np.array_equal(got_bo, ref_bo) and np.array_equal(got_b, ref_b)
    zero = torch.zeros(1, dtype=torch.int64, device="cuda")
    bo = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    tok.decode_static(ids, zero, torch.empty(16, dtype=torch.uint8, device="cuda"), bo)
    tok.check()
    assert bo.cpu().tolist() == [0]


def test_more_records_than_the_static_scratch_holds_are_rejected():
    tok = dn.DNATok(mode="kmer", k=6)
    n = dn.DECODE_STATIC_MAX_RECORDS + 1
    out = torch.zeros(n + 1, dtype=torch.int64, device="cuda")             # n empty records
    ids = torch.zeros(1, dtype=torch.int32, device="cuda")
    buf = torch.empty(16, dtype=torch.uint8, device="cuda")
    bo = torch.full((n + 1,), -1, dtype=torch.int64, device="cuda")
    launches = tok.launch_count
    with pytest.raises(dn.DNATokError) as e:
        tok.decode_static(ids, out, buf, bo)
    assert e.value.code == dn.ECAPACITY and "static scratch" in str(e.value)
    assert tok.launch_count == launches and int(bo[0].item()) == -1        # nothing was launched
    # exactly the maximum is served
    tok.decode_static(ids, out[: n], buf, bo[: n])
    tok.check()
    assert int(bo[: n].abs().sum().item()) == 0
