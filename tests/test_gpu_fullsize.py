"""GPU parity at the full BASELINE.json sizes, in the launch configuration bench.py times: EVERY id and EVERY
out_offsets entry against the CPU oracle (PAPER.md:183 section 2.3 "equivalence checks", :305 section 4.4), plus the
paths only a full-size run or a capped grid reaches deterministically: one persistent CTA walking many super-tiles /
reads (dnatok_set_grid_cap), tickets far beyond the grid, stream-buffer reuse, and a 200x stress of the chained scan.
Config 5 is checked STREAMED: every batch of the 64 MiB x 4-stream run is copied back and compared with oracle rows
computed on the fly (SURVEY.md 8(d) protocol)."""
import numpy as np
import pytest

import dnagen
import oracle
from oracle_mt import encode_mt

torch = pytest.importorskip("torch")
pytestmark = [pytest.mark.gpu]

if torch.cuda.is_available():
    import paper_2601_05531_b200 as dn

MIB = 1 << 20


def dense_lut():
    """default table with no SKIP class: '\\n' and '\\r' are ordinary UNK bytes (the no-scan fast path's spec)"""
    lut = oracle.default_lut()
    lut[10] = lut[13] = oracle.CLS_UNK
    return lut


def gpu_full(w, **kw):
    tok = dn.DNATok(**kw)
    d, o = torch.from_numpy(w.data).cuda(), torch.from_numpy(w.offsets).cuda()
    ids, out = tok.encode(d, o)
    tok.check()
    out = out.cpu().numpy()
    return ids[: out[-1]].cpu().numpy(), out, tok


def assert_same(got_ids, got_off, want_ids, want_off):
    bad = np.flatnonzero(got_off != want_off)
    assert bad.size == 0, ("out_offsets", bad[:5], got_off[bad[:5]], want_off[bad[:5]])
    assert got_ids.shape == want_ids.shape
    neq = got_ids != want_ids
    assert not neq.any(), ("ids", np.flatnonzero(neq)[:8])


def test_config2_full_every_id_and_offset():
    w = dnagen.config2()                                     # 4,096 x 65,536 bases = 256 MiB
    for kw, okw in ((dict(), dict()),
                    (dict(class_lut=dense_lut(), strip_headers=False), dict(class_lut=dense_lut(), strip_headers=False))):
        want_ids, want_off = encode_mt(w.data, w.offsets, oracle.Config(mode=oracle.KMER, k=6, **okw))
        got_ids, got_off, _ = gpu_full(w, mode="kmer", k=6, **kw)
        assert_same(got_ids, got_off, want_ids, want_off)


@pytest.mark.parametrize("k", [1, 6, 8])
def test_config3_quarter_gib_every_id_and_offset(k):
    w = dnagen.config3(total_bases=256 * MIB)                # FASTA layout, log-uniform record lengths
    want_ids, want_off = encode_mt(w.data, w.offsets, oracle.Config(mode=oracle.KMER, k=k))
    got_ids, got_off, _ = gpu_full(w, mode="kmer", k=k, id_dtype=2 if k <= 6 else 4)
    assert_same(got_ids, got_off, want_ids, want_off)


def test_config1_times_64_single_nt():
    w = dnagen.config1(n_records=16 * 64)                    # the streaming-rate variant of config 1 (64 copies' worth)
    want_ids, want_off = encode_mt(w.data, w.offsets, oracle.Config(mode=oracle.SINGLE_NT))
    got_ids, got_off, _ = gpu_full(w, mode="single_nt")
    assert_same(got_ids, got_off, want_ids, want_off)


def test_config4_full_every_id_and_offset():
    w = dnagen.config4()                                     # 65,536 reads, 4,092 merges
    want_ids, want_off = encode_mt(w.data, w.offsets, oracle.Config(mode=oracle.BPE, merges=w.merges))
    got_ids, got_off, _ = gpu_full(w, mode="bpe", merges=w.merges, max_record_bytes=1536)
    assert_same(got_ids, got_off, want_ids, want_off)


def test_config5_streamed_one_gib_every_batch_against_oracle_rows():
    """1 GiB of config 5 through dnatok_stream_encode with 64 MiB chunks x 4 streams: each delivered batch (CSR counts,
    batch_ids, mask) is copied back inside the callback and compared with oracle rows of exactly those records."""
    total = 1 << 30
    pinned = torch.empty(total, dtype=torch.uint8).pin_memory()
    w = dnagen.config5(total_bytes=total, out=pinned.numpy())
    L = 8192
    tok = dn.DNATok(mode="kmer", k=6, seq_len=L, max_record_bytes=65536)
    cfg = oracle.Config(mode=oracle.KMER, k=6, seq_len=L)
    seen = [0]
    cuts = []

    def on_batch(b):
        s = torch.cuda.ExternalStream(b.stream)
        with torch.cuda.stream(s):
            off = b.out_offsets().cpu().numpy()
            rows = b.batch_ids().cpu().numpy() if b.n_records else np.zeros((0, L), np.int32)
            msk = b.mask().cpu().numpy() if b.n_records else np.zeros((0, L), np.uint8)
        assert b.first_record == seen[0]
        r0, r1 = b.first_record, b.first_record + b.n_records
        lo, hi = int(w.offsets[r0]), int(w.offsets[r1])
        want_ids, want_off = encode_mt(w.data[lo:hi], w.offsets[r0:r1 + 1] - lo, cfg)
        assert np.array_equal(off, want_off), b.chunk_index
        wb, wm = oracle.pad(want_ids, want_off, cfg)
        assert np.array_equal(rows, wb), b.chunk_index
        assert np.array_equal(msk, wm), b.chunk_index
        seen[0] = r1
        cuts.append(b.n_records)

    tok.stream_encode(pinned, w.offsets, 64 * MIB, 4, max_rows_per_chunk=2100, on_batch=on_batch)
    assert seen[0] == w.n_records and len(cuts) == total // (64 * MIB)
    assert min(cuts[:-1]) >= 2047                            # every interior boundary cut a record (Q18)


# ---------------------------------------------------------------------------------- capped grids
@pytest.fixture(params=[1, 2, 7], ids=lambda c: f"cap{c}")
def grid_cap(request):
    old = dn.GRID_CAP
    dn.GRID_CAP = request.param
    yield request.param
    dn.GRID_CAP = old


@pytest.fixture(params=[0, 1], ids=lambda s: f"S{s}")
def small_super_tile(request):
    old = dn.SUPER_TILE
    dn.SUPER_TILE = request.param
    yield request.param
    dn.SUPER_TILE = old


def small_check(w, okw=None, **kw):
    m = {"single_nt": oracle.SINGLE_NT, "kmer": oracle.KMER, "bpe": oracle.BPE}[kw["mode"]]
    cfg = oracle.Config(mode=m, k=kw.get("k", 1), merges=kw.get("merges"), **(okw or {}))
    want_ids, want_off = oracle.encode(w.data, w.offsets, cfg)
    got_ids, got_off, _ = gpu_full(w, **kw)
    assert_same(got_ids.astype(np.int32), got_off, want_ids, want_off)


def test_capped_grid_walks_many_super_tiles_fasta(grid_cap, small_super_tile):
    """3 MiB of FASTA on 1 / 2 / 7 persistent CTAs: each CTA walks >= 6 super-tiles, both stream buffers are reused
    many times, tickets run far beyond the grid"""
    w = dnagen.config3(total_bases=3 * MIB)
    for k, dt in ((6, 2), (1, 2), (8, 4)):
        small_check(w, mode="kmer", k=k, id_dtype=dt)
    small_check(w, mode="single_nt")


def test_capped_grid_single_line_records_and_dense_spec(grid_cap, small_super_tile):
    w = dnagen.config2(n_records=40, bases=65536, n_frac=0.01)
    small_check(w, mode="kmer", k=6)
    small_check(w, okw=dict(class_lut=dense_lut(), strip_headers=False), mode="kmer", k=6,
                class_lut=dense_lut(), strip_headers=False)
    small_check(w, okw=dict(class_lut=dense_lut(), strip_headers=False), mode="kmer", k=5, id_dtype=2,
                class_lut=dense_lut(), strip_headers=False)


def test_capped_grid_bpe_many_reads_per_cta(grid_cap):
    """400 reads on 1 / 2 / 7 CTAs: every CTA takes many reads in turn (workspace reuse between reads)"""
    w = dnagen.config4(n_reads=400, n_merges=1000, corpus_bases=65536)
    small_check(w, mode="bpe", merges=w.merges, max_record_bytes=1536)


def test_capped_grid_pad(grid_cap):
    w = dnagen.config3(total_bases=300_000, lo=1000, hi=9000)
    tok = dn.DNATok(mode="kmer", k=6, seq_len=700)
    d, o = torch.from_numpy(w.data).cuda(), torch.from_numpy(w.offsets).cuda()
    batch, mask, _ = tok.encode_padded(d, o)
    tok.check()
    cfg = oracle.Config(mode=oracle.KMER, k=6, seq_len=700)
    want_ids, want_off = oracle.encode(w.data, w.offsets, cfg)
    wb, wm = oracle.pad(want_ids, want_off, cfg)
    assert np.array_equal(batch.cpu().numpy(), wb) and np.array_equal(mask.cpu().numpy(), wm)


# ---------------------------------------------------------------------------------- stress of the chained scan
def test_stress_200_full_config3_encodes_bit_exact_each_time():
    """200 back-to-back encodes of the full 1 GiB config 3 input on one handle (generation tags advance, scratch is
    never cleared): the first result is checked against the oracle in full, every later one against the first on the
    device; dnatok_check must never report ESTATE / ECAPACITY."""
    w = dnagen.config3()
    want_ids, want_off = encode_mt(w.data, w.offsets, oracle.Config(mode=oracle.KMER, k=6))
    tok = dn.DNATok(mode="kmer", k=6, id_dtype=2)
    d, o = torch.from_numpy(w.data).cuda(), torch.from_numpy(w.offsets).cuda()
    n_tok = int(want_off[-1])
    ids0 = torch.empty(n_tok + 64, dtype=torch.int16, device="cuda")
    off0 = torch.empty(w.n_records + 1, dtype=torch.int64, device="cuda")
    tok.encode(d, o, ids_out=ids0, out_offsets=off0)
    tok.check()
    assert np.array_equal(off0.cpu().numpy(), want_off)
    assert np.array_equal(ids0[:n_tok].cpu().numpy(), want_ids.astype(np.int16))
    del want_ids
    ids = torch.empty_like(ids0)
    off = torch.empty_like(off0)
    for it in range(199):
        ids.fill_(-1)
        tok.encode(d, o, ids_out=ids, out_offsets=off)
        tok.check()
        assert torch.equal(off, off0), it
        assert torch.equal(ids[:n_tok], ids0[:n_tok]), it
