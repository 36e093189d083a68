"""GPU parity of the pinned multi-stream scheduler (step 7): the streamed result must equal the whole-buffer
result for every chunk size and stream count (SURVEY.md 8(c) 'Streaming' pin; "keep tokenizer
logic unchanged").  Chunk boundaries fall inside header lines, on '\\n' and between the bases of one k-mer."""
import numpy as np
import pytest

import dnagen
import oracle

torch = pytest.importorskip("torch")
pytestmark = [pytest.mark.gpu, pytest.mark.usefixtures("super_tile")]

if torch.cuda.is_available():
    import paper_2601_05531_b200 as dn


def run_stream(w, chunk_bytes, n_streams, source="pinned", **kw):
    tok = dn.DNATok(**kw)
    pinned = torch.from_numpy(w.data.copy()).pin_memory() if source == "pinned" else w.data.copy()   # pageable numpy array
    got_ids, got_cnt, got_batch, got_mask, firsts = [], [], [], [], []
    keep = []

    def on_batch(b: dn.Batch):
        s = torch.cuda.ExternalStream(b.stream)
        with torch.cuda.stream(s):
            off = b.out_offsets().cpu()                    # sync copy on that stream: fine for a test
            n_tok = int(off[-1])
            got_cnt.append(np.diff(off.numpy()))
            got_ids.append(b.ids(n_tok).cpu().numpy().astype(np.int32) if n_tok else np.zeros(0, np.int32))
            if tok.cfg.seq_len:
                got_batch.append(b.batch_ids().cpu().numpy())
                got_mask.append(b.mask().cpu().numpy())
            firsts.append((b.first_record, b.n_records))

    if source == "file":
        import tempfile
        with tempfile.NamedTemporaryFile() as f:
            f.write(w.data.tobytes()); f.flush()
            with open(f.name, "rb", buffering=0) as rd:
                def fill(i, off, dst):
                    rd.seek(off)
                    assert rd.readinto(dst) == dst.size
                tok.stream_encode_from(fill, w.data.size, w.offsets, chunk_bytes, n_streams, max_rows_per_chunk=w.n_records + 1,
                                       on_batch=on_batch)
    else:
        tok.stream_encode(pinned, w.offsets, chunk_bytes, n_streams, max_rows_per_chunk=w.n_records + 1, on_batch=on_batch)
    # batches arrive in record order and cover every record exactly once
    pos = 0
    for f, n in firsts:
        assert f == pos
        pos += n
    assert pos == w.n_records
    ids = np.concatenate(got_ids) if got_ids else np.zeros(0, np.int32)
    cnt = np.concatenate(got_cnt) if got_cnt else np.zeros(0, np.int64)
    batch = np.concatenate(got_batch) if got_batch else None
    mask = np.concatenate(got_mask) if got_mask else None
    return ids, cnt, batch, mask


def oracle_ref(w, **kw):
    m = {"single_nt": oracle.SINGLE_NT, "kmer": oracle.KMER, "bpe": oracle.BPE}
    cfg = oracle.Config(mode=m[kw["mode"]], k=kw.get("k", 1), seq_len=kw.get("seq_len", 0),
                        pad_side=kw.get("pad_side", 0), merges=kw.get("merges"))
    ids, off = oracle.encode(w.data, w.offsets, cfg)
    batch, mask = oracle.pad(ids, off, cfg) if cfg.seq_len else (None, None)
    return ids, np.diff(off), batch, mask


@pytest.mark.parametrize("chunk_bytes", [4099, 65536 + 7, 1 << 20])
@pytest.mark.parametrize("n_streams", [1, 2, 4])
def test_chunk_size_invariance_fasta(chunk_bytes, n_streams):
    w = dnagen.config3(total_bases=400_000, lo=1000, hi=20000)
    kw = dict(mode="kmer", k=6, seq_len=512, max_record_bytes=32768)
    want = oracle_ref(w, **kw)
    got = run_stream(w, chunk_bytes, n_streams, **kw)
    for g, x in zip(got, want):
        assert np.array_equal(g, x)


@pytest.mark.parametrize("chunk_bytes", [4099, 40000])
def test_config5_shape_records_cut_by_every_boundary(chunk_bytes):
    w = dnagen.config5(total_bytes=60 * 4097 + 8, bases=4096)
    kw = dict(mode="kmer", k=6, seq_len=1024, pad_side=1, max_record_bytes=8192)
    want = oracle_ref(w, **kw)
    got = run_stream(w, chunk_bytes, 4, **kw)
    for g, x in zip(got, want):
        assert np.array_equal(g, x)


def test_record_spanning_several_chunks_and_no_padding():
    w = dnagen.config3(total_bases=300_000, lo=50_000, hi=131072)
    kw = dict(mode="single_nt", max_record_bytes=200_000)
    want = oracle_ref(w, **kw)
    got = run_stream(w, 30_000, 2, **kw)
    assert np.array_equal(got[0], want[0]) and np.array_equal(got[1], want[1])


def test_stream_bpe():
    w = dnagen.config4(n_reads=400, n_merges=500, corpus_bases=16384)
    kw = dict(mode="bpe", merges=w.merges, max_record_bytes=2048)
    want = oracle_ref(w, **kw)
    got = run_stream(w, 50_000, 3, **kw)
    assert np.array_equal(got[0], want[0]) and np.array_equal(got[1], want[1])


def test_carry_capacity_error_and_device_pointer_rejected():
    w = dnagen.config3(total_bases=100_000, lo=50_000, hi=100_000)
    tok = dn.DNATok(mode="kmer", k=6, max_record_bytes=1024)
    with pytest.raises(dn.DNATokError) as e:
        tok.stream_encode(torch.from_numpy(w.data.copy()).pin_memory(), w.offsets, 8192, 2)
    assert e.value.code == dn.ECAPACITY
    with pytest.raises(dn.DNATokError) as e:                              # a device pointer is not host memory
        dn.dnatok_stream_encode(tok.h, torch.from_numpy(w.data.copy()).cuda().data_ptr(), w.data.size, w.offsets.ctypes.data,
                                w.n_records, 8192, 2, 0, dn._BATCH_FN(lambda *_: None))
    assert e.value.code == dn.EINVAL


@pytest.mark.parametrize("source", ["pageable", "file"])
@pytest.mark.parametrize("chunk_bytes,n_streams", [(4099, 1), (65536 + 7, 4), (1 << 20, 2)])
def test_pageable_and_file_input_go_through_the_pinned_staging_ring(source, chunk_bytes, n_streams):
    """a producer reading from a file or pageable memory fills a ring of n_streams + 1 pinned slots
    (PAPER.md:181 persistent pinned buffers); the result is the whole-buffer result"""
    w = dnagen.config3(total_bases=300_000, lo=1000, hi=20000)
    kw = dict(mode="kmer", k=6, seq_len=512, max_record_bytes=32768)
    want = oracle_ref(w, **kw)
    got = run_stream(w, chunk_bytes, n_streams, source=source, **kw)
    for g, x in zip(got, want):
        assert np.array_equal(g, x)


def test_failed_stream_call_leaves_nothing_in_flight_and_the_handle_usable():
    """a capacity failure in the middle of the chunk loop (a record longer than the carry buffer) drains the ring; the next
    call on the same handle works; a failing producer is reported as EINVAL"""
    w = dnagen.config3(total_bases=300_000, lo=50_000, hi=131072)
    tok = dn.DNATok(mode="kmer", k=6, max_record_bytes=4096)
    pinned = torch.from_numpy(w.data.copy()).pin_memory()
    with pytest.raises(dn.DNATokError) as e:
        tok.stream_encode(pinned, w.offsets, 16384, 4, max_rows_per_chunk=64)
    assert e.value.code == dn.ECAPACITY
    torch.cuda.synchronize()
    small = dnagen.config3(total_bases=50_000, lo=100, hi=2000)
    cnt = []

    def on_batch(b):
        with torch.cuda.stream(torch.cuda.ExternalStream(b.stream)):      # read on the batch's own stream
            cnt.append(np.diff(b.out_offsets().cpu().numpy()))
    tok.stream_encode(torch.from_numpy(small.data.copy()).pin_memory(), small.offsets, 16384, 4, max_rows_per_chunk=small.n_records + 1,
                      on_batch=on_batch)
    _, want_off = oracle.encode(small.data, small.offsets, oracle.Config(mode=oracle.KMER, k=6))
    assert np.array_equal(np.concatenate(cnt), np.diff(want_off))

    def bad_fill(i, off, dst):
        raise IOError("no such chunk")
    with pytest.raises(dn.DNATokError) as e:
        tok.stream_encode_from(bad_fill, small.data.size, small.offsets, 16384, 2)
    assert e.value.code == dn.EINVAL
