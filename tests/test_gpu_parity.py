"""GPU parity: the CUDA path (through the C-ABI) against the CPU oracle, bit-exact, ID for ID and offset
for offset, on seeded inputs.  Small shapes span several 16 KiB sub-tiles and ragged tails (tests/test_gpu_fullsize.py
holds the full-size configs); edge cases cover
empty / tiny / huge records, headers across tiles, unaligned pointers and capacity overflow."""
import json
import os
import random

import numpy as np
import pytest

import dnagen
import oracle

torch = pytest.importorskip("torch")
pytestmark = [pytest.mark.gpu, pytest.mark.usefixtures("super_tile")]

if torch.cuda.is_available():
    import paper_2601_05531_b200 as dn


def ocfg(**kw):
    """oracle.Config from binding-style kwargs"""
    m = {"single_nt": oracle.SINGLE_NT, "kmer": oracle.KMER, "bpe": oracle.BPE}
    kw = dict(kw)
    kw["mode"] = m[kw.get("mode", "kmer")]
    kw.pop("id_dtype", None)
    kw.pop("max_record_bytes", None)
    if "class_lut" in kw and kw["class_lut"] is None:
        kw.pop("class_lut")
    return oracle.Config(**kw)


def gpu_encode(data, offsets, misalign=0, **kw):
    tok = dn.DNATok(**kw)
    data = np.ascontiguousarray(data, dtype=np.uint8)
    buf = torch.zeros(data.size + misalign + 64, dtype=torch.uint8, device="cuda")
    d = buf[misalign:misalign + data.size]
    d.copy_(torch.from_numpy(data))
    o = torch.from_numpy(np.ascontiguousarray(offsets, dtype=np.int64)).cuda()
    ids, out = tok.encode(d, o)
    tok.check()
    out = out.cpu().numpy()
    return ids[: out[-1]].cpu().numpy().astype(np.int32), out, tok


def check(data, offsets, **kw):
    if not isinstance(data, np.ndarray):
        data = np.frombuffer(bytes(data), dtype=np.uint8)
    offsets = np.asarray(offsets, dtype=np.int64)
    mis_list = kw.pop("_mis", (0,))
    want_ids, want_off = oracle.encode(data, offsets, ocfg(**kw))
    for mis in mis_list:
        got_ids, got_off, _ = gpu_encode(data, offsets, misalign=mis, **kw)
        assert np.array_equal(got_off, want_off), (np.flatnonzero(got_off != want_off)[:5], got_off[:8], want_off[:8])
        assert got_ids.shape == want_ids.shape
        bad = np.flatnonzero(got_ids != want_ids)
        assert bad.size == 0, (bad[:8], got_ids[bad[:8]], want_ids[bad[:8]])


ALL_MODES = [dict(mode="single_nt"), dict(mode="kmer", k=1), dict(mode="kmer", k=3), dict(mode="kmer", k=6),
             dict(mode="kmer", k=8), dict(mode="kmer", k=15),
             dict(mode="kmer", k=6, tail_policy=1), dict(mode="kmer", k=4, tail_policy=2),
             dict(mode="kmer", k=6, id_dtype=2)]


def test_handworked_example(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "handworked_example.json")))
    data = (g["record0"] + g["record1"]).encode()
    ids, out, _ = gpu_encode(np.frombuffer(data, dtype=np.uint8), g["rec_offsets"], mode="single_nt")
    assert ids.tolist() == g["single_nt"]["ids"] and out.tolist() == g["single_nt"]["out_offsets"]
    ids, out, _ = gpu_encode(np.frombuffer(data, dtype=np.uint8), g["rec_offsets"], mode="kmer", k=3)
    assert ids.tolist() == g["kmer3"]["ids"] and out.tolist() == g["kmer3"]["out_offsets"]
    ids, out, _ = gpu_encode(np.frombuffer(data, dtype=np.uint8), g["rec_offsets"], mode="bpe",
                             merges=np.array(g["bpe"]["merges"], dtype=np.int32), n_id=2)
    assert ids.tolist() == g["bpe"]["ids"] and out.tolist() == g["bpe"]["out_offsets"]


def test_config1_small_and_full():
    for w in (dnagen.config1(n_records=3, bases=20000), dnagen.config1()):
        check(w.data, w.offsets, mode="single_nt")


@pytest.mark.parametrize("kw", ALL_MODES)
def test_config2_small(kw):
    w = dnagen.config2(n_records=24, bases=5000 + 37, n_frac=0.01)
    check(w.data, w.offsets, **kw)


@pytest.mark.parametrize("k", [1, 2, 3, 4, 5, 6, 8])
def test_config3_small_fasta(k):
    w = dnagen.config3(total_bases=300_000)
    check(w.data, w.offsets, mode="kmer", k=k, id_dtype=2 if k <= 6 else 4)


def test_config3_small_single_nt_and_no_header_strip():
    w = dnagen.config3(total_bases=100_000)
    check(w.data, w.offsets, mode="single_nt")
    check(w.data, w.offsets, mode="kmer", k=6, strip_headers=False)


def test_config5_small_records_with_terminator():
    w = dnagen.config5(total_bytes=40 * 4097 + 8, bases=4096)
    check(w.data, w.offsets, mode="kmer", k=6)


def test_unaligned_input_pointer():
    w = dnagen.config3(total_bases=60_000)
    check(w.data, w.offsets, mode="kmer", k=6, _mis=(1, 7, 15))


def test_offsets_not_covering_buffer():
    w = dnagen.config3(total_bases=200_000, lo=1000, hi=8000)
    assert w.n_records > 10
    offs = w.offsets[2:-3]
    check(w.data, offs, mode="kmer", k=6)
    check(w.data, offs, mode="single_nt")


@pytest.mark.parametrize("kw", [dict(mode="single_nt"), dict(mode="kmer", k=6), dict(mode="kmer", k=2)])
def test_degenerate_inputs(kw):
    check(b"", [0], **kw)                                  # no records, no bytes
    check(b"", [0, 0, 0], **kw)                            # empty records only
    check(b"ACGT", [0, 0, 4, 4], **kw)                     # empty records around a real one
    check(b"A", [0, 1], **kw)
    check(b">only header", [0, 12], **kw)
    check(b">h\n", [0, 3], **kw)
    check(b"\n\n\n", [0, 1, 3], **kw)
    check(b"ACGTNNNNacgtRYK-*", [0, 17], **kw)
    check(b"AC\r\nGT\r\n>x\r\nAC", [0, 14], **kw)
    check(b"\r>hdr\nAC>GT\n", [0, 12], **kw)


def test_many_tiny_records_in_one_tile():
    # > 256 record starts per 8 KiB tile: exercises the chunked event loop and warp-per-segment emit
    rng = np.random.default_rng(5)
    lens = rng.integers(0, 9, size=5000)
    data = rng.choice(np.frombuffer(b"ACGTN", dtype=np.uint8), size=int(lens.sum()))
    offs = np.concatenate([[0], np.cumsum(lens)])
    for kw in (dict(mode="kmer", k=3), dict(mode="single_nt"), dict(mode="kmer", k=6, tail_policy=2)):
        check(data, offs, **kw)


@pytest.mark.parametrize("n_rec", [31, 32, 33, 63, 127, 128, 1023, 1024, 4095, 4096, 4097])
def test_record_counts_around_the_search_fanout(n_rec):
    # the per-tile record search is 32-ary: counts where a narrowed range is a multiple of 32 hit its edge cases
    rng = np.random.default_rng(n_rec)
    lens = rng.integers(250, 350, size=n_rec)
    data = rng.choice(np.frombuffer(b"ACGTN", dtype=np.uint8), size=int(lens.sum()), p=[.245, .245, .245, .245, .02])
    offs = np.concatenate([[0], np.cumsum(lens)])
    check(data, offs, mode="kmer", k=6)


def test_records_aligned_to_tile_boundaries():
    rng = np.random.default_rng(6)
    data = rng.choice(np.frombuffer(b"ACGT", dtype=np.uint8), size=8192 * 5)
    check(data, [0, 8192, 16384, 16384, 8192 * 4, 8192 * 5], mode="kmer", k=6)
    check(data, [8192, 8192 * 3], mode="kmer", k=5)
    check(data, [8191, 8193, 8192 * 2 + 1, 8192 * 5], mode="kmer", k=6)


def test_long_header_and_single_line_record_across_tiles():
    rng = np.random.default_rng(7)
    seq = rng.choice(np.frombuffer(b"ACGT", dtype=np.uint8), size=40_000).tobytes()
    hdr = b">" + b"x" * 20_000 + b"\n"                     # header longer than two tiles
    rec0 = hdr + seq[:30_000] + b"\n" + hdr + seq[30_000:]
    rec1 = b">" + b"ACGT" * 5_000                          # header with no newline: runs to the record's end
    rec2 = seq                                             # one 40 kB line, no newline at all
    data = rec0 + rec1 + rec2
    offs = [0, len(rec0), len(rec0) + len(rec1), len(data)]
    for kw in (dict(mode="kmer", k=6), dict(mode="single_nt"), dict(mode="kmer", k=6, strip_headers=False)):
        check(data, offs, **kw)


def test_gt_at_tile_start_and_newline_at_tile_end():
    # '\n' is the last byte of tile 0 and '>' the first byte of tile 1: header detection crosses the tile edge
    body = b"ACGT" * 2047 + b"ACG\n"                        # 8192 bytes ending in '\n'
    data = body + b">hdr in the next tile\nACGTACGTAC\n"
    check(data, [0, len(data)], mode="kmer", k=6)
    data2 = body[:-1] + b"A" + b">not a header: mid-line\nACGT\n"
    check(data2, [0, len(data2)], mode="kmer", k=6)
    data3 = body[:-2] + b"\n\r" + b">hdr after a CR at the line start\nACGT\n"
    check(data3, [0, len(data3)], mode="single_nt")


@pytest.mark.parametrize("edge", [16384, 32768, 65536, 131072])
def test_line_state_across_super_tile_edges(edge):
    """The entry line state of a super-tile is read off the 128 bytes in front of it when they hold a newline or the
    record start, else it comes from the chain (and the super-tile is redone if it was not IN_LINE).  `edge` is a
    super-tile boundary for every super-tile size that divides it."""
    rng = np.random.default_rng(edge)
    acgt = lambda n: rng.choice(np.frombuffer(b"ACGT", dtype=np.uint8), size=n).tobytes()
    cases = {
        "newline last, '>' first": acgt(edge - 1) + b"\n" + b">hdr\n" + acgt(300) + b"\n",
        "header starts 100 before, ends 200 after": acgt(edge - 101) + b"\n>" + b"h" * 299 + b"\n" + acgt(500),
        "header starts 200 before (no newline in the last 128)": acgt(edge - 201) + b"\n>" + b"h" * 500 + b"\n" + acgt(500),
        "header spans several super-tiles": acgt(50) + b"\n>" + b"h" * (edge + 70_000) + b"\n" + acgt(500),
        "long line, no newline for 1000 bytes": acgt(edge - 1001) + b"\n" + acgt(1000 + 700) + b"\n>x\n" + acgt(9),
        "CR LF then '>'": acgt(edge - 2) + b"\r\n" + b">hdr\r\n" + acgt(77) + b"\r\n",
        "newline, CR at the edge, then '>'": acgt(edge - 1) + b"\n" + b"\r>hdr\n" + acgt(77),
        "'>' mid-line at the edge": acgt(edge) + b">not a header\n" + acgt(77),
        "record starts 60 before with '>' (record start inside the window)": None,
    }
    for name, data in cases.items():
        if data is None:
            data = acgt(edge - 60) + b">" + b"h" * 200 + b"\n" + acgt(400)
            offs = [0, edge - 60, len(data)]
        else:
            offs = [0, len(data)]
        for kw in (dict(mode="kmer", k=6), dict(mode="single_nt")):
            check(data, offs, **kw)


@pytest.mark.parametrize("k", [5, 6, 8])
def test_walk_back_over_many_super_tiles(k):
    """3 MiB in three records: with 16 KiB super-tiles the look-back walks through several windows of 32 aggregates
    that hold no record start, carrying the open record's (q, r) and pending bases"""
    w = dnagen.config2(n_records=3, bases=(1 << 20) + 12345, n_frac=0.002)
    check(w.data, w.offsets, mode="kmer", k=k)


@pytest.mark.parametrize("seed", range(12))
def test_fuzz_fasta_like(seed):
    rng = random.Random(seed)
    recs = []
    for _ in range(rng.randrange(1, 60)):
        n = rng.choice([0, 1, 5, rng.randrange(0, 3000), rng.randrange(0, 30000)])
        body = "".join(rng.choice("ACGTACGTACGTNacgtnR") for _ in range(n))
        style = rng.randrange(4)
        if style == 0:
            rec = body
        elif style == 1:
            w = rng.choice([1, 7, 60, 80, 8191])
            rec = ">r %d\n" % n + "\n".join(body[i:i + w] for i in range(0, n, w)) + "\n"
        elif style == 2:
            rec = ">h1\r\n>h2\r\n" + "\r\n".join(body[i:i + 61] for i in range(0, n, 61))
        else:
            rec = body[: n // 2] + "\n>mid header " + "z" * rng.randrange(0, 200) + "\n" + body[n // 2:] + "\n\n"
        recs.append(rec.encode())
    data = np.frombuffer(b"".join(recs), dtype=np.uint8)
    offs = np.cumsum([0] + [len(r) for r in recs])
    kw = rng.choice(ALL_MODES)
    check(data, offs, _mis=(rng.randrange(16),), **kw)
    check(data, offs, strip_headers=False, **kw)


def test_custom_lut_and_vocab():
    lut = oracle.default_lut()
    lut[ord("-")] = oracle.CLS_SKIP
    lut[ord("U")] = 3
    lut[ord("u")] = 3
    data = b"AC-GU\n->x\nacgu--NNR\n" * 700
    check(data, [0, len(data)], mode="kmer", k=4, class_lut=lut, unk_id=9, base_id=100)
    check(data, [0, len(data)], mode="single_nt", class_lut=lut, nt_ids=(1, 2, 3, 4, 0), unk_id=0)   # paper LUT (Q1)


def test_capacity_overflow_reports_and_writes_nothing_past_the_end():
    w = dnagen.config2(n_records=4, bases=4000, n_frac=0)
    tok = dn.DNATok(mode="single_nt")
    d = torch.from_numpy(w.data).cuda()
    o = torch.from_numpy(w.offsets).cuda()
    ids = torch.full((10_000 + 64,), -7, dtype=torch.int32, device="cuda")
    tok.encode(d, o, ids_out=ids[:10_000])
    with pytest.raises(dn.DNATokError) as e:
        tok.check()
    assert e.value.code == dn.ECAPACITY
    assert (ids[10_000:] == -7).all()
    want, _ = oracle.encode(w.data, w.offsets, oracle.Config(mode=oracle.SINGLE_NT))
    assert np.array_equal(ids[:10_000].cpu().numpy(), want[:10_000])
    tok.check()                                             # status is sticky only until read


def test_create_rejects_bad_configs():
    for kw in (dict(mode="kmer", k=0), dict(mode="kmer", k=16), dict(mode="kmer", k=8, id_dtype=2),
               dict(mode="bpe", merges=np.array([[0, 4]], dtype=np.int32)),
               dict(mode="bpe", merges=np.array([[0, 1], [0, 1]], dtype=np.int32)),
               dict(mode="kmer", k=6, seq_len=-1)):
        with pytest.raises(dn.DNATokError) as e:
            dn.DNATok(**kw)
        assert e.value.code == dn.EINVAL


def test_repeated_calls_on_one_handle_reuse_scratch():
    tok = dn.DNATok(mode="kmer", k=6)
    for n in (3, 40, 5, 17):
        w = dnagen.config2(n_records=n, bases=3001, n_frac=0.01, seed=n)
        d, o = torch.from_numpy(w.data).cuda(), torch.from_numpy(w.offsets).cuda()
        ids, out = tok.encode(d, o)
        tok.check()
        want_ids, want_off = oracle.encode(w.data, w.offsets, oracle.Config(mode=oracle.KMER, k=6))
        out = out.cpu().numpy()
        assert np.array_equal(out, want_off) and np.array_equal(ids[: out[-1]].cpu().numpy(), want_ids)


# ------------------------------------------------------------------------------------------- BPE
def test_bpe_config4_small():
    w = dnagen.config4(n_reads=300, n_merges=4092)
    check(w.data, w.offsets, mode="bpe", merges=w.merges, max_record_bytes=2048)


@pytest.mark.parametrize("seed", range(6))
def test_bpe_fuzz(seed):
    rng = random.Random(seed)
    merges = dnagen.merge_table(seed=seed, n_merges=rng.choice([1, 5, 60, 500]), corpus_bases=8192)
    recs = []
    for _ in range(rng.randrange(1, 80)):
        n = rng.choice([0, 1, 2, rng.randrange(0, 200), rng.randrange(0, 2000)])
        alphabet = rng.choice(["ACGT", "ACGTN", "A", "AAAAAC", "ACGTACGTACGTACGTNR\n"])
        recs.append("".join(rng.choice(alphabet) for _ in range(n)).encode())
    data = np.frombuffer(b"".join(recs), dtype=np.uint8)
    offs = np.cumsum([0] + [len(r) for r in recs])
    check(data, offs, mode="bpe", merges=merges, max_record_bytes=2048)


def test_bpe_homopolymer_runs_and_fasta_layout():
    merges = np.array([[0, 0], [4, 4], [5, 5], [3, 3], [7, 0]], dtype=np.int32)
    data = (b">r\n" + b"A" * 777 + b"\n" + b"T" * 300 + b"A" * 5 + b"\nNN" + b"A" * 64 + b"\n")
    check(data, [0, len(data)], mode="bpe", merges=merges, max_record_bytes=2048)


def test_bpe_segment_lengths_around_the_group_sizes():
    """segments on both sides of every length class of the merge kernel (one segment per lane up to 64 symbols, per 2 / 4 /
    8 lanes up to 128 / 256 / 512, per warp up to 2048, the giant kernel beyond), side by side in the same reads, and
    lengths on both sides of a 32-class step of the segment finder"""
    rng = random.Random(7)
    merges = dnagen.merge_table(seed=3, n_merges=200, corpus_bases=8192)
    seg = lambda n: "".join(rng.choice("ACGT") for _ in range(n))
    recs = [seg(63) + "N" + seg(64) + "N" + seg(65) + "N" + seg(1), seg(127) + "NN" + seg(128) + "N" + seg(129) + "N",
            seg(255) + "R" + seg(256) + "N" + seg(257), seg(511) + "N" + seg(512) + "N" + seg(513), seg(2047) + "N" + seg(2), seg(2048),
            "N" + seg(2049) + "R" + seg(50), seg(5000), seg(31) + "N" + seg(32) + "N" + seg(33) + "N" + seg(31), seg(32), seg(64) + "N",
            "", "N", seg(1), seg(2), "NN", seg(8) + "N" + seg(9) + "N" + seg(16) + "N" + seg(17)]
    data = np.frombuffer("".join(recs).encode(), dtype=np.uint8)
    offs = np.cumsum([0] + [len(r) for r in recs])
    check(data, offs, mode="bpe", merges=merges, max_record_bytes=8192)


def test_bpe_many_segments_of_every_bin():
    """a few thousand segments of every length from 1 to 520 (every 8-wide length bin, work items that are not full) and
    a table whose rules keep firing on random ACGT"""
    rng = random.Random(11)
    merges = dnagen.merge_table(seed=5, n_merges=1500, corpus_bases=65536)
    recs, cur = [], []
    for n in list(range(1, 521)) * 3:
        cur.append("".join(rng.choice("ACGT") for _ in range(n)))
        if len(cur) == 7:
            recs.append("N".join(cur)); cur = []
    recs.append("N".join(cur))
    data = np.frombuffer("".join(recs).encode(), dtype=np.uint8)
    offs = np.cumsum([0] + [len(r) for r in recs])
    check(data, offs, mode="bpe", merges=merges, max_record_bytes=8192)


def test_bpe_segment_longer_than_workspace_reports_capacity():
    """the merge kernels hold ACGT segments of up to max(2048, max_record_bytes) symbols (at most 49152); a longer run between
    two N / UNK bytes is reported as ECAPACITY"""
    merges = np.array([[0, 1]], dtype=np.int32)
    tok = dn.DNATok(mode="bpe", merges=merges, max_record_bytes=256)
    d = torch.from_numpy(np.frombuffer(b"AC" * 1500, dtype=np.uint8).copy()).cuda()
    o = torch.tensor([0, 3000], dtype=torch.int64, device="cuda")
    tok.encode(d, o)
    with pytest.raises(dn.DNATokError) as e:
        tok.check()
    assert e.value.code == dn.ECAPACITY


# ------------------------------------------------------------------------------------------- pad + mask
@pytest.mark.parametrize("side", [0, 1])
@pytest.mark.parametrize("seq_len", [5, 64, 700, 8192])
@pytest.mark.parametrize("id_dtype", [2, 4])
def test_pad_mask(side, seq_len, id_dtype):
    w = dnagen.config3(total_bases=80_000)
    kw = dict(mode="kmer", k=6, seq_len=seq_len, pad_side=side, id_dtype=id_dtype)
    tok = dn.DNATok(**kw)
    d, o = torch.from_numpy(w.data).cuda(), torch.from_numpy(w.offsets).cuda()
    ids, out = tok.encode(d, o)
    batch, mask = tok.pad(ids, out)
    tok.check()
    cfg = ocfg(**kw)
    want_ids, want_off = oracle.encode(w.data, w.offsets, cfg)
    want_batch, want_mask = oracle.pad(want_ids, want_off, cfg)
    assert np.array_equal(batch.cpu().numpy(), want_batch) and np.array_equal(mask.cpu().numpy(), want_mask)


def test_pad_handworked(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "handworked_example.json")))
    data = np.frombuffer((g["record0"] + g["record1"]).encode(), dtype=np.uint8).copy()
    for side, key in ((0, "kmer3_pad5_left"), (1, "kmer3_pad5_right")):
        tok = dn.DNATok(mode="kmer", k=3, seq_len=5, pad_side=side)
        batch, mask, _ = tok.encode_padded(torch.from_numpy(data).cuda(), torch.tensor(g["rec_offsets"]).cuda())
        tok.check()
        assert batch.cpu().tolist() == g[key]["ids"] and mask.cpu().tolist() == g[key]["mask"]


# ------------------------------------------------------------------------------------------- custom tables on every path
def _lut(**over):
    lut = oracle.default_lut()
    for ch, c in over.items():
        lut[ord(ch)] = c
    return lut


@pytest.mark.parametrize("name,lut", [
    ("soft-masked lowercase is N (no arithmetic classification of acgt)", dict(a=4, c=4, g=4, t=4)),
    ("N is UNK (runs of N take the table)", dict(N=5, n=5)),
    ("'-' and '*' are skipped, 'U' is T", {"-": 255, "*": 255, "U": 3, "u": 3}),
    ("'>' itself is a SKIP byte but still opens a header", {">": 255}),
])
@pytest.mark.parametrize("k", [1, 6])
def test_custom_luts_on_multi_super_tile_fasta(name, lut, k):
    """EncParams.fast_lut = 0 / fast_n = 0 and extra SKIP bytes, on FASTA that spans many super-tiles, with headers and skipped
    bytes sprinkled around the super-tile edges (16 KiB multiples)"""
    w = dnagen.config3(total_bases=600_000, lo=1000, hi=70_000, seed=5)
    data = w.data.copy()
    rng = np.random.default_rng(k)
    edges = np.arange(16384, data.size - 200, 16384)
    for e in edges:                                           # soft-masked runs, gaps and stops around every edge
        a = int(e + rng.integers(-150, 150))
        run = data[a: a + 40]
        keep = run != 10
        if rng.random() < 0.5:
            run[keep] = np.char.lower(run[keep].view("S1")).view(np.uint8)
        else:
            run[keep & (rng.random(40) < 0.3)] = ord("-")
        data[int(e + rng.integers(-3, 3))] = rng.choice(np.frombuffer(b"*-Nn>U", dtype=np.uint8))
    data[data == 0] = ord("A")
    check(data, w.offsets, mode="kmer", k=k, class_lut=_lut(**lut))


@pytest.mark.parametrize("mode,k,dt", [("single_nt", 1, 4), ("kmer", 6, 2), ("kmer", 3, 4)])
def test_ids_out_pointer_that_is_not_16_byte_aligned(mode, k, dt):
    w = dnagen.config3(total_bases=200_000, lo=100, hi=30_000)
    kw = dict(mode=mode, k=k, id_dtype=dt)
    tok = dn.DNATok(**kw)
    d, o = torch.from_numpy(w.data).cuda(), torch.from_numpy(w.offsets).cuda()
    buf = torch.empty(w.data.size + 8, dtype=tok.id_torch_dtype, device="cuda")
    want_ids, want_off = oracle.encode(w.data, w.offsets, ocfg(**kw))
    for shift in (1, 3):
        ids, out = tok.encode(d, o, ids_out=buf[shift:])
        tok.check()
        out = out.cpu().numpy()
        assert np.array_equal(out, want_off) and np.array_equal(ids[: out[-1]].cpu().numpy().astype(np.int32), want_ids)


def test_pad_into_unaligned_views():
    w = dnagen.config3(total_bases=60_000, lo=10, hi=3000)
    tok = dn.DNATok(mode="kmer", k=6, seq_len=64)
    d, o = torch.from_numpy(w.data).cuda(), torch.from_numpy(w.offsets).cuda()
    ids, out = tok.encode(d, o)
    n = w.n_records
    bbuf = torch.empty(n * 64 + 4, dtype=torch.int32, device="cuda")
    mbuf = torch.empty(n * 64 + 4, dtype=torch.uint8, device="cuda")
    batch, mask = tok.pad(ids, out, batch_ids=bbuf[1: 1 + n * 64].view(n, 64), mask=mbuf[1: 1 + n * 64].view(n, 64))
    tok.check()
    c = oracle.Config(mode=oracle.KMER, k=6, seq_len=64)
    wi, wo = oracle.encode(w.data, w.offsets, c)
    wb, wm = oracle.pad(wi, wo, c)
    assert np.array_equal(batch.cpu().numpy(), wb) and np.array_equal(mask.cpu().numpy(), wm)
