"""GPU parity of the regular-layout FASTA encoder (csrc/encode_fasta.cuh) and of its hand-over to the chained-scan encoder.
Every case compares IDs and offsets bit for bit with the CPU oracle AND asserts which of the two encoders served the call
(dnatok_fast_path_taken), so that neither "always falls back" nor "never falls back" can pass unnoticed: layouts the
closed form covers must be taken, every violation of it -- planted at tile, chunk and record edges -- must be caught."""
import random

import numpy as np
import pytest

import oracle

torch = pytest.importorskip("torch")
pytestmark = [pytest.mark.gpu]

if torch.cuda.is_available():
    import paper_2601_05531_b200 as dn

M = {"single_nt": oracle.SINGLE_NT, "kmer": oracle.KMER}
MODES = [dict(mode="single_nt"), dict(mode="kmer", k=1), dict(mode="kmer", k=3), dict(mode="kmer", k=6), dict(mode="kmer", k=8),
         dict(mode="kmer", k=15), dict(mode="kmer", k=6, tail_policy=1), dict(mode="kmer", k=4, tail_policy=2),
         dict(mode="kmer", k=6, id_dtype=2)]


@pytest.fixture(autouse=True)
def fast_path_on_every_size():
    old = dn.FAST_PATH
    dn.FAST_PATH = 2
    yield
    dn.FAST_PATH = old


def run(data, offsets, taken, misalign=0, **kw):
    """encode on the GPU and with the oracle; taken = True / False / None (either)"""
    if not isinstance(data, np.ndarray):
        data = np.frombuffer(bytes(data), dtype=np.uint8)
    offsets = np.asarray(offsets, dtype=np.int64)
    okw = dict(kw)
    okw["mode"] = M[okw.get("mode", "kmer")]
    okw.pop("id_dtype", None)
    want_ids, want_off = oracle.encode(data, offsets, oracle.Config(**okw))
    tok = dn.DNATok(**kw)
    buf = torch.zeros(data.size + misalign + 64, dtype=torch.uint8, device="cuda")
    d = buf[misalign:misalign + data.size]
    d.copy_(torch.from_numpy(np.ascontiguousarray(data)))
    o = torch.from_numpy(offsets).cuda()
    ids, out = tok.encode(d, o)
    tok.check()
    got_taken = tok.fast_path_taken()
    out = out.cpu().numpy()
    got = ids[: out[-1]].cpu().numpy().astype(np.int32)
    assert np.array_equal(out, want_off), (np.flatnonzero(out != want_off)[:5], out[:6], want_off[:6])
    bad = np.flatnonzero(got != want_ids)
    assert bad.size == 0, (bad[:8], got[bad[:8]], want_ids[bad[:8]])
    if taken is not None:
        assert got_taken == taken, "fast path %s" % ("not taken" if taken else "taken on a layout it must reject")
    return got_taken


def fasta(rng, n_rec, width, lo, hi, header=True, last_newline=True, alphabet="ACGT"):
    recs = []
    for i in range(n_rec):
        n = rng.randrange(lo, hi + 1)
        seq = "".join(rng.choice(alphabet) for _ in range(n))
        w = width(i) if callable(width) else width
        body = "\n".join(seq[j:j + w] for j in range(0, n, w))
        if n and last_newline:
            body += "\n"
        recs.append((((">rec%d len=%d\n" % (i, n)) if header else "") + body).encode())
    return np.frombuffer(b"".join(recs), dtype=np.uint8), np.cumsum([0] + [len(r) for r in recs])


# ------------------------------------------------------------------------------------------------ layouts that are taken
@pytest.mark.parametrize("W", [1, 2, 3, 15, 16, 17, 31, 59, 60, 63, 64, 65, 66, 80, 100, 127, 128, 129, 200, 500, 511])
def test_every_line_width(W):
    rng = random.Random(W)
    data, offs = fasta(rng, 12, W, 1500, 9000)
    for kw in (dict(mode="kmer", k=6), dict(mode="single_nt"), dict(mode="kmer", k=1 + W % 9)):
        run(data, offs, True, **kw)


@pytest.mark.parametrize("kw", MODES, ids=lambda kw: "-".join("%s%s" % kv for kv in kw.items()))
def test_every_mode_on_wrapped_records(kw):
    rng = random.Random(7)
    data, offs = fasta(rng, 20, 60, 0, 12000, alphabet="ACGTACGTACGTNacgtnRY-")
    run(data, offs, True, **kw)
    run(data, offs, True, misalign=rng.randrange(1, 16), **kw)


def test_records_without_header_or_last_line_end():
    rng = random.Random(1)
    for header in (True, False):
        for last in (True, False):
            data, offs = fasta(rng, 15, 70, 0, 5000, header=header, last_newline=last)
            run(data, offs, True, mode="kmer", k=6)
            if not header:
                run(data, offs, True, mode="kmer", k=6, strip_headers=False)


def test_body_lengths_that_are_multiples_of_the_width():
    rng = random.Random(2)
    recs = []
    for n in (60, 120, 600, 6000, 59, 60 * 137, 61, 1, 0):                   # at most 16 records touch one 16 KiB tile
        seq = "".join(rng.choice("ACGT") for _ in range(n))
        recs.append((">x\n" + "".join(seq[j:j + 60] + "\n" for j in range(0, n, 60))).encode())
    run(b"".join(recs), np.cumsum([0] + [len(r) for r in recs]), True, mode="kmer", k=6)
    run(b"".join(recs), np.cumsum([0] + [len(r) for r in recs]), True, mode="kmer", k=7, tail_policy=2)


def test_a_different_width_in_every_record():
    rng = random.Random(3)
    widths = [60, 80, 7, 200, 65, 64, 1, 333, 70, 61, 100, 50]
    data, offs = fasta(rng, len(widths), lambda i: widths[i], 2000, 7000)
    run(data, offs, True, mode="kmer", k=6)
    run(data, offs, True, mode="single_nt")


def test_header_only_empty_and_unterminated_header_records():
    recs = [b">only a header\n", b"", b">", b">no line end", b">h\nACGTACGTAC\n", b"", b">h2\nA", b">h3\n", b"\nACGT\n", b"\n", b"ACGT",
            b">z\nAC\nGT\nA\n"]
    offs = np.cumsum([0] + [len(r) for r in recs])
    # "\nACGT\n": a body that starts with an empty line is not regular -- the call as a whole falls back
    run(b"".join(recs), offs, False, mode="kmer", k=3)
    recs.remove(b"\nACGT\n")
    for part in (recs[:6], recs[5:]):                                          # at most 16 records per 16 KiB tile are taken
        offs = np.cumsum([0] + [len(r) for r in part])
        run(b"".join(part), offs, True, mode="kmer", k=3)
        run(b"".join(part), offs, True, mode="single_nt")


def test_one_line_records_longer_than_the_parse_bound():
    """config 5's shape: a single line of some thousand bases ended by one line end, no header"""
    rng = random.Random(4)
    recs = [("".join(rng.choice("ACGT") for _ in range(rng.randrange(1000, 30000))) + "\n").encode() for _ in range(14)]
    offs = np.cumsum([0] + [len(r) for r in recs])
    run(b"".join(recs), offs, True, mode="kmer", k=6)
    recs = [r[:-1] for r in recs]                                             # ... and without the line end
    run(b"".join(recs), np.cumsum([0] + [len(r) for r in recs]), True, mode="kmer", k=6)


def test_header_lengths_up_to_the_parse_bound():
    rng = random.Random(5)
    recs = []
    for hl in (1, 2, 63, 64, 65, 1000, 4094, 4095):
        seq = "".join(rng.choice("ACGT") for _ in range(700))
        recs.append((">" + "h" * (hl - 1) + "\n" + "\n".join(seq[j:j + 60] for j in range(0, 700, 60)) + "\n").encode())
    run(b"".join(recs), np.cumsum([0] + [len(r) for r in recs]), True, mode="kmer", k=6)
    seq = "ACGT" * 100
    long_hdr = (">" + "h" * 4200 + "\n" + seq + "\n").encode()                # header line beyond the bound: chained-scan encoder
    run(long_hdr + b"".join(recs), np.cumsum([0, len(long_hdr)] + [len(r) for r in recs]), False, mode="kmer", k=6)


def test_up_to_sixteen_records_per_warp_tile_are_taken_and_more_fall_back():
    rng = random.Random(6)
    data, offs = fasta(rng, 64, 60, 1300, 1500)                               # ~1.4 KiB records: at most 13 pieces per 16 KiB tile
    run(data, offs, True, mode="kmer", k=6)
    data, offs = fasta(rng, 400, 60, 0, 300)                                  # dozens of records per tile
    run(data, offs, False, mode="kmer", k=6)


def test_offsets_that_leave_gaps_and_do_not_start_at_zero():
    rng = random.Random(8)
    data, offs = fasta(rng, 10, 60, 3000, 9000)
    lead = np.frombuffer(b"garbage in front of the first record\n>>>\n", dtype=np.uint8)
    data = np.concatenate([lead, data, lead])
    run(data, offs + lead.size, None, mode="kmer", k=6)


# ------------------------------------------------------------------------------------------------ violations that are caught
def regular_input(seed, n_rec=6, W=60):
    rng = random.Random(seed)
    data, offs = fasta(rng, n_rec, W, 4000, 9000)
    return data.copy(), offs


def edge_positions(data, offs):
    """bytes next to warp-tile (16 KiB) and chunk (2 KiB) edges, record edges, and the ends of the input"""
    pos = set()
    for e in list(range(0, data.size, 2048)) + list(offs) + [data.size]:
        for dlt in (-66, -65, -64, -63, -17, -16, -2, -1, 0, 1, 2, 15, 16, 17, 63, 64, 65):
            if 0 <= e + dlt < data.size:
                pos.add(int(e + dlt))
    return sorted(pos)


@pytest.mark.parametrize("kind", ["base_to_newline", "newline_to_base", "gt_at_line_start", "base_to_cr"])
def test_one_violation_anywhere_near_an_edge_is_caught(kind):
    data, offs = regular_input(11)
    hdr_end = {}
    for r in range(len(offs) - 1):
        a = int(offs[r])
        hdr_end[r] = a + bytes(data[a:offs[r + 1]]).index(b"\n") + 1
    n_caught = n_run = 0
    cand = edge_positions(data, offs)
    if kind in ("gt_at_line_start", "newline_to_base"):                        # every line start / line end within two lines of an edge
        near = np.zeros(data.size, dtype=bool)
        for p in cand:
            near[max(0, p - 130):p + 130] = True
        nl = np.flatnonzero(near[:-1] & (data[:-1] == 10))
        cand = [int(p) + (kind == "gt_at_line_start") for p in nl]
    for p in cand:
        r = int(np.searchsorted(offs, p, side="right")) - 1
        if p < hdr_end[r]:
            continue                                                           # header bytes are free text
        mut = data.copy()
        if kind == "base_to_newline" and mut[p] != 10:
            mut[p] = 10
        elif kind == "newline_to_base" and mut[p] == 10 and p + 1 < offs[r + 1]:
            mut[p] = ord("A")
        elif kind == "gt_at_line_start" and mut[p] != 10 and mut[p - 1] == 10:
            mut[p] = ord(">")
        elif kind == "base_to_cr" and mut[p] != 10:
            mut[p] = 13
        else:
            continue
        n_run += 1
        # a mutation may leave another regular layout (e.g. the record's last line split in two is still "lines of width W,
        # a short one last" only if it is the last line): the oracle decides the IDs, the flag is checked where it must be set
        taken = run(mut, offs, None, mode="kmer", k=6)
        n_caught += not taken
    assert n_run >= 20
    if kind in ("gt_at_line_start", "base_to_cr"):
        assert n_caught == n_run                                               # never a regular layout
    else:
        assert n_caught >= n_run - 12                                          # all but mutations inside a record's last line or first line


def test_violations_in_the_middle_of_long_records():
    data, offs = regular_input(12, n_rec=3, W=80)
    rng = random.Random(12)
    for _ in range(25):
        mut = data.copy()
        p = rng.randrange(200, data.size - 200)
        if mut[p] == 10:
            mut[p] = ord("C")
        else:
            mut[p] = 10
        run(mut, offs, None, mode="kmer", k=6)


def test_crlf_blank_lines_and_second_header_lines():
    seq = "ACGTTGCA" * 400
    lines = [seq[j:j + 60] for j in range(0, len(seq), 60)]
    crlf = (">h\r\n" + "\r\n".join(lines) + "\r\n").encode()
    blank = (">h\n" + "\n".join(lines[:20]) + "\n\n" + "\n".join(lines[20:]) + "\n").encode()
    two_hdr = (">h\n>second header line\n" + "\n".join(lines) + "\n").encode()
    mid_hdr = (">h\n" + "\n".join(lines[:30]) + "\n>mid\n" + "\n".join(lines[30:]) + "\n").encode()
    ragged = (">h\n" + "\n".join(lines[:10]) + "\n" + seq[:61] + "\n" + "\n".join(lines[10:]) + "\n").encode()
    ok = (">h\n" + "\n".join(lines) + "\n").encode()
    for rec in (crlf, blank, two_hdr, mid_hdr, ragged):
        both = ok + rec + ok
        run(both, [0, len(ok), len(ok) + len(rec), len(both)], False, mode="kmer", k=6)
        run(both, [0, len(ok), len(ok) + len(rec), len(both)], False, mode="single_nt")
    run(ok + ok, [0, len(ok), 2 * len(ok)], True, mode="kmer", k=6)


def test_first_line_longer_than_the_parse_bound_followed_by_more_lines():
    rng = random.Random(13)
    seq = "".join(rng.choice("ACGT") for _ in range(5000))
    rec = (">h\n" + seq[:700] + "\n" + seq[700:1400] + "\n" + seq[1400:2100] + "\n").encode()     # lines of 700 > 512
    run(rec, [0, len(rec)], False, mode="kmer", k=6)
    one = (">h\n" + seq + "\n").encode()                                       # one long line: regular
    run(one, [0, len(one)], True, mode="kmer", k=6)


def test_custom_lut_that_keeps_line_ends_or_skips_other_bytes():
    lut = oracle.default_lut().copy()
    lut[ord("-")] = oracle.CLS_SKIP                                            # gaps are skipped: wherever one occurs the layout check fails
    rng = random.Random(14)
    data, offs = fasta(rng, 5, 60, 3000, 6000, alphabet="ACGT")
    run(data, offs, True, mode="kmer", k=6, class_lut=lut)
    gapped = data.copy()
    p = int(offs[2]) + 500
    p += int(gapped[p] == 10)
    gapped[p] = ord("-")
    run(gapped, offs, False, mode="kmer", k=6, class_lut=lut)
    lut2 = oracle.default_lut().copy()
    lut2[10] = oracle.CLS_UNK                                                  # a table that keeps '\n' as an unknown base
    data, offs = fasta(rng, 5, 60, 3000, 6000, header=False)
    run(data, offs, False, mode="kmer", k=6, class_lut=lut2, strip_headers=False)


def test_fuzz_mixture_of_regular_and_irregular_inputs():
    n_taken = 0
    for seed in range(24):
        rng = random.Random(1000 + seed)
        W = rng.choice([1, 5, 60, 61, 64, 65, 80, 120, 300])
        data, offs = fasta(rng, rng.randrange(1, 9), W, 0, 20000, header=rng.random() < 0.8, last_newline=rng.random() < 0.8,
                           alphabet=rng.choice(["ACGT", "ACGTN", "ACGTacgtNnRYKM"]))
        data = data.copy()
        if seed % 3 == 0 and data.size > 10:
            for _ in range(rng.randrange(1, 4)):
                data[rng.randrange(data.size)] = rng.choice([10, 10, ord(">"), ord(" "), ord("A"), 13])
        kw = rng.choice(MODES)
        n_taken += run(data, offs, True if seed % 3 else None, misalign=rng.randrange(16), **kw)
    assert n_taken >= 16


def test_threshold_small_inputs_skip_the_fast_path_by_default():
    import dnagen
    dn.FAST_PATH = 1
    rng = random.Random(15)
    data, offs = fasta(rng, 8, 60, 3000, 6000)
    run(data, offs, False, mode="kmer", k=6)                                   # under 48 MiB: chained-scan encoder directly
    w = dnagen.config3(total_bases=52 << 20, lo=1000, hi=131072, seed=15)
    run(w.data, w.offsets, True, mode="kmer", k=6)                             # 48 MiB and more: regular-layout encoder
    dn.FAST_PATH = 0
    run(w.data, w.offsets, False, mode="kmer", k=6)


# ------------------------------------------------------------------------------------------------ fused encode + pad
def run_padded(data, offsets, taken, seq_len, pad_side, misalign=0, **kw):
    """dnatok_encode_pad against oracle encode + pad; a call served by the regular-layout encoder must leave ids_out untouched"""
    if not isinstance(data, np.ndarray):
        data = np.frombuffer(bytes(data), dtype=np.uint8)
    offsets = np.asarray(offsets, dtype=np.int64)
    okw = dict(kw)
    okw["mode"] = {"single_nt": oracle.SINGLE_NT, "kmer": oracle.KMER, "bpe": oracle.BPE}[okw.get("mode", "kmer")]
    okw.pop("id_dtype", None)
    okw.pop("max_record_bytes", None)
    ocfg = oracle.Config(seq_len=seq_len, pad_side=pad_side, **okw)
    want_ids, want_off = oracle.encode(data, offsets, ocfg)
    want_b, want_m = oracle.pad(want_ids, want_off, ocfg)
    tok = dn.DNATok(seq_len=seq_len, pad_side=pad_side, **kw)
    buf = torch.zeros(data.size + misalign + 64, dtype=torch.uint8, device="cuda")
    d = buf[misalign:misalign + data.size]
    d.copy_(torch.from_numpy(np.ascontiguousarray(data)))
    o = torch.from_numpy(offsets).cuda()
    poison = -12345 if tok.id_torch_dtype == torch.int32 else -1234
    ids = torch.full((max(data.size, 1),), poison, dtype=tok.id_torch_dtype, device="cuda")
    n_rec = offsets.size - 1
    batch = torch.full((n_rec, seq_len), -777, dtype=torch.int32, device="cuda")
    mask = torch.full((n_rec, seq_len), 9, dtype=torch.uint8, device="cuda")
    b, m, out = tok.encode_padded(d, o, ids_out=ids, batch_ids=batch, mask=mask)
    tok.check()
    got_taken = tok.fast_path_taken()
    assert np.array_equal(out.cpu().numpy(), want_off)
    gb, gm = b.cpu().numpy(), m.cpu().numpy()
    assert np.array_equal(gm, want_m), np.argwhere(gm != want_m)[:5]
    bad = np.argwhere(gb != want_b)
    assert bad.size == 0, (bad[:5], gb[tuple(bad[0])], want_b[tuple(bad[0])])
    if taken is not None:
        assert got_taken == taken
    if got_taken:
        assert bool((ids == poison).all()), "the CSR ids were written although the tokens went straight into the batch"
    return got_taken


@pytest.mark.parametrize("pad_side", [0, 1])
@pytest.mark.parametrize("seq_len", [512, 333, 8, 2048])
def test_fused_pad_on_wrapped_records(seq_len, pad_side):
    rng = random.Random(seq_len + pad_side)
    # records from empty to several times seq_len tokens (truncation: the first seq_len tokens are kept)
    data, offs = fasta(rng, 14, 60, 0, 9000, alphabet="ACGTACGTACGTN")
    for kw in (dict(mode="kmer", k=6), dict(mode="kmer", k=6, id_dtype=2), dict(mode="single_nt"), dict(mode="kmer", k=3, tail_policy=2),
               dict(mode="kmer", k=5, tail_policy=1), dict(mode="kmer", k=15)):
        run_padded(data, offs, True, seq_len, pad_side, **kw)
    run_padded(data, offs, True, seq_len, pad_side, misalign=5, mode="kmer", k=4)


def test_fused_pad_one_line_records_config5_shape():
    rng = random.Random(21)
    recs = [("".join(rng.choice("ACGT") for _ in range(rng.choice([4096, 4096, 100, 5000, 0, 1]))) + "\n").encode() for _ in range(40)]
    offs = np.cumsum([0] + [len(r) for r in recs])
    run_padded(b"".join(recs), offs, True, 683, 0, mode="kmer", k=6)          # 4096 / 6 = 682.67: full rows, short rows, cut rows
    run_padded(b"".join(recs), offs, True, 683, 1, mode="kmer", k=6)
    run_padded(b"".join(recs), offs, True, 700, 0, mode="kmer", k=6, tail_policy=2)


def test_fused_pad_falls_back_on_irregular_input_and_small_inputs_skip_it():
    rng = random.Random(22)
    data, offs = fasta(rng, 10, 60, 100, 6000)
    bad = data.copy()
    p = int(offs[4]) + 700
    p += int(bad[p] == 10)
    bad[p] = 10                                                                # a line cut in two: the chained-scan encoder + pad kernel
    run_padded(bad, offs, False, 256, 0, mode="kmer", k=6)
    run_padded(bad, offs, False, 256, 1, mode="kmer", k=6, id_dtype=2)
    dn.FAST_PATH = 1
    run_padded(data, offs, False, 256, 0, mode="kmer", k=6)                    # under the size threshold (48 MiB): encode + pad as before
    dn.FAST_PATH = 0
    run_padded(data, offs, False, 256, 0, mode="kmer", k=6)


def test_fused_entry_point_serves_bpe_and_dense_specs_through_the_pad_kernel():
    import dnagen
    rng = random.Random(23)
    merges = dnagen.merge_table(seed=3, n_merges=200, corpus_bases=8192)
    recs = ["".join(rng.choice("ACGTN") for _ in range(rng.randrange(0, 400))).encode() for _ in range(30)]
    offs = np.cumsum([0] + [len(r) for r in recs])
    run_padded(b"".join(recs), offs, False, 64, 0, mode="bpe", merges=merges)
    lut = oracle.default_lut().copy()
    lut[lut == oracle.CLS_SKIP] = oracle.CLS_UNK                               # no SKIP class + no header strip: the dense encoder
    run_padded(b"".join(recs), offs, False, 64, 1, mode="kmer", k=3, class_lut=lut, strip_headers=False)


def test_after_a_failed_layout_check_the_next_calls_skip_the_attempt():
    """dnatok_set_fast_path(1), the default: a fall-back is reported to the host, which then sends the next 8 eligible calls on the
    handle to the chained-scan encoder directly (results are the oracle's either way)"""
    import dnagen
    dn.FAST_PATH = 1
    w = dnagen.config3(total_bases=50 << 20, lo=1000, hi=131072, seed=31)       # over the 48 MiB threshold
    bad = w.data.copy()
    p = bad.size // 3
    p += int(bad[p] == 10)
    bad[p] = 13                                                                # one '\r' inside a line
    cfg = oracle.Config(mode=oracle.KMER, k=6)
    want_ok, want_off_ok = oracle.encode(w.data, w.offsets, cfg)
    want_bad, want_off_bad = oracle.encode(bad, w.offsets, cfg)
    tok = dn.DNATok(mode="kmer", k=6)
    d_ok, d_bad = torch.from_numpy(w.data).cuda(), torch.from_numpy(bad).cuda()
    o = torch.from_numpy(w.offsets).cuda()

    def call(d, want, want_off):
        ids, out = tok.encode(d, o)
        tok.check()
        taken = tok.fast_path_taken()
        out = out.cpu().numpy()
        assert np.array_equal(out, want_off) and np.array_equal(ids[: out[-1]].cpu().numpy(), want)
        return taken

    assert call(d_ok, want_ok, want_off_ok) is True
    assert call(d_bad, want_bad, want_off_bad) is False                        # tried, failed, redone by the chained scan
    skipped = [call(d_ok, want_ok, want_off_ok) for _ in range(8)]
    assert skipped == [False] * 8                                              # not even tried
    assert call(d_ok, want_ok, want_off_ok) is True                            # ... and tried again afterwards
    small = w.data[: int(w.offsets[5])]
    tok2 = dn.DNATok(mode="kmer", k=6)
    ids, out = tok2.encode(torch.from_numpy(small.copy()).cuda(), torch.from_numpy(w.offsets[:6].copy()).cuda())
    tok2.check()
    assert tok2.fast_path_taken() is False                                     # under the threshold: never tried
