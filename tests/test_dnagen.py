"""Generator statistics (SURVEY.md 8(c) last row: generators are inputs, 'parity unpinned' by the paper;
only their stated statistics are pinned) and determinism."""
import numpy as np

import dnagen


def test_config1_layout_and_rates():
    w = dnagen.config1()
    assert w.n_bytes == 1_066_064 and w.n_records == 16                 # Q24
    assert np.all(np.diff(w.offsets) == 66_629)
    d = w.data
    assert (d == 10).sum() == 16 * 1093
    rec = bytes(d[:66_629])
    assert all(len(l) == 60 for l in rec.split(b"\n")[:-2]) and rec.endswith(b"\n")
    bases = d[d != 10]
    assert abs(np.isin(bases, [78, 110]).mean() - 0.01) < 0.002
    assert abs((bases >= 97).mean() - 0.05) < 0.005


def test_config2_statistics():
    w = dnagen.config2(n_records=128)
    d = w.data
    assert w.n_bytes == 128 * 65536 and not (d == 10).any()
    acgt = np.isin(d, [65, 67, 71, 84])
    gc = np.isin(d, [67, 71]).sum() / acgt.sum()
    assert abs(gc - 0.41) < 0.01                                        # Q22
    assert abs((d == 78).mean() - 0.005) < 0.0005                       # Q23
    assert (acgt | (d == 78)).all()


def test_config3_fasta_layout():
    w = dnagen.config3(total_bases=1 << 22)
    assert w.n_bases.sum() == 1 << 22
    assert w.n_bases[:-1].min() >= 1000 and w.n_bases.max() <= 131072    # Q19
    for r in (0, 1, w.n_records - 1):
        rec = bytes(w.data[w.offsets[r]:w.offsets[r + 1]])
        lines = rec.split(b"\n")
        assert lines[0] == b">r%d len=%d" % (r, w.n_bases[r]) and lines[-1] == b""
        assert all(len(l) == 80 for l in lines[1:-2]) and sum(len(l) for l in lines[1:]) == w.n_bases[r]


def test_config4_reads_and_merge_table():
    w = dnagen.config4(n_reads=512, n_merges=200, corpus_bases=16384)
    assert w.n_bases.min() >= 500 and w.n_bases.max() <= 1500           # BJ config 4
    assert abs((w.data == 78).mean() - 0.02) < 0.004
    m = w.merges
    assert m.shape == (200, 2)
    assert all(m[r, 0] < 4 + r and m[r, 1] < 4 + r for r in range(200))  # Q12 validity
    assert len({(int(a), int(b)) for a, b in m}) == 200


def test_config5_layout():
    w = dnagen.config5(total_bytes=10 * 32769 + 8)
    assert w.n_records == 11 and w.n_bytes == 10 * 32769 + 8             # Q18
    assert np.all(w.data[w.offsets[1:-1] - 1] == 10) and w.data[-1] != 10
    assert w.n_bases[-1] == 8


def test_determinism_and_thread_independence():
    a = dnagen.config3(total_bases=1 << 20)
    b = dnagen.config3(total_bases=1 << 20)
    assert np.array_equal(a.data, b.data) and np.array_equal(a.offsets, b.offsets)
    c = dnagen._make("x", a.n_bases, 0, 3, 0, None, 0.0, 0.0, True, 80, False, threads=1)
    assert np.array_equal(a.data, c.data)
    assert not np.array_equal(dnagen.config1(seed=1).data, dnagen.config1(seed=0).data)
