"""World-size-2 and -3 runs of the multi-GPU host logic on CPU (gloo): records are partitioned into contiguous ranges of about
equal byte count, each rank encodes its own range (here with the CPU oracle standing in for the rank's GPU), the only
exchange is one int64 per rank, and the stitched result must equal the whole-buffer encoding."""
import os
import socket

import numpy as np
import pytest

import dnagen
import oracle
from paper_2601_05531_b200.shard import exclusive_token_base, partition_records

torch = pytest.importorskip("torch")


def test_partition_records_balances_bytes_and_covers_everything():
    w = dnagen.config3(total_bases=400_000)
    for world in (1, 2, 3, 8):
        parts = partition_records(w.offsets, world)
        assert parts[0][0] == 0 and parts[-1][1] == w.n_records
        assert all(a[1] == b[0] for a, b in zip(parts, parts[1:]))
        sizes = [int(w.offsets[b] - w.offsets[a]) for a, b in parts]
        longest = int(np.diff(w.offsets).max())
        assert max(sizes) - min(sizes) <= 2 * longest
    assert partition_records(np.array([0], dtype=np.int64), 4) == [(0, 0)] * 4
    assert partition_records(np.array([0, 10], dtype=np.int64), 2)[-1][1] == 1


def _rank_main(rank, world, port, q, few_records=False):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = dnagen.config3(total_bases=150_000, lo=500, hi=9000)          # same seeded input on every rank
        if few_records:                                                   # two records for three ranks: one range is empty
            w = dnagen.config3(total_bases=9000, lo=4000, hi=5000)
            assert w.n_records == 2
        cfg = oracle.Config(mode=oracle.KMER, k=6)
        r0, r1 = partition_records(w.offsets, world)[rank]
        a, b = int(w.offsets[r0]), int(w.offsets[r1])
        ids, off = oracle.encode(w.data[a:b], w.offsets[r0:r1 + 1] - a, cfg)
        base, total = exclusive_token_base(int(off[-1]))
        pieces = [None] * world
        dist.all_gather_object(pieces, (r0, r1, base, total, ids, off))
        if rank == 0:
            want_ids, want_off = oracle.encode(w.data, w.offsets, cfg)
            got_ids = np.concatenate([p[4] for p in pieces])
            got_off = np.concatenate([p[5][:-1] + p[2] for p in pieces] + [[pieces[-1][3]]])
            ok = (np.array_equal(got_ids, want_ids) and np.array_equal(got_off, want_off)
                  and all(p[3] == int(want_off[-1]) for p in pieces) and pieces[0][2] == 0)
            ok = ok and (not few_records or any(p[0] == p[1] for p in pieces))
            q.put(bool(ok))
    finally:
        dist.destroy_process_group()


def _run_ranks(world, few_records):
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_rank_main, args=(r, world, port, q, few_records)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    assert q.get(timeout=10) is True


def test_two_ranks_gloo_stitch_equals_whole_buffer():
    _run_ranks(2, False)


def test_three_ranks_gloo_with_an_empty_range():
    _run_ranks(3, True)


def test_bench_gpus_flag_starts_that_many_ranks():
    """`bench.py --gpus 2` outside torchrun re-launches itself under torch.distributed.run; --dry-run-ranks joins the ranks on
    gloo and shows the record ranges (no GPU needed)."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--dry-run-ranks"], capture_output=True,
                         text=True, timeout=300, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    assert line["n_gpus"] == 2 and len(line["ranks"]) == 2 and line["ranks"][0]["records"][1] == line["ranks"][1]["records"][0]
