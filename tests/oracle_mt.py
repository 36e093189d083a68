"""Test helper: the CPU oracle run over record ranges on several host threads (ctypes releases the GIL) and
stitched back into one CSR result.  Records are independent, so this is the oracle's own
result, only faster to obtain at the full BASELINE.json sizes.  Calls nothing but `oracle/`."""
from __future__ import annotations

import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np

import oracle


def host_threads() -> int:
    try:
        return max(1, min(32, len(os.sched_getaffinity(0))))
    except AttributeError:
        return max(1, min(32, os.cpu_count() or 1))


def encode_mt(data: np.ndarray, offsets: np.ndarray, cfg: "oracle.Config", threads: int | None = None):
    """oracle.encode on contiguous record ranges of about equal byte count -> (ids int32, out_offsets int64)."""
    threads = threads or host_threads()
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    n = offsets.size - 1
    if n <= 1 or threads == 1:
        return oracle.encode(data, offsets, cfg)
    targets = np.linspace(int(offsets[0]), int(offsets[-1]), threads * 4 + 1)
    cuts = np.unique(np.concatenate([[0], np.searchsorted(offsets, targets, side="left"), [n]]))
    cuts = cuts[cuts <= n]
    jobs = [(int(a), int(b)) for a, b in zip(cuts[:-1], cuts[1:]) if b > a]

    def job(ab):
        a, b = ab
        lo, hi = int(offsets[a]), int(offsets[b])
        return oracle.encode(data[lo:hi], offsets[a:b + 1] - lo, cfg)

    with ThreadPoolExecutor(max_workers=threads) as ex:
        parts = list(ex.map(job, jobs))
    ids = np.concatenate([p[0] for p in parts]) if parts else np.zeros(0, np.int32)
    out = np.zeros(n + 1, dtype=np.int64)
    base = 0
    for (a, b), (pi, po) in zip(jobs, parts):
        out[a:b + 1] = po + base
        base += int(po[-1])
    return ids, out
