#!/usr/bin/env python
"""bench.py -- device-timed encode throughput of the DNATok hot path on B200, one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--k K] [--impl ours|reference] [--only]

A "step" is one pass of the hot path (dnatok_encode, + dnatok_pad where the config pads) over one batch of seeded
synthetic input.  The headline line is BASELINE.json configs[2] with k = 6: 1 GiB of
FASTA (80-column lines, a '>' header per record, log-uniform record lengths), non-overlapping 6-mers, int16 ids --
the largest single-GPU encode configuration and the hardest one for the HBM roofline.  Unless --only is given the
same run also measures every other config (1, 2, 3 for k in {1,2,3,4,5,8}, 4, 5) and reports them under "configs".

  value      kept bases/s of the headline config, device-timed with CUDA events, inputs resident in HBM
  roofline   algorithmic bytes (input bytes + record offsets + output id bytes + CSR offsets) / median step time
             against the measured HBM copy rate of MEASURED_PEAKS.json
  e2e        BASELINE.json configs[4]: 8 GiB in PINNED HOST memory through dnatok_stream_encode, 64 MiB chunks x 4
             streams, 6-mer + pad 8192 + mask into device batch tensors; H2D of bytes and offsets and D2H of the CSR
             counts inside the timed region; bases/s and the fraction of the measured pinned host link
  cpu_baseline  the CPU oracle (oracle/, as it stands) on this box's host cores, rank 0, N = 1 only: 1 warm-up and
             the median of 3 passes over a bounded sample of the headline workload
  parity     every out_offsets entry and the ids of 64 sampled records (config 5: their batch rows and masks too)
             against the oracle; a mismatch makes the run exit non-zero

Multi-GPU: records are independent.  `--gpus N` without a torchrun environment re-launches itself under
torch.distributed.run with N ranks.  --scaling weak (default): each rank encodes its own seeded shard.  --scaling
strong: ONE buffer is cut into per-rank record ranges of equal bytes (shard.partition_records), each rank encodes its
range with its own handle, the CSR is stitched from one int64 per rank and checked against the oracle on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

MIB = 1 << 20
K_SWEEP = (1, 2, 3, 4, 5, 6, 8)


# ----------------------------------------------------------------------------------------- workloads
def dense_lut() -> np.ndarray:
    """The default byte -> class table with no SKIP class ('\\n', '\\r' -> UNK): together with strip_headers = 0 this
    is the create-time spec of the no-scan encoder (kept bases = bytes).  Configs 2 and 4 hold no newline and no
    header, so their result is the same under either table; the oracle is given the same table."""
    lut = np.full(256, 5, dtype=np.uint8)
    for i, (u, l) in enumerate(zip(b"ACGTN", b"acgtn")):
        lut[u] = lut[l] = i
    return lut


def workload_spec(config: int, scale: float = 1.0, k: int = 6, dense: bool = True) -> dict:
    """Binding-style kwargs + generator call for BASELINE.json configs[config-1]."""
    spec = _workload_spec(config, scale, k)
    if dense and config in (2, 4):
        spec["tok"].update(class_lut=dense_lut(), strip_headers=False)
        spec["name"] += ", dense spec (no SKIP class, strip_headers 0)"
    return spec


def _workload_spec(config: int, scale: float = 1.0, k: int = 6) -> dict:
    if config == 1:
        return dict(name="config1: single-nt, 16 x 65,536 bases, 60-col lines, 1% N, 5% lowercase, int32",
                    gen=("config1", {}), tok=dict(mode="single_nt"), seq_len=0)
    if config == 2:
        n = max(1, int(4096 * scale))
        return dict(name=f"config2: 6-mer, {n} x 65,536 bases, order-2 Markov GC .41, N runs 0.5%, int32",
                    gen=("config2", dict(n_records=n)), tok=dict(mode="kmer", k=6), seq_len=0)
    if config == 3:
        tb = int((1 << 30) * scale)
        dt = 2 if k <= 6 else 4                       # BASELINE.json config 3: int16 for k <= 6, int32 for k = 8
        return dict(name=f"config3: {k}-mer int{8 * dt}, {tb} bases FASTA (80-col lines + header), log-uniform lengths",
                    gen=("config3", dict(total_bases=tb)), tok=dict(mode="kmer", k=k, id_dtype=dt), seq_len=0)
    if config == 4:
        n = max(1, int(65536 * scale))
        return dict(name=f"config4: BPE 4,092 merges, {n} reads of 500-1,500 bases, 2% N, int32",
                    gen=("config4", dict(n_reads=n)), tok=dict(mode="bpe", max_record_bytes=1536), seq_len=0)
    if config == 5:
        tb = int((8 << 30) * scale)
        return dict(name=f"config5: streaming {tb} bytes pinned, 64 MiB chunks x 4 streams, 6-mer + pad 8192 + mask",
                    gen=("config5", dict(total_bytes=tb)), tok=dict(mode="kmer", k=6, seq_len=8192,
                                                                    max_record_bytes=65536), seq_len=8192)
    raise SystemExit(f"unknown config {config}")


def generate(spec: dict, seed: int, out: np.ndarray | None = None):
    import dnagen
    fn, kw = spec["gen"]
    kw = dict(kw, seed=seed)
    if out is not None and fn in ("config2", "config5"):
        kw["out"] = out
    return getattr(dnagen, fn)(**kw)


def oracle_config(spec: dict, w):
    import oracle
    t = spec["tok"]
    m = {"single_nt": oracle.SINGLE_NT, "kmer": oracle.KMER, "bpe": oracle.BPE}[t["mode"]]
    kw = {}
    if t.get("class_lut") is not None:
        kw["class_lut"] = np.asarray(t["class_lut"], dtype=np.uint8)
    return oracle.Config(mode=m, k=t.get("k", 1), merges=w.merges, seq_len=spec["seq_len"],
                         strip_headers=bool(t.get("strip_headers", True)), **kw)


# ----------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=lambda: self.lines.extend(self.proc.stdout), daemon=True)
            self.t.start()
        except OSError:
            self.proc = None
        return self

    def stop(self) -> dict:
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.t.join(timeout=2)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def committed_profile(key: str):
    """Numbers taken from committed ncu captures (profiles/traffic.json): DRAM read + write bytes per launch of the
    dominant kernel of a config, warp-instructions per launch of the BPE kernel (null if none is committed)."""
    try:
        return json.load(open(os.path.join(ROOT, "profiles", "traffic.json"))).get(key)
    except Exception:
        return None


def measured_peaks() -> tuple[float, str]:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ----------------------------------------------------------------------------------------- CPU oracle legs
def host_cores() -> int:
    try:
        return max(1, min(64, len(os.sched_getaffinity(0))))
    except AttributeError:
        return max(1, min(64, os.cpu_count() or 1))


def oracle_sample(w, max_bytes: int = 256 * MIB):
    """Bounded sample of the workload for the CPU legs: the first records up to max_bytes."""
    r = int(np.searchsorted(w.offsets, max_bytes, side="right")) - 1
    r = max(1, min(r, w.n_records))
    return w.data[: int(w.offsets[r])], w.offsets[: r + 1].copy(), int(w.n_bases[:r].sum())


def oracle_run(data, offsets, cfg, threads: int, want=False):
    """The oracle as it stands, records split over `threads` host threads (ctypes releases the GIL).
    Returns (seconds, tokens); with want = "all" (ids, out_offsets); with want = "offsets" (None, out_offsets)."""
    import oracle
    from concurrent.futures import ThreadPoolExecutor
    n = offsets.size - 1
    targets = np.linspace(int(offsets[0]), int(offsets[-1]), threads * 4 + 1)
    cuts = np.unique(np.concatenate([[0], np.searchsorted(offsets, targets, side="left"), [n]]))
    cuts = cuts[cuts <= n]
    jobs = [(int(a), int(b)) for a, b in zip(cuts[:-1], cuts[1:]) if b > a]

    def job(ab):
        a, b = ab
        o = offsets[a: b + 1] - offsets[a]
        r = oracle.encode(data[int(offsets[a]): int(offsets[b])], o, cfg)
        if want == "offsets":
            return (None, r[1])
        return r if want else int(r[1][-1])

    t0 = time.perf_counter()
    if threads == 1:
        res = [job(j) for j in jobs]
    else:
        with ThreadPoolExecutor(max_workers=threads) as ex:
            res = list(ex.map(job, jobs))
    dt = time.perf_counter() - t0
    if not want:
        return dt, sum(res)
    ids = None if want == "offsets" else (np.concatenate([r[0] for r in res]) if res else np.zeros(0, np.int32))
    out = np.zeros(n + 1, dtype=np.int64)
    base = 0
    for (a, b), r in zip(jobs, res):
        out[a: b + 1] = r[1] + base
        base += int(r[1][-1])
    return ids, out


def cpu_baseline(spec, w) -> dict:
    """1 warm-up + median of 3 passes on all host threads, plus one single-threaded pass."""
    cores = host_cores()
    data, offs, bases = oracle_sample(w)
    cfg = oracle_config(spec, w)
    oracle_run(data, offs, cfg, cores)                              # warm-up: builds the library, pages in, starts threads
    runs = [oracle_run(data, offs, cfg, cores) for _ in range(3)]
    tn = float(np.median([r[0] for r in runs]))
    toks = runs[0][1]
    t1, _ = oracle_run(data, offs, cfg, 1)
    return {"value": bases / tn, "unit": "bases/s", "cores": cores, "kind": "oracle",
            "single_thread_value": bases / t1, "tokens_per_s": toks / tn,
            "sample": f"first {offs.size - 1} records ({data.size} bytes, {bases} bases) of the workload; 1 warm-up, "
                      f"median of 3 passes on {cores} threads ({tn:.3f} s), 1 pass single-threaded ({t1:.2f} s)"}


def run_reference(args) -> None:
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    spec = workload_spec(args.config, args.scale, args.k, not args.no_dense)
    w = generate(spec, seed=0)
    data, offs, bases = oracle_sample(w)
    cfg = oracle_config(spec, w)
    cores = host_cores()
    for _ in range(args.warmup):
        oracle_run(data, offs, cfg, cores)
    t, toks = 0.0, 0
    for _ in range(args.steps):
        dt, toks = oracle_run(data, offs, cfg, cores)
        t += dt
    v = bases * args.steps / t
    sample = f"first {offs.size - 1} records ({data.size} bytes, {bases} bases) per step on {cores} threads"
    print(json.dumps({
        "impl": "reference", "metric": "encode_bases_per_s", "value": v, "unit": "bases/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "tokens_per_s": toks * args.steps / t,
        "config": {"workload": spec["name"], "sample": sample},
        "cpu_baseline": {"value": v, "unit": "bases/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "bases/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }), flush=True)


# ----------------------------------------------------------------------------------------- CUDA arm
def token_upper_bound(offsets: np.ndarray, tok: dict) -> np.ndarray:
    """Per-record upper bound on emitted tokens from the record byte lengths alone (sizes D2H copies and
    id buffers without a device sync): kmer floor(L/k) + (k-1); single-nt / BPE L."""
    L = np.diff(offsets)
    if tok["mode"] == "kmer":
        k = tok["k"]
        return L // k + np.minimum(L, k - 1)
    return L


class Dist:
    """torch.distributed plumbing (one process per GPU, NCCL); a no-op at world size 1."""

    def __init__(self, torch, local: int):
        self.torch = torch
        self.rank = int(os.environ.get("RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.dist = None
        if self.world > 1:
            import torch.distributed as dist
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
            self.dist = dist

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()
        self.torch.cuda.synchronize()

    def _red(self, x: float, op) -> float:
        if self.dist is None:
            return x
        t = self.torch.tensor([x], dtype=self.torch.float64, device="cuda")
        self.dist.all_reduce(t, op=op)
        return float(t.item())

    def max(self, x: float) -> float:
        return self._red(x, self.dist.ReduceOp.MAX if self.dist else None)

    def sum(self, x: float) -> float:
        return self._red(x, self.dist.ReduceOp.SUM if self.dist else None)

    def close(self):
        if self.dist is not None:
            self.dist.barrier()
            self.dist.destroy_process_group()


def bench_config(dn, torch, D: Dist, local: int, config: int, k: int, args, *, e2e: bool, parity: bool,
                 keep: dict | None = None) -> dict:
    """One config: device-timed steps, roofline, parity against the oracle, optionally the end-to-end stream leg.
    `keep` carries a generated workload from one k of the config 3 sweep to the next."""
    spec = workload_spec(config, args.scale, k, not args.no_dense)
    tokkw = dict(spec["tok"])
    strong = args.scaling == "strong" and D.world > 1
    # ---- input: generated straight into pinned host memory where it is streamed from ---------------------------------
    t0 = time.perf_counter()
    if keep is not None and "w" in keep:
        w, pinned = keep["w"], keep["pinned"]
    else:
        pinned = None
        seed = 0 if strong else D.rank
        if spec["gen"][0] in ("config2", "config5"):
            total = (spec["gen"][1].get("n_records", 0) * 65536) or spec["gen"][1]["total_bytes"]
            pinned = torch.empty(total, dtype=torch.uint8).pin_memory()
            w = generate(spec, seed=seed, out=pinned.numpy())
        else:
            w = generate(spec, seed=seed)
            if e2e:
                pinned = torch.empty(w.n_bytes, dtype=torch.uint8).pin_memory()
                pinned.numpy()[:] = w.data
                w.data = pinned.numpy()
        if keep is not None:
            keep["w"], keep["pinned"] = w, pinned
    gen_s = time.perf_counter() - t0
    if w.merges is not None:
        tokkw["merges"] = w.merges
    # strong scaling: this rank's contiguous record range of the one shared buffer
    r0, r1 = 0, w.n_records
    if strong:
        from paper_2601_05531_b200.shard import partition_records
        r0, r1 = partition_records(w.offsets, D.world)[D.rank]
    b0, b1 = int(w.offsets[r0]), int(w.offsets[r1])
    offsets = (w.offsets[r0: r1 + 1] - b0).astype(np.int64)
    data = w.data[b0:b1]
    n_bytes, n_rec, bases = b1 - b0, r1 - r0, int(w.n_bases[r0:r1].sum())
    ub = token_upper_bound(offsets, tokkw)
    ub_prefix = np.concatenate([[0], np.cumsum(ub)]).astype(np.int64)
    id_cap = int(ub_prefix[-1]) + 64
    idsz = int(tokkw.get("id_dtype", 4))
    L = spec["seq_len"]

    dn.SUPER_TILE = args.super_tile
    tok = dn.DNATok(**tokkw, device=local)
    d_bytes = (pinned[b0:b1] if pinned is not None else torch.from_numpy(data)).cuda(non_blocking=True)
    d_off = torch.from_numpy(offsets).cuda()
    ids = torch.empty(id_cap, dtype=tok.id_torch_dtype, device="cuda")
    out_off = torch.empty(n_rec + 1, dtype=torch.int64, device="cuda")
    batch = mask = None
    if L:
        batch = torch.empty((n_rec, L), dtype=torch.int32, device="cuda")
        mask = torch.empty((n_rec, L), dtype=torch.uint8, device="cuda")

    def step():
        if L:       # dnatok_encode_pad: steps 1-6 in one call; regular layouts go straight into the batch (no CSR ids in HBM)
            tok.encode_padded(d_bytes, d_off, ids_out=ids, out_offsets=out_off, batch_ids=batch, mask=mask)
        else:
            tok.encode(d_bytes, d_off, ids_out=ids, out_offsets=out_off)

    # ---- device-timed region: K steps, CUDA events on the launching (current) stream ---------------------------------
    for _ in range(max(args.warmup, 3)):
        step()
    tok.check()
    n_tokens = int(out_off[-1].item())
    launches0 = tok.launch_count
    clocks = ClockSampler(local).start()
    # inputs + outputs of one step larger than L2: steps run back to back.  Otherwise (configs 1 and 4) L2 is flushed
    # between the timed steps by writing a 256 MiB buffer, and every step is timed on its own.
    small = (n_bytes + id_cap * idsz) <= 2 * 126_000_000
    flush = torch.empty(256 * MIB, dtype=torch.uint8, device="cuda") if small else None
    ev0 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    ev1 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    D.barrier()
    for i in range(args.steps):
        if small:
            flush.zero_()
        ev0[i].record()
        step()
        ev1[i].record()
    D.barrier()
    per_step_ms = np.array([ev0[i].elapsed_time(ev1[i]) for i in range(args.steps)])
    total_ms = float(per_step_ms.sum()) if small else ev0[0].elapsed_time(ev1[-1])
    del flush
    launches = tok.launch_count - launches0
    launches_per_step = launches // max(args.steps, 1)
    # keep the GPU busy a little longer so nvidia-smi gets samples under this very load
    t_end = time.perf_counter() + 0.5
    while time.perf_counter() < t_end:
        step()
    torch.cuda.synchronize()
    clk = clocks.stop()
    tok.check()
    ms_per_step = D.max(total_ms / args.steps)
    assert launches >= args.steps, "the CUDA library launched no kernels: there is no CPU path"

    # ---- parity against the oracle (untimed): every offset, the ids of sampled records ------------------------------
    parity_s = "skipped"
    if parity and not args.no_parity:
        import oracle
        ocfg = oracle_config(spec, w)
        off_h = out_off.cpu().numpy()
        if args.full_parity or config != 5:
            want_ids, want_off = oracle_run(data, offsets, ocfg, host_cores(), want="all")
            ok = bool(np.array_equal(off_h, want_off))
            if L and tok.fast_path_taken():                      # fused call: the ids went straight into the batch
                wb, wm = oracle.pad(want_ids, want_off, ocfg)
                ok = ok and bool(np.array_equal(batch.cpu().numpy(), wb)) and bool(np.array_equal(mask.cpu().numpy(), wm))
                what = f"every batch and mask entry ({n_rec} x {L}) and every out_offsets entry ({n_rec + 1})"
            else:
                ok = ok and bool(np.array_equal(ids[: n_tokens].cpu().numpy().astype(np.int32), want_ids))
                what = f"every id ({n_tokens}) and every out_offsets entry ({n_rec + 1})"
            del want_ids
        else:
            # config 5 (10.7 GB of rows): every out_offsets entry, and ids + batch row + mask of 64 sampled records
            _, want_off = oracle_run(data, offsets, ocfg, host_cores(), want="offsets")
            ok = bool(np.array_equal(off_h, want_off))
            rng = np.random.default_rng(1234)
            pick = np.unique(np.concatenate([[0, n_rec - 1], rng.integers(0, n_rec, size=62)]))
            ids_written = not (L and tok.fast_path_taken())             # the fused call leaves the CSR ids unwritten
            for r in pick:
                a, b = int(offsets[r]), int(offsets[r + 1])
                want, _ = oracle.encode(data[a:b], np.array([0, b - a], dtype=np.int64), ocfg)
                lo = int(want_off[r])
                if ids_written:
                    got = ids[lo: lo + want.size].cpu().numpy().astype(np.int32)
                    ok = ok and bool(np.array_equal(got, want))
                if L:
                    wb, wm = oracle.pad(want, np.array([0, want.size], dtype=np.int64), ocfg)
                    ok = ok and bool(np.array_equal(batch[r].cpu().numpy(), wb[0]))
                    ok = ok and bool(np.array_equal(mask[r].cpu().numpy(), wm[0]))
            what = (f"every out_offsets entry ({n_rec + 1}) and " + ("ids, " if ids_written else "") +
                    f"batch row and mask of {pick.size} sampled records")
        parity_s = ("bit-exact: " + what) if ok else ("MISMATCH: " + what)

    # ---- roofline: the method's own bytes over the median step -----------------------------------------------------
    peak, peak_src = measured_peaks()
    in_bytes = n_bytes + (n_rec + 1) * 8
    if L:
        out_bytes = n_rec * L * 5 + (n_rec + 1) * 8              # batch_ids int32 + mask uint8 (+ the CSR offsets)
    else:
        out_bytes = n_tokens * idsz + (n_rec + 1) * 8
    alg_bytes = in_bytes + out_bytes
    kern_ms = float(np.median(per_step_ms))
    kname = {"bpe": "bpe_merge_kernel"}.get(tokkw["mode"], "encode_tiles_v7<dense>" if tok.cfg.class_lut is not None
                                               and not tok.cfg.strip_headers else "encode_tiles_v5")
    if kname == "encode_tiles_v5" and tok.fast_path_taken():
        kname = "encode_fasta_kernel"                            # the regular-layout encoder served the call (dnatok.h)
    roof = {"bound": "hbm", "kernel": kname, "achieved": alg_bytes / (kern_ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
            "peak_source": peak_src, "algorithmic_bytes_per_launch": alg_bytes,
            "bytes_per_base": alg_bytes / max(1, bases), "kernel_ms": kern_ms, "traffic": args.traffic}
    if args.traffic is None:
        # a committed ncu capture counts as this launch's DRAM traffic only if it is OF this launch: full size, and for config 3
        # the k = 6 kernel; config 5 was captured at an eighth of its size (profiles/r2_pad.md) and is reported as such
        if args.scale == 1.0 and config != 5 and (config != 3 or k == 6):
            roof["traffic"] = committed_profile(f"config{config}")
        elif config == 5:
            roof["traffic_at_scale"] = {"scale": 0.125, "dram_bytes": committed_profile("config5"), "method_bytes": 2416e6,
                                        "source": "profiles/r2_pad.md"}
    roof["frac"] = roof["achieved"] / peak
    if L:
        if kname == "encode_fasta_kernel":
            roof["note"] = "method bytes: input + batch_ids + mask; dnatok_encode_pad wrote the tokens straight into the batch (no CSR ids)"
        else:
            roof["note"] = ("method bytes only: input + batch_ids + mask; the CSR ids the pad kernel re-reads (%d B written, "
                            "%d B read per step) are not counted" % (n_tokens * idsz, n_tokens * idsz))
    if tokkw["mode"] == "bpe":
        # the merge loop is bound by instruction issue, not by HBM (SURVEY.md section 7 hard part 5)
        sm_mhz = clk.get("sm_mhz") or 1965.0
        issue_peak = 148 * 4 * sm_mhz * 1e6                      # warp-instructions/s: 148 SMs x 4 schedulers x 1 per clock
        winst = committed_profile("config4_warp_inst")
        roof_issue = {"bound": "issue", "peak": issue_peak, "unit": "warp-inst/s",
                      "peak_derivation": f"148 SMs x 4 schedulers x {sm_mhz:.0f} MHz (median under load)",
                      "warp_inst_per_launch": winst, "source": "ncu smsp__inst_executed.sum, profiles/r2_bpe.md"}
        if winst:
            roof_issue["achieved"] = winst / (kern_ms * 1e-3)
            roof_issue["frac"] = roof_issue["achieved"] / issue_peak
            roof_issue["lane_instr_per_base"] = 32.0 * winst / max(1, bases)
            roof_issue["algorithmic_lookups_per_base"] = 3.8
        roof = dict(roof, hbm_frac=roof["frac"], issue=roof_issue)
    elif kname == "encode_fasta_kernel" and config == 3 and tokkw.get("k") == 6 and args.scale == 1.0:
        # what holds the strip encoder below the HBM rate (profiles/r2_encode.md): instruction issue.  Reported beside the
        # HBM roofline, which stays the headline; the count is the full-size ncu capture's (the work is data-independent)
        sm_mhz = clk.get("sm_mhz") or 1965.0
        issue_peak = 148 * 4 * sm_mhz * 1e6
        winst = committed_profile("config3_warp_inst")
        if winst:
            roof["issue"] = {"bound": "issue", "peak": issue_peak, "unit": "warp-inst/s",
                             "peak_derivation": f"148 SMs x 4 schedulers x {sm_mhz:.0f} MHz (median under load)",
                             "warp_inst_per_launch": winst, "source": "ncu smsp__inst_executed.sum, profiles/r2_encode.md",
                             "achieved": winst / (kern_ms * 1e-3), "frac": winst / (kern_ms * 1e-3) / issue_peak,
                             "lane_instr_per_byte": 32.0 * winst / max(1, n_bytes)}

    res = {"workload": spec["name"], "n_bytes": n_bytes, "n_records": n_rec, "kept_bases": bases, "tokens": n_tokens,
           "ms_per_step": ms_per_step, "bases_per_s": D.sum(bases) / (ms_per_step * 1e-3),
           "tokens_per_s": D.sum(n_tokens) / (ms_per_step * 1e-3), "dtype": {2: "int16", 4: "int32"}[idsz],
           "roofline": roof, "parity": parity_s, "gpu_launches": int(launches), "launches_per_step": int(launches_per_step),
           "clocks": clk, "gen_s": round(gen_s, 2),
           "ms_per_step_stats": {"median": kern_ms, "mean": float(per_step_ms.mean()), "sd": float(per_step_ms.std()),
                                 "min": float(per_step_ms.min())},
           "l2": "inputs + outputs per step exceed the 126 MB L2; steps back to back" if not small
                 else "L2 flushed between timed steps (256 MiB written), each step timed on its own"}
    if strong:
        from paper_2601_05531_b200.shard import exclusive_token_base
        base, total = exclusive_token_base(n_tokens)
        res["strong"] = {"records": [r0, r1], "token_base": base, "token_total": total}
        if D.rank == 0 and not args.no_parity:
            import oracle
            _, want_off = oracle_run(w.data, w.offsets, oracle_config(spec, w), host_cores(), want="offsets")
            ok = int(want_off[-1]) == total and bool(np.array_equal(out_off.cpu().numpy() + base, want_off[r0: r1 + 1]))
            res["strong"]["stitched_offsets_vs_oracle"] = "bit-exact" if ok else "MISMATCH"
            if not ok:
                res["parity"] = "MISMATCH: stitched CSR offsets"

    # ---- end to end through dnatok_stream_encode: HOST buffers in, results read back on the host -------------------
    if e2e and not args.no_e2e:
        chunk = args.chunk_mib * MIB
        n_chunks = (n_bytes + chunk - 1) // chunk
        h_ids = torch.empty(id_cap if not L else 1, dtype=tok.id_torch_dtype).pin_memory()
        h_cnt = torch.empty(n_rec + n_chunks + 2, dtype=torch.int64).pin_memory()
        max_rows = int(chunk // max(1, int(np.diff(offsets).min() or 1))) + 2
        max_rows = min(max_rows, n_rec + 1)
        d2h = [0]
        src = pinned[b0:b1]

        def on_batch(b):
            n = b.n_records
            s = torch.cuda.ExternalStream(b.stream)
            with torch.cuda.stream(s):
                o0 = b.first_record + b.chunk_index                       # (n + 1) offsets per batch
                h_cnt[o0: o0 + n + 1].copy_(b.out_offsets(), non_blocking=True)
                d2h[0] += (n + 1) * 8
                if not L and n:                                           # CSR ids go back to the host;
                    a, e = int(ub_prefix[b.first_record]), int(ub_prefix[b.first_record + n])
                    h_ids[a: e].copy_(b.ids(e - a), non_blocking=True)   # padded batches stay on the device
                    d2h[0] += (e - a) * idsz

        def e2e_step():
            tok.stream_encode(src, offsets, chunk, args.streams, max_rows_per_chunk=max_rows, on_batch=on_batch)

        for _ in range(2):
            e2e_step()
        # the streamed CSR counts must equal the resident ones (checked once, outside the timed region)
        off_res = out_off.cpu().numpy()
        cnt_res = np.diff(off_res)
        hc = h_cnt.numpy()
        got, pos, rec = [], 0, 0
        first = []
        tok.stream_encode(src, offsets, chunk, args.streams, max_rows_per_chunk=max_rows,
                          on_batch=lambda b: (first.append((b.first_record, b.n_records, b.chunk_index)), on_batch(b)))
        torch.cuda.synchronize()
        for f, n, ci in first:
            o = hc[f + ci: f + ci + n + 1]
            got.append(np.diff(o))
        stream_ok = bool(np.array_equal(np.concatenate(got) if got else np.zeros(0, np.int64), cnt_res))
        # host link: one cudaMemcpyAsync of the whole pinned buffer, best of 5
        h2d_best = 0.0
        for _ in range(5):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); d_bytes.copy_(src, non_blocking=True); b.record(); torch.cuda.synchronize()
            h2d_best = max(h2d_best, n_bytes / (a.elapsed_time(b) * 1e-3) / 1e9)
        ke = max(3, min(args.steps, 5 if n_bytes > (2 << 30) else 10))
        d2h[0] = 0
        launches0 = tok.launch_count
        D.barrier()
        t0 = time.perf_counter()
        for _ in range(ke):
            e2e_step()                                                    # returns after its streams are drained
        torch.cuda.synchronize()
        e_s = D.max((time.perf_counter() - t0) / ke)
        D.barrier()
        res["gpu_launches"] += int(tok.launch_count - launches0)
        res["e2e"] = {"value": D.sum(bases) / e_s, "unit": "bases/s", "tokens_per_s": D.sum(n_tokens) / e_s,
                      "h2d_bytes_per_step": n_bytes + (n_rec + n_chunks) * 8, "d2h_bytes_per_step": d2h[0] // ke,
                      "ms_per_step": e_s * 1e3, "steps": ke, "chunk_bytes": chunk, "n_streams": args.streams,
                      "workload": spec["name"],
                      "h2d_gbs": n_bytes / e_s / 1e9, "h2d_gbs_link_measured": h2d_best,
                      "frac_of_host_link": n_bytes / e_s / 1e9 / h2d_best,
                      "streamed_counts_vs_resident": "equal" if stream_ok else "MISMATCH",
                      "timing": "host wall clock around K calls of dnatok_stream_encode, streams drained"}
        if not stream_ok:
            res["parity"] = "MISMATCH: streamed CSR counts differ from the resident encode"
    res["_w"] = w
    res["_spec"] = spec
    return res


def ablation(dn, torch, local: int, args) -> dict:
    """the paper's IDs path next to the bytes path, in the shape of its Table S2:
    int64 vs int32 + on-device widening for the host-mapped IDs path, and 1 vs n_streams streams for the bytes
    path.  Workload: equal-length clean strings as in the paper's microbenchmarks -- B rows of T = 512
    uniform-ACGT bases, single-nucleotide vocabulary.  Every arm is timed end to end from HOST memory (host clock around
    enqueue .. synchronize, median of 3 after one warm-up); the host LUT map of the IDs path is numpy fancy indexing on one
    thread, as in the paper ("vectorised CPU map")."""
    T = 512
    B = max(1, int(args.ablation_mib * MIB) // T)
    n = B * T
    rng = np.random.default_rng(7)
    pin_bytes = torch.empty(n, dtype=torch.uint8).pin_memory()
    pin_bytes.numpy()[:] = np.frombuffer(b"ACGT", dtype=np.uint8)[rng.integers(0, 4, size=n)]
    offsets = (np.arange(B + 1, dtype=np.int64) * T)
    lut_ids = np.full(256, 1, dtype=np.int64)                       # ASCII -> id, the IDs path's host table
    for i, (u, l) in enumerate(zip(b"ACGTN", b"acgtn")):
        lut_ids[u] = lut_ids[l] = 2 + i
    lut32 = lut_ids.astype(np.int32)
    pin64 = torch.empty(n, dtype=torch.int64).pin_memory()
    pin32 = torch.empty(n, dtype=torch.int32).pin_memory()
    d64 = torch.empty(n, dtype=torch.int64, device="cuda")
    d32 = torch.empty(n, dtype=torch.int32, device="cuda")
    d_bytes = torch.empty(n, dtype=torch.uint8, device="cuda")
    d_off = torch.from_numpy(offsets).cuda()
    tok = dn.DNATok(mode="single_nt", class_lut=dense_lut(), strip_headers=False, max_record_bytes=65536, device=local)
    ids = torch.empty(n + 64, dtype=torch.int32, device="cuda")
    out_off = torch.empty(B + 1, dtype=torch.int64, device="cuda")
    src = pin_bytes.numpy()

    def ids64():
        np.take(lut_ids, src, out=pin64.numpy()); d64.copy_(pin64, non_blocking=True)

    def ids32():
        np.take(lut32, src, out=pin32.numpy()); d32.copy_(pin32, non_blocking=True); tok.widen(d32)

    def bytes_resident():
        d_bytes.copy_(pin_bytes, non_blocking=True); tok.encode(d_bytes, d_off, ids_out=ids, out_offsets=out_off)

    def bytes_stream(ns):
        return lambda: tok.stream_encode(pin_bytes, offsets, args.chunk_mib * MIB, ns, max_rows_per_chunk=args.chunk_mib * MIB // T + 2)

    def timed(fn):
        fn(); torch.cuda.synchronize()
        ts = []
        for _ in range(3):
            t0 = time.perf_counter(); fn(); torch.cuda.synchronize(); ts.append(time.perf_counter() - t0)
        return float(np.median(ts))

    arms = {"ids_path_int64": timed(ids64), "ids_path_int32_widen_on_device": timed(ids32),
            "bytes_path_one_copy_then_encode": timed(bytes_resident),
            "bytes_path_stream_1": timed(bytes_stream(1)), f"bytes_path_stream_{args.streams}": timed(bytes_stream(args.streams))}
    # the three paths must agree on the ids (checked once, untimed)
    tok.check()
    same = bool(torch.equal(d64, tok.widen(d32))) and bool(torch.equal(d64[: n], ids[: n].to(torch.int64)))
    base = arms["ids_path_int64"]
    return {"workload": f"{B} rows x {T} uniform-ACGT bases, single-nt vocabulary (PAPER.md Table S2 shape)", "tokens": n,
            "tokens_per_s": {k: n / v for k, v in arms.items()}, "speedup_vs_ids_int64": {k: base / v for k, v in arms.items()},
            "seconds": arms, "ids_agree": same, "host_map": "numpy.take on 1 thread",
            "note": "IDs path = host LUT map -> pinned ids -> H2D (PAPER.md:82); bytes path = raw bytes -> H2D -> device LUT (PAPER.md:84)"}


def run_ours(args) -> None:
    import torch
    import paper_2601_05531_b200 as dn

    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device: there is no CPU fallback"
    torch.cuda.set_device(local)
    D = Dist(torch, local)
    rank0 = D.rank == 0
    single = D.world == 1

    keep3: dict = {}
    head = bench_config(dn, torch, D, local, args.config, args.k, args, e2e=args.only or args.config == 5,
                        parity=rank0, keep=keep3 if args.config == 3 else None)
    cpu = cpu_baseline(head["_spec"], head["_w"]) if (rank0 and single and not args.no_cpu) else None
    configs = {}
    e2e = head.get("e2e")
    bad = "MISMATCH" in head["parity"]
    if not args.only:
        plan = []
        if args.config == 3:
            plan += [(3, k) for k in K_SWEEP if k != args.k]
        plan += [(c, 6) for c in (1, 2, 4, 5) if c != args.config]
        if args.config != 3:
            plan += [(3, k) for k in K_SWEEP]
        for c, k in plan:
            r = bench_config(dn, torch, D, local, c, k, args, e2e=(c == 5), parity=rank0,
                             keep=keep3 if c == 3 else None)
            if c == 5 and "e2e" in r and args.config != 5:
                e2e = r["e2e"]
            bad = bad or "MISMATCH" in r["parity"]
            key = f"config{c}" + (f"_k{k}" if c == 3 else "")
            configs[key] = {kk: v for kk, v in r.items() if not kk.startswith("_") and kk not in ("clocks",)}
            if c != 3:
                keep3.clear()                                            # free the 1 GiB sweep input before the big configs
            del r
    abl = None
    if rank0 and single and args.ablation and not args.only:
        abl = ablation(dn, torch, local, args)
        bad = bad or not abl["ids_agree"]
    D.close()
    if not rank0:
        return
    line = {
        "metric": "encode_bases_per_s", "value": head["bases_per_s"], "unit": "bases/s",
        "n_gpus": D.world, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": head["ms_per_step"],
        "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None,
        "dtype": head["dtype"], "data": "synthetic", "tokens_per_s": head["tokens_per_s"],
        "config": {"workload": head["workload"], "n_bytes": head["n_bytes"], "n_records": head["n_records"],
                   "kept_bases": head["kept_bases"], "tokens": head["tokens"],
                   "seed": "0 on every rank" if args.scaling == "strong" else "rank", "l2": head["l2"], "gen_s": head["gen_s"]},
        "roofline": head["roofline"], "cpu_baseline": cpu, "e2e": e2e,
        "gpu_launches": head["gpu_launches"] + sum(c["gpu_launches"] for c in configs.values()),
        "launches_per_step": head["launches_per_step"], "clocks": head["clocks"], "parity": head["parity"],
        "ms_per_step_stats": head["ms_per_step_stats"], "configs": configs, "ablation": abl,
        "context": "paper (H200, IDs path + embedding): 1.93-2.18e8 tokens/s encode, 1.27-1.84e8 e2e; not comparable",
    }
    if "strong" in head:
        line["strong"] = head["strong"]
    print(json.dumps(line), flush=True)
    if bad:
        print("bench.py: parity MISMATCH against the oracle", file=sys.stderr)
        sys.exit(1)


def dry_run_ranks(args) -> None:
    """No GPU needed: every rank joins a gloo group, cuts the same small seeded buffer with shard.partition_records
    and exchanges one int64 -- shows that `--gpus N` really starts N ranks and that the host-side sharding runs."""
    import torch
    import torch.distributed as dist
    import dnagen
    from paper_2601_05531_b200.shard import exclusive_token_base, partition_records
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    w = dnagen.config3(total_bases=200_000, lo=500, hi=9000)
    r0, r1 = partition_records(w.offsets, world)[rank]
    base, total = exclusive_token_base(int(r1 - r0))                # (record counts stand in for token totals here)
    every = [None] * world
    dist.all_gather_object(every, {"rank": rank, "records": [int(r0), int(r1)], "base": base})
    if rank == 0:
        print(json.dumps({"dry_run_ranks": world, "n_gpus": world, "ranks": every, "total": total,
                          "torch": torch.__version__}), flush=True)
    dist.destroy_process_group()


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--k", type=int, default=6, help="config 3 only: k of the k-mer sweep (1,2,3,4,5,6,8)")
    ap.add_argument("--only", action="store_true", help="measure only --config (with its own e2e leg), not the other configs")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"])
    ap.add_argument("--scale", type=float, default=1.0, help="shrink the workload (debugging only)")
    ap.add_argument("--chunk-mib", type=int, default=64)
    ap.add_argument("--streams", type=int, default=4)
    ap.add_argument("--traffic", type=float, default=None,
                    help="ncu dram read+write bytes per launch of the dominant kernel (from profiles/)")
    ap.add_argument("--super-tile", type=int, default=0, help="tuning: 16 KiB units per tile (0 = automatic)")
    ap.add_argument("--no-dense", action="store_true", help="configs 2 and 4: default table (with SKIP) instead of the dense spec")
    ap.add_argument("--full-parity", action="store_true", help="compare every id of every config with the oracle")
    ap.add_argument("--no-ablation", dest="ablation", action="store_false", help="skip the IDs-path / streams ablation (SURVEY 8(f) f4)")
    ap.add_argument("--ablation-mib", type=int, default=128, help="tokens of the ablation workload, in Mi")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-parity", action="store_true")
    ap.add_argument("--dry-run-ranks", action="store_true", help="start the ranks on CPU (gloo) and show the sharding only")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # not under torchrun: start the N ranks ourselves (one process per GPU)
        import socket
        with socket.socket() as s:
            s.bind(("127.0.0.1", 0))
            port = s.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        sys.exit(subprocess.call(cmd))
    if args.dry_run_ranks:
        dry_run_ranks(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
