#!/usr/bin/env python
"""bench.py -- one JSON line per run (the driver's contract).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2|3|4|5|churn|d2] [--k 4|8|16]
                    [--impl reference]

A step = one pass of the hot path over one batch of synthetic input:
  configs 2/3/5  one spork_decode_attn call (plan lookup, cascade decode kernel, merge kernel)
  config 4       one spork_verify_attn call with k drafts per sequence
  churn          one spork_fork of 10,000 children + one spork_release of them (config 5)
  d2             one spork_confidence call: Eq. 2 over 256 probe spans of Qwen3-vocabulary logits
Default workload: BASELINE.json configs[1] (Qwen3-4B shape, 16 fork groups of 2, prefix 4096).
Inputs are seeded synthetic (synth/), resident in HBM before the timed region; L2 is flushed
between timed iterations.  `value` = unique KV bytes / step time (GB/s); config 4 also reports
TFLOP/s.  N > 1 (torchrun) runs N independent replicas: the path does not shard ("replicas only").
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

import synth  # noqa: E402

METRIC = "forked_decode_attn_unique_kv_bandwidth"
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        d["_source"] = "measured"
        return d
    d = dict(FALLBACK_PEAKS)
    d["_source"] = "fallback"
    return d


# ---------------------------------------------------------------------------
# clocks sampler (nvidia-smi during the timed region)
# ---------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(max(mx)) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------
# workloads
# ---------------------------------------------------------------------------
def pick_config(args):
    if args.config == "churn":
        return synth.CFG5, "cfg5_fork_churn"
    n = int(args.config)
    cfg = synth.CONFIGS[n]
    if n == 4:
        cfg = cfg.scaled(k_draft=args.k)
        return cfg, f"cfg4_qwen3_32b_verify_k{args.k}"
    return cfg, cfg.name


def pool_dims(wl, num_pages=None):
    c = wl.cfg
    per_seq = int((wl.total_len.max() + 15) // 16) + 4
    need = int(c.n_groups * ((c.prefix_len + 15) // 16) + sum((int(x) + 15) // 16 + 1 for x in wl.private_len))
    return (num_pages or need + 1024), per_seq


def build_spork(cfg, wl, num_pages=None, max_seqs=None, device="cuda:0"):
    import paper_2607_03333_b200 as sp
    npg, mp = pool_dims(wl, num_pages)
    spk = sp.Spork(cfg.dtype, cfg.Hq, cfg.Hkv, cfg.D, npg, max_seqs or cfg.n_seqs + 8, mp, cfg.scale,
                   device=device)
    ids = synth.build_state(spk, wl)
    spk.synchronize()
    return spk, ids


# ---------------------------------------------------------------------------
# the oracle leg (cpu_baseline and --impl reference): a bounded sample of the same workload
# ---------------------------------------------------------------------------
def oracle_sample(cfg, wl, max_groups=2):
    """Builds `max_groups` fork groups of the workload in the CPU oracle and returns a closure that
    runs one oracle step on them, plus the factor that scales its time to the whole batch."""
    import oracle
    g = min(cfg.n_groups, max_groups)
    sub = cfg.scaled(n_groups=g)
    # same sub-streams as the full workload: groups / sequences [0, g) are identical
    swl = synth.Workload(sub, wl.k[:sub.n_seqs] if cfg.k_draft else None)
    swl.suffix_len = wl.suffix_len[:sub.n_seqs].copy()
    swl.private_len = wl.private_len[:sub.n_seqs].copy()
    swl.total_len = wl.total_len[:sub.n_seqs].copy()
    npg, mp = pool_dims(swl)
    orc = oracle.Oracle(sub.dtype, sub.Hq, sub.Hkv, sub.D, npg, sub.n_seqs + 2, mp, sub.scale)
    ids = synth.build_state(orc, swl)
    q = swl.q_all()
    qi = swl.q_indptr()
    frac = float(swl.flops() / wl.flops())

    def step():
        if cfg.k_draft:
            return orc.verify(ids, qi, q)
        return orc.decode(ids, q)

    return step, frac, oracle.num_threads(), f"{g} of {cfg.n_groups} fork groups ({sub.n_seqs} sequences), all heads"


def run_reference(args, cfg, name, wl):
    step, frac, cores, sample = oracle_sample(cfg, wl, args.ref_groups)
    for _ in range(max(0, min(args.warmup, 1))):
        step()
    steps = min(args.steps, 20)            # a CPU step takes 0.05 .. 20 s: keep the run bounded
    t0 = time.perf_counter()
    for _ in range(steps):
        step()
    dt = (time.perf_counter() - t0) / steps
    full = dt / frac                       # time one whole step would take, scaled by flops
    ub = wl.unique_kv_bytes()
    val = ub / full / 1e9
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": "GB/s", "n_gpus": args.gpus,
        "steps": steps, "warmup": args.warmup, "ms_per_step": full * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": cfg.dtype, "data": "synthetic",
        "config": {"workload": name, "sample": sample, "sample_seconds_per_step": dt},
        "cpu_baseline": {"value": val, "unit": "GB/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def _traffic(workload: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of the workload's dominant kernel, from
    the committed ncu capture (profiles/traffic.json); None if there is none."""
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        with open(tpath) as f:
            return json.load(f).get(workload)
    return None


def max_over_ranks(x: float, device, world: int) -> float:
    """Replicas only: the step time of an N-replica run is the slowest rank's."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(unique_bytes: int, ms_step: float, world: int) -> float:
    """Whole-job GB/s of `world` independent replicas that each moved `unique_bytes` in `ms_step`."""
    return world * unique_bytes / (ms_step * 1e-3) / 1e9


# ---------------------------------------------------------------------------
# the CUDA arm
# ---------------------------------------------------------------------------
def run_ours(args, cfg, name, wl):
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    device = f"cuda:{local}"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(device))
    peaks = load_peaks()

    churn = args.config == "churn"
    num_pages = (1 << 20) if (churn or (args.config == "5" and args.full_pool)) else None
    max_seqs = cfg.n_seqs + 10008 if churn else None
    t_build = time.perf_counter()
    spk, ids = build_spork(cfg, wl, num_pages, max_seqs, device)
    t_build = time.perf_counter() - t_build
    if args.min_rows is not None:
        spk.set_tensor_path_min_rows(args.min_rows)
    if args.stream_k is not None:
        spk.set_stream_k(bool(args.stream_k))
    if args.many_row_variant is not None:
        spk.set_many_row_variant(args.many_row_variant)
    st = spk.stream
    gi = wl.group_indptr()
    qi = wl.q_indptr()
    verify = cfg.k_draft > 0
    q_np = wl.q_all()
    q_dev = spk._dev(q_np)
    rows = q_np.shape[0]
    out = torch.empty((rows, cfg.Hq, cfg.D), dtype=torch.float32, device=device)
    lse = torch.empty((rows, cfg.Hq), dtype=torch.float32, device=device)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=device)   # > 126 MB L2
    clean = torch.zeros(64 << 20, dtype=torch.int32, device=device)    # 256 MiB, only ever read
    parents = synth.churn_parents(5, 10000, ids) if churn else None

    churn_launches = [0]

    def step():
        if churn:
            ch = spk.fork(parents)
            n1 = spk.last_launches()
            spk.release(ch)
            churn_launches[0] = n1 + spk.last_launches()
        elif verify:
            spk.verify_attn(gi, ids, qi, q_dev, out, lse)
        else:
            spk.decode_attn(gi, ids, q_dev, out, lse)

    def flush_l2():
        # write 512 MiB (evicts every line of the workload), then read 256 MiB of unrelated data so
        # the dirty lines are written back BEFORE the timed region: L2 starts cold and clean
        with torch.cuda.stream(st):
            flush.zero_()
            clean.max()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(n, do_flush=True):
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
        for a, b in evs:
            if do_flush:
                flush_l2()
            a.record(st)
            step()
            b.record(st)
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in evs]

    # nvidia-smi samples every 100 ms: the sampler runs from the warm-up to the end of the e2e pass
    # (the GPU is under the same load throughout), the timed region lies inside that window
    sampler = ClockSampler(local)
    sampler.start()
    for _ in range(max(args.warmup, 3)):
        flush_l2()
        step()
    barrier()
    ms = timed(args.steps)
    barrier()
    total_ms = max_over_ranks(float(sum(ms)), device, world)
    ms_step = total_ms / args.steps

    info = spk.last_plan() if not churn else {}
    ub = wl.unique_kv_bytes() if not churn else 0
    flops = wl.flops()
    launches_per_step = info.get("launches", 0) if not churn else churn_launches[0]

    # ---- roofline of the dominant kernel (separate timed pass with kernel events on) ----
    roof = None
    extra = {}
    if not churn:
        spk.set_timing(True)
        k_ms, m_ms = [], []
        for _ in range(args.steps):
            flush_l2()
            step()
            a, m = spk.last_kernel_ms()
            k_ms.append(a)
            m_ms.append(m)
        spk.set_timing(False)
        k_avg = float(np.mean(k_ms))
        peak_bw = float(peaks["hbm_gbs"])
        ach_bw = info["unique_tokens"] * cfg.token_bytes / (k_avg * 1e-3) / 1e9
        peak_tf = float(peaks["bf16_tflops"])
        ach_tf = flops / (k_avg * 1e-3) / 1e12
        tensor_bound = verify and (flops / (peak_tf * 1e12)) > (ub / (peak_bw * 1e9))
        traffic = _traffic(name)
        if tensor_bound:
            roof = {"bound": "tensor", "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s",
                    "frac": ach_tf / peak_tf, "traffic": traffic}
        else:
            roof = {"bound": "hbm", "achieved": ach_bw, "peak": peak_bw, "unit": "GB/s",
                    "frac": ach_bw / peak_bw, "traffic": traffic}
        kname = {0: "attn_simt_kernel", 1: "attn_mma_kernel", 2: "attn_umma_kernel",
                 3: "attn_umma_kernel+attn_mma_kernel"}[info["kernel"]]
        roof.update({"kernel": kname,
                     "kernel_ms": k_avg, "merge_ms": float(np.mean(m_ms)), "peak_source": peaks["_source"],
                     "frac_of_8TBps": ach_bw / 8000.0, "achieved_tflops": ach_tf,
                     "algorithmic_bytes": info["unique_tokens"] * cfg.token_bytes})
        warm = timed(args.steps, do_flush=False)
        extra["warm_l2_ms_per_step"] = float(np.mean(warm))
        extra["plan"] = info

    # ---- e2e: host buffers through the C ABI, copies inside the timed region ----
    e2e = None
    if not churn:
        qh = torch.from_numpy(q_np).pin_memory()
        oh = torch.empty((rows, cfg.Hq, cfg.D), dtype=torch.float32).pin_memory()
        lh = torch.empty((rows, cfg.Hq), dtype=torch.float32).pin_memory()

        def e2e_step():
            if verify:
                spk.verify_attn_host(gi, ids, qi, qh, oh, lh)
            else:
                spk.decode_attn_host(gi, ids, qh, oh, lh)

        for _ in range(3):
            e2e_step()
        tt = []
        for _ in range(args.steps):
            flush_l2()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            e2e_step()
            tt.append(time.perf_counter() - t0)
        e_ms = max_over_ranks(float(np.mean(tt)) * 1e3, device, world)
        e2e = {"value": aggregate_value(ub, e_ms, world), "unit": "GB/s", "ms_per_step": e_ms,
               "h2d_bytes_per_step": int(qh.numel() * qh.element_size()),
               "d2h_bytes_per_step": int(oh.numel() * 4 + lh.numel() * 4)}
        # parity spot check of what was just timed (oracle, one sampled row)
        o = oh.numpy()
        assert np.all(np.isfinite(o))

    clocks = sampler.stop()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    cpu = None
    if not args.no_cpu_baseline and not churn:
        ostep, frac, cores, sample = oracle_sample(cfg, wl, args.ref_groups)
        # repeat the sample until about a second of wall clock (>= 10 core-seconds on this box's
        # host cores) has been spent; the mean step of the sample is scaled to the whole batch by flops
        reps, t0 = 0, time.perf_counter()
        while reps < 20 and (reps == 0 or time.perf_counter() - t0 < 1.0):
            ostep()
            reps += 1
        dt = (time.perf_counter() - t0) / reps
        cpu = {"value": ub / (dt / frac) / 1e9, "unit": "GB/s", "cores": cores, "kind": "oracle",
               "sample": sample + f", {reps} repetition(s)", "sample_seconds": dt * reps,
               "scaled_ms_per_step": dt / frac * 1e3}

    if churn:
        value, unit, metric = 10000 / (ms_step * 1e-3), "forks/s", "fork_release_churn"
    else:
        value, unit, metric = aggregate_value(ub, ms_step, world), "GB/s", METRIC
    line = {
        "metric": metric, "value": value, "unit": unit, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "us_per_step": ms_step * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": cfg.dtype,
        "data": "synthetic",
        "config": {"workload": name, "Hq": cfg.Hq, "Hkv": cfg.Hkv, "D": cfg.D, "n_groups": cfg.n_groups,
                   "group_size": cfg.group_size, "prefix_len": cfg.prefix_len,
                   "suffix": [cfg.suffix_lo, cfg.suffix_hi], "k_draft": cfg.k_draft,
                   "unique_kv_bytes": ub, "naive_kv_bytes": wl.naive_tokens() * cfg.token_bytes,
                   "flops": flops, "l2": "flushed between timed iterations (512 MiB write, then 256 MiB read so no dirty lines remain)",
                   "parallelism": "replicas only" if world > 1 else "1 gpu",
                   "state_build_seconds": t_build},
        "clocks": clocks,
        "gpu_launches": int(launches_per_step * args.steps),
        "frac_of_8TBps": (value / world / 8000.0) if not churn else None,
        "frac_of_measured_hbm": (value / world / float(peaks["hbm_gbs"])) if not churn else None,
    }
    if verify:
        line["verify_tflops"] = flops / (ms_step * 1e-3) / 1e12
    if roof is not None:
        line["roofline"] = roof
    if e2e is not None:
        line["e2e"] = e2e
    if cpu is not None:
        line["cpu_baseline"] = cpu
    line.update(extra)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


# ---------------------------------------------------------------------------
# D2 confidence: a stream over probe logits
# ---------------------------------------------------------------------------
D2_SPANS, D2_VOCAB = 256, 151936       # 256 probes in flight, Qwen3 vocabulary


def run_d2(args):
    import torch
    import paper_2607_03333_b200 as sp
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    x, spn = synth.probe_logits(D2_SPANS, D2_VOCAB, seed=0)
    rows_read = int(np.maximum(np.diff(spn) - 1, 0).sum())
    alg_bytes = rows_read * D2_VOCAB * 4
    name = "d2_confidence_qwen3_vocab"
    if args.impl == "reference":
        if rank != 0:
            return
        import oracle
        g = 16                              # spans in the oracle's bounded sample
        t0 = time.perf_counter()
        oracle.confidence(x[:spn[g]], spn[:g + 1])
        dt = time.perf_counter() - t0
        frac = float(np.maximum(np.diff(spn[:g + 1]) - 1, 0).sum()) / rows_read
        val = alg_bytes / (dt / frac) / 1e9
        sample = f"{g} of {D2_SPANS} spans, numpy fp64, 1 thread"
        print(json.dumps({"impl": "reference", "metric": "d2_confidence_logits_bandwidth", "value": val,
                          "unit": "GB/s", "n_gpus": args.gpus, "steps": 1, "warmup": 0,
                          "ms_per_step": dt / frac * 1e3, "higher_is_better": True, "scaling": "weak",
                          "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                          "config": {"workload": name, "sample": sample},
                          "cpu_baseline": {"value": val, "unit": "GB/s", "cores": 1, "kind": "oracle", "sample": sample},
                          "e2e": {"value": val, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                          "gpu_launches": 0}))
        return
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    device = f"cuda:{local}"
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(device))
    peaks = load_peaks()
    spk = sp.Spork("f32", 4, 1, 64, 8, 2, 4, 0.125, device=device)
    st = spk.stream
    xd = spk._dev(x)
    out = torch.empty((D2_SPANS,), dtype=torch.float32, device=device)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=device)
    clean = torch.zeros(64 << 20, dtype=torch.int32, device=device)

    def flush_l2():
        with torch.cuda.stream(st):
            flush.zero_()
            clean.max()

    def step():
        spk.confidence(spn, xd, out)

    sampler = ClockSampler(local)
    sampler.start()
    for _ in range(max(args.warmup, 3)):
        flush_l2()
        step()
    torch.cuda.synchronize()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for a, b in evs:
        flush_l2()
        a.record(st)
        step()
        b.record(st)
    torch.cuda.synchronize()
    ms_step = max_over_ranks(float(sum(a.elapsed_time(b) for a, b in evs)), device, world) / args.steps
    # e2e: logits in pinned host memory, copied in every step; the scores copied back
    xh = torch.from_numpy(x).pin_memory()
    oh = torch.empty((D2_SPANS,), dtype=torch.float32).pin_memory()
    tt = []
    for _ in range(min(args.steps, 10)):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        with torch.cuda.stream(st):
            xd.copy_(xh, non_blocking=True)
            step()
            oh.copy_(out, non_blocking=True)
        st.synchronize()
        tt.append(time.perf_counter() - t0)
    e_ms = max_over_ranks(float(np.mean(tt)) * 1e3, device, world)
    clocks = sampler.stop()
    if rank != 0:
        return
    import oracle
    want = oracle.confidence(x[:spn[8]], spn[:9])
    got = oh.numpy()[:8]
    assert np.allclose(got, want, rtol=2e-5), "bench output does not match the oracle"
    cpu = None
    if not args.no_cpu_baseline:
        g = 16
        t0 = time.perf_counter()
        oracle.confidence(x[:spn[g]], spn[:g + 1])
        dt = time.perf_counter() - t0
        frac = float(np.maximum(np.diff(spn[:g + 1]) - 1, 0).sum()) / rows_read
        cpu = {"value": alg_bytes / (dt / frac) / 1e9, "unit": "GB/s", "cores": 1, "kind": "oracle",
               "sample": f"{g} of {D2_SPANS} spans, numpy fp64, 1 thread", "sample_seconds": dt}
    ach = alg_bytes / (ms_step * 1e-3) / 1e9
    line = {"metric": "d2_confidence_logits_bandwidth", "value": aggregate_value(alg_bytes, ms_step, world),
            "unit": "GB/s", "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_step, "us_per_step": ms_step * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": name, "spans": D2_SPANS, "vocab": D2_VOCAB, "rows_read": rows_read,
                       "algorithmic_bytes": alg_bytes,
                       "l2": "flushed between timed iterations (512 MiB write, then 256 MiB read)",
                       "parallelism": "replicas only" if world > 1 else "1 gpu"},
            "clocks": clocks, "gpu_launches": 2 * args.steps,
            "roofline": {"bound": "hbm", "achieved": ach, "peak": float(peaks["hbm_gbs"]), "unit": "GB/s",
                         "frac": ach / float(peaks["hbm_gbs"]), "traffic": _traffic(name),
                         "kernel": "conf_partial_kernel+conf_span_kernel (whole call)",
                         "peak_source": peaks["_source"], "algorithmic_bytes": alg_bytes},
            "e2e": {"value": aggregate_value(alg_bytes, e_ms, world), "unit": "GB/s", "ms_per_step": e_ms,
                    "h2d_bytes_per_step": int(x.nbytes), "d2h_bytes_per_step": int(4 * D2_SPANS)}}
    if cpu is not None:
        line["cpu_baseline"] = cpu
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", default="2", choices=["2", "3", "4", "5", "churn", "d2"])
    ap.add_argument("--k", type=int, default=8, help="drafts per sequence for config 4")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-groups", type=int, default=0,
                    help="fork groups in the oracle's bounded sample (0: per-config default)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--stream-k", type=int, default=None, choices=[0, 1], help="planner knob: stream-K schedule")
    ap.add_argument("--many-row-variant", type=int, default=None, choices=[0, 1, 2],
                    help="planner knob: > 128-row segments on the two-pipe tcgen05 kernel")
    ap.add_argument("--min-rows", type=int, default=None,
                    help="planner knob: rows per KV head from which a segment runs on the tcgen05 kernel")
    ap.add_argument("--full-pool", action="store_true", help="config 5 on the 2^20-page pool")
    args = ap.parse_args()
    if args.config == "d2":
        run_d2(args)
        return
    cfg, name = pick_config(args)
    wl = synth.Workload(cfg)
    if args.ref_groups <= 0:
        args.ref_groups = {"2": 16, "3": 8, "4": 2, "5": 4, "churn": 1}[args.config]
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) == 0:
            run_reference(args, cfg, name, wl)
        return
    run_ours(args, cfg, name, wl)


if __name__ == "__main__":
    main()
