#!/usr/bin/env python
"""bench.py -- one JSON line per run (the driver's contract).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config all|1|2|3|4|5|churn|loop|turn|successive|layers|d2] [--kv bf16|e4m3]
                    [--k 4|8|16] [--impl reference]

A step = one pass of the hot path over one batch of synthetic input:
  configs 2/3/5  one spork_decode_attn call (plan lookup, cascade decode kernel, merge kernel)
  config 4       one spork_verify_attn call with k drafts per sequence
  config 1       the tiny fp32 group (us/step only: launch-latency bound, no roofline target)
  churn          one spork_fork of 10,000 children + one spork_release of them (config 5, 2^20-page pool)
  loop           spork_append of one token to every sequence + spork_decode_attn (Alg. 1 step 5,
                 PAPER.md:261; the paper's decode loop), on config 2
  successive     config 3's shape with probes forked at successive CoT positions: multi-level vs one-level cascade
  layers         config 2's batch over 36 layers: one plan, 36 chained (attention, merge) launches
  turn           one partial-token-accept turn of config 4's batch (append k drafts, verify, accept +
                 rollback, append one token, decode) captured in ONE CUDA graph and replayed (spork_turn_*)
  d2             one spork_confidence call: Eq. 2 over 256 probe spans of Qwen3-vocabulary logits
Default (`--config all`): the headline is the LARGEST single-GPU decode config of BASELINE.json
(config 5: 16 fork groups of 8, prefix 32768, 1.59 GB of unique KV); the same JSON line carries a
`per_config` object with the same measurements for config 2, config 3, config 4 at k = 4, 8, 16
(with verify TFLOP/s), the fork churn, the append+decode loop and config 1.
Inputs are seeded synthetic (synth/), resident in HBM before the timed region; L2 is flushed
between timed iterations.  `value` = unique KV bytes / step time (GB/s); config 4 also reports
TFLOP/s.  N > 1 (torchrun) runs N independent replicas: the path does not shard ("replicas only").
"""
from __future__ import annotations

import argparse
import gc
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
L2_NOTE = "flushed between timed iterations (512 MiB write, then 256 MiB read so no dirty lines remain)"
OUT_TOL = {"f32": 1e-5, "bf16": 1e-2, "e4m3": 1e-2}     # BASELINE.json north_star; e4m3 KV: DESIGN.md section 6
LSE_RTOL = 1e-4


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
        return self

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
def workload_name(cfg) -> str:
    name = f"cfg4_qwen3_32b_verify_k{cfg.k_draft}" if cfg.cfg_no == 4 else cfg.name
    return name + ("_e4m3kv" if cfg.dtype == "e4m3" else "")


def pool_dims(wl, num_pages=None):
    c = wl.cfg
    per_seq = int((wl.total_len.max() + 15) // 16) + 4
    need = int(c.n_groups * ((c.prefix_len + 15) // 16) + sum((int(x) + 15) // 16 + 1 for x in wl.private_len))
    return (num_pages or need + 1024), per_seq


def build_spork(cfg, wl, num_pages=None, max_seqs=None, device="cuda:0", extra_pages_per_seq=0):
    import paper_2607_03333_b200 as sp
    npg, mp = pool_dims(wl, num_pages)
    spk = sp.Spork(cfg.dtype, cfg.Hq, cfg.Hkv, cfg.D, npg, max_seqs or cfg.n_seqs + 8, mp + extra_pages_per_seq,
                   cfg.scale, device=device)
    ids = synth.build_state(spk, wl)
    spk.synchronize()
    return spk, ids


# ---------------------------------------------------------------------------
# the oracle leg (cpu_baseline, parity spot check, --impl reference): bounded samples of the workload
# ---------------------------------------------------------------------------
REF_GROUPS = {1: 1, 2: 16, 3: 8, 4: 2, 5: 4}


def oracle_sample(cfg, wl, max_groups=0):
    """Builds `max_groups` fork groups of the workload in the CPU oracle and returns a closure that
    runs one oracle step on them, plus the factor that scales its time to the whole batch."""
    import oracle
    g = min(cfg.n_groups, max_groups or REF_GROUPS[cfg.cfg_no])
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


def cpu_baseline_attn(cfg, wl, ub, max_groups=0):
    ostep, frac, cores, sample = oracle_sample(cfg, wl, max_groups)
    # repeat the sample until about a second of wall clock (>= 10 core-seconds on this box's host
    # cores) has been spent; the mean step of the sample is scaled to the whole batch by flops
    reps, t0 = 0, time.perf_counter()
    while reps < 20 and (reps == 0 or time.perf_counter() - t0 < 1.0):
        ostep()
        reps += 1
    dt = (time.perf_counter() - t0) / reps
    rec = {"value": ub / (dt / frac) / 1e9, "unit": "GB/s", "cores": cores, "kind": "oracle",
           "sample": sample + f", {reps} repetition(s)", "sample_seconds": dt * reps,
           "scaled_ms_per_step": dt / frac * 1e3}
    if cfg.cfg_no <= 2:
        # configs 1-2 also on ONE thread (one repetition of the same sample)
        import oracle
        oracle.set_num_threads(1)
        t0 = time.perf_counter()
        ostep()
        d1 = time.perf_counter() - t0
        oracle.set_num_threads(cores)
        rec["one_thread"] = {"value": ub / (d1 / frac) / 1e9, "unit": "GB/s", "cores": 1,
                             "scaled_ms_per_step": d1 / frac * 1e3, "sample_seconds": d1}
    return rec


def parity_spot_check(cfg, wl, out_np, lse_np, n_rows=2, seed=0):
    """What was just timed, against the oracle's plain dense definition on regenerated K/V: `n_rows`
    sampled (sequence, draft row) pairs, ALL heads of each.  Asserts the north_star tolerances."""
    import oracle
    r = np.random.default_rng([23, cfg.cfg_no, seed])
    qi = wl.q_indptr()
    worst, worst_l = 0.0, 0.0
    for _ in range(n_rows):
        seq = int(r.integers(0, cfg.n_seqs))
        k = int(wl.k[seq])
        j = int(r.integers(0, max(1, k)))
        K, V = wl.dense_kv(seq)
        Q = wl.q(seq)
        L = int(wl.total_len[seq])
        n_att = L if k == 0 else L - k + j + 1
        row = int(qi[seq]) + j
        for h in range(cfg.Hq):
            o_ref, l_ref = oracle.attend_dense(cfg.dtype, cfg.scale, Q[j, h], K[:n_att, h // cfg.G],
                                               V[:n_att, h // cfg.G])
            err = float(np.max(np.abs(out_np[row, h].astype(np.float64) - o_ref)))
            lerr = abs(float(lse_np[row, h]) - l_ref) / max(1.0, abs(l_ref))
            worst, worst_l = max(worst, err), max(worst_l, lerr)
    assert worst <= OUT_TOL[cfg.dtype] and worst_l <= LSE_RTOL, \
        f"bench output does not match the oracle: out err {worst:.3e}, lse rel err {worst_l:.3e}"
    return {"rows_checked": n_rows * cfg.Hq, "max_abs_err": worst, "max_lse_rel_err": worst_l,
            "tolerance": OUT_TOL[cfg.dtype], "against": "oracle.attend_dense (fp64)"}


def reference_line(args, cfg, wl):
    name = workload_name(cfg)
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
    return {
        "impl": "reference", "metric": METRIC, "value": val, "unit": "GB/s", "n_gpus": args.gpus,
        "steps": steps, "warmup": args.warmup, "ms_per_step": full * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": cfg.dtype, "data": "synthetic",
        "config": {"workload": name, "sample": sample, "sample_seconds_per_step": dt},
        "cpu_baseline": {"value": val, "unit": "GB/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }


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
class Env:
    """Per-process GPU context shared by all records of a run."""

    def __init__(self, args):
        import torch
        self.torch = torch
        self.args = args
        self.rank = int(os.environ.get("RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
        self.device = f"cuda:{self.local}"
        torch.cuda.set_device(self.local)
        if self.world > 1:
            import torch.distributed as dist
            dist.init_process_group("nccl", device_id=torch.device(self.device))
        self.peaks = load_peaks()
        self.flush = torch.empty(512 << 20, dtype=torch.uint8, device=self.device)   # > 126 MB L2
        self.clean = torch.zeros(64 << 20, dtype=torch.int32, device=self.device)    # 256 MiB, only ever read

    def flush_l2(self, st):
        # write 512 MiB (evicts every line of the workload), then read 256 MiB of unrelated data so
        # the dirty lines are written back BEFORE the timed region: L2 starts cold and clean
        with self.torch.cuda.stream(st):
            self.flush.zero_()
            self.clean.max()

    def barrier(self):
        self.torch.cuda.synchronize()
        if self.world > 1:
            import torch.distributed as dist
            dist.barrier()
        self.torch.cuda.synchronize()

    def timed(self, st, step, n, do_flush=True, pre=None):
        """CUDA events on the launch stream around each of n steps (L2 flushed before each)."""
        torch = self.torch
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
        for a, b in evs:
            if pre is not None:
                pre()
            if do_flush:
                self.flush_l2(st)
            a.record(st)
            step()
            b.record(st)
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in evs]

    def mx(self, x):
        return max_over_ranks(float(x), self.device, self.world)

    def read_peak(self, spk):
        """GB/s a plain read-only stream reaches on this GPU now (spork_hbm_read_probe over the 512 MiB
        flush buffer, best of 10 after a warm-up pass).  Reported beside the driver's copy figure: the
        attention kernels read, they do not copy."""
        if getattr(self, "_read_peak", None) is None:
            torch = self.torch
            st = spk.stream
            nbytes = self.flush.numel()
            spk.hbm_read_probe(self.flush)
            best = 0.0
            for _ in range(10):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(st)
                spk.hbm_read_probe(self.flush)
                b.record(st)
                b.synchronize()
                best = max(best, nbytes / (a.elapsed_time(b) * 1e-3) / 1e9)
            self._read_peak = best
        return self._read_peak

    def close(self):
        if self.world > 1:
            import torch.distributed as dist
            dist.destroy_process_group()


def measure_attn(env: Env, spk, ids, cfg, wl, cpu=True):
    """One record: step time, roofline of the dominant kernel, e2e through the host-buffer ABI calls,
    the oracle on the host cores, and a parity spot check of the timed output."""
    torch, args = env.torch, env.args
    name = workload_name(cfg)
    st = spk.stream
    gi, qi = wl.group_indptr(), wl.q_indptr()
    verify = cfg.k_draft > 0
    q_np = wl.q_all()
    q_dev = spk._dev(q_np)
    rows = q_np.shape[0]
    out = torch.empty((rows, cfg.Hq, cfg.D), dtype=torch.float32, device=env.device)
    lse = torch.empty((rows, cfg.Hq), dtype=torch.float32, device=env.device)

    def step():
        if verify:
            spk.verify_attn(gi, ids, qi, q_dev, out, lse)
        else:
            spk.decode_attn(gi, ids, q_dev, out, lse)

    # nvidia-smi samples every 100 ms: the sampler runs from the warm-up to the end of the e2e pass
    # (the GPU is under the same load throughout), the timed region lies inside that window
    sampler = ClockSampler(env.local).start()
    t0 = time.perf_counter()
    step()
    spk.synchronize()
    first_call_us = (time.perf_counter() - t0) * 1e6      # plan build + upload + first launch, host clock
    info0 = spk.last_plan()
    for _ in range(max(args.warmup, 3)):
        env.flush_l2(st)
        step()
    # steady-state plan rebuild (workspace already sized): invalidate the cached plan, time the next call
    spk.set_cascade_levels(7)
    spk.synchronize()
    t0 = time.perf_counter()
    step()
    rebuild_call_us = (time.perf_counter() - t0) * 1e6    # host time of a call that rebuilds the plan
    info1 = spk.last_plan()
    assert info1["plan_cached"] == 0
    env.barrier()
    ms = env.timed(st, step, args.steps)
    env.barrier()
    ms_step = env.mx(sum(ms)) / args.steps
    info = spk.last_plan()
    assert info["plan_cached"] == 1
    ub = wl.unique_kv_bytes()
    assert info["unique_tokens"] * cfg.token_bytes == ub, "library and synth disagree on the unique KV bytes"
    flops = wl.flops()

    # ---- roofline of the dominant kernel (separate timed pass with kernel events on) ----
    peaks = env.peaks
    spk.set_timing(True)
    k_ms, m_ms = [], []
    for _ in range(args.steps):
        env.flush_l2(st)
        step()
        a, m = spk.last_kernel_ms()
        k_ms.append(a)
        m_ms.append(m)
    spk.set_timing(False)
    k_avg = float(np.mean(k_ms))
    bf16_path = info["kernel"] != 0
    peak_bw, peak_tf = float(peaks["hbm_gbs"]), float(peaks["bf16_tflops"])
    ach_bw = ub / (k_avg * 1e-3) / 1e9
    ach_tf = flops / (k_avg * 1e-3) / 1e12
    tensor_bound = verify and bf16_path and (flops / (peak_tf * 1e12)) > (ub / (peak_bw * 1e9))
    kname = {0: "attn_simt_kernel", 1: "attn_mma_kernel", 2: "attn_umma_kernel",
             3: "attn_umma_kernel+attn_mma_kernel"}[info["kernel"]]
    if tensor_bound:
        roof = {"bound": "tensor", "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s",
                "frac": ach_tf / peak_tf, "traffic": _traffic(name)}
    else:
        roof = {"bound": "hbm", "achieved": ach_bw, "peak": peak_bw, "unit": "GB/s",
                "frac": ach_bw / peak_bw, "traffic": _traffic(name)}
    read_peak = env.read_peak(spk)
    roof.update({"kernel": kname, "kernel_ms": k_avg, "merge_ms": float(np.mean(m_ms)),
                 "peak_source": peaks["_source"], "frac_of_8TBps": ach_bw / 8000.0,
                 "read_peak": read_peak, "frac_of_read_peak": ach_bw / read_peak,
                 "peak_note": "peak = MEASURED_PEAKS.json's copy (read + write) figure; read_peak = a plain "
                              "read-only stream of bulk copies timed in this run (spork_hbm_read_probe), the "
                              "ceiling of a read-dominated kernel",
                 "achieved_tflops": ach_tf, "algorithmic_bytes": ub, "algorithmic_flops": flops})
    warm = env.timed(st, step, args.steps, do_flush=False)

    # ---- e2e: host buffers through the C ABI, copies inside the timed region ----
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
        env.flush_l2(st)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        e2e_step()
        tt.append(time.perf_counter() - t0)
    e_ms = env.mx(float(np.mean(tt)) * 1e3)
    e2e = {"value": aggregate_value(ub, e_ms, env.world), "unit": "GB/s", "ms_per_step": e_ms,
           "h2d_bytes_per_step": int(qh.numel() * qh.element_size()),
           "d2h_bytes_per_step": int(oh.numel() * 4 + lh.numel() * 4)}
    clocks = sampler.stop()

    rec = {
        "workload": name, "ms_per_step": ms_step, "us_per_step": ms_step * 1e3,
        "value": aggregate_value(ub, ms_step, env.world), "unit": "GB/s",
        "frac_of_8TBps": ub / (ms_step * 1e-3) / 1e9 / 8000.0,
        "frac_of_measured_hbm": ub / (ms_step * 1e-3) / 1e9 / peak_bw,
        "dtype": cfg.dtype, "unique_kv_bytes": ub, "naive_kv_bytes": wl.naive_tokens() * cfg.token_bytes,
        "flops": flops, "roofline": roof, "e2e": e2e, "clocks": clocks,
        "warm_l2_ms_per_step": float(np.mean(warm)), "first_call_us": first_call_us,
        "plan_rebuild_us": info1.get("plan_host_us"), "plan_rebuild_call_us": rebuild_call_us,
        "plan_first_build_us": info0.get("plan_host_us"),
        "launches_per_step": info["launches"], "plan": info,
        "shape": {"Hq": cfg.Hq, "Hkv": cfg.Hkv, "D": cfg.D, "n_groups": cfg.n_groups,
                  "group_size": cfg.group_size, "prefix_len": cfg.prefix_len,
                  "suffix": [cfg.suffix_lo, cfg.suffix_hi], "k_draft": cfg.k_draft},
    }
    if verify:
        rec["verify_tflops"] = flops / (ms_step * 1e-3) / 1e12
    if env.rank == 0 and cpu and not args.no_cpu_baseline:
        rec["parity"] = parity_spot_check(cfg, wl, oh.numpy(), lh.numpy())
        rec["cpu_baseline"] = cpu_baseline_attn(cfg, wl, ub, args.ref_groups)
    return rec


def churn_bytes(cfg, wl, ids, parents, num_pages):
    """Algorithmic bytes of the churn step, computed exactly.  SURVEY.md 8(d)'s churn row counts the
    LOGICAL traffic (every child reads its parent's row and tail: 87 + 87 + 328 + 328 MB); the 10,000
    children have only 128 distinct parents, whose rows and tail pages are read from HBM once and
    then served by L2, so the bytes that must cross the HBM interface -- the roofline's numerator --
    are: fork = the DISTINCT parents' table rows and tail pages read, the children's rows
    (floor(L/16) + 1 entries of 4 B) and duplicated tail pages (K and V) written, one scan of the
    refcount array; release = the children's table rows read once more."""
    L = {int(s): int(wl.total_len[i]) for i, s in enumerate(ids)}
    page_bytes = cfg.Hkv * 16 * cfg.D * cfg.elt_bytes          # one pool
    entries = sum(L[int(p)] // 16 + 1 for p in parents)
    tails = sum(1 for p in parents if L[int(p)] % 16)
    distinct = sorted(set(int(p) for p in parents))
    d_entries = sum(L[p] // 16 + 1 for p in distinct)
    d_tails = sum(1 for p in distinct if L[p] % 16)
    fork_clone = 4 * (d_entries + entries) + (d_tails + tails) * 2 * page_bytes
    logical = 2 * 4 * entries + tails * 2 * 2 * page_bytes
    return {"fork_clone_kernel": fork_clone, "fork_clone_kernel_logical": logical,
            "refcount_scan": 4 * num_pages, "release_table_read": 4 * entries,
            "step": fork_clone + 4 * num_pages + 4 * entries,
            "step_logical": logical + 4 * num_pages + 4 * entries,
            "table_entries": entries, "tail_pages": tails, "distinct_parents": len(distinct)}


def measure_churn(env: Env, spk, ids, cfg, wl, num_pages):
    """config 5 fork stress: 10,000 spork_fork + spork_release per step on the 2^20-page pool."""
    args = env.args
    st = spk.stream
    parents = synth.churn_parents(5, 10000, ids)
    launches = [0]

    def step():
        ch = spk.fork(parents)
        n1 = spk.last_launches()
        spk.release(ch)
        launches[0] = n1 + spk.last_launches()

    sampler = ClockSampler(env.local).start()
    for _ in range(max(args.warmup, 3)):
        env.flush_l2(st)
        step()
    env.barrier()
    ms = env.timed(st, step, args.steps)
    env.barrier()
    ms_step = env.mx(sum(ms)) / args.steps
    # dominant kernel: fork_clone_kernel (table rows + tail pages), timed live with events on the stream
    spk.set_timing(True)
    k_ms = []
    for _ in range(args.steps):
        env.flush_l2(st)
        ch = spk.fork(parents)
        k_ms.append(spk.last_kernel_ms()[0])
        spk.release(ch)
    spk.set_timing(False)
    clocks = sampler.stop()
    k_avg = float(np.mean(k_ms))
    by = churn_bytes(cfg, wl, ids, parents, num_pages)
    peak_bw = float(env.peaks["hbm_gbs"])
    ach = by["fork_clone_kernel"] / (k_avg * 1e-3) / 1e9
    rec = {
        "workload": "cfg5_fork_churn", "ms_per_step": ms_step, "us_per_step": ms_step * 1e3,
        "value": env.world * 10000 / (ms_step * 1e-3), "unit": "forks/s", "dtype": "int32",
        "step_gbs": by["step"] / (ms_step * 1e-3) / 1e9, "algorithmic_bytes_step": by["step"],
        "roofline": {"bound": "hbm", "achieved": ach, "peak": peak_bw, "unit": "GB/s", "frac": ach / peak_bw,
                     "traffic": _traffic("cfg5_fork_churn"), "kernel": "fork_clone_kernel", "kernel_ms": k_avg,
                     "peak_source": env.peaks["_source"], "algorithmic_bytes": by["fork_clone_kernel"]},
        "e2e": {"value": env.world * 10000 / (ms_step * 1e-3), "unit": "forks/s", "ms_per_step": ms_step,
                "h2d_bytes_per_step": 4 * 10000 * 2, "d2h_bytes_per_step": 0,
                "note": "the ABI takes HOST id arrays: the timed step already contains their staging copies"},
        "clocks": clocks, "launches_per_step": launches[0], "bytes": by,
        "shape": {"forks": 10000, "live_parents": int(len(ids)), "num_pages": num_pages},
    }
    if env.rank == 0 and not args.no_cpu_baseline:
        rec["cpu_baseline"] = cpu_baseline_churn(cfg, wl, num_pages)
    return rec


def cpu_baseline_churn(cfg, wl, num_pages, n_forks=10000):
    """oracle fork x 10,000 + release on the 2^20-page pool, single thread (the
    lowest-free-id policy is sequential).  State is built with lengths only (no KV values: the oracle's
    allocator does not look at them; its tail copies are skipped)."""
    import oracle
    npg, mp = pool_dims(wl, num_pages)
    orc = oracle.Oracle(cfg.dtype, cfg.Hq, cfg.Hkv, cfg.D, npg, cfg.n_seqs + n_forks + 8, mp, cfg.scale,
                        store_kv=False)
    ids = synth.build_state(orc, wl, values=False)
    parents = synth.churn_parents(5, n_forks, ids)
    t0 = time.perf_counter()
    ch = orc.fork(parents)
    orc.release(ch)
    dt = time.perf_counter() - t0
    return {"value": n_forks / dt, "unit": "forks/s", "cores": 1, "kind": "oracle",
            "sample": f"the whole step once: {n_forks} forks + releases, table and refcount work only (no tail copies)",
            "sample_seconds": dt, "scaled_ms_per_step": dt * 1e3}


def measure_cfg1(env: Env):
    """config 1: us/step of the tiny fp32 fork group (launch latency; excluded from the 70 % target)."""
    args = env.args
    cfg = synth.CFG1
    wl = synth.Workload(cfg)
    spk, ids = build_spork(cfg, wl, device=env.device)
    st = spk.stream
    gi = wl.group_indptr()
    q_np = wl.q_all()
    q_dev = spk._dev(q_np)
    out, lse = spk.decode_attn(gi, ids, q_dev)

    def step():
        spk.decode_attn(gi, ids, q_dev, out, lse)

    for _ in range(max(args.warmup, 3)):
        step()
    ms = env.timed(st, step, args.steps)
    ms_step = env.mx(sum(ms)) / args.steps
    spk.set_timing(True)
    k_ms = []
    for _ in range(args.steps):
        step()
        k_ms.append(spk.last_kernel_ms()[0])
    spk.set_timing(False)
    ub = wl.unique_kv_bytes()
    rec = {"workload": cfg.name, "ms_per_step": ms_step, "us_per_step": ms_step * 1e3, "dtype": "f32",
           "value": aggregate_value(ub, ms_step, env.world), "unit": "GB/s", "unique_kv_bytes": ub,
           "roofline": None, "kernel": "attn_simt_kernel", "kernel_ms": float(np.mean(k_ms)),
           "note": "0.16 MB problem: launch-latency bound, excluded from the 70 % target (SURVEY 8(d))",
           "plan": spk.last_plan()}
    if env.rank == 0 and not args.no_cpu_baseline:
        import oracle
        o = oracle.Oracle(cfg.dtype, cfg.Hq, cfg.Hkv, cfg.D, 64, 8, 32, cfg.scale)
        oids = synth.build_state(o, wl)
        ref, lref = o.decode(oids, q_np)
        err = float(np.max(np.abs(out.cpu().numpy() - ref)))
        assert err <= OUT_TOL["f32"], f"config 1 does not match the oracle: {err:.3e}"
        t0 = time.perf_counter()
        for _ in range(20):
            o.decode(oids, q_np)
        dt = (time.perf_counter() - t0) / 20
        rec["parity"] = {"rows_checked": int(ref.shape[0] * ref.shape[1]), "max_abs_err": err, "tolerance": 1e-5}
        rec["cpu_baseline"] = {"value": ub / dt / 1e9, "unit": "GB/s", "cores": oracle.num_threads(),
                               "kind": "oracle", "sample": "the whole step, 20 repetitions",
                               "scaled_ms_per_step": dt * 1e3}
        cores = oracle.num_threads()
        oracle.set_num_threads(1)
        t0 = time.perf_counter()
        for _ in range(20):
            o.decode(oids, q_np)
        d1 = (time.perf_counter() - t0) / 20
        oracle.set_num_threads(cores)
        rec["cpu_baseline"]["one_thread"] = {"value": ub / d1 / 1e9, "unit": "GB/s", "cores": 1,
                                             "scaled_ms_per_step": d1 * 1e3}
    spk.close()
    return rec


def measure_loop(env: Env, cfg, n_steps=None):
    """The paper's decode loop (Alg. 1 step 5; SURVEY 8(b) call order): each timed step
    appends ONE token to every sequence and then attends.  Reports the step, the append's share and
    how often the plan had to be rebuilt."""
    torch, args = env.torch, env.args
    wl = synth.Workload(cfg)
    n_steps = n_steps or max(args.steps, 64)
    total = n_steps + max(args.warmup, 3) + 8
    spk, ids = build_spork(cfg, wl, device=env.device, extra_pages_per_seq=total // 16 + 2,
                           num_pages=pool_dims(wl)[0] + cfg.n_seqs * (total // 16 + 2))
    st = spk.stream
    gi = wl.group_indptr()
    q_dev = spk._dev(wl.q_all())
    out = torch.empty((cfg.n_seqs, cfg.Hq, cfg.D), dtype=torch.float32, device=env.device)
    lse = torch.empty((cfg.n_seqs, cfg.Hq), dtype=torch.float32, device=env.device)
    r = synth.rng(cfg.cfg_no, synth.T_MISC, 77)
    kv = spk._dev(synth.to_storage(r.standard_normal((2, cfg.n_seqs, cfg.Hkv, cfg.D), dtype=np.float32), cfg.dtype))
    ones = np.ones(cfg.n_seqs, np.int32)
    cached, rebuild_us = [], []

    def step():
        spk.append(ids, ones, kv[0], kv[1])
        spk.decode_attn(gi, ids, q_dev, out, lse)

    for _ in range(max(args.warmup, 3)):
        env.flush_l2(st)
        step()
    env.barrier()
    evs = []
    for _ in range(n_steps):
        env.flush_l2(st)
        a, b, c = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        a.record(st)
        spk.append(ids, ones, kv[0], kv[1])
        b.record(st)
        spk.decode_attn(gi, ids, q_dev, out, lse)
        c.record(st)
        info = spk.last_plan()
        cached.append(info["plan_cached"])
        if not info["plan_cached"]:
            rebuild_us.append(info.get("plan_host_us"))
        evs.append((a, b, c))
    torch.cuda.synchronize()
    env.barrier()
    app = float(np.mean([a.elapsed_time(b) for a, b, _ in evs]))
    att = float(np.mean([b.elapsed_time(c) for _, b, c in evs]))
    ms_step = env.mx(float(np.mean([a.elapsed_time(c) for a, _, c in evs])))
    # host-side pace: the same loop without flushes or events, wall clock per step
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(n_steps):
        step()
    torch.cuda.synchronize()
    wall = (time.perf_counter() - t0) / n_steps
    L_end = wl.total_len + (2 * n_steps + 2 * max(args.warmup, 3))
    spk.close()
    return {"workload": f"{cfg.name}_append_decode_loop", "steps": n_steps, "ms_per_step": ms_step,
            "us_per_step": ms_step * 1e3, "append_us": app * 1e3, "attn_us": att * 1e3,
            "wall_us_per_step_back_to_back": wall * 1e6,
            "plan_cached_frac": float(np.mean(cached)), "plan_rebuilds": int(len(cached) - sum(cached)),
            "plan_rebuild_us": float(np.mean([x for x in rebuild_us if x is not None])) if any(
                x is not None for x in rebuild_us) else None,
            "value": aggregate_value(wl.unique_kv_bytes(), ms_step, env.world), "unit": "GB/s",
            "note": "unique KV bytes of the initial state; sequences grow by one token per step",
            "final_mean_len": float(np.mean(L_end))}


def measure_successive(env: Env):
    """Successive probes (Algorithm 1 steps 4-6): config 3's shape,
    32 mains, 3 probes forked after 500 / 1000 / 1500 further CoT tokens.  The multi-level cascade reads
    every shared run once; with one level (the round-1 planner) everything beyond the first fork point is
    read once per member.  Same kernels, same outputs: only the plan differs."""
    args = env.args
    cfg = synth.CFG3
    wl = synth.SuccessiveWorkload(cfg, 500)
    per_seq = int(wl.total_len.max()) // 16 + 4
    npg = int(sum(int(x) // 16 + 2 for x in wl.total_len)) + 1024
    import paper_2607_03333_b200 as sp
    spk = sp.Spork(cfg.dtype, cfg.Hq, cfg.Hkv, cfg.D, npg, cfg.n_seqs + 8, per_seq, cfg.scale, device=env.device)
    ids = synth.build_state_successive(spk, wl)
    spk.synchronize()
    st = spk.stream
    gi = wl.group_indptr()
    q_dev = spk._dev(wl.q_all())
    out, lse = spk.decode_attn(gi, ids, q_dev)
    rec = {"workload": "cfg3_successive_probes_500_1000_1500", "dtype": cfg.dtype,
           "nested_unique_tokens": wl.unique_tokens(), "single_level_tokens": wl.single_level_tokens(),
           "naive_tokens": wl.naive_tokens()}
    for name, lv in (("multi_level", 7), ("single_level", 1)):
        spk.set_cascade_levels(lv)

        def step():
            spk.decode_attn(gi, ids, q_dev, out, lse)

        for _ in range(max(args.warmup, 3)):
            env.flush_l2(st)
            step()
        env.barrier()
        ms = env.mx(sum(env.timed(st, step, args.steps))) / args.steps
        info = spk.last_plan()
        by = info["unique_tokens"] * cfg.token_bytes
        rec[name] = {"us_per_step": ms * 1e3, "plan_tokens_read": info["unique_tokens"], "bytes_read_model": by,
                     "GBps": by / (ms * 1e-3) / 1e9, "n_levels": info["n_levels"], "n_items": info["n_items"]}
    assert rec["multi_level"]["plan_tokens_read"] == wl.unique_tokens()
    assert rec["single_level"]["plan_tokens_read"] == wl.single_level_tokens()
    ub = wl.unique_tokens() * cfg.token_bytes
    ms = rec["multi_level"]["us_per_step"] * 1e-3
    rec.update({"ms_per_step": ms, "us_per_step": ms * 1e3, "unique_kv_bytes": ub,
                "value": aggregate_value(ub, ms, env.world), "unit": "GB/s", "frac_of_8TBps": ub / (ms * 1e-3) / 1e9 / 8000.0,
                "speedup_vs_single_level": rec["single_level"]["us_per_step"] / rec["multi_level"]["us_per_step"]})
    if env.rank == 0 and not args.no_cpu_baseline:
        rec["parity"] = parity_spot_check(cfg, wl, out.cpu().numpy(), lse.cpu().numpy())
    spk.close()
    return rec


def measure_layers(env: Env, n_layers=36):
    """Multi-layer step: config 2's batch over the 36 layers of Qwen3-4B:
    ONE plan, 36 x (attention, merge) launches chained programmatically.  Layers 1.. hold copies of layer
    0's K/V (the values do not matter for the time)."""
    torch, args = env.torch, env.args
    cfg = synth.CFG2
    wl = synth.Workload(cfg)
    spk, ids = build_spork(cfg, wl, device=env.device)
    spk.layers(n_layers)
    with torch.cuda.stream(spk.stream):
        for l in range(1, n_layers):
            spk.k_pools[l].copy_(spk.k_pool)
            spk.v_pools[l].copy_(spk.v_pool)
    st = spk.stream
    gi = wl.group_indptr()
    q0 = spk._dev(wl.q_all())
    qs = [q0] + [q0.clone() for _ in range(n_layers - 1)]
    outs = [torch.empty((cfg.n_seqs, cfg.Hq, cfg.D), dtype=torch.float32, device=env.device) for _ in range(n_layers)]
    lses = [torch.empty((cfg.n_seqs, cfg.Hq), dtype=torch.float32, device=env.device) for _ in range(n_layers)]

    def step():
        spk.attn_layers(gi, ids, qs, outs, lses)

    def single():
        spk.decode_attn(gi, ids, q0, outs[0], lses[0])

    for _ in range(max(args.warmup, 3)):
        env.flush_l2(st)
        step()
    env.barrier()
    n = max(5, args.steps // 2)
    ms = env.mx(sum(env.timed(st, step, n))) / n
    single()
    ms1 = env.mx(sum(env.timed(st, single, args.steps))) / args.steps
    launches = spk.last_plan()["launches"]
    ub = wl.unique_kv_bytes()
    same = bool(torch.equal(outs[0], outs[n_layers - 1]))     # identical pools and q: identical results
    spk.close()
    return {"workload": f"cfg2_x{n_layers}_layers", "layers": n_layers, "ms_per_step": ms, "us_per_step": ms * 1e3,
            "us_per_layer": ms * 1e3 / n_layers, "single_layer_call_us": ms1 * 1e3,
            "value": aggregate_value(ub * n_layers, ms, env.world), "unit": "GB/s",
            "frac_of_8TBps": ub * n_layers / (ms * 1e-3) / 1e9 / 8000.0, "unique_kv_bytes_per_layer": ub,
            "last_layer_equals_first": same, "dtype": cfg.dtype,
            "note": "K/V of 36 layers = 14 GB: nothing of a layer survives in L2 until its next use"}


def measure_turn(env: Env, k=16, n_turns=30):
    """config 4's batch, one partial-token-accept turn per step, captured in ONE CUDA graph and replayed
    (spork_turn_*: no host round trip): append k drafts -> verify -> accept + rollback -> append 1 token ->
    decode.  Random accept lengths (uniform in 0..k), so sequences grow by k/2 + 1 tokens per turn."""
    torch, args = env.torch, env.args
    cfg = synth.CFG4.scaled(k_draft=0)
    wl = synth.Workload(cfg)
    grow = (n_turns + max(args.warmup, 3) + 4) * (k + 1) + k
    spk, ids = build_spork(cfg, wl, device=env.device, extra_pages_per_seq=grow // 16 + 2,
                           num_pages=pool_dims(wl)[0] + cfg.n_seqs * (grow // 16 + 2))
    st = spk.stream
    n, tot = cfg.n_seqs, cfg.n_seqs * k
    ks = np.full(n, k, np.int64)
    qi = np.concatenate([[0], np.cumsum(ks)]).astype(np.int32)
    r = synth.rng(cfg.cfg_no, synth.T_MISC, 99)
    f = lambda *shape: spk._dev(synth.to_storage(r.standard_normal(shape, dtype=np.float32), cfg.dtype))
    kd, vd, qv = f(tot, cfg.Hkv, cfg.D), f(tot, cfg.Hkv, cfg.D), f(tot, cfg.Hq, cfg.D)
    k1, v1, qd = f(n, cfg.Hkv, cfg.D), f(n, cfg.Hkv, cfg.D), f(n, cfg.Hq, cfg.D)
    draft_np = r.integers(0, 50000, size=tot).astype(np.int32)
    target_np = draft_np.copy()
    acc_want = r.integers(0, k + 1, size=n)
    for i in range(n):
        target_np[qi[i] + acc_want[i]:qi[i + 1]] += 1
    draft, target = spk._dev(draft_np), spk._dev(target_np)
    dev = env.device
    out_v = torch.empty((tot, cfg.Hq, cfg.D), dtype=torch.float32, device=dev)
    lse_v = torch.empty((tot, cfg.Hq), dtype=torch.float32, device=dev)
    out_d = torch.empty((n, cfg.Hq, cfg.D), dtype=torch.float32, device=dev)
    lse_d = torch.empty((n, cfg.Hq), dtype=torch.float32, device=dev)
    acc = torch.zeros(n, dtype=torch.int32, device=dev)
    turn = spk.turn(wl.group_indptr(), ids, qi)
    launches = [0]

    def enqueue():
        turn.append(0, kd, vd)
        a = spk.last_launches()
        turn.verify(qv, out_v, lse_v)
        b = spk.last_launches()
        turn.accept(draft, target, acc)
        c = spk.last_launches()
        turn.append(1, k1, v1)
        d = spk.last_launches()
        turn.decode(qd, out_d, lse_d)
        launches[0] = a + b + c + d + spk.last_launches()

    enqueue()                                   # eager warm-up turn
    spk.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=st):
        enqueue()
    with torch.cuda.stream(st):
        for _ in range(max(args.warmup, 3)):
            env.flush_l2(st)
            g.replay()
    env.barrier()
    evs = []
    with torch.cuda.stream(st):
        for _ in range(n_turns):
            env.flush_l2(st)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(st)
            g.replay()
            b.record(st)
            evs.append((a, b))
    torch.cuda.synchronize()
    ms_turn = env.mx(float(np.mean([a.elapsed_time(b) for a, b in evs])))
    # the same turn issued call by call (eager launches, no graph), wall clock per turn back to back
    t0 = time.perf_counter()
    for _ in range(4):
        enqueue()
    spk.synchronize()
    eager = (time.perf_counter() - t0) / 4
    rc = turn.sync(check=False)
    assert rc == 0 and np.array_equal(acc.cpu().numpy(), acc_want), "turn state went wrong"
    lens = np.array([spk.export(int(s))[0] for s in ids])
    turn.close()
    spk.close()
    return {"workload": f"cfg4_turn_k{k}_cuda_graph", "turn_us": ms_turn * 1e3, "ms_per_step": ms_turn,
            "us_per_step": ms_turn * 1e3, "turns": n_turns, "kernels_per_turn": launches[0],
            "eager_wall_us_per_turn": eager * 1e6, "mean_accept_len": float(acc_want.mean()),
            "value": env.world * cfg.n_seqs * (k + 1) / (ms_turn * 1e-3), "unit": "query rows/s",
            "note": "one graph replay = append k drafts, verify, accept + rollback, append 1 token, decode; "
                    "L2 flushed before every replay; no host round trip inside the turn",
            "final_mean_len": float(lens.mean())}


def release_all(spk):
    spk.close()
    gc.collect()
    import torch
    torch.cuda.empty_cache()


def headline_line(env: Env, rec, cfg):
    args = env.args
    line = {
        "metric": METRIC, "value": rec["value"], "unit": "GB/s", "n_gpus": env.world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": rec["ms_per_step"], "us_per_step": rec["us_per_step"],
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": cfg.dtype, "data": "synthetic",
        "config": dict(rec["shape"], workload=rec["workload"], unique_kv_bytes=rec["unique_kv_bytes"],
                       naive_kv_bytes=rec["naive_kv_bytes"], flops=rec["flops"], l2=L2_NOTE,
                       parallelism="replicas only" if env.world > 1 else "1 gpu"),
        "clocks": rec["clocks"], "gpu_launches": int(rec["launches_per_step"] * args.steps),
        "frac_of_8TBps": rec["frac_of_8TBps"], "frac_of_measured_hbm": rec["frac_of_measured_hbm"],
        "roofline": rec["roofline"], "e2e": rec["e2e"],
        "warm_l2_ms_per_step": rec["warm_l2_ms_per_step"], "first_call_us": rec["first_call_us"],
        "plan_rebuild_us": rec["plan_rebuild_us"], "plan_rebuild_call_us": rec["plan_rebuild_call_us"],
        "plan_first_build_us": rec["plan_first_build_us"], "plan": rec["plan"],
    }
    for k in ("verify_tflops", "cpu_baseline", "parity"):
        if k in rec:
            line[k] = rec[k]
    return line


def run_single(env: Env, args):
    """--config 2|3|4|5: one workload, one line (the per-config form of the default run)."""
    n = int(args.config)
    cfg = synth.CONFIGS[n]
    if n == 4:
        cfg = cfg.scaled(k_draft=args.k)
    if args.kv == "e4m3":
        cfg = cfg.scaled(dtype="e4m3")
    wl = synth.Workload(cfg)
    num_pages = (1 << 20) if (n == 5 and args.full_pool) else None
    spk, ids = build_spork(cfg, wl, num_pages, None, env.device)
    apply_knobs(spk, args)
    rec = measure_attn(env, spk, ids, cfg, wl)
    spk.close()
    return headline_line(env, rec, cfg)


def apply_knobs(spk, args):
    if args.min_rows is not None:
        spk.set_tensor_path_min_rows(args.min_rows)
    if args.stream_k is not None:
        spk.set_stream_k(bool(args.stream_k))
    if args.many_row_variant is not None:
        spk.set_many_row_variant(args.many_row_variant)


def run_all(env: Env, args):
    """The default run: config 5 at the top level (the largest single-GPU decode config), everything
    else under per_config."""
    t_all = time.perf_counter()
    per = {}
    # ---- config 5 on the 2^20-page pool (BASELINE.json configs[4]) + its fork churn: one state ----
    cfg5 = synth.CFG5
    wl5 = synth.Workload(cfg5)
    NP5 = 1 << 20
    t0 = time.perf_counter()
    spk, ids = build_spork(cfg5, wl5, NP5, cfg5.n_seqs + 10008, env.device)
    build5 = time.perf_counter() - t0
    head = measure_attn(env, spk, ids, cfg5, wl5)
    head["state_build_seconds"] = build5
    per["churn"] = measure_churn(env, spk, ids, cfg5, wl5, NP5)
    release_all(spk)
    # ---- configs 2 and 3 ----
    for n in (2, 3):
        cfg = synth.CONFIGS[n]
        wl = synth.Workload(cfg)
        spk, ids = build_spork(cfg, wl, None, None, env.device)
        per[f"cfg{n}"] = measure_attn(env, spk, ids, cfg, wl)
        release_all(spk)
    # ---- config 4: built once with k = 16 drafts per sequence; k = 8 and k = 4 are the same state
    # rolled back by spork_truncate (the sub-streams make its values identical to a direct build) ----
    cfg16 = synth.CFG4.scaled(k_draft=16)
    wl16 = synth.Workload(cfg16)
    spk, ids = build_spork(cfg16, wl16, None, None, env.device)
    per["cfg4_k16"] = measure_attn(env, spk, ids, cfg16, wl16)
    for k in (8, 4):
        cfgk = synth.CFG4.scaled(k_draft=k)
        wlk = synth.Workload(cfgk)
        spk.truncate(ids, wlk.total_len.astype(np.int32))
        per[f"cfg4_k{k}"] = measure_attn(env, spk, ids, cfgk, wlk)
    release_all(spk)
    # ---- FP8-KV variant: configs 5 and 2 with an e4m3 cache (half the unique bytes) ----
    for n in (5, 2):
        cfg = synth.CONFIGS[n].scaled(dtype="e4m3")
        wl = synth.Workload(cfg)
        spk, ids = build_spork(cfg, wl, None, None, env.device)
        per[f"cfg{n}_e4m3kv"] = measure_attn(env, spk, ids, cfg, wl)
        release_all(spk)
    # ---- the append + decode loop on config 2, and config 1 ----
    per["loop_cfg2"] = measure_loop(env, synth.CFG2)
    per["turn_cfg4_k16"] = measure_turn(env, 16)
    per["successive_cfg3"] = measure_successive(env)
    per["layers_cfg2_x36"] = measure_layers(env, 36)
    per["cfg1"] = measure_cfg1(env)
    line = headline_line(env, head, cfg5)
    line["config"]["pool_pages"] = NP5
    line["config"]["state_build_seconds"] = build5
    line["per_config"] = per
    line["bench_seconds"] = time.perf_counter() - t_all
    return line


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
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", default="all",
                    choices=["all", "1", "2", "3", "4", "5", "churn", "loop", "turn", "successive", "layers", "d2"])
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
    ap.add_argument("--kv", default="bf16", choices=["bf16", "e4m3"],
                    help="KV storage of configs 2-5: bf16 (BASELINE.json) or the FP8-KV variant (e4m3 K/V, bf16 Q)")
    args = ap.parse_args()
    if args.config == "d2":
        run_d2(args)
        return
    if args.impl == "reference":
        # the oracle on the host cores, on this arm's headline workload (config 5 unless --config says otherwise)
        if int(os.environ.get("RANK", "0")) != 0:
            return
        n = 5 if args.config in ("all", "churn", "loop", "turn", "successive", "layers") else int(args.config)
        cfg = synth.CONFIGS[n]
        if n == 4:
            cfg = cfg.scaled(k_draft=args.k)
        print(json.dumps(reference_line(args, cfg, synth.Workload(cfg))))
        return
    env = Env(args)
    if args.config == "all":
        line = run_all(env, args)
    elif args.config == "churn":
        cfg, wl = synth.CFG5, synth.Workload(synth.CFG5)
        spk, ids = build_spork(cfg, wl, 1 << 20, cfg.n_seqs + 10008, env.device)
        rec = measure_churn(env, spk, ids, cfg, wl, 1 << 20)
        spk.close()
        line = dict(rec, metric="fork_release_churn", n_gpus=env.world, steps=args.steps,
                    warmup=max(args.warmup, 3), higher_is_better=True, scaling="weak", vs_baseline=None,
                    data="synthetic", config=dict(rec["shape"], workload=rec["workload"], l2=L2_NOTE),
                    gpu_launches=int(rec["launches_per_step"] * args.steps))
    elif args.config == "loop":
        rec = measure_loop(env, synth.CFG2)
        line = dict(rec, metric="append_decode_loop_us_per_step", n_gpus=env.world, higher_is_better=True,
                    scaling="weak", vs_baseline=None, dtype="bf16", data="synthetic",
                    config={"workload": rec["workload"], "l2": L2_NOTE})
    elif args.config in ("successive", "layers"):
        rec = measure_successive(env) if args.config == "successive" else measure_layers(env, 36)
        line = dict(rec, metric=METRIC, n_gpus=env.world, steps=args.steps, warmup=max(args.warmup, 3),
                    higher_is_better=True, scaling="weak", vs_baseline=None, data="synthetic",
                    config={"workload": rec["workload"], "l2": L2_NOTE})
    elif args.config == "turn":
        rec = measure_turn(env, args.k if args.k else 16)
        line = dict(rec, metric="partial_token_accept_turn_us", n_gpus=env.world, higher_is_better=False,
                    scaling="weak", vs_baseline=None, dtype="bf16", data="synthetic", steps=rec["turns"],
                    warmup=max(args.warmup, 3), gpu_launches=rec["kernels_per_turn"] * rec["turns"],
                    config={"workload": rec["workload"], "l2": L2_NOTE})
    elif args.config == "1":
        rec = measure_cfg1(env)
        line = dict(rec, metric=METRIC, n_gpus=env.world, steps=args.steps, warmup=max(args.warmup, 3),
                    higher_is_better=True, scaling="weak", vs_baseline=None, data="synthetic",
                    config={"workload": rec["workload"]})
    else:
        line = run_single(env, args)
    if env.rank == 0:
        print(json.dumps(line))
    env.close()


if __name__ == "__main__":
    main()
