#!/usr/bin/env python
"""bench.py -- rows/s of CA-SGD outer iterations on B200 (BASELINE.json:metric), one JSON line.

A "step" is one CA-SGD outer iteration (Alg. 1): gather s*b rows, Gram + margin,
s-step recurrence, gradient + update + shadow -- the whole hot path on one batch of s*b sampled rows.
Headline workload: BASELINE.json:configs[2] (synth dense linear regression, m = 1,000,000, n = 4096, b = 128)
at s = 32, the largest single-GPU configuration (33.5 MB of Y and 6.66e10 Gram flop per step); the other four
workloads are measured in the same run and reported under "extras". Synthetic data.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 0..4] [--s S] [--impl reference]

Timing: W warm-up steps, then the K-step region is run R times back to back (R chosen so that the timed work
lasts >= ~0.5 s: K = 20 steps of 100 us would not load the chip), each repeat bracketed by CUDA events on the
library's stream; ms_per_step = median over the repeats / K. Clocks and throttle reasons are sampled through NVML
for the whole timed region.

N > 1 (torchrun): the path does not shard at P = 1 (replicas only), so every rank
runs an independent replica on its own seeded dataset; value = all ranks' rows / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_18463_b200 import synth  # noqa: E402

METRIC = "rows/sec of CA-SGD outer iterations"
UNIT = "rows/s"
HEADLINE_WORKLOAD = 2                                 # synth-linear: the largest single-GPU config of BASELINE.json
DEFAULT_S = {0: 4, 1: 32, 2: 32, 3: 64, 4: 32}       # headline s per workload: the largest of its sweep
LOSS_NAMES = ("logistic", "linear", "poisson")


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--workload", type=int, default=HEADLINE_WORKLOAD, help="index into BASELINE.json:configs (0-based)")
    ap.add_argument("--s", type=int, default=0, help="inner steps per outer iteration (0: the workload's headline s)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--m", type=int, default=0, help="override the row count (debugging only; noted in config)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the other four workloads")
    ap.add_argument("--min-timed-s", type=float, default=0.5, help="the K-step region is repeated until this much device time")
    return ap.parse_args()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(hbm=p["hbm_gbs"], bf16_burst=p["bf16_tflops"], bf16_sustained=p["bf16_tflops_sustained"],
                    source="measured")
    return dict(hbm=6650.0, bf16_burst=1590.0, bf16_sustained=1400.0, source="fallback")   # B200_PROFILING.md


def config_dict(cfg, s, world=1):
    """The `config` object of the JSON line -- the SAME keys and values in both arms (--impl ours / reference)."""
    return dict(workload=cfg.name, m=cfg.m, n=cfg.n, b=cfg.b, s=s, rows_per_step=s * cfg.b, eta=cfg.eta,
                loss=LOSS_NAMES[cfg.loss], parallelism=f"replicas x{world}")


def step_indices(cfg, seed, n_steps, sb):
    """Row indices of n_steps consecutive outer iterations: seeded per-epoch permutations (epoch rule of
    DESIGN.md reading 12), continuing into further epochs as needed."""
    need = n_steps * sb
    chunks, have, epoch = [], 0, 0
    while have < need:
        e = synth.epoch_indices(cfg, seed, epoch)
        e = e[: (len(e) // sb) * sb]
        chunks.append(e)
        have += len(e)
        epoch += 1
    return np.ascontiguousarray(np.concatenate(chunks)[:need])


# ------------------------------------------------------------------ algorithmic work per outer step ---

def stage_work(n, s, b, pk):
    """SURVEY.md 8(d) / DESIGN.md "Roofline": algorithmic bytes and flops of each stage of one outer step."""
    sb = s * b
    gl_bytes = 2 * b * b * s * (s - 1)                    # strict block-lower G, FP32
    w = {
        "gather": dict(bytes=2 * sb * n + 8 * sb + 2 * sb * n + 4 * sb, flops=0, bound="hbm"),
        "gram": dict(bytes=2 * sb * n + gl_bytes, flops=n * b * b * s * (s - 1), bound="hbm"),
        "margin": dict(bytes=2 * sb * n + 2 * n + 4 * sb, flops=2 * sb * n, bound="hbm"),
        "recurrence": dict(bytes=gl_bytes + 16 * sb, flops=b * b * s * (s - 1), bound="hbm"),
        "gradient": dict(bytes=2 * sb * n + 10 * n + 4 * sb, flops=2 * sb * n, bound="hbm"),
    }
    g = w["gram"]
    knee = pk["bf16_sustained"] * 1e12 / (pk["hbm"] * 1e9)
    if g["bytes"] and g["flops"] / g["bytes"] > knee:
        g["bound"] = "tensor"
    return w


_NCU_ROWS = None


def ncu_metrics(lib_version, workload, s, stage):
    """Per-launch ncu --set full numbers of a stage's kernel (dram bytes, tensor-pipe active %) -- ONLY if the
    committed capture (profiles/r2_ncu_metrics.csv: lib_version,workload,s,stage,kernel,dram_read_bytes,
    dram_write_bytes,tensor_pipe_active_pct,report) was taken on this very build of the library; else None
    (a capture of another build says nothing about this one)."""
    global _NCU_ROWS
    if _NCU_ROWS is None:
        _NCU_ROWS = []
        path = os.path.join(ROOT, "profiles", "r2_ncu_metrics.csv")
        if os.path.exists(path):
            import csv
            with open(path) as f:
                _NCU_ROWS = list(csv.DictReader(f))
    for row in _NCU_ROWS:
        if (row["lib_version"] == lib_version and row["workload"] == workload and int(row["s"]) == s
                and row["stage"] == stage):
            tp = row.get("tensor_pipe_active_pct") or ""
            return dict(traffic=int(float(row["dram_read_bytes"]) + float(row["dram_write_bytes"])),
                        tensor_pipe_active_pct=float(tp) if tp else None, report=row.get("report"))
    return None


def roofline_of(stage, work, ms, pk, ncu=None):
    """achieved = algorithmic bytes (or flops) / the stage's device time. A tensor-bound stage is a tens-of-us
    kernel timed alone by its own first/last-CTA stamps, so its peak is the BURST bf16 figure; the sustained one
    is quoted beside it."""
    if ms <= 0:
        return None
    out = dict(kernel=stage, bound=work["bound"])
    if work["bound"] == "tensor":
        achieved = work["flops"] / (ms * 1e-3) / 1e12
        out.update(achieved=round(achieved, 3), peak=pk["bf16_burst"], unit="TFLOP/s", frac=round(achieved / pk["bf16_burst"], 4),
                   peak_sustained=pk["bf16_sustained"], frac_of_sustained=round(achieved / pk["bf16_sustained"], 4),
                   flops_counted="strict block-lower G (n b^2 s (s-1))" + (" + margin (2 sb n)" if "margin" in work.get("fused", []) else ""))
    else:
        achieved = work["bytes"] / (ms * 1e-3) / 1e9
        out.update(achieved=round(achieved, 3), peak=pk["hbm"], unit="GB/s", frac=round(achieved / pk["hbm"], 4))
    out.update(traffic=ncu["traffic"] if ncu else None, peak_source=pk["source"], avg_launch_ms=round(ms, 6))
    if ncu and ncu.get("tensor_pipe_active_pct") is not None:
        out["tensor_pipe_active_pct"] = ncu["tensor_pipe_active_pct"]
    return out


# ------------------------------------------------------------------------------------- clocks ---

class ClockSampler:
    """SM clock, power and throttle reasons DURING the timed regions, through NVML (nvidia_ml_py) from a thread
    started at process start; nvidia-smi once as a fallback. Samples are kept only while `active` is set."""
    REASONS = (("hw_slowdown", 0x8), ("hw_thermal_slowdown", 0x40), ("sw_thermal_slowdown", 0x20), ("sw_power_cap", 0x4))

    def __init__(self, index, period_s=0.005):
        self.index, self.period = index, period_s
        self.sm, self.power, self.reasons, self.sm_all = [], [], set(), []
        self.active = False
        self.stop_flag = False
        self.max_mhz = None
        self.h = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            phys = index
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            if vis:
                tok = vis.split(",")[index].strip()
                if tok.isdigit():
                    phys = int(tok)
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.h = None
        self.t = threading.Thread(target=self._run, daemon=True)
        self.t.start()

    def _sample(self):
        nv = self.nv
        mhz = float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
        self.sm_all.append(mhz)
        if not self.active:
            return
        self.sm.append(mhz)
        try:
            self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            bits = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h) if hasattr(nv, "nvmlDeviceGetCurrentClocksEventReasons") \
                else nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
            for nm, bit in self.REASONS:
                if bits & bit:
                    self.reasons.add(nm)
        except Exception:
            pass

    def _run(self):
        while not self.stop_flag:
            if self.h is not None:
                try:
                    self._sample()
                except Exception:
                    pass
            time.sleep(self.period)

    def window(self, on):
        if on and self.h is not None:
            try:
                self.active = True
                self._sample()                          # at least one sample per window, however short
            except Exception:
                pass
        self.active = on

    def _smi_once(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        try:
            out = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={q}", "--format=csv,noheader,nounits"],
                                 capture_output=True, text=True, timeout=20).stdout.strip().splitlines()[0]
            parts = [t.strip() for t in out.split(",")]
            names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
            return dict(sm_mhz=float(parts[0]), sm_max_mhz=float(parts[1]),
                        reasons=[nm for nm, v in zip(names, parts[3:7]) if v.lower().startswith("active")], samples=1,
                        source="nvidia-smi after the timed region (NVML unavailable)")
        except Exception:
            return None

    def stop(self):
        self.stop_flag = True
        self.t.join(timeout=2)
        if self.sm:
            return dict(sm_mhz=statistics.median(self.sm), sm_min_mhz=min(self.sm), sm_max_mhz=self.max_mhz,
                        power_w_max=max(self.power) if self.power else None, reasons=sorted(self.reasons),
                        samples=len(self.sm), source="NVML, sampled every 5 ms during the timed regions")
        smi = self._smi_once()
        if smi:
            return smi
        return dict(sm_mhz=None, sm_max_mhz=self.max_mhz, reasons=[], samples=0, source="no sampler available")


# ------------------------------------------------------------------------------ oracle legs ---

def _compact_rows(A_dev, y_dev, seg):
    """Only the rows an index segment touches are brought to the host: compact BF16 bits, labels, remapped indices."""
    uniq, inv = np.unique(seg, return_inverse=True)
    sel = torch.from_numpy(uniq.astype(np.int64)).to(A_dev.device)
    A_bits = A_dev[sel].contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
    yy = y_dev[sel].cpu().numpy()
    return A_bits, yy, np.ascontiguousarray(inv.astype(np.int32))


def oracle_rows_per_s(cfg, s, A_dev, y_dev, idx_np, seed, budget_s=10.0, form="gram"):
    """Time the oracle as it stands, on this host's cores, on the first steps of the same index stream: form "gram" =
    O1 (Alg. 1 as the GPU computes it: full FP64 Gram), form "seq" = O2 (s sequential SGD steps, PAPER.md:L176 -- the
    sensible CPU algorithm at P = 1). Returns rows/s, steps, seconds, threads."""
    import oracle
    sb = s * cfg.b

    def run(lo, hi, x):
        A_bits, yy, local = _compact_rows(A_dev, y_dev, idx_np[lo * sb: hi * sb])
        t0 = time.perf_counter()
        x = oracle.train(A_bits, yy, local, x, s, cfg.b, cfg.eta, cfg.loss, shadow=True, form=form)
        return time.perf_counter() - t0, x

    t1, x = run(0, 1, np.zeros(cfg.n))
    steps = int(max(1, min(budget_s / max(t1, 1e-6), 20000)))
    if steps + 1 > len(idx_np) // sb:                    # the same seeded stream, continued
        idx_np = step_indices(cfg, seed, steps + 1, sb)
    t, _ = run(1, 1 + steps, x)
    return steps * sb / t, steps, t, oracle.num_threads()


def main_reference(args, cfg, s):
    """--impl reference: the oracle (test infrastructure) timed on the host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    sb = s * cfg.b
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    ds = synth.make_dataset(cfg, seed=42, device=dev)
    total = args.warmup + args.steps
    idx = step_indices(cfg, 42, total + 1, sb)
    import oracle
    # bound each step so that the whole run ends within a few minutes: the first s_eff blocks of every step
    s_eff = s
    while s_eff > 1 and 2.0 * (s_eff * cfg.b) ** 2 * cfg.n * total > 2.0e11:
        s_eff //= 2
    sb_eff = s_eff * cfg.b
    x = np.zeros(cfg.n)
    times = []
    for h in range(total):
        A_bits, yy, local = _compact_rows(ds.X_bf16, ds.y, idx[h * sb: h * sb + sb_eff])
        t0 = time.perf_counter()
        ref = oracle.outer_step_gram(A_bits, yy, local, x, s_eff, cfg.b, cfg.eta, cfg.loss, shadow=True)
        x = ref.x_out
        dt = time.perf_counter() - t0
        if h >= args.warmup:
            times.append(dt)
    t = sum(times)
    value = len(times) * sb_eff / t
    sample = (f"oracle O1 (FP64 Gram form), {len(times)} outer steps of s={s_eff} x b={cfg.b} rows"
              + ("" if s_eff == s else f" (bounded: the workload's s={s} cut to its first {s_eff} blocks per step)"))
    line = dict(impl="reference", metric=METRIC, value=value, unit=UNIT, n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=1e3 * t / len(times), higher_is_better=True, scaling="weak",
                vs_baseline=None, dtype="f64", data="synthetic", config=config_dict(cfg, s, max(1, args.gpus)),
                cpu_baseline=dict(value=value, unit=UNIT, cores=oracle.num_threads(), kind="oracle", sample=sample),
                e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))


# --------------------------------------------------------------------------------- our arm ---

def replica_seed(rank):
    """Replicas only: rank r trains its own dataset, drawn from seed 42 + r."""
    return 42 + rank


def max_over_ranks(values, dist, device):
    """Element-wise MAX over ranks of a list of floats (the timing rule: the slowest rank sets the time)."""
    if dist is None:
        return [float(v) for v in values]
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.tolist()]


def aggregate_rows_per_s(world, steps, sb, ms):
    """Whole-job rows/s: every rank processed steps*sb rows in (max-over-ranks) ms."""
    return world * steps * sb / (ms * 1e-3)


def time_call(stream, fn):
    """Device milliseconds of fn() on the library's stream (CUDA events recorded on that very stream)."""
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    fn()
    e1.record(stream)
    stream.synchronize()
    return e0.elapsed_time(e1)


def prime_graphs(cg, cfg, seed, s, sb):
    """Make the library capture and instantiate the graph lengths it replays (64 steps, and the 9-step remainder of this
    call as a graph of its own; a timed call's own remainder length is captured by the untimed sizing call), on a scratch x."""
    idx_p = torch.from_numpy(step_indices(cfg, seed, 73, sb)).cuda()
    cg.outer_steps(idx_p, torch.zeros(cfg.n, device="cuda"), s, cfg.b, cfg.eta, n_steps=73)
    cg.sync()


def timed_steps(cg, cfg, s, idx_d, x, K, W, stream, min_timed_s, clocks=None, max_repeats=400):
    """W warm-up steps, then R repeats of exactly K steps each (R so that the timed work lasts >= min_timed_s),
    consecutive segments of one index stream; returns the per-repeat device times (ms) and R."""
    sb = s * cfg.b
    cg.outer_steps(idx_d[: W * sb], x, s, cfg.b, cfg.eta, n_steps=W)
    cg.sync()
    have = idx_d.numel() // sb - W                         # steps of indices available after the warm-up
    t_first = time_call(stream, lambda: cg.outer_steps(idx_d[W * sb:], x, s, cfg.b, cfg.eta, n_steps=K))
    R = int(min(max_repeats, max(5, min_timed_s * 1e3 / max(t_first, 1e-3))))
    if clocks:
        clocks.window(True)
    times = []
    l0 = cg.launch_count()
    for rep in range(R):
        lo = W + ((rep * K) % max(1, have - K + 1))        # wraps around the stream when it is shorter than R * K steps
        times.append(time_call(stream, lambda: cg.outer_steps(idx_d[lo * sb:], x, s, cfg.b, cfg.eta, n_steps=K)))
    launches = (cg.launch_count() - l0) / R               # kernels of the library per K-step region
    if clocks:
        clocks.window(False)
    return times, R, launches


def stage_report(cg, binding, cfg, s, idx_d, x, W, Kp, pk, lib_version, overlap=None):
    """Per-stage device times measured INSIDE the CUDA-graph replays (CASGD_OPT_STAMPS: first-CTA start after the PDL
    wait to last-CTA end, %globaltimer), the algorithmic work of each stage and its roofline fraction."""
    sb = s * cfg.b
    if overlap is not None:
        cg.set_option(binding.OPT_OVERLAP, overlap)
    cg.set_option(binding.OPT_STAMPS, 1)
    prime_graphs(cg, cfg, 7, s, sb)                         # the option rebuilt the graphs
    cg.stage_times(reset=True)
    cg.outer_steps(idx_d[W * sb:], x, s, cfg.b, cfg.eta, n_steps=Kp)
    st = cg.stage_times(reset=True)
    cg.set_option(binding.OPT_STAMPS, 0)
    if overlap is not None:
        cg.set_option(binding.OPT_OVERLAP, 2)
    work = stage_work(cfg.n, s, cfg.b, pk)
    # fused stages: a stage with no launch of its own ran inside its neighbour (n <= 64: gather inside the Gram
    # kernel; small steps: gradient + update inside the recurrence kernel; s = 1: l' inside the margin kernel)
    # (not pipelined: r rides in the Gram kernel's B operand)
    for absent, host in (("margin", "gram"), ("gather", "gram"), ("gradient", "recurrence"), ("recurrence", "gram")):
        if st[absent][1] == 0 and st[host][1] > 0:
            work[host]["bytes"] += work[absent]["bytes"]
            work[host]["flops"] += work[absent]["flops"]
            work[host]["fused"] = work[host].get("fused", []) + [absent]
    stages = {}
    launched = [k for k in work if st[k][1] > 0]
    if launched == ["gram"] and st["gram"][1] < Kp / 2:
        # mini_step.cu: ALL iterations of the call in one persistent one-CTA launch (gather -> Gram -> recurrence ->
        # update, x resident in shared memory): one stage, its time divided by the iterations it ran
        per_step = st["gram"][0] / Kp
        wk = dict(bytes=sum(w["bytes"] for w in work.values()), flops=sum(w["flops"] for w in work.values()), bound="hbm")
        rl = roofline_of("fused_step", wk, per_step, pk, None)
        rl["note"] = "latency-bound by design: one CTA, %d iterations per launch" % Kp
        stages["fused_step"] = dict(ms_per_step=round(per_step, 6), launches_per_step=st["gram"][1] / Kp, roofline=rl,
                                    alg_bytes=wk["bytes"], alg_flops=wk["flops"])
        return stages
    for name, wk in work.items():
        tot_ms, cnt = st[name]
        if not cnt:
            continue
        per_launch = tot_ms / cnt
        rl = roofline_of(name, wk, per_launch, pk, ncu_metrics(lib_version, cfg.name, s, name))
        if rl and name == "recurrence" and s > 1:
            rl["chain"] = dict(hops=s - 1, kernel_us_per_hop=round(per_launch * 1e3 / (s - 1), 3),
                               note="latency chain of s - 1 dependent hops (one distributed-shared-memory broadcast each)")
        if rl and wk.get("fused"):
            rl["includes"] = wk["fused"]
        stages[name] = dict(ms_per_step=round(per_launch, 6), launches_per_step=cnt / Kp, roofline=rl,
                            alg_bytes=wk["bytes"], alg_flops=wk["flops"])
    return stages


def gemv_report(cg, binding, cfg, x, pk, lib_version, stream, reps=5):
    """casgd_loss: the pure streaming GEMV over all of A (BASELINE metric's "GEMV HBM GB/s")."""
    cg.loss(x)
    cg.set_option(binding.OPT_PROFILE, 1)
    cg.stage_times(reset=True)
    for _ in range(reps):
        cg.loss(x)
    loss_ms = cg.stage_times(reset=True)["loss"][0] / reps
    cg.set_option(binding.OPT_PROFILE, 0)
    loss_bytes = 2 * cfg.m * cfg.n + 4 * cfg.m
    ncu = ncu_metrics(lib_version, cfg.name, 0, "loss")
    return dict(kernel="casgd_loss", bound="hbm", achieved=round(loss_bytes / loss_ms / 1e6, 2), peak=pk["hbm"],
                unit="GB/s", frac=round(loss_bytes / loss_ms / 1e6 / pk["hbm"], 4), avg_call_ms=round(loss_ms, 5),
                traffic=ncu["traffic"] if ncu else None, peak_source=pk["source"])


def run_workload(args, cfg, s, binding, pk, dist, world, rank, stream, clocks, full):
    """Everything measured on one workload. full: the headline (e2e, on-device sampling, sweep, FP32 baseline,
    oracle legs); else the light set for `extras` (rows/s, stages, GEMV)."""
    lib_version = binding.version()
    sb = s * cfg.b
    seed = replica_seed(rank)                            # independent replicas
    ds = synth.make_dataset(cfg, seed=seed, device="cuda")
    K, W = args.steps, max(args.warmup, 3)
    n_idx_steps = W + max(K, min(8 * K, 4096), min(max(K, 64), 256))   # (the stage report replays min(max(K, 64), 256) steps)
    idx_np = step_indices(cfg, seed, n_idx_steps, sb)
    out = {}
    with torch.cuda.stream(stream):                      # every allocation / fill below is ordered on the library's stream
        idx_d = torch.from_numpy(idx_np).cuda()
        cg = binding.Casgd(ds.X_bf16, ds.y, cfg.loss, stream=stream)
        x = torch.zeros(cfg.n, device="cuda")
        stream.synchronize()
        # graph instantiation is not a step: casgd_outer_steps captures its CUDA graphs (64 steps, and one per remainder length) on first use
        prime_graphs(cg, cfg, seed, s, sb)
        if dist:
            dist.barrier()
        torch.cuda.synchronize()
        times, R, launches_per_region = timed_steps(cg, cfg, s, idx_d, x, K, W, stream, args.min_timed_s, clocks)
        torch.cuda.synchronize()
        if dist:
            dist.barrier()
        ms_med, ms_min, ms_max = max_over_ranks([statistics.median(times), min(times), max(times)], dist, "cuda")
        out.update(ms=ms_med, ms_min=ms_min, ms_max=ms_max, repeats=R, launches=launches_per_region,
                   final_loss=cg.loss(x), sb=sb)
        Kp = min(max(K, 64), 256)
        out["stages"] = stage_report(cg, binding, cfg, s, idx_d, x, W, Kp, pk, lib_version)
        # ... and each kernel with the chip to itself (CASGD_OPT_OVERLAP = 0: kernels strictly in sequence, the margin
        # fused into the Gram): what the kernels can do, as opposed to what they get beside one another
        out["stages_alone"] = stage_report(cg, binding, cfg, s, idx_d, x, W, Kp, pk, lib_version, overlap=0)
        out["gemv"] = gemv_report(cg, binding, cfg, x, pk, lib_version, stream)
        if not full:
            cg.close()
            del ds
            return out

        # ---- the same K steps with the indices drawn on the device (Alg. 1 line 1 as the paper states it: i.i.d. with
        # replacement, Philox4x32-10; casgd_outer_steps_sampled) -- no index buffer at all
        xs_ = torch.zeros(cfg.n, device="cuda")
        cg.outer_steps_sampled(xs_, s, cfg.b, cfg.eta, n_steps=W, seed=seed, first_step=0)
        reps = max(3, min(R, 20))
        ts = [time_call(stream, lambda: cg.outer_steps_sampled(xs_, s, cfg.b, cfg.eta, n_steps=K, seed=seed, first_step=W + i * K))
              for i in range(reps)]
        out["sampled_ms"], = max_over_ranks([statistics.median(ts)], dist, "cuda")

        # ---- end to end through the C ABI with HOST buffers: every step copies its indices and x in, x out
        idx_h = torch.from_numpy(idx_np[W * sb:]).pin_memory()
        x_h = torch.zeros(cfg.n).pin_memory()
        Ke = min(idx_h.numel() // sb, max(K, 500))
        cg.outer_steps_host(idx_h[: sb], x_h, s, cfg.b, cfg.eta, n_steps=1)
        x_h.zero_()
        if dist:
            dist.barrier()
        clocks.window(True)
        t0 = time.perf_counter()
        for h in range(Ke):
            cg.outer_steps_host(idx_h[h * sb:(h + 1) * sb], x_h, s, cfg.b, cfg.eta, n_steps=1)
        e2e_s = time.perf_counter() - t0
        # the same with one call per 64 steps (indices of 64 steps copied at once, x in/out once per call); the graph of the
        # last, shorter call is captured by an untimed call first
        if Ke % 64 > 1:
            cg.outer_steps_host(idx_h[: (Ke % 64) * sb], x_h, s, cfg.b, cfg.eta, n_steps=Ke % 64)
        x_h.zero_()
        t0 = time.perf_counter()
        done = 0
        while done < Ke:
            c = min(64, Ke - done)
            cg.outer_steps_host(idx_h[done * sb:(done + c) * sb], x_h, s, cfg.b, cfg.eta, n_steps=c)
            done += c
        e2e64_s = time.perf_counter() - t0
        clocks.window(False)
        e2e_s, e2e64_s = max_over_ranks([e2e_s, e2e64_s], dist, "cuda")
        out.update(e2e_s=e2e_s, e2e64_s=e2e64_s, Ke=Ke)

        # ---- in-library FP32 s = 1 SGD baseline (Recipe A) and the s sweep, same index stream
        sweep = {}
        if not args.no_sweep:
            Ks = max(50, min(K * s, 4000))
            idx_s = torch.from_numpy(step_indices(cfg, seed, Ks, cfg.b)).cuda()
            xs = torch.zeros(cfg.n, device="cuda")
            cg.sgd_steps_fp32(idx_s[: 10 * cfg.b], xs, cfg.b, cfg.eta, n_steps=10)
            ms32 = time_call(stream, lambda: cg.sgd_steps_fp32(idx_s, xs, cfg.b, cfg.eta, n_steps=Ks))
            sweep["fp32_sgd_s1"] = dict(rows_per_s=Ks * cfg.b / (ms32 * 1e-3), ms_per_step=ms32 / Ks)
            for s2 in cfg.s_list:
                sb2 = s2 * cfg.b
                k2 = max(20, min(2000, (K * sb) // sb2))
                idx2 = torch.from_numpy(step_indices(cfg, seed, 4 * k2 + 5, sb2)).cuda()
                prime_graphs(cg, cfg, seed, s2, sb2)
                x2 = torch.zeros(cfg.n, device="cuda")
                t2, R2, _ = timed_steps(cg, cfg, s2, idx2, x2, k2, 5, stream, 0.1, None, 50)
                ms2 = statistics.median(t2)
                sweep[f"s{s2}"] = dict(rows_per_s=k2 * sb2 / (ms2 * 1e-3), ms_per_outer_step=ms2 / k2, repeats=R2)
                if s2 != s:
                    sweep[f"s{s2}"]["stages"] = stage_report(cg, binding, cfg, s2, idx2, x2, 5, min(k2, 128), pk, lib_version)
        out["sweep"] = sweep

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v1, st1, t1, cores = oracle_rows_per_s(cfg, s, ds.X_bf16, ds.y, idx_np, seed, 10.0, "gram")
        v2, st2, t2, _ = oracle_rows_per_s(cfg, s, ds.X_bf16, ds.y, idx_np, seed, 5.0, "seq")
        out["cpu_baseline"] = dict(
            value=v1, unit=UNIT, cores=cores, kind="oracle",
            sample=f"oracle O1 (FP64 Gram form, what the GPU computes) on the first {st1} outer steps (s={s}, b={cfg.b}) "
                   f"of the same index stream, {t1:.1f} s",
            sequential_form=dict(value=v2, unit=UNIT, cores=cores, kind="oracle",
                                 sample=f"oracle O2 (s sequential FP64 SGD steps, PAPER.md:L176: the sensible CPU algorithm "
                                        f"at P = 1) on the first {st2} outer steps, {t2:.1f} s"))
    cg.close()
    del ds
    return out


def main_ours(args, cfg, s):
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU path)"
    torch.cuda.set_device(local)
    clocks = ClockSampler(local)                         # started at process start; samples kept during timed windows
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2606_18463_b200 import build
    if rank == 0:
        build.build()
    if dist:
        dist.barrier()
    from paper_2606_18463_b200 import binding
    pk = peaks()
    stream = torch.cuda.Stream()
    K, W = args.steps, max(args.warmup, 3)
    sb = s * cfg.b

    r = run_workload(args, cfg, s, binding, pk, dist, world, rank, stream, clocks, full=True)

    extras = {}
    if not args.no_extras and not args.m:
        for wi in range(len(synth.CONFIGS)):
            if wi == args.workload:
                continue
            cfg2, s2 = synth.config(wi), DEFAULT_S[wi]
            torch.cuda.empty_cache()
            e = run_workload(args, cfg2, s2, binding, pk, dist, world, rank, stream, None, full=False)
            extras[cfg2.name] = dict(config=config_dict(cfg2, s2, world), value=aggregate_rows_per_s(world, K, e["sb"], e["ms"]),
                                     unit=UNIT, ms_per_step=e["ms"] / K, repeats=e["repeats"], final_loss=e["final_loss"],
                                     stages=e["stages"], stages_alone=e["stages_alone"], gemv=e["gemv"])
    clk = clocks.stop()

    stages = r["stages"]
    # the roofline object: the dominant kernel of the headline step (for synth-linear: the tcgen05 Gram, tensor-bound)
    dominant = max(stages, key=lambda k: stages[k]["ms_per_step"])
    roofline = dict(stages[dominant]["roofline"])
    alone = r["stages_alone"].get(dominant)
    if alone:
        # the same kernel with the chip to itself (kernels in sequence): its own quality, next to what it gets when the
        # schedule runs it on part of the SMs beside the latency-bound chain
        roofline["alone"] = dict(achieved=alone["roofline"]["achieved"], frac=alone["roofline"]["frac"],
                                 avg_launch_ms=alone["roofline"]["avg_launch_ms"], includes=alone["roofline"].get("includes"))
        roofline["note"] = ("as scheduled: the pipelined graph runs this kernel on part of the SMs, sharing L2 with the chain "
                            "of the previous iteration; `alone` is the same kernel in a strictly sequential graph")
    ms, Ke = r["ms"], r["Ke"]
    config = config_dict(cfg, s, world)
    notes = dict(l2="inputs larger than L2: rows are gathered at random from A "
                    f"({cfg.m * max(cfg.n, 8) * 2 / 1e6:.0f} MB)" if cfg.m * cfg.n * 2 > 126e6 else
                    "A fits in L2; not flushed (the step's own working set is L2-resident by design)",
                 timing=f"median of {r['repeats']} back-to-back repeats of the K = {K}-step region (CUDA events on the library's "
                        f"stream around each); min {r['ms_min'] / K:.6f} / max {r['ms_max'] / K:.6f} ms per step",
                 stage_times="inside the CUDA-graph replays: first-CTA start (after the PDL wait) to last-CTA end, %globaltimer",
                 schedule="pipelined (CASGD_OPT_OVERLAP = 2): gather + Gram of outer iteration t + 1 run on a side branch of the "
                          "graph beside margin -> recurrence -> update of iteration t, so stage times OVERLAP and do not add "
                          "up to ms_per_step; the Gram runs on the SMs the chain leaves it and shares L2 with it",
                 outer_iters_per_s=K / (ms * 1e-3), final_loss=r["final_loss"], lib=binding.version())
    line = dict(metric=METRIC, value=aggregate_rows_per_s(world, K, sb, ms), unit=UNIT, n_gpus=world, steps=K, warmup=W,
                ms_per_step=ms / K, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="bf16 in / f32 accumulate",
                data="synthetic", config=config, notes=notes, clocks=clk,
                e2e=dict(value=aggregate_rows_per_s(world, Ke, sb, r["e2e_s"] * 1e3), unit=UNIT,
                         h2d_bytes_per_step=sb * 4 + cfg.n * 4, d2h_bytes_per_step=cfg.n * 4, steps=Ke,
                         batched64=dict(value=aggregate_rows_per_s(world, Ke, sb, r["e2e64_s"] * 1e3),
                                        h2d_bytes_per_step=sb * 4 + cfg.n * 4 / 64, d2h_bytes_per_step=cfg.n * 4 / 64)),
                gpu_launches=int(round(r["launches"])),
                sampled_on_device=dict(value=aggregate_rows_per_s(world, K, sb, r["sampled_ms"]), unit=UNIT,
                                       ms_per_step=r["sampled_ms"] / K,
                                       sampler="Philox4x32-10, i.i.d. with replacement (PAPER.md:L111)"),
                roofline=roofline, stages=stages, stages_alone=r["stages_alone"], gemv=r["gemv"], sweep=r.get("sweep", {}), extras=extras)
    if "cpu_baseline" in r:
        line["cpu_baseline"] = r["cpu_baseline"]
    if rank == 0:
        print(json.dumps(line))
    if dist:
        dist.destroy_process_group()


def main():
    args = parse_args()
    cfg = synth.config(args.workload, m=args.m or None)
    s = args.s or DEFAULT_S[args.workload]
    if args.impl == "reference":
        main_reference(args, cfg, s)
    else:
        main_ours(args, cfg, s)


if __name__ == "__main__":
    main()
