#!/usr/bin/env python
"""bench.py -- rows/s of CA-SGD outer iterations on B200 (BASELINE.json:metric), one JSON line.

A "step" is one CA-SGD outer iteration (Alg. 1): gather s*b rows, Gram + margin,
s-step recurrence, gradient + update + shadow -- the whole hot path on one batch of s*b sampled rows.
Default workload: BASELINE.json:configs[1] (SUSY-shaped logistic, m = 5,000,000, n = 18, b = 64) at full
size, synthetic (the LIBSVM file is not available).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 0..4] [--s S] [--impl reference]

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
import tempfile
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_18463_b200 import synth  # noqa: E402

METRIC = "rows/sec of CA-SGD outer iterations"
UNIT = "rows/s"
DEFAULT_S = {0: 4, 1: 32, 2: 32, 3: 64, 4: 32}       # headline s per workload: the largest of its sweep


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--workload", type=int, default=1, help="index into BASELINE.json:configs (0-based)")
    ap.add_argument("--s", type=int, default=0, help="inner steps per outer iteration (0: the workload's headline s)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--m", type=int, default=0, help="override the row count (debugging only; noted in config)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sweep", action="store_true")
    return ap.parse_args()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(hbm=p["hbm_gbs"], bf16_burst=p["bf16_tflops"], bf16_sustained=p["bf16_tflops_sustained"],
                    source="measured")
    return dict(hbm=6650.0, bf16_burst=1590.0, bf16_sustained=1400.0, source="fallback")   # B200_PROFILING.md


def step_indices(cfg, seed, n_steps, sb):
    """Row indices of n_steps consecutive outer iterations: seeded per-epoch permutations (epoch rule of
    DESIGN.md reading 16), continuing into further epochs as needed."""
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
        "gram": dict(bytes=2 * sb * n + gl_bytes + 4 * sb, flops=n * b * b * s * (s - 1) + 2 * sb * n, bound="hbm"),
        "recurrence": dict(bytes=gl_bytes + 16 * sb, flops=b * b * s * (s - 1), bound="hbm"),
        "gradient": dict(bytes=2 * sb * n + 10 * n + 4 * sb, flops=2 * sb * n, bound="hbm"),
    }
    g = w["gram"]
    knee = pk["bf16_sustained"] * 1e12 / (pk["hbm"] * 1e9)
    if g["bytes"] and g["flops"] / g["bytes"] > knee:
        g["bound"] = "tensor"
    return w


def ncu_traffic(workload, s, stage):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of a stage's kernel, from the committed ncu
    --set full summaries (profiles/r1_traffic.csv: workload,s,stage,kernel,dram_read_bytes,dram_write_bytes,report)."""
    path = os.path.join(ROOT, "profiles", "r1_traffic.csv")
    if not os.path.exists(path):
        return None
    import csv
    with open(path) as f:
        for row in csv.DictReader(f):
            if row["workload"] == workload and int(row["s"]) == s and row["stage"] == stage:
                return int(float(row["dram_read_bytes"]) + float(row["dram_write_bytes"]))
    return None


def roofline_of(stage, work, ms, pk, traffic=None):
    if ms <= 0:
        return None
    if work["bound"] == "tensor":
        achieved = work["flops"] / (ms * 1e-3) / 1e12
        peak, unit = pk["bf16_sustained"], "TFLOP/s"
    else:
        achieved = work["bytes"] / (ms * 1e-3) / 1e9
        peak, unit = pk["hbm"], "GB/s"
    return dict(kernel=stage, bound=work["bound"], achieved=round(achieved, 3), peak=peak, unit=unit,
                frac=round(achieved / peak, 4), traffic=traffic, peak_source=pk["source"],
                avg_launch_ms=round(ms, 6))


# ------------------------------------------------------------------------------------- clocks ---

class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "20"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = dict(sm_mhz=None, sm_max_mhz=None, reasons=[])
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.f.read().splitlines():
            parts = [t.strip() for t in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
            except ValueError:
                continue
            for nm, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out = dict(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))
        return out


# ------------------------------------------------------------------------------ oracle legs ---

def oracle_rows_per_s(cfg, s, A_dev, y_dev, idx_np, seed, budget_s=12.0, max_steps=None):
    """Time oracle O1 (the Gram form, what the GPU computes) as it stands, on this host's cores, on the
    first steps of the same index stream. Only the rows those steps touch are brought to the host."""
    import oracle
    sb = s * cfg.b
    x = np.zeros(cfg.n)

    def run(lo, hi):
        nonlocal x
        seg = idx_np[lo * sb: hi * sb]
        uniq, inv = np.unique(seg, return_inverse=True)
        rows = A_dev[torch.from_numpy(uniq.astype(np.int64)).to(A_dev.device)].contiguous()
        A_bits = rows.view(torch.int16).cpu().numpy().view(np.uint16)
        yy = y_dev[torch.from_numpy(uniq.astype(np.int64)).to(y_dev.device)].cpu().numpy()
        local = inv.astype(np.int32)
        t0 = time.perf_counter()
        for h in range(hi - lo):
            ref = oracle.outer_step_gram(A_bits, yy, np.ascontiguousarray(local[h * sb:(h + 1) * sb]), x, s, cfg.b,
                                         cfg.eta, cfg.loss, shadow=True)
            x = ref.x_out
        return time.perf_counter() - t0

    t1 = run(0, 1)
    steps = int(max(1, budget_s / max(t1, 1e-6)))
    if max_steps:
        steps = min(steps, max_steps)
    if steps + 1 > len(idx_np) // sb:                    # the same seeded stream, continued
        idx_np = step_indices(cfg, seed, steps + 1, sb)
    t = run(1, 1 + steps)
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
    # bound each step so that the whole run ends within a few minutes
    per_step_flop = 2.0 * sb * sb * cfg.n + 6.0 * sb * cfg.n
    frac_blocks = s
    while frac_blocks > 1 and 2.0 * (frac_blocks * cfg.b) ** 2 * cfg.n * total > 2.0e11:
        frac_blocks //= 2
    s_eff = frac_blocks
    sb_eff = s_eff * cfg.b
    x = np.zeros(cfg.n)
    times = []
    for h in range(total):
        seg = idx[h * sb: h * sb + sb_eff]
        uniq, inv = np.unique(seg, return_inverse=True)
        sel = torch.from_numpy(uniq.astype(np.int64)).to(ds.X_bf16.device)
        A_bits = ds.X_bf16[sel].contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
        yy = ds.y[sel].cpu().numpy()
        t0 = time.perf_counter()
        ref = oracle.outer_step_gram(A_bits, yy, inv.astype(np.int32), x, s_eff, cfg.b, cfg.eta, cfg.loss, shadow=True)
        x = ref.x_out
        dt = time.perf_counter() - t0
        if h >= args.warmup:
            times.append(dt)
    t = sum(times)
    value = len(times) * sb_eff / t
    sample = (f"oracle O1 (FP64 Gram form), {len(times)} outer steps of s={s_eff} x b={cfg.b} rows"
              + ("" if s_eff == s else f" (bounded: the workload's s={s} cut to {s_eff} blocks per step)"))
    line = dict(impl="reference", metric=METRIC, value=value, unit=UNIT, n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=1e3 * t / len(times), higher_is_better=True, scaling="weak",
                vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=cfg.name, m=cfg.m, n=cfg.n, b=cfg.b, s=s, eta=cfg.eta, loss=cfg.loss,
                            per_step_flop_full=per_step_flop),
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


def time_steps(binding, cg, idx_d, x, s, b, eta, n_steps, stream):
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        e0.record(stream)
        cg.outer_steps(idx_d, x, s, b, eta, n_steps=n_steps)
        e1.record(stream)
    stream.synchronize()
    return e0.elapsed_time(e1)


def prime_graphs(cg, cfg, seed, s, sb):
    """Make the library capture and instantiate every graph length it replays (64 + 8 + 1 steps), on a scratch x."""
    idx_p = torch.from_numpy(step_indices(cfg, seed, 73, sb)).cuda()
    cg.outer_steps(idx_p, torch.zeros(cfg.n, device="cuda"), s, cfg.b, cfg.eta, n_steps=73)
    cg.sync()
    cg.invalidate_shadow()


def main_ours(args, cfg, s):
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU path)"
    torch.cuda.set_device(local)
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
    sb = s * cfg.b
    seed = replica_seed(rank)                            # independent replicas
    ds = synth.make_dataset(cfg, seed=seed, device="cuda")
    K, W = args.steps, max(args.warmup, 3)
    idx_np = step_indices(cfg, seed, W + K, sb)
    idx_d = torch.from_numpy(idx_np).cuda()
    stream = torch.cuda.Stream()
    out = {}
    with torch.cuda.stream(stream):
        cg = binding.Casgd(ds.X_bf16, ds.y, cfg.loss, stream=stream)
    x = torch.zeros(cfg.n, device="cuda")
    torch.cuda.synchronize()

    # ---- graph instantiation is not a step: casgd_outer_steps captures its 64 / 8 / 1-step CUDA graphs on first use,
    # so run 73 steps on a scratch iterate first (untimed, x untouched), then the W warm-up steps proper
    prime_graphs(cg, cfg, seed, s, sb)
    # ---- warm-up, then the timed region: K outer steps, device-resident inputs
    cg.outer_steps(idx_d[: W * sb], x, s, cfg.b, cfg.eta, n_steps=W)
    cg.sync()
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    clocks = ClockSampler(local)
    l0 = cg.launch_count()
    ms = time_steps(binding, cg, idx_d[W * sb:], x, s, cfg.b, cfg.eta, K, stream)
    torch.cuda.synchronize()
    launches = cg.launch_count() - l0
    if dist:
        dist.barrier()
    ms, = max_over_ranks([ms], dist, "cuda")
    cg.sync()
    F_after = cg.loss(x)

    # ---- the same K steps with the indices drawn on the device (Alg. 1 line 1 as the paper states it: i.i.d. with
    # replacement, Philox4x32-10; casgd_outer_steps_sampled) -- no index buffer at all
    xs_ = torch.zeros(cfg.n, device="cuda")
    cg.outer_steps_sampled(xs_, s, cfg.b, cfg.eta, n_steps=W, seed=seed, first_step=0)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        e0.record(stream)
        cg.outer_steps_sampled(xs_, s, cfg.b, cfg.eta, n_steps=K, seed=seed, first_step=W)
        e1.record(stream)
    stream.synchronize()
    sampled_ms, = max_over_ranks([e0.elapsed_time(e1)], dist, "cuda")
    cg.invalidate_shadow()

    # ---- end to end through the C ABI with HOST buffers: every step copies its indices and x in, x out
    idx_h = torch.from_numpy(idx_np[W * sb:]).pin_memory()
    x_h = torch.zeros(cfg.n).pin_memory()
    Ke = min(K, 2000)
    cg.outer_steps_host(idx_h[: sb], x_h, s, cfg.b, cfg.eta, n_steps=1)
    if dist:
        dist.barrier()
    t0 = time.perf_counter()
    for h in range(Ke):
        cg.outer_steps_host(idx_h[h * sb:(h + 1) * sb], x_h, s, cfg.b, cfg.eta, n_steps=1)
    e2e_s = time.perf_counter() - t0
    # the same with one call per 64 steps (indices of 64 steps copied at once, x in/out once per call)
    x_h.zero_()
    t0 = time.perf_counter()
    done = 0
    while done < Ke:
        c = min(64, Ke - done)
        cg.outer_steps_host(idx_h[done * sb:(done + c) * sb], x_h, s, cfg.b, cfg.eta, n_steps=c)
        done += c
    e2e64_s = time.perf_counter() - t0
    clk = clocks.stop()
    e2e_s, e2e64_s = max_over_ranks([e2e_s, e2e64_s], dist, "cuda")

    # ---- per-stage device times (CUDA events on the library's stream, same kernels launched directly)
    Kp = min(K, 200)
    cg.set_option(binding.OPT_PROFILE, 1)
    cg.outer_steps(idx_d[W * sb:], x, s, cfg.b, cfg.eta, n_steps=min(Kp, 5))
    cg.stage_times(reset=True)
    cg.outer_steps(idx_d[W * sb:], x, s, cfg.b, cfg.eta, n_steps=Kp)
    st = cg.stage_times(reset=True)
    cg.set_option(binding.OPT_PROFILE, 0)
    work = stage_work(cfg.n, s, cfg.b, pk)
    # fused stages: a stage with no launch of its own ran inside its neighbour (n <= 64: gather inside the Gram
    # kernel; small steps: gradient + update inside the recurrence kernel; s = 1: l' inside the Gram epilogue)
    for absent, host in (("gather", "gram"), ("gradient", "recurrence"), ("recurrence", "gram")):
        if st[absent][1] == 0 and st[host][1] > 0:
            work[host]["bytes"] += work[absent]["bytes"]
            work[host]["flops"] += work[absent]["flops"]
            work[host]["fused"] = work[host].get("fused", []) + [absent]
    stages = {}
    for name, wk in work.items():
        tot_ms, cnt = st[name]
        per_step = tot_ms / Kp
        rl = roofline_of(name, wk, per_step, pk, ncu_traffic(cfg.name, s, name)) if cnt else None
        if rl and name == "recurrence" and s > 1:
            # the chain is s - 1 dependent hops of one distributed-shared-memory broadcast each: its own floor
            rl["chain"] = dict(hops=s - 1, kernel_us_per_hop=round(per_step * 1e3 / (s - 1), 3),
                               note="latency chain: the kernel's time over its s - 1 dependent hops (start-up, launch "
                                    "latency and any fused update included); ~0.42 us per hop in steady state "
                                    "(DESIGN.md section 6)")
        if rl and wk.get("fused"):
            rl["includes"] = wk["fused"]
        stages[name] = dict(ms_per_step=round(per_step, 6), launches_per_step=cnt / Kp, roofline=rl,
                            alg_bytes=wk["bytes"], alg_flops=wk["flops"])
    dominant = max(stages, key=lambda k: stages[k]["ms_per_step"])
    roofline = stages[dominant]["roofline"]

    # ---- casgd_loss: the pure streaming GEMV over all of A (BASELINE metric's "GEMV HBM GB/s")
    cg.loss(x)
    cg.set_option(binding.OPT_PROFILE, 1)
    cg.stage_times(reset=True)
    reps = 5
    for _ in range(reps):
        cg.loss(x)
    loss_ms = cg.stage_times(reset=True)["loss"][0] / reps
    cg.set_option(binding.OPT_PROFILE, 0)
    loss_bytes = 2 * cfg.m * cfg.n + 4 * cfg.m
    gemv = dict(kernel="casgd_loss", bound="hbm", achieved=round(loss_bytes / loss_ms / 1e6, 2), peak=pk["hbm"],
                unit="GB/s", frac=round(loss_bytes / loss_ms / 1e6 / pk["hbm"], 4), avg_call_ms=round(loss_ms, 5),
                traffic=ncu_traffic(cfg.name, 0, "loss"), peak_source=pk["source"])

    # ---- in-library FP32 s = 1 SGD baseline (Recipe A) and the s sweep, same index stream
    sweep = {}
    if not args.no_sweep:
        Ks = max(50, min(K * s, 4000))
        idx_s = torch.from_numpy(step_indices(cfg, seed, Ks, cfg.b)).cuda()
        xs = torch.zeros(cfg.n, device="cuda")
        cg.sgd_steps_fp32(idx_s[: 10 * cfg.b], xs, cfg.b, cfg.eta, n_steps=10)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(stream):
            e0.record(stream)
            cg.sgd_steps_fp32(idx_s, xs, cfg.b, cfg.eta, n_steps=Ks)
            e1.record(stream)
        stream.synchronize()
        sweep["fp32_sgd_s1"] = dict(rows_per_s=Ks * cfg.b / (e0.elapsed_time(e1) * 1e-3))
        for s2 in cfg.s_list:
            sb2 = s2 * cfg.b
            k2 = max(20, min(2000, (K * sb) // sb2))
            idx2 = torch.from_numpy(step_indices(cfg, seed, k2 + 5, sb2)).cuda()
            prime_graphs(cg, cfg, seed, s2, sb2)
            x2 = torch.zeros(cfg.n, device="cuda")
            cg.outer_steps(idx2[: 5 * sb2], x2, s2, cfg.b, cfg.eta, n_steps=5)
            ms2 = time_steps(binding, cg, idx2[5 * sb2:], x2, s2, cfg.b, cfg.eta, k2, stream)
            sweep[f"s{s2}"] = dict(rows_per_s=k2 * sb2 / (ms2 * 1e-3), ms_per_outer_step=ms2 / k2)

    value = aggregate_rows_per_s(world, K, sb, ms)
    e2e_value = aggregate_rows_per_s(world, Ke, sb, e2e_s * 1e3)
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=K, warmup=W, ms_per_step=ms / K,
                higher_is_better=True, scaling="weak", vs_baseline=None, dtype="bf16 in / f32 accumulate",
                data="synthetic",
                config=dict(workload=cfg.name, m=cfg.m, n=cfg.n, b=cfg.b, s=s, rows_per_step=sb, eta=cfg.eta,
                            loss=("logistic", "linear", "poisson")[cfg.loss], parallelism=f"replicas x{world}",
                            l2="inputs larger than L2: rows are gathered at random from A "
                               f"({cfg.m * max(cfg.n, 8) * 2 / 1e6:.0f} MB)" if cfg.m * cfg.n * 2 > 126e6 else
                               "A fits in L2; not flushed (the step's own working set is L2-resident by design)",
                            outer_iters_per_s=K / (ms * 1e-3), final_loss=F_after),
                clocks=clk,
                e2e=dict(value=e2e_value, unit=UNIT, h2d_bytes_per_step=sb * 4 + cfg.n * 4,
                         d2h_bytes_per_step=cfg.n * 4, steps=Ke,
                         batched64=dict(value=aggregate_rows_per_s(world, Ke, sb, e2e64_s * 1e3), h2d_bytes_per_step=sb * 4 + cfg.n * 4 / 64,
                                        d2h_bytes_per_step=cfg.n * 4 / 64)),
                gpu_launches=int(launches),
                sampled_on_device=dict(value=aggregate_rows_per_s(world, K, sb, sampled_ms), unit=UNIT, ms_per_step=sampled_ms / K,
                                       sampler="Philox4x32-10, i.i.d. with replacement (PAPER.md:L111)"),
                roofline=roofline, stages=stages, gemv=gemv, sweep=sweep)

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, steps_o, t_o, cores = oracle_rows_per_s(cfg, s, ds.X_bf16, ds.y, idx_np, seed)
        line["cpu_baseline"] = dict(value=v, unit=UNIT, cores=cores, kind="oracle",
                                    sample=f"oracle O1 (FP64 Gram form) on the first {steps_o} outer steps "
                                           f"(s={s}, b={cfg.b}) of the same index stream, {t_o:.1f} s")
    cg.close()
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
