"""The N > 1 path of bench.py on CPU (gloo, world size 2). The method does not shard at P = 1 (DESIGN.md
section 10: replicas only), so what N > 1 adds is host logic: per-rank seeds, MAX-over-ranks timing,
whole-job aggregation, and the reference arm printing one line from rank 0 only."""
import json
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = [10.0 + 5.0 * rank, 3.0 - rank]                 # rank 1 is slower on the first, faster on the second
    got = bench.max_over_ranks(ms, dist, "cpu")
    out.put((rank, got, bench.replica_seed(rank)))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_replica_seeds_gloo_world2():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [[15.0, 3.0], [15.0, 3.0]]      # every rank holds the max
    assert [r[2] for r in res] == [42, 43]                         # replicas draw different datasets
    sys.path.insert(0, ROOT)
    import bench
    # 2 ranks x 100 steps x 1024 rows in 15 ms
    assert bench.aggregate_rows_per_s(2, 100, 1024, 15.0) == 2 * 100 * 1024 / 0.015
    assert bench.max_over_ranks([1.5], None, "cpu") == [1.5]


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
           "--workload", "0", "--steps", "3", "--warmup", "1"]
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="", OMP_NUM_THREADS="2")
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["steps"] == 3 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["config"]["workload"] == "tiny-logistic"
