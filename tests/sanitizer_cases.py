"""Tiny shapes through every kernel variant of libcasgd.so, for compute-sanitizer:

    compute-sanitizer --tool memcheck  python tests/sanitizer_cases.py
    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py
    compute-sanitizer --tool synccheck python tests/sanitizer_cases.py
    compute-sanitizer --tool initcheck python tests/sanitizer_cases.py

(one tool per GPU-box call; B200_PROFILING.md). Not a pytest file: it only drives the kernels -- parity is what
tests/test_gpu_*.py check -- and prints one line per case so that a sanitizer report can be matched to it.
`--only NAME` runs the cases whose name contains NAME."""
from __future__ import annotations

import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_2606_18463_b200 import binding, synth  # noqa: E402


def dataset(ci, m, n):
    cfg = synth.config(ci, m=m, n=n)
    ds = synth.make_dataset(cfg, seed=42, device="cpu")
    return cfg, ds.X_bf16.cuda(), ds.y.cuda()


def step_case(name, ci, m, n, s, b, opts=(), steps=1, eta=None):
    cfg, X, y = dataset(ci, m, n)
    eta = cfg.eta if eta is None else eta
    with binding.Casgd(X, y, cfg.loss) as cg:
        for o, v in opts:
            cg.set_option(o, v)
        idx = torch.from_numpy(synth.iid_indices(m, steps * s * b, 3)).cuda()
        x = torch.zeros(n, device="cuda")
        if steps == 1:
            cg.outer_step(idx, x, s, b, eta)
        else:
            cg.outer_steps(idx, x, s, b, eta)
        cg.sync()
        assert torch.isfinite(x).all()
        damage = int(cg.debug(binding.DBG_GUARDS)[0])
        assert damage == 0, f"{name}: {damage} guard bytes around the workspaces were overwritten"
    print(f"case {name}: ok, guard bands intact", flush=True)


def cases():
    B = binding
    yield "gram_simt", lambda: step_case("gram_simt", 3, 600, 72, 3, 32, [(B.OPT_GRAM_IMPL, 1)])
    yield "gram_tile128", lambda: step_case("gram_tile128", 3, 600, 200, 5, 32, [(B.OPT_GRAM_IMPL, 2)])
    yield "gram_tile128_ksplit", lambda: step_case("gram_tile128_ksplit", 3, 600, 200, 5, 32, [(B.OPT_GRAM_IMPL, 2), (B.OPT_GRAM_KSPLIT, 2)])
    yield "gram_pair256", lambda: step_case("gram_pair256", 4, 900, 136, 5, 64, [(B.OPT_GRAM_IMPL, 3)], eta=0.01)
    yield "gram_pair256_ksplit", lambda: step_case("gram_pair256_ksplit", 4, 900, 136, 5, 64, [(B.OPT_GRAM_IMPL, 3), (B.OPT_GRAM_KSPLIT, 2)], eta=0.01)
    yield "gram_pair512", lambda: step_case("gram_pair512", 4, 900, 136, 9, 64, [(B.OPT_GRAM_IMPL, 4)], eta=0.01)
    yield "gram_narrow", lambda: step_case("gram_narrow", 1, 900, 18, 3, 64, [(B.OPT_GRAM_IMPL, 5)])
    yield "gram_narrow_s1", lambda: step_case("gram_narrow_s1", 1, 900, 18, 1, 64, [(B.OPT_MINI, 0)])
    yield "mini_s1", lambda: step_case("mini_s1", 1, 900, 18, 1, 64, steps=5)
    yield "mini_s4", lambda: step_case("mini_s4", 0, 900, 64, 4, 16, steps=5)
    yield "mini_odd", lambda: step_case("mini_odd", 0, 900, 33, 3, 13, steps=3)
    yield "mini_split", lambda: step_case("mini_split", 0, 900, 64, 4, 16, [(B.OPT_MARGIN_SPLIT, 1)], steps=3)
    yield "margin_s1", lambda: step_case("margin_s1", 4, 900, 136, 1, 64, [(B.OPT_MINI, 0)], eta=0.01)
    yield "s1_cluster", lambda: step_case("s1_cluster", 4, 900, 520, 1, 64, steps=5, eta=0.01)
    yield "s1_cluster_odd", lambda: step_case("s1_cluster_odd", 3, 900, 1001, 1, 40, steps=3)
    for impl, nm in ((1, "cta"), (2, "grid"), (3, "cluster"), (4, "stream"), (5, "chain")):
        yield f"rec_{nm}", (lambda impl=impl, nm=nm: step_case(f"rec_{nm}", 0, 900, 24, 6, 32, [(B.OPT_RECURRENCE_IMPL, impl)]))
    yield "rec_stream_two_groups", lambda: step_case("rec_stream_two_groups", 0, 1200, 24, 3, 128, [(B.OPT_RECURRENCE_IMPL, 4)])
    yield "rec_stream_unfused", lambda: step_case("rec_stream_unfused", 0, 900, 24, 6, 32, [(B.OPT_RECURRENCE_IMPL, 4), (B.OPT_NO_FUSED_UPDATE, 1)])
    yield "rec_chain_unfused", lambda: step_case("rec_chain_unfused", 0, 900, 24, 9, 64, [(B.OPT_RECURRENCE_IMPL, 5), (B.OPT_NO_FUSED_UPDATE, 1)])
    yield "rec_grid_scalar", lambda: step_case("rec_grid_scalar", 0, 900, 24, 5, 13, [(B.OPT_RECURRENCE_IMPL, 2)])
    yield "gather_bulk_gradient_stream", lambda: step_case("gather_bulk_gradient_stream", 2, 1200, 1024, 4, 128)
    yield "graph_sequential", lambda: step_case("graph_sequential", 4, 900, 136, 3, 64, [(B.OPT_OVERLAP, 0)], steps=9, eta=0.01)
    yield "graph_gather_aside", lambda: step_case("graph_gather_aside", 2, 1200, 1024, 3, 128, [(B.OPT_OVERLAP, 1)], steps=9)
    yield "graph_pipelined_wide", lambda: step_case("graph_pipelined_wide", 2, 1200, 1024, 3, 128, steps=9)
    yield "split_fused_tile128", lambda: step_case("split_fused_tile128", 3, 600, 200, 5, 32, [(B.OPT_OVERLAP, 0), (B.OPT_GRAM_IMPL, 2), (B.OPT_MARGIN_SPLIT, 1)])
    yield "split_fused_pair", lambda: step_case("split_fused_pair", 4, 900, 136, 5, 64, [(B.OPT_OVERLAP, 0), (B.OPT_GRAM_IMPL, 3), (B.OPT_MARGIN_SPLIT, 1)], eta=0.01)
    yield "split_margin_kernel", lambda: step_case("split_margin_kernel", 3, 600, 200, 5, 32, [(B.OPT_MARGIN_SPLIT, 1)], steps=3)
    yield "graph_replay", lambda: step_case("graph_replay", 4, 900, 136, 3, 64, steps=9, eta=0.01)
    yield "graph_replay_stamps", lambda: step_case("graph_replay_stamps", 4, 900, 136, 3, 64, [(B.OPT_STAMPS, 1)], steps=9, eta=0.01)

    def loss_cases():
        for ci, m, n in ((0, 700, 64), (1, 3001, 18), (2, 301, 1040), (0, 333, 19), (2, 40, 8200)):
            cfg, X, y = dataset(ci, m, n)
            with binding.Casgd(X, y, cfg.loss) as cg:
                for impl in (0, 1):
                    cg.set_option(B.OPT_LOSS_IMPL, impl)
                    F = cg.loss(torch.full((n,), 0.01, device="cuda"))
                    assert np.isfinite(F)
        print("case loss: ok", flush=True)
    yield "loss", loss_cases

    def sgd32():
        cfg, X, y = dataset(4, 900, 136)
        with binding.Casgd(X, y, cfg.loss) as cg:
            x = torch.zeros(cfg.n, device="cuda")
            cg.sgd_steps_fp32(torch.from_numpy(synth.iid_indices(cfg.m, 3 * 64, 1)).cuda(), x, 64, 0.01)
            cg.sync()
        print("case sgd32: ok", flush=True)
    yield "sgd32", sgd32

    def sampled_and_host():
        cfg, X, y = dataset(1, 900, 18)
        with binding.Casgd(X, y, cfg.loss) as cg:
            x = torch.zeros(cfg.n, device="cuda")
            cg.outer_steps_sampled(x, 3, 64, cfg.eta, n_steps=3, seed=5, first_step=0)
            xh = torch.zeros(cfg.n)
            cg.outer_steps_host(torch.from_numpy(synth.iid_indices(cfg.m, 2 * 192, 2)), xh, 3, 64, cfg.eta)
            cg.sync()
        print("case sampled_and_host: ok", flush=True)
    yield "sampled_and_host", sampled_and_host

    def partition_case():
        from paper_2606_18463_b200 import partition
        cfg, X, y = dataset(4, 900, 136)
        s, b, P = 3, 64, 3
        slabs = [partition.column_slab(cfg.n, r, P) for r in range(P)]
        ctxs = [binding.Casgd(X[:, sl], y, cfg.loss) for sl in slabs]
        idx = torch.from_numpy(synth.iid_indices(cfg.m, s * b, 4)).cuda()
        xs = [torch.zeros(sl.stop - sl.start, device="cuda") for sl in slabs]
        pays = [torch.empty(binding.payload_count(s, b), device="cuda") for _ in slabs]
        for cg, xp, pay in zip(ctxs, xs, pays):
            cg.step_local(idx, xp, s, b, pay)
        for cg, xp in zip(ctxs, xs):
            cg.reduce_peers(pays, s, b)
            cg.step_finish(xp, s, b, 0.01, None)
        total = torch.stack(pays).sum(0)
        for cg, xp in zip(ctxs, xs):
            cg.step_finish(xp, s, b, 0.01, total)
            cg.sync()
            cg.close()
        print("case partition: ok", flush=True)
    yield "partition", partition_case


def main():
    only = sys.argv[sys.argv.index("--only") + 1] if "--only" in sys.argv else ""
    skip = sys.argv[sys.argv.index("--skip") + 1].split(",") if "--skip" in sys.argv else []
    assert torch.cuda.is_available()
    from paper_2606_18463_b200 import build
    build.build()
    for name, fn in cases():
        if only in name and not any(k and k in name for k in skip):
            fn()
    print("sanitizer cases done", flush=True)


if __name__ == "__main__":
    main()
