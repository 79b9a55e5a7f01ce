"""P > 1 (Alg. 1 line 5, L141 section 4.2, L154 Table 2): the host logic of the 1-D
block-column partition on CPU -- column slabs, the payload layout, and the sum over ranks through torch.distributed
(gloo, world size 2) -- and the oracle's partitioned form pinned to its P = 1 form. The CUDA halves of the split outer
iteration are tested in tests/test_gpu_partition.py."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2606_18463_b200 import partition, synth  # noqa: E402


@pytest.mark.parametrize("n,P", [(4096, 8), (2000, 4), (18, 2), (18, 3), (512, 7), (64, 64), (9984, 16)])
def test_column_slabs_tile_the_columns_in_rank_order(n, P):
    slabs = [partition.column_slab(n, r, P) for r in range(P)]
    assert slabs[0].start == 0 and slabs[-1].stop == n
    for a, c in zip(slabs, slabs[1:]):
        assert a.stop == c.start                       # contiguous, ordered, disjoint
    assert all(sl.stop > sl.start for sl in slabs)     # nobody is left without columns
    sizes = [sl.stop - sl.start for sl in slabs]
    if n >= 8 * P:
        assert all(sl.start % 8 == 0 for sl in slabs)  # 16-byte aligned BF16 slab starts: used in place by the library
        assert max(sizes) - min(sizes) <= 8 + (8 - n % 8) % 8
    with pytest.raises(ValueError):
        partition.column_slab(3, 0, 4)


@pytest.mark.parametrize("s,b", [(1, 16), (4, 16), (5, 7), (32, 64)])
def test_payload_layout_is_a_bijection_onto_r_and_the_strict_block_lower_G(s, b):
    sb = s * b
    count = partition.payload_words(s, b)
    assert count == sb + b * b * s * (s - 1) // 2       # Table 2's sb + (sb)^2 with the symmetric half dropped (L154, L180)
    seen = np.zeros(count, bool)
    seen[:sb] = True                                    # r
    for i in range(b, sb, max(1, sb // 37)):            # sampled rows, every column they own
        for k in range((i // b) * b):
            t = partition.payload_index(i, k, s, b)
            assert sb <= t < count and not seen[t]
            seen[t] = True
    if sb <= 128:                                       # small: every entry
        seen[sb:] = False
        for i in range(b, sb):
            for k in range((i // b) * b):
                seen[partition.payload_index(i, k, s, b)] = True
        assert seen.all()


@pytest.mark.parametrize("ci,m,n,s,b,P", [(0, 600, 64, 4, 16, 2), (1, 500, 18, 3, 8, 3), (2, 300, 200, 3, 16, 7),
                                          (4, 400, 96, 5, 8, 1)])
@pytest.mark.parametrize("shadow", [True, False])
def test_partitioned_oracle_equals_the_single_rank_form(ci, m, n, s, b, P, shadow):
    """The sum of the slab Grams is the Gram matrix and the sum of the slab margins the margin (block-column identity
    behind L141), so Alg. 1 with line 5 gives the x of Alg. 1 at P = 1 -- to rounding, for every loss."""
    cfg = synth.config(ci, m=m, n=n)
    ds = synth.make_dataset(cfg, seed=7, device="cpu")
    A_bits, y = ds.X_bits_numpy(), ds.y_numpy()
    idx = np.random.default_rng(3).integers(0, m, s * b).astype(np.int32)          # with duplicates
    x0 = (np.random.default_rng(4).standard_normal(n) * 0.4).astype(np.float32).astype(np.float64)
    slabs = [partition.column_slab(n, r, P) for r in range(P)]
    one = oracle.outer_step_gram(A_bits, y, idx, x0, s, b, cfg.eta, cfg.loss, shadow=shadow)
    par = oracle.outer_step_gram_partitioned(A_bits, y, idx, x0, s, b, cfg.eta, cfg.loss, slabs, shadow=shadow)
    scale = max(1.0, np.abs(one.G).max())
    assert np.abs(par.G - one.G).max() <= 1e-12 * scale
    assert np.abs(par.r - one.r).max() <= 1e-12 * max(1.0, np.abs(one.r).max())
    assert np.abs(par.u - one.u).max() <= 1e-11 * max(1.0, np.abs(one.u).max())
    assert np.linalg.norm(par.x_out - one.x_out) <= 1e-12 * max(1.0, np.linalg.norm(one.x_out))
    # a slab's Gram alone is NOT the Gram (the reduce is needed): negative control
    if P > 1:
        _, G0 = oracle.slab_payload(A_bits, idx, x0, s, b, slabs[0], shadow)
        assert np.abs(G0 - one.G).max() > 1e-3 * scale


class _NumpySlab:
    """Stand-in for the CUDA backend in the host-logic test: the rank's share of the step in FP64 numpy, using the same
    payload layout as the library (partition.payload_index)."""

    def __init__(self, A_bits, y, loss, cols):
        self.A, self.y, self.loss, self.cols = A_bits, y, loss, cols

    def new_payload(self, s, b):
        return torch.zeros(partition.payload_words(s, b), dtype=torch.float64)

    def local(self, idx, x_slab, s, b, payload):
        x_full = np.zeros(self.A.shape[1])
        x_full[self.cols] = x_slab
        r, G = oracle.slab_payload(self.A, idx, x_full, s, b, self.cols, shadow=True)
        out = payload.numpy()
        out[: s * b] = r
        for i in range(b, s * b):
            j = i // b
            t0 = partition.payload_index(i, 0, s, b)
            out[t0: t0 + j * b] = G[i, : j * b]
        self._idx = idx

    def finish(self, x_slab, s, b, eta, payload):
        p = payload.numpy()
        sb, alpha = s * b, eta / b
        u = np.zeros(sb)
        yI = self.y[self._idx].astype(np.float64)
        for j in range(s):
            for i in range(j * b, (j + 1) * b):
                corr = p[partition.payload_index(i, 0, s, b): partition.payload_index(i, 0, s, b) + j * b] @ u[: j * b] if j else 0.0
                u[i] = oracle.lprime(p[i] - alpha * corr, yI[i], self.loss)
        Y = oracle.bf16_to_f64(self.A[self._idx][:, self.cols])
        x_slab -= alpha * (Y.T @ u)


def _free_port():
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        return sk.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = synth.config(0, m=700, n=50)
    ds = synth.make_dataset(cfg, seed=11, device="cpu")
    A_bits, y = ds.X_bits_numpy(), ds.y_numpy()
    s, b, steps = 3, 8, 4
    idx = np.random.default_rng(5).integers(0, cfg.m, steps * s * b).astype(np.int32)
    cols = partition.column_slab(cfg.n, rank, world)
    step = partition.PartitionedCasgd(_NumpySlab(A_bits, y, cfg.loss, cols), group=dist.group.WORLD)
    x_slab = np.zeros(cols.stop - cols.start)
    for h in range(steps):
        step.outer_step(idx[h * s * b:(h + 1) * s * b], x_slab, s, b, cfg.eta)
    out.put((rank, cols.start, cols.stop, x_slab.tolist()))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_over_gloo_reproduce_the_single_rank_trajectory():
    """World size 2 on CPU: column slabs, payload packing, the AllReduce of line 5 and the per-slab update, driven by
    the product's PartitionedCasgd, give the oracle's P = 1 trajectory (BF16 shadow per outer step) to rounding."""
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    cfg = synth.config(0, m=700, n=50)
    ds = synth.make_dataset(cfg, seed=11, device="cpu")
    A_bits, y = ds.X_bits_numpy(), ds.y_numpy()
    s, b, steps = 3, 8, 4
    idx = np.random.default_rng(5).integers(0, cfg.m, steps * s * b).astype(np.int32)
    x = np.zeros(cfg.n)
    for h in range(steps):
        x = oracle.outer_step_gram(A_bits, y, idx[h * s * b:(h + 1) * s * b], x, s, b, cfg.eta, cfg.loss, shadow=True).x_out
    got = np.zeros(cfg.n)
    assert res[0][1] == 0 and res[0][2] == res[1][1] and res[1][2] == cfg.n
    for _, c0, c1, xs in res:
        got[c0:c1] = xs
    # the numpy stand-in keeps an FP64 master, the oracle's outer_step_gram takes an FP64 x too: only summation order differs
    assert np.linalg.norm(got - x) <= 1e-10 * np.linalg.norm(x)
