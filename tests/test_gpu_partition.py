"""P > 1 on the GPU: the CUDA halves of the split outer iteration (casgd_step_local /
casgd_reduce_peers / casgd_step_finish, include/casgd.h) with the P ranks emulated as P contexts -- one per column
slab -- on ONE device, their kernels run one after the other on one stream (no kernel waits for another). Checked against
oracle O1 on the unpartitioned matrix at north_star's tolerances. A scaling curve needs more GPUs than this run has."""
import os
import socket

import numpy as np
import pytest
import torch

from paper_2606_18463_b200 import partition, synth

from gpu_common import TOL_G, TOL_R, TOL_X, block_lower_mask, device_dataset, random_x

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    from paper_2606_18463_b200 import binding as b
    b.load()
    return b


@pytest.fixture(scope="module")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle


SHAPES = [(0, 8192, 64, 4, 16, 2), (1, 20000, 18, 5, 64, 2), (4, 6000, 512, 6, 64, 3), (3, 5000, 2000, 9, 32, 4),
          (2, 4200, 4096, 3, 128, 8), (4, 6000, 512, 1, 64, 2), (2, 5000, 1000, 6, 128, 3)]


@pytest.mark.parametrize("reduce", ["peers-kernel", "callers-sum"])
@pytest.mark.parametrize("ci,m,n,s,b,P", SHAPES)
def test_p_slabs_on_one_device_match_the_oracle(binding, oracle_mod, ci, m, n, s, b, P, reduce):
    cfg = synth.config(ci, m=m, n=n)
    X_d, y_d, A_bits, y = device_dataset(cfg)
    idx = synth.epoch_indices(cfg, 42, 0)[: s * b].copy()
    idx_d = torch.from_numpy(idx).cuda()
    x0 = random_x(n, 9, 0.5)
    slabs = [partition.column_slab(n, r, P) for r in range(P)]
    ref = oracle_mod.outer_step_gram(A_bits, y, idx, x0.astype(np.float64), s, b, cfg.eta, cfg.loss, shadow=True)
    sb = s * b
    count = binding.payload_count(s, b)
    assert count == partition.payload_words(s, b)
    ctxs = [binding.Casgd(X_d[:, sl], y_d, cfg.loss) for sl in slabs]
    try:
        xs = [torch.from_numpy(x0[sl].copy()).cuda() for sl in slabs]
        pays = [torch.empty(count, device="cuda") for _ in slabs]
        for cg, xp, pay in zip(ctxs, xs, pays):
            cg.step_local(idx_d, xp, s, b, pay)
        torch.cuda.synchronize()
        # each slab's payload: r_loc and the strict block-lower G_loc in the documented layout
        Yf = oracle_mod.bf16_to_f64(ref.Y_bits)
        for sl, pay in zip(slabs, pays):
            r_loc, G_loc = oracle_mod.slab_payload(A_bits, idx, x0.astype(np.float64), s, b, sl, shadow=True)
            p = pay.cpu().numpy().astype(np.float64)
            nrm = np.sqrt((Yf[:, sl] ** 2).sum(1))
            xh = oracle_mod.bf16_to_f64(oracle_mod.f32_to_bf16(x0[sl]))
            assert np.all(np.abs(p[:sb] - r_loc) <= TOL_R * nrm * np.linalg.norm(xh) + 1e-30)
            for i in range(b, sb, max(1, sb // 23)):
                j = i // b
                t0 = partition.payload_index(i, 0, s, b)
                assert np.all(np.abs(p[t0: t0 + j * b] - G_loc[i, : j * b]) <= TOL_G * nrm[i] * nrm[: j * b] + 1e-30)
        # the sum over ranks (Alg. 1 line 5), then the second half on every rank
        if reduce == "peers-kernel":
            for cg, xp in zip(ctxs, xs):
                cg.reduce_peers(pays, s, b)
                cg.step_finish(xp, s, b, cfg.eta, None)
        else:
            total = torch.stack(pays).sum(0)            # stands in for the caller's AllReduce
            for cg, xp in zip(ctxs, xs):
                cg.step_finish(xp, s, b, cfg.eta, total)
        torch.cuda.synchronize()
        norms = np.sqrt((Yf * Yf).sum(1))
        xhat = oracle_mod.bf16_to_f64(oracle_mod.f32_to_bf16(x0))
        mask = block_lower_mask(s, b)
        u0 = None
        for cg in ctxs:
            r = cg.debug(binding.DBG_R).astype(np.float64)
            assert np.all(np.abs(r - ref.r) <= TOL_R * norms * np.linalg.norm(xhat) + 1e-30)
            if mask.any():
                G = cg.debug(binding.DBG_G).astype(np.float64)
                assert np.all((np.abs(G - ref.G) <= TOL_G * np.outer(norms, norms) + 1e-30)[mask])
            u = cg.debug(binding.DBG_U)
            if reduce == "peers-kernel" and u0 is not None:
                assert np.array_equal(u, u0)            # rank-ordered sum: every rank's recurrence saw identical bits
            u0 = u
        x1 = np.concatenate([xp.cpu().numpy() for xp in xs]).astype(np.float64)
        rel = np.linalg.norm(x1 - ref.x_out) / np.linalg.norm(ref.x_out)
        assert rel <= TOL_X, f"x after one partitioned outer step: relative error {rel:.3g}"
    finally:
        for cg in ctxs:
            cg.close()


def test_one_rank_through_the_split_calls_equals_casgd_outer_step(binding):
    cfg = synth.config(4, m=6000, n=512)
    X_d, y_d, _, _ = device_dataset(cfg)
    s, b = 6, 64
    idx_d = torch.from_numpy(synth.epoch_indices(cfg, 42, 0)[: s * b].copy()).cuda()
    x0 = random_x(cfg.n, 3, 0.3)
    with binding.Casgd(X_d, y_d, cfg.loss) as cg:
        xa = torch.from_numpy(x0.copy()).cuda()
        cg.outer_step(idx_d, xa, s, b, cfg.eta)
        xb = torch.from_numpy(x0.copy()).cuda()
        pay = torch.empty(binding.payload_count(s, b), device="cuda")
        cg.step_local(idx_d, xb, s, b, pay)
        cg.step_finish(xb, s, b, cfg.eta, pay)
        cg.sync()
        assert torch.equal(xa, xb)
        # argument checks of the split calls
        with pytest.raises(binding.CasgdError):
            cg.step_finish(xb, s + 1, b, cfg.eta, pay)
        assert binding.payload_count(0, 4) == -1


def test_partitioned_step_over_nccl_world_of_one(binding, oracle_mod):
    """PartitionedCasgd with a real NCCL process group (one rank: the only size this box allows): the AllReduce of the
    payload runs through torch.distributed on the device tensor the library packed."""
    import torch.distributed as dist
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK="0", WORLD_SIZE="1")
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda:0"))
    try:
        cfg = synth.config(3, m=5000, n=520)
        X_d, y_d, A_bits, y = device_dataset(cfg)
        s, b = 5, 32
        idx = synth.epoch_indices(cfg, 42, 0)[: s * b].copy()
        x0 = random_x(cfg.n, 4, 0.5)
        back = partition.CudaSlab(X_d, y_d, cfg.loss)
        step = partition.PartitionedCasgd(back, group=dist.group.WORLD)
        x = torch.from_numpy(x0.copy()).cuda()
        step.outer_step(torch.from_numpy(idx).cuda(), x, s, b, cfg.eta)
        torch.cuda.synchronize()
        ref = oracle_mod.outer_step_gram(A_bits, y, idx, x0.astype(np.float64), s, b, cfg.eta, cfg.loss, shadow=True)
        x1 = x.cpu().numpy().astype(np.float64)
        assert np.linalg.norm(x1 - ref.x_out) <= TOL_X * np.linalg.norm(ref.x_out)
        back.close()
    finally:
        dist.destroy_process_group()


def _peer_worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)       # control plane only: handles and barriers
    try:
        import oracle
        from paper_2606_18463_b200 import binding
        torch.cuda.set_device(0)
        cfg = synth.config(4, m=6000, n=520)
        X_d, y_d, A_bits, y = device_dataset(cfg)
        s, b = 6, 64
        idx = synth.epoch_indices(cfg, 42, 0)[: 2 * s * b].copy()
        x0 = random_x(cfg.n, 21, 0.4)
        sl = partition.column_slab(cfg.n, rank, world)
        back = partition.CudaSlab(X_d[:, sl], y_d, cfg.loss)
        step = partition.PeerPartitionedCasgd(back, dist.group.WORLD)
        x = torch.from_numpy(x0[sl].copy()).cuda()
        xs = []
        for h in range(2):
            step.outer_step(torch.from_numpy(idx[h * s * b:(h + 1) * s * b]).cuda(), x, s, b, cfg.eta)
            xs.append(x.cpu().numpy().copy())
        u_bits = back.cg.debug(binding.DBG_U).tobytes()
        out.put((rank, sl.start, sl.stop, xs, u_bits))
        dist.barrier()
        step.close()
        back.close()
    finally:
        dist.destroy_process_group()


def test_two_processes_sum_their_payloads_through_peer_memory(oracle_mod):
    """Two PROCESSES (one column slab each, both on this box's one GPU, gloo for the control plane): the payloads are
    dedicated allocations shared by CUDA IPC handles, each process's casgd_reduce_peers kernel reads both and writes
    the rank-ordered sum into its own G and r -- the library's own one-shot all-reduce, no NCCL. Two outer iterations
    against oracle O1 on the unpartitioned matrix; both processes end with identical u bits."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    procs = [ctx.Process(target=_peer_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=300) for _ in procs)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    cfg = synth.config(4, m=6000, n=520)
    ds = synth.make_dataset(cfg, seed=42, device="cpu")
    A_bits, y = ds.X_bits_numpy(), ds.y_numpy()
    s, b = 6, 64
    idx = synth.epoch_indices(cfg, 42, 0)[: 2 * s * b].copy()
    x_prev = random_x(cfg.n, 21, 0.4)
    assert res[0][1] == 0 and res[0][2] == res[1][1] and res[1][2] == cfg.n
    for h in range(2):
        ref = oracle_mod.outer_step_gram(A_bits, y, idx[h * s * b:(h + 1) * s * b], x_prev.astype(np.float64), s, b, cfg.eta,
                                         cfg.loss, shadow=True)
        got = np.concatenate([r[3][h] for r in res])
        rel = np.linalg.norm(got.astype(np.float64) - ref.x_out) / np.linalg.norm(ref.x_out)
        assert rel <= TOL_X, f"iteration {h}: relative error {rel:.3g}"
        x_prev = got                                     # the next iteration starts from the library's own FP32 bits
    assert res[0][4] == res[1][4]                        # rank-ordered sum: identical u on both ranks
