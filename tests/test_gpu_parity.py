"""GPU parity: the CUDA path (through the C ABI) against the FP64 oracle, element by element, on the same
seeded inputs. Sizes here are ones the oracle finishes in seconds and that still span several 128-row
Gram tiles and a ragged tail; tests/test_gpu_fullsize.py covers BASELINE.json's full sizes on sampled
outputs. Tolerances: tests/gpu_common.py (BASELINE.json:north_star)."""
import math

import numpy as np
import pytest
import torch

from paper_2606_18463_b200 import synth

from gpu_common import (TOL_FINAL_LOSS, TOL_LOSS_CALL, check_step_against_oracle, compare_last_step, device_dataset, random_x,
                        require_cuda)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    require_cuda()
    from paper_2606_18463_b200 import build
    build.build()
    from paper_2606_18463_b200 import binding as b
    b.load()
    return b


# (config index, m, n, s, b): down-sized rows, BASELINE shapes of (n, b); sb spans several tiles + a tail
SMALL = [
    (0, 8192, 64, 4, 16),        # configs[0] as is
    (1, 20000, 18, 4, 64),       # SUSY-shaped: n = 18 goes through the padded repack
    (1, 20000, 18, 5, 64),       # sb = 320: ragged tail of a 128-row tile
    (2, 3000, 4096, 3, 128),     # dense linear, full n
    (3, 5000, 2000, 9, 32),      # epsilon-shaped, n = 2000: ragged K tail (2000 = 31*64 + 16)
    (4, 6000, 512, 5, 64),       # Poisson
    (4, 6000, 512, 1, 64),       # s = 1: plain mini-batch SGD with a BF16 shadow
    (2, 3000, 4096, 1, 128),     # s = 1, wide rows: the warp-per-row gather + margin + l' kernel
    (3, 3000, 203, 1, 13),       # s = 1, odd n, odd b
    (0, 4096, 64, 7, 1),         # b = 1
    (3, 3000, 203, 11, 13),      # odd n, odd b: nothing aligned
]


GRAM_IMPLS = dict(argvalues=[0, 1, 2, 3, 4, 5], ids=["auto", "simt", "tile128", "pair256", "pair512", "narrow"])


@pytest.mark.parametrize("gram_impl", **GRAM_IMPLS)
@pytest.mark.parametrize("ci,m,n,s,b", SMALL)
def test_one_outer_step_matches_the_oracle(binding, oracle_mod, ci, m, n, s, b, gram_impl):
    cfg = synth.config(ci, m=m, n=n)
    X_d, y_d, A_bits, y = device_dataset(cfg)
    if gram_impl == 5 and n > 64:
        gram_impl = 2                                   # the fused gather + Gram kernel takes n <= 64 only
    with binding.Casgd(X_d, y_d, cfg.loss) as cg:
        cg.set_option(binding.OPT_GRAM_IMPL, gram_impl)
        idx = np.random.default_rng(42).permutation(m)[: s * b].astype(np.int32)      # without replacement
        # from x = 0 (first block has the closed form u_0 = l'(0, y)) and from a generic iterate
        for x0 in (np.zeros(n, np.float32), random_x(n, 7, 0.5 if cfg.loss != synth.POISSON else 0.2)):
            check_step_against_oracle(oracle_mod, cg, A_bits, y, idx, x0, s, b, cfg.eta, cfg.loss, binding)


@pytest.mark.parametrize("ci,m,n,s,b", [(0, 8192, 64, 4, 16), (1, 20000, 18, 5, 64), (4, 6000, 512, 1, 64), (4, 6000, 512, 6, 64)])
def test_unfused_kernels_match_the_oracle(binding, oracle_mod, ci, m, n, s, b):
    """CASGD_OPT_NO_FUSED_UPDATE: the outer update as its own kernel after the recurrence, and at s = 1 the margin through
    the Gram kernel followed by the recurrence kernel -- the paths the fused kernels replace by default."""
    cfg = synth.config(ci, m=m, n=n)
    X_d, y_d, A_bits, y = device_dataset(cfg)
    eta = cfg.eta if cfg.loss != synth.POISSON else 0.01
    with binding.Casgd(X_d, y_d, cfg.loss) as cg:
        cg.set_option(binding.OPT_NO_FUSED_UPDATE, 1)
        idx = synth.iid_indices(m, s * b, 77)
        check_step_against_oracle(oracle_mod, cg, A_bits, y, idx, random_x(n, 5, 0.2), s, b, eta, cfg.loss, binding)


# shapes that span several 256-row pair tiles with a ragged tail, for the cta_group::2 Gram kernel
PAIR_SHAPES = [
    (4, 6000, 512, 9, 128),      # sb = 1152 = 4.5 pair tiles; b = 128: the block diagonal cuts every diagonal tile
    (3, 5000, 336, 40, 32),      # sb = 1280, K tail (336 = 5*64 + 16)
    (2, 4000, 1024, 17, 64),     # sb = 1088: a 64-row tail
]


@pytest.mark.parametrize("ksplit", [0, 3])
@pytest.mark.parametrize("gram_impl", [0, 2, 3, 4], ids=["auto", "tile128", "pair256", "pair512"])
@pytest.mark.parametrize("ci,m,n,s,b", PAIR_SHAPES)
def test_pair_gram_kernel_matches_the_oracle(binding, oracle_mod, ci, m, n, s, b, gram_impl, ksplit):
    cfg = synth.config(ci, m=m, n=n)
    X_d, y_d, A_bits, y = device_dataset(cfg)
    eta = cfg.eta if cfg.loss != synth.POISSON else 0.01
    with binding.Casgd(X_d, y_d, cfg.loss) as cg:
        cg.set_option(binding.OPT_GRAM_IMPL, gram_impl)
        cg.set_option(binding.OPT_GRAM_KSPLIT, ksplit)
        for rep, full in enumerate((0, 1)):
            cg.set_option(binding.OPT_GRAM_FULL_LOWER, full)
            idx = synth.iid_indices(m, s * b, 200 + rep)
            x0 = random_x(n, 17 + rep, 0.3 if cfg.loss != synth.POISSON else 0.1)
            check_step_against_oracle(oracle_mod, cg, A_bits, y, idx, x0, s, b, eta, cfg.loss, binding,
                                      full_lower=bool(full))


@pytest.mark.parametrize("gram_impl", **GRAM_IMPLS)
def test_full_lower_triangle_and_duplicates(binding, oracle_mod, gram_impl):
    """i.i.d. sampling with replacement (Alg. 1 line 1) gives duplicate rows inside and
    across blocks; with CASGD_OPT_GRAM_FULL_LOWER the whole lower triangle (diagonal G_ii = ||y_i||^2
    included) is exported and checked."""
    cfg = synth.config(3, m=300, n=520)
    X_d, y_d, A_bits, y = device_dataset(cfg)
    s, b = 6, 50
    idx = synth.iid_indices(cfg.m, s * b, 5)
    assert len(np.unique(idx)) < len(idx)
    if gram_impl == 5:
        cfg = synth.config(3, m=300, n=52)              # the fused gather + Gram kernel takes n <= 64 only
        X_d, y_d, A_bits, y = device_dataset(cfg)
    with binding.Casgd(X_d, y_d, cfg.loss) as cg:
        cg.set_option(binding.OPT_GRAM_IMPL, gram_impl)
        cg.set_option(binding.OPT_GRAM_FULL_LOWER, 1)
        check_step_against_oracle(oracle_mod, cg, A_bits, y, idx, random_x(cfg.n, 3), s, b, cfg.eta, cfg.loss,
                                  binding, full_lower=True)


# (config index, m, n, s, b): shapes that stress the recurrence kernels; n kept small so that O1 stays fast
RECURRENCE = [
    (2, 6000, 64, 32, 128),      # configs[2]'s largest block: sb = 4096, 31 dependent steps, 4 rows per warp
    (3, 5000, 40, 64, 32),       # configs[3]: s = 64, b = 32 (a quarter of a 128-column chunk)
    (1, 20000, 18, 32, 64),      # configs[1]: sb = 2048
    (0, 9000, 24, 50, 13),       # b % 4 != 0: the one-column-per-lane path, ragged everything
    (4, 6000, 32, 3, 256),       # b = 256: two 128-column chunks per block
    (0, 20000, 16, 9, 1300),     # sb = 11700: up to 10 rows per warp
    (0, 3000, 16, 300, 1),       # b = 1: 299 dependent steps of one column each
    (0, 9000, 24, 21, 20),       # b = 20: blocks straddle the 128-column chunks; CTAs own 2 or 1 rows per block
    (3, 5000, 40, 130, 16),      # b = 16: one row per CTA, 129 hops, eight blocks per chunk
    (0, 9000, 24, 40, 96),       # b = 96: a "bulk" chunk can hold part of the newest block
    (0, 3000, 16, 200, 4),       # b = 4: bulk warps run 64 blocks ahead of the chain (the stream kernel declines)
    (3, 5000, 40, 130, 8),       # b = 8: 32 blocks ahead, inside the stream kernel's partial-sum ring
]


@pytest.mark.parametrize("rec_impl", [1, 2, 3, 4, 5], ids=["cta", "grid", "cluster", "stream", "chain"])
@pytest.mark.parametrize("ci,m,n,s,b", RECURRENCE)
def test_recurrence_kernels_match_the_oracle(binding, oracle_mod, ci, m, n, s, b, rec_impl):
    """Every recurrence kernel (one CTA; all SMs with tagged words through L2; one cluster with plain loads of G;
    one cluster with G streamed through a shared-memory ring; one cluster with the chain on a single CTA and the older
    part of every sum from 15 helper CTAs) on the same inputs, forced with
    CASGD_OPT_RECURRENCE_IMPL, twice in a row (the second launch sees the first one's retired epoch). Shapes a
    kernel does not take (b % 4 != 0, more than 8 rows of a block per CTA) fall through to the next one."""
    cfg = synth.config(ci, m=m, n=n)
    X_d, y_d, A_bits, y = device_dataset(cfg)
    eta = cfg.eta if cfg.loss != synth.POISSON else 0.01
    with binding.Casgd(X_d, y_d, cfg.loss) as cg:
        cg.set_option(binding.OPT_RECURRENCE_IMPL, rec_impl)
        for rep in range(2):
            idx = synth.iid_indices(m, s * b, 100 + rep)
            x0 = random_x(n, 7 + rep, 0.3 if cfg.loss != synth.POISSON else 0.1)
            check_step_against_oracle(oracle_mod, cg, A_bits, y, idx, x0, s, b, eta, cfg.loss, binding)


def test_grid_recurrence_replays_from_a_graph(binding):
    """The cooperative grid-wide recurrence inside casgd_outer_steps' CUDA graph gives bitwise the x of
    single launches, and of the one-CTA kernel up to FP32 summation order."""
    cfg = synth.config(4, m=30000, n=128)
    X_d, y_d, _, _ = device_dataset(cfg)
    s, b, steps = 16, 64, 19
    idx_d = torch.from_numpy(synth.epoch_indices(cfg, 42, 0)[: steps * s * b].copy()).cuda()
    xs = {}
    with binding.Casgd(X_d, y_d, cfg.loss) as cg:
        for impl in (1, 2, 3, 4, 5):
            cg.set_option(binding.OPT_RECURRENCE_IMPL, impl)
            xa = torch.zeros(cfg.n, device="cuda")
            for h in range(steps):
                cg.outer_step(idx_d[h * s * b:(h + 1) * s * b], xa, s, b, cfg.eta)
            xb = torch.zeros(cfg.n, device="cuda")
            cg.outer_steps(idx_d, xb, s, b, cfg.eta)
            cg.sync()
            if impl in (2, 3):
                assert torch.equal(xa, xb)              # sequential graphs: the very kernels of the single steps
            else:                                       # pipelined graphs: the margin is a kernel of its own there
                assert torch.linalg.norm(xa - xb) <= 1e-5 * torch.linalg.norm(xa)
            xs[impl] = xa
    for impl in (2, 3, 4, 5):
        assert torch.linalg.norm(xs[1] - xs[impl]) <= 1e-5 * torch.linalg.norm(xs[1])


def test_gather_special_index_sets(binding, oracle_mod):
    """idx = identity gives Y = A[:sb]; a constant idx gives equal rows; a strided X (row stride > n)
    is used in place."""
    cfg = synth.config(4, m=1000, n=96)
    ds = synth.make_dataset(cfg, device="cpu")
    wide = torch.zeros((cfg.m, 128), dtype=torch.bfloat16)
    wide[:, :96] = ds.X_bf16
    wide[:, 96:] = 7.0                                   # junk in the padding must never reach Y
    X_d = wide.cuda()[:, :96]
    assert X_d.stride(0) == 128
    y_d = ds.y.cuda()
    A_bits = ds.X_bits_numpy()
    x = torch.zeros(cfg.n, device="cuda")
    with binding.Casgd(X_d, y_d, cfg.loss) as cg:
        idx = np.arange(256, dtype=np.int32)
        cg.outer_step(torch.from_numpy(idx).cuda(), x, 4, 64, 0.0)
        assert np.array_equal(cg.debug(binding.DBG_Y), A_bits[:256])
        idx = np.full(256, 17, np.int32)
        cg.outer_step(torch.from_numpy(idx).cuda(), x, 4, 64, 0.0)
        Y = cg.debug(binding.DBG_Y)
        assert np.array_equal(Y, np.broadcast_to(A_bits[17], (256, 96)))
        assert torch.count_nonzero(x).item() == 0        # eta = 0 leaves x alone


def test_out_of_range_index_is_reported_not_read(binding):
    cfg = synth.config(0, m=512, n=64)
    X_d, y_d, A_bits, y = device_dataset(cfg)
    with binding.Casgd(X_d, y_d, cfg.loss) as cg:
        idx = np.arange(64, dtype=np.int32)
        idx[5] = cfg.m
        idx[9] = -1
        x = torch.zeros(cfg.n, device="cuda")
        cg.outer_step(torch.from_numpy(idx).cuda(), x, 4, 16, 0.5)
        with pytest.raises(binding.CasgdError) as e:
            cg.sync()
        assert e.value.status == binding.EINDEX
        Y = cg.debug(binding.DBG_Y)
        assert not Y[5].any() and not Y[9].any() and np.array_equal(Y[6], A_bits[6])
        cg.sync()                                        # the flag is cleared by the failing sync


@pytest.mark.parametrize("n,stride", [(1024, 1024), (2040, 2048), (4096, 4096), (520, 520)])
def test_wide_row_gather_is_bit_exact(binding, n, stride):
    """Wide rows go through the copy-engine gather (cp.async.bulk global -> shared -> global): duplicates within and
    across a warp's batches of 32 rows, out-of-range indices (zero rows + CASGD_EINDEX), a row stride larger
    than n (used in place), row lengths that are not a multiple of the 4 KB slot."""
    m, sb, b = 3000, 1408, 64
    rng = np.random.default_rng(n)
    bits = rng.integers(0, 1 << 16, size=(m, stride), dtype=np.uint16)
    bits[(bits & 0x7f80) == 0x7f80] = 0x3f80                         # no NaN / Inf patterns: the step also runs the math
    X_full = torch.from_numpy(bits.view(np.int16)).cuda().view(torch.bfloat16)
    X_d = X_full[:, :n]
    y_d = torch.from_numpy(rng.standard_normal(m).astype(np.float32)).cuda()
    idx = rng.integers(0, m, size=sb).astype(np.int32)
    idx[100:140] = idx[7]                                             # duplicates
    bad = [3, 64, 65, 700, sb - 1]
    idx[bad] = [m, -1, m + 5, -7, 2 ** 31 - 1]
    x = torch.zeros(n, device="cuda")
    with binding.Casgd(X_d, y_d, synth.LINEAR) as cg:
        cg.outer_step(torch.from_numpy(idx).cuda(), x, sb // b, b, 0.0)
        with pytest.raises(binding.CasgdError) as e:
            cg.sync()
        assert e.value.status == binding.EINDEX
        Y = cg.debug(binding.DBG_Y)
        ylab = cg.debug(binding.DBG_YLAB)
        good = np.ones(sb, bool)
        good[bad] = False
        assert np.array_equal(Y[good], bits[idx[good], :n])
        assert not Y[~good].any()
        assert np.array_equal(ylab[good], y_d.cpu().numpy()[idx[good]]) and not ylab[~good].any()


def test_bad_arguments_are_rejected_before_any_launch(binding):
    cfg = synth.config(0, m=256, n=64)
    X_d, y_d, _, _ = device_dataset(cfg)
    with binding.Casgd(X_d, y_d, cfg.loss) as cg:
        x = torch.zeros(cfg.n, device="cuda")
        idx = torch.zeros(64, dtype=torch.int32, device="cuda")
        before = cg.launch_count()
        lib, ctx = cg._lib, cg._ctx
        assert lib.casgd_outer_step(ctx, idx.data_ptr(), x.data_ptr(), 0, 16, 0.5) == binding.EINVAL
        assert lib.casgd_outer_step(ctx, idx.data_ptr(), x.data_ptr(), 4, 0, 0.5) == binding.EINVAL
        assert lib.casgd_outer_step(ctx, None, x.data_ptr(), 4, 16, 0.5) == binding.EINVAL
        assert lib.casgd_outer_step(ctx, idx.data_ptr(), x.data_ptr(), 4, 16, float("nan")) == binding.EINVAL
        assert lib.casgd_outer_step(ctx, idx.data_ptr(), x.data_ptr(), 2, binding.MAX_SB, 0.5) == binding.EINVAL
        assert lib.casgd_outer_steps(ctx, idx.data_ptr(), -1, x.data_ptr(), 4, 16, 0.5) == binding.EINVAL
        assert cg.launch_count() == before
        cg.outer_steps(idx, x, 4, 16, 0.5, n_steps=0)    # zero steps: a no-op
        assert cg.launch_count() == before


# shapes: the five configs' n, plus ragged ones -- odd n and odd row counts (unaligned narrow rows, a last slot
# that is not a multiple of 16 bytes), n just past a 2 KB segment, one row, fewer rows than warps
LOSS_SHAPES = [(0, 8192, 64), (1, 30000, 18), (2, 4000, 1024), (3, 6000, 2000), (4, 20000, 512), (2, 1501, 4096),
               (1, 30001, 18), (0, 7777, 19), (0, 5003, 7), (4, 3001, 1032), (3, 999, 1001), (0, 1, 64), (1, 37, 18),
               (4, 4099, 40), (2, 300, 8200)]


@pytest.mark.parametrize("impl", [0, 1], ids=["stream", "plain"])
@pytest.mark.parametrize("ci,m,n", LOSS_SHAPES)
def test_full_loss_matches_the_oracle(binding, oracle_mod, ci, m, n, impl):
    cfg = synth.config(ci, m=m, n=n)
    X_d, y_d, A_bits, y = device_dataset(cfg)
    with binding.Casgd(X_d, y_d, cfg.loss) as cg:
        cg.set_option(binding.OPT_LOSS_IMPL, impl)
        F0 = cg.loss(torch.zeros(n, device="cuda"))
        closed = {0: math.log(2.0), 1: float(np.mean(y.astype(np.float64) ** 2) / 2), 2: 1.0}[cfg.loss]
        assert F0 == pytest.approx(closed, rel=1e-6)                       # F(0) in closed form
        x = random_x(n, 11, 0.3)
        F = cg.loss(torch.from_numpy(x).cuda())
        ref = oracle_mod.full_loss(A_bits, y, x.astype(np.float64), cfg.loss)
        assert abs(F - ref) <= TOL_LOSS_CALL * abs(ref)


@pytest.mark.parametrize("ci,m,n", [(1, 20000, 18), (2, 4200, 4096), (4, 6000, 512)])
def test_fp32_sgd_baseline_matches_the_oracle(binding, oracle_mod, ci, m, n):
    """casgd_sgd_steps_fp32 is Alg. 1 with s = 1 and no BF16 shadow (Recipe A): O2 with shadow off."""
    cfg = synth.config(ci, m=m, n=n)
    X_d, y_d, A_bits, y = device_dataset(cfg)
    steps = 6
    idx = synth.epoch_indices(cfg, 42, 0)[: steps * cfg.b].copy()
    x0 = random_x(n, 2, 0.1)
    with binding.Casgd(X_d, y_d, cfg.loss) as cg:
        x_d = torch.from_numpy(x0.copy()).cuda()
        cg.sgd_steps_fp32(torch.from_numpy(idx).cuda(), x_d, cfg.b, cfg.eta)
        cg.sync()
        ref = oracle_mod.train(A_bits, y, idx, x0.astype(np.float64), 1, cfg.b, cfg.eta, cfg.loss, shadow=False)
        x1 = x_d.cpu().numpy().astype(np.float64)
        assert np.linalg.norm(x1 - ref) <= 1e-5 * np.linalg.norm(ref)


def test_graph_replay_and_host_entry_point_equal_single_steps(binding):
    """casgd_outer_steps (CUDA-graph replay) and casgd_outer_steps_host against repeated casgd_outer_step: bitwise-equal
    x wherever the same kernels run (every reduction in the library has a fixed order), equal to rounding otherwise."""
    cfg = synth.config(4, m=20000, n=512)
    X_d, y_d, _, _ = device_dataset(cfg)
    s, b, steps = 8, 64, 21                     # 21 = 8 + 8 + 5 singles: exercises both graph lengths
    idx = synth.epoch_indices(cfg, 42, 0)[: steps * s * b].copy()
    idx_d = torch.from_numpy(idx).cuda()
    with binding.Casgd(X_d, y_d, cfg.loss) as cg:
        xa = torch.zeros(cfg.n, device="cuda")
        for h in range(steps):
            cg.outer_step(idx_d[h * s * b:(h + 1) * s * b], xa, s, b, cfg.eta)
        xb = torch.zeros(cfg.n, device="cuda")
        n0 = cg.launch_count()
        cg.outer_steps(idx_d, xb, s, b, cfg.eta)
        assert cg.launch_count() > n0
        cg.sync()
        # the pipelined graphs compute r in a kernel of its own (FP32 FMA order instead of the tensor core's): same
        # iterate up to rounding; with CASGD_OPT_OVERLAP = 0 the graphs replay the single steps' kernels, bit for bit
        assert torch.linalg.norm(xa - xb) <= 1e-5 * torch.linalg.norm(xa)
        cg.set_option(binding.OPT_OVERLAP, 0)
        xs = torch.zeros(cfg.n, device="cuda")
        cg.outer_steps(idx_d, xs, s, b, cfg.eta)
        cg.sync()
        assert torch.equal(xa, xs)
        cg.set_option(binding.OPT_OVERLAP, 2)
        xh = torch.zeros(cfg.n).pin_memory()
        idx_h = torch.from_numpy(idx).pin_memory()
        cg.outer_steps_host(idx_h, xh, s, b, cfg.eta)
        assert torch.equal(xb.cpu(), xh)
        # one step per call (the static host graph: staging copies, shadow rebuild, step, copy back), from pageable memory too
        x1 = torch.zeros(cfg.n)
        for h in range(steps):
            cg.outer_steps_host(torch.from_numpy(idx[h * s * b:(h + 1) * s * b].copy()), x1, s, b, cfg.eta, n_steps=1)
        assert torch.equal(xa.cpu(), x1)
        # the synchronous entry point reports a row index outside [0, m) itself; the next call is clean again
        bad = idx[: s * b].copy()
        bad[5] = cfg.m
        with pytest.raises(binding.CasgdError):
            cg.outer_steps_host(torch.from_numpy(bad), torch.zeros(cfg.n), s, b, cfg.eta, n_steps=1)
        x2 = torch.zeros(cfg.n)
        cg.outer_steps_host(torch.from_numpy(idx[: s * b].copy()), x2, s, b, cfg.eta, n_steps=1)
        assert torch.isfinite(x2).all()


@pytest.mark.parametrize("overlap", [0, 1, 2], ids=["sequential", "gather-aside", "pipelined"])
@pytest.mark.parametrize("ci,m,n,s,b", [(3, 6000, 520, 5, 32), (2, 5000, 1024, 3, 128)])
def test_next_step_gather_on_the_side_branch_changes_nothing(binding, oracle_mod, ci, m, n, s, b, overlap):
    """CASGD_OPT_OVERLAP: inside the graphs of casgd_outer_steps the next step's rows are gathered (mode 1), or gathered
    and their Gram matrix computed (mode 2, the margin then being a kernel of its own), on a side branch beside this
    step's recurrence and update. The iterate equals repeated casgd_outer_step bit for bit in modes 0 and 1 (same
    kernels), to rounding in mode 2 (its margin is a kernel of its own), and the last step's exported intermediates (taken
    from the stage that step used) match oracle O1."""
    cfg = synth.config(ci, m=m, n=n)
    X_d, y_d, A_bits, y = device_dataset(cfg)
    steps = 64 + 8 + 8 + 1                      # a 64-step graph, two 8-step graphs, a single
    idx = np.concatenate([synth.epoch_indices(cfg, 42, e) for e in range(-(-steps * s * b // m) + 1)])[: steps * s * b].copy()
    idx_d = torch.from_numpy(idx).cuda()
    eta = cfg.eta * 0.25
    with binding.Casgd(X_d, y_d, cfg.loss) as cg:
        cg.set_option(binding.OPT_OVERLAP, overlap)
        xa = torch.zeros(cfg.n, device="cuda")
        for h in range(steps - 9):
            cg.outer_step(idx_d[h * s * b:(h + 1) * s * b], xa, s, b, eta)
        xb = torch.zeros(cfg.n, device="cuda")
        cg.outer_steps(idx_d[: (steps - 9) * s * b], xb, s, b, eta)      # 64 + 8: ends on an 8-step graph (stage 1)
        cg.sync()
        same = (lambda p, q: torch.equal(p, q)) if overlap < 2 else (lambda p, q: bool(torch.linalg.norm(p - q) <= 1e-4 * torch.linalg.norm(p)))
        assert same(xa, xb)
        x0 = xb.cpu().numpy().copy()
        cg.outer_steps(idx_d[(steps - 9) * s * b: (steps - 1) * s * b], xb, s, b, eta)
        cg.sync()
        for h in range(steps - 9, steps - 2):
            cg.outer_step(idx_d[h * s * b:(h + 1) * s * b], xa, s, b, eta)
        x_before_last = xa.cpu().numpy().copy()
        cg.outer_step(idx_d[(steps - 2) * s * b:(steps - 1) * s * b], xa, s, b, eta)
        cg.sync()
        assert same(xa, xb)
        # the last step of the 8-step graph, against the oracle from the same FP32 bits
        xc = torch.from_numpy(x0.copy()).cuda()
        cg.outer_steps(idx_d[(steps - 9) * s * b: (steps - 1) * s * b], xc, s, b, eta)
        cg.sync()
        last = idx[(steps - 2) * s * b:(steps - 1) * s * b]
        ref = oracle_mod.outer_step_gram(A_bits, y, last, x_before_last.astype(np.float64), s, b, eta, cfg.loss, shadow=True)
        compare_last_step(oracle_mod, cg, ref, y[last], x_before_last, xc, s, b, eta, cfg.loss, binding)


def _random_shapes(count, seed):
    rng = np.random.default_rng(seed)
    out = []
    for _ in range(count):
        loss_cfg = int(rng.choice([0, 2, 4]))               # logistic, linear, Poisson generators
        n = int(rng.choice([9, 18, 40, 64, 100, 257, 520, 777, 1024, 1500]))
        b = int(rng.choice([4, 8, 13, 16, 24, 32, 48, 64, 100, 128]))
        s = int(rng.choice([1, 1, 2, 3, 5, 8, 12]))
        while s * b > 1200:
            s = max(1, s // 2)
        out.append((loss_cfg, n, s, b))
    return out


@pytest.mark.parametrize("ci,n,s,b", _random_shapes(28, 2026))
def test_default_paths_on_random_shapes(binding, oracle_mod, ci, n, s, b):
    """Whatever kernels the library picks by itself for a shape (one-launch kernels, narrow / 128-tile / pair Gram, each
    recurrence kernel, fused or stand-alone update): one step against oracle O1, then an 8-step call (pipelined graph or
    one launch) whose last step is checked from the bits it started from."""
    m = 3000
    cfg = synth.config(ci, m=m, n=n)
    X_d, y_d, A_bits, y = device_dataset(cfg)
    rng = np.random.default_rng(n * 1000 + s * 10 + b)
    idx = rng.integers(0, m, 8 * s * b).astype(np.int32)                   # with duplicates
    eta = min(cfg.eta, 0.05)
    x0 = random_x(n, 17, 0.3)
    with binding.Casgd(X_d, y_d, cfg.loss) as cg:
        check_step_against_oracle(oracle_mod, cg, A_bits, y, idx[: s * b], x0, s, b, eta, cfg.loss, binding)
        cg.set_option(binding.OPT_SNAPSHOT, 1)
        x7 = torch.from_numpy(x0.copy()).cuda()
        cg.outer_steps(torch.from_numpy(idx[: 7 * s * b]).cuda(), x7, s, b, eta)
        cg.sync()
        x8 = torch.from_numpy(x0.copy()).cuda()
        n0 = cg.launch_count()
        cg.outer_steps(torch.from_numpy(idx).cuda(), x8, s, b, eta)
        cg.sync()
        one_launch = cg.launch_count() - n0 == 1
        x_before = x7.cpu().numpy().copy() if one_launch else cg.debug(binding.DBG_XSNAP).copy()
        last = idx[7 * s * b:]
        ref = oracle_mod.outer_step_gram(A_bits, y, last, x_before.astype(np.float64), s, b, eta, cfg.loss, shadow=True)
        compare_last_step(oracle_mod, cg, ref, y[last], x_before, x8, s, b, eta, cfg.loss, binding)


def test_pipelined_graphs_of_two_contexts_and_shapes_interleaved(binding):
    """Robustness of the graph plumbing: two contexts on one device, each replaying pipelined graphs of two different
    (s, b) in alternation, with a workspace growth in between -- every call must give what the same call gives on a fresh
    context in the sequential schedule (to FP32 rounding: the pipelined margin is a kernel of its own)."""
    cfgs = [synth.config(4, m=6000, n=512), synth.config(3, m=5000, n=1000)]
    data = [device_dataset(c) for c in cfgs]
    shapes = [(3, 64), (8, 32), (5, 64), (12, 32)]                 # the last one grows the workspaces
    steps = 16
    rng = np.random.default_rng(8)
    idxs = {(ci, sh): torch.from_numpy(rng.integers(0, cfgs[ci].m, steps * sh[0] * sh[1]).astype(np.int32)).cuda()
            for ci in range(2) for sh in shapes}

    def run(schedule, interleaved):
        out = {}
        ctxs = [binding.Casgd(d[0], d[1], c.loss) for d, c in zip(data, cfgs)]
        try:
            for cg in ctxs:
                cg.set_option(binding.OPT_OVERLAP, schedule)
            order = [(ci, sh) for sh in shapes for ci in range(2)] if interleaved else [(ci, sh) for ci in range(2) for sh in shapes]
            for rep in range(2):
                for ci, sh in order:
                    x = torch.full((cfgs[ci].n,), 0.01 * (rep + 1), device="cuda")
                    ctxs[ci].outer_steps(idxs[(ci, sh)], x, sh[0], sh[1], min(cfgs[ci].eta, 0.02))
                    out[(ci, sh, rep)] = x
            for cg in ctxs:
                cg.sync()
        finally:
            for cg in ctxs:
                cg.close()
        return out

    ref = run(0, False)
    got = run(2, True)
    for k in ref:
        assert torch.isfinite(got[k]).all()
        assert torch.linalg.norm(got[k] - ref[k]) <= 2e-5 * torch.linalg.norm(ref[k]), k


# (config, m, n, s, b, CASGD_OPT_MINI): 2 / 3 = the one-CTA / the cluster kernel whenever the step fits it, whatever the
# measured crossovers
MINI_SHAPES = [(0, 8192, 64, 4, 16, 2), (1, 20000, 18, 1, 64, 2), (1, 20000, 18, 2, 64, 2), (4, 6000, 512, 1, 16, 2),
               (0, 4097, 64, 7, 13, 2), (3, 3000, 100, 3, 24, 2), (0, 5000, 33, 2, 5, 2), (4, 6000, 512, 2, 16, 2),
               (2, 20000, 1024, 1, 8, 2), (1, 9000, 18, 1, 500, 2), (0, 9000, 120, 1, 130, 1), (0, 8192, 64, 4, 16, 1),
               # s = 1 with wide rows: one launch of one column-split cluster (s1_cluster.cu)
               (4, 6000, 512, 1, 64, 1), (3, 5000, 2000, 1, 32, 1), (2, 20000, 4096, 1, 128, 1), (3, 5000, 1001, 1, 40, 1),
               (4, 6000, 256, 1, 16, 1), (0, 7000, 300, 1, 256, 1), (0, 8192, 64, 1, 16, 3), (1, 9000, 100, 1, 7, 3),
               # ... with eight rows per lane group in its margin (b >= 8 x the groups), ragged rows and chunks
               (4, 6000, 512, 1, 256, 1), (3, 5000, 1100, 1, 200, 1)]


@pytest.mark.parametrize("ci,m,n,s,b,mode", MINI_SHAPES)
def test_one_launch_kernel_for_tiny_steps(binding, oracle_mod, ci, m, n, s, b, mode):
    """mini_step.cu / s1_cluster.cu: steps that fit one SM, and s = 1 steps with wide rows (one
    column-split cluster), run all iterations of a call in ONE launch. One
    step against oracle O1 element by element (gather bit-exact, G, r, z, u, x); a 9-step call equals 9 single-step
    calls bit for bit and is a single launch; the kernel-per-stage path gives the same iterate up to FP32 summation
    order; an out-of-range index is reported, not read."""
    cfg = synth.config(ci, m=m, n=n)
    X_d, y_d, A_bits, y = device_dataset(cfg)
    steps = 9
    idx = np.concatenate([synth.epoch_indices(cfg, 42, e) for e in range(-(-steps * s * b // m) + 1)])[: steps * s * b].copy()
    idx_d = torch.from_numpy(idx).cuda()
    x0 = random_x(n, 11, 0.4)
    eta = cfg.eta * 0.5
    with binding.Casgd(X_d, y_d, cfg.loss) as cg:
        cg.set_option(binding.OPT_MINI, mode)
        n0 = cg.launch_count()
        check_step_against_oracle(oracle_mod, cg, A_bits, y, idx[: s * b], x0, s, b, eta, cfg.loss, binding)
        assert cg.launch_count() - n0 == 1, "the step did not run as one launch"
        xa = torch.from_numpy(x0.copy()).cuda()
        for h in range(steps):
            cg.outer_step(idx_d[h * s * b:(h + 1) * s * b], xa, s, b, eta)
        xc = torch.from_numpy(x0.copy()).cuda()
        cg.outer_steps(idx_d[: (steps - 1) * s * b], xc, s, b, eta)
        cg.sync()
        x_before = xc.cpu().numpy().copy()
        xb = torch.from_numpy(x0.copy()).cuda()
        n0 = cg.launch_count()
        cg.outer_steps(idx_d, xb, s, b, eta)
        cg.sync()
        assert cg.launch_count() - n0 == 1
        assert torch.equal(xa, xb)
        # the last step of the 9-step launch, against the oracle from the iterate before it
        last = idx[(steps - 1) * s * b:]
        ref = oracle_mod.outer_step_gram(A_bits, y, last, x_before.astype(np.float64), s, b, eta, cfg.loss, shadow=True)
        compare_last_step(oracle_mod, cg, ref, y[last], x_before, xb, s, b, eta, cfg.loss, binding)
        # kernel-per-stage path: same iterate up to summation order
        cg.set_option(binding.OPT_MINI, 0)
        xd = torch.from_numpy(x0.copy()).cuda()
        cg.outer_steps(idx_d, xd, s, b, eta)
        cg.sync()
        assert torch.linalg.norm(xd - xb) <= 2e-5 * torch.linalg.norm(xb)
        cg.set_option(binding.OPT_MINI, mode)
        bad = idx[: s * b].copy()
        bad[3] = m + 5
        xe = torch.from_numpy(x0.copy()).cuda()
        cg.outer_step(torch.from_numpy(bad).cuda(), xe, s, b, eta)
        with pytest.raises(binding.CasgdError):
            cg.sync()
        assert torch.isfinite(xe).all()


SPLIT_SHAPES = [(0, 8192, 64, 4, 16), (1, 20000, 18, 5, 64), (2, 4200, 4096, 3, 128), (3, 5000, 2000, 9, 32), (4, 6000, 512, 6, 64),
                (4, 6000, 512, 1, 64), (2, 5000, 1024, 6, 128)]


@pytest.mark.parametrize("mode", ["sequential-auto", "sequential-simt", "sequential-tile128", "sequential-pair256", "pipelined"])
@pytest.mark.parametrize("ci,m,n,s,b", SPLIT_SHAPES)
def test_margin_of_the_fp32_master(binding, oracle_mod, ci, m, n, s, b, mode):
    """CASGD_OPT_MARGIN_SPLIT (Eq. 8, Table 3 column B): the margin is taken of
    the FP32 master -- as three BF16 rows hi / lo / lo2 of the fused tensor-core margin, or by the stand-alone margin kernel
    reading x itself -- so r, and the whole step, match oracle O1 run WITHOUT the BF16 shadow (shadow=False) at the same
    1e-5 tolerances. A negative control shows the default (shadow) margin does not."""
    cfg = synth.config(ci, m=m, n=n)
    X_d, y_d, A_bits, y = device_dataset(cfg)
    idx = synth.epoch_indices(cfg, 42, 0)[: s * b].copy()
    x0 = random_x(n, 5, 0.7)
    gram = {"sequential-auto": 0, "sequential-simt": 1, "sequential-tile128": 2, "sequential-pair256": 3, "pipelined": 0}[mode]
    if gram == 3 and (n < 64 or s * b < 256):
        pytest.skip("the pair kernel needs whole 256-row tiles worth of work")
    with binding.Casgd(X_d, y_d, cfg.loss) as cg:
        cg.set_option(binding.OPT_OVERLAP, 2 if mode == "pipelined" else 0)
        cg.set_option(binding.OPT_GRAM_IMPL, gram)
        cg.set_option(binding.OPT_MARGIN_SPLIT, 1)
        check_step_against_oracle(oracle_mod, cg, A_bits, y, idx, x0, s, b, cfg.eta, cfg.loss, binding, shadow=False)
        # a second step from the updated iterate: the residue rows follow the fused update
        x1 = torch.from_numpy(x0.copy()).cuda()
        cg.outer_step(torch.from_numpy(idx).cuda(), x1, s, b, cfg.eta)
        cg.sync()
        check_step_against_oracle(oracle_mod, cg, A_bits, y, idx, x1.cpu().numpy(), s, b, cfg.eta, cfg.loss, binding, shadow=False)
        if mode == "pipelined":
            # the pipelined GRAPH computes r in the stand-alone margin kernel, from the FP32 x itself: its last step
            # against the oracle from the bits it started from (CASGD_OPT_SNAPSHOT)
            cg.set_option(binding.OPT_SNAPSHOT, 1)
            idx8 = np.concatenate([synth.epoch_indices(cfg, 42, e) for e in range(-(-8 * s * b // m) + 1)])[: 8 * s * b].copy()
            xg = torch.from_numpy(x0.copy()).cuda()
            n0 = cg.launch_count()
            cg.outer_steps(torch.from_numpy(idx8).cuda(), xg, s, b, cfg.eta * 0.25)
            cg.sync()
            if cg.launch_count() - n0 > 1:              # (not the one-launch kernel)
                xs = cg.debug(binding.DBG_XSNAP).copy()
                last = idx8[7 * s * b:]
                ref = oracle_mod.outer_step_gram(A_bits, y, last, xs.astype(np.float64), s, b, cfg.eta * 0.25, cfg.loss, shadow=False)
                compare_last_step(oracle_mod, cg, ref, y[last], xs, xg, s, b, cfg.eta * 0.25, cfg.loss, binding, shadow=False)
        # negative control: with the split off, r is the margin of bf16(x), which is NOT within 1e-5 of Y x
        cg.set_option(binding.OPT_MARGIN_SPLIT, 0)
        with pytest.raises(AssertionError, match="margin"):
            check_step_against_oracle(oracle_mod, cg, A_bits, y, idx, x0, s, b, cfg.eta, cfg.loss, binding, shadow=False)


@pytest.mark.parametrize("ci,m,n,s,b", [(1, 20000, 18, 5, 64), (4, 6000, 512, 3, 64), (0, 4097, 64, 7, 13)])
def test_on_device_sampling_matches_the_oracle_sampler(binding, oracle_mod, ci, m, n, s, b):
    """casgd_outer_steps_sampled draws Alg. 1 line 1's indices on the device (Philox4x32-10, with replacement): the rows it
    gathers are exactly A[oracle.sample_indices(...)], and the iterate equals casgd_outer_steps on those indices bit
    for bit; step numbers continue across calls (first_step)."""
    cfg = synth.config(ci, m=m, n=n)
    X_d, y_d, A_bits, y = device_dataset(cfg)
    seed, steps, sb = 0xC0FFEE1234, 11, s * b
    idx = np.concatenate([oracle_mod.sample_indices(seed, h, sb, m) for h in range(steps)])
    assert len(np.unique(idx)) < len(idx) or m > 50 * len(idx)             # with replacement
    eta = cfg.eta if cfg.loss != synth.POISSON else 0.01
    with binding.Casgd(X_d, y_d, cfg.loss) as cg:
        xa = torch.zeros(n, device="cuda")
        idx_d = torch.from_numpy(idx).cuda()
        cg.outer_steps(idx_d[: 4 * sb], xa, s, b, eta)                      # the same split into calls as below: the same
        cg.outer_steps(idx_d[4 * sb:], xa, s, b, eta)                      # schedules (graph lengths), hence the same kernels
        cg.sync()
        xb = torch.zeros(n, device="cuda")
        cg.outer_steps_sampled(xb, s, b, eta, n_steps=4, seed=seed, first_step=0)
        cg.outer_steps_sampled(xb, s, b, eta, n_steps=steps - 4, seed=seed, first_step=4)
        cg.sync()
        assert torch.equal(xa, xb)
        assert np.array_equal(cg.debug(binding.DBG_Y), A_bits[idx[-sb:]])   # the last step's gathered rows
        # and one sampled step against the oracle itself
        x0 = random_x(n, 9, 0.2)
        xc = torch.from_numpy(x0.copy()).cuda()
        cg.invalidate_shadow()
        cg.outer_steps_sampled(xc, s, b, eta, n_steps=1, seed=seed, first_step=(1 << 40) + 3)
        cg.sync()
        idx1 = oracle_mod.sample_indices(seed, (1 << 40) + 3, sb, m)
        ref = oracle_mod.outer_step_gram(A_bits, y, idx1, x0.astype(np.float64), s, b, eta, cfg.loss, shadow=True)
        from gpu_common import compare_last_step
        compare_last_step(oracle_mod, cg, ref, y[idx1], x0, xc, s, b, eta, cfg.loss, binding)


def _train_gpu(binding, cg, cfg, idx, s):
    x = torch.zeros(cfg.n, device="cuda")
    cg.invalidate_shadow()
    cg.outer_steps(torch.from_numpy(idx).cuda(), x, s, cfg.b, cfg.eta)
    cg.sync()
    return x


def test_config1_training_loss_matches_the_trajectory_oracle(binding, oracle_mod):
    """BASELINE.json:configs[0] in full: 5 epochs = 640 outer steps from x = 0; final F within 0.5 %."""
    cfg = synth.config(0)
    X_d, y_d, A_bits, y = device_dataset(cfg)
    idx = synth.training_indices(cfg, seed=42)
    s = cfg.s_list[0]
    with binding.Casgd(X_d, y_d, cfg.loss) as cg:
        x = _train_gpu(binding, cg, cfg, idx, s)
        F_gpu = cg.loss(x)
    x_ref = oracle_mod.train(A_bits, y, idx, np.zeros(cfg.n), s, cfg.b, cfg.eta, cfg.loss, shadow=True, form="gram")
    F_ref = oracle_mod.full_loss(A_bits, y, x_ref, cfg.loss)
    assert F_ref < 0.6 * math.log(2.0)                    # it trained
    assert abs(F_gpu - F_ref) <= TOL_FINAL_LOSS * F_ref
    # far tighter in practice; the iterate itself stays close too
    assert np.linalg.norm(x.cpu().numpy() - x_ref) <= 1e-3 * np.linalg.norm(x_ref)


@pytest.mark.parametrize("ci,m,n", [(1, 65536, 18), (2, 16384, 1024), (3, 16384, 2000), (4, 32768, 512)])
def test_downsized_training_loss_across_the_s_sweep(binding, oracle_mod, ci, m, n):
    """Configs 2-5 with fewer rows, every s of the sweep, the configured epochs: final F within 0.5 % of
    the trajectory oracle (O2 form), and the losses of different s agree with each other."""
    cfg = synth.config(ci, m=m, n=n)
    X_d, y_d, A_bits, y = device_dataset(cfg)
    idx = synth.training_indices(cfg, seed=42)
    losses = []
    with binding.Casgd(X_d, y_d, cfg.loss) as cg:
        for s in cfg.s_list:
            x = _train_gpu(binding, cg, cfg, idx, s)
            F_gpu = cg.loss(x)
            x_ref = oracle_mod.train(A_bits, y, idx, np.zeros(n), s, cfg.b, cfg.eta, cfg.loss, shadow=True)
            F_ref = oracle_mod.full_loss(A_bits, y, x_ref, cfg.loss)
            assert abs(F_gpu - F_ref) <= TOL_FINAL_LOSS * abs(F_ref), (s, F_gpu, F_ref)
            losses.append(F_gpu)
    assert max(losses) - min(losses) <= 1e-3 * abs(losses[0])
