"""casgd_loss_noalloc (csrc/loss_noalloc.cu): the loss without a context and without any allocation -- its partial sums in
a static __device__ array -- against the existing path (casgd_loss, the context's streaming kernel), on two calls in a
row with different x (the array keeps the first call's contents), on aligned and unaligned rows, a strided X, several
chunks with a ragged tail, and the size limit. Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest
import torch

from paper_2606_18463_b200 import synth

from gpu_common import TOL_LOSS_CALL, require_cuda

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    require_cuda()
    from paper_2606_18463_b200 import build
    build.build()
    from paper_2606_18463_b200 import binding as b
    b.load()
    return b


# (config, m, n): 36-byte rows (2-byte loads), 16-byte-aligned rows, a ragged last chunk, one row
SHAPES = [(1, 20001, 18), (4, 6000, 512), (3, 5000, 1001), (2, 1537, 4096), (0, 1, 64)]


@pytest.mark.parametrize("ci,m,n", SHAPES)
def test_loss_without_allocation_matches_casgd_loss_twice_in_a_row(binding, ci, m, n):
    cfg = synth.config(ci, m=m, n=n)
    ds = synth.make_dataset(cfg, seed=7, device="cuda")
    gen = torch.Generator().manual_seed(3)
    xs = [(torch.randn(n, generator=gen) * s).cuda() for s in (0.2, 0.05)]
    out = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    with binding.Casgd(ds.X_bf16, ds.y, cfg.loss) as cg:
        want = [cg.loss(x) for x in xs]
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    got = []
    for x in xs:                                        # two calls in a row, the second on the first one's leftovers
        binding.loss_noalloc(ds.X_bf16, ds.y, cfg.loss, x, out)
        torch.cuda.synchronize()
        got.append(float(out.item()))
    assert torch.cuda.memory_allocated() == before
    for g, w in zip(got, want):
        assert np.isfinite(g)
        assert abs(g - w) <= TOL_LOSS_CALL * abs(w), (g, w)
    # the same bits on a repeat (fixed summation order), and a strided X (row stride > n) is used in place
    binding.loss_noalloc(ds.X_bf16, ds.y, cfg.loss, xs[0], out)
    torch.cuda.synchronize()
    assert float(out.item()) == got[0]
    wide = torch.zeros(m, n + 11, dtype=torch.bfloat16, device="cuda")
    wide[:, :n] = ds.X_bf16
    binding.loss_noalloc(wide[:, :n], ds.y, cfg.loss, xs[1], out)
    torch.cuda.synchronize()
    assert abs(float(out.item()) - want[1]) <= TOL_LOSS_CALL * abs(want[1])


def test_loss_without_allocation_rejects_sizes_beyond_its_scratch(binding):
    m = 256 * 16384 + 1                                 # one row more than the static array covers
    X = torch.zeros(m, 1, dtype=torch.bfloat16, device="cuda")
    y = torch.ones(m, device="cuda")
    x = torch.zeros(1, device="cuda")
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    with pytest.raises(binding.CasgdError) as e:
        binding.loss_noalloc(X, y, synth.LOGISTIC, x, out)
    assert e.value.status == binding.EINVAL and "exceeds the static scratch" in str(e.value)
    binding.loss_noalloc(X[: m - 1], y[: m - 1], synth.LOGISTIC, x, out)     # the maximum itself: F(0) = log 2
    torch.cuda.synchronize()
    assert float(out.item()) == pytest.approx(np.log(2.0), rel=1e-6)
