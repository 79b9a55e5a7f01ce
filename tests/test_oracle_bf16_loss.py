"""Pins for the oracle's BF16 helpers and loss family (CPU only).

Each test checks the oracle against something other than itself: torch's BF16 cast, hand-built
rounding ties, constants the paper prints (tests/golden/paper_constants.txt), finite differences,
closed forms and scipy's expit.
"""
import math
import os

import numpy as np
import pytest
import torch
from scipy.special import expit

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")) as fh:
    for line in fh:
        line = line.split("#")[0].split()
        if len(line) == 2:
            GOLD[line[0]] = float(line[1])

LOSSES = (0, 1, 2)  # logistic, linear, poisson


# ------------------------------------------------------------------ BF16 ---

def test_bf16_widen_narrow_identity_exhaustive(oracle_mod):
    bits = np.arange(1 << 16, dtype=np.uint16)
    wide = oracle_mod.bf16_to_f64(bits)
    finite = np.isfinite(wide)
    back = oracle_mod.f32_to_bf16(wide[finite].astype(np.float32))
    assert np.array_equal(back, bits[finite])
    back64 = oracle_mod.f64_to_bf16(wide[finite])
    assert np.array_equal(back64, bits[finite])
    # widening agrees with torch bit for bit on every pattern (NaNs compare as bits of float32)
    t = torch.from_numpy(bits.view(np.int16)).view(torch.bfloat16).double().numpy()
    assert np.array_equal(t[finite], wide[finite])


def test_bf16_rounding_matches_torch(oracle_mod):
    rng = np.random.default_rng(0)
    vals = np.concatenate([
        rng.standard_normal(20000).astype(np.float32),
        (rng.standard_normal(5000) * 1e-30).astype(np.float32),
        (rng.standard_normal(5000) * 1e30).astype(np.float32),
        rng.integers(0, 1 << 32, 20000, dtype=np.uint64).astype(np.uint32).view(np.float32),
        np.array([0.0, -0.0, np.inf, -np.inf, 3.3895314e38, 1e-45, 1.17549435e-38], dtype=np.float32),
    ])
    vals = vals[~np.isnan(vals)]
    ours = oracle_mod.f32_to_bf16(vals)
    ref = torch.from_numpy(vals).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(ours, ref)


def test_bf16_ties_to_even_hand_built(oracle_mod):
    # 1 + 2^-8 lies exactly between BF16 1.0 (0x3f80, even) and 1.0078125 (0x3f81): -> even
    assert oracle_mod.f32_to_bf16(np.float32(1 + 2.0 ** -8))[()] == 0x3F80
    # 1 + 3*2^-8 lies between 0x3f81 (odd) and 0x3f82 (even): -> 0x3f82
    assert oracle_mod.f32_to_bf16(np.float32(1 + 3 * 2.0 ** -8))[()] == 0x3F82
    # just above / below a tie
    assert oracle_mod.f32_to_bf16(np.float32(1 + 2.0 ** -8 + 2.0 ** -20))[()] == 0x3F81
    assert oracle_mod.f32_to_bf16(np.float32(1 + 2.0 ** -8 - 2.0 ** -20))[()] == 0x3F80
    assert oracle_mod.f32_to_bf16(np.float32(-(1 + 3 * 2.0 ** -8)))[()] == 0xBF82


def test_f64_to_bf16_has_no_double_rounding(oracle_mod):
    # d is above the tie by 2^-40: the binary32 route rounds d to the tie first and then to even (0x3f80),
    # a correctly rounded binary64 -> BF16 conversion gives 0x3f81.
    d = 1 + 2.0 ** -8 + 2.0 ** -40
    assert np.float32(d) == np.float32(1 + 2.0 ** -8)
    assert oracle_mod.f64_to_bf16(d)[()] == 0x3F81
    assert oracle_mod.f64_to_bf16(1 + 2.0 ** -8 - 2.0 ** -40)[()] == 0x3F80
    assert oracle_mod.f64_to_bf16(-d)[()] == 0xBF81
    # nearest in binary64 on random values: |bf16(d) - d| is minimal among neighbours
    rng = np.random.default_rng(1)
    ds = rng.standard_normal(3000) * np.exp(rng.uniform(-20, 20, 3000))
    got = oracle_mod.f64_to_bf16(ds)
    for d_, b_ in zip(ds, got):
        err = abs(oracle_mod.bf16_to_f64(b_) - d_)
        for nb in (b_ - 1, b_ + 1):
            assert err <= abs(oracle_mod.bf16_to_f64(np.uint16(nb)) - d_)


def test_bf16_unit_roundoff_is_the_papers(oracle_mod):
    # Table 3: u_BF16 ~ 4e-3. RNE to 8 significand bits has max relative error 2^-8 = 3.9e-3.
    rng = np.random.default_rng(2)
    v = (rng.uniform(1.0, 2.0, 50000)).astype(np.float32)
    rel = np.abs(oracle_mod.bf16_to_f64(oracle_mod.f32_to_bf16(v)) - v.astype(np.float64)) / v
    assert rel.max() <= 2.0 ** -8
    assert rel.max() > 0.9 * 2.0 ** -8
    assert abs(rel.max() - GOLD["u_bf16"]) < 0.1 * GOLD["u_bf16"]
    assert abs(2.0 ** -24 - GOLD["u_fp32"]) < 0.1 * GOLD["u_fp32"]
    assert abs(2 * 2.0 ** -8 - GOLD["two_u16"]) < 0.1 * GOLD["two_u16"]


# ------------------------------------------------------------ loss family ---

def _labels(loss, rng, k):
    if loss == 0:
        return rng.choice([-1.0, 1.0], k)
    if loss == 1:
        return rng.standard_normal(k)
    return rng.poisson(1.5, k).astype(np.float64)


@pytest.mark.parametrize("loss", LOSSES)
def test_lprime_is_derivative_of_L(oracle_mod, loss):
    """u = dL/dr (PAPER.md:L31 gives L, L59 gives delta = -dL/dr): central finite difference in binary64."""
    rng = np.random.default_rng(3 + loss)
    zs = rng.uniform(-6, 6, 200)
    ys = _labels(loss, rng, 200)
    h = 1e-5
    for z, y in zip(zs, ys):
        fd = (oracle_mod.loss_value(z + h, y, loss) - oracle_mod.loss_value(z - h, y, loss)) / (2 * h)
        assert abs(oracle_mod.lprime(z, y, loss) - fd) <= 1e-8 * max(1.0, abs(fd)) + 1e-9


def test_residual_formulas_printed_in_the_paper(oracle_mod):
    """delta = y(1 - sigma(y r)) logistic; y - r linear; y - exp(r) Poisson; u = -delta."""
    rng = np.random.default_rng(7)
    for z in rng.uniform(-30, 30, 300):
        for y in (-1.0, 1.0):
            delta = y * (1.0 - expit(y * z))
            assert abs(oracle_mod.lprime(z, y, 0) + delta) <= 1e-15 + 1e-13 * abs(delta)
        y = rng.standard_normal()
        assert oracle_mod.lprime(z, y, 1) == z - y
        yk = float(rng.poisson(2.0))
        assert abs(oracle_mod.lprime(z, yk, 2) - (math.exp(z) - yk)) <= 1e-15 * math.exp(abs(z))


def test_logistic_is_stable_at_large_margins(oracle_mod):
    for t in (50.0, 500.0, 800.0, 5000.0):
        assert oracle_mod.lprime(t, 1.0, 0) == pytest.approx(-math.exp(-t) if t < 700 else 0.0, abs=1e-300, rel=1e-12)
        assert oracle_mod.lprime(-t, 1.0, 0) == pytest.approx(-1.0, rel=1e-15)
        assert oracle_mod.loss_value(-t, 1.0, 0) == pytest.approx(t, rel=1e-15)
        assert oracle_mod.loss_value(t, 1.0, 0) == pytest.approx(math.exp(-t) if t < 700 else 0.0, abs=1e-300, rel=1e-12)
        assert math.isfinite(oracle_mod.loss_value(-t, -1.0, 0))


def test_lipschitz_constants_of_the_residual(oracle_mod):
    """L_sigma = 1/4 (logistic), 1 (linear) and |delta| <= 1 (logistic): PAPER.md:L31, L164."""
    zs = np.linspace(-12, 12, 4801)
    for y in (-1.0, 1.0):
        u = np.array([oracle_mod.lprime(z, y, 0) for z in zs])
        slope = np.abs(np.diff(u) / np.diff(zs))
        assert slope.max() <= GOLD["lsigma_logistic"] + 1e-9
        assert slope.max() >= GOLD["lsigma_logistic"] - 1e-4          # attained at z = 0
        assert np.abs(u).max() <= GOLD["dmax_logistic"]
    u = np.array([oracle_mod.lprime(z, 0.3, 1) for z in zs])
    assert np.allclose(np.diff(u) / np.diff(zs), GOLD["lsigma_linear"], rtol=0, atol=1e-9)


@pytest.mark.parametrize("loss", LOSSES)
def test_full_loss_closed_form_at_zero(oracle_mod, loss):
    """F(0): logistic ln 2; Poisson e^0 - y*0 = 1; linear mean(y^2)/2 (from L at PAPER.md:L31)."""
    rng = np.random.default_rng(11)
    m, n = 257, 13
    A = oracle_mod.f32_to_bf16(rng.standard_normal((m, n)).astype(np.float32))
    y = _labels(loss, rng, m).astype(np.float32)
    F0 = oracle_mod.full_loss(A, y, np.zeros(n), loss)
    want = {0: math.log(2.0), 1: float(np.mean(y.astype(np.float64) ** 2) / 2), 2: 1.0}[loss]
    assert F0 == pytest.approx(want, rel=1e-14)


@pytest.mark.parametrize("loss", LOSSES)
def test_full_loss_matches_numpy_definition(oracle_mod, loss):
    rng = np.random.default_rng(12)
    m, n = 300, 21
    A = oracle_mod.f32_to_bf16((rng.standard_normal((m, n)) / math.sqrt(n)).astype(np.float32))
    y = _labels(loss, rng, m).astype(np.float32)
    x = rng.standard_normal(n)
    r = oracle_mod.bf16_to_f64(A) @ x
    yd = y.astype(np.float64)
    want = {0: np.logaddexp(0.0, -yd * r), 1: (r - yd) ** 2 / 2, 2: np.exp(r) - yd * r}[loss].mean()
    assert oracle_mod.full_loss(A, y, x, loss) == pytest.approx(want, rel=1e-13)
    # row stride larger than n (padded storage) gives the same value
    Apad = np.zeros((m, n + 11), np.uint16)
    Apad[:, :n] = A
    Apad[:, n:] = 0x7FC0  # NaN padding must never be read
    assert oracle_mod.full_loss(Apad[:, :n], y, x, loss) == pytest.approx(want, rel=1e-13)
