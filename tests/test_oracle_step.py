"""Pins for the oracle's outer step (O1 Gram form, O2 sequential form), CPU only.

What fixes the answers here is the paper and the mathematics, not the oracle: pure-Python brute
force written separately (O0), the closed-form first block from x = 0, textbook mini-batch SGD
in numpy, the identity "one CA-SGD block == s mini-batch SGD steps", LAPACK's
triangular solve and the terminating Neumann series for the linear loss (L180), and the
structure of a Gram matrix (L166).
"""
import math

import numpy as np
import pytest
import scipy.linalg
from scipy.special import expit

from paper_2606_18463_b200 import synth

LOSSES = (0, 1, 2)


def _problem(oracle_mod, loss, m, n, seed, row_scale=None):
    rng = np.random.default_rng(seed)
    X = rng.standard_normal((m, n)) / math.sqrt(n) * (row_scale or 1.0)
    A = oracle_mod.f32_to_bf16(X.astype(np.float32))
    w = rng.standard_normal(n)
    score = oracle_mod.bf16_to_f64(A) @ w
    if loss == 0:
        y = np.where(score + 0.3 * rng.standard_normal(m) >= 0, 1.0, -1.0)
    elif loss == 1:
        y = score + 0.1 * rng.standard_normal(m)
    else:
        y = rng.poisson(np.exp(0.5 * score)).astype(np.float64)
    return A, y.astype(np.float32), rng


def _lprime_np(z, y, loss):
    """The residuals as the paper prints them, u = -delta, via scipy's expit."""
    if loss == 0:
        return -y * (1.0 - expit(y * z))
    if loss == 1:
        return z - y
    return np.exp(z) - y


# ----------------------------------------------------------- O0 brute force ---

def _brute_force(A_bits, y, idx, x_master, x_hat, s, b, eta, loss):
    """O0: scalar Python loops over (row, row, feature); no numpy arithmetic, no symmetry, no blocking."""
    n = A_bits.shape[1]
    sb = s * b

    def widen(h):
        import struct
        return struct.unpack("<f", struct.pack("<I", int(h) << 16))[0]

    Y = [[widen(A_bits[idx[t], k]) for k in range(n)] for t in range(sb)]
    yI = [float(y[idx[t]]) for t in range(sb)]
    r = [math.fsum(Y[t][k] * x_hat[k] for k in range(n)) for t in range(sb)]
    G = [[math.fsum(Y[i][k] * Y[j][k] for k in range(n)) for j in range(sb)] for i in range(sb)]
    alpha = eta / b
    u, z = [0.0] * sb, [0.0] * sb
    for j in range(s):
        for i in range(b):
            row = j * b + i
            corr = math.fsum(G[row][t] * u[t] for t in range(j * b))
            z[row] = r[row] - alpha * corr
            t_ = yI[row] * z[row]
            if loss == 0:
                u[row] = -yI[row] / (1.0 + math.exp(t_))
            elif loss == 1:
                u[row] = z[row] - yI[row]
            else:
                u[row] = math.exp(z[row]) - yI[row]
    g = [math.fsum(Y[t][k] * u[t] for t in range(sb)) for k in range(n)]
    x_out = [x_master[k] - alpha * g[k] for k in range(n)]
    return np.array(G), np.array(r), np.array(z), np.array(u), np.array(g), np.array(x_out)


@pytest.mark.parametrize("loss", LOSSES)
@pytest.mark.parametrize("s,b,n", [(1, 5, 7), (3, 4, 6), (4, 3, 9), (6, 2, 3)])
def test_gram_form_matches_brute_force(oracle_mod, loss, s, b, n):
    A, y, rng = _problem(oracle_mod, loss, 40, n, 100 + loss)
    idx = synth.iid_indices(40, s * b, seed=5)            # with replacement: duplicates occur
    x = rng.standard_normal(n).astype(np.float32).astype(np.float64)
    x_hat = oracle_mod.bf16_to_f64(oracle_mod.f64_to_bf16(x))
    res = oracle_mod.outer_step_gram(A, y, idx, x, s, b, 0.7, loss, shadow=True)
    G, r, z, u, g, x_out = _brute_force(A, y, idx, x, x_hat, s, b, 0.7, loss)
    for got, want in ((res.G, G), (res.r, r), (res.z, z), (res.u, u), (res.g, g), (res.x_out, x_out)):
        assert np.allclose(got, want, rtol=1e-13, atol=1e-15)
    assert np.array_equal(res.Y_bits, A[idx])


# --------------------------------------------- closed forms and special cases ---

@pytest.mark.parametrize("loss", LOSSES)
def test_first_block_from_zero(oracle_mod, loss):
    """x = 0 => r = 0 => u_0 = -y/2 (logistic), -y (linear), 1 - y (Poisson); s = 1: x_1 = -alpha Y^T u_0."""
    A, y, _ = _problem(oracle_mod, loss, 64, 10, 200 + loss)
    b, eta = 8, 0.3
    idx = np.arange(16, 16 + b, dtype=np.int32)
    res = oracle_mod.outer_step_gram(A, y, idx, np.zeros(10), 1, b, eta, loss)
    yd = y[idx].astype(np.float64)
    want_u = {0: -yd / 2, 1: -yd, 2: 1.0 - yd}[loss]
    assert np.array_equal(res.r, np.zeros(b))
    assert np.allclose(res.u, want_u, rtol=1e-15, atol=0)
    Y = oracle_mod.bf16_to_f64(A[idx])
    assert np.allclose(res.x_out, -(eta / b) * (Y.T @ want_u), rtol=1e-14, atol=1e-17)


@pytest.mark.parametrize("loss", LOSSES)
def test_s1_is_textbook_minibatch_sgd(oracle_mod, loss):
    """s = 1, no BF16 shadow: x+ = x - (eta/b) Y^T l'(Y x, y_I)."""
    A, y, rng = _problem(oracle_mod, loss, 90, 12, 300 + loss)
    b, eta = 10, 0.4
    idx = synth.iid_indices(90, b, seed=1)
    x = rng.standard_normal(12) * 0.5
    Y = oracle_mod.bf16_to_f64(A[idx])
    want = x - (eta / b) * (Y.T @ _lprime_np(Y @ x, y[idx].astype(np.float64), loss))
    o1 = oracle_mod.outer_step_gram(A, y, idx, x, 1, b, eta, loss, shadow=False)
    o2 = oracle_mod.outer_step_seq(A, y, idx, x, 1, b, eta, loss, shadow=False)
    assert np.allclose(o1.x_out, want, rtol=1e-14, atol=1e-16)
    assert np.allclose(o2.x_out, want, rtol=1e-14, atol=1e-16)


@pytest.mark.parametrize("loss", LOSSES)
@pytest.mark.parametrize("s,b,n", [(2, 3, 5), (8, 4, 16), (16, 8, 40), (64, 2, 12), (5, 16, 3)])
def test_ca_block_equals_s_sgd_steps(oracle_mod, loss, s, b, n):
    """"the exact CA-SGD block with parameter s is the composition of s mini-batch SGD
    steps". Gram form (O1) vs s separate textbook steps in numpy, vs O2, to 1e-12 relative;
    indices drawn with replacement so rows repeat inside and across mini-batches."""
    m = 50
    A, y, rng = _problem(oracle_mod, loss, m, n, 400 + loss, row_scale=0.5)
    idx = synth.iid_indices(m, s * b, seed=s * 31 + b)
    assert len(set(idx.tolist())) < s * b or s * b < 8          # duplicates really occur
    eta = 0.25
    x = (rng.standard_normal(n) * 0.3).astype(np.float32).astype(np.float64)
    x_hat = oracle_mod.bf16_to_f64(oracle_mod.f64_to_bf16(x))
    # s textbook steps starting from the margin input x_hat
    v = x_hat.copy()
    z_ref, u_ref = [], []
    for j in range(s):
        rows = idx[j * b:(j + 1) * b]
        Y = oracle_mod.bf16_to_f64(A[rows])
        zj = Y @ v
        uj = _lprime_np(zj, y[rows].astype(np.float64), loss)
        v = v - (eta / b) * (Y.T @ uj)
        z_ref.append(zj)
        u_ref.append(uj)
    x_ref = x + (v - x_hat)                                      # displacement applied to the master
    o1 = oracle_mod.outer_step_gram(A, y, idx, x, s, b, eta, loss, shadow=True)
    o2 = oracle_mod.outer_step_seq(A, y, idx, x, s, b, eta, loss, shadow=True)
    scale = max(1.0, np.abs(np.concatenate(u_ref)).max())
    for o in (o1, o2):
        assert np.linalg.norm(o.x_out - x_ref) <= 1e-12 * max(np.linalg.norm(x_ref), 1e-3)
        assert np.abs(o.z - np.concatenate(z_ref)).max() <= 1e-12 * max(1.0, np.abs(np.concatenate(z_ref)).max())
        assert np.abs(o.u - np.concatenate(u_ref)).max() <= 1e-12 * scale
    assert np.linalg.norm(o1.x_out - o2.x_out) <= 1e-12 * max(np.linalg.norm(o2.x_out), 1e-3)


def test_linear_loss_recurrence_is_a_triangular_solve(oracle_mod):
    """Linear loss: u = z - y and z = r - alpha G_L u  =>  (I + alpha G_L) u = r - y with G_L the strict
    block-lower part of G. Check against LAPACK and the terminating Neumann series."""
    s, b, n, m = 7, 5, 11, 60
    A, y, rng = _problem(oracle_mod, 1, m, n, 500)
    idx = synth.iid_indices(m, s * b, seed=9)
    x = rng.standard_normal(n)
    eta = 0.9
    res = oracle_mod.outer_step_gram(A, y, idx, x, s, b, eta, 1, shadow=False)
    Y = oracle_mod.bf16_to_f64(A[idx])
    G = Y @ Y.T
    blk = np.arange(s * b) // b
    GL = np.where(blk[:, None] > blk[None, :], G, 0.0)
    alpha = eta / b
    rhs = Y @ x - y[idx].astype(np.float64)
    u_solve = scipy.linalg.solve_triangular(np.eye(s * b) + alpha * GL, rhs, lower=True, unit_diagonal=True)
    assert np.allclose(res.u, u_solve, rtol=1e-12, atol=1e-14)
    # nilpotency: G_L^s = 0, so the Neumann series terminates after s terms
    assert np.count_nonzero(np.linalg.matrix_power(GL, s)) == 0
    term, u_series = rhs.copy(), rhs.copy()
    for _ in range(1, s):
        term = -alpha * (GL @ term)
        u_series += term
    assert np.allclose(res.u, u_series, rtol=1e-12, atol=1e-14)
    # the entries inside a diagonal block must not matter: an oracle that used the full lower
    # triangle (k <= j within a block) would differ from the block-strict solve
    GT = np.tril(G, -1)
    u_wrong = scipy.linalg.solve_triangular(np.eye(s * b) + alpha * GT, rhs, lower=True, unit_diagonal=True)
    assert np.abs(u_wrong - res.u).max() > 1e-6


def test_gram_matrix_structure(oracle_mod):
    """G = Y Y^T: symmetric, G_ii = ||y_i||^2, |G_ij| <= ||y_i|| ||y_j||, PSD, rank <= n, ||G||_F <= sb for
    rows of norm <= 1 (Assumption 5.3)."""
    m, n, s, b = 200, 6, 8, 4
    rng = np.random.default_rng(600)
    X = rng.standard_normal((m, n))
    X /= np.linalg.norm(X, axis=1, keepdims=True) * 1.01
    A = oracle_mod.f32_to_bf16(X.astype(np.float32))
    y = np.ones(m, np.float32)
    idx = synth.iid_indices(m, s * b, seed=3)
    res = oracle_mod.outer_step_gram(A, y, idx, np.zeros(n), s, b, 0.1, 0)
    G = res.G
    norms = np.linalg.norm(oracle_mod.bf16_to_f64(A[idx]), axis=1)
    assert np.array_equal(G, G.T)
    assert np.allclose(np.diag(G), norms ** 2, rtol=1e-14)
    assert (np.abs(G) <= np.outer(norms, norms) * (1 + 1e-14)).all()
    ev = np.linalg.eigvalsh(G)
    assert ev.min() >= -1e-12 * np.trace(G)
    assert np.linalg.matrix_rank(G, tol=1e-9) <= n
    assert norms.max() <= 1.0 and np.linalg.norm(G) <= s * b
    ent, nr = oracle_mod.gram_entries(A, idx, [(3, 1), (17, 17), (0, 31), (31, 0)])
    assert np.allclose(ent, [G[3, 1], G[17, 17], G[0, 31], G[31, 0]], rtol=1e-15)
    assert np.allclose(nr, norms, rtol=1e-15)


def test_gather_is_exact(oracle_mod):
    """Alg. 1 line 2: identity indices, a constant index, a permutation; padded row stride."""
    m, n = 33, 7
    rng = np.random.default_rng(700)
    store = rng.integers(0, 1 << 16, (m, n + 5), dtype=np.uint64).astype(np.uint16)
    store[(store & 0x7F80) == 0x7F80] = 0x3F80                   # keep values finite
    A = store[:, :n]                                               # row stride n + 5
    y = rng.standard_normal(m).astype(np.float32)
    x = np.zeros(n)
    ident = np.arange(12, dtype=np.int32)
    assert np.array_equal(oracle_mod.outer_step_gram(A, y, ident, x, 3, 4, 0.1, 1).Y_bits, A[:12])
    const = np.full(12, 20, np.int32)
    Yc = oracle_mod.outer_step_gram(A, y, const, x, 3, 4, 0.1, 1).Y_bits
    assert (Yc == A[20]).all()
    perm = np.random.default_rng(1).permutation(m).astype(np.int32)[:32]
    Yp = oracle_mod.outer_step_gram(A, y, perm, x, 4, 8, 0.1, 1).Y_bits
    assert sorted(map(bytes, Yp)) == sorted(bytes(A[i]) for i in perm)
    # labels ride along: r = 0 at x = 0, so the linear loss gives u = -y_I exactly
    assert np.array_equal(oracle_mod.outer_step_gram(A, y, perm, x, 1, 32, 0.1, 1).u, -y[perm].astype(np.float64))
    for bad in (-1, m):
        with pytest.raises(IndexError):
            oracle_mod.outer_step_gram(A, y, np.array([0, bad, 1, 2], np.int32), x, 2, 2, 0.1, 1)
        with pytest.raises(IndexError):
            oracle_mod.outer_step_seq(A, y, np.array([0, bad, 1, 2], np.int32), x, 2, 2, 0.1, 1)


@pytest.mark.parametrize("loss", LOSSES)
def test_shadow_enters_the_margin_only(oracle_mod, loss):
    """r uses BF16(x), the update lands on the un-rounded master x (Table 1)."""
    A, y, rng = _problem(oracle_mod, loss, 80, 9, 800 + loss)
    s, b, eta = 3, 4, 0.2
    idx = synth.iid_indices(80, s * b, seed=2)
    x = rng.standard_normal(9)
    res = oracle_mod.outer_step_gram(A, y, idx, x, s, b, eta, loss, shadow=True)
    Y = oracle_mod.bf16_to_f64(A[idx])
    x_hat = oracle_mod.bf16_to_f64(oracle_mod.f64_to_bf16(x))
    assert np.abs(x_hat - x).max() > 1e-4                         # the rounding is visible
    assert np.allclose(res.r, Y @ x_hat, rtol=1e-14, atol=1e-16)
    assert np.allclose(res.x_out - x, -(eta / b) * res.g, rtol=1e-12, atol=1e-16)
    assert np.allclose(res.g, Y.T @ res.u, rtol=1e-13, atol=1e-16)
    off = oracle_mod.outer_step_gram(A, y, idx, x, s, b, eta, loss, shadow=False)
    assert np.allclose(off.r, Y @ x, rtol=1e-14, atol=1e-16)


def test_step_scale_is_eta_over_b_not_eta_over_sb(oracle_mod):
    """alpha = eta/b: with s blocks of identical rows and the linear loss at
    x = 0, eta/(sb) would give a different, smaller step."""
    n, b, s = 4, 2, 3
    A = oracle_mod.f32_to_bf16(np.tile(np.array([[0.5, -0.25, 0.125, 1.0]], np.float32), (8, 1)))
    y = np.full(8, 2.0, np.float32)
    idx = np.zeros(s * b, np.int32)
    eta = 0.1
    res = oracle_mod.outer_step_gram(A, y, idx, np.zeros(n), s, b, eta, 1, shadow=False)
    a = np.array([0.5, -0.25, 0.125, 1.0])
    # one row repeated: each mini-batch step is x <- x - eta * a (a.x - 2)
    v = np.zeros(n)
    for _ in range(s):
        v = v - eta * a * (a @ v - 2.0)
    assert np.allclose(res.x_out, v, rtol=1e-14)
