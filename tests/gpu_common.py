"""Shared helpers of the `-m gpu` parity tests: seeded inputs on the device, oracle inputs on the host.

The CUDA path is reached only through the C ABI (paper_2606_18463_b200.binding -> libcasgd.so); the
expected values come only from `oracle/` on the same BF16 bits, labels, indices and FP32 x bits.
Tolerances are BASELINE.json:north_star's, written out here once:

  Y, y_I, idx            bit-exact
  |dG_ij|                <= 1e-5 * ||y_i|| * ||y_j||
  |dr_i|                 <= 1e-5 * ||y_i|| * ||x_hat||
  ||dx||_2 / ||x||_2     <= 1e-5 after one outer step
  final training loss    within 0.5 % of the trajectory oracle's
and DESIGN.md's additional ones (z and u within the bound the recurrence implies, `chain_bounds`;
casgd_loss within 1e-6 relative).
"""
from __future__ import annotations

import numpy as np
import torch

from paper_2606_18463_b200 import synth

TOL_G = 1e-5
TOL_R = 1e-5
TOL_X = 1e-5
TOL_U = 2e-6          # evaluating l' in FP32 (fast exp / divide on the chain: ~2^-21 relative), relative to max(1, |u|)
TOL_LOSS_CALL = 1e-6
TOL_FINAL_LOSS = 5e-3


def require_cuda():
    assert torch.cuda.is_available(), "GPU tests selected on a box without a CUDA device"


def device_dataset(cfg, seed=42):
    """Draw the dataset on the CPU generator (same bits on every box) and upload it."""
    ds = synth.make_dataset(cfg, seed=seed, device="cpu")
    A_bits = ds.X_bits_numpy()
    y = ds.y_numpy()
    return ds.X_bf16.cuda(), ds.y.cuda(), A_bits, y


def random_x(n, seed, scale=1.0):
    """An FP32 iterate with entries of mixed magnitude (so that its BF16 rounding matters)."""
    rng = np.random.default_rng(seed)
    return (rng.standard_normal(n) * scale).astype(np.float32)


def block_lower_mask(s, b):
    """mask[i, k] = block(k) < block(i): the entries of G the recurrence reads."""
    blk = np.arange(s * b) // b
    return blk[None, :] < blk[:, None]


def chain_bounds(ref, y_idx, z_gpu, s, b, eta, loss, bound_r, bound_g, tol_scale=1.0):
    """Forward propagation of the admitted input errors through Alg. 1 lines 6-15 (the recurrence is a unit
    block-lower-triangular system): returns (bound_z, bound_u), element-wise."""
    sb = s * b
    alpha = eta / b
    absG, absu = np.abs(ref.G), np.abs(ref.u)
    if loss == 0:
        lip = np.full(sb, 0.25) * np.abs(y_idx.astype(np.float64)) ** 2     # |d/dz (-y / (1 + e^{yz}))| <= y^2 / 4
    elif loss == 1:
        lip = np.ones(sb)
    else:                                            # Poisson: d/dz e^z = e^z, taken at the larger of the two margins
        lip = np.exp(np.maximum(z_gpu, ref.z))
    eps_u = TOL_U * tol_scale * np.maximum(1.0, absu)
    bz, bu = np.zeros(sb), np.zeros(sb)
    for j in range(s):
        rows = slice(j * b, (j + 1) * b)
        L = j * b
        corr = alpha * (bound_g[rows, :L] @ absu[:L] + absG[rows, :L] @ bu[:L])
        fp32 = (L / 32 + 8) * 2.0 ** -24 * (np.abs(ref.r[rows]) + alpha * (absG[rows, :L] @ absu[:L]))
        bz[rows] = bound_r[rows] + corr + fp32
        if loss == 2:
            lip[rows] = lip[rows] * np.exp(bz[rows])
        bu[rows] = lip[rows] * bz[rows] + eps_u[rows]
    return bz, bu


def check_step_against_oracle(oracle, cg, A_bits, y, idx, x0, s, b, eta, loss, binding, full_lower=False,
                              check_g=True, tol_scale=1.0, shadow=True):
    """Run one casgd_outer_step from the FP32 bits x0 and compare every exported intermediate with O1."""
    idx_d = torch.from_numpy(idx).cuda()
    x_d = torch.from_numpy(x0.copy()).cuda()
    cg.invalidate_shadow()
    cg.outer_step(idx_d, x_d, s, b, eta)
    cg.sync()
    ref = oracle.outer_step_gram(A_bits, y, idx, x0.astype(np.float64), s, b, eta, loss, shadow=shadow)
    return compare_last_step(oracle, cg, ref, y[idx], x0, x_d, s, b, eta, loss, binding, full_lower, check_g, tol_scale,
                             shadow=shadow)


def compare_last_step(oracle, cg, ref, y_idx, x0, x_d, s, b, eta, loss, binding, full_lower=False, check_g=True,
                      tol_scale=1.0, shadow=True):
    """Compare the intermediates of the LAST outer step the context ran (casgd_debug_export) and the iterate
    `x_d` it left with `ref`, oracle O1's result for the same rows, labels `y_idx`, indices and FP32 x0 bits."""
    sb = s * b
    # gather: bit-exact rows and labels (Alg. 1 line 2)
    Y = cg.debug(binding.DBG_Y)
    assert Y.dtype == np.uint16 and np.array_equal(Y, ref.Y_bits), "gathered rows differ bitwise"
    assert np.array_equal(cg.debug(binding.DBG_YLAB), y_idx), "gathered labels differ bitwise"

    Yf = oracle.bf16_to_f64(ref.Y_bits)
    norms = np.sqrt((Yf * Yf).sum(axis=1))
    xhat = oracle.bf16_to_f64(oracle.f32_to_bf16(x0)) if shadow else x0.astype(np.float64)   # (False: CASGD_OPT_MARGIN_SPLIT)
    xnorm = np.sqrt((xhat * xhat).sum())

    # margin (line 3)
    r = cg.debug(binding.DBG_R).astype(np.float64)
    bound_r = TOL_R * tol_scale * norms * xnorm + 1e-30
    assert np.all(np.abs(r - ref.r) <= bound_r), f"margin: max ratio {np.max(np.abs(r - ref.r) / bound_r):.3g}"

    # Gram (line 4): the entries include/casgd.h declares valid
    mask = np.tril(np.ones((sb, sb), bool)) if full_lower else block_lower_mask(s, b)
    bound_g = TOL_G * tol_scale * np.outer(norms, norms) + 1e-30
    if check_g and mask.any():
        G = cg.debug(binding.DBG_G).astype(np.float64)
        ratio = np.abs(G - ref.G) / bound_g
        assert np.all(ratio[mask] <= 1.0), f"Gram: max ratio {ratio[mask].max():.3g}"

    # recurrence (lines 6-15), FP32: the bound the recurrence itself implies, propagated forward
    # block by block from the oracle's own G and u:
    #   |dz_j| <= |dr_j| + alpha * sum_{k<j} (|dG_jk| |u_k| + |G_jk| |du_k|) + fp32(j),   |du_k| <= Lip_k |dz_k| + eps_u
    # with |dr|, |dG| the admitted margin / Gram errors, fp32(j) the worst-case rounding of an FP32 sum of j*b terms
    # split over >= 32 lanes (depth j*b/32 + 8), and eps_u = TOL_U * max(1, |u|) the admitted error of evaluating l'.
    z = cg.debug(binding.DBG_Z).astype(np.float64)
    u = cg.debug(binding.DBG_U).astype(np.float64)
    bound_z, bound_u = chain_bounds(ref, y_idx, z, s, b, eta, loss, bound_r, bound_g, tol_scale)
    assert np.all(np.abs(z - ref.z) <= bound_z), f"z: max ratio {np.max(np.abs(z - ref.z) / bound_z):.3g}"
    assert np.all(np.abs(u - ref.u) <= bound_u), f"u: max ratio {np.max(np.abs(u - ref.u) / bound_u):.3g}"

    # update (lines 16-17): relative 2-norm of x after one outer step
    x1 = x_d.cpu().numpy().astype(np.float64)
    denom = max(np.linalg.norm(ref.x_out), 1e-300)
    rel = np.linalg.norm(x1 - ref.x_out) / denom
    assert rel <= TOL_X * tol_scale, f"x after one outer step: relative error {rel:.3g}"

    # shadow: bf16_rne of the library's own new master, bit for bit
    xbf = cg.debug(binding.DBG_XBF)
    assert np.array_equal(xbf, oracle.f32_to_bf16(x_d.cpu().numpy())), "BF16 shadow is not bf16_rne(x)"
    # no kernel wrote past a workspace (1 KB guard bands around Y, y_I, G, r, z, u)
    assert int(cg.debug(binding.DBG_GUARDS)[0]) == 0, "guard bytes around the workspaces were overwritten"
    return ref, dict(r=r, z=z, u=u, x=x1)
