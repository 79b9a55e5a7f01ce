"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json:configs).

This module is the one thing the CUDA path's callers and the CPU oracle's
callers share. It holds none of the method's arithmetic (no margin, Gram,
recurrence, loss or update), imports neither ``oracle`` nor the CUDA binding,
and only draws data: a BF16 feature matrix, FP32 labels from a planted model,
and per-epoch row permutations. The real epsilon / SUSY LIBSVM files the paper
uses (Table 4) are not available; these stand in for them
(DESIGN.md "Input recipe").

"N(0, v)" is variance v throughout. X is rounded to BF16 (round-to-nearest-even,
torch's cast) once; those bits are the dataset for every consumer.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Tuple

import numpy as np
import torch

LOGISTIC, LINEAR, POISSON = 0, 1, 2


@dataclass(frozen=True)
class Config:
    name: str
    m: int
    n: int
    loss: int
    b: int
    s_list: Tuple[int, ...]
    eta: float
    epochs: int
    kind: str                      # which generator below


# BASELINE.json:configs, in order.
CONFIGS: Tuple[Config, ...] = (
    Config("tiny-logistic", 8192, 64, LOGISTIC, 16, (4,), 0.5, 5, "gauss_logistic"),
    Config("susy-shaped", 5_000_000, 18, LOGISTIC, 64, (1, 4, 16, 32), 0.1, 3, "susy"),
    Config("synth-linear", 1_000_000, 4096, LINEAR, 128, (1, 8, 32), 0.05, 2, "gauss_linear"),
    Config("epsilon-shaped", 400_000, 2000, LOGISTIC, 32, (1, 8, 16, 64), 1.0, 2, "epsilon"),
    Config("poisson-synth", 2_000_000, 512, POISSON, 64, (1, 8, 32), 0.01, 2, "poisson"),
)


def config(i: int, m: int | None = None, n: int | None = None) -> Config:
    """Config i of BASELINE.json (0-based), optionally down-sized in m / n for CPU-side tests."""
    c = CONFIGS[i]
    if m is None and n is None:
        return c
    return Config(c.name, m or c.m, n or c.n, c.loss, c.b, c.s_list, c.eta, c.epochs, c.kind)


@dataclass
class Dataset:
    cfg: Config
    X_bf16: torch.Tensor           # [m, n] torch.bfloat16, on `device`
    y: torch.Tensor                # [m] float32
    w_star: torch.Tensor           # [n] float32 (the planted model; not used by the method)
    seed: int = 42
    extra: dict = field(default_factory=dict)

    def X_bits_numpy(self) -> np.ndarray:
        """The BF16 bit patterns as a host uint16 array [m, n]."""
        return self.X_bf16.view(torch.int16).cpu().numpy().view(np.uint16)

    def y_numpy(self) -> np.ndarray:
        return self.y.cpu().numpy()


def _gen(device, seed: int) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    return g


def _rows_chunk(m: int, n: int) -> int:
    return max(1, min(m, (1 << 27) // max(n, 1)))       # <= 128 Mi elements per chunk


def _planted_scores(X_bf16: torch.Tensor, w: torch.Tensor) -> torch.Tensor:
    """X_bf16 @ w in FP32, chunked over rows (label generation only)."""
    m, n = X_bf16.shape
    out = torch.empty(m, dtype=torch.float32, device=X_bf16.device)
    step = _rows_chunk(m, n)
    for lo in range(0, m, step):
        out[lo:lo + step] = X_bf16[lo:lo + step].float() @ w
    return out


def make_dataset(cfg: Config, seed: int = 42, device: str | torch.device = "cpu") -> Dataset:
    """Draw the dataset of `cfg` from `seed` on `device` (CPU and CUDA streams differ; a run uses one)."""
    device = torch.device(device)
    g = _gen(device, seed)
    m, n = cfg.m, cfg.n
    X = torch.empty((m, n), dtype=torch.bfloat16, device=device)
    step = _rows_chunk(m, n)
    kind = cfg.kind

    if kind in ("gauss_logistic", "gauss_linear", "poisson"):
        sd = 1.0 / math.sqrt(n)
        for lo in range(0, m, step):
            rows = min(step, m - lo)
            X[lo:lo + rows] = (torch.randn((rows, n), generator=g, device=device) * sd).to(torch.bfloat16)
    elif kind == "epsilon":
        for lo in range(0, m, step):
            rows = min(step, m - lo)
            blk = torch.randn((rows, n), generator=g, device=device)
            blk = blk / blk.norm(dim=1, keepdim=True)
            X[lo:lo + rows] = blk.to(torch.bfloat16)
    elif kind == "susy":
        half = n // 2
        raw = torch.randn((m, n), generator=g, device=device)
        raw[:, half:] = torch.exp(raw[:, half:])
        mean = raw.mean(dim=0, keepdim=True)
        std = raw.std(dim=0, unbiased=False, keepdim=True)
        X[:] = ((raw - mean) / std).to(torch.bfloat16)
        del raw
    else:
        raise ValueError(kind)

    if kind == "poisson":
        w = torch.randn(n, generator=g, device=device) * 0.5        # N(0, 0.25)
    else:
        w = torch.randn(n, generator=g, device=device)
    score = _planted_scores(X, w)

    if kind == "gauss_logistic":
        score = score + torch.randn(m, generator=g, device=device) * math.sqrt(0.1)
        y = torch.where(score >= 0, 1.0, -1.0)
    elif kind == "gauss_linear":
        y = score + torch.randn(m, generator=g, device=device) * 0.1   # N(0, 0.01)
    elif kind == "epsilon":
        y = torch.where(score >= 0, 1.0, -1.0)
        flip = torch.rand(m, generator=g, device=device) < 0.10
        y = torch.where(flip, -y, y)
    elif kind == "susy":
        score = score + torch.randn(m, generator=g, device=device)
        kth = max(1, min(m, int(round(0.54 * m))))
        thresh = torch.kthvalue(score.double().cpu(), kth).values.item()   # 54th percentile: ~46% positive
        y = torch.where(score > thresh, 1.0, -1.0)
    elif kind == "poisson":
        y = torch.poisson(torch.exp(score), generator=g)
    return Dataset(cfg, X, y.to(torch.float32).contiguous(), w.to(torch.float32), seed)


def minibatches_per_epoch(m: int, b: int, s_list) -> int:
    """Epoch rule (reading 16): floor(m / (b*s_max)) * s_max mini-batches, the tail dropped,
    so every s of a sweep consumes the same mini-batch sequence."""
    s_max = max(s_list)
    return (m // (b * s_max)) * s_max


def epoch_indices(cfg: Config, seed: int, epoch: int) -> np.ndarray:
    """Row indices of one epoch: a seeded permutation of range(m) (BASELINE.json:configs[0]: "sampled
    without replacement per epoch from seed"), truncated to whole mini-batches. int32 [N_mb * b]."""
    perm = np.random.default_rng([seed, epoch]).permutation(cfg.m).astype(np.int32)
    return np.ascontiguousarray(perm[: minibatches_per_epoch(cfg.m, cfg.b, cfg.s_list) * cfg.b])


def training_indices(cfg: Config, seed: int = 42, epochs: int | None = None) -> np.ndarray:
    """All epochs' indices concatenated."""
    e = cfg.epochs if epochs is None else epochs
    return np.concatenate([epoch_indices(cfg, seed, k) for k in range(e)])


def iid_indices(m: int, count: int, seed: int) -> np.ndarray:
    """i.i.d. uniform WITH replacement (Alg. 1 line 1): duplicates are expected."""
    return np.random.default_rng(seed).integers(0, m, size=count, dtype=np.int64).astype(np.int32)


def checksum(a: np.ndarray) -> int:
    """64-bit FNV-style checksum of an array's bytes, logged so runs are comparable."""
    v = np.frombuffer(np.ascontiguousarray(a).tobytes(), dtype=np.uint8)
    pad = (-len(v)) % 8
    if pad:
        v = np.concatenate([v, np.zeros(pad, np.uint8)])
    w = v.view(np.uint64)
    mult = np.uint64(0x100000001B3)
    with np.errstate(over="ignore"):
        idx = np.arange(1, len(w) + 1, dtype=np.uint64)
        return int(np.bitwise_xor.reduce(w * (idx * mult + np.uint64(0xCBF29CE484222325))))
