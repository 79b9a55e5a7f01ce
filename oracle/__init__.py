"""FP64 CPU oracle for one CA-SGD outer iteration -- TEST INFRASTRUCTURE.

ctypes front end of ``casgd_oracle.c`` (read that file's header first). Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package; the product
(``paper_2606_18463_b200``) never does, and this package never imports the
product. Arrays are numpy; nothing here touches CUDA.

Citations are to /root/reference/PAPER.md (arxiv/paper_2606_18463).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import NamedTuple, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "casgd_oracle.c")
_LIB = os.path.join(_HERE, "libcasgd_oracle.so")

LOGISTIC, LINEAR, POISSON = 0, 1, 2
LOSSES = {"logistic": LOGISTIC, "linear": LINEAR, "poisson": POISSON}


def build(force: bool = False) -> str:
    """Compile casgd_oracle.c with gcc (-O2, OpenMP); returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-std=c11", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        c_u16p = ctypes.POINTER(ctypes.c_uint16)
        c_f32p = ctypes.POINTER(ctypes.c_float)
        c_f64p = ctypes.POINTER(ctypes.c_double)
        c_i32p = ctypes.POINTER(ctypes.c_int32)
        c_i64p = ctypes.POINTER(ctypes.c_int64)
        i64, i32, f64 = ctypes.c_int64, ctypes.c_int32, ctypes.c_double
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_bf16_to_f64.restype = f64
        lib.oracle_bf16_to_f64.argtypes = [ctypes.c_uint16]
        lib.oracle_f32_to_bf16.restype = ctypes.c_uint16
        lib.oracle_f32_to_bf16.argtypes = [ctypes.c_float]
        lib.oracle_f64_to_bf16.restype = ctypes.c_uint16
        lib.oracle_f64_to_bf16.argtypes = [f64]
        lib.oracle_loss_value.restype = f64
        lib.oracle_loss_value.argtypes = [f64, f64, ctypes.c_int]
        lib.oracle_lprime.restype = f64
        lib.oracle_lprime.argtypes = [f64, f64, ctypes.c_int]
        lib.oracle_full_loss.restype = f64
        lib.oracle_full_loss.argtypes = [c_u16p, i64, c_f32p, i64, i32, c_f64p, ctypes.c_int]
        lib.oracle_outer_step_gram.restype = ctypes.c_int
        lib.oracle_outer_step_gram.argtypes = [
            c_u16p, i64, c_f32p, i64, i32, c_i32p, i32, i32, f64, ctypes.c_int, ctypes.c_int,
            c_f64p, c_u16p, c_f64p, c_f64p, c_f64p, c_f64p, c_f64p, c_f64p]
        lib.oracle_gram_entries.restype = ctypes.c_int
        lib.oracle_gram_entries.argtypes = [c_u16p, i64, i64, i32, c_i32p, i64, c_i64p, i64, c_f64p, c_f64p]
        lib.oracle_train_seq.restype = ctypes.c_int
        lib.oracle_train_seq.argtypes = [
            c_u16p, i64, c_f32p, i64, i32, c_i32p, i64, i32, i32, f64, ctypes.c_int, ctypes.c_int,
            c_f64p, c_f64p, c_f64p]
        lib.oracle_train_gram.restype = ctypes.c_int
        lib.oracle_train_gram.argtypes = [
            c_u16p, i64, c_f32p, i64, i32, c_i32p, i64, i32, i32, f64, ctypes.c_int, ctypes.c_int, c_f64p]
        _lib = lib
    return _lib


def _p(a: Optional[np.ndarray], ctype):
    return None if a is None else a.ctypes.data_as(ctypes.POINTER(ctype))


def _check_data(A_bits, y, idx):
    assert A_bits.dtype == np.uint16 and A_bits.ndim == 2 and A_bits.strides[1] == 2, "A: uint16 [m, n] BF16 bits"
    assert A_bits.strides[0] % 2 == 0
    assert y.dtype == np.float32 and y.ndim == 1 and y.flags.c_contiguous and y.shape[0] == A_bits.shape[0]
    assert idx.dtype == np.int32 and idx.ndim == 1 and idx.flags.c_contiguous


def _rc(rc: int):
    if rc == 1:
        raise IndexError("oracle: row index outside [0, m)")
    if rc:
        raise ValueError(f"oracle: bad arguments or out of memory (rc={rc})")


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def bf16_to_f64(bits) -> np.ndarray:
    """Exact widening of BF16 bit patterns (uint16) to float64."""
    bits = np.asarray(bits, dtype=np.uint16)
    with np.errstate(invalid="ignore"):          # signalling-NaN patterns widen quietly
        return (bits.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


def f32_to_bf16(x) -> np.ndarray:
    """Round-to-nearest-even binary32 -> BF16 bits, elementwise through the C helper."""
    lib = _load()
    x = np.asarray(x, dtype=np.float32)
    return np.fromiter((lib.oracle_f32_to_bf16(float(v)) for v in x.ravel()), dtype=np.uint16,
                       count=x.size).reshape(x.shape)


def f64_to_bf16(x) -> np.ndarray:
    lib = _load()
    x = np.asarray(x, dtype=np.float64)
    return np.fromiter((lib.oracle_f64_to_bf16(float(v)) for v in x.ravel()), dtype=np.uint16,
                       count=x.size).reshape(x.shape)


def loss_value(r: float, y: float, loss: int) -> float:
    """L(r, y)."""
    return float(_load().oracle_loss_value(float(r), float(y), int(loss)))


def lprime(z: float, y: float, loss: int) -> float:
    """u = dL/dr = -delta, delta as printed at PAPER.md:L59."""
    return float(_load().oracle_lprime(float(z), float(y), int(loss)))


def full_loss(A_bits: np.ndarray, y: np.ndarray, x: np.ndarray, loss: int) -> float:
    """F(x) = mean_i L(a_i^T x, y_i); x float64."""
    _check_data(A_bits, y, np.zeros(0, np.int32))
    x = np.ascontiguousarray(x, dtype=np.float64)
    m, n = A_bits.shape
    assert x.shape == (n,)
    return float(_load().oracle_full_loss(_p(A_bits, ctypes.c_uint16), A_bits.strides[0] // 2,
                                          _p(y, ctypes.c_float), m, n, _p(x, ctypes.c_double), int(loss)))


class GramStep(NamedTuple):
    Y_bits: np.ndarray   # [sb, n] uint16, the gathered rows, bit for bit
    G: np.ndarray        # [sb, sb] float64, Y Y^T
    r: np.ndarray        # [sb]   Y x_hat
    z: np.ndarray        # [sb]   corrected margins
    u: np.ndarray        # [sb]   l'(z, y_I)
    g: np.ndarray        # [n]    Y^T u
    x_out: np.ndarray    # [n]    x - (eta/b) g


def outer_step_gram(A_bits, y, idx, x, s, b, eta, loss, shadow=True) -> GramStep:
    """O1: one outer iteration in the Gram form, Algorithm 1 at P = 1."""
    _check_data(A_bits, y, idx)
    m, n = A_bits.shape
    sb = s * b
    assert idx.shape[0] == sb
    x = np.ascontiguousarray(x, dtype=np.float64)
    assert x.shape == (n,)
    Yb = np.empty((sb, n), np.uint16)
    G = np.empty((sb, sb), np.float64)
    r, z, u = (np.empty(sb, np.float64) for _ in range(3))
    g, x_out = np.empty(n, np.float64), np.empty(n, np.float64)
    d = ctypes.c_double
    _rc(_load().oracle_outer_step_gram(
        _p(A_bits, ctypes.c_uint16), A_bits.strides[0] // 2, _p(y, ctypes.c_float), m, n,
        _p(idx, ctypes.c_int32), s, b, float(eta), int(loss), int(bool(shadow)), _p(x, d),
        _p(Yb, ctypes.c_uint16), _p(G, d), _p(r, d), _p(z, d), _p(u, d), _p(g, d), _p(x_out, d)))
    return GramStep(Yb, G, r, z, u, g, x_out)


def slab_payload(A_bits, idx, x, s, b, cols, shadow=True):
    """One rank's contribution to Alg. 1 line 5 in the 1-D block-column partition (L33, L141): with the
    rank holding columns `cols` of A and x, r_loc = Y_loc x_hat_loc and G_loc = Y_loc Y_loc^T (FP64, plain numpy)."""
    Y = bf16_to_f64(A_bits[idx][:, cols])
    xl = np.asarray(x, np.float64)[cols]
    xh = bf16_to_f64(f32_to_bf16(xl.astype(np.float32))) if shadow else xl
    return Y @ xh, Y @ Y.T


def outer_step_gram_partitioned(A_bits, y, idx, x, s, b, eta, loss, slabs, shadow=True) -> GramStep:
    """O1 on P ranks: Algorithm 1 WITH its line 5 (section 4.2). `slabs` is a list of column
    slices, one per rank. Each rank forms r_loc, G_loc on its slab; the AllReduce sums them (in rank order here);
    every rank runs the same recurrence (lines 6-15); rank p updates its slab of x with its own Y_loc^T u (lines 16-17).
    Plain numpy FP64, no blocking beyond the partition the paper states."""
    _check_data(A_bits, y, idx)
    m, n = A_bits.shape
    sb = s * b
    x = np.asarray(x, np.float64)
    alpha = eta / b
    r, G = np.zeros(sb), np.zeros((sb, sb))
    for cols in slabs:                                   # line 5: the sum over ranks of [r; G]
        rl, Gl = slab_payload(A_bits, idx, x, s, b, cols, shadow)
        r += rl
        G += Gl
    yI = y[idx].astype(np.float64)
    z, u = np.zeros(sb), np.zeros(sb)
    for j in range(s):                                   # lines 6-15, redundantly on every rank
        rows = slice(j * b, (j + 1) * b)
        z[rows] = r[rows] - alpha * (G[rows, : j * b] @ u[: j * b])
        u[rows] = [lprime(zz, yy, loss) for zz, yy in zip(z[rows], yI[rows])]
    g, x_out = np.zeros(n), x.copy()
    for cols in slabs:                                   # lines 16-17, each rank on its slab
        Y = bf16_to_f64(A_bits[idx][:, cols])
        g[cols] = Y.T @ u
        x_out[cols] = x[cols] - alpha * g[cols]
    return GramStep(A_bits[idx].copy(), G, r, z, u, g, x_out)


class SeqStep(NamedTuple):
    z: np.ndarray
    u: np.ndarray
    x_out: np.ndarray


def outer_step_seq(A_bits, y, idx, x, s, b, eta, loss, shadow=True) -> SeqStep:
    """O2: the same outer iteration as s sequential mini-batch SGD steps."""
    _check_data(A_bits, y, idx)
    m, n = A_bits.shape
    sb = s * b
    assert idx.shape[0] == sb
    x_out = np.array(x, dtype=np.float64, copy=True)
    z, u = np.empty(sb, np.float64), np.empty(sb, np.float64)
    d = ctypes.c_double
    _rc(_load().oracle_train_seq(
        _p(A_bits, ctypes.c_uint16), A_bits.strides[0] // 2, _p(y, ctypes.c_float), m, n,
        _p(idx, ctypes.c_int32), 1, s, b, float(eta), int(loss), int(bool(shadow)), _p(x_out, d), _p(z, d), _p(u, d)))
    return SeqStep(z, u, x_out)


def train(A_bits, y, idx, x0, s, b, eta, loss, shadow=True, form="seq") -> np.ndarray:
    """Trajectory oracle: len(idx)/(s*b) consecutive outer iterations from x0 (float64 master).

    form="seq" uses O2 (cheap), form="gram" uses O1 (what the GPU computes)."""
    _check_data(A_bits, y, idx)
    m, n = A_bits.shape
    sb = s * b
    assert idx.shape[0] % sb == 0
    n_outer = idx.shape[0] // sb
    x = np.array(x0, dtype=np.float64, copy=True)
    d = ctypes.c_double
    lib = _load()
    if form == "seq":
        _rc(lib.oracle_train_seq(_p(A_bits, ctypes.c_uint16), A_bits.strides[0] // 2, _p(y, ctypes.c_float), m, n,
                                 _p(idx, ctypes.c_int32), n_outer, s, b, float(eta), int(loss),
                                 int(bool(shadow)), _p(x, d), None, None))
    elif form == "gram":
        _rc(lib.oracle_train_gram(_p(A_bits, ctypes.c_uint16), A_bits.strides[0] // 2, _p(y, ctypes.c_float), m, n,
                                  _p(idx, ctypes.c_int32), n_outer, s, b, float(eta), int(loss),
                                  int(bool(shadow)), _p(x, d)))
    else:
        raise ValueError(form)
    return x


def gram_entries(A_bits, idx, pairs):
    """G[i, j] for selected (i, j) positions of the sampled block, and all row norms ||Y_t||."""
    m, n = A_bits.shape
    pairs = np.ascontiguousarray(pairs, dtype=np.int64).reshape(-1, 2)
    out = np.empty(pairs.shape[0], np.float64)
    norms = np.empty(idx.shape[0], np.float64)
    _rc(_load().oracle_gram_entries(_p(A_bits, ctypes.c_uint16), A_bits.strides[0] // 2, m, n,
                                    _p(idx, ctypes.c_int32), idx.shape[0], _p(pairs, ctypes.c_int64),
                                    pairs.shape[0], _p(out, ctypes.c_double), _p(norms, ctypes.c_double)))
    return out, norms


# ---------------------------------------------------------------- index sampling (Alg. 1 line 1) ---
# The paper samples the s*b row indices of an outer step i.i.d. uniformly WITH replacement (PAPER.md:L111-L112,
# L59). For the on-device sampler (include/casgd.h: casgd_outer_steps_sampled) both sides implement the same
# counter-based generator, Philox4x32-10 (Salmon, Moraes, Dror, Shaw: "Parallel random numbers: as easy as 1, 2, 3",
# SC'11), written here from the paper's definition in plain numpy integer arithmetic:
#   index t of outer step h:  counter = (t // 4, h mod 2^32, h div 2^32, 0xCA5D), key = (seed mod 2^32, seed div 2^32),
#   w = Philox4x32-10(counter, key)[t mod 4],  idx = floor(w * m / 2^32)     (multiply-shift: bias < m / 2^32)
_PHILOX_M0, _PHILOX_M1 = np.uint64(0xD2511F53), np.uint64(0xCD9E8D57)
_PHILOX_W0, _PHILOX_W1 = 0x9E3779B9, 0xBB67AE85
_MASK32 = np.uint64(0xFFFFFFFF)
SAMPLING_DOMAIN = 0xCA5D


def philox4x32_10(counter, key):
    """Philox4x32 with 10 rounds. counter: [..., 4] and key: [..., 2] arrays of values < 2^32; returns uint32 [..., 4]."""
    c = np.asarray(counter, dtype=np.uint64) & _MASK32
    k = np.asarray(key, dtype=np.uint64) & _MASK32
    c0, c1, c2, c3 = (c[..., i].copy() for i in range(4))
    k0, k1 = k[..., 0].copy(), k[..., 1].copy()
    for _ in range(10):
        p0 = _PHILOX_M0 * c0                      # 32 x 32 -> 64 bit products
        p1 = _PHILOX_M1 * c2
        hi0, lo0 = p0 >> np.uint64(32), p0 & _MASK32
        hi1, lo1 = p1 >> np.uint64(32), p1 & _MASK32
        c0, c1, c2, c3 = hi1 ^ c1 ^ k0, lo1, hi0 ^ c3 ^ k1, lo0
        k0 = (k0 + np.uint64(_PHILOX_W0)) & _MASK32
        k1 = (k1 + np.uint64(_PHILOX_W1)) & _MASK32
    return np.stack([c0, c1, c2, c3], axis=-1).astype(np.uint32)


def sample_indices(seed: int, step: int, sb: int, m: int) -> np.ndarray:
    """The s*b row indices of outer step `step` under `seed`: i.i.d. uniform on [0, m), with replacement. int32 [sb]."""
    t = np.arange(sb, dtype=np.uint64)
    nblk = (sb + 3) // 4
    ctr = np.zeros((nblk, 4), dtype=np.uint64)
    ctr[:, 0] = np.arange(nblk, dtype=np.uint64)
    ctr[:, 1] = step & 0xFFFFFFFF
    ctr[:, 2] = (step >> 32) & 0xFFFFFFFF
    ctr[:, 3] = SAMPLING_DOMAIN
    key = np.array([seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF], dtype=np.uint64)
    w = philox4x32_10(ctr, np.broadcast_to(key, (nblk, 2))).reshape(-1)[:sb].astype(np.uint64)
    return ((w * np.uint64(m)) >> np.uint64(32)).astype(np.int32)
