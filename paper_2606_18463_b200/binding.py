"""Thin ctypes binding of libcasgd.so (C ABI: include/casgd.h). Argument marshalling only.

PyTorch is used for device memory and streams; every step of the path runs in the library's
CUDA kernels. There is no CPU path: if the library is missing or cannot be loaded, `load()`
raises, and so does everything that needs it.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcasgd.so")

LOGISTIC, LINEAR, POISSON = 0, 1, 2
OK, EINVAL, ENOMEM, ECUDA, EARCH, EINDEX = range(6)
STATUS_NAMES = ("CASGD_OK", "CASGD_EINVAL", "CASGD_ENOMEM", "CASGD_ECUDA", "CASGD_EARCH", "CASGD_EINDEX")
DBG_Y, DBG_YLAB, DBG_G, DBG_R, DBG_Z, DBG_U, DBG_XBF, DBG_STAMPS, DBG_GUARDS, DBG_XSNAP = range(10)
OPT_GRAM_IMPL, OPT_GRAM_FULL_LOWER, OPT_PROFILE, OPT_NO_GRAPH, OPT_GRAM_KSPLIT, OPT_RECURRENCE_IMPL, OPT_LOSS_IMPL, OPT_NO_FUSED_UPDATE, OPT_STAMPS, OPT_OVERLAP, OPT_CHAIN_SMS, OPT_MARGIN_SPLIT, OPT_MINI, OPT_SNAPSHOT = range(14)
STAGES = ("gather", "gram", "recurrence", "gradient", "margin", "other", "loss")
MAX_SB = 16384

# every symbol include/casgd.h declares
EXPORTS = (
    "casgd_init", "casgd_outer_step", "casgd_outer_steps", "casgd_outer_steps_sampled", "casgd_outer_steps_host",
    "casgd_sgd_step_fp32",
    "casgd_sgd_steps_fp32", "casgd_loss", "casgd_loss_noalloc", "casgd_loss_noalloc_error", "casgd_invalidate_shadow", "casgd_sync", "casgd_debug_export",
    "casgd_set_option", "casgd_stage_times", "casgd_launch_count", "casgd_last_error", "casgd_destroy",
    "casgd_version", "casgd_payload_count", "casgd_step_local", "casgd_reduce_peers", "casgd_step_finish",
    "casgd_payload_alloc", "casgd_payload_free", "casgd_ipc_export", "casgd_ipc_open", "casgd_ipc_close",
)


def payload_count(s: int, b: int) -> int:
    """casgd_payload_count: FP32 words of one outer iteration's [r; strict block-lower G] (Alg. 1 line 5)."""
    return int(load().casgd_payload_count(s, b))


def loss_noalloc(X_bf16: torch.Tensor, y: torch.Tensor, loss: int, x: torch.Tensor, out: torch.Tensor,
                 stream: Optional[torch.cuda.Stream] = None) -> None:
    """casgd_loss_noalloc: F(x) into `out` (one float64 on the device) without a context and without any allocation;
    asynchronous on `stream` (default: torch's current stream). m <= 4,194,304 rows (static scratch)."""
    assert X_bf16.is_cuda and X_bf16.dtype == torch.bfloat16 and X_bf16.dim() == 2 and X_bf16.stride(1) == 1
    m, n = X_bf16.shape
    assert y.is_cuda and y.dtype == torch.float32 and y.is_contiguous() and y.numel() == m
    assert x.is_cuda and x.dtype == torch.float32 and x.is_contiguous() and x.numel() == n
    assert out.is_cuda and out.dtype == torch.float64 and out.numel() == 1
    st = stream if stream is not None else torch.cuda.current_stream(X_bf16.device)
    lib = load()
    rc = lib.casgd_loss_noalloc(X_bf16.data_ptr(), X_bf16.stride(0), y.data_ptr(), m, n, int(loss), x.data_ptr(), out.data_ptr(),
                                st.cuda_stream)
    if rc:
        raise CasgdError(rc, (lib.casgd_loss_noalloc_error() or b"").decode())


class CasgdError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{STATUS_NAMES[status] if 0 <= status < 6 else status}: {message}")
        self.status = status


_lib = None


def load() -> ctypes.CDLL:
    """dlopen libcasgd.so and declare the prototypes. Raises if the library has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2606_18463_b200.build` "
            "(or __graft_entry__.build()). There is no CPU fallback.")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i64, i32, f32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_float
    lib.casgd_init.restype = ctypes.c_int
    lib.casgd_init.argtypes = [ctypes.POINTER(vp), vp, i64, vp, i64, i32, ctypes.c_int, vp]
    lib.casgd_outer_step.restype = ctypes.c_int
    lib.casgd_outer_step.argtypes = [vp, vp, vp, i32, i32, f32]
    lib.casgd_outer_steps.restype = ctypes.c_int
    lib.casgd_outer_steps.argtypes = [vp, vp, i64, vp, i32, i32, f32]
    lib.casgd_outer_steps_sampled.restype = ctypes.c_int
    lib.casgd_outer_steps_sampled.argtypes = [vp, i64, vp, i32, i32, f32, ctypes.c_uint64, ctypes.c_uint64]
    lib.casgd_outer_steps_host.restype = ctypes.c_int
    lib.casgd_outer_steps_host.argtypes = [vp, vp, i64, vp, i32, i32, f32]
    lib.casgd_sgd_step_fp32.restype = ctypes.c_int
    lib.casgd_sgd_step_fp32.argtypes = [vp, vp, vp, i32, f32]
    lib.casgd_sgd_steps_fp32.restype = ctypes.c_int
    lib.casgd_sgd_steps_fp32.argtypes = [vp, vp, i64, vp, i32, f32]
    lib.casgd_payload_count.restype = ctypes.c_int64
    lib.casgd_payload_count.argtypes = [i32, i32]
    lib.casgd_payload_alloc.restype = ctypes.c_int
    lib.casgd_payload_alloc.argtypes = [i64, ctypes.POINTER(vp)]
    lib.casgd_payload_free.restype = ctypes.c_int
    lib.casgd_payload_free.argtypes = [vp]
    lib.casgd_ipc_export.restype = ctypes.c_int
    lib.casgd_ipc_export.argtypes = [vp, ctypes.c_char_p]
    lib.casgd_ipc_open.restype = ctypes.c_int
    lib.casgd_ipc_open.argtypes = [ctypes.c_char_p, ctypes.POINTER(vp)]
    lib.casgd_ipc_close.restype = ctypes.c_int
    lib.casgd_ipc_close.argtypes = [vp]
    lib.casgd_step_local.restype = ctypes.c_int
    lib.casgd_step_local.argtypes = [vp, vp, vp, i32, i32, vp]
    lib.casgd_reduce_peers.restype = ctypes.c_int
    lib.casgd_reduce_peers.argtypes = [vp, ctypes.POINTER(vp), i32, i32, i32]
    lib.casgd_step_finish.restype = ctypes.c_int
    lib.casgd_step_finish.argtypes = [vp, vp, i32, i32, f32, vp]
    lib.casgd_loss.restype = ctypes.c_int
    lib.casgd_loss.argtypes = [vp, vp, ctypes.POINTER(ctypes.c_double)]
    lib.casgd_loss_noalloc.restype = ctypes.c_int
    lib.casgd_loss_noalloc.argtypes = [vp, i64, vp, i64, i32, ctypes.c_int, vp, vp, vp]
    lib.casgd_loss_noalloc_error.restype = ctypes.c_char_p
    lib.casgd_loss_noalloc_error.argtypes = []
    lib.casgd_invalidate_shadow.restype = ctypes.c_int
    lib.casgd_invalidate_shadow.argtypes = [vp]
    lib.casgd_sync.restype = ctypes.c_int
    lib.casgd_sync.argtypes = [vp]
    lib.casgd_debug_export.restype = ctypes.c_int
    lib.casgd_debug_export.argtypes = [vp, ctypes.c_int, vp, i64]
    lib.casgd_set_option.restype = ctypes.c_int
    lib.casgd_set_option.argtypes = [vp, ctypes.c_int, i64]
    lib.casgd_stage_times.restype = ctypes.c_int
    lib.casgd_stage_times.argtypes = [vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(i64), ctypes.c_int]
    lib.casgd_launch_count.restype = i64
    lib.casgd_launch_count.argtypes = [vp]
    lib.casgd_last_error.restype = ctypes.c_char_p
    lib.casgd_last_error.argtypes = [vp]
    lib.casgd_destroy.restype = None
    lib.casgd_destroy.argtypes = [vp]
    lib.casgd_version.restype = ctypes.c_char_p
    lib.casgd_version.argtypes = []
    _lib = lib
    return lib


def version() -> str:
    return load().casgd_version().decode()


class DevBuf:
    """A device buffer of float32 words that is not a torch tensor: a payload allocated by casgd_payload_alloc (a
    dedicated allocation, so that its CUDA IPC handle can be exported) or a peer's payload opened from such a handle."""
    is_cuda = True
    dtype = torch.float32

    def __init__(self, ptr: int, numel: int, owned: bool):
        self.ptr, self._numel, self.owned = ptr, numel, owned

    def data_ptr(self) -> int:
        return self.ptr

    def numel(self) -> int:
        return self._numel

    def is_contiguous(self) -> bool:
        return True

    def export_handle(self) -> bytes:
        h = ctypes.create_string_buffer(64)
        rc = load().casgd_ipc_export(self.ptr, h)
        if rc != OK:
            raise CasgdError(rc, "casgd_ipc_export failed")
        return h.raw

    def close(self):
        if self.ptr:
            (load().casgd_payload_free if self.owned else load().casgd_ipc_close)(self.ptr)
            self.ptr = 0


def payload_alloc(s: int, b: int) -> DevBuf:
    """casgd_payload_alloc: an IPC-exportable payload buffer on the current device."""
    p = ctypes.c_void_p()
    n = payload_count(s, b)
    rc = load().casgd_payload_alloc(n, ctypes.byref(p))
    if rc != OK:
        raise CasgdError(rc, "casgd_payload_alloc failed")
    return DevBuf(p.value, n, True)


def ipc_open(handle: bytes, numel: int) -> DevBuf:
    """casgd_ipc_open: map another process's payload into this one."""
    p = ctypes.c_void_p()
    rc = load().casgd_ipc_open(handle, ctypes.byref(p))
    if rc != OK:
        raise CasgdError(rc, "casgd_ipc_open failed")
    return DevBuf(p.value, numel, False)


def _dev_ptr(t) -> int:
    assert t.is_cuda and t.is_contiguous(), "device tensors must be contiguous CUDA tensors"
    return t.data_ptr()


class Casgd:
    """One context per (A, y) dataset: the calls of include/casgd.h with torch tensors for memory.

    X_bf16: [m, n] torch.bfloat16 CUDA tensor (row stride may exceed n); y: [m] float32 CUDA tensor.
    Both are borrowed: keep them alive as long as this object (it holds references)."""

    def __init__(self, X_bf16: torch.Tensor, y: torch.Tensor, loss: int, stream: Optional[torch.cuda.Stream] = None):
        lib = load()
        assert X_bf16.is_cuda and X_bf16.dtype == torch.bfloat16 and X_bf16.dim() == 2 and X_bf16.stride(1) == 1
        assert y.is_cuda and y.dtype == torch.float32 and y.dim() == 1 and y.is_contiguous()
        assert y.shape[0] == X_bf16.shape[0]
        self._lib = lib
        self.X, self.y = X_bf16, y
        self.m, self.n = X_bf16.shape
        self.loss_kind = int(loss)
        self.stream = stream if stream is not None else torch.cuda.current_stream(X_bf16.device)
        self._ctx = ctypes.c_void_p()
        with torch.cuda.device(X_bf16.device):
            rc = lib.casgd_init(ctypes.byref(self._ctx), X_bf16.data_ptr(), X_bf16.stride(0), y.data_ptr(),
                                self.m, self.n, self.loss_kind, self.stream.cuda_stream)
        if rc != OK:
            self._ctx = ctypes.c_void_p()
            raise CasgdError(rc, "casgd_init failed (device not sm_100, bad arguments or out of memory)")
        self._last_sb = 0

    # -- plumbing ---------------------------------------------------------------------------
    def _check(self, rc: int):
        if rc != OK:
            raise CasgdError(rc, self._lib.casgd_last_error(self._ctx).decode())

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self._lib.casgd_destroy(self._ctx)
            self._ctx = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- the path -----------------------------------------------------------------------------
    def outer_step(self, idx: torch.Tensor, x: torch.Tensor, s: int, b: int, eta: float):
        """casgd_outer_step: idx int32 [s*b] (device), x float32 [n] (device, updated in place)."""
        assert idx.dtype == torch.int32 and idx.numel() == s * b and x.dtype == torch.float32 and x.numel() == self.n
        self._check(self._lib.casgd_outer_step(self._ctx, _dev_ptr(idx), _dev_ptr(x), s, b, eta))
        self._last_sb = s * b

    def outer_steps(self, idx: torch.Tensor, x: torch.Tensor, s: int, b: int, eta: float, n_steps: Optional[int] = None):
        """casgd_outer_steps: idx int32 [n_steps*s*b] (device)."""
        assert idx.dtype == torch.int32 and x.dtype == torch.float32 and x.numel() == self.n
        if n_steps is None:
            assert idx.numel() % (s * b) == 0
            n_steps = idx.numel() // (s * b)
        assert idx.numel() >= n_steps * s * b
        self._check(self._lib.casgd_outer_steps(self._ctx, _dev_ptr(idx), n_steps, _dev_ptr(x), s, b, eta))
        if n_steps:
            self._last_sb = s * b

    # ---- P > 1: the two halves of an outer iteration around the sum over ranks (Alg. 1 line 5) ----
    def step_local(self, idx: torch.Tensor, x: torch.Tensor, s: int, b: int, payload: torch.Tensor):
        """casgd_step_local: this slab's [r; strict block-lower G] into `payload` (payload_count(s, b) float32)."""
        assert idx.is_cuda and idx.dtype == torch.int32 and idx.is_contiguous() and idx.numel() == s * b
        assert x.is_cuda and x.dtype == torch.float32 and x.is_contiguous() and x.numel() == self.n
        assert payload.is_cuda and payload.dtype == torch.float32 and payload.is_contiguous()
        assert payload.numel() == payload_count(s, b)      # (a torch tensor or a DevBuf)
        self._check(self._lib.casgd_step_local(self._ctx, _dev_ptr(idx), _dev_ptr(x), s, b, _dev_ptr(payload)))
        self._last_sb = s * b

    def reduce_peers(self, payloads, s: int, b: int):
        """casgd_reduce_peers: sum the ranks' payloads (device tensors, possibly peer memory) into this context."""
        arr = (ctypes.c_void_p * len(payloads))(*[_dev_ptr(p) for p in payloads])
        self._check(self._lib.casgd_reduce_peers(self._ctx, arr, len(payloads), s, b))

    def step_finish(self, x: torch.Tensor, s: int, b: int, eta: float, payload: Optional[torch.Tensor] = None):
        """casgd_step_finish: recurrence on the summed [r; G] and the update of this slab of x."""
        assert x.is_cuda and x.dtype == torch.float32 and x.is_contiguous() and x.numel() == self.n
        self._check(self._lib.casgd_step_finish(self._ctx, _dev_ptr(x), s, b, eta,
                                                _dev_ptr(payload) if payload is not None else None))

    def outer_steps_sampled(self, x: torch.Tensor, s: int, b: int, eta: float, n_steps: int, seed: int, first_step: int = 0):
        """casgd_outer_steps_sampled: indices drawn on the device (Philox4x32-10, with replacement)."""
        assert x.dtype == torch.float32 and x.numel() == self.n
        self._check(self._lib.casgd_outer_steps_sampled(self._ctx, n_steps, _dev_ptr(x), s, b, eta, seed, first_step))
        if n_steps:
            self._last_sb = s * b

    def outer_steps_host(self, idx_host: torch.Tensor, x_host: torch.Tensor, s: int, b: int, eta: float,
                         n_steps: Optional[int] = None):
        """casgd_outer_steps_host: idx_host int32 and x_host float32 are HOST tensors (pinned for async copies)."""
        assert not idx_host.is_cuda and not x_host.is_cuda
        assert idx_host.dtype == torch.int32 and idx_host.is_contiguous()
        assert x_host.dtype == torch.float32 and x_host.is_contiguous() and x_host.numel() == self.n
        if n_steps is None:
            n_steps = idx_host.numel() // (s * b)
        assert idx_host.numel() >= n_steps * s * b
        self._check(self._lib.casgd_outer_steps_host(self._ctx, idx_host.data_ptr(), n_steps, x_host.data_ptr(), s, b, eta))
        if n_steps:
            self._last_sb = s * b

    def sgd_steps_fp32(self, idx: torch.Tensor, x: torch.Tensor, b: int, eta: float, n_steps: Optional[int] = None):
        """casgd_sgd_steps_fp32: the all-FP32 s = 1 baseline."""
        assert idx.dtype == torch.int32 and x.dtype == torch.float32 and x.numel() == self.n
        if n_steps is None:
            n_steps = idx.numel() // b
        assert idx.numel() >= n_steps * b
        self._check(self._lib.casgd_sgd_steps_fp32(self._ctx, _dev_ptr(idx), n_steps, _dev_ptr(x), b, eta))

    def loss(self, x: torch.Tensor) -> float:
        """casgd_loss: F(x) over the whole dataset."""
        assert x.dtype == torch.float32 and x.numel() == self.n
        out = ctypes.c_double()
        self._check(self._lib.casgd_loss(self._ctx, _dev_ptr(x), ctypes.byref(out)))
        return out.value

    def sync(self):
        self._check(self._lib.casgd_sync(self._ctx))

    def invalidate_shadow(self):
        self._check(self._lib.casgd_invalidate_shadow(self._ctx))

    def set_option(self, option: int, value: int):
        self._check(self._lib.casgd_set_option(self._ctx, option, value))

    def launch_count(self) -> int:
        return int(self._lib.casgd_launch_count(self._ctx))

    def stage_times(self, reset: bool = False):
        ms = (ctypes.c_double * len(STAGES))()
        cnt = (ctypes.c_int64 * len(STAGES))()
        self._check(self._lib.casgd_stage_times(self._ctx, ms, cnt, int(reset)))
        return {name: (ms[i], int(cnt[i])) for i, name in enumerate(STAGES)}

    def debug(self, what: int, sb: Optional[int] = None) -> np.ndarray:
        """casgd_debug_export into a fresh numpy array (see include/casgd.h for layouts)."""
        sb = self._last_sb if sb is None else sb
        shapes = {DBG_Y: ((sb, self.n), np.uint16), DBG_YLAB: ((sb,), np.float32), DBG_G: ((sb, sb), np.float32),
                  DBG_R: ((sb,), np.float32), DBG_Z: ((sb,), np.float32), DBG_U: ((sb,), np.float32),
                  DBG_XBF: ((self.n,), np.uint16), DBG_STAMPS: ((64, 8, 2), np.uint64), DBG_GUARDS: ((1,), np.int64), DBG_XSNAP: ((self.n,), np.float32)}
        shape, dt = shapes[what]
        out = np.empty(shape, dt)
        self._check(self._lib.casgd_debug_export(self._ctx, what, out.ctypes.data, out.nbytes))
        return out
