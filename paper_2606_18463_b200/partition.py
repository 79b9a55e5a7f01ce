"""P > 1 ranks: the paper's 1-D block-column partition (section 4.2) around the C ABI's split outer
iteration (include/casgd.h: casgd_step_local / casgd_reduce_peers / casgd_step_finish).

Host logic only -- who owns which columns, what is summed, in which order the calls go; every arithmetic step runs in
libcasgd.so (or, in the CPU tests of this logic, in a stand-in backend the test supplies). One process per GPU;
`torch.distributed` provides the sum over ranks of Alg. 1 line 5 (L118): an AllReduce of sb + b^2 s (s-1) / 2 FP32
words (r and the strict block-lower part of G; Table 2, counts the whole symmetric G).

    slab = column_slab(n, rank, P)
    step = PartitionedCasgd(CudaSlab(X[:, slab], y, loss), group)      # y: the FULL label vector on every rank
    step.outer_step(idx, x_slab, s, b, eta)                            # same idx on every rank
"""
from __future__ import annotations

from typing import Optional, Protocol

import torch


def column_slab(n: int, rank: int, P: int, align: int = 8) -> slice:
    """Columns [c0, c1) of rank `rank` of P: contiguous, in rank order, sizes as equal as `align`-column units allow
    (slab starts on 16-byte boundaries of a BF16 row, so the library can use the caller's matrix in place); the last
    rank takes the ragged tail. Every rank gets at least one column or the partition is refused."""
    if not (0 <= rank < P) or n < P:
        raise ValueError(f"cannot give each of P = {P} ranks a column of n = {n}")
    units = -(-n // align)
    if units < P:
        align, units = 1, n
    lo, rem = divmod(units, P)
    start = lambda r: (r * lo + min(r, rem)) * align
    return slice(min(start(rank), n), min(start(rank + 1), n))


def payload_words(s: int, b: int) -> int:
    """FP32 words summed per outer iteration: r (sb) and the strict block-lower G (b^2 s (s-1) / 2)."""
    return s * b + b * b * s * (s - 1) // 2


def payload_index(i: int, k: int, s: int, b: int) -> int:
    """Where entry (i, k) of G, block(k) < block(i), sits in the payload (include/casgd.h)."""
    j = i // b
    assert 0 <= k < j * b <= i < s * b
    return s * b + b * b * j * (j - 1) // 2 + (i - j * b) * j * b + k


class SlabBackend(Protocol):
    """One rank's share of an outer iteration."""

    def new_payload(self, s: int, b: int) -> torch.Tensor: ...

    def local(self, idx, x_slab, s: int, b: int, payload: torch.Tensor) -> None: ...

    def finish(self, x_slab, s: int, b: int, eta: float, payload: torch.Tensor) -> None: ...


class CudaSlab:
    """The CUDA backend: a libcasgd context on this rank's column slab."""

    def __init__(self, X_slab_bf16: torch.Tensor, y: torch.Tensor, loss: int, stream: Optional[torch.cuda.Stream] = None):
        from . import binding
        self.cg = binding.Casgd(X_slab_bf16, y, loss, stream=stream)
        self._count = binding.payload_count

    def new_payload(self, s, b):
        return torch.empty(self._count(s, b), dtype=torch.float32, device=self.cg.X.device)

    def local(self, idx, x_slab, s, b, payload):
        self.cg.step_local(idx, x_slab, s, b, payload)

    def finish(self, x_slab, s, b, eta, payload):
        self.cg.step_finish(x_slab, s, b, eta, payload)

    def close(self):
        self.cg.close()


class PartitionedCasgd:
    """One outer iteration of Alg. 1 on P ranks: local [r; G] -> sum over ranks -> recurrence + slab update.

    `group` is a torch.distributed process group (NCCL on GPUs: the paper's grouped AllReduce, L276; gloo in the CPU
    tests). With `group=None` (P = 1) the sum is the identity."""

    def __init__(self, backend: SlabBackend, group=None):
        self.backend = backend
        self.group = group
        self._payloads = {}

    def outer_step(self, idx, x_slab, s: int, b: int, eta: float):
        payload = self._payloads.get((s, b))
        if payload is None:
            payload = self._payloads[(s, b)] = self.backend.new_payload(s, b)
            assert payload.numel() == payload_words(s, b)
        self.backend.local(idx, x_slab, s, b, payload)
        if self.group is not None:
            import torch.distributed as dist
            # NCCL orders its work after the CURRENT torch stream and the stream after it: the backend's context must
            # have been created on that stream (binding.Casgd's default)
            dist.all_reduce(payload, op=dist.ReduceOp.SUM, group=self.group)
        self.backend.finish(x_slab, s, b, eta, payload)


class PeerPartitionedCasgd:
    """The same outer iteration with the library's OWN sum over ranks instead of a collective call: every rank's payload
    lives in a dedicated device allocation whose CUDA IPC handle the ranks exchange once (through `group`, any backend);
    per iteration each rank's `casgd_reduce_peers` kernel reads all P payloads -- peer memory over NVLink when the ranks
    sit on different GPUs -- and writes the rank-ordered sum straight into its recurrence's G and r.

    Ordering between the ranks is kept on the host here, the simplest correct protocol: a barrier after every rank's
    local half has finished on its stream (payloads complete), and another after every rank's reduce has finished
    (payloads may be overwritten). Device-side flags would remove both host round trips; they need one GPU per rank to
    be measured, which this build's test box does not have."""

    def __init__(self, backend: "CudaSlab", group):
        import torch.distributed as dist
        from . import binding
        self.backend, self.group, self._dist, self._binding = backend, group, dist, binding
        self._bufs = {}

    def _setup(self, s, b):
        mine = self._binding.payload_alloc(s, b)
        handles = [None] * self._dist.get_world_size(self.group)
        self._dist.all_gather_object(handles, mine.export_handle(), group=self.group)
        rank = self._dist.get_rank(self.group)
        peers = [mine if q == rank else self._binding.ipc_open(h, mine.numel()) for q, h in enumerate(handles)]
        self._bufs[(s, b)] = (mine, peers)
        return mine, peers

    def outer_step(self, idx, x_slab, s: int, b: int, eta: float):
        mine, peers = self._bufs.get((s, b)) or self._setup(s, b)
        cg = self.backend.cg
        cg.step_local(idx, x_slab, s, b, mine)
        cg.sync()
        self._dist.barrier(group=self.group)            # every rank's payload is complete
        cg.reduce_peers(peers, s, b)
        cg.step_finish(x_slab, s, b, eta, None)
        cg.sync()
        self._dist.barrier(group=self.group)            # every rank has read every payload

    def close(self):
        for mine, peers in self._bufs.values():
            for p in peers:
                p.close()
        self._bufs = {}
