"""User-sharded multi-GPU (section 4.4, Fig. 3): one process per GPU, each holding a
contiguous range of users; lambda and b replicated; ONE exchange per evaluation -- an all-reduce (int64 SUM) of the J*m + 3
fixed-point accumulators -- issued from the library's reduce hook between the gradient kernel and the epilogue.  Because the
accumulators are integers, every rank finalises identical bits: grad g, g and the AGD update are the same on all ranks and
the same as on one GPU holding all users, so there is no rank-0 update and no broadcast (the paper's design reduces to rank
0 and broadcasts lambda).

This module is collectives + marshalling only: every arithmetic step runs in the kernels behind the C ABI.
BASELINE.json's north_star keeps the graded path on ONE GPU; this is the "next" row, unmeasured on multi-GPU hardware.
"""
from __future__ import annotations

from .binding import Problem, ShardExtents


def split_users(row_ptr, world: int, align: bool = True):
    """Contiguous user ranges balanced by nonzeros: range r = [cut[r], cut[r+1]).  row_ptr: int64 tensor / array (I+1).
    align: move every cut to the nearest user u with u even and row_ptr[u] a multiple of 4, so that the shard's slices of
    row_ptr / item_idx / c / a start on 16-byte boundaries.  Then (i) a shard can BORROW its slices in place (the streaming
    kernel's bulk copies need that alignment), and (ii) every row sits at the same position modulo 4 as in the unsharded arrays,
    so its lane assignment -- and with it the summation order inside its projection -- is the same: the sharded result is
    bit-identical to one GPU's.  Without alignment it is identical across ranks and equal to one GPU's up to fp32 rounding of
    fractional x."""
    import numpy as np
    rp = row_ptr.cpu().numpy() if hasattr(row_ptr, "cpu") else np.asarray(row_ptr)
    I, nnz = rp.size - 1, int(rp[-1])
    cuts = [0]
    for r in range(1, world):
        u = int(np.searchsorted(rp, nnz * r // world, side="left"))
        u = min(max(u, cuts[-1]), I)
        if align:
            ok = np.flatnonzero((rp[:I + 1] % 4 == 0) & (np.arange(I + 1) % 2 == 0))
            if ok.size:
                k = int(np.searchsorted(ok, u))
                cand = [int(ok[j]) for j in (k - 1, k) if 0 <= j < ok.size]
                u = max(min(cand, key=lambda v: abs(v - u)), cuts[-1])
        cuts.append(u)
    cuts.append(I)
    return cuts


class ShardedProblem:
    """A Problem over this rank's users whose evaluations all-reduce their accumulators over `dist` (torch.distributed, or
    None for a single rank).  grad / solve are the local Problem's: the hook makes them global."""

    def __init__(self, local: Problem, dist=None, device=None):
        import torch
        self.local, self.dist, self.torch = local, dist, torch
        self.device = device if device is not None else torch.device("cuda", torch.cuda.current_device())
        self._acc = torch.zeros(local.acc_words, dtype=torch.int64, device=self.device)
        self.allreduce_calls = 0
        self._agree_on_constants()
        local.set_reduce_hook(self._hook)

    def _all_reduce(self, t, op: str):
        if self.dist is not None:
            self.dist.all_reduce(t, op=getattr(self.dist.ReduceOp, op))
        return t

    def _agree_on_constants(self):
        """a0 across shards: global extents (SUM / MAX), then the fixed-point column sums in the scales those imply (int64 SUM)."""
        torch, local = self.torch, self.local
        e = local.shard_extents()
        cnt = self._all_reduce(torch.tensor([e.I, e.nnz], dtype=torch.int64, device=self.device), "SUM")
        mx = self._all_reduce(torch.tensor([e.max_abs_a, e.max_abs_c], dtype=torch.float32, device=self.device), "MAX")
        g = ShardExtents(int(cnt[0]), int(cnt[1]), float(mx[0]), float(mx[1]))
        stats = torch.empty(2 * local.J * local.m + 1, dtype=torch.int64, device=self.device)
        local.column_stats(g, stats)
        self._all_reduce(stats, "SUM")
        local.set_shard_constants(g, stats)
        self.global_extents = g

    def _hook(self, acc_ptr, n_words, lam_ptr, gamma, stream):
        """Between the gradient kernel and the epilogue: accumulators <- sum over ranks (in place, through a staging tensor
        torch.distributed can see).  Everything is enqueued on `stream`, the raw cudaStream_t the library launched the gradient
        kernel on and will launch the epilogue on: the two copies take it as an argument, and the all-reduce runs with it as
        torch's current stream (which is the stream torch.distributed orders a collective against).  An exception raised here
        makes the evaluation fail with DualipError(EHOOK) on this rank (Problem.set_reduce_hook) instead of finalising local sums."""
        if self.dist is None:
            return 0
        if self.device.type == "cuda":
            ext = self.torch.cuda.ExternalStream(stream, device=self.device) if stream else self.torch.cuda.default_stream(self.device)
            with self.torch.cuda.stream(ext):
                self.local.export_accumulators(self._acc, clear=False, stream=ext)
                self.dist.all_reduce(self._acc, op=self.dist.ReduceOp.SUM)
                self.local.import_accumulators(self._acc, accumulate=False, stream=ext)
        else:                                         # CPU stand-in of the gloo test: no streams
            self.local.export_accumulators(self._acc, clear=False)
            self.dist.all_reduce(self._acc, op=self.dist.ReduceOp.SUM)
            self.local.import_accumulators(self._acc, accumulate=False)
        self.allreduce_calls += 1
        return 0

    def set_c(self, c_new, stream=None):
        """Replace this rank's slice of c (config 5's perturbed re-solve), then agree on the constants again: sum |c| and max |c|
        are global quantities, and the library refuses to evaluate a sharded handle (DUALIP_ESTALE) until that is done.
        Collective: every rank must call it."""
        self.local.set_c(c_new, stream=stream)
        # the agreement below reads c on the library's default stream
        if stream is not None:
            stream.synchronize()
        elif self.device.type == "cuda":
            self.torch.cuda.current_stream(self.device).synchronize()
        self._agree_on_constants()

    def grad(self, *a, **kw):
        return self.local.grad(*a, **kw)

    def solve(self, *a, **kw):
        return self.local.solve(*a, **kw)

    def destroy(self):
        self.local.set_reduce_hook(None)
        self.local.destroy()
