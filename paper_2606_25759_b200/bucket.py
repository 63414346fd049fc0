"""Device-side buffers of one gradient bucket (memory plumbing only, no arithmetic).

`BucketBuffers` owns the metadata tensors (off/len/elig), the outputs and the plan/workspace
scratch that the C-ABI calls need for one bucket layout, so tests and bench.py do not repeat the
allocation boilerplate. Every computation is done by the calls in `binding`.
"""
from __future__ import annotations

from typing import Sequence

import torch

from . import binding as nf


class BucketBuffers:
    def __init__(self, off: Sequence[int], length: Sequence[int], elig: Sequence[int], n: int, W: int,
                 device="cuda", planes: bool = True, counts: bool = False, health: bool = True,
                 plane_stride: int | None = None, workspace: torch.Tensor | None = None, replicas: int = 1):
        dev = torch.device(device)
        self.T, self.n, self.W = len(off), int(n), int(W)
        T = max(self.T, 1)
        self.off = torch.tensor(list(off), dtype=torch.int64, device=dev)
        self.len = torch.tensor(list(length), dtype=torch.int64, device=dev)
        self.elig = torch.tensor(list(elig), dtype=torch.uint8, device=dev)
        self.route = torch.zeros(T, dtype=torch.uint8, device=dev)
        self.woff = torch.zeros(T, dtype=torch.int64, device=dev)
        self.summary = torch.zeros(nf.SUM_LEN, dtype=torch.int64, device=dev)
        self.plan = torch.zeros(nf.nf_plan_bytes(self.T, max(self.W, int(replicas))), dtype=torch.uint8, device=dev)
        # the fused call's scratch: the caller may share one (large enough) buffer between buckets whose calls
        # are ordered on one stream
        self.workspace = workspace if workspace is not None else torch.zeros(
            nf.nf_workspace_bytes(self.T, self.n), dtype=torch.uint8, device=dev)
        self.Wd_max = sum((int(l) + 31) // 32 for l in length)
        ps = plane_stride if plane_stride is not None else (self.Wd_max + 3) // 4 * 4
        self.plane_stride = max(ps, 4)
        self.P = self.N = None
        if planes:
            self.P = torch.zeros((W, self.plane_stride), dtype=torch.int32, device=dev)
            self.N = torch.zeros((W, self.plane_stride), dtype=torch.int32, device=dev)
        self.abs_sum = torch.zeros((W, T), dtype=torch.float64, device=dev)
        self.sumsq = self.nan_cnt = self.inf_cnt = None
        if health:
            self.sumsq = torch.zeros((W, T), dtype=torch.float64, device=dev)
            self.nan_cnt = torch.zeros((W, T), dtype=torch.int64, device=dev)
            self.inf_cnt = torch.zeros((W, T), dtype=torch.int64, device=dev)
        self.out = torch.zeros(max(self.n, 4), dtype=torch.float32, device=dev)
        self.scale = torch.zeros(T, dtype=torch.float32, device=dev)
        self.cpos = self.cneg = None
        if counts:
            self.cpos = torch.zeros(max(self.n, 1), dtype=torch.uint8, device=dev)
            self.cneg = torch.zeros(max(self.n, 1), dtype=torch.uint8, device=dev)

    # -- the five calls + the fused call, with this bucket's buffers filled in --------------------
    def route_bucket(self, state, stream=None):
        nf.nf_route_bucket(self.off, self.len, self.elig, self.T, self.n, state, self.route, self.woff,
                           self.summary, self.plan, stream)

    def sign_pack(self, g, worker_stride, mode, tau=None, stream=None):
        nf.nf_sign_pack(g, worker_stride, self.W, self.n, self.off, self.len, self.route, self.woff,
                        self.T, mode, tau, self.P, self.N if mode == nf.MODE_GTERNARY else None,
                        self.plane_stride, self.abs_sum, self.plan, stream)

    def sign_count_reduce(self, mode, margin=0, stream=None):
        nf.nf_sign_count_reduce(self.P, self.N if mode == nf.MODE_GTERNARY else None, self.plane_stride,
                                self.W, self.n, self.off, self.len, self.route, self.woff, self.T, mode,
                                margin, self.abs_sum, self.out, self.cpos, self.cneg, self.scale,
                                self.plan, stream)

    def fp32_reduce(self, g, worker_stride, alpha=1.0, stream=None):
        nf.nf_fp32_reduce(g, worker_stride, self.W, self.n, self.off, self.len, self.route, self.T,
                          alpha, self.out, self.plan, stream)

    def health_stats(self, x, replica_stride, R=None, stream=None):
        nf.nf_health_stats(x, replica_stride, self.W if R is None else R, self.n, self.off, self.len,
                           self.T, self.sumsq, self.nan_cnt, self.inf_cnt, self.plan, stream)

    def aggregate(self, g, worker_stride, state=(1, 0, 1), mode=nf.MODE_GTERNARY, tau=None, margin=0,
                  alpha=1.0, planes=None, stream=None):
        use_planes = (self.P is not None) if planes is None else planes
        nf.nf_aggregate_bucket(g, worker_stride, self.W, self.n, self.off, self.len, self.elig, self.T,
                               state, mode, tau, margin, alpha, self.route, self.woff, self.summary,
                               self.P if use_planes else None,
                               self.N if (use_planes and mode == nf.MODE_GTERNARY) else None,
                               self.plane_stride, self.abs_sum, self.sumsq, self.nan_cnt, self.inf_cnt,
                               self.out, self.scale, self.plan, self.workspace, stream)


class ModelBuffers:
    """Device buffers of a whole model's buckets, in the arrangement bench.py times (memory plumbing only):
    every bucket has its own metadata, plan, accumulators, output and — when `planes` — its own packed
    planes P/N (the "wire payload" of that bucket); the 2-bit direction workspace between the two passes of
    the fused path is one buffer with a slice per bucket (an L2-resident intermediate: a slice is written and
    read back within one bucket's kernel time). `step()` is ONE nf_aggregate_step call: one fused kernel per bucket, back to back
    on one stream, chained into a pipeline by the library."""

    def __init__(self, layouts, W: int, device="cuda", planes: bool = True, health: bool = True):
        """layouts: sequence of (off, length, elig, n) per bucket."""
        dev = torch.device(device)
        self.W = int(W)
        self.planes = planes
        self.buckets = []
        self.workspace = torch.zeros(sum(nf.nf_workspace_bytes(len(l[0]), int(l[3])) for l in layouts), dtype=torch.uint8,
                                     device=dev)
        for off, length, elig, n in layouts:
            bb = BucketBuffers(off, length, elig, n, W, dev, planes=planes, health=health, workspace=self.workspace)
            self.buckets.append(bb)
        self._desc = (nf.NfBucket * len(self.buckets))()

    def _fill(self, G, mode, tau):
        ptr = lambda t: None if t is None else t.data_ptr()
        for i, (g, bb) in enumerate(zip(G, self.buckets)):
            d = self._desc[i]
            use_planes = self.planes and bb.P is not None
            d.g, d.worker_stride, d.n = g.data_ptr(), g.shape[1], bb.n
            d.off, d.len, d.elig, d.T = bb.off.data_ptr(), bb.len.data_ptr(), bb.elig.data_ptr(), bb.T
            d.tau = ptr(tau[i]) if tau is not None else None
            d.route, d.woff, d.summary = bb.route.data_ptr(), bb.woff.data_ptr(), bb.summary.data_ptr()
            d.P = ptr(bb.P) if use_planes else None
            d.N = ptr(bb.N) if (use_planes and mode == nf.MODE_GTERNARY) else None
            d.plane_stride = bb.plane_stride
            d.abs_sum, d.sumsq = bb.abs_sum.data_ptr(), ptr(bb.sumsq)
            d.nan_cnt, d.inf_cnt = ptr(bb.nan_cnt), ptr(bb.inf_cnt)
            d.out, d.scale_out = bb.out.data_ptr(), bb.scale.data_ptr()
            d.plan, d.plan_bytes = bb.plan.data_ptr(), bb.plan.numel()

    def step(self, G, state=(1, 0, 1), mode=nf.MODE_GTERNARY, tau=None, margin=0, alpha=1.0, stream=None):
        """G: per-bucket gradient tensors [W][stride]; tau: per-bucket [T] tensors or None."""
        self._fill(G, mode, tau)
        nf.nf_aggregate_step(self._desc, self.W, state, mode, margin, alpha, self.workspace, stream)
