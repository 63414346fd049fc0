"""Seeded synthetic gradient buckets for the five configs (SURVEY.md §8(d) recipe).

Inputs only: random draws, per-tensor scales, injected zeros / NaNs. None of the method's
arithmetic lives here. The same function feeds the oracle (CPU tensors -> numpy) and the
CUDA path (device tensors); on a GPU box the tests generate on the device and copy the very
same values to the host for the oracle.

Seeds: stream(config c, bucket b, worker w) = 1_000_000*c + 1000*b + w;
       per-tensor sigma of bucket b      = 1_000_000*c + 1000*b + 999 (CPU generator, shared by all workers).
"""
from __future__ import annotations

import math

import torch

from .shapes import Bucket, Config


def _seed(cfg: Config, b: int, w: int) -> int:
    return 1_000_000 * cfg.index + 1000 * b + w


def tensor_sigmas(cfg: Config, bucket: Bucket) -> torch.Tensor:
    """[T] float64 per-tensor sigma for this bucket (same for every worker)."""
    T = len(bucket.tensors)
    if cfg.sigma_schedule == "loguniform":
        g = torch.Generator(device="cpu").manual_seed(_seed(cfg, bucket.index, 999))
        u = torch.rand(T, generator=g, dtype=torch.float64)
        lo, hi = math.log10(cfg.sigma_lo), math.log10(cfg.sigma_hi)
        return torch.pow(torch.tensor(10.0, dtype=torch.float64), lo + (hi - lo) * u)
    if cfg.sigma_schedule == "const":
        return torch.full((T,), cfg.sigma_hi, dtype=torch.float64)
    if cfg.sigma_schedule == "gpt_layer":
        # sigma decays by a TOTAL factor of 2 from the last layer to the first
        nl = 1 + max([t.layer for b in cfg.buckets for t in b.tensors])
        out = []
        for t in bucket.tensors:
            if t.layer < 0:
                out.append(cfg.sigma_hi)
            else:
                out.append(cfg.sigma_hi * 2.0 ** (-(nl - 1 - t.layer) / max(nl - 1, 1)))
        return torch.tensor(out, dtype=torch.float64)
    raise ValueError(cfg.sigma_schedule)


def gen_worker(cfg: Config, bucket: Bucket, w: int, device="cpu", out: torch.Tensor | None = None
               ) -> torch.Tensor:
    """One worker's flat FP32 gradient bucket, [n] float32 on `device`."""
    dev = torch.device(device)
    n = bucket.n
    g = torch.Generator(device=dev).manual_seed(_seed(cfg, bucket.index, w))
    if out is None:
        out = torch.empty(n, dtype=torch.float32, device=dev)
    assert out.shape == (n,) and out.dtype == torch.float32
    out.normal_(0.0, 1.0, generator=g)
    if cfg.dist == "student3":
        # t(3) = Z / sqrt(chi2_3 / 3): heavy tails
        chi = torch.zeros(n, dtype=torch.float32, device=dev)
        tmp = torch.empty(n, dtype=torch.float32, device=dev)
        for _ in range(3):
            tmp.normal_(0.0, 1.0, generator=g)
            chi.addcmul_(tmp, tmp)
        out.div_(chi.div_(3.0).sqrt_())
        del chi, tmp
    sig = tensor_sigmas(cfg, bucket).to(torch.float32)
    lens = torch.tensor(bucket.length, dtype=torch.int64)
    out.mul_(torch.repeat_interleave(sig, lens).to(dev))
    if cfg.zero_frac > 0.0:
        m = torch.rand(n, generator=g, device=dev) < cfg.zero_frac
        out.masked_fill_(m, 0.0)
    if cfg.nan_frac > 0.0 and bucket.index == cfg.nan_bucket and w == cfg.nan_worker:
        m = torch.rand(n, generator=g, device=dev) < cfg.nan_frac
        out.masked_fill_(m, float("nan"))
    return out


def stride_for(n: int) -> int:
    """Worker stride in elements: n rounded up to a multiple of 4 (16-byte aligned rows)."""
    return (n + 3) // 4 * 4


def gen_bucket(cfg: Config, bucket: Bucket, device="cpu") -> torch.Tensor:
    """[W][stride] float32 (stride = n rounded up to 4; the pad is zero)."""
    s = stride_for(bucket.n)
    g = torch.zeros((cfg.W, s), dtype=torch.float32, device=device)
    for w in range(cfg.W):
        gen_worker(cfg, bucket, w, device, g[w, :bucket.n])
    return g
