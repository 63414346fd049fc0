"""`-m gpu` parity of WHOLE configs at BASELINE.json's full sizes, in exactly the buffer arrangement and
launch sequence `bench.py` times (`ModelBuffers`: every bucket resident in HBM, per-bucket planes,
accumulators and direction-workspace slices, ONE `nf_aggregate_step` call per step: one fused kernel per bucket,
chained, on one stream with no host synchronisation in between). Two full steps are run before anything is compared, so
that what is checked is the steady state (plans, accumulators and workspace reused from the previous step);
then EVERY bucket of the config is compared with the oracle element by element (planes, abs-sums, decoded and
FP32-route outputs, scales, health statistics, route codes). PAPER.md L285 / L455-456: zero aggregate-output
and local-count mismatches; BASELINE.json target "all five configs match the oracle".

The C oracle streams bucket by bucket from a host copy (about 0.5 GB/s of gradient input: ~10 s for ViT-B/16,
~80 s for GPT-2-1.3B)."""
import numpy as np
import pytest
import torch

from oracle import nf_oracle as O
from paper_2606_25759_b200 import ModelBuffers, binding as nf
from tests.parity import compare, _np
from workloads import shapes, gen

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _whole_config(cfg, mode=O.MODE_GTERNARY, steps=2):
    G = [gen.gen_bucket(cfg, b, DEV) for b in cfg.buckets]
    mb = ModelBuffers([(b.off, b.length, b.elig, b.n) for b in cfg.buckets], cfg.W, DEV, planes=True, health=True)
    for bb in mb.buckets:
        bb.out.fill_(-77.0)
    for _ in range(steps):
        mb.step(G, (1, 0, 1), mode, None, 0, 1.0)
    torch.cuda.synchronize()
    worst = 0.0
    for b, g, bb in zip(cfg.buckets, G, mb.buckets):
        gh = np.ascontiguousarray(_np(g)[:, :b.n])
        ref = O.aggregate_bucket(gh, b.off, b.length, b.elig, (1, 0, 1), mode)
        del gh
        worst = max(worst, compare(bb, ref, cfg.W, mode, what=f"{cfg.name} bucket {b.index} (whole-config step)"))
        if cfg.nan_frac and b.index == cfg.nan_bucket:
            assert ref.nan_cnt[cfg.nan_worker].sum() > 0
            assert ref.nan_cnt.sum() == ref.nan_cnt[cfg.nan_worker].sum()
        del ref
    del G, mb
    torch.cuda.empty_cache()
    return worst


def test_tiny_whole_config():
    assert _whole_config(shapes.tiny(), steps=3) <= 1e-6


def test_resnet50_whole_config():
    cfg = shapes.resnet50()
    assert len(cfg.buckets) == 4
    _whole_config(cfg)
    _whole_config(cfg, mode=O.MODE_GBINARY)


def test_vit_b16_whole_config():
    cfg = shapes.vit_b16()
    assert (cfg.n_tensors, cfg.n_params, len(cfg.buckets)) == (152, 86_567_656, 13)
    _whole_config(cfg)


def test_gpt2_1p3b_whole_config():
    """All 37 buckets (42 GB of gradients resident), incl. the NaN-injected bucket 1 and the 401 MB all-FP32
    embedding bucket 36."""
    cfg = shapes.gpt2_1p3b()
    assert (cfg.n_tensors, cfg.n_params, len(cfg.buckets)) == (292, 1_313_626_112, 37)
    _whole_config(cfg)


@pytest.mark.parametrize("W", shapes.SWEEP_W)
def test_sweep_whole_config(W):
    _whole_config(shapes.sweep(W), steps=2)


def test_step_chain_with_breakers_and_bitwise_equal_to_single_calls():
    """nf_aggregate_step on an irregular sequence of buckets: small and large, a bucket of 300 tensors (routed by a
    separate kernel: breaks the chain), a one-tile bucket, W > 8, repeated three times. Every bucket must match the
    oracle AND be bitwise identical to what a stand-alone nf_aggregate_bucket call produces for it."""
    from tests.util import layout
    rng = np.random.default_rng(2024)
    W = 12
    specs = []
    for T, big in ((5, 2048 * 120 + 7), (300, 2048 * 40), (3, 100), (40, 2048 * 300 + 1), (7, 2048 * 9), (1, 2048 * 64), (20, 5000)):
        lens = [int(x) for x in rng.integers(1, 4000, T)]
        lens[T // 2] = big
        off, ln, n = layout(lens)
        elig = [int(x) for x in rng.integers(0, 2, T)]
        elig[T // 2] = 1
        specs.append((off, ln, elig, n))
    G, refs = [], []
    for off, ln, elig, n in specs:
        g = (rng.standard_normal((W, n)) * 10 ** rng.uniform(-4, 0, (1, n))).astype(np.float32)
        g[rng.random((W, n)) < 0.03] = 0.0
        gd = torch.zeros((W, (n + 3) // 4 * 4), dtype=torch.float32, device=DEV)
        gd[:, :n] = torch.from_numpy(g)
        G.append(gd)
        refs.append(O.aggregate_bucket(g, off, ln, elig))
    mb = ModelBuffers(specs, W, DEV, planes=True, health=True)
    for _ in range(3):
        for bb in mb.buckets:
            bb.out.fill_(-5.0)
        mb.step(G)
    torch.cuda.synchronize()
    for i, (bb, ref) in enumerate(zip(mb.buckets, refs)):
        compare(bb, ref, W, O.MODE_GTERNARY, what=f"step bucket {i}")
    # bitwise against stand-alone calls
    from paper_2606_25759_b200 import BucketBuffers
    for i, ((off, ln, elig, n), g, bb) in enumerate(zip(specs, G, mb.buckets)):
        one = BucketBuffers(off, ln, elig, n, W, DEV, planes=True, health=True)
        one.aggregate(g, g.shape[1])
        torch.cuda.synchronize()
        for name in ("out", "scale", "abs_sum", "sumsq", "nan_cnt", "inf_cnt", "P", "N", "route", "woff"):
            a, b = getattr(bb, name), getattr(one, name)
            assert torch.equal(a.view(torch.uint8), b.view(torch.uint8)), f"bucket {i}: {name} differs from the stand-alone call"


def test_step_with_a_refused_bucket_in_the_middle():
    """A bucket with a bad layout inside a step: it is refused on the device (status in its summary, nothing written),
    its neighbours are aggregated as usual, and the next step works again."""
    from tests.util import layout
    rng = np.random.default_rng(7)
    W = 4
    off, ln, n = layout([3000, 2048 * 30, 500])
    specs = [(off, ln, [1, 1, 0], n), (np.array([0, 8], np.int64), np.array([16, 8], np.int64), [1, 1], 32), (off, ln, [0, 1, 1], n)]
    G, refs = [], []
    for off_, ln_, elig_, n_ in specs:
        g = rng.standard_normal((W, n_)).astype(np.float32)
        gd = torch.zeros((W, (n_ + 3) // 4 * 4), dtype=torch.float32, device=DEV)
        gd[:, :n_] = torch.from_numpy(g)
        G.append(gd)
        refs.append(None if n_ == 32 else O.aggregate_bucket(g, off_, ln_, elig_))
    mb = ModelBuffers(specs, W, DEV, planes=True, health=True)
    for _ in range(2):
        mb.buckets[1].out.fill_(9.0)
        mb.step(G)
        torch.cuda.synchronize()
        assert int(mb.buckets[1].summary[nf.SUM_STATUS]) == nf.NF_ERR_ARG
        assert bool((mb.buckets[1].out == 9.0).all())
        for i in (0, 2):
            compare(mb.buckets[i], refs[i], W, O.MODE_GTERNARY, what=f"bucket {i} beside a refused bucket")


@pytest.mark.parametrize("seed,W,lean", [(1, 4, False), (2, 12, False), (3, 40, False), (4, 8, False), (5, 8, True), (6, 20, True)])
def test_random_step_chains_bitwise_equal_to_single_calls(seed, W, lean):
    """Random sequences of buckets through nf_aggregate_step: runs of tiny buckets (kernels of a few CTAs that overlap
    their neighbours, grids of different sizes handing decode units on to each other), large ones, chain breakers
    (T > 256, empty buckets), all-FP32 and all-low-bit buckets, four steps in a row on the same plans. Every output of
    every bucket must be bitwise what a stand-alone nf_aggregate_bucket call produces (itself checked against the
    oracle elsewhere), after the last step and after the first. `lean`: G-Binary, no planes, no health statistics (the
    other template instances of the chained kernel)."""
    from tests.util import layout
    from paper_2606_25759_b200 import BucketBuffers
    rng = np.random.default_rng(9000 + seed)
    specs = []
    for _ in range(int(rng.integers(9, 14))):
        kind = rng.integers(0, 6)
        if kind == 0:
            T = int(rng.integers(1, 4)); lens = [int(x) for x in rng.integers(1, 300, T)]                 # tiny
        elif kind == 1:
            T = int(rng.integers(2, 30)); lens = [int(x) for x in rng.integers(1, 6000, T)]               # small
        elif kind == 2:
            T = int(rng.integers(1, 6)); lens = [int(x) for x in rng.integers(2048 * 50, 2048 * 400, T)]   # large
        elif kind == 3:
            T = int(rng.integers(257, 300)); lens = [int(x) for x in rng.integers(1, 500, T)]              # breaks the chain
        elif kind == 4:
            T = 0; lens = []                                                                                # empty bucket
        else:
            T = int(rng.integers(3, 12)); lens = [int(x) for x in rng.integers(1, 2048 * 12, T)]
        off, ln, n = layout(lens)
        mode = rng.integers(0, 3)
        elig = [1] * T if mode == 0 else ([0] * T if mode == 1 else [int(x) for x in rng.integers(0, 2, T)])
        specs.append((off, ln, elig, n))
    G = []
    for off, ln, elig, n in specs:
        g = (rng.standard_normal((W, max(n, 1))) * 10 ** rng.uniform(-4, 0, (1, max(n, 1)))).astype(np.float32)
        g[rng.random(g.shape) < 0.03] = 0.0
        gd = torch.zeros((W, (max(n, 1) + 3) // 4 * 4), dtype=torch.float32, device=DEV)
        gd[:, :g.shape[1]] = torch.from_numpy(g)
        G.append(gd)
    names = ("out", "scale", "abs_sum", "route", "woff", "summary") + (() if lean else ("sumsq", "nan_cnt", "inf_cnt", "P", "N"))
    mode = O.MODE_GBINARY if lean else O.MODE_GTERNARY
    ones = []
    for (off, ln, elig, n), g in zip(specs, G):
        one = BucketBuffers(off, ln, elig, n, W, DEV, planes=not lean, health=not lean)
        one.out.fill_(-5.0)
        one.aggregate(g, g.shape[1], (1, 0, 1), mode, None, 1 if lean else 0, 1.0)
        ones.append(one)
    mb = ModelBuffers(specs, W, DEV, planes=not lean, health=not lean)
    for step in range(4):
        for bb in mb.buckets:
            bb.out.fill_(-5.0)
        mb.step(G, (1, 0, 1), mode, None, 1 if lean else 0, 1.0)
        if step in (0, 3):
            torch.cuda.synchronize()
            for i, (bb, one) in enumerate(zip(mb.buckets, ones)):
                assert int(bb.summary[nf.SUM_STATUS]) == nf.NF_OK
                for name in names:
                    a, b = getattr(bb, name), getattr(one, name)
                    assert torch.equal(a.view(torch.uint8), b.view(torch.uint8)), \
                        f"seed {seed} step {step} bucket {i} (T = {bb.T}, n = {bb.n}): {name} differs from the stand-alone call"
