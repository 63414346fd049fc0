"""`-m gpu` parity of WHOLE configs at BASELINE.json's full sizes, in exactly the buffer arrangement and
launch sequence `bench.py` times (`ModelBuffers`: every bucket resident in HBM, per-bucket planes and
accumulators, ONE shared direction workspace, one `nf_aggregate_bucket` per bucket issued back to back on
one stream with no host synchronisation in between). Two full steps are run before anything is compared, so
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
