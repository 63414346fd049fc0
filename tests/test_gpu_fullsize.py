"""`-m gpu` parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(fused nf_aggregate_bucket, planes + health on). The C oracle handles ~0.5 GB/s of gradient input,
so whole buckets are compared element by element: every bucket of ResNet-50, selected buckets of
ViT-B/16 and GPT-2-1.3B (first low-bit bucket, the NaN-injected bucket, the 401 MB embedding
bucket), and the reducer sweep at every W."""
import numpy as np
import pytest
import torch

from oracle import nf_oracle as O
from paper_2606_25759_b200 import BucketBuffers, binding as nf
from tests.parity import compare, _np
from workloads import shapes, gen

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _check_bucket(cfg, b, mode=O.MODE_GTERNARY, five_call=False):
    g = gen.gen_bucket(cfg, b, DEV)
    gh = np.ascontiguousarray(_np(g)[:, :b.n])
    ref = O.aggregate_bucket(gh, b.off, b.length, b.elig, (1, 0, 1), mode)
    del gh
    bb = BucketBuffers(b.off, b.length, b.elig, b.n, cfg.W, DEV, planes=True, counts=five_call, health=True)
    bb.aggregate(g, g.shape[1], (1, 0, 1), mode)
    err = compare(bb, ref, cfg.W, mode, what=f"{cfg.name} bucket {b.index} fused")
    if five_call:
        bb.out.zero_()
        bb.route_bucket((1, 0, 1))
        bb.sign_pack(g, g.shape[1], mode)
        bb.sign_count_reduce(mode)
        bb.fp32_reduce(g, g.shape[1])
        bb.health_stats(g, g.shape[1])
        compare(bb, ref, cfg.W, mode, check_counts=True, what=f"{cfg.name} bucket {b.index} 5-call")
    del g, bb
    torch.cuda.empty_cache()
    return ref, err


def test_resnet50_full_all_buckets():
    cfg = shapes.resnet50()
    assert (cfg.n_tensors, cfg.n_params, len(cfg.buckets)) == (161, 25_557_032, 4)
    for b in cfg.buckets:
        _check_bucket(cfg, b, five_call=True)


def test_vit_b16_full_selected_buckets():
    cfg = shapes.vit_b16()
    assert (cfg.n_tensors, cfg.n_params, len(cfg.buckets)) == (152, 86_567_656, 13)
    for i in (0, 5, 12):
        _check_bucket(cfg, cfg.buckets[i], five_call=(i == 0))


def test_gpt2_1p3b_full_selected_buckets():
    cfg = shapes.gpt2_1p3b()
    assert (cfg.n_tensors, cfg.n_params, len(cfg.buckets)) == (292, 1_313_626_112, 37)
    _check_bucket(cfg, cfg.buckets[0])
    ref, _ = _check_bucket(cfg, cfg.buckets[1], five_call=True)       # NaN-injected bucket
    assert ref.nan_cnt[3].sum() > 0 and ref.nan_cnt.sum() == ref.nan_cnt[3].sum()
    b = cfg.buckets[1]
    for t, (o, l, r) in enumerate(zip(b.off, b.length, ref.route.route)):
        if r == O.ROUTE_L and ref.nan_cnt[3, t] > 0:
            assert np.isnan(ref.out[o:o + l]).all()                    # reading #11
    _check_bucket(cfg, cfg.buckets[36])                                # wte + wpe, 105 M elements, all FP32


@pytest.mark.parametrize("W", shapes.SWEEP_W)
def test_reducer_sweep_full(W):
    cfg = shapes.sweep(W)
    _check_bucket(cfg, cfg.buckets[0], five_call=(W <= 32))
    if W == 8:
        _check_bucket(cfg, cfg.buckets[0], mode=O.MODE_GBINARY, five_call=True)


@pytest.mark.parametrize("n", [131_072, 524_288])
def test_paper_local_count_shapes(n):
    """8 x 131K and 8 x 524K logical buckets, zero mismatches."""
    cfg = shapes.paper_local_count(n)
    _check_bucket(cfg, cfg.buckets[0], five_call=True)


def test_gpt2_bucket_binary_mode_full_size():
    """G-Binary (one plane, cneg = W - cpos) on a full 33.6 M-element GPT bucket through the fused call."""
    cfg = shapes.gpt2_1p3b()
    _check_bucket(cfg, cfg.buckets[2], mode=O.MODE_GBINARY)
