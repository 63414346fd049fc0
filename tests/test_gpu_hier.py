"""`-m gpu` parity of NEXT-1 (two-level hierarchical sign count) through the C ABI:
nf_partial_count per group of workers, nf_partial_count_merge over the groups. Partial-count planes
are bit-exact with the oracle; the merged result is bit-exact with the flat nf_sign_count_reduce (and
with the oracle within the decode tolerance)."""
import numpy as np
import pytest
import torch

from oracle import nf_oracle as O
from paper_2606_25759_b200 import BucketBuffers, binding as nf
from tests.parity import compare, _np
from workloads import shapes, gen

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _hier(cfg, b, groups, mode, margin=0, cs_pad=0, ps_pad=0):
    W = cfg.W
    assert sum(groups) == W
    g = gen.gen_bucket(cfg, b, DEV)
    ref = O.aggregate_bucket(np.ascontiguousarray(_np(g)[:, :b.n]), b.off, b.length, b.elig, (1, 0, 1), mode, None, margin)
    # plane_stride a multiple of 4 words: level 1 runs on the bulk-copy ring kernel; anything else: register-staged
    Wd0 = sum((int(l) + 31) // 32 for l, e in zip(b.length, b.elig) if e)
    bb = BucketBuffers(b.off, b.length, b.elig, b.n, W, DEV, planes=True, counts=True, health=True,
                       plane_stride=(Wd0 + 3) // 4 * 4 + ps_pad)
    bb.route_bucket((1, 0, 1))
    bb.sign_pack(g, g.shape[1], mode)
    bb.fp32_reduce(g, g.shape[1])
    bb.health_stats(g, g.shape[1])
    torch.cuda.synchronize()
    Wd = int(bb.summary[nf.SUM_WD])
    ternary = mode == nf.MODE_GTERNARY
    G = len(groups)
    B = max(nf.nf_count_planes(x) for x in groups)
    # count_stride a multiple of 4 words: bulk-copy ring kernel; anything else: register-staged merge kernel
    cs = (max(Wd, 1) + 3) // 4 * 4
    if cs_pad and (G == 1 or (B * (cs + cs_pad)) % 4 == 0):     # every group's planes must stay 16-byte aligned
        cs += cs_pad
    cnt_pos = torch.zeros((G, B, cs), dtype=torch.int32, device=DEV)
    cnt_neg = torch.zeros((G, B, cs), dtype=torch.int32, device=DEV) if ternary else None
    w0 = 0
    for gi, Wg in enumerate(groups):
        nf.nf_partial_count(bb.P[w0:], bb.N[w0:] if ternary else None, bb.plane_stride, Wg, Wd, mode, B,
                            cnt_pos[gi], cnt_neg[gi] if ternary else None, cs)
        w0 += Wg
    torch.cuda.synchronize()
    # level 1: bit-exact against the oracle's partial counts of the oracle's planes
    w0 = 0
    for gi, Wg in enumerate(groups):
        exp_p = O.partial_count(ref.P[w0:w0 + Wg], B)
        assert np.array_equal(_np(cnt_pos[gi]).view(np.uint32)[:, :Wd], exp_p), f"pos partial counts, group {gi}"
        if ternary:
            exp_n = O.partial_count(ref.N[w0:w0 + Wg], B)
            assert np.array_equal(_np(cnt_neg[gi]).view(np.uint32)[:, :Wd], exp_n), f"neg partial counts, group {gi}"
        w0 += Wg
    # flat a3 for the bit-for-bit comparison
    bb.sign_count_reduce(mode, margin)
    torch.cuda.synchronize()
    flat_out, flat_cp, flat_cn = bb.out.clone(), bb.cpos.clone(), bb.cneg.clone()
    # level 2 (L positions are overwritten; FP32-route positions stay)
    bb.cpos.zero_(); bb.cneg.zero_(); bb.scale.zero_()
    nf.nf_partial_count_merge(cnt_pos, cnt_neg, cs, G, B, W, b.n, bb.off, bb.len, bb.route, bb.woff, bb.T, mode,
                              margin, bb.abs_sum, bb.out, bb.cpos, bb.cneg, bb.scale, bb.plan)
    compare(bb, ref, W, mode, check_counts=True, what=f"{cfg.name} bucket {b.index} hierarchical {groups}")
    a, c = _np(bb.out), _np(flat_out)
    assert np.array_equal(a, c, equal_nan=True), "hierarchical vs flat output"
    assert torch.equal(bb.cpos, flat_cp) and torch.equal(bb.cneg, flat_cn)
    # without count outputs (the fast write-back path)
    out2 = torch.full_like(bb.out, -5.0)
    nf.nf_partial_count_merge(cnt_pos, cnt_neg, cs, G, B, W, b.n, bb.off, bb.len, bb.route, bb.woff, bb.T, mode,
                              margin, bb.abs_sum, out2, None, None, None, bb.plan)
    torch.cuda.synchronize()
    isL = np.zeros(b.n, bool)
    for o, l, r in zip(b.off, b.length, ref.route.route):
        if r == O.ROUTE_L:
            isL[o:o + l] = True
    assert np.array_equal(_np(out2)[:b.n][isL], a[:b.n][isL], equal_nan=True)
    assert bool((out2[:b.n][torch.from_numpy(~isL).to(DEV)] == -5.0).all())


@pytest.mark.parametrize("mode", [nf.MODE_GBINARY, nf.MODE_GTERNARY])
@pytest.mark.parametrize("groups", [[2, 2], [4], [1, 1, 1, 1], [3, 1]])
def test_tiny_hierarchical(groups, mode):
    cfg = shapes.tiny()
    _hier(cfg, cfg.buckets[0], groups, mode)
    _hier(cfg, cfg.buckets[0], groups, mode, margin=1)
    _hier(cfg, cfg.buckets[0], groups, mode, cs_pad=2)
    if len(groups) == 1:          # (several groups: their base pointers must stay 16-byte aligned)
        _hier(cfg, cfg.buckets[0], groups, mode, ps_pad=1)
        _hier(cfg, cfg.buckets[0], groups, mode, ps_pad=3, margin=1)


@pytest.mark.parametrize("name,groups", [("resnet50", [4, 4]), ("vit_b16", [8, 8]), ("vit_b16", [4, 4, 4, 4]),
                                         ("sweep_w32", [8, 8, 8, 8]), ("sweep_w128", [16] * 8), ("sweep_w128", [100, 28])])
def test_configs_hierarchical_small(name, groups):
    cfg = shapes.get(name, small=True)
    for b in cfg.buckets[:3]:
        _hier(cfg, b, groups, nf.MODE_GTERNARY)
    _hier(cfg, cfg.buckets[0], groups, nf.MODE_GBINARY, cs_pad=2)


def test_sweep_full_size_hierarchical():
    """Config 5 at full size (n = 6,553,600), W = 32 as 4 nodes of 8."""
    cfg = shapes.sweep(32)
    _hier(cfg, cfg.buckets[0], [8, 8, 8, 8], nf.MODE_GTERNARY)


@pytest.mark.parametrize("mode", [nf.MODE_GBINARY, nf.MODE_GTERNARY])
@pytest.mark.parametrize("name", ["tiny", "resnet50", "vit_b16", "sweep_w32"])
def test_stock_packed_sign_replicated_counting(name, mode):
    """NEXT-2 (Fig. 3): nf_stock_packed_sign — W gathered copies of the planes, W local
    unpack-and-count passes into W outputs. Every replica's output matches the oracle's replica, all W are bitwise
    identical to each other, to the flat nf_sign_count_reduce and to the two-level hierarchical path."""
    cfg = shapes.get(name, small=(name != "tiny"))
    W = cfg.W
    for b in cfg.buckets[:2]:
        g = gen.gen_bucket(cfg, b, DEV)
        ref = O.aggregate_bucket(np.ascontiguousarray(_np(g)[:, :b.n]), b.off, b.length, b.elig, (1, 0, 1), mode)
        ref_outs, gathered = O.stock_packed_sign(ref.P, ref.N if mode == O.MODE_GTERNARY else None, W, b.n, b.off, b.length,
                                                 ref.route.route, ref.route.woff, mode, 0, ref.abs_sum)
        bb = BucketBuffers(b.off, b.length, b.elig, b.n, W, DEV, planes=True, counts=False, health=True)
        bb.route_bucket((1, 0, 1))
        bb.sign_pack(g, g.shape[1], mode)
        ternary = mode == nf.MODE_GTERNARY
        recvP = torch.zeros((W, W, bb.plane_stride), dtype=torch.int32, device=DEV)
        recvN = torch.zeros_like(recvP) if ternary else None
        stride = (b.n + 3) // 4 * 4
        outs = torch.full((W, max(stride, 4)), -9.0, dtype=torch.float32, device=DEV)
        nf.nf_stock_packed_sign(bb.P, bb.N if ternary else None, bb.plane_stride, W, b.n, bb.off, bb.len, bb.route, bb.woff,
                                bb.T, mode, 0, bb.abs_sum, recvP, recvN, outs, outs.shape[1], bb.plan)
        bb.out.fill_(-9.0)
        bb.sign_count_reduce(mode)
        torch.cuda.synchronize()
        Wd = ref.route.Wd
        assert gathered == W * W * Wd * 4 * (2 if ternary else 1)
        for r in range(W):                                           # the gathered streams are the workers' planes
            assert np.array_equal(_np(recvP[r]).view(np.uint32)[:, :Wd], ref.P)
        isL = np.zeros(b.n, bool)
        for o, l, rt in zip(b.off, b.length, ref.route.route):
            if rt == O.ROUTE_L:
                isL[o:o + l] = True
        flat = _np(bb.out)[:b.n]
        from tests.util import assert_float_match
        for r in range(W):
            got = _np(outs[r])[:b.n]
            assert_float_match(got[isL], ref_outs[r][isL], 1e-6, f"{cfg.name} bucket {b.index} replica {r}")
            assert np.array_equal(got[isL], flat[isL], equal_nan=True), f"replica {r} differs from the flat reduce"
            assert np.all(got[~isL] == -9.0)                         # only low-bit positions are written
