"""GPU-vs-oracle comparison of one bucket (comparison rules of SURVEY.md §8(c)).

Tolerances (BASELINE.json north_star): packed planes and sign counts bit-exact; decoded low-bit
and FP32-route outputs max relative error <= 1e-6 against the fixed-worker-order oracle; health
norms <= 1e-5 relative; NaN/Inf tallies exact; route codes / word offsets / summary exact.
"""
import numpy as np
import torch

from oracle import nf_oracle as O
from paper_2606_25759_b200 import BucketBuffers, binding as nf
from tests.util import assert_float_match

RTOL_OUT = 1e-6
RTOL_NORM = 1e-5
RTOL_ABS = 1e-6


def _np(t):
    return t.detach().cpu().numpy()


def compare(bb: BucketBuffers, ref: O.BucketResult, W, mode, check_planes=True, check_counts=False,
            check_health=True, check_scale=True, what=""):
    T, n = bb.T, bb.n
    torch.cuda.synchronize()
    summ = _np(bb.summary)
    assert summ[nf.SUM_STATUS] == 0, what
    assert np.array_equal(_np(bb.route)[:T], ref.route.route), what + " route"
    assert np.array_equal(_np(bb.woff)[:T], ref.route.woff), what + " woff"
    assert [int(x) for x in summ[:6]] == [ref.route.Wd, ref.route.nL, ref.route.nF, ref.route.nP,
                                          ref.route.e, ref.route.f], what + " summary"
    Wd = ref.route.Wd
    if check_planes and Wd > 0:
        P = _np(bb.P).view(np.uint32)[:, :Wd]
        assert np.array_equal(P, ref.P), what + " pos plane"
        if mode == O.MODE_GTERNARY:
            N = _np(bb.N).view(np.uint32)[:, :Wd]
            assert np.array_equal(N, ref.N), what + " neg plane"
            assert not (P & N).any()
    A = _np(bb.abs_sum)[:, :T]
    assert_float_match(A, ref.abs_sum, RTOL_ABS, what + " abs_sum")
    out = _np(bb.out)[:n]
    # only positions covered by tensors are defined
    cover = np.zeros(n, bool)
    isL = np.zeros(n, bool)
    for o, l, r in zip(_np(bb.off), _np(bb.len), ref.route.route):
        cover[o:o + l] = True
        if r == O.ROUTE_L:
            isL[o:o + l] = True
    err = assert_float_match(out[cover], ref.out[cover], RTOL_OUT, what + " out")
    if check_scale:
        assert_float_match(_np(bb.scale)[:T], ref.scale, RTOL_OUT, what + " scale")
    if check_counts:
        cp, cn = _np(bb.cpos)[:n], _np(bb.cneg)[:n]
        assert np.array_equal(cp[isL], ref.cpos[isL]), what + " cpos"
        assert np.array_equal(cn[isL], ref.cneg[isL]), what + " cneg"
        cz = W - cp[isL].astype(int) - cn[isL].astype(int)
        assert cz.min(initial=0) >= 0                      # cpos + cneg + czero = W, czero >= 0
    if check_health:
        Q = _np(bb.sumsq)[:, :T]
        assert_float_match(np.sqrt(Q), np.sqrt(ref.sumsq), RTOL_NORM, what + " l2 norm")
        assert np.array_equal(_np(bb.nan_cnt)[:, :T].astype(np.uint64), ref.nan_cnt), what + " nan"
        assert np.array_equal(_np(bb.inf_cnt)[:, :T].astype(np.uint64), ref.inf_cnt), what + " inf"
    return err


def run_both(g: torch.Tensor, off, length, elig, state=(1, 0, 1), mode=O.MODE_GTERNARY, tau=None,
             margin=0, alpha=1.0, what=""):
    """Runs the fused call and the 5-call sequence on the device tensor g [W][stride] and checks
    both against the oracle on the same values. Returns the oracle result."""
    W, stride = g.shape
    n = int(off[-1] + length[-1]) if len(off) else 0
    n = max(n, 0)
    ref = O.aggregate_bucket(np.ascontiguousarray(_np(g)[:, :n]), off, length, elig, state, mode, tau,
                             margin, alpha)
    tau_d = None if tau is None else torch.tensor(np.asarray(tau, np.float32), device=g.device)
    # fused
    bb = BucketBuffers(off, length, elig, n, W, g.device, planes=True, counts=False, health=True)
    bb.out.fill_(-77.0)
    bb.aggregate(g, stride, state, mode, tau_d, margin, alpha)
    compare(bb, ref, W, mode, what=what + " [fused]")
    # fused without planes / health
    bb2 = BucketBuffers(off, length, elig, n, W, g.device, planes=False, counts=False, health=False)
    bb2.aggregate(g, stride, state, mode, tau_d, margin, alpha)
    compare(bb2, ref, W, mode, check_planes=False, check_health=False, what=what + " [fused lean]")
    # five calls
    bc = BucketBuffers(off, length, elig, n, W, g.device, planes=True, counts=True, health=True)
    bc.route_bucket(state)
    bc.sign_pack(g, stride, mode, tau_d)
    bc.sign_count_reduce(mode, margin)
    bc.fp32_reduce(g, stride, alpha)
    bc.health_stats(g, stride)
    compare(bc, ref, W, mode, check_counts=True, what=what + " [5-call]")
    # a3 once more WITHOUT count outputs (its 512-byte write-back path): the same bits at every low-bit position,
    # nothing written elsewhere
    if ref.route.Wd:
        out_nc = torch.full_like(bc.out, -123.0)
        nf.nf_sign_count_reduce(bc.P, bc.N if mode == O.MODE_GTERNARY else None, bc.plane_stride, W, n, bc.off, bc.len,
                                bc.route, bc.woff, bc.T, mode, margin, bc.abs_sum, out_nc, None, None, None, bc.plan)
        torch.cuda.synchronize()
        isL = np.zeros(n, bool)
        for o, l, r in zip(off, length, ref.route.route):
            if r == O.ROUTE_L:
                isL[o:o + l] = True
        a_nc, b_c = _np(out_nc)[:n], _np(bc.out)[:n]
        assert np.array_equal(a_nc[isL].view(np.uint32), b_c[isL].view(np.uint32)), what + " a3 without count outputs"
        assert np.all(a_nc[~isL] == -123.0), what + " a3 without count outputs wrote outside the low-bit tensors"
    # fused == 5-call bit for bit on planes and outputs
    torch.cuda.synchronize()
    if ref.route.Wd:
        assert torch.equal(bb.P[:, :ref.route.Wd], bc.P[:, :ref.route.Wd])
    a, b = _np(bb.out)[:n], _np(bc.out)[:n]
    m = ~(np.isnan(a) & np.isnan(b))
    cover = np.zeros(n, bool)
    for o, l in zip(off, length):
        cover[o:o + l] = True
    # same directions everywhere; magnitudes (the per-tensor scale, summed in a different order by
    # the two paths) within twice the oracle tolerance of each other; FP32-route values identical
    sel = m & cover
    assert np.array_equal(np.sign(a[sel]), np.sign(b[sel])), what + " fused vs 5-call directions"
    fin = sel & np.isfinite(a) & np.isfinite(b)
    assert np.all(np.abs(a[fin] - b[fin]) <= 2 * RTOL_OUT * np.abs(b[fin])), what + " fused vs 5-call out"
    inf = sel & ~np.isfinite(a)
    assert np.array_equal(a[inf], b[inf]), what + " fused vs 5-call inf"
    isP = cover.copy()
    for o, l, r in zip(off, length, ref.route.route):
        if r == O.ROUTE_L:
            isP[o:o + l] = False
    assert np.array_equal(a[m & isP], b[m & isP]), what + " fused vs 5-call FP32 route"
    return ref
