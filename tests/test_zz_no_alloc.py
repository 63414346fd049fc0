"""nf_aggregate_bucket_noalloc (include/nf.h): the fused per-bucket call with its direction workspace in the
library's static device array instead of a caller buffer, for callers that may not allocate. Checked against the
existing path (nf_aggregate_bucket with a caller workspace) on the same inputs, on two calls in a row that share
the static array: the second bucket has another layout, fan-in and data, so whatever the first call left in the
array lies under it. Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest
import torch

from paper_2606_25759_b200 import BucketBuffers, binding as nf
from tests.util import assert_float_match, layout

DEV = "cuda"
RTOL = 1e-6          # the bound the parity tests use for outputs, scales and abs-sums (tests/parity.py)
RTOL_NORM = 1e-5


def _np(t):
    return t.detach().cpu().numpy()


def _noalloc(bb, g, mode, margin):
    nf.nf_aggregate_bucket_noalloc(g, g.shape[1], bb.W, bb.n, bb.off, bb.len, bb.elig, bb.T, (1, 0, 1), mode, None,
                                   margin, 1.0, bb.route, bb.woff, bb.summary, bb.P,
                                   bb.N if mode == nf.MODE_GTERNARY else None, bb.plane_stride, bb.abs_sum, bb.sumsq,
                                   bb.nan_cnt, bb.inf_cnt, bb.out, bb.scale, bb.plan)


def _case(seed, W, lens, mode, margin):
    rng = np.random.default_rng(seed)
    off, ln, n = layout(lens)
    elig = [int(x) for x in rng.integers(0, 4, len(lens)) > 0]
    elig[int(np.argmax(lens))] = 1
    g = (rng.standard_normal((W, n)) * 10 ** rng.uniform(-4, 0, (1, n))).astype(np.float32)
    g[rng.random((W, n)) < 0.05] = 0.0
    g[W // 2, off[0]] = np.nan
    gd = torch.zeros((W, (n + 3) // 4 * 4), dtype=torch.float32, device=DEV)
    gd[:, :n] = torch.from_numpy(g)
    return off, ln, elig, n, gd


@pytest.mark.gpu
def test_noalloc_entry_matches_the_existing_path_on_two_calls_in_a_row():
    cases = [(11, 8, [3000, 2048 * 70 + 13, 17, 2048 * 9, 640], nf.MODE_GTERNARY, 0),
             (12, 20, [5, 2048 * 33 + 1, 2048 * 150 + 77, 900, 1, 2048 * 4], nf.MODE_GBINARY, 2)]
    for seed, W, lens, mode, margin in cases:
        off, ln, elig, n, gd = _case(seed, W, lens, mode, margin)
        ref = BucketBuffers(off, ln, elig, n, W, DEV, planes=True, health=True)
        ref.aggregate(gd, gd.shape[1], (1, 0, 1), mode, None, margin, 1.0)
        new = BucketBuffers(off, ln, elig, n, W, DEV, planes=True, health=True)
        new.out.fill_(-3.0)
        _noalloc(new, gd, mode, margin)
        torch.cuda.synchronize()
        what = f"no-alloc call, W={W}"
        assert int(new.summary[nf.SUM_STATUS]) == nf.NF_OK and int(ref.summary[nf.SUM_STATUS]) == nf.NF_OK
        for name in ("route", "woff", "summary", "P", "nan_cnt", "inf_cnt") + (("N",) if mode == nf.MODE_GTERNARY else ()):
            assert torch.equal(getattr(new, name), getattr(ref, name)), f"{what}: {name}"
        assert int(ref.nan_cnt.sum()) == 1 and int(ref.summary[nf.SUM_NL]) > 0
        cover = np.zeros(n, bool)
        for o, l in zip(off, ln):
            cover[o:o + l] = True
        finite = ~np.isnan(_np(ref.out)[:n])
        assert np.array_equal(np.isnan(_np(new.out)[:n]), ~finite)
        assert_float_match(_np(new.out)[:n][cover & finite], _np(ref.out)[:n][cover & finite], RTOL, what + " out")
        assert bool((new.out[:n][torch.from_numpy(~cover).to(DEV)] == -3.0).all())      # gaps untouched
        assert_float_match(_np(new.scale), _np(ref.scale), RTOL, what + " scale")
        assert_float_match(_np(new.abs_sum), _np(ref.abs_sum), RTOL, what + " abs_sum")
        assert_float_match(np.sqrt(_np(new.sumsq)), np.sqrt(_np(ref.sumsq)), RTOL_NORM, what + " l2 norm")


def test_noalloc_entry_refuses_a_bucket_beyond_its_static_scratch():
    """Host-side check, nothing is launched and no pointer dereferenced: n/32 + T + 1 words of 8 bytes must fit in
    NF_NOALLOC_WORKSPACE_BYTES."""
    from paper_2606_25759_b200 import build
    build.build()
    lib = nf.lib()
    st = nf.NfState(1, 0, 1)
    fake = 0x1000
    limit = nf.NF_NOALLOC_WORKSPACE_BYTES
    n_big = 32 * (limit // 8)
    assert nf.nf_workspace_bytes(4, n_big) > limit
    args = lambda n, W=2: (fake, n, W, n, fake, fake, fake, 4, st, nf.MODE_GTERNARY, None, 0, 1.0, fake, fake, fake,
                           None, None, 0, fake, None, None, None, fake, None, fake, 1 << 20, None)
    assert lib.nf_aggregate_bucket_noalloc(*args(n_big)) == nf.NF_ERR_TOO_LARGE
    assert "NF_NOALLOC_WORKSPACE_BYTES" in nf.status_string(nf.NF_ERR_TOO_LARGE)
    assert lib.nf_aggregate_bucket_noalloc(*args(n_big, W=300)) == nf.NF_ERR_RANGE
