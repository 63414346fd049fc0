"""Shared test helpers: golden-file reader and the comparison rules of SURVEY.md §8(c)."""
import os

import numpy as np

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_golden(name):
    d = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, v = line.split(":", 1)
            d[k.strip()] = v.split()
    return d


def layout(lengths):
    off, o = [], 0
    for l in lengths:
        off.append(o)
        o += l
    return np.array(off, np.int64), np.array(lengths, np.int64), o


def assert_float_match(got, ref, rtol=1e-6, what="out"):
    """NaN where ref is NaN; equal where ref is +-Inf; zero where ref is zero (sign ignored);
    else |got-ref|/|ref| <= rtol. Returns the max relative error."""
    got = np.asarray(got)
    ref = np.asarray(ref)
    assert got.shape == ref.shape, (what, got.shape, ref.shape)
    rn = np.isnan(ref)
    assert np.array_equal(np.isnan(got), rn), f"{what}: NaN positions differ"
    ri = np.isinf(ref)
    assert np.array_equal(got[ri], ref[ri]), f"{what}: Inf positions/signs differ"
    rz = (ref == 0) & ~rn
    assert np.all(got[rz] == 0), f"{what}: nonzero where reference is zero"
    m = ~(rn | ri | rz)
    if not m.any():
        return 0.0
    r64 = ref[m].astype(np.float64)
    rel = np.abs(got[m].astype(np.float64) - r64) / np.abs(r64)
    mx = float(rel.max())
    assert mx <= rtol, f"{what}: max rel err {mx:.3e} > {rtol}"
    return mx
