"""`-m "not gpu"` pins of the oracle's NEXT-1 functions (two-level hierarchical sign count, PAPER L243,
L267): node-local partial counts as bit-sliced planes, partial-count merge + decode."""
import numpy as np
import pytest

from oracle import nf_oracle as O
from tests.util import read_golden, layout


def _bits(words):
    return ((words[..., None] >> np.arange(32, dtype=np.uint32)) & 1).astype(np.int64)   # [..., Wd, 32]


def test_plane_count_closed_form():
    """B = number of bits of Wg = floor(log2 Wg) + 1."""
    for Wg in range(1, 256):
        assert O.count_planes(Wg) == int(np.floor(np.log2(Wg))) + 1 == Wg.bit_length()


def test_handworked_two_groups_of_two():
    d = read_golden("handworked_w4.txt")
    P = np.array([int(x, 16) for x in d["P"]], np.uint32).reshape(4, 1)
    N = np.array([int(x, 16) for x in d["N"]], np.uint32).reshape(4, 1)
    G, B = int(d["hier_G"][0]), int(d["hier_B"][0])
    for g in range(G):
        got_p = O.partial_count(P[2 * g:2 * g + 2], B)[:, 0]
        got_n = O.partial_count(N[2 * g:2 * g + 2], B)[:, 0]
        assert [int(x) for x in got_p] == [int(x, 16) for x in d[f"hier_pos_g{g}"]]
        assert [int(x) for x in got_n] == [int(x, 16) for x in d[f"hier_neg_g{g}"]]
    # level 2 reproduces the hand-worked flat result
    off, ln, n = layout([int(x) for x in d["len"]])
    route = np.array([1, 0], np.uint8)
    woff = np.array([0, -1], np.int64)
    A = np.zeros((4, 2)); A[:, 0] = [float(x) for x in d["abs_sum"]]
    cp = np.stack([O.partial_count(P[2 * g:2 * g + 2], B) for g in range(G)])
    cn = np.stack([O.partial_count(N[2 * g:2 * g + 2], B) for g in range(G)])
    out, cpos, cneg, scale = O.partial_count_merge(cp, cn, 4, n, off, ln, route, woff, O.MODE_GTERNARY, 0, A)
    S = np.float32(float(d["scale"][0]))
    assert [int(x) for x in cpos[:8]] == [int(x) for x in d["cpos"]]
    assert [int(x) for x in cneg[:8]] == [int(x) for x in d["cneg_ternary"]]
    assert np.array_equal(out[:8], np.array([S * int(x) for x in d["d_ternary"]], np.float32))
    out_b, _, _, _ = O.partial_count_merge(cp, None, 4, n, off, ln, route, woff, O.MODE_GBINARY, 0, A)
    assert np.array_equal(out_b[:8], np.array([S * int(x) for x in d["d_binary"]], np.float32))


@pytest.mark.parametrize("Wg", [1, 2, 3, 7, 8, 31, 64])
def test_partial_count_brute_force_and_plane_encoding(Wg):
    """Planes decode back to the per-bit population counts computed straight from the words."""
    rng = np.random.default_rng(Wg)
    words = rng.integers(0, 2 ** 32, size=(Wg, 37), dtype=np.uint64).astype(np.uint32)
    B = O.count_planes(Wg)
    cnt = O.partial_count(words)
    assert cnt.shape == (B, 37)
    decoded = sum(_bits(cnt[b]) << b for b in range(B))
    assert np.array_equal(decoded, _bits(words).sum(axis=0))
    assert decoded.max() <= Wg
    # extra planes beyond the necessary ones stay zero
    if B < 8:
        assert not O.partial_count(words, B + 1)[B].any()


def test_one_worker_per_group_is_the_packed_plane():
    """Wg = 1: the single partial-count plane IS the worker's packed plane (special case = the input)."""
    rng = np.random.default_rng(11)
    words = rng.integers(0, 2 ** 32, size=(1, 50), dtype=np.uint64).astype(np.uint32)
    assert np.array_equal(O.partial_count(words)[0], words[0])


@pytest.mark.parametrize("W,groups", [(4, [2, 2]), (8, [8]), (8, [1] * 8), (9, [4, 4, 1]), (16, [4] * 4), (33, [16, 16, 1])])
@pytest.mark.parametrize("mode", [O.MODE_GBINARY, O.MODE_GTERNARY])
def test_hierarchical_equals_flat(W, groups, mode):
    """Level 1 per group + level 2 == the flat sign-count reduce O3, bit for bit (counts, votes, output),
    for equal and unequal group sizes, with margin and tau."""
    rng = np.random.default_rng(100 + W)
    lens = [70, 33, 5, 64]
    off, ln, n = layout(lens)
    elig = [1, 0, 1, 1]
    g = (rng.standard_normal((W, n)) * 10 ** rng.uniform(-3, 1, (1, n))).astype(np.float32)
    g[rng.random((W, n)) < 0.15] = 0.0
    r = O.route_bucket(off, ln, elig, n)
    tau = (rng.random(len(lens)) * 1e-2).astype(np.float32)
    P, N, A = O.sign_pack(g, off, ln, r.route, r.woff, mode, tau)
    for margin in (0, 2):
        flat = O.sign_count_reduce(P, N if mode == O.MODE_GTERNARY else None, W, n, off, ln, r.route, r.woff, mode, margin, A)
        B = max(O.count_planes(x) for x in groups)
        cps, cns, w0 = [], [], 0
        for Wg in groups:
            cps.append(O.partial_count(P[w0:w0 + Wg], B))
            cns.append(O.partial_count(N[w0:w0 + Wg], B) if mode == O.MODE_GTERNARY else None)
            w0 += Wg
        cp = np.stack(cps)
        cn = np.stack(cns) if mode == O.MODE_GTERNARY else None
        hier = O.partial_count_merge(cp, cn, W, n, off, ln, r.route, r.woff, mode, margin, A)
        for a, b in zip(flat, hier):
            assert np.array_equal(a, b, equal_nan=True)


@pytest.mark.parametrize("mode", [O.MODE_GBINARY, O.MODE_GTERNARY])
def test_stock_packed_sign_every_replica_reconstructs_the_same_aggregate(mode):
    """NEXT-2: with stock packed-sign transport every worker unpacks and counts all W streams itself and
    must arrive at the same aggregate: W identical outputs, equal to the flat reduce, whose counts equal the
    brute-force counts taken straight from the floats (no words involved)."""
    rng = np.random.default_rng(11)
    W = 5
    lens = [70, 33, 400]
    off, ln, n = layout(lens)
    g = rng.standard_normal((W, n)).astype(np.float32)
    g[rng.random((W, n)) < 0.2] = 0.0
    r = O.route_bucket(off, ln, [1, 0, 1], n)
    P, N, A = O.sign_pack(g, off, ln, r.route, r.woff, mode, None, r.Wd)
    outs, gathered = O.stock_packed_sign(P, N, W, n, off, ln, r.route, r.woff, mode, 0, A)
    assert outs.shape == (W, n)
    assert gathered == W * W * r.Wd * 4 * (2 if mode == O.MODE_GTERNARY else 1)
    flat, cpos, cneg, scale = O.sign_count_reduce(P, N, W, n, off, ln, r.route, r.woff, mode, 0, A)
    for rr in range(W):
        assert np.array_equal(outs[rr], flat)
    # brute force from the floats for the two low-bit tensors
    for t in (0, 2):
        x = g[:, off[t]:off[t] + ln[t]]
        cp = (x > 0).sum(0)
        cn = (x < 0).sum(0) if mode == O.MODE_GTERNARY else W - cp
        d = np.sign(cp.astype(int) - cn.astype(int)).astype(np.float32)
        assert np.array_equal(outs[0][off[t]:off[t] + ln[t]], scale[t] * d)
