"""Pins of the CPU oracle against things other than itself (`-m "not gpu"`).

Each test states the PAPER.md passage (or the SURVEY §8(c) reading) it pins. The brute-force
sides below are pure-Python loops over the floats, written from the definitions, and share
nothing with oracle/nf_oracle.c.
"""
import itertools
import math

import numpy as np
import pytest

from oracle import nf_oracle as O
from tests.util import read_golden, layout, assert_float_match


# ------------------------------------------------------------------ O1 route (L108, L132, L205, L229)
# The 16 rows, written out literally from the paper's prose — (admitted, veto, capacity_ok, elig) -> route
# code (P = 0, L = 1, F = 2). Not admitted (FP32 warm-up, L66 / L207): everything plain FP32, whatever the
# other flags say. Admitted but elig = 0 (sensitive or unmapped tensor, L132 / L205): plain FP32, never
# low-bit and never counted as a fallback. Admitted, eligible, and a Supervisor veto or a capacity-guard
# reject (L108, L229, L273): FP32 fallback F. Admitted, eligible, no veto, guard ok: low-bit L.
ROUTE_TABLE = {
    (0, 0, 0, 0): 0, (0, 0, 0, 1): 0, (0, 0, 1, 0): 0, (0, 0, 1, 1): 0,
    (0, 1, 0, 0): 0, (0, 1, 0, 1): 0, (0, 1, 1, 0): 0, (0, 1, 1, 1): 0,
    (1, 0, 0, 0): 0, (1, 0, 0, 1): 2, (1, 0, 1, 0): 0, (1, 0, 1, 1): 1,
    (1, 1, 0, 0): 0, (1, 1, 0, 1): 2, (1, 1, 1, 0): 0, (1, 1, 1, 1): 2,
}


def expected_route(admitted, veto, cap, elig):
    return ROUTE_TABLE[(admitted, veto, cap, elig)]


def test_route_table_is_complete_and_has_one_low_bit_row():
    assert len(ROUTE_TABLE) == 16
    assert [k for k, v in ROUTE_TABLE.items() if v == 1] == [(1, 0, 1, 1)]      # L needs all four conditions
    assert sorted(k for k, v in ROUTE_TABLE.items() if v == 2) == [(1, 0, 0, 1), (1, 1, 0, 1), (1, 1, 1, 1)]


def test_route_truth_table_16_rows():
    off, ln, n = layout([5, 40, 1, 64])
    for a, v, c in itertools.product((0, 1), repeat=3):
        for eligs in itertools.product((0, 1), repeat=4):
            r = O.route_bucket(off, ln, eligs, n, a, v, c)
            exp = [expected_route(a, v, c, e) for e in eligs]
            assert list(r.route) == exp
            assert r.nL + r.nF + r.nP == 4
            # woff: running ceil(len/32) over L tensors; -1 elsewhere
            w = 0
            for t in range(4):
                if exp[t] == 1:
                    assert r.woff[t] == w
                    w += (int(ln[t]) + 31) // 32
                else:
                    assert r.woff[t] == -1
            assert r.Wd == w
            assert r.e == sum(int(ln[t]) for t in range(4) if exp[t] == 1)
            assert r.e + r.f == n


def test_route_rejects_bad_layout():
    with pytest.raises(ValueError):
        O.route_bucket([0, 4], [8, 4], [1, 1], 12)       # overlap
    with pytest.raises(ValueError):
        O.route_bucket([0, 8], [8, 8], [1, 1], 12)       # beyond n


# ------------------------------------------------------------------ hand-worked bucket (L211, L60, L50)
def _hand():
    d = read_golden("handworked_w4.txt")
    W = int(d["W"][0])
    ln = [int(x) for x in d["len"]]
    elig = [int(x) for x in d["elig"]]
    g = np.array([[float(x) for x in d[f"g{w}"]] for w in range(W)], np.float32)
    return d, W, ln, elig, g


def test_handworked_bucket_ternary_and_binary():
    d, W, ln, elig, g = _hand()
    off, ln, n = layout(ln)
    for mode, dkey in ((O.MODE_GTERNARY, "d_ternary"), (O.MODE_GBINARY, "d_binary")):
        r = O.aggregate_bucket(g, off, ln, elig, (1, 0, 1), mode)
        assert list(r.route.route) == [1, 0]
        assert [int(x) for x in r.P[:, 0]] == [int(x, 16) for x in d["P"]]
        if mode == O.MODE_GTERNARY:
            assert [int(x) for x in r.N[:, 0]] == [int(x, 16) for x in d["N"]]
        assert list(r.abs_sum[:, 0]) == [float(x) for x in d["abs_sum"]]
        S = float(d["scale"][0])
        assert r.scale[0] == np.float32(S)
        assert list(r.cpos[:8]) == [int(x) for x in d["cpos"]]
        if mode == O.MODE_GTERNARY:
            assert list(r.cneg[:8]) == [int(x) for x in d["cneg_ternary"]]
            cz = W - r.cpos[:8].astype(int) - r.cneg[:8].astype(int)
            assert list(cz) == [int(x) for x in d["czero_ternary"]]
        else:
            assert list(r.cneg[:8].astype(int)) == [W - int(x) for x in d["cpos"]]
        exp = np.array([S * int(x) for x in d[dkey]], np.float32)
        assert np.array_equal(r.out[:8], exp)
        assert list(r.out[8:]) == [float(x) for x in d["fp32_sum"]]
        assert list(r.sumsq[:, 0]) == [float(x) for x in d["sumsq_t0"]]
        assert list(r.sumsq[:, 1]) == [float(x) for x in d["sumsq_t1"]]
        assert not r.nan_cnt.any() and not r.inf_cnt.any()


# ------------------------------------------------------------------ brute force on tiny inputs
def brute(g, off, ln, route, mode, tau, margin):
    """Pure-Python restatement of L211 from the floats. Returns per-position dicts."""
    W = g.shape[0]
    res = {}
    for t in range(len(off)):
        if route[t] != 1:
            continue
        th = float(np.float32(0.0 if tau is None else tau[t]))
        s = []
        for w in range(W):
            a = 0.0
            for i in range(ln[t]):
                a += abs(float(g[w, off[t] + i]))
            s.append(float(np.float32(a / ln[t])))
        S = np.float32(sum(s) / W)
        for i in range(ln[t]):
            cp = cn = 0
            for w in range(W):
                x = float(g[w, off[t] + i])
                if x > th:
                    cp += 1
                if x < -th:
                    cn += 1
            if mode == O.MODE_GBINARY:
                cn = W - cp
            D = cp - cn
            dd = 1 if D > margin else (-1 if D < -margin else 0)
            res[off[t] + i] = (cp, cn, np.float32(S * np.float32(dd)))
    return res


@pytest.mark.parametrize("W", [1, 2, 3, 4])
@pytest.mark.parametrize("mode", [O.MODE_GBINARY, O.MODE_GTERNARY])
def test_bruteforce_counts_and_decode_small(W, mode):
    rng = np.random.default_rng(100 + W)
    lens = [1, 31, 32, 33, 7, 64][: 3 + W]
    off, ln, n = layout(lens)
    assert n <= 64 * 3
    elig = [1, 1, 0, 1, 1, 0][: len(lens)]
    g = rng.standard_normal((W, n)).astype(np.float32)
    g[rng.random((W, n)) < 0.25] = 0.0                      # plenty of exact zeros
    g[0, 0] = -0.0
    tau = (rng.random(len(lens)) * 0.5).astype(np.float32)
    for tt, margin in ((None, 0), (tau, 0), (None, 1), (tau, 2)):
        r = O.aggregate_bucket(g, off, ln, elig, (1, 0, 1), mode, tt, margin)
        b = brute(g, off, ln, r.route.route, mode, tt, margin)
        rc, rn = O.sign_count_reference(g, off, ln, r.route.route, mode, tt)
        for pos, (cp, cn, o) in b.items():
            assert r.cpos[pos] == cp == rc[pos]
            assert r.cneg[pos] == cn == rn[pos]
            assert r.out[pos] == o
            assert 0 <= cp <= W and 0 <= cn <= W and cp + cn <= W     # czero >= 0; sums to W
        # packed bits agree with the floats, bit by bit; padding bits are zero; P & N == 0
        for t in range(len(lens)):
            if r.route.route[t] != 1:
                continue
            th = 0.0 if tt is None else float(tt[t])
            nw = (lens[t] + 31) // 32
            for w in range(W):
                for k in range(nw):
                    word_p = int(r.P[w, r.route.woff[t] + k])
                    word_n = int(r.N[w, r.route.woff[t] + k]) if r.N is not None else 0
                    assert word_p & word_n == 0
                    for j in range(32):
                        i = 32 * k + j
                        if i < lens[t]:
                            x = float(g[w, off[t] + i])
                            assert (word_p >> j) & 1 == int(x > th)
                            if r.N is not None:
                                assert (word_n >> j) & 1 == int(x < -th)
                        else:
                            assert (word_p >> j) & 1 == 0 and (word_n >> j) & 1 == 0


@pytest.mark.parametrize("W", [1, 2, 3, 4])
def test_exhaustive_vote_table(W):
    """All 3^W sign patterns laid across element positions: the vote is sign(#pos - #neg)
    (G-Ternary, readings #5/#6) and sign(2#pos - W) (G-Binary, reading #2)."""
    pats = list(itertools.product((-1.0, 0.0, 1.0), repeat=W))
    n = len(pats)
    g = np.array(pats, np.float32).T.copy()                 # [W][n]
    off, ln, _ = layout([n])
    for mode in (O.MODE_GTERNARY, O.MODE_GBINARY):
        r = O.aggregate_bucket(g, off, ln, [1], (1, 0, 1), mode)
        S = r.scale[0]
        for i, p in enumerate(pats):
            cp = sum(1 for v in p if v > 0)
            cn = sum(1 for v in p if v < 0) if mode == O.MODE_GTERNARY else W - cp
            assert (r.cpos[i], r.cneg[i]) == (cp, cn)
            sgn = (cp > cn) - (cp < cn)
            assert r.out[i] == np.float32(S * sgn)


# ------------------------------------------------------------------ closed forms and special cases
def test_pack_all_positive_all_zero_closed_forms():
    for L in (1, 31, 32, 33, 100):
        off, ln, n = layout([L])
        for val, full in ((2.0, True), (0.0, False), (-3.0, False)):
            g = np.full((2, n), val, np.float32)
            r = O.route_bucket(off, ln, [1], n)
            P, N, A = O.sign_pack(g, off, ln, r.route, r.woff, O.MODE_GTERNARY)
            nw = (L + 31) // 32
            for k in range(nw):
                bits = min(32, L - 32 * k)
                fullword = (1 << bits) - 1
                assert int(P[0, k]) == (fullword if full else 0)
                assert int(N[0, k]) == (fullword if val < 0 else 0)
            assert A[0, 0] == L * abs(val) and A[1, 0] == L * abs(val)


def test_scale_constant_tensor_and_numpy_abs_sum():
    # constant c, len power of two: A = len*|c| exactly
    off, ln, n = layout([1024, 4096])
    g = np.empty((3, n), np.float32)
    g[:, :1024] = -0.375
    g[:, 1024:] = 2.0 ** -20
    r = O.route_bucket(off, ln, [1, 1], n)
    _, _, A = O.sign_pack(g, off, ln, r.route, r.woff, O.MODE_GBINARY)
    assert np.all(A[:, 0] == 1024 * 0.375) and np.all(A[:, 1] == 4096 * 2.0 ** -20)
    # library routine: float64 sum of |x| (numpy pairwise sum; agree to fp64 rounding)
    rng = np.random.default_rng(7)
    g = (rng.standard_normal((4, n)) * 1e-3).astype(np.float32)
    _, _, A = O.sign_pack(g, off, ln, r.route, r.woff, O.MODE_GBINARY)
    for w in range(4):
        for t in range(2):
            ref = np.abs(g[w, off[t]:off[t] + ln[t]]).astype(np.float64).sum()
            assert abs(A[w, t] - ref) <= 1e-12 * ref
    # popcount identity: popcount(P_w over tensor t) = #{x > 0}
    P, N, _ = O.sign_pack(g, off, ln, r.route, r.woff, O.MODE_GTERNARY)
    for w in range(4):
        for t in range(2):
            words = P[w, r.woff[t]: r.woff[t] + (ln[t] + 31) // 32]
            assert sum(bin(int(x)).count("1") for x in words) == int((g[w, off[t]:off[t] + ln[t]] > 0).sum())


def test_identical_workers_is_scaled_sign_sgd_and_sign_flip():
    """W identical workers, tau=0, m=0 => out = mean|g| * sign(g) (textbook scaled signSGD);
    W=1 the same; flipping all signs negates out exactly (G-Ternary)."""
    rng = np.random.default_rng(3)
    off, ln, n = layout([100, 37])
    x = rng.standard_normal(n).astype(np.float32)
    x[::9] = 0.0
    for W in (1, 2, 5):
        g = np.tile(x, (W, 1))
        r = O.aggregate_bucket(g, off, ln, [1, 1], (1, 0, 1), O.MODE_GTERNARY)
        for t in range(2):
            seg = x[off[t]:off[t] + ln[t]]
            # all s_w are the same float, so their fp64 mean rounds back to it exactly
            S = np.float32(np.abs(seg).astype(np.float64).sum() / ln[t])
            assert abs(float(r.scale[t]) - float(S)) <= 2e-7 * float(S)
            assert np.array_equal(r.out[off[t]:off[t] + ln[t]], r.scale[t] * np.sign(seg))
            assert set(np.unique(r.cpos[off[t]:off[t] + ln[t]])) <= {0, W}
        r2 = O.aggregate_bucket(-g, off, ln, [1, 1], (1, 0, 1), O.MODE_GTERNARY)
        assert np.array_equal(r2.out, -r.out)


def test_counts_permutation_invariant_and_sum_to_W():
    rng = np.random.default_rng(11)
    W = 7
    off, ln, n = layout([70, 50])
    g = rng.standard_normal((W, n)).astype(np.float32)
    g[rng.random((W, n)) < 0.2] = 0.0
    r = O.aggregate_bucket(g, off, ln, [1, 1], (1, 0, 1), O.MODE_GTERNARY)
    perm = rng.permutation(W)
    r2 = O.aggregate_bucket(g[perm], off, ln, [1, 1], (1, 0, 1), O.MODE_GTERNARY)
    assert np.array_equal(r.cpos, r2.cpos) and np.array_equal(r.cneg, r2.cneg)
    cz = W - r.cpos.astype(int) - r.cneg.astype(int)
    assert cz.min() >= 0
    assert np.array_equal(cz, (g == 0).sum(axis=0))
    # out only takes the three values {-S, 0, +S} per tensor
    for t in range(2):
        seg = r.out[off[t]:off[t] + ln[t]]
        assert set(np.unique(np.abs(seg))) <= {np.float32(0), r.scale[t]}


# ------------------------------------------------------------------ O4a FP32 route (L50, L144)
def test_fp32_route_is_plain_ordered_sum():
    rng = np.random.default_rng(5)
    W = 6
    off, ln, n = layout([33, 17, 64])
    g = (rng.standard_normal((W, n)) * 10 ** rng.uniform(-3, 3, (W, n))).astype(np.float32)
    r = O.route_bucket(off, ln, [0, 0, 0], n)
    out = O.fp32_reduce(g, off, ln, r.route, 1.0)
    acc = g[0].copy()
    for w in range(1, W):
        acc = (acc + g[w]).astype(np.float32)              # numpy float32 add, worker order
    assert np.array_equal(out, acc)
    # integer-valued floats: exact in any order
    gi = rng.integers(-1000, 1000, (W, n)).astype(np.float32)
    assert np.array_equal(O.fp32_reduce(gi, off, ln, r.route, 1.0), gi.sum(axis=0, dtype=np.float64).astype(np.float32))
    # W = 1: identity copy times alpha
    assert np.array_equal(O.fp32_reduce(g[:1], off, ln, r.route, 0.5), (g[0] * np.float32(0.5)))
    # NaN / Inf propagate
    g2 = g.copy(); g2[2, 5] = np.nan; g2[1, 6] = np.inf; g2[3, 7] = -np.inf; g2[4, 7] = np.inf
    o2 = O.fp32_reduce(g2, off, ln, r.route, 1.0)
    assert np.isnan(o2[5]) and o2[6] == np.inf and np.isnan(o2[7])


def test_three_state_preflight_whole_bucket_fp32(tmp_path):
    """L207: the same binding through FP32 warm-up -> admission -> forced veto. In warm-up and
    under veto the whole bucket output is bit-identical to the FP32 route over all tensors."""
    rng = np.random.default_rng(9)
    off, ln, n = layout([40, 8, 100, 3])
    elig = [1, 0, 1, 0]
    g = rng.standard_normal((4, n)).astype(np.float32)
    plain = O.fp32_reduce(g, off, ln, np.zeros(4, np.uint8), 1.0)
    warm = O.aggregate_bucket(g, off, ln, elig, (0, 0, 1))
    veto = O.aggregate_bucket(g, off, ln, elig, (1, 1, 1))
    guard = O.aggregate_bucket(g, off, ln, elig, (1, 0, 0))
    adm = O.aggregate_bucket(g, off, ln, elig, (1, 0, 1))
    assert np.array_equal(warm.out, plain) and (warm.route.nP, warm.route.nL, warm.route.nF) == (4, 0, 0)
    assert np.array_equal(veto.out, plain) and (veto.route.nP, veto.route.nL, veto.route.nF) == (2, 0, 2)
    assert np.array_equal(guard.out, plain) and guard.route.nF == 2
    assert (adm.route.nP, adm.route.nL, adm.route.nF) == (2, 2, 0)
    for t in (1, 3):                                         # sensitive tensors never change route
        assert np.array_equal(adm.out[off[t]:off[t] + ln[t]], plain[off[t]:off[t] + ln[t]])


# ------------------------------------------------------------------ O4b health (BASELINE.json step 4)
def test_health_closed_form_injection_and_numpy_norm():
    off, ln, n = layout([256, 1000])
    x = np.empty((2, n), np.float32)
    x[:, :256] = 0.5
    x[:, 256:] = -3.0
    Q, cn, ci = O.health_stats(x, off, ln)
    assert np.all(Q[:, 0] == 256 * 0.25) and np.all(Q[:, 1] == 1000 * 9.0)
    rng = np.random.default_rng(2)
    x = (rng.standard_normal((3, n)) * 1e-2).astype(np.float32)
    nan_pos = rng.choice(1000, 13, replace=False) + 256
    inf_pos = rng.choice(256, 5, replace=False)
    x[1, nan_pos] = np.nan
    x[1, inf_pos[:3]] = np.inf
    x[1, inf_pos[3:]] = -np.inf
    Q, cn, ci = O.health_stats(x, off, ln)
    assert cn.tolist() == [[0, 0], [0, 13], [0, 0]] and ci.tolist() == [[0, 0], [5, 0], [0, 0]]
    for r in range(3):
        for t in range(2):
            seg = x[r, off[t]:off[t] + ln[t]].astype(np.float64)
            ref = np.linalg.norm(seg[np.isfinite(seg)])
            assert abs(math.sqrt(Q[r, t]) - ref) <= 1e-12 * ref


def test_nan_propagation_reading_11():
    """Reading #11: NaN votes 'zero'; the (worker,tensor) scale and hence the decoded tensor become NaN."""
    off, ln, n = layout([64, 32])
    rng = np.random.default_rng(1)
    g = rng.standard_normal((3, n)).astype(np.float32)
    g[1, 5] = np.nan
    r = O.aggregate_bucket(g, off, ln, [1, 1])
    assert np.all(np.isnan(r.out[:64])) and not np.isnan(r.out[64:]).any()
    assert r.cpos[5] == (g[[0, 2], 5] > 0).sum() and r.cneg[5] == (g[[0, 2], 5] < 0).sum()
    assert r.nan_cnt[1, 0] == 1 and r.nan_cnt.sum() == 1
