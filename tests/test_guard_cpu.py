"""`-m "not gpu"`: NEXT-3, MGTR accounting and the endpoint-capacity guard (L273-275).
Pins of the oracle (oracle/guard_oracle.py), then the product's host functions nf_mgtr / nf_capacity_guard
(libnf.so, no GPU needed) against it."""
import math

import numpy as np
import pytest

from oracle import guard_oracle as G


def test_mgtr_closed_forms():
    ev_fp32 = [(1000, G.ROUTE_P, 0), (500, G.ROUTE_F, G.MODE_GTERNARY)]
    assert G.mgtr(ev_fp32) == 1.0                                     # fallback and plain FP32 count as FP32
    # all low-bit, G-Binary, no scale bytes: 1 bit instead of 32
    assert G.mgtr([(4096, G.ROUTE_L, G.MODE_GBINARY)], scale_bytes=0) == pytest.approx(1 / 32)
    assert G.mgtr([(4096, G.ROUTE_L, G.MODE_GTERNARY)], scale_bytes=0) == pytest.approx(math.log2(3) / 32)
    # mixture: share s of the bytes low-bit at b bits -> 1 - s (1 - b/32)
    n = 10_000
    ev = [(n, G.ROUTE_L, G.MODE_GBINARY)] * 3 + [(n, G.ROUTE_P, 0)] * 7
    assert G.mgtr(ev, scale_bytes=0) == pytest.approx(1 - 0.3 * (1 - 1 / 32))
    # the scale adds 4 bytes per low-bit tensor event
    assert G.mgtr([(8, G.ROUTE_L, G.MODE_GBINARY)]) == pytest.approx((1 + 4) / 32)
    assert G.mgtr([]) == 1.0


def test_mgtr_against_the_papers_distilbert_row():
    """PAPER L327 / Table 13: MGTR 0.824x at 29.1 % low-bit route share (DistilBERT). With G-Ternary at
    log2(3) bits (reading #14) this needs 63.4 % of an event's bytes to be low-bit eligible (SURVEY §8(c) #14:
    the eight DistilBERT rows share that factor); the formula then reproduces the printed ratio to 3 digits."""
    per_event = [(634, G.ROUTE_L, G.MODE_GTERNARY), (366, G.ROUTE_P, 0)]       # one low-bit step
    fp32_event = [(1000, G.ROUTE_P, 0)]
    ev = per_event * 291 + fp32_event * 709
    assert G.mgtr(ev, scale_bytes=0) == pytest.approx(0.824, abs=1.5e-3)


def test_guard_break_even_and_monotonicities():
    n, nodes, F, bw, p = 6_553_600, 4, 8, 25e9, 2
    # closed-form break-even service rate: t_hier == t_fp32
    ring = 2 * (nodes - 1) / nodes
    B = G.count_planes(nodes * F)
    r_star = F * (p * n / 8) / (ring * 4 * n / bw - ring * (p * B * n / 8) / bw)
    assert G.guard(n, nodes, F, r_star * 1.01, bw, p) == 1
    assert G.guard(n, nodes, F, r_star * 0.99, bw, p) == 0
    # L275: losses concentrate under fast networks, high fan-in, low endpoint service rate
    r = r_star * 1.5
    assert G.guard(n, nodes, F, r, bw, p) == 1
    assert G.guard(n, nodes, F, r, bw * 4, p) == 0                    # faster network -> reject
    assert G.guard(n, nodes, F * 4, r, bw, p) == 0                    # higher fan-in -> reject
    assert G.guard(n, nodes, F, r / 4, bw, p) == 0                    # slower endpoint -> reject
    # the decision does not depend on the bucket size (every term is linear in n)
    assert G.guard(10 * n, nodes, F, r, bw, p) == G.guard(n, nodes, F, r, bw, p)
    # G-Binary halves the compact payload
    th2, _ = G.guard_times(n, nodes, F, r, bw, 2)
    th1, _ = G.guard_times(n, nodes, F, r, bw, 1)
    assert th1 == pytest.approx(th2 / 2)


@pytest.fixture(scope="module")
def nf():
    from paper_2606_25759_b200 import build, binding
    build.build()
    return binding


def test_library_mgtr_and_guard_match_oracle(nf):
    rng = np.random.default_rng(0)
    for _ in range(20):
        E = int(rng.integers(1, 200))
        numel = rng.integers(1, 10 ** 7, E)
        route = rng.integers(0, 3, E)
        mode = rng.integers(1, 3, E)
        ev = [(int(a), int(b), int(c)) for a, b, c in zip(numel, route, mode)]
        for sb in (0, 4):
            assert nf.nf_mgtr(numel, route, mode, scale_bytes=sb) == pytest.approx(G.mgtr(ev, scale_bytes=sb), rel=1e-12)
    assert nf.nf_mgtr([], [], []) == 1.0
    for _ in range(200):
        n = int(rng.integers(1, 10 ** 8)); nodes = int(rng.integers(2, 65)); F = int(rng.integers(1, 17))
        if nodes * F > 255:
            continue
        r = 10 ** rng.uniform(8, 13); bw = 10 ** rng.uniform(9, 12); p = int(rng.integers(1, 3))
        th, tf = G.guard_times(n, nodes, F, r, bw, p)
        if abs(th - tf) < 1e-9 * tf:
            continue
        adm, lt_h, lt_f = nf.nf_capacity_guard(n, nodes, F, r, bw, p)
        assert adm == G.guard(n, nodes, F, r, bw, p)
        assert lt_h == pytest.approx(th, rel=1e-12) and lt_f == pytest.approx(tf, rel=1e-12)
