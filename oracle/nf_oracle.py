"""ctypes front-end of the CPU oracle (oracle/nf_oracle.c). TEST INFRASTRUCTURE ONLY.

Argument marshalling only (numpy arrays <-> C pointers); every operation is the C function of
the same name, which cites the PAPER.md passage it follows. Nothing here imports the product
package, and the product package never imports this module.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass

import numpy as np

from . import build as _build

ROUTE_P, ROUTE_L, ROUTE_F = 0, 1, 2
MODE_GBINARY, MODE_GTERNARY = 1, 2

_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        for name in ("nfo_route_bucket", "nfo_sign_pack", "nfo_sign_count_reference",
                     "nfo_sign_count_reduce", "nfo_fp32_reduce", "nfo_health_stats", "nfo_count_planes",
                     "nfo_partial_count", "nfo_partial_count_merge"):
            getattr(_lib, name).restype = C.c_int
    return _lib


def _p(a, ctype):
    return None if a is None else a.ctypes.data_as(C.POINTER(ctype))


def _i64(a):
    return np.ascontiguousarray(a, dtype=np.int64)


def _check(rc: int, what: str):
    if rc != 0:
        raise ValueError(f"{what} failed with status {rc}")


@dataclass
class Route:
    route: np.ndarray      # [T] uint8
    woff: np.ndarray       # [T] int64, -1 if not L
    Wd: int
    nL: int
    nF: int
    nP: int
    e: int
    f: int


def route_bucket(off, length, elig, n, admitted=1, veto=0, capacity_ok=1) -> Route:
    off, length = _i64(off), _i64(length)
    elig = np.ascontiguousarray(elig, dtype=np.uint8)
    T = len(off)
    route = np.zeros(T, np.uint8)
    woff = np.zeros(T, np.int64)
    summary = np.zeros(6, np.int64)
    rc = lib().nfo_route_bucket(_p(off, C.c_int64), _p(length, C.c_int64), _p(elig, C.c_uint8),
                                C.c_int(T), C.c_int64(n), C.c_int(admitted), C.c_int(veto),
                                C.c_int(capacity_ok), _p(route, C.c_uint8), _p(woff, C.c_int64),
                                _p(summary, C.c_int64))
    _check(rc, "nfo_route_bucket")
    return Route(route, woff, *[int(v) for v in summary])


def _g2d(g):
    g = np.ascontiguousarray(g, dtype=np.float32)
    assert g.ndim == 2, "g must be [W][stride]"
    return g


def sign_pack(g, off, length, route, woff, mode, tau=None, Wd=None):
    """g: [W][stride] float32. Returns (P [W][Wd] u32, N or None, abs_sum [W][T] f64)."""
    g = _g2d(g)
    W, stride = g.shape
    off, length, woff = _i64(off), _i64(length), _i64(woff)
    route = np.ascontiguousarray(route, dtype=np.uint8)
    T = len(off)
    if Wd is None:
        Wd = int(sum((int(l) + 31) // 32 for l, r in zip(length, route) if r == ROUTE_L))
    ps = max(Wd, 1)
    P = np.zeros((W, ps), np.uint32)
    N = np.zeros((W, ps), np.uint32) if mode == MODE_GTERNARY else None
    A = np.zeros((W, T), np.float64)
    tau_a = None if tau is None else np.ascontiguousarray(tau, dtype=np.float32)
    rc = lib().nfo_sign_pack(_p(g, C.c_float), C.c_int64(stride), C.c_int(W), C.c_int64(stride),
                             _p(off, C.c_int64), _p(length, C.c_int64), _p(route, C.c_uint8),
                             _p(woff, C.c_int64), C.c_int(T), C.c_int(mode), _p(tau_a, C.c_float),
                             _p(P, C.c_uint32), _p(N, C.c_uint32), C.c_int64(ps), _p(A, C.c_double))
    _check(rc, "nfo_sign_pack")
    return P[:, :Wd], (None if N is None else N[:, :Wd]), A


def sign_count_reference(g, off, length, route, mode, tau=None):
    """Counts straight from the floats (paper's 'reference sign-count', L285). [n] uint8 each."""
    g = _g2d(g)
    W, stride = g.shape
    off, length = _i64(off), _i64(length)
    route = np.ascontiguousarray(route, dtype=np.uint8)
    cpos = np.zeros(stride, np.uint8)
    cneg = np.zeros(stride, np.uint8)
    tau_a = None if tau is None else np.ascontiguousarray(tau, dtype=np.float32)
    rc = lib().nfo_sign_count_reference(_p(g, C.c_float), C.c_int64(stride), C.c_int(W),
                                        C.c_int64(stride), _p(off, C.c_int64), _p(length, C.c_int64),
                                        _p(route, C.c_uint8), C.c_int(len(off)), C.c_int(mode),
                                        _p(tau_a, C.c_float), _p(cpos, C.c_uint8), _p(cneg, C.c_uint8))
    _check(rc, "nfo_sign_count_reference")
    return cpos, cneg


def sign_count_reduce(P, N, W, n, off, length, route, woff, mode, margin, abs_sum, out=None):
    """Returns (out [n] f32, cpos [n] u8, cneg [n] u8, scale [T] f32). `out` is updated in place
    at L positions when given (so the FP32 route can share the buffer)."""
    P = np.ascontiguousarray(P, dtype=np.uint32)
    assert P.ndim == 2 and P.shape[0] == W
    ps = P.shape[1]
    if N is not None:
        N = np.ascontiguousarray(N, dtype=np.uint32)
        assert N.shape == P.shape
    off, length, woff = _i64(off), _i64(length), _i64(woff)
    route = np.ascontiguousarray(route, dtype=np.uint8)
    T = len(off)
    A = np.ascontiguousarray(abs_sum, dtype=np.float64)
    assert A.shape == (W, T)
    if out is None:
        out = np.zeros(n, np.float32)
    assert out.dtype == np.float32 and out.flags.c_contiguous and out.shape == (n,)
    cpos = np.zeros(n, np.uint8)
    cneg = np.zeros(n, np.uint8)
    scale = np.zeros(T, np.float32)
    rc = lib().nfo_sign_count_reduce(_p(P, C.c_uint32), _p(N, C.c_uint32), C.c_int64(ps), C.c_int(W),
                                     C.c_int64(n), _p(off, C.c_int64), _p(length, C.c_int64),
                                     _p(route, C.c_uint8), _p(woff, C.c_int64), C.c_int(T),
                                     C.c_int(mode), C.c_int(margin), _p(A, C.c_double),
                                     _p(out, C.c_float), _p(cpos, C.c_uint8), _p(cneg, C.c_uint8),
                                     _p(scale, C.c_float))
    _check(rc, "nfo_sign_count_reduce")
    return out, cpos, cneg, scale


def count_planes(Wg: int) -> int:
    """NEXT-1: bit-planes of a partial count of Wg workers (smallest B with 2^B > Wg)."""
    return int(lib().nfo_count_planes(C.c_int(int(Wg))))


def partial_count(planes, B=None):
    """NEXT-1 level 1 (PAPER L243/L267 node-local counting): planes [Wg][Wd] uint32 of one group ->
    bit-sliced partial counts [B][Wd] uint32."""
    planes = np.ascontiguousarray(planes, dtype=np.uint32)
    Wg, Wd = planes.shape
    B = count_planes(Wg) if B is None else int(B)
    cnt = np.zeros((B, max(Wd, 1)), np.uint32)
    rc = lib().nfo_partial_count(_p(planes, C.c_uint32), C.c_int64(planes.shape[1]), C.c_int(Wg), C.c_int64(Wd),
                                 C.c_int(B), _p(cnt, C.c_uint32), C.c_int64(cnt.shape[1]))
    _check(rc, "nfo_partial_count")
    return cnt[:, :Wd]


def partial_count_merge(cnt_pos, cnt_neg, W, n, off, length, route, woff, mode, margin, abs_sum, out=None):
    """NEXT-1 level 2: cnt_pos/cnt_neg [G][B][Wd] uint32 (cnt_neg None for G-Binary) -> (out, cpos, cneg, scale)
    exactly as sign_count_reduce."""
    cnt_pos = np.ascontiguousarray(cnt_pos, dtype=np.uint32)
    G, B, cs = cnt_pos.shape
    if cnt_neg is not None:
        cnt_neg = np.ascontiguousarray(cnt_neg, dtype=np.uint32)
        assert cnt_neg.shape == cnt_pos.shape
    off, length, woff = _i64(off), _i64(length), _i64(woff)
    route = np.ascontiguousarray(route, dtype=np.uint8)
    T = len(off)
    A = np.ascontiguousarray(abs_sum, dtype=np.float64)
    assert A.shape == (W, T)
    if out is None:
        out = np.zeros(n, np.float32)
    cpos = np.zeros(n, np.uint8)
    cneg = np.zeros(n, np.uint8)
    scale = np.zeros(T, np.float32)
    rc = lib().nfo_partial_count_merge(_p(cnt_pos, C.c_uint32), _p(cnt_neg, C.c_uint32), C.c_int64(cs), C.c_int(G),
                                       C.c_int(B), C.c_int(W), C.c_int64(n), _p(off, C.c_int64),
                                       _p(length, C.c_int64), _p(route, C.c_uint8), _p(woff, C.c_int64),
                                       C.c_int(T), C.c_int(mode), C.c_int(margin), _p(A, C.c_double),
                                       _p(out, C.c_float), _p(cpos, C.c_uint8), _p(cneg, C.c_uint8),
                                       _p(scale, C.c_float))
    _check(rc, "nfo_partial_count_merge")
    return out, cpos, cneg, scale


def fp32_reduce(g, off, length, route, alpha=1.0, out=None):
    g = _g2d(g)
    W, stride = g.shape
    off, length = _i64(off), _i64(length)
    route = np.ascontiguousarray(route, dtype=np.uint8)
    if out is None:
        out = np.zeros(stride, np.float32)
    assert out.dtype == np.float32 and out.flags.c_contiguous
    rc = lib().nfo_fp32_reduce(_p(g, C.c_float), C.c_int64(stride), C.c_int(W), C.c_int64(stride),
                               _p(off, C.c_int64), _p(length, C.c_int64), _p(route, C.c_uint8),
                               C.c_int(len(off)), C.c_float(alpha), _p(out, C.c_float))
    _check(rc, "nfo_fp32_reduce")
    return out


def health_stats(x, off, length):
    """x: [R][stride] float32. Returns (sumsq [R][T] f64, nan [R][T] u64, inf [R][T] u64)."""
    x = _g2d(x)
    R, stride = x.shape
    off, length = _i64(off), _i64(length)
    T = len(off)
    Q = np.zeros((R, T), np.float64)
    cn = np.zeros((R, T), np.uint64)
    ci = np.zeros((R, T), np.uint64)
    rc = lib().nfo_health_stats(_p(x, C.c_float), C.c_int64(stride), C.c_int(R), C.c_int64(stride),
                                _p(off, C.c_int64), _p(length, C.c_int64), C.c_int(T),
                                _p(Q, C.c_double), _p(cn, C.c_uint64), _p(ci, C.c_uint64))
    _check(rc, "nfo_health_stats")
    return Q, cn, ci


@dataclass
class BucketResult:
    route: Route
    P: np.ndarray
    N: np.ndarray | None
    abs_sum: np.ndarray
    out: np.ndarray
    cpos: np.ndarray
    cneg: np.ndarray
    scale: np.ndarray
    sumsq: np.ndarray
    nan_cnt: np.ndarray
    inf_cnt: np.ndarray


def aggregate_bucket(g, off, length, elig, state=(1, 0, 1), mode=MODE_GTERNARY, tau=None,
                     margin=0, alpha=1.0) -> BucketResult:
    """The whole per-bucket path in the paper's order (§3.3): O1 -> O2 -> O3 -> O4a -> O4b."""
    g = _g2d(g)
    W, n = g.shape
    r = route_bucket(off, length, elig, n, *state)
    P, N, A = sign_pack(g, off, length, r.route, r.woff, mode, tau, r.Wd)
    out = np.zeros(n, np.float32)
    out, cpos, cneg, scale = sign_count_reduce(P, N, W, n, off, length, r.route, r.woff, mode,
                                               margin, A, out)
    fp32_reduce(g, off, length, r.route, alpha, out)
    Q, cn, ci = health_stats(g, off, length)
    return BucketResult(r, P, N, A, out, cpos, cneg, scale, Q, cn, ci)


def stock_packed_sign(P, N, W, n, off, length, route, woff, mode, margin, abs_sum):
    """NEXT-2, the stock packed-sign path ("packed-sign all-gather followed by local unpack-and-count",
    L267 "each worker receives sign streams and reconstructs the same count locally"), written out: every replica r
    gets its own copy of all W workers' planes (the all-gather) and runs O3 on it. Returns (out [W][n], gathered
    bytes). That the W results are equal is NOT assumed here: the tests check it."""
    outs = []
    gathered = 0
    for _ in range(W):
        rP = np.array(P, copy=True)
        rN = None if N is None else np.array(N, copy=True)
        gathered += rP.nbytes + (0 if rN is None else rN.nbytes)
        out, _, _, _ = sign_count_reduce(rP, rN, W, n, off, length, route, woff, mode, margin, abs_sum)
        outs.append(out)
    return np.stack(outs), gathered
