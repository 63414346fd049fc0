"""Thin Python binding of libnf.so (include/nf.h): argument marshalling only.

Every function has the name and argument order of its C entry point and takes torch CUDA
tensors (or None for optional pointers); PyTorch is used for device memory and streams only.
There is NO CPU fallback: if libnf.so is missing or fails to load, the first call raises.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libnf.so")

NF_OK, NF_ERR_ARG, NF_ERR_ALIGN, NF_ERR_RANGE, NF_ERR_CUDA, NF_ERR_TOO_LARGE = 0, -1, -2, -3, -4, -5
NF_NOALLOC_WORKSPACE_BYTES = 16 << 20   # nf.h: the static scratch array behind nf_aggregate_bucket_noalloc
ROUTE_P, ROUTE_L, ROUTE_F = 0, 1, 2
MODE_GBINARY, MODE_GTERNARY = 1, 2
SUM_WD, SUM_NL, SUM_NF, SUM_NP, SUM_E, SUM_F, SUM_TILES, SUM_STATUS, SUM_LEN = range(9)

EXPORTS = ("nf_status_string", "nf_version", "nf_plan_bytes", "nf_workspace_bytes", "nf_route_bucket",
           "nf_sign_pack", "nf_sign_count_reduce", "nf_fp32_reduce", "nf_health_stats",
           "nf_aggregate_bucket", "nf_aggregate_bucket_host", "nf_aggregate_step", "nf_step_workspace_bytes", "nf_stock_packed_sign",
           "nf_count_planes", "nf_partial_count", "nf_partial_count_merge", "nf_supervisor_init",
           "nf_supervisor_step", "nf_mgtr", "nf_capacity_guard", "nf_debug_trace", "nf_aggregate_bucket_noalloc")


class NfState(C.Structure):
    _fields_ = [("admitted", C.c_int32), ("veto", C.c_int32), ("capacity_ok", C.c_int32)]


class NfSupervisorCfg(C.Structure):
    _fields_ = [("warmup_steps", C.c_int32), ("cooldown_steps", C.c_int32), ("guard_steps", C.c_int32),
                ("reserved", C.c_int32), ("ema_beta", C.c_double), ("slack", C.c_double), ("threshold", C.c_double)]


class NfSupervisor(C.Structure):
    _fields_ = [("cfg", NfSupervisorCfg), ("phase", C.c_int32), ("remaining", C.c_int32), ("step", C.c_int64),
                ("detections", C.c_int64), ("ema", C.c_double), ("cusum", C.c_double)]


class NfBucket(C.Structure):
    """struct nf_bucket of include/nf.h (one bucket of nf_aggregate_step)."""
    _fields_ = [("g", C.c_void_p), ("worker_stride", C.c_int64), ("n", C.c_int64), ("off", C.c_void_p),
                ("len", C.c_void_p), ("elig", C.c_void_p), ("T", C.c_int32), ("reserved", C.c_int32),
                ("tau", C.c_void_p), ("route", C.c_void_p), ("woff", C.c_void_p), ("summary", C.c_void_p),
                ("P", C.c_void_p), ("N", C.c_void_p), ("plane_stride", C.c_int64), ("abs_sum", C.c_void_p),
                ("sumsq", C.c_void_p), ("nan_cnt", C.c_void_p), ("inf_cnt", C.c_void_p), ("out", C.c_void_p),
                ("scale_out", C.c_void_p), ("plan", C.c_void_p), ("plan_bytes", C.c_size_t)]


class NfError(RuntimeError):
    def __init__(self, fn: str, status: int):
        self.status = status
        super().__init__(f"{fn}: {status_string(status)} ({status})")


_lib = None


def lib() -> C.CDLL:
    """Load libnf.so. Fails loudly: the product has no other implementation to fall back to."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_25759_b200.build` "
                           "(there is no CPU or PyTorch fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i64, i32, sz, f32 = C.c_void_p, C.c_int64, C.c_int, C.c_size_t, C.c_float
    L.nf_status_string.restype = C.c_char_p
    L.nf_status_string.argtypes = [i32]
    L.nf_version.restype = i32
    L.nf_plan_bytes.restype = sz
    L.nf_plan_bytes.argtypes = [i32, i32]
    L.nf_workspace_bytes.restype = sz
    L.nf_workspace_bytes.argtypes = [i32, i64]
    L.nf_route_bucket.restype = i32
    L.nf_route_bucket.argtypes = [vp, vp, vp, i32, i64, NfState, vp, vp, vp, vp, sz, vp]
    L.nf_sign_pack.restype = i32
    L.nf_sign_pack.argtypes = [vp, i64, i32, i64, vp, vp, vp, vp, i32, i32, vp, vp, vp, i64, vp, vp, vp]
    L.nf_sign_count_reduce.restype = i32
    L.nf_sign_count_reduce.argtypes = [vp, vp, i64, i32, i64, vp, vp, vp, vp, i32, i32, i32, vp,
                                       vp, vp, vp, vp, vp, vp]
    L.nf_fp32_reduce.restype = i32
    L.nf_fp32_reduce.argtypes = [vp, i64, i32, i64, vp, vp, vp, i32, f32, vp, vp, vp]
    L.nf_health_stats.restype = i32
    L.nf_health_stats.argtypes = [vp, i64, i32, i64, vp, vp, i32, vp, vp, vp, vp, vp]
    L.nf_aggregate_bucket.restype = i32
    L.nf_aggregate_bucket.argtypes = [vp, i64, i32, i64, vp, vp, vp, i32, NfState, i32, vp, i32, f32,
                                      vp, vp, vp, vp, vp, i64, vp, vp, vp, vp, vp, vp,
                                      vp, sz, vp, sz, vp]
    L.nf_aggregate_bucket_noalloc.restype = i32
    L.nf_aggregate_bucket_noalloc.argtypes = [vp, i64, i32, i64, vp, vp, vp, i32, NfState, i32, vp, i32, f32,
                                              vp, vp, vp, vp, vp, i64, vp, vp, vp, vp, vp, vp,
                                              vp, sz, vp]
    L.nf_aggregate_bucket_host.restype = i32
    L.nf_aggregate_bucket_host.argtypes = [vp, vp, i64, i32, i64, vp, vp, vp, i32, NfState, i32, vp, i32,
                                           f32, vp, vp, vp, vp, vp, i64, vp, vp, vp, vp, vp, vp,
                                           vp, sz, vp, sz, vp]
    L.nf_debug_trace.restype = i32
    L.nf_debug_trace.argtypes = [i32, vp]
    L.nf_step_workspace_bytes.restype = sz
    L.nf_step_workspace_bytes.argtypes = [C.POINTER(NfBucket), i32]
    L.nf_aggregate_step.restype = i32
    L.nf_aggregate_step.argtypes = [C.POINTER(NfBucket), i32, i32, NfState, i32, i32, f32, vp, sz, vp]
    L.nf_stock_packed_sign.restype = i32
    L.nf_stock_packed_sign.argtypes = [vp, vp, i64, i32, i64, vp, vp, vp, vp, i32, i32, i32, vp, vp, vp, vp, i64, vp, vp]
    L.nf_count_planes.restype = i32
    L.nf_count_planes.argtypes = [i32]
    L.nf_partial_count.restype = i32
    L.nf_partial_count.argtypes = [vp, vp, i64, i32, i64, i32, i32, vp, vp, i64, vp]
    L.nf_partial_count_merge.restype = i32
    L.nf_partial_count_merge.argtypes = [vp, vp, i64, i32, i32, i32, i64, vp, vp, vp, vp, i32, i32, i32, vp,
                                         vp, vp, vp, vp, vp, vp]
    L.nf_supervisor_init.restype = i32
    L.nf_supervisor_init.argtypes = [C.POINTER(NfSupervisor), C.POINTER(NfSupervisorCfg)]
    L.nf_supervisor_step.restype = i32
    L.nf_supervisor_step.argtypes = [C.POINTER(NfSupervisor), C.c_double, C.c_uint64, C.c_uint64, i32, C.POINTER(NfState)]
    L.nf_mgtr.restype = i32
    L.nf_mgtr.argtypes = [vp, vp, vp, i64, C.c_double, C.c_double, i32, C.POINTER(C.c_double)]
    L.nf_capacity_guard.restype = i32
    L.nf_capacity_guard.argtypes = [i64, i32, i32, C.c_double, C.c_double, i32, C.POINTER(C.c_double),
                                    C.POINTER(C.c_double)]
    _lib = L
    return L


def status_string(status: int) -> str:
    return lib().nf_status_string(int(status)).decode()


def _ptr(t: Optional[torch.Tensor], cuda: bool = True) -> Optional[int]:
    if t is None:
        return None
    if cuda and not t.is_cuda:
        raise TypeError("expected a CUDA tensor")
    if not t.is_contiguous():
        raise TypeError("expected a contiguous tensor")
    return t.data_ptr()


def _stream(stream) -> Optional[int]:
    if stream is None:
        return torch.cuda.current_stream().cuda_stream or None
    if isinstance(stream, torch.cuda.Stream):
        return stream.cuda_stream or None
    return int(stream) or None


def _state(state) -> NfState:
    if isinstance(state, NfState):
        return state
    a, v, c = state
    return NfState(int(a), int(v), int(c))


def _check(fn: str, rc: int):
    if rc != NF_OK:
        raise NfError(fn, rc)


def nf_plan_bytes(T: int, R: int = 1) -> int:
    return int(lib().nf_plan_bytes(int(T), int(R)))


def nf_workspace_bytes(T: int, n: int) -> int:
    return int(lib().nf_workspace_bytes(int(T), int(n)))


def nf_route_bucket(off, length, elig, T, n, state, route, woff, summary, plan, stream=None):
    _check("nf_route_bucket", lib().nf_route_bucket(
        _ptr(off), _ptr(length), _ptr(elig), int(T), int(n), _state(state), _ptr(route), _ptr(woff),
        _ptr(summary), _ptr(plan), plan.numel() * plan.element_size(), _stream(stream)))


def nf_sign_pack(g, worker_stride, W, n, off, length, route, woff, T, mode, tau, P, N, plane_stride,
                 abs_sum, plan, stream=None):
    _check("nf_sign_pack", lib().nf_sign_pack(
        _ptr(g), int(worker_stride), int(W), int(n), _ptr(off), _ptr(length), _ptr(route), _ptr(woff),
        int(T), int(mode), _ptr(tau), _ptr(P), _ptr(N), int(plane_stride), _ptr(abs_sum), _ptr(plan),
        _stream(stream)))


def nf_sign_count_reduce(P, N, plane_stride, W, n, off, length, route, woff, T, mode, margin, abs_sum,
                         out, cpos, cneg, scale_out, plan, stream=None):
    _check("nf_sign_count_reduce", lib().nf_sign_count_reduce(
        _ptr(P), _ptr(N), int(plane_stride), int(W), int(n), _ptr(off), _ptr(length), _ptr(route),
        _ptr(woff), int(T), int(mode), int(margin), _ptr(abs_sum), _ptr(out), _ptr(cpos), _ptr(cneg),
        _ptr(scale_out), _ptr(plan), _stream(stream)))


def nf_fp32_reduce(g, worker_stride, W, n, off, length, route, T, alpha, out, plan, stream=None):
    _check("nf_fp32_reduce", lib().nf_fp32_reduce(
        _ptr(g), int(worker_stride), int(W), int(n), _ptr(off), _ptr(length), _ptr(route), int(T),
        float(alpha), _ptr(out), _ptr(plan), _stream(stream)))


def nf_health_stats(x, replica_stride, R, n, off, length, T, sumsq, nan_cnt, inf_cnt, plan, stream=None):
    _check("nf_health_stats", lib().nf_health_stats(
        _ptr(x), int(replica_stride), int(R), int(n), _ptr(off), _ptr(length), int(T), _ptr(sumsq),
        _ptr(nan_cnt), _ptr(inf_cnt), _ptr(plan), _stream(stream)))


def nf_aggregate_bucket(g, worker_stride, W, n, off, length, elig, T, state, mode, tau, margin, alpha,
                        route, woff, summary, P, N, plane_stride, abs_sum, sumsq, nan_cnt, inf_cnt,
                        out, scale_out, plan, workspace, stream=None):
    _check("nf_aggregate_bucket", lib().nf_aggregate_bucket(
        _ptr(g), int(worker_stride), int(W), int(n), _ptr(off), _ptr(length), _ptr(elig), int(T),
        _state(state), int(mode), _ptr(tau), int(margin), float(alpha), _ptr(route), _ptr(woff),
        _ptr(summary), _ptr(P), _ptr(N), int(plane_stride), _ptr(abs_sum), _ptr(sumsq), _ptr(nan_cnt),
        _ptr(inf_cnt), _ptr(out), _ptr(scale_out), _ptr(plan), plan.numel() * plan.element_size(),
        _ptr(workspace), workspace.numel() * workspace.element_size(), _stream(stream)))


def nf_aggregate_bucket_noalloc(g, worker_stride, W, n, off, length, elig, T, state, mode, tau, margin, alpha,
                                route, woff, summary, P, N, plane_stride, abs_sum, sumsq, nan_cnt, inf_cnt,
                                out, scale_out, plan, stream=None):
    """nf_aggregate_bucket with the direction workspace in the library's static device array (nf.h): no buffer to
    pass, nothing allocated; buckets beyond NF_NOALLOC_WORKSPACE_BYTES of scratch raise NF_ERR_TOO_LARGE."""
    _check("nf_aggregate_bucket_noalloc", lib().nf_aggregate_bucket_noalloc(
        _ptr(g), int(worker_stride), int(W), int(n), _ptr(off), _ptr(length), _ptr(elig), int(T),
        _state(state), int(mode), _ptr(tau), int(margin), float(alpha), _ptr(route), _ptr(woff),
        _ptr(summary), _ptr(P), _ptr(N), int(plane_stride), _ptr(abs_sum), _ptr(sumsq), _ptr(nan_cnt),
        _ptr(inf_cnt), _ptr(out), _ptr(scale_out), _ptr(plan), plan.numel() * plan.element_size(), _stream(stream)))


def nf_aggregate_bucket_host(g_host, g_dev, worker_stride, W, n, off, length, elig, T, state, mode, tau,
                             margin, alpha, route, woff, summary, P, N, plane_stride, abs_sum, sumsq, nan_cnt,
                             inf_cnt, out, out_host, plan, workspace, stream=None):
    _check("nf_aggregate_bucket_host", lib().nf_aggregate_bucket_host(
        _ptr(g_host, cuda=False), _ptr(g_dev), int(worker_stride), int(W), int(n), _ptr(off),
        _ptr(length), _ptr(elig), int(T), _state(state), int(mode), _ptr(tau), int(margin), float(alpha),
        _ptr(route), _ptr(woff), _ptr(summary), _ptr(P), _ptr(N), int(plane_stride), _ptr(abs_sum), _ptr(sumsq),
        _ptr(nan_cnt), _ptr(inf_cnt), _ptr(out), _ptr(out_host, cuda=False), _ptr(plan), plan.numel() * plan.element_size(),
        _ptr(workspace), workspace.numel() * workspace.element_size(), _stream(stream)))


def nf_step_workspace_bytes(buckets) -> int:
    """buckets: a ctypes array of NfBucket."""
    return int(lib().nf_step_workspace_bytes(buckets, len(buckets)))


def nf_aggregate_step(buckets, W, state, mode, margin, alpha, workspace, stream=None):
    """buckets: a ctypes array of NfBucket (host memory, device pointers inside)."""
    _check("nf_aggregate_step", lib().nf_aggregate_step(
        buckets, len(buckets), int(W), _state(state), int(mode), int(margin), float(alpha), _ptr(workspace),
        workspace.numel() * workspace.element_size(), _stream(stream)))


def nf_stock_packed_sign(P, N, plane_stride, W, n, off, length, route, woff, T, mode, margin, abs_sum, recvP, recvN,
                         out, out_stride, plan, stream=None):
    _check("nf_stock_packed_sign", lib().nf_stock_packed_sign(
        _ptr(P), _ptr(N), int(plane_stride), int(W), int(n), _ptr(off), _ptr(length), _ptr(route), _ptr(woff), int(T),
        int(mode), int(margin), _ptr(abs_sum), _ptr(recvP), _ptr(recvN), _ptr(out), int(out_stride), _ptr(plan),
        _stream(stream)))


def nf_count_planes(Wg: int) -> int:
    B = lib().nf_count_planes(int(Wg))
    if B < 0:
        raise NfError("nf_count_planes", B)
    return B


def nf_partial_count(P, N, plane_stride, Wg, Wd, mode, B, cnt_pos, cnt_neg, count_stride, stream=None):
    _check("nf_partial_count", lib().nf_partial_count(
        _ptr(P), _ptr(N), int(plane_stride), int(Wg), int(Wd), int(mode), int(B), _ptr(cnt_pos), _ptr(cnt_neg),
        int(count_stride), _stream(stream)))


def nf_partial_count_merge(cnt_pos, cnt_neg, count_stride, G, B, W, n, off, length, route, woff, T, mode, margin,
                           abs_sum, out, cpos, cneg, scale_out, plan, stream=None):
    _check("nf_partial_count_merge", lib().nf_partial_count_merge(
        _ptr(cnt_pos), _ptr(cnt_neg), int(count_stride), int(G), int(B), int(W), int(n), _ptr(off), _ptr(length),
        _ptr(route), _ptr(woff), int(T), int(mode), int(margin), _ptr(abs_sum), _ptr(out), _ptr(cpos),
        _ptr(cneg), _ptr(scale_out), _ptr(plan), _stream(stream)))


def nf_mgtr(numel, route, mode, bits_binary=1.0, bits_ternary=1.584962500721156, scale_bytes=4) -> float:
    """Host call: MGTR of a route log."""
    import numpy as np
    a = np.ascontiguousarray(numel, dtype=np.int64)
    r = np.ascontiguousarray(route, dtype=np.uint8)
    m = np.ascontiguousarray(mode, dtype=np.uint8)
    out = C.c_double(0.0)
    _check("nf_mgtr", lib().nf_mgtr(a.ctypes.data, r.ctypes.data, m.ctypes.data, int(a.size), float(bits_binary),
                                    float(bits_ternary), int(scale_bytes), C.byref(out)))
    return out.value


def nf_capacity_guard(n, nodes, local_fan_in, service_rate, net_bw, planes):
    """Host call: (admit, t_hier, t_fp32) of the endpoint-capacity guard."""
    th, tf = C.c_double(0.0), C.c_double(0.0)
    rc = lib().nf_capacity_guard(int(n), int(nodes), int(local_fan_in), float(service_rate), float(net_bw),
                                 int(planes), C.byref(th), C.byref(tf))
    if rc < 0:
        raise NfError("nf_capacity_guard", rc)
    return rc, th.value, tf.value


class Supervisor:
    """Marshalling for nf_supervisor_init / nf_supervisor_step (host functions of libnf.so)."""

    def __init__(self, warmup_steps, ema_beta, slack, threshold, cooldown_steps, guard_steps):
        self._s = NfSupervisor()
        cfg = NfSupervisorCfg(int(warmup_steps), int(cooldown_steps), int(guard_steps), 0, float(ema_beta),
                              float(slack), float(threshold))
        _check("nf_supervisor_init", lib().nf_supervisor_init(C.byref(self._s), C.byref(cfg)))

    def step(self, signal, nan_count=0, inf_count=0, capacity_ok=1):
        st = NfState()
        _check("nf_supervisor_step", lib().nf_supervisor_step(C.byref(self._s), float(signal), int(nan_count),
                                                               int(inf_count), int(capacity_ok), C.byref(st)))
        return st.admitted, st.veto, st.capacity_ok

    phase = property(lambda self: self._s.phase)
    detections = property(lambda self: self._s.detections)
    cusum = property(lambda self: self._s.cusum)
    ema = property(lambda self: self._s.ema)


def nf_debug_trace(on: int, fetch: bool = False):
    """Debugging aid (single-threaded): per-CTA globaltimer stamps of the last two fused
    kernels, [2][256][16] uint64, or None."""
    import numpy as np
    buf = np.zeros(2 * 256 * 16, np.uint64) if fetch else None
    rc = lib().nf_debug_trace(int(on), buf.ctypes.data if fetch else None)
    if rc != NF_OK:
        raise NfError("nf_debug_trace", rc)
    return buf.reshape(2, 256, 16) if fetch else None
