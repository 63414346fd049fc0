#!/usr/bin/env python
"""bench.py — throughput of the fused low-bit bucket-aggregation hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config NAME]

A "step" is one pass of the whole hot path (route + pack + sign-count + decode + FP32 route +
health statistics, i.e. nf_aggregate_bucket) over every DDP bucket of the workload, W emulated
workers resident in HBM. Default workload: BASELINE.json configs[3], the GPT-2-1.3B-shaped model
(W=8, 1.31 G params, 37 buckets, 42 GB of FP32 gradients) — the config the metric is quoted on.
Prints ONE JSON line. Metric: FP32-gradient input bytes consumed per second, 4*W*n/t, in GB/s.

N > 1 (torchrun): the path does not shard across GPUs in this build (BASELINE.json: one GPU, no
collectives): every rank runs an independent replica ("replicas only"),
value = N * per-replica bytes / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "bucket FP32-grad GB/s aggregated (W emulated workers, 1 B200), % HBM peak"
UNIT = "GB/s"
HBM_FALLBACK_GBS = 6650.0      # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
HBM_NOMINAL_GBS = 8000.0       # BASELINE.json "~8 TB/s peak"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="nf", choices=["nf", "reference"])
    ap.add_argument("--config", default="gpt2_1p3b")
    ap.add_argument("--small", action="store_true", help="scaled-down shapes (debug only; invalid as a bench number)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-planes", action="store_true", help="do not materialise the packed planes")
    ap.add_argument("--mode", default="ternary", choices=["ternary", "binary"])
    ap.add_argument("--max-buckets", type=int, default=0, help="profiling aid: only the first K buckets "
                    "(invalid as a bench number)")
    return ap.parse_args()


# ------------------------------------------------------------------------------------------------
def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy)"
    except Exception:
        return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic():
    """dram bytes per launch of the dominant kernel from the committed ncu --set full summary."""
    p = os.path.join(ROOT, "profiles", "roofline_traffic.json")
    try:
        with open(p) as f:
            return json.load(f)
    except Exception:
        return None


class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "20"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1]))
            except ValueError:
                continue
            for nme, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out = {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                   "samples": len(sm)}
        return out


def dist_setup(n_gpus):
    import torch
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        backend = "nccl" if torch.cuda.is_available() else "gloo"
        dist.init_process_group(backend=backend)
    return rank, world, local


def max_over_ranks(ms: float, world: int, device) -> float:
    """Barrier-bracketed timing is taken as the MAX over ranks (replicas run independently)."""
    if world <= 1:
        return ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def barrier(world):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


# ------------------------------------------------------------------------------------------------
def algorithmic_bytes(cfg, planes: bool, ternary: bool):
    """fused path moves 4*W*n (in) + 4*n (out) + e/4 + e/4 (2-bit directions written
    by pass A and read by pass B) + p*W*e/8 (planes, when materialised) bytes per bucket."""
    p = 2 if ternary else 1
    tot_in = tot_all = passA = 0
    for b in cfg.buckets:
        e, n = b.n_eligible, b.n
        f = n - e
        inp = 4 * cfg.W * n
        pl = (p * cfg.W * e) // 8 if planes else 0
        a = inp + pl + e // 4 + 4 * f          # pass A: read all, write planes + dirs + FP32-route out
        bb = e // 4 + 4 * e                    # pass B: read dirs, write low-bit out
        tot_in += inp
        passA += a
        tot_all += a + bb
    return tot_in, tot_all, passA


def run_nf(args):
    import torch
    from paper_2606_25759_b200 import ModelBuffers, binding as nf
    from paper_2606_25759_b200 import build as nf_build
    from workloads import shapes, gen

    rank, world, local = dist_setup(args.gpus)
    nf_build.build()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    cfg = shapes.get(args.config, small=args.small)
    if args.max_buckets > 0:
        cfg.buckets = cfg.buckets[:args.max_buckets]
    W = cfg.W
    ternary = args.mode == "ternary"
    mode = nf.MODE_GTERNARY if ternary else nf.MODE_GBINARY
    planes = not args.no_planes

    # ---- resident inputs: every bucket's [W][stride] gradients in HBM (42 GB for the GPT config); every
    # bucket owns its outputs, accumulators and packed planes (2.4 GB of planes for the GPT config: plane
    # bytes written in one step are never overwritten inside L2 before they reach HBM); the 2-bit direction
    # workspace (8.4 MB) is one buffer shared by all buckets, an L2-resident intermediate by design
    t0 = time.time()
    G = [gen.gen_bucket(cfg, b, dev) for b in cfg.buckets]
    MB = ModelBuffers([(b.off, b.length, b.elig, b.n) for b in cfg.buckets], W, dev, planes=planes, health=True)
    BB = MB.buckets
    torch.cuda.synchronize()
    gen_s = time.time() - t0
    stream = torch.cuda.current_stream()

    def step():
        MB.step(G, (1, 0, 1), mode, None, 0, 1.0)

    in_bytes, all_bytes, passA_bytes = algorithmic_bytes(cfg, planes, ternary)
    n_total = cfg.n_params

    sampler = ClockSampler(local) if rank == 0 else None
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    # ---- timed region: device-resident inputs (inputs are 42 GB >> 126 MB L2: no flush needed)
    barrier(world)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    torch.cuda.synchronize()
    barrier(world)
    ms = max_over_ranks(e0.elapsed_time(e1), world, dev)
    clocks = sampler.stop() if sampler else None
    ms_per_step = ms / args.steps
    value = world * in_bytes / (ms_per_step * 1e-3) / 1e9

    # ---- duration of the dominant kernel, measured live: one nf_aggregate_bucket call = one launch of
    # nf::fused_passA_kernel (every bucket here has <= 256 tensors), bracketed by CUDA events recorded on the
    # launching stream (torch's current stream, the one the call is enqueued on)
    nb = len(cfg.buckets)
    prof_steps = min(args.steps, 5)
    evs = [[(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(nb)]
           for _ in range(prof_steps)]
    for k in range(prof_steps):
        for i, (g, bb) in enumerate(zip(G, BB)):
            evs[k][i][0].record(stream)
            bb.aggregate(g, g.shape[1], (1, 0, 1), mode, None, 0, 1.0)
            evs[k][i][1].record(stream)
    torch.cuda.synchronize()
    fused_ms = sum(a.elapsed_time(b) for step_evs in evs for a, b in step_evs) / prof_steps
    launches_per_step = sum(1 if len(b.tensors) <= 256 else 2 for b in cfg.buckets)
    peak, peak_src = measured_peak()
    # dominant kernel: nf::fused_passA_kernel = pass A + pass B of one bucket in one launch, so its
    # algorithmic bytes are the whole path's (SURVEY 8(d) "fused floor" + planes)
    # Inside a step the kernels of consecutive buckets overlap (the tail of bucket k is drained by the kernel of
    # bucket k+1), so the kernel's average duration in the timed region is the step time over the launches: the
    # timed region contains nothing but these launches, on the stream the CUDA events were recorded on.
    achieved = all_bytes / (ms_per_step * 1e-3) / 1e9
    traffic = ncu_traffic()
    roofline = {"bound": "hbm", "kernel": "nf::fused_passA_kernel (pass A + pass B of one bucket, TMA ring)",
                "achieved": round(achieved, 1), "peak": peak, "unit": "GB/s",
                "frac": round(achieved / peak, 4), "peak_source": peak_src,
                "frac_of_nominal_8TBs": round(achieved / HBM_NOMINAL_GBS, 4),
                "algorithmic_bytes_per_step": all_bytes, "launches_per_step": nb,
                "avg_launch_ms": round(ms_per_step / nb, 4),
                "avg_launch_ms_unchained": round(fused_ms / nb, 4),
                "traffic": (traffic or {}).get("dram_bytes_per_launch_avg"),
                "traffic_note": (traffic or {}).get("note"),
                "whole_path": {"algorithmic_bytes_per_step": all_bytes,
                               "achieved": round(all_bytes / (ms_per_step * 1e-3) / 1e9, 1),
                               "frac": round(all_bytes / (ms_per_step * 1e-3) / 1e9 / peak, 4)},
                "kernel_ms_per_step": {"fused_in_step": round(ms_per_step, 4), "fused_unchained_sum": round(fused_ms, 4)},
                "note": "avg_launch_ms = timed region (CUDA events on the launching stream) / launches: the step is "
                        "nothing but these launches. avg_launch_ms_unchained = the same kernel as stand-alone "
                        "nf_aggregate_bucket calls, one CUDA event pair per launch (no overlap between buckets)"}

    # ---- e2e: same metric through the C-ABI call with HOST buffers (H2D + D2H inside the region)
    e2e = None
    if not args.no_e2e:
        e2e = run_e2e(args, cfg, BB, mode, dev, world)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(cfg, G, budget_s=20.0)

    if rank == 0:
        line = {"metric": METRIC, "value": round(value, 1), "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": round(ms_per_step, 4),
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
                "data": "synthetic", "impl": "nf",
                "config": {"workload": f"{cfg.name}: W={W} emulated workers, {cfg.n_params} FP32 params, "
                                       f"{nb} DDP buckets, {cfg.n_tensors} tensors, mode=G-"
                                       f"{'Ternary' if ternary else 'Binary'}, planes={'on' if planes else 'off'}",
                           "W": W, "n_params": n_total, "buckets": nb, "input_bytes_per_step": in_bytes,
                           "l2": "inputs (42 GB) are larger than L2 (126 MB); no flush",
                           "parallelism": "replicas only" if world > 1 else "single GPU",
                           "small": bool(args.small), "max_buckets": args.max_buckets},
                "elements_per_s": round(world * n_total / (ms_per_step * 1e-3), 1),
                "input_elements_per_s": round(world * n_total * W / (ms_per_step * 1e-3), 1),
                "pct_hbm_peak_measured": round(100 * all_bytes / (ms_per_step * 1e-3) / 1e9 / peak, 2),
                "pct_hbm_peak_nominal_8TBs": round(100 * all_bytes / (ms_per_step * 1e-3) / 1e9 / HBM_NOMINAL_GBS, 2),
                "gpu_launches": args.steps * launches_per_step,
                "roofline": roofline, "clocks": clocks, "e2e": e2e, "cpu_baseline": cpu,
                "setup_s": round(gen_s, 1)}
        print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def run_e2e(args, cfg, BB, mode, dev, world):
    """nf_aggregate_bucket_host per bucket: H2D of the bucket's W x n floats from pinned host memory,
    the fused path, D2H of the n aggregated floats. Buckets alternate between two CUDA streams, each
    with its own device staging buffer, workspace and pinned result buffer, so that the H2D copy of
    bucket k+1 overlaps the kernels and the D2H copy of bucket k (two copy engines, full duplex).
    The pinned source holds one bucket's worth of gradients (the largest), read by every bucket: the
    bytes cross PCIe every step."""
    import torch
    from paper_2606_25759_b200 import binding as nf
    W = cfg.W
    max_stride = max((b.n + 3) // 4 * 4 for b in cfg.buckets)
    g_host = torch.empty(W * max_stride, dtype=torch.float32, pin_memory=True)
    slots = []
    for _ in range(2):
        g_dev = torch.empty(W * max_stride, dtype=torch.float32, device=dev)
        g_dev.normal_(0.0, 1e-3)
        ws = torch.zeros_like(BB[0].workspace) if BB[0].workspace is not None else None
        slots.append({"g_dev": g_dev, "out_host": torch.empty(max_stride, dtype=torch.float32, pin_memory=True),
                      "ws": ws, "stream": torch.cuda.Stream(device=dev)})
    g_host.copy_(slots[0]["g_dev"])
    torch.cuda.synchronize()
    main = torch.cuda.current_stream()
    steps = max(1, min(args.steps, 2))

    def step():
        for i, (b, bb) in enumerate(zip(cfg.buckets, BB)):
            sl = slots[i & 1]
            s = (b.n + 3) // 4 * 4
            nf.nf_aggregate_bucket_host(g_host, sl["g_dev"], s, W, b.n, bb.off, bb.len, bb.elig, bb.T, (1, 0, 1),
                                        mode, None, 0, 1.0, bb.route, bb.woff, bb.summary, bb.P,
                                        bb.N if mode == nf.MODE_GTERNARY else None, bb.plane_stride, bb.abs_sum,
                                        bb.sumsq, bb.nan_cnt, bb.inf_cnt, bb.out, sl["out_host"], bb.plan,
                                        sl["ws"], sl["stream"])
    step()
    torch.cuda.synchronize()
    barrier(world)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(main)
    for sl in slots:
        sl["stream"].wait_stream(main)                  # both streams start after e0
    for _ in range(steps):
        step()
    for sl in slots:
        main.wait_stream(sl["stream"])                  # e1 fires after both streams drained
    e1.record(main)
    torch.cuda.synchronize()
    barrier(world)
    ms = max_over_ranks(e0.elapsed_time(e1), world, dev) / steps
    h2d = sum(4 * ((W - 1) * ((b.n + 3) // 4 * 4) + b.n) for b in cfg.buckets)
    d2h = sum(4 * b.n for b in cfg.buckets)
    in_bytes = sum(4 * W * b.n for b in cfg.buckets)
    del slots, g_host
    return {"value": round(world * in_bytes / (ms * 1e-3) / 1e9, 2), "unit": UNIT,
            "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "ms_per_step": round(ms, 2),
            "steps": steps, "api": "nf_aggregate_bucket_host (pinned host buffers, cudaMemcpyAsync; same mode, planes "
                                   "and health outputs as the device-resident leg), buckets alternating between two "
                                   "streams; PCIe-bound"}


def cpu_baseline(cfg, G, budget_s=20.0):
    """The oracle as it stands, single-threaded, on a bounded sample of the same workload: whole
    buckets in order until ~budget_s of CPU work. Input values are the device-resident ones."""
    from oracle import nf_oracle as O
    done_bytes, t_total, used, last = 0, 0.0, [], 0.0
    for b, g in zip(cfg.buckets, G):
        if used and t_total + last > budget_s:
            break
        if b.n * cfg.W > 600_000_000:            # keep the host copy of one bucket under ~2.4 GB
            continue
        gh = g.cpu().numpy()[:, :b.n].copy()
        t0 = time.perf_counter()
        O.aggregate_bucket(gh, b.off, b.length, b.elig, (1, 0, 1), O.MODE_GTERNARY)
        last = time.perf_counter() - t0
        t_total += last
        done_bytes += 4 * cfg.W * b.n
        used.append(b.index)
        del gh
    if not used:
        return None
    out = {"value": round(done_bytes / t_total / 1e9, 4), "unit": UNIT, "cores": 1, "kind": "oracle",
           "sample": f"buckets {used} of {cfg.name} ({done_bytes / 1e9:.2f} GB of FP32 gradient input, "
                     f"{t_total:.1f} s single-threaded, host has {os.cpu_count()} cores)"}
    # the same (unchanged, single-threaded) oracle on all host cores at once: one bucket per thread, the C calls run
    # outside the GIL; reported beside the 1-core figure, never as the target
    try:
        from concurrent.futures import ThreadPoolExecutor
        nthr = max(1, min(os.cpu_count() or 1, len(used), 16))
        todo = [(b, g.cpu().numpy()[:, :b.n].copy()) for b, g in zip(cfg.buckets, G) if b.index in used[:nthr]]
        t0 = time.perf_counter()
        with ThreadPoolExecutor(max_workers=nthr) as ex:
            list(ex.map(lambda bg: O.aggregate_bucket(bg[1], bg[0].off, bg[0].length, bg[0].elig, (1, 0, 1),
                                                      O.MODE_GTERNARY) and None, todo))
        dt = time.perf_counter() - t0
        nb = sum(4 * cfg.W * b.n for b, _ in todo)
        out["all_cores"] = {"value": round(nb / dt / 1e9, 4), "unit": UNIT, "cores": nthr,
                            "sample": f"buckets {[b.index for b, _ in todo]} concurrently, one oracle call per thread "
                                      f"({nb / 1e9:.2f} GB in {dt:.1f} s)"}
    except Exception as e:                                   # the 1-core figure stands on its own
        out["all_cores"] = {"error": str(e)[:200]}
    return out


def run_reference(args):
    """--impl reference: the CPU oracle (oracle/), as it stands, on a bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import numpy as np
    import torch
    from oracle import nf_oracle as O
    from workloads import shapes, gen
    cfg = shapes.get(args.config, small=args.small)
    # bounded sample: the first bucket of the workload (GPT config: bucket 0, 33.6 M elements x W = 8, two 16.8 M
    # low-bit weight matrices + biases / LayerNorm on the FP32 route, no injected NaN: a clean, typical bucket)
    b = cfg.buckets[0]
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    gh = gen.gen_bucket(cfg, b, dev).cpu().numpy()[:, :b.n].copy()
    in_bytes = 4 * cfg.W * b.n

    def step():
        O.aggregate_bucket(gh, b.off, b.length, b.elig, (1, 0, 1), O.MODE_GTERNARY)
    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = (time.perf_counter() - t0) / args.steps
    val = round(in_bytes / dt / 1e9, 4)
    sample = (f"bucket {b.index} of {cfg.name} per step ({in_bytes / 1e9:.2f} GB of FP32 gradient input, "
              f"{b.n} elements x W={cfg.W}, no injected NaN); single-threaded C oracle; host has {os.cpu_count()} cores")
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT,
                      "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
                      "ms_per_step": round(dt * 1e3, 2), "higher_is_better": True, "scaling": "weak",
                      "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                      "config": {"workload": f"{cfg.name}: W={cfg.W}, bounded sample = {sample}"},
                      "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
                      "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                      "gpu_launches": 0}))


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_nf(a)
