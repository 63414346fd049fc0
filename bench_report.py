#!/usr/bin/env python
"""bench_report.py — the measurement tables of SURVEY.md §8(d) beyond bench.py's single JSON line.

    python bench_report.py [--out gpurun_out/report.md] [--quick]

Table 1: the five BASELINE.json configs (plus the paper's two local-count shapes)
through the fused call nf_aggregate_bucket: time per step, FP32-gradient GB/s (4*W*n/t),
elements/s, algorithmic bytes, % of the nominal and of the measured HBM peak.
Table 2: the reducer-capacity sweep (config 5): for W in {2, 8, 32, 64, 128} on one 25 MB
all-eligible bucket: (i) nf_sign_count_reduce alone on pre-packed planes, (ii) nf_sign_pack +
nf_sign_count_reduce, (iii) the fused call, (iv) nf_fp32_reduce on the same W x n — the paper's
"endpoint service rate vs fan-in" question measured on one B200.
Timing: median of CUDA-event-timed iterations after 3 warm-ups, inputs resident in HBM. Buckets
smaller than L2 are rotated over enough copies to exceed 126 MB (stated per row). Tables 2-4 time the
calls replayed from a CUDA graph (a call shorter than the ~15 us Python/ctypes needs to issue it is
otherwise host-bound); table 1 gives both the eager and the graph-replay time.
No oracle is used here (parity is the job of tests/); this only times the CUDA path.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

L2_BYTES = 126 * 2 ** 20
NOMINAL = 8000.0


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"])
    except Exception:
        return 6650.0


def time_fn(fn, iters, warmup=3, reps=1, graph=False):
    """Median over `iters` samples of the time of `reps` back-to-back calls, per call (ms). reps > 1 keeps the
    launch latency of a short call from being counted as its duration. graph=True captures the `reps` calls into
    a CUDA graph and times its replay: the calls then follow each other on the device without waiting for the
    host, which otherwise bounds calls shorter than the ~15 us Python/ctypes takes to issue one."""
    import torch
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    run = None
    if graph:
        side = torch.cuda.Stream()
        with torch.cuda.stream(side):          # the library's lazy one-time setup must not happen under capture
            fn()
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            for _ in range(reps):
                fn()
        g.replay()
        torch.cuda.synchronize()
        run = g.replay
    ts = []
    for _ in range(iters):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        if run is not None:
            run()
        else:
            for _ in range(reps):
                fn()
        e1.record()
        e1.synchronize()
        ts.append(e0.elapsed_time(e1) / reps)
    return statistics.median(ts)


def fused_bytes(cfg, planes=True, p=2):
    tot = 0
    for b in cfg.buckets:
        e, n = b.n_eligible, b.n
        tot += 4 * cfg.W * n + 4 * n + e // 2 + ((p * cfg.W * e) // 8 if planes else 0)
    return tot


def run_config(cfg, iters, dev):
    """Whole model per iteration: ONE nf_aggregate_step call over all buckets (the kernels of consecutive buckets
    chained by the library), and for comparison one nf_aggregate_bucket call per bucket; small models are
    replicated so that one iteration touches more than L2 (the step then runs over all copies)."""
    import torch
    from paper_2606_25759_b200 import ModelBuffers, binding as nf
    from workloads import gen
    in_bytes = sum(4 * cfg.W * b.n for b in cfg.buckets)
    copies = max(1, -(-2 * L2_BYTES // in_bytes)) if in_bytes < 2 * L2_BYTES else 1
    G, layouts = [], []
    for _ in range(copies):
        for b in cfg.buckets:
            G.append(gen.gen_bucket(cfg, b, dev))
            layouts.append((b.off, b.length, b.elig, b.n))
    mb = ModelBuffers(layouts, cfg.W, dev, planes=True, health=True)

    def step():
        mb.step(G, (1, 0, 1), nf.MODE_GTERNARY)

    def calls():
        for g, bb in zip(G, mb.buckets):
            bb.aggregate(g, g.shape[1], (1, 0, 1), nf.MODE_GTERNARY)
    ms = time_fn(step, iters) / copies
    ms_graph = time_fn(step, iters, graph=True) / copies
    ms_calls = time_fn(calls, iters, graph=True) / copies
    del G, mb
    torch.cuda.empty_cache()
    return ms, ms_graph, ms_calls, copies


def table_configs(args, dev, peak):
    from workloads import shapes
    names = ["tiny", "resnet50", "vit_b16", "gpt2_1p3b"] + [f"sweep_w{w}" for w in shapes.SWEEP_W]
    rows = []
    for nme in names:
        cfg = shapes.get(nme)
        ms, msg, msc, copies = run_config(cfg, args.iters if cfg.n_params < 5e8 else max(5, args.iters // 4), dev)
        rows.append((cfg.name, cfg.W, cfg.n_params, len(cfg.buckets), ms, msg, msc, copies, fused_bytes(cfg)))
    for n in (131_072, 524_288):
        cfg = shapes.paper_local_count(n)
        ms, msg, msc, copies = run_config(cfg, args.iters, dev)
        rows.append((cfg.name + " (PAPER L456 shape)", cfg.W, cfg.n_params, 1, ms, msg, msc, copies, fused_bytes(cfg)))
    out = ["| config | W | n (elements) | buckets | time / step (nf_aggregate_step, eager) | FP32-grad GB/s | elements/s | algorithmic bytes | "
           f"% of 8000 GB/s | % of {peak:.1f} GB/s | nf_aggregate_step replayed from a CUDA graph | one nf_aggregate_bucket call per bucket, "
           "graph replay | note |", "|---|---|---|---|---|---|---|---|---|---|---|---|---|"]
    for name, W, n, nb, ms, msg, msc, copies, ab in rows:
        t = ms * 1e-3
        note = f"{copies} rotating copies (input < 2 x L2), chained into one step" if copies > 1 else "input > L2"
        out.append(f"| {name} | {W} | {n:,} | {nb} | {ms * 1e3:.1f} us | {4 * W * n / t / 1e9:.1f} | {n / t:.3e} | "
                   f"{ab / 1e6:.1f} MB | {100 * ab / t / 1e9 / NOMINAL:.1f} | {100 * ab / t / 1e9 / peak:.1f} | "
                   f"{msg * 1e3:.1f} us, {100 * ab / (msg * 1e-3) / 1e9 / peak:.1f} % | "
                   f"{msc * 1e3:.1f} us, {100 * ab / (msc * 1e-3) / 1e9 / peak:.1f} % | {note} |")
    return "\n".join(out)


def table_sweep(args, dev, peak):
    import torch
    from paper_2606_25759_b200 import BucketBuffers, binding as nf
    from workloads import shapes, gen
    out = ["| W | planes in (MB) | (i) count-reduce alone | (ii) pack + count-reduce | (iii) fused | (iv) fp32_reduce | "
           "rotating copies (i) / (ii)-(iv) |", "|---|---|---|---|---|---|---|"]
    for W in ([args.sweep_w] if args.sweep_w else shapes.SWEEP_W):
        cfg = shapes.sweep(W)
        b = cfg.buckets[0]
        n = b.n
        in_bytes = 4 * W * n
        copies = max(1, -(-2 * L2_BYTES // in_bytes))
        G = [gen.gen_bucket(cfg, b, dev) for _ in range(copies)]
        BB = [BucketBuffers(b.off, b.length, b.elig, n, W, dev, planes=True, health=True) for _ in range(copies)]
        for g, bb in zip(G, BB):
            bb.route_bucket((1, 0, 1))
            bb.sign_pack(g, g.shape[1], nf.MODE_GTERNARY)
        plane_bytes = 2 * W * n // 8
        # (i) reads only the planes: its own rotating set, sized on the bytes a3 touches (planes + output)
        rcopies = max(1, -(-2 * L2_BYTES // (plane_bytes + 4 * n)))
        RB = BB[:rcopies] + [BucketBuffers(b.off, b.length, b.elig, n, W, dev, planes=True, health=False)
                             for _ in range(max(0, rcopies - copies))]
        for rb in RB[copies:]:
            rb.route_bucket((1, 0, 1))
            rb.sign_pack(G[0], G[0].shape[1], nf.MODE_GTERNARY)
        torch.cuda.synchronize()

        def reduce_only():
            for rb in RB:
                rb.sign_count_reduce(nf.MODE_GTERNARY)

        def pack_reduce():
            for g, bb in zip(G, BB):
                bb.sign_pack(g, g.shape[1], nf.MODE_GTERNARY)
                bb.sign_count_reduce(nf.MODE_GTERNARY)

        def fused():
            for g, bb in zip(G, BB):
                bb.aggregate(g, g.shape[1], (1, 0, 1), nf.MODE_GTERNARY)

        # (iv): the same bucket with every tensor on the FP32 route
        FB = [BucketBuffers(b.off, b.length, [0] * len(b.off), n, W, dev, planes=False, health=False) for _ in range(copies)]
        for fb in FB:
            fb.route_bucket((1, 0, 1))

        def fp32():
            for g, fb in zip(G, FB):
                fb.fp32_reduce(g, g.shape[1])
        cells = []
        for fn, own in ((reduce_only, plane_bytes + 4 * n), (pack_reduce, in_bytes + 2 * plane_bytes + 4 * n),
                        (fused, in_bytes + plane_bytes + n // 2 + 4 * n), (fp32, in_bytes + 4 * n)):
            ncp = rcopies if fn is reduce_only else copies
            t = time_fn(fn, args.iters, reps=max(1, 8 // ncp), graph=True) / ncp * 1e-3
            cells.append(f"{t * 1e6:.1f} us, {in_bytes / t / 1e9:.0f} GB/s FP32-equiv, {100 * own / t / 1e9 / peak:.0f} % HBM on own bytes")
        out.append(f"| {W} | {plane_bytes / 1e6:.1f} | " + " | ".join(cells) + f" | {rcopies} / {copies} |")
        del G, BB, FB, RB
        torch.cuda.empty_cache()
    return "\n".join(out)


def table_hier(args, dev, peak):
    """NEXT-1: node-local counting per group of W/G workers (level 1), merge of the G
    partial-count sets + decode (level 2), against the flat count-reduce over all W."""
    import torch
    from paper_2606_25759_b200 import BucketBuffers, binding as nf
    from workloads import shapes, gen
    out = ["| W | G (nodes) | workers/node | B planes | payload per node: packed signs -> partial counts | level 1 (one node) | "
           "level 2 merge + decode | flat count-reduce | NEXT-2: stock packed-sign (all-gather of the planes to W replicas + W local counts) | hierarchical, all nodes "
           "(G x level 1 + level 2) | NEXT-3: measured endpoint service rate | guard verdict at 12.5 / 50 / 400 GB/s per node |",
           "|---|---|---|---|---|---|---|---|---|---|---|---|"]
    for W, G in ((32, 4), (32, 8), (128, 4), (128, 8), (128, 16)):
        cfg = shapes.sweep(W)
        b = cfg.buckets[0]
        n = b.n
        g = gen.gen_bucket(cfg, b, dev)
        Wg = W // G
        B = nf.nf_count_planes(Wg)
        Wd = (n + 31) // 32
        cs = (Wd + 3) // 4 * 4
        # rotating sets of (planes, partial counts, output) so that every timed function streams from HBM, not L2
        per_copy = 2 * W * Wd * 4 + 2 * G * B * cs * 4 + 4 * n
        rc = max(1, -(-2 * L2_BYTES // per_copy))
        BBs, CPs, CNs = [], [], []
        for _ in range(rc):
            bb = BucketBuffers(b.off, b.length, b.elig, n, W, dev, planes=True, health=False)
            bb.route_bucket((1, 0, 1))
            bb.sign_pack(g, g.shape[1], nf.MODE_GTERNARY)
            BBs.append(bb)
            CPs.append(torch.zeros((G, B, cs), dtype=torch.int32, device=dev))
            CNs.append(torch.zeros((G, B, cs), dtype=torch.int32, device=dev))
        torch.cuda.synchronize()
        assert int(BBs[0].summary[nf.SUM_WD]) == Wd

        def node_counts(bb, cp, cn):      # level 1 of every node of one copy
            for gi in range(G):
                nf.nf_partial_count(bb.P[gi * Wg:], bb.N[gi * Wg:], bb.plane_stride, Wg, Wd, nf.MODE_GTERNARY, B, cp[gi], cn[gi], cs)

        def merge(bb, cp, cn):
            nf.nf_partial_count_merge(cp, cn, cs, G, B, W, n, bb.off, bb.len, bb.route, bb.woff, bb.T, nf.MODE_GTERNARY, 0,
                                      bb.abs_sum, bb.out, None, None, bb.scale, bb.plan)
        for bb, cp, cn in zip(BBs, CPs, CNs):
            node_counts(bb, cp, cn)

        def level1():     # rc x G node-local counts
            for bb, cp, cn in zip(BBs, CPs, CNs):
                node_counts(bb, cp, cn)

        def level2():
            for bb, cp, cn in zip(BBs, CPs, CNs):
                merge(bb, cp, cn)

        def flat():
            for bb in BBs:
                bb.sign_count_reduce(nf.MODE_GTERNARY)

        # NEXT-2: stock packed-sign transport: every worker receives all W sign streams (W gathered
        # copies of the planes, device-to-device) and counts them itself into its own output (nf_stock_packed_sign)
        bb0 = BBs[0]
        recvP = torch.empty((W, W, bb0.plane_stride), dtype=torch.int32, device=dev)
        recvN = torch.empty_like(recvP)
        ostride = (n + 3) // 4 * 4
        outs = torch.zeros((W, ostride), dtype=torch.float32, device=dev)

        def stock():
            nf.nf_stock_packed_sign(bb0.P, bb0.N, bb0.plane_stride, W, n, bb0.off, bb0.len, bb0.route, bb0.woff, bb0.T,
                                    nf.MODE_GTERNARY, 0, bb0.abs_sum, recvP, recvN, outs, ostride, bb0.plan)
        stock()
        merge(bb0, CPs[0], CNs[0])
        torch.cuda.synchronize()
        for r in range(W):      # every replica reconstructs the same aggregate, and it is the hierarchical path's
            assert torch.equal(outs[r, :n].view(torch.int32), bb0.out[:n].view(torch.int32)), f"replica {r} differs"
        gathered = 2 * W * W * Wd * 4

        def hier_all():   # all G nodes count locally, one merge + decode
            for bb, cp, cn in zip(BBs, CPs, CNs):
                node_counts(bb, cp, cn)
                merge(bb, cp, cn)
        t1, t2, t3, t4, t5 = (time_fn(f, args.iters if f is not stock else max(3, args.iters // 5), reps=1, graph=True) * 1e3 / div
                              for f, div in ((level1, rc * G), (level2, rc), (flat, rc), (stock, 1), (hier_all, rc)))
        packed, partial = 2 * Wg * Wd * 4, 2 * B * Wd * 4
        out.append(f"| {W} | {G} | {Wg} | {B} | {packed / 1e6:.1f} MB -> {partial / 1e6:.1f} MB | {t1:.1f} us | {t2:.1f} us | {t3:.1f} us | "
                   f"{t4:.0f} us ({gathered / 1e9:.2f} GB gathered, {W} outputs, all identical) | {t5:.1f} us | "
                   f"{packed / (t1 * 1e-6) / 1e9:.0f} GB/s | "
                   + " / ".join("admit" if nf.nf_capacity_guard(n, G, Wg, packed / (t1 * 1e-6), bw, 2)[0] else "FP32"
                                for bw in (12.5e9, 50e9, 400e9)) + " |")
        del g, bb, cp, cn, BBs, CPs, CNs, recvP, recvN, outs
        torch.cuda.empty_cache()
    return "\n".join(out)


def table_five_calls(args, dev, peak):
    """The five stand-alone calls of include/nf.h and the fused call on one GPT-2-1.3B-shaped bucket (bucket 0:
    33,568,768 elements, W = 8, all low-bit) and on its 401 MB FP32-route bucket: time and % of the measured HBM
    peak on each call's own algorithmic bytes; 8 back-to-back calls per sample."""
    import torch
    from paper_2606_25759_b200 import BucketBuffers, binding as nf
    from workloads import shapes, gen
    cfg = shapes.gpt2_1p3b()
    out = ["| bucket | call | time | own algorithmic bytes | % of measured HBM peak |", "|---|---|---|---|---|"]
    for bi in (0, 36):
        b = cfg.buckets[bi]
        W, n, e = cfg.W, b.n, b.n_eligible
        f = n - e
        g = gen.gen_bucket(cfg, b, dev)
        bb = BucketBuffers(b.off, b.length, b.elig, n, W, dev, planes=True, health=True)
        bb.aggregate(g, g.shape[1])
        torch.cuda.synchronize()
        planes = 2 * W * e // 8
        calls = [("nf_route_bucket (a1)", lambda: bb.route_bucket((1, 0, 1)), 0),
                 ("nf_sign_pack (a2)", lambda: bb.sign_pack(g, g.shape[1], nf.MODE_GTERNARY), 4 * W * e + planes),
                 ("nf_sign_count_reduce (a3)", lambda: bb.sign_count_reduce(nf.MODE_GTERNARY), planes + 4 * e),
                 ("nf_fp32_reduce (a4a)", lambda: bb.fp32_reduce(g, g.shape[1]), 4 * W * f + 4 * f),
                 ("nf_health_stats (a4b)", lambda: bb.health_stats(g, g.shape[1]), 4 * W * n),
                 ("nf_aggregate_bucket (fused)", lambda: bb.aggregate(g, g.shape[1]), 4 * W * n + planes + e // 2 + 4 * n)]
        for name, fn, own in calls:
            t = time_fn(fn, args.iters, reps=8, graph=True) * 1e-3
            pct = f"{100 * own / t / 1e9 / peak:.0f}" if own > 1e6 else "- (O(T) latency)"
            out.append(f"| {bi} (n = {n:,}, {100 * e / n:.0f} % low-bit) | {name} | {t * 1e6:.1f} us | {own / 1e6:.1f} MB | {pct} |")
        del g, bb
        torch.cuda.empty_cache()
    return "\n".join(out)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default="")
    ap.add_argument("--iters", type=int, default=20)
    ap.add_argument("--skip-configs", action="store_true")
    ap.add_argument("--only", default="", choices=["", "configs", "five", "sweep", "hier"],
                    help="print one table only (short runs under ncu: see profiles/)")
    ap.add_argument("--sweep-w", type=int, default=0, help="restrict the sweep table to one worker count")
    args = ap.parse_args()
    import torch
    from paper_2606_25759_b200 import build as nf_build
    nf_build.build()
    if not torch.cuda.is_available():
        raise SystemExit("bench_report.py needs a CUDA device (no CPU fallback)")
    dev = "cuda"
    peak = measured_peak()
    parts = [f"GPU: {torch.cuda.get_device_name(0)}; measured HBM copy peak {peak:.1f} GB/s; "
             f"median of {args.iters} CUDA-event-timed iterations after 3 warm-ups; mode G-Ternary, planes and health on. "
             "The stand-alone calls, the sweep and the hierarchical table are timed as replays of a CUDA graph holding the "
             "calls back to back (issued one by one from Python, a call shorter than ~15 us is host-bound); the config "
             "table gives both.", ""]
    want = lambda name: args.only in ("", name)
    if want("configs") and not args.skip_configs:
        parts += ["### Configs through nf_aggregate_bucket (route + fused kernel per bucket)", "", table_configs(args, dev, peak), ""]
    if want("five"):
        parts += ["### The five stand-alone calls and the fused call on GPT buckets 0 (all low-bit) and 36 (all FP32 route)", "",
                  table_five_calls(args, dev, peak), ""]
    if want("sweep"):
        parts += ["### Reducer-capacity sweep (config 5: one 25 MB all-eligible bucket, n = 6,553,600)", "", table_sweep(args, dev, peak), ""]
    if want("hier"):
        parts += ["### NEXT-1 / NEXT-2: two-level hierarchical sign count vs replicated counting of stock packed-sign transport, same bucket "
                  "(G-Ternary; results identical to the flat reduce; all work of all nodes / workers emulated on ONE GPU, no exchange; every cell rotates over enough copies of the planes, partial counts and output to stream from HBM)", "",
                  table_hier(args, dev, peak), ""]
    text = "\n".join(parts)
    print(text)
    if args.out:
        with open(args.out, "w") as f:
            f.write(text + "\n")


if __name__ == "__main__":
    main()
