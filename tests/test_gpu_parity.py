"""`-m gpu` parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by
element on the same seeded inputs. Sizes span several tiles (tile = 2048 elements) and ragged
tails; full-size configs are in test_gpu_fullsize.py."""
import numpy as np
import pytest
import torch

from oracle import nf_oracle as O
from paper_2606_25759_b200 import BucketBuffers, binding as nf
from tests.parity import run_both, compare, _np
from tests.util import read_golden, layout
from workloads import shapes, gen

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _dev(g_np, pad_to4=True):
    W, n = g_np.shape
    s = (n + 3) // 4 * 4 if pad_to4 else n
    g = torch.zeros((W, max(s, 4)), dtype=torch.float32, device=DEV)
    g[:, :n] = torch.from_numpy(g_np)
    return g


def test_handworked_bucket_on_gpu():
    d = read_golden("handworked_w4.txt")
    W = int(d["W"][0])
    off, ln, n = layout([int(x) for x in d["len"]])
    elig = [int(x) for x in d["elig"]]
    g = np.array([[float(x) for x in d[f"g{w}"]] for w in range(W)], np.float32)
    for mode, dkey in ((O.MODE_GTERNARY, "d_ternary"), (O.MODE_GBINARY, "d_binary")):
        ref = run_both(_dev(g), off, ln, elig, mode=mode, what="handworked")
        S = np.float32(float(d["scale"][0]))
        assert np.array_equal(ref.out[:8], np.array([S * int(x) for x in d[dkey]], np.float32))


@pytest.mark.parametrize("W", [1, 2, 3, 4, 8, 9, 17, 32, 33, 64, 100, 255])     # (records of 32 workers: whole, one over, ragged)
@pytest.mark.parametrize("mode", [O.MODE_GBINARY, O.MODE_GTERNARY])
def test_adversarial_lengths_and_offsets(W, mode):
    """Lengths 1, 31, 32, 33, 4099, a multi-tile tensor, offsets that are not multiples of 4,
    gaps between tensors, -0.0, denormals, +-Inf, a tensor that is entirely NaN."""
    rng = np.random.default_rng(1000 + W)
    lens = [1, 31, 32, 33, 4099, 2048 * 3 + 5, 7, 2048, 64]
    off, o = [], 3                                            # first tensor starts at 3: misaligned
    for i, l in enumerate(lens):
        off.append(o)
        o += l + (2 if i % 3 == 0 else 0)                     # gaps
    n = o + 1
    off, ln = np.array(off, np.int64), np.array(lens, np.int64)
    elig = [1, 1, 0, 1, 1, 1, 0, 1, 1]
    g = (rng.standard_normal((W, n)) * 10 ** rng.uniform(-6, 2, (1, n))).astype(np.float32)
    g[rng.random((W, n)) < 0.1] = 0.0
    g[0, off[4] + 5] = -0.0
    g[W - 1, off[4] + 6] = 1e-42                              # denormal
    g[0, off[5] + 100] = np.inf
    g[W - 1, off[5] + 101] = -np.inf
    g[:, off[8]:off[8] + 64] = np.nan                         # tensor entirely NaN
    g[0, off[2] + 3] = np.nan                                 # NaN on the FP32 route
    tau = (rng.random(len(lens)) * 1e-3).astype(np.float32)
    gd = _dev(g)
    run_both(gd, off, ln, elig, mode=mode, what=f"adv W={W}")
    run_both(gd, off, ln, elig, mode=mode, tau=tau, margin=1, alpha=1.0 / W, what=f"adv tau W={W}")


@pytest.mark.parametrize("state", [(0, 0, 1), (1, 1, 1), (1, 0, 0), (1, 0, 1)])
def test_three_state_preflight(state):
    """warm-up / admitted / forced veto (and guard reject) over the same binding."""
    cfg = shapes.tiny()
    b = cfg.buckets[0]
    g = gen.gen_bucket(cfg, b, DEV)
    ref = run_both(g, b.off, b.length, b.elig, state=state, what=f"tiny state={state}")
    if state != (1, 0, 1):
        plain = O.fp32_reduce(_np(g)[:, :b.n].copy(), b.off, b.length, np.zeros(len(b.off), np.uint8))
        assert np.array_equal(ref.out, plain)


def test_no_L_and_no_P_buckets_and_empty():
    rng = np.random.default_rng(5)
    off, ln, n = layout([5000, 333])
    g = _dev(rng.standard_normal((4, n)).astype(np.float32))
    run_both(g, off, ln, [0, 0], what="zero L")
    run_both(g, off, ln, [1, 1], what="zero P")
    # zero-length tensor in the middle, and T = 0
    off2, ln2 = np.array([0, 100, 100], np.int64), np.array([100, 0, 200], np.int64)
    run_both(g, off2, ln2, [1, 1, 0], what="empty tensor")
    bb = BucketBuffers([], [], [], 0, 4, DEV)
    bb.aggregate(g, g.shape[1])
    torch.cuda.synchronize()
    assert int(bb.summary[nf.SUM_STATUS]) == 0 and int(bb.summary[nf.SUM_WD]) == 0


def test_bad_layout_is_flagged_on_device_and_nothing_runs():
    g = torch.ones((2, 64), device=DEV)
    bb = BucketBuffers([0, 8], [16, 8], [1, 1], 32, 2, DEV)   # overlap
    bb.out.fill_(5.0)
    bb.aggregate(g, 64)
    torch.cuda.synchronize()
    assert int(bb.summary[nf.SUM_STATUS]) == nf.NF_ERR_ARG
    assert bool((bb.out == 5.0).all())


@pytest.mark.parametrize("name", ["tiny", "resnet50", "vit_b16", "gpt2_1p3b", "sweep_w2", "sweep_w32", "sweep_w128"])
def test_config_shapes_small(name):
    """The five BASELINE configs, structurally identical but scaled down (tiny is full size)."""
    cfg = shapes.get(name, small=True)
    for b in cfg.buckets:
        g = gen.gen_bucket(cfg, b, DEV)
        ref = run_both(g, b.off, b.length, b.elig, what=f"{cfg.name} bucket {b.index}")
        if cfg.nan_frac and b.index == cfg.nan_bucket:
            assert ref.nan_cnt[cfg.nan_worker].sum() > 0 and ref.nan_cnt.sum() == ref.nan_cnt[cfg.nan_worker].sum()


def test_gpu_invariants_without_oracle():
    """Properties that hold at any size, checked on the GPU's own outputs."""
    cfg = shapes.tiny()
    b = cfg.buckets[0]
    g = gen.gen_bucket(cfg, b, DEV)
    bb = BucketBuffers(b.off, b.length, b.elig, b.n, cfg.W, DEV, counts=True)
    bb.route_bucket((1, 0, 1))
    bb.sign_pack(g, g.shape[1], nf.MODE_GTERNARY)
    bb.sign_count_reduce(nf.MODE_GTERNARY)
    torch.cuda.synchronize()
    assert not bool((bb.P & bb.N).any())
    cz = cfg.W - bb.cpos.to(torch.int32) - bb.cneg.to(torch.int32)
    assert int(cz.min()) >= 0
    # permuting workers leaves counts unchanged
    cp0 = bb.cpos.clone()
    g2 = g[torch.tensor([2, 0, 3, 1], device=DEV)].contiguous()
    bb.sign_pack(g2, g2.shape[1], nf.MODE_GTERNARY)
    bb.sign_count_reduce(nf.MODE_GTERNARY)
    torch.cuda.synchronize()
    assert torch.equal(cp0, bb.cpos)


@pytest.mark.parametrize("name", ["tiny", "sweep_w8", "sweep_w32", "resnet50"])
@pytest.mark.parametrize("mode", [O.MODE_GBINARY, O.MODE_GTERNARY])
def test_count_reduce_without_count_outputs(name, mode):
    """nf_sign_count_reduce with cpos/cneg == NULL takes its own write-back path (1024-element runs of one
    tensor through the direction table); the count-output variant is covered by run_both."""
    cfg = shapes.get(name, small=(name != "tiny"))
    for b in cfg.buckets:
        g = gen.gen_bucket(cfg, b, DEV)
        ref = O.aggregate_bucket(np.ascontiguousarray(_np(g)[:, :b.n]), b.off, b.length, b.elig, (1, 0, 1), mode)
        bb = BucketBuffers(b.off, b.length, b.elig, b.n, cfg.W, DEV, planes=True, counts=False, health=True)
        bb.out.fill_(-77.0)
        bb.route_bucket((1, 0, 1))
        bb.sign_pack(g, g.shape[1], mode)
        bb.sign_count_reduce(mode)
        bb.fp32_reduce(g, g.shape[1])
        bb.health_stats(g, g.shape[1])
        compare(bb, ref, cfg.W, mode, check_counts=False, what=f"{cfg.name} bucket {b.index} 5-call, no counts")


@pytest.mark.parametrize("stride_pad", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("counts", [False, True])
@pytest.mark.parametrize("name,mode", [("tiny", O.MODE_GTERNARY), ("sweep_w32", O.MODE_GBINARY), ("vit_b16", O.MODE_GTERNARY)])
def test_count_reduce_both_kernels(name, mode, counts, stride_pad):
    """nf_sign_count_reduce has two kernels: the bulk-copy ring (plane rows 16-byte aligned, i.e. plane_stride a
    multiple of 4 words) and the register-staged one (any plane_stride). Both must give the oracle's result, with
    and without count outputs; the ring's last unit copies whole 16-byte chunks up to the row's end."""
    cfg = shapes.get(name, small=(name != "tiny"))
    for b in cfg.buckets:
        g = gen.gen_bucket(cfg, b, DEV)
        ref = O.aggregate_bucket(np.ascontiguousarray(_np(g)[:, :b.n]), b.off, b.length, b.elig, (1, 0, 1), mode)
        Wd = sum((int(l) + 31) // 32 for l, e in zip(b.length, b.elig) if e)
        ps = (Wd + 3) // 4 * 4 + stride_pad
        bb = BucketBuffers(b.off, b.length, b.elig, b.n, cfg.W, DEV, planes=True, counts=counts, health=True,
                           plane_stride=ps)
        assert bb.plane_stride == max(ps, 4)
        bb.out.fill_(-77.0)
        bb.route_bucket((1, 0, 1))
        bb.sign_pack(g, g.shape[1], mode)
        bb.sign_count_reduce(mode)
        bb.fp32_reduce(g, g.shape[1])
        bb.health_stats(g, g.shape[1])
        compare(bb, ref, cfg.W, mode, check_counts=counts,
                what=f"{cfg.name} bucket {b.index} plane_stride {bb.plane_stride} counts {counts}")


@pytest.mark.parametrize("T", [256, 257, 700])
def test_many_tensor_buckets(T):
    """Buckets around and above the fused kernel's shared-memory metadata capacity (256 tensors): T <= 256 routes
    inside the fused kernel, larger T goes through the route kernel and global-memory lookups."""
    rng = np.random.default_rng(T)
    lens = [int(x) for x in rng.integers(1, 3000, T)]
    lens[5] = 2048 * 3            # a few multi-tile tensors
    lens[T // 2] = 2048 * 2 + 17
    off, ln, n = layout(lens)
    elig = [int(x) for x in rng.integers(0, 2, T)]
    W = 5
    g = (rng.standard_normal((W, n)) * 10 ** rng.uniform(-4, 0, (1, n))).astype(np.float32)
    g[rng.random((W, n)) < 0.05] = 0.0
    run_both(_dev(g), off, ln, elig, what=f"T={T}")


def test_host_buffer_entry_point_matches_oracle():
    """nf_aggregate_bucket_host (the call bench.py's e2e leg times): pinned host gradients in, aggregated bucket
    back in pinned host memory, same values as the oracle."""
    cfg = shapes.tiny()
    b = cfg.buckets[0]
    g_dev_src = gen.gen_bucket(cfg, b, DEV)
    stride = g_dev_src.shape[1]
    g_host = torch.empty((cfg.W, stride), dtype=torch.float32, pin_memory=True)
    g_host.copy_(g_dev_src)
    ref = O.aggregate_bucket(np.ascontiguousarray(g_host.numpy()[:, :b.n]), b.off, b.length, b.elig)
    bb = BucketBuffers(b.off, b.length, b.elig, b.n, cfg.W, DEV, planes=True, health=True)
    staging = torch.zeros((cfg.W, stride), dtype=torch.float32, device=DEV)
    out_host = torch.full((b.n,), -3.0, dtype=torch.float32).pin_memory()
    nf.nf_aggregate_bucket_host(g_host, staging, stride, cfg.W, b.n, bb.off, bb.len, bb.elig, bb.T, (1, 0, 1),
                                nf.MODE_GTERNARY, None, 0, 1.0, bb.route, bb.woff, bb.summary, bb.P, bb.N,
                                bb.plane_stride, bb.abs_sum, bb.sumsq, bb.nan_cnt, bb.inf_cnt, bb.out, out_host, bb.plan,
                                bb.workspace)
    torch.cuda.synchronize()
    compare(bb, ref, cfg.W, O.MODE_GTERNARY, check_scale=False,      # the host call has no scale_out
            what="host entry point")
    assert np.array_equal(out_host.numpy(), _np(bb.out)[:b.n])
    # rows `stride` apart with a host / staging buffer that ends with the last row (the copy must not
    # run past (W-1)*stride + n floats)
    stride2 = b.n + 8
    flat = torch.zeros((cfg.W - 1) * stride2 + b.n, dtype=torch.float32).pin_memory()
    for w in range(cfg.W):
        flat[w * stride2: w * stride2 + b.n] = g_host[w, :b.n]
    staging2 = torch.zeros_like(flat, device=DEV)
    nf.nf_aggregate_bucket_host(flat, staging2, stride2, cfg.W, b.n, bb.off, bb.len, bb.elig, bb.T, (1, 0, 1),
                                nf.MODE_GTERNARY, None, 0, 1.0, bb.route, bb.woff, bb.summary, None, None, 0,
                                bb.abs_sum, bb.sumsq, bb.nan_cnt, bb.inf_cnt, bb.out, out_host, bb.plan, bb.workspace)
    torch.cuda.synchronize()
    compare(bb, ref, cfg.W, O.MODE_GTERNARY, check_planes=False, check_scale=False, what="host entry point, tight buffer")


@pytest.mark.parametrize("seed", range(24))
def test_random_layouts(seed):
    """Seeded random buckets: tensor counts, lengths (from 1 element to several tiles), gaps, unaligned offsets
    and strides, W (one or several worker groups), mode, tau, margin, alpha, state — fused call and five calls
    against the oracle."""
    rng = np.random.default_rng(9000 + seed)
    T = int(rng.integers(1, 40))
    lens = []
    for _ in range(T):
        kind = rng.integers(0, 4)
        lens.append(int({0: rng.integers(1, 40), 1: rng.integers(40, 2100), 2: rng.integers(2100, 9000),
                         3: 2048 * int(rng.integers(1, 4))}[int(kind)]))
    align = bool(rng.integers(0, 2))
    off, o = [], 0 if align else int(rng.integers(0, 4))
    for l in lens:
        off.append(o)
        o += l
        if rng.random() < 0.2:
            o += int(rng.integers(1, 9))                      # gap
        if align:
            o = (o + 3) // 4 * 4
    n = o + int(rng.integers(0, 3))
    W = int(rng.choice([1, 2, 3, 5, 8, 9, 16, 23, 40]))
    elig = [int(x) for x in rng.integers(0, 2, T)]
    mode = O.MODE_GTERNARY if rng.random() < 0.6 else O.MODE_GBINARY
    g = (rng.standard_normal((W, n)) * 10 ** rng.uniform(-5, 1, (1, n))).astype(np.float32)
    g[rng.random((W, n)) < 0.08] = 0.0
    if rng.random() < 0.3:
        g[rng.integers(0, W), rng.integers(0, n)] = np.nan
    if rng.random() < 0.3:
        g[rng.integers(0, W), rng.integers(0, n)] = np.inf
    tau = (rng.random(T) * 1e-3).astype(np.float32) if rng.random() < 0.5 else None
    margin = int(rng.integers(0, 3))
    alpha = 1.0 if rng.random() < 0.5 else 1.0 / W
    state = (1, 0, 1) if rng.random() < 0.8 else (1, 1, 1)
    pad = rng.random() < 0.5                                   # worker stride a multiple of 4 or exactly n
    gd = _dev(g, pad_to4=pad)
    if gd.shape[1] < n:                                        # _dev pads tiny buckets to 4 columns
        pytest.skip("degenerate")
    run_both(gd, np.array(off, np.int64), np.array(lens, np.int64), elig, state=state, mode=mode, tau=tau,
             margin=margin, alpha=alpha, what=f"random layout seed {seed}")


@pytest.mark.parametrize("T,W", [(257, 16), (700, 16), (300, 40), (700, 40), (256, 40)])
def test_many_tensor_buckets_wide_fan_in(T, W):
    """T around / above the 256-tensor shared-memory metadata capacity with SEVERAL worker groups (W > 8) and a few
    tensors of several hundred tiles each (so that the tile scheduler, the group-major runs and the per-tensor
    completion counters are all exercised on the T > 256 path: separate route kernel, global-memory lookups)."""
    rng = np.random.default_rng(7000 + T + W)
    lens = [int(x) for x in rng.integers(1, 1500, T)]
    big = {3: 2048 * 310 + 1234, T // 3: 2048 * 205, T - 2: 2048 * 140 + 31}
    for t, l in big.items():
        lens[t] = l
    lens[T // 2] = 2048 * 2 + 17
    off, ln, n = layout(lens)
    elig = [int(x) for x in rng.integers(0, 2, T)]
    elig[3], elig[T // 3], elig[T - 2] = 1, 0, 1             # big low-bit, big FP32-route, big low-bit
    g = (rng.standard_normal((W, n)) * 10 ** rng.uniform(-4, 0, (1, n))).astype(np.float32)
    g[rng.random((W, n)) < 0.05] = 0.0
    g[W - 1, off[T - 2] + 77] = np.inf
    run_both(_dev(g), off, ln, elig, what=f"T={T} W={W}")


@pytest.mark.parametrize("R", [1, 3, 11])
def test_health_stats_replica_counts_other_than_W(R):
    """nf_health_stats with R != W ('applied to the W inputs and/or to the aggregated output,
    R = 1'), plan routed for another worker count."""
    cfg = shapes.get("resnet50", small=True)
    b = cfg.buckets[-1]
    rng = np.random.default_rng(40 + R)
    x = (rng.standard_normal((R, b.n)) * 10 ** rng.uniform(-5, 1, (1, b.n))).astype(np.float32)
    x[rng.random((R, b.n)) < 0.01] = np.nan
    x[rng.random((R, b.n)) < 0.01] = np.inf
    x[0, : min(b.n, 5)] = -np.inf
    xd = _dev(x)
    bb = BucketBuffers(b.off, b.length, b.elig, b.n, max(R, 2), DEV, planes=False, health=True)
    bb.route_bucket((1, 0, 1))
    bb.health_stats(xd, xd.shape[1], R=R)
    torch.cuda.synchronize()
    Q, cn, ci = O.health_stats(x, b.off, b.length)
    from tests.util import assert_float_match
    T = bb.T
    got = _np(bb.sumsq).reshape(-1)[:R * T].reshape(R, T)
    assert_float_match(np.sqrt(got), np.sqrt(Q), 1e-5, "l2 norm")
    assert np.array_equal(_np(bb.nan_cnt).reshape(-1)[:R * T].reshape(R, T).astype(np.uint64), cn)
    assert np.array_equal(_np(bb.inf_cnt).reshape(-1)[:R * T].reshape(R, T).astype(np.uint64), ci)


@pytest.mark.parametrize("name", ["tiny", "vit_b16", "gpt2_1p3b"])
def test_health_stats_of_the_aggregated_output(name):
    """R = 1 on `out`: the health statistics of the aggregate the hook hands back (consumer: the Supervisor, PAPER
    L158 / L177), computed by nf_health_stats from the fused call's own output buffer."""
    cfg = shapes.get(name, small=(name != "tiny"))
    for b in cfg.buckets:
        g = gen.gen_bucket(cfg, b, DEV)
        bb = BucketBuffers(b.off, b.length, b.elig, b.n, cfg.W, DEV, planes=False, health=True)
        bb.aggregate(g, g.shape[1])
        torch.cuda.synchronize()
        ref = O.aggregate_bucket(np.ascontiguousarray(_np(g)[:, :b.n]), b.off, b.length, b.elig)
        Q, cn, ci = O.health_stats(ref.out.reshape(1, -1), b.off, b.length)
        bb.health_stats(bb.out, b.n, R=1)
        torch.cuda.synchronize()
        from tests.util import assert_float_match
        T = bb.T
        assert_float_match(np.sqrt(_np(bb.sumsq)[0, :T]), np.sqrt(Q[0]), 1e-5, f"{cfg.name} bucket {b.index} out l2")
        assert np.array_equal(_np(bb.nan_cnt)[0, :T].astype(np.uint64), cn[0])
        assert np.array_equal(_np(bb.inf_cnt)[0, :T].astype(np.uint64), ci[0])


@pytest.mark.parametrize("name", ["tiny", "resnet50", "vit_b16", "sweep_w32"])
def test_run_to_run_bitwise_reproducible(name):
    """PAPER L243 'synchronized aggregate direction': every replica of the hook must produce the same bits. Same
    input ten times through the fused call and through the stand-alone calls: out, scale, abs_sum, sumsq and the
    planes are BITWISE identical between runs (tile scheduling is dynamic; the totals must not depend on it)."""
    cfg = shapes.get(name, small=(name not in ("tiny",)))
    for b in cfg.buckets[:3]:
        g = gen.gen_bucket(cfg, b, DEV)
        bb = BucketBuffers(b.off, b.length, b.elig, b.n, cfg.W, DEV, planes=True, health=True)
        first = None
        for rep in range(10):
            bb.out.fill_(float(rep))
            bb.aggregate(g, g.shape[1])
            torch.cuda.synchronize()
            cur = [bb.out.clone(), bb.scale.clone(), bb.abs_sum.clone(), bb.sumsq.clone(), bb.P.clone(), bb.N.clone(),
                   bb.nan_cnt.clone(), bb.inf_cnt.clone()]
            if first is None:
                first = cur
            else:
                for k, (x, y) in enumerate(zip(first, cur)):
                    assert torch.equal(x.view(torch.uint8), y.view(torch.uint8)), f"fused run {rep}, output {k} differs"
        first = None
        for rep in range(10):
            bb.route_bucket((1, 0, 1))
            bb.sign_pack(g, g.shape[1], nf.MODE_GTERNARY)
            bb.sign_count_reduce(nf.MODE_GTERNARY)
            bb.fp32_reduce(g, g.shape[1])
            bb.health_stats(g, g.shape[1])
            torch.cuda.synchronize()
            cur = [bb.out.clone(), bb.scale.clone(), bb.abs_sum.clone(), bb.sumsq.clone()]
            if first is None:
                first = cur
            else:
                for k, (x, y) in enumerate(zip(first, cur)):
                    assert torch.equal(x.view(torch.uint8), y.view(torch.uint8)), f"5-call run {rep}, output {k} differs"


def test_full_size_bucket_run_to_run_bitwise():
    """The same on a full 33.6 M-element GPT bucket (16 400 tiles over 148 persistent CTAs: which CTA processes
    which tile differs from run to run)."""
    cfg = shapes.gpt2_1p3b()
    b = cfg.buckets[0]
    g = gen.gen_bucket(cfg, b, DEV)
    bb = BucketBuffers(b.off, b.length, b.elig, b.n, cfg.W, DEV, planes=False, health=True)
    first = None
    for rep in range(10):
        bb.aggregate(g, g.shape[1])
        torch.cuda.synchronize()
        cur = [bb.out.clone(), bb.scale.clone(), bb.abs_sum.clone(), bb.sumsq.clone()]
        if first is None:
            first = cur
        else:
            for k, (x, y) in enumerate(zip(first, cur)):
                assert torch.equal(x.view(torch.uint8), y.view(torch.uint8)), f"run {rep}, output {k} differs"


@pytest.mark.parametrize("T", [64, 700])
def test_concurrent_calls_on_two_streams_behind_foreign_work(T):
    """The DDP-hook setting: the aggregation runs while other kernels (backward compute) hold part of the SMs, and
    two buckets may be in flight on two streams. No call may depend on all of its CTAs being resident at once.
    A long-running filler kernel occupies the device, then two nf_aggregate_bucket calls (separate plans, workspaces
    and outputs) are issued on two streams, 50 times; both must match the oracle."""
    rng = np.random.default_rng(T)
    lens = [int(x) for x in rng.integers(1, 3000, T)]
    lens[2] = 2048 * 150 + 5
    lens[T - 1] = 2048 * 90
    off, ln, n = layout(lens)
    elig = [int(x) for x in rng.integers(0, 2, T)]
    elig[2] = elig[T - 1] = 1
    W = 8
    gs, refs, bbs = [], [], []
    for k in range(2):
        g = (rng.standard_normal((W, n)) * 10 ** rng.uniform(-4, 0, (1, n))).astype(np.float32)
        gs.append(_dev(g))
        refs.append(O.aggregate_bucket(g, off, ln, elig))
        bbs.append(BucketBuffers(off, ln, elig, n, W, DEV, planes=True, health=True))
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    filler_stream = torch.cuda.Stream()
    a = torch.randn((8192, 8192), device=DEV, dtype=torch.float32)
    torch.cuda.synchronize()
    for it in range(50):
        with torch.cuda.stream(filler_stream):
            for _ in range(2):
                a = torch.tanh(a @ a * 1e-3)                 # a few ms of foreign work on all SMs
        for k in range(2):
            bbs[k].aggregate(gs[k], gs[k].shape[1], stream=streams[k])
        if it % 10 == 9:
            torch.cuda.synchronize()
            for k in range(2):
                compare(bbs[k], refs[k], W, O.MODE_GTERNARY, what=f"concurrent T={T} iteration {it} stream {k}")
    torch.cuda.synchronize()


@pytest.mark.parametrize("W", [4, 24])
def test_adjacent_lowbit_tensors_meeting_inside_a_warp_of_the_count_reduce(W):
    """Low-bit tensors that are adjacent in the bucket and a whole number of 32-element words long, with word offsets
    that are not multiples of 32: a warp of nf_sign_count_reduce (32 consecutive word positions) then holds words of
    two tensors whose elements are contiguous in `out`, and must still give each its own scale (the 512-byte
    write-back path once took them for one tensor)."""
    rng = np.random.default_rng(4242 + W)
    lens = [2080, 4096, 96, 32 * 77, 5000, 32 * 33, 32 * 31, 2048 * 3]
    off, ln, n = layout(lens)
    elig = [1, 1, 1, 1, 1, 1, 1, 1]
    g = (rng.standard_normal((W, n)) * 10 ** rng.uniform(-4, 0, (1, n))).astype(np.float32)
    for t, (o, l) in enumerate(zip(off, ln)):          # very different scales per tensor
        g[:, o:o + l] *= 10.0 ** (t - 4)
    gd = _dev(g)
    ref = run_both(gd, off, ln, elig, what=f"adjacent low-bit tensors W={W}")
    # the five calls WITHOUT count outputs: nf_sign_count_reduce then writes back 512 contiguous bytes per store
    bc = BucketBuffers(off, ln, elig, n, W, gd.device, planes=True, counts=False, health=True)
    bc.out.fill_(-77.0)
    bc.route_bucket((1, 0, 1))
    bc.sign_pack(gd, gd.shape[1], O.MODE_GTERNARY)
    bc.sign_count_reduce(O.MODE_GTERNARY, 0)
    bc.fp32_reduce(gd, gd.shape[1], 1.0)
    bc.health_stats(gd, gd.shape[1])
    compare(bc, ref, W, O.MODE_GTERNARY, what=f"adjacent low-bit tensors W={W} [5-call, no count outputs]")
