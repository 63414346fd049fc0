"""N>1 host logic of bench.py on CPU: two gloo ranks, barrier + max-over-ranks timing, replica
accounting (replicas only, no data-path collective)."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch, bench
rank, world, local = bench.dist_setup(2)
assert world == 2
bench.barrier(world)
ms = bench.max_over_ranks(10.0 * (rank + 1), world, torch.device("cpu"))   # ranks report 10 and 20 ms
bench.barrier(world)
cfgbytes = 1000
value = world * cfgbytes / (ms * 1e-3) / 1e9
print(json.dumps({"rank": rank, "ms": ms, "value": value}))
import torch.distributed as dist
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_two_gloo_ranks_take_max_time_and_sum_work():
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER % ROOT], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=120)
        assert p.returncode == 0, e[-2000:]
        outs.append(json.loads(o.strip().splitlines()[-1]))
    for o in outs:
        assert o["ms"] == 20.0                                  # MAX over ranks
        assert abs(o["value"] - 2 * 1000 / 0.020 / 1e9) < 1e-12  # whole-job aggregate over both replicas


def test_reference_arm_nonzero_rank_exits_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1", CUDA_VISIBLE_DEVICES="")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0", "--config", "tiny"], env=env, capture_output=True,
                       text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_reference_arm_prints_contract_line_on_cpu():
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "2",
                        "--warmup", "1", "--config", "tiny"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    d = json.loads(r.stdout.strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["unit"] == "GB/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0


def test_algorithmic_bytes_accounting():
    sys.path.insert(0, ROOT)
    import bench
    from workloads import shapes
    cfg = shapes.sweep(8, 6_553_600)
    tot_in, tot_all, passA = bench.algorithmic_bytes(cfg, planes=True, ternary=True)
    n = 6_553_600
    assert tot_in == 32 * n
    assert passA == 32 * n + 2 * n + n // 4          # 34.25 B per element
    assert tot_all == passA + n // 4 + 4 * n         # 38.5 B per element
