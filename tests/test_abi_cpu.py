"""`-m "not gpu"`: the C-ABI library loads, exports every symbol include/nf.h declares, and its
host-side argument checks answer without a GPU (no compute calls)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def nf():
    from paper_2606_25759_b200 import build, binding
    build.build()
    return binding


def test_every_declared_symbol_is_exported(nf):
    hdr = open(os.path.join(ROOT, "include", "nf.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(nf_[a-z0-9_]+)\s*\(", hdr))
    assert {"nf_route_bucket", "nf_sign_pack", "nf_sign_count_reduce", "nf_fp32_reduce",
            "nf_health_stats", "nf_aggregate_bucket"} <= declared
    lib = nf.lib()
    for name in declared:
        assert hasattr(lib, name), name
    assert declared == set(nf.EXPORTS)


def test_host_side_checks_need_no_gpu(nf):
    lib = nf.lib()
    assert lib.nf_version() >= 100
    assert nf.status_string(0) == "NF_OK"
    assert nf.nf_plan_bytes(0) >= 64 and nf.nf_plan_bytes(100) > nf.nf_plan_bytes(10)
    assert nf.nf_plan_bytes(10, 8) - nf.nf_plan_bytes(10, 1) == 7 * 10 * 256      # 256-byte exact accumulator per (replica, tensor)
    assert nf.nf_workspace_bytes(3, 1 << 20) >= (1 << 20) // 4
    st = nf.NfState(1, 0, 1)
    fake = 0x1000                     # never dereferenced: the range/alignment checks come first
    # W out of range
    rc = lib.nf_fp32_reduce(fake, 64, 0, 64, fake, fake, fake, 1, 1.0, fake, fake, None)
    assert rc == nf.NF_ERR_RANGE
    rc = lib.nf_fp32_reduce(fake, 64, 256, 64, fake, fake, fake, 1, 1.0, fake, fake, None)
    assert rc == nf.NF_ERR_RANGE
    # worker_stride < n
    rc = lib.nf_fp32_reduce(fake, 32, 2, 64, fake, fake, fake, 1, 1.0, fake, fake, None)
    assert rc == nf.NF_ERR_ARG
    # misaligned base pointer
    rc = lib.nf_fp32_reduce(fake + 4, 64, 2, 64, fake, fake, fake, 1, 1.0, fake, fake, None)
    assert rc == nf.NF_ERR_ALIGN
    # bad mode / margin
    rc = lib.nf_sign_count_reduce(fake, fake, 64, 2, 64, fake, fake, fake, fake, 1, 7, 0, fake, fake,
                                  None, None, None, fake, None)
    assert rc == nf.NF_ERR_ARG
    rc = lib.nf_sign_count_reduce(fake, fake, 64, 2, 64, fake, fake, fake, fake, 1, 2, 300, fake, fake,
                                  None, None, None, fake, None)
    assert rc == nf.NF_ERR_RANGE
    # plan too small
    rc = lib.nf_route_bucket(fake, fake, fake, 4, 64, st, fake, fake, fake, fake, 8, None)
    assert rc == nf.NF_ERR_ARG
    # G-Ternary without a neg plane
    rc = lib.nf_sign_pack(fake, 64, 2, 64, fake, fake, fake, fake, 1, 2, None, fake, None, 64, fake, fake, None)
    assert rc == nf.NF_ERR_ARG


def test_missing_library_fails_loudly(nf, monkeypatch):
    monkeypatch.setattr(nf, "_lib", None)
    monkeypatch.setattr(nf, "LIB_PATH", "/nonexistent/libnf.so")
    with pytest.raises(RuntimeError, match="no CPU or PyTorch fallback"):
        nf.lib()
