"""CPU-only: the C-ABI library loads and exports every symbol include/ajt.h declares; host-side argument
validation works without a GPU; the product path fails loudly without a device (no fallback)."""
import ctypes as C
import os
import re
import shutil

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = "".join(open(os.path.join(ROOT, "include", f)).read() for f in sorted(os.listdir(os.path.join(ROOT, "include")))
                  if f.endswith(".h"))
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ajt_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_04484_b200 import build as b
    if shutil.which("nvcc") or os.path.exists("/usr/local/cuda/bin/nvcc"):
        b.build()
    import paper_2606_04484_b200 as ajt
    return ajt


def test_header_symbols_are_exported(lib):
    names = declared_symbols()
    assert len(names) >= 11
    L = lib.lib()
    for n in names:
        assert hasattr(L, n), n
    assert sorted(lib.exported_symbols()) == names


def test_version_and_strerror(lib):
    assert lib.version() >= 100
    assert lib.strerror(0) == "ok"
    assert "workspace" in lib.strerror(-2)
    assert "unknown" in lib.strerror(-99)


def test_workspace_queries(lib):
    assert lib.merge_workspace_bytes(0, 0) > 0
    assert lib.merge_workspace_bytes(512, 1 << 20) > lib.merge_workspace_bytes(16, 1 << 10)
    assert lib.merge_workspace_bytes(-1, 0) == 0
    a, b = lib.loss_workspace_bytes(1024, 32000, 8), lib.loss_workspace_bytes(65536, 151936, 256)
    assert 0 < a < b
    assert lib.loss_host_arena_bytes(64, 1024, 4, 1024, lib.DT_BF16) > 64 * 1024 * 2
    assert lib.merge_host_arena_bytes(8, 4096) > 4096 * 4


def test_host_detectable_errors_without_gpu(lib):
    L = lib.lib()
    one = (C.c_uint8 * 512)()
    # invalid arguments are rejected before any CUDA call
    rc = L.ajt_policy_loss_fwd_bwd(None, None, None, None, None, None, C.c_float(0.2), C.c_float(0.2), C.c_int64(4),
                                   C.c_int32(0), C.c_int32(1), C.c_int64(8), C.c_int32(0), None, C.c_float(0), C.c_float(1),
                                   None, None, None, None, None, C.c_size_t(0), None)
    assert rc == -1
    rc = L.ajt_merge_timelines(None, None, None, None, None, None, C.c_int32(-1), C.c_int64(0), C.c_int32(0), C.c_uint32(0),
                               None, None, None, None, None, None, None, None, None, None, C.c_size_t(0), None)
    assert rc == -1
    rc = L.ajt_merge_timelines(one, one, one, one, None, None, C.c_int32(1), C.c_int64(1), C.c_int32(5), C.c_uint32(0),
                               one, one, one, None, one, one, one, one, one, one, C.c_size_t(512), None)
    assert rc == -1   # unknown owner rule


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_cpu_fallback(lib):
    t = torch.zeros(4, dtype=torch.int32)
    with pytest.raises((RuntimeError, TypeError)):
        lib.merge_timelines(t, torch.zeros(2, dtype=torch.int64), t[:1], t[:1])
    with pytest.raises((RuntimeError, TypeError)):
        lib.policy_loss_fwd_bwd(torch.zeros(2, 8, dtype=torch.bfloat16), t[:2], torch.zeros(2), torch.zeros(2),
                                torch.zeros(2, dtype=torch.uint8), t[:2], 1, 0.2, 0.2)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_04484_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                s = open(os.path.join(dp, f)).read()
                assert "import oracle" not in s and "from oracle" not in s and "ajt_oracle" not in s, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            s = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2606_04484_b200" not in s and "from paper_2606_04484_b200" not in s and "csrc" not in s.replace(
                "paper_2606_04484_b200/csrc/", ""), f
