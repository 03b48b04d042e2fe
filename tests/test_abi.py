"""The C-ABI boundary without a GPU: the library builds, loads and exports every symbol include/lgf.h declares;
argument checking and the no-CPU-fallback rule hold.  No compute call is made here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_1301_3460_b200 as lgf

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_symbols():
    txt = open(os.path.join(ROOT, "include", "lgf.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(lgf_[a-z_0-9]+)\s*\(", txt)))


def test_library_builds_and_exports_every_header_symbol():
    L = lgf.lib()
    syms = header_symbols()
    assert len(syms) >= 20
    for s in syms:
        assert hasattr(L, s), f"{s} declared in include/lgf.h but not exported"
    assert sorted(lgf.EXPORTS) == syms


def test_status_strings_and_kernel_names():
    L = lgf.lib()
    for st in (0, 1, 2, 3, 4, 5, 6, 100):
        assert len(L.lgf_status_string(st)) > 0
    names = [L.lgf_kernel_name(i).decode() for i in range(lgf.LGF_MAX_KERNELS)]
    assert "k_update_quad" in names and "k_fft23_mid" in names and "k_fa_delta_fwd" in names
    assert L.lgf_kernel_name(99) == b""


def test_workspace_bytes_and_supported_sizes():
    L = lgf.lib()
    d = lambda *v: (C.c_int * 4)(*v)
    V = 32 ** 4
    n12 = L.lgf_workspace_bytes(d(32, 32, 32, 32), lgf.LGF_FP64, lgf.LGF_STORE_12)
    n18 = L.lgf_workspace_bytes(d(32, 32, 32, 32), lgf.LGF_FP64, lgf.LGF_STORE_18)
    # links 384 / 576 B per site, one buffer (updated in place), field 64 B, stored g 96 B
    assert V * (384 + 64) <= n12 <= V * (384 + 64 + 96) + (80 << 20) and n18 - n12 == V * 192
    assert L.lgf_workspace_bytes(d(64, 64, 64, 64), lgf.LGF_FP64, lgf.LGF_STORE_12) >= 64 ** 4 * 448
    assert L.lgf_workspace_bytes(d(32, 32, 32, 64), lgf.LGF_FP64, lgf.LGF_STORE_12) > 0
    assert L.lgf_workspace_bytes(d(8, 8, 8, 8), lgf.LGF_FP64, lgf.LGF_STORE_18) > 0
    # fp32 (LGF_FP32): half the link and field bytes
    n12f = L.lgf_workspace_bytes(d(32, 32, 32, 32), lgf.LGF_FP32, lgf.LGF_STORE_12)
    assert V * (192 + 32) <= n12f < n12 - V * 192
    # unsupported: non power of two, too small, bad precision, bad storage
    assert L.lgf_workspace_bytes(d(12, 8, 8, 8), lgf.LGF_FP64, lgf.LGF_STORE_12) == 0
    assert L.lgf_workspace_bytes(d(2, 8, 8, 8), lgf.LGF_FP64, lgf.LGF_STORE_12) == 0
    assert L.lgf_workspace_bytes(d(8, 8, 8, 8), 7, lgf.LGF_STORE_12) == 0
    assert L.lgf_workspace_bytes(d(8, 8, 8, 8), lgf.LGF_FP64, 10) == 0


def test_argument_errors_before_any_device_work():
    L = lgf.lib()
    h = C.c_void_p()
    d = (C.c_int * 4)(8, 8, 8, 8)
    assert L.lgf_create(None, 0, 12, C.byref(h)) == lgf.LGF_ERR_INVALID_ARG
    assert L.lgf_create(d, 7, 12, C.byref(h)) == lgf.LGF_ERR_INVALID_ARG
    assert L.lgf_create(d, 0, 13, C.byref(h)) == lgf.LGF_ERR_INVALID_ARG
    st = L.lgf_create(d, lgf.LGF_FP32, 12, C.byref(h))            # fp32 is built: only the missing device can refuse it
    assert st in (lgf.LGF_ERR_CUDA, lgf.LGF_OK)
    if st == lgf.LGF_OK:
        L.lgf_destroy(h)
    bad = (C.c_int * 4)(8, 8, 6, 8)
    assert L.lgf_create(bad, 0, 12, C.byref(h)) == lgf.LGF_ERR_UNSUPPORTED
    neg = (C.c_int * 4)(8, 8, -1, 8)
    assert L.lgf_create(neg, 0, 12, C.byref(h)) == lgf.LGF_ERR_INVALID_ARG
    # NULL contexts
    F = C.c_double()
    assert L.lgf_iterate(None, 1, 0.08, C.byref(F), C.byref(F)) == lgf.LGF_ERR_INVALID_ARG
    assert L.lgf_fix(None, 0.08, 1e-15, 10, None, None, None) == lgf.LGF_ERR_INVALID_ARG
    assert L.lgf_load_links(None, None) == lgf.LGF_ERR_INVALID_ARG
    assert L.lgf_launch_count(None) == 0
    L.lgf_destroy(None)


def test_create_error_text_belongs_to_the_last_create():
    """lgf_last_error(NULL) describes the LAST lgf_create* of the calling thread on every failing path -- argument
    errors and fp32 contexts included -- and never a stale text of an earlier one."""
    L = lgf.lib()
    h = C.c_void_p()
    d = lambda *v: (C.c_int * 4)(*v)
    assert L.lgf_create(d(8, 8, 6, 8), lgf.LGF_FP64, 12, C.byref(h)) == lgf.LGF_ERR_UNSUPPORTED
    assert b"powers of two" in L.lgf_last_error(None)
    assert L.lgf_create(d(8, 8, 8, 8), 7, 12, C.byref(h)) == lgf.LGF_ERR_INVALID_ARG
    assert b"precision" in L.lgf_last_error(None)                        # not the text of the call before
    assert L.lgf_create(d(8, 8, 8, 8), lgf.LGF_FP64, 13, C.byref(h)) == lgf.LGF_ERR_INVALID_ARG
    assert b"storage" in L.lgf_last_error(None)
    assert L.lgf_create(d(8, 8, 6, 8), lgf.LGF_FP32, 12, C.byref(h)) == lgf.LGF_ERR_UNSUPPORTED
    assert b"powers of two" in L.lgf_last_error(None)                    # forwarded from the fp32 translation unit
    assert L.lgf_create_ex(d(8, 8, 8, 8), lgf.LGF_MIXED, 12, None, 0, None, C.byref(h)) == lgf.LGF_ERR_INVALID_ARG
    assert b"workspace" in L.lgf_last_error(None)
    st = L.lgf_create(d(8, 8, 8, 8), lgf.LGF_FP64, 12, C.byref(h))
    if st == lgf.LGF_OK:                                                 # a device is present: a success leaves no text
        assert L.lgf_last_error(None) == b""
        L.lgf_destroy(h)
    else:
        assert st == lgf.LGF_ERR_CUDA and b"no CUDA device" in L.lgf_last_error(None)


def test_sharded_create_failures_leave_a_text():
    L = lgf.lib()
    h = C.c_void_p()
    d = lambda *v: (C.c_int * 4)(*v)
    assert L.lgf_create_sharded(d(8, 8, 8, 8), 3, 12, C.byref(h)) == lgf.LGF_ERR_INVALID_ARG
    assert b"power of two" in L.lgf_last_error_sharded(None)
    assert L.lgf_create_sharded(d(16, 4, 16, 16), 8, 12, C.byref(h)) == lgf.LGF_ERR_UNSUPPORTED
    assert b"n_ranks must not exceed" in L.lgf_last_error_sharded(None)
    with pytest.raises(lgf.LgfError) as e:
        lgf.ShardedGaugeFixer((16, 16, 16, 16), 3)
    assert "power of two" in str(e.value)


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    L = lgf.lib()
    h = C.c_void_p()
    d = (C.c_int * 4)(8, 8, 8, 8)
    assert L.lgf_create(d, 0, 12, C.byref(h)) == lgf.LGF_ERR_CUDA
    assert not h.value
    with pytest.raises(lgf.LgfError):
        lgf.GaugeFixer((8, 8, 8, 8), 12)
    with pytest.raises(lgf.LgfError):
        lgf.GaugeFixer((8, 8, 8, 8), 12, use_torch_workspace=False)


def test_product_does_not_import_the_oracle():
    """The product path shares nothing with oracle/: no import, no file read (judge's rule, section 3)."""
    pkg = os.path.join(ROOT, "paper_1301_3460_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "lgf_oracle" not in txt, f
    for dirpath, _, files in os.walk(os.path.join(ROOT, "oracle")):
        for f in files:
            if f.endswith((".py", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import paper_1301_3460_b200" not in txt and "liblgf.so" not in txt and "csrc" not in txt, f
