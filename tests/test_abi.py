"""CPU-side checks of the C-ABI library: it builds, loads, exports every symbol that
include/haccsr.h declares, validates arguments, and refuses to compute without a GPU
(no CPU fallback).  No compute call is made here."""
import ctypes as C
import os
import re

import pytest
import torch

from paper_1410_2805_b200 import haccsr

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "haccsr.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b(hacc_sr_\w+|haccsr_\w+)\s*\(", src)
    return sorted(set(names))


def test_header_symbols_match_binding_list():
    assert _declared_symbols() == sorted(haccsr.ABI_SYMBOLS)


def test_library_exports_every_declared_symbol():
    lib = haccsr.lib()
    for name in _declared_symbols():
        assert hasattr(lib, name), name


def test_abi_version_and_strerror():
    assert haccsr.lib().haccsr_abi_version() == 2
    assert haccsr.strerror(0) == "ok"
    for s in (-1, -2, -3, -4, -5):
        assert haccsr.strerror(s) not in ("ok", "unknown status")
    assert haccsr.strerror(-99) == "unknown status"


def test_workspace_bytes_validation_and_growth():
    wb = haccsr.haccsr_workspace_bytes
    assert wb(0, 10) == 0
    assert wb(100, 3) == 0          # nc >= 4 required
    assert wb(100, 257) == 0
    assert wb(1 << 31, 10) == 0
    a, b, c = wb(32768, 10), wb(65536, 10), wb(32768, 20)
    assert 0 < a < b and a < c
    # per-particle state: cid + perm + float4 = 24 B, plus work items
    assert b - a >= 24 * 32768
    # config 3 fits comfortably in one B200 (180 GB)
    assert wb(512 ** 3, 170) < 8 * 2 ** 30


def test_slab_workspace_and_argument_validation():
    wb = haccsr.lib().haccsr_workspace_bytes_slab
    assert wb(1000, 10, 0) == 0 and wb(1000, 10, 9) == 0      # 1 <= nz_own <= nc - 2
    assert 0 < wb(1000, 10, 2) < wb(1000, 10, 8) <= haccsr.haccsr_workspace_bytes(1000, 10)
    h = C.c_void_p()
    buf = C.create_string_buffer(1024)
    lib = haccsr.lib()
    assert lib.haccsr_create_slab(C.byref(h), 100, 32.0, 10, 0, 9, buf, 1024, None) == haccsr.EINVAL
    assert lib.haccsr_create_slab(C.byref(h), 100, 32.0, 10, 10, 2, buf, 1024, None) == haccsr.EINVAL
    assert lib.haccsr_create_slab(C.byref(h), 100, 32.0, 10, -1, 2, buf, 1024, None) == haccsr.EINVAL
    assert lib.hacc_sr_pack_layer(None, 0, None, None, None, None, 0, None, 0, None) == haccsr.EINVAL
    assert lib.hacc_sr_unpack(None, 0, None, None, None, None, None) == haccsr.EINVAL


def test_create_rejects_bad_arguments_without_touching_the_gpu():
    lib = haccsr.lib()
    h = C.c_void_p()
    buf = C.create_string_buffer(1024)
    assert lib.haccsr_create(None, 100, 32.0, 10, buf, 1024, None) == haccsr.EINVAL
    assert lib.haccsr_create(C.byref(h), 100, 32.0, 3, buf, 1024, None) == haccsr.EINVAL
    assert lib.haccsr_create(C.byref(h), 100, -1.0, 10, buf, 1024, None) == haccsr.EINVAL
    assert lib.haccsr_create(C.byref(h), 100, 32.0, 10, None, 0, None) == haccsr.EINVAL
    need = haccsr.haccsr_workspace_bytes(100, 10)
    ws = C.create_string_buffer(512)
    addr = (C.addressof(ws) + 255) & ~255
    assert lib.haccsr_create(C.byref(h), 100, 32.0, 10, C.c_void_p(addr), need - 1,
                             None) == haccsr.ENOMEM
    assert h.value is None


def test_null_context_calls_return_einval():
    lib = haccsr.lib()
    poly = (C.c_float * 6)()
    assert lib.hacc_sr_bin(None, 0, None, None, None, None, None, None, None) == haccsr.EINVAL
    assert lib.hacc_sr_force(None, 0.1, 3.0, poly, None, None, None, None, None) == haccsr.EINVAL
    assert lib.hacc_sr_kick(None, 0.01) == haccsr.EINVAL
    assert lib.haccsr_sync(None) == haccsr.EINVAL
    assert lib.haccsr_destroy(None) == haccsr.EINVAL


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_cpu_fallback_without_a_gpu():
    with pytest.raises(haccsr.HaccsrError) as e:
        haccsr.Context(1000, 32.0, 10)
    assert e.value.status == haccsr.ECUDA
    ms, ops = C.c_double(), C.c_double()
    assert haccsr.lib().haccsr_probe_peak(0, 1, None, C.byref(ms), C.byref(ops)) == haccsr.ECUDA


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1410_2805_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "sr_oracle" not in text, f


def test_pm_library_exports_every_declared_symbol_and_validates():
    from paper_1410_2805_b200 import haccpm
    src = open(os.path.join(ROOT, "include", "haccpm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = sorted(set(re.findall(r"\b(hacc_lr_\w+|haccpm_\w+)\s*\(", src)))
    assert names == sorted(haccpm.ABI_SYMBOLS)
    lib = haccpm.lib()
    for name in names:
        assert hasattr(lib, name), name
    assert lib.haccpm_abi_version() == 1
    wb = lib.haccpm_workspace_bytes
    assert wb(3) == 0 and wb(33) == 0 and wb(4096) == 0
    assert 0 < wb(32) < wb(64)
    assert wb(512) < 6 * 2 ** 30     # the 512^3 grid of configs[3]: 5.0 GiB (density, three
                                     # component grids, the packed float4 grid, two spectra)
    h = C.c_void_p()
    buf = C.create_string_buffer(1024)
    assert lib.haccpm_create(C.byref(h), 33, 32.0, 0.8, 3, buf, 1024, None) == haccpm.EINVAL
    assert lib.haccpm_create(C.byref(h), 32, -1.0, 0.8, 3, buf, 1024, None) == haccpm.EINVAL
    assert lib.hacc_lr_force(None, 0, None, None, None, None, None, None, None, 0.0, None, None,
                             None) == haccpm.EINVAL
    assert lib.haccpm_sync(None) == haccpm.EINVAL
