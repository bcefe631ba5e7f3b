"""Host-side checks of the C ABI that need no GPU: the library builds, loads and exports every
symbol include/vx.h declares; argument validation; and the loud failure without a CUDA device."""
import ctypes
import os
import re

import pytest

import paper_2606_14007_b200 as vx
import vx_inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_functions():
    text = open(os.path.join(ROOT, "include", "vx.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(vx_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    L = vx.load_library()
    declared = header_functions()
    assert declared, "no declarations parsed from include/vx.h"
    assert sorted(vx.EXPORTS) == declared
    for name in declared:
        assert getattr(L, name) is not None


def test_workspace_bytes_arithmetic():
    assert vx.workspace_bytes(0) == 0 and vx.workspace_bytes(41) == 0 and vx.workspace_bytes(37) == 0
    # K = 34..36: bucket-range passes, each the size of a K = 33 plot
    assert 170e9 < vx.workspace_bytes(34) < 178e9 and 170e9 < vx.workspace_bytes(36) < 178e9
    assert vx.workspace_bytes(20, 24, vx.VX_CREATE_PASSES_LOG(2)) < vx.workspace_bytes(20, 24)
    assert vx.workspace_bytes(12, 24, vx.VX_CREATE_PASSES_LOG(1)) == 0   # one partition cannot be split
    a, b = vx.workspace_bytes(27), vx.workspace_bytes(28)
    assert 0 < a < b
    # K=31: Table 1 in place in the partition array (2^31 x 16 B x 1.125 slack = 38.7 GB)
    # + Table 2 (17.2 GB) + offsets
    assert 50e9 < vx.workspace_bytes(31) < 60e9
    assert vx.workspace_bytes(32) < 120e9
    # K=33: wide layout, 10-byte Table-1 records in place (96.6 GB) + 9-byte Table-2 records (77.3 GB)
    assert 170e9 < vx.workspace_bytes(33) < 178e9
    # the test-only wide layout is smaller than the 16-byte-record layout at the same K
    assert 0 < vx.workspace_bytes(20, 24, vx.VX_CREATE_WIDE_LAYOUT) < vx.workspace_bytes(20, 24)
    assert 0 < vx.workspace_bytes(20, 24, vx.VX_CREATE_BIG_TILES)
    assert vx.workspace_bytes(20, 24, 4) == 0              # unknown flag
    assert vx.workspace_bytes(16, 12) > 0 and vx.workspace_bytes(16, 4) == 0


def test_create_validates_arguments():
    L = vx.load_library()
    h = ctypes.c_void_p()
    key = vx_inputs.key_from_seed(1)
    assert L.vx_plot_create(0, key, ctypes.byref(h)) == -1
    assert L.vx_plot_create(41, key, ctypes.byref(h)) == -1
    assert L.vx_plot_create(20, None, ctypes.byref(h)) == -1
    assert L.vx_plot_create(20, key, None) == -1
    assert L.vx_plot_create_ex(16, key, 25, ctypes.byref(h)) == -1
    assert L.vx_plot_create_ex(16, key, 4, ctypes.byref(h)) == -1      # mean bucket > 512
    assert L.vx_plot_create_opts(16, key, 12, 4, ctypes.byref(h)) == -1  # unknown flag
    assert L.vx_plot_create(33, key, ctypes.byref(h)) == 0 and h.value   # 5-byte nonces, wide layout
    ns = ctypes.c_uint32()
    assert L.vx_plot_info(h, None, None, ctypes.byref(ns), None, None, None) == 0 and ns.value == 5
    # wide layout: 2 clears, 4 rounds of hash+scatter and compaction, the partition scan
    l1, l2 = ctypes.c_uint32(), ctypes.c_uint32()
    assert L.vx_plot_launches(h, ctypes.byref(l1), ctypes.byref(l2)) == 0 and (l1.value, l2.value) == (11, 2)
    # streamed egress: not before vx_build_table1 (and never for 5-byte nonces)
    assert L.vx_sort_match_table2_to_host(h, None, ctypes.c_void_p(8), 4, ctypes.c_void_p(8), 0, None, None) == -2
    assert L.vx_sort_match_table2_to_file(h, None, ctypes.c_void_p(8), 4, -1, None, 0, None) == -1
    assert L.vx_status_string(-8) == b"VX_ERR_IO"
    L.vx_free(h)
    assert L.vx_plot_create(20, key, ctypes.byref(h)) == 0 and h.value
    info = [ctypes.c_uint32() for _ in range(5)]
    t2 = ctypes.c_uint64()
    assert L.vx_plot_info(h, *[ctypes.byref(x) for x in info], ctypes.byref(t2)) == 0
    assert [x.value for x in info[:4]] == [20, 24, 4, 8]
    assert L.vx_plot_launches(h, ctypes.byref(l1), ctypes.byref(l2)) == 0 and (l1.value, l2.value) == (3, 2)
    # out-of-order calls
    assert L.vx_build_table1(h, None) == -2
    assert L.vx_sort_match_table2(h, None) == -2
    assert L.vx_synchronize(h) == -2
    need = ctypes.c_size_t()
    assert L.vx_read_tables(h, 1, 0, 1, None, None, 0, ctypes.byref(need)) == -2
    assert b"VX_ERR_STATE" in L.vx_last_error(h)
    assert L.vx_status_string(-5) == b"VX_ERR_OVERFLOW"
    L.vx_free(h)
    L.vx_free(None)


def test_no_cuda_device_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(vx.VxError) as ei:
        vx.Plot(12, vx_inputs.key_from_seed(1), 8)
    assert ei.value.status == -4
    with pytest.raises(vx.VxError):
        vx.hash_range(20, vx_inputs.key_from_seed(1), 0, 16)
    # and straight through the C ABI: binding a workspace needs a device
    L = vx.load_library()
    h = ctypes.c_void_p()
    assert L.vx_plot_create(12, vx_inputs.key_from_seed(1), ctypes.byref(h)) == 0
    assert L.vx_plot_bind(h, ctypes.c_void_p(256), 1 << 30) == -4
    assert b"VX_ERR_CUDA" in L.vx_last_error(h)
    L.vx_free(h)


def test_product_and_oracle_are_independent():
    pkg = os.path.join(ROOT, "paper_2606_14007_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"\boracle\b|vxo_|vx_oracle", src), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"import\s+paper_2606|from\s+paper_2606|libvx\.so|vx_blake3\.cuh|#include\s+\"vx", src), f
