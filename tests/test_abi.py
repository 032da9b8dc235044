"""The C-ABI boundary without a GPU: libpeek.so builds (nvcc cross-compiles), loads, exports every
function include/peek.h declares, and its host-side argument checks answer before any CUDA call."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2607_02525_b200 import build
    path = build.build_libpeek()
    return ctypes.CDLL(path)


def declared_functions():
    src = open(os.path.join(ROOT, "include", "peek.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b(peek_[a-z_0-9]+)\s*\(", src)
    return sorted(set(names))


def test_every_declared_symbol_is_exported(lib):
    names = declared_functions()
    assert {"peek_block_hash", "peek_lpm", "peek_pending_tree", "peek_demand_rank",
            "peek_workspace_bytes", "peek_set_option"} <= set(names)
    for n in names:
        assert hasattr(lib, n), "libpeek.so does not export %s" % n


def test_binding_export_list_matches_header():
    from paper_2607_02525_b200 import binding
    assert sorted(binding.EXPORTS) == declared_functions()


def test_status_strings_and_version(lib):
    lib.peek_status_string.restype = ctypes.c_char_p
    lib.peek_status_string.argtypes = [ctypes.c_int32]
    assert lib.peek_status_string(0) == b"PEEK_OK"
    assert lib.peek_status_string(-3) == b"PEEK_ERR_WORKSPACE"
    assert lib.peek_status_string(-99) == b"PEEK_ERR_UNKNOWN"
    assert lib.peek_version() >= 100


def test_workspace_bytes_host_only(lib):
    out = ctypes.c_int64(0)
    f = lib.peek_workspace_bytes
    f.argtypes = [ctypes.c_int32] + [ctypes.c_int64] * 5 + [ctypes.POINTER(ctypes.c_int64)]
    prev = 0
    for call in range(4):
        assert f(call, 1 << 20, 0, 0, 1 << 23, 0, ctypes.byref(out)) == 0
        assert out.value >= 256 and out.value % 256 == 0
    for n in (1, 1000, 1 << 20):   # monotone in N
        assert f(2, n, 0, 0, 0, 0, ctypes.byref(out)) == 0
        assert out.value >= prev
        prev = out.value
    assert f(9, 1, 0, 0, 0, 0, ctypes.byref(out)) == -1
    assert f(0, -1, 0, 0, 0, 0, ctypes.byref(out)) == -1


def test_argument_errors_before_any_cuda_call(lib):
    vp, i64, i32, u64 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_uint64
    lib.peek_block_hash.argtypes = [vp, vp, i64, i32, u64, vp, vp, i64, vp, i64, vp]
    assert lib.peek_block_hash(None, None, -1, 16, 0, None, None, 0, None, 0, None) == -1
    assert lib.peek_block_hash(None, None, 4, 8, 0, None, None, 0, None, 0, None) == -5
    assert lib.peek_block_hash(None, None, 0, 16, 0, None, None, 0, None, 0, None) == 0
    assert lib.peek_block_hash(None, None, 4, 16, 0, None, None, 0, None, 0, None) == -1
    lib.peek_pending_tree.argtypes = [vp, vp, i64] + [vp] * 9 + [i64, vp]
    assert lib.peek_pending_tree(None, None, 0, None, None, None, None, None, None, None, None, None, 0, None) == 0
    assert lib.peek_pending_tree(None, None, 5, None, None, None, None, None, None, None, None, None, 0, None) == -1
    lib.peek_set_option.argtypes = [i32, i64]
    assert lib.peek_set_option(1, 2) == 0
    assert lib.peek_set_option(1, 0) == 0
    assert lib.peek_set_option(77, 0) == -1
    lib.peek_last_error.restype = ctypes.c_char_p
    assert b"peek_set_option" in lib.peek_last_error()


def test_binding_refuses_cpu_tensors():
    import torch
    from paper_2607_02525_b200 import binding
    with pytest.raises(binding.PeekError):
        binding.peek_block_hash(torch.zeros(16, dtype=torch.int32), torch.tensor([0, 16]), 1)


def test_next_row_calls_argument_errors(lib):
    """Host-side checks of the SURVEY 8(f) calls answer before any CUDA call."""
    vp, i64, i32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32
    dbl = ctypes.c_double
    lib.peek_clpm_signals.argtypes = [vp, vp, i64, vp, vp, vp, i32, vp, vp, vp, vp, vp, vp, i64, vp]
    assert lib.peek_clpm_signals(None, None, -1, None, None, None, 0, None, None, None, None, None, None, 0, None) == -1
    assert lib.peek_clpm_signals(None, None, 0, None, None, None, 0, None, None, None, None, None, None, 0, None) == 0
    lib.peek_clpm_order_full.argtypes = [vp, vp, vp, vp, vp, i64, vp, vp, i64, vp]
    assert lib.peek_clpm_order_full(None, None, None, None, None, 0, None, None, 0, None) == 0
    assert lib.peek_clpm_order_full(None, None, None, None, None, 3, None, None, 0, None) == -1
    lib.peek_clpm_group_major.argtypes = [vp, vp, i64, vp, vp, i64, vp]
    assert lib.peek_clpm_group_major(None, None, 3, None, None, 0, None) == -1
    lib.peek_clpm_lane_b.argtypes = [vp, vp, vp, i64, vp, vp, i64, vp]
    assert lib.peek_clpm_lane_b(None, None, None, 3, None, None, 0, None) == -1
    lib.peek_stride_interleave.argtypes = [vp, vp, i64, dbl, vp, vp, i64, vp]
    assert lib.peek_stride_interleave(None, None, 0, 0.7, None, None, 0, None) == 0
    assert lib.peek_stride_interleave(None, None, 4, 1.5, None, None, 0, None) == -1      # alpha outside [0, 1]
    assert lib.peek_stride_interleave(None, None, 4, float("nan"), None, None, 0, None) == -1
    lib.peek_dynamic_lane.argtypes = [vp, i64, dbl, dbl, vp, vp, i64, vp]
    assert lib.peek_dynamic_lane(None, 4, 0.0, 0.15, None, None, 0, None) == -1
    lib.peek_offline_phase1.argtypes = [vp, vp, i64, i32, vp, vp, vp, i64, vp]
    assert lib.peek_offline_phase1(None, None, 4, 0, None, None, None, 0, None) == -1     # depth_blocks 1..16
    assert lib.peek_offline_phase1(None, None, 4, 17, None, None, None, 0, None) == -1
    assert lib.peek_offline_phase1(None, None, 0, 8, None, None, None, 0, None) == 0
    lib.peek_radix_demand.argtypes = [vp, vp, i64, vp, vp, vp, vp]
    assert lib.peek_radix_demand(None, None, 4, None, None, None, None) == -1
    lib.peek_pending_tree_update.argtypes = [vp, vp, i64, i64, vp, vp, i64, vp] + [vp] * 8 + [vp, i64, vp]
    assert lib.peek_pending_tree_update(None, None, 4, 5, None, None, 0, None, *([None] * 8), None, 0, None) == -1  # M > N_new
    assert lib.peek_pending_tree_update(None, None, 0, 0, None, None, 0, None, *([None] * 8), None, 0, None) == 0
    out = ctypes.c_int64(0)
    f = lib.peek_workspace_bytes
    f.argtypes = [ctypes.c_int32] + [ctypes.c_int64] * 5 + [ctypes.POINTER(ctypes.c_int64)]
    for call in (4, 5, 6, 7):
        assert f(call, 1 << 16, 0, 0, 1 << 18, 0, ctypes.byref(out)) == 0 and out.value % 256 == 0
    assert f(8, 1 << 16, 1 << 16, 100, 0, 0, ctypes.byref(out)) == 0 and out.value >= 256
    assert f(8, 1 << 16, -1, 100, 0, 0, ctypes.byref(out)) == -1
