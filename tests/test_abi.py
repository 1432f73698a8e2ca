"""CPU-side checks of the boundary: the library loads, exports every symbol include/tri_attn.h declares,
validates arguments before any launch, and reports O(N^2) workspace sizes.  No compute calls."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2506_20686_b200 import build as b

    b.build()
    from paper_2506_20686_b200 import binding

    return binding.load()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "tri_attn.h")).read()
    return sorted(set(re.findall(r"TRI_API[^;(]*?\b(tri_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_expected_entry_points():
    syms = declared_symbols()
    for s in ("tri_attn_fwd", "tri_attn_bwd", "tri_attn_fwd_workspace_bytes", "tri_attn_bwd_workspace_bytes",
              "tri_attn_step_host", "tri_status_string"):
        assert s in syms


def test_library_exports_every_declared_symbol(lib):
    from paper_2506_20686_b200 import binding

    for s in declared_symbols():
        assert hasattr(lib, s), s
        assert s in binding.SIGNATURES, f"binding lacks {s}"


def test_argument_validation_happens_before_any_launch(lib):
    n0 = lib.tri_attn_launch_count()
    # null pointers
    assert lib.tri_attn_fwd(None, None, None, None, None, None, None, None, 1, 32, 4, 32, 0, 0, None, 0, None) == 1
    # bad sizes / enums
    p = ctypes.c_void_p(4096)
    assert lib.tri_attn_fwd(p, p, p, p, p, None, p, p, 0, 32, 4, 32, 0, 0, p, 1 << 20, None) == 1
    assert lib.tri_attn_fwd(p, p, p, p, p, None, p, p, 1, 32, 4, 32, 7, 0, p, 1 << 20, None) == 1
    # misaligned
    q = ctypes.c_void_p(4100)
    assert lib.tri_attn_fwd(q, p, p, p, p, None, p, p, 1, 32, 4, 32, 0, 0, p, 1 << 20, None) == 1
    # unsupported head dim
    assert lib.tri_attn_fwd(p, p, p, p, p, None, p, p, 1, 32, 4, 48, 0, 0, p, 1 << 20, None) == 2
    # workspace too small / null
    assert lib.tri_attn_bwd(*([p] * 5), p, None, p, p, p, p, p, p, p, 1, 32, 4, 32, 0, 0, None, 0, None) == 3
    assert lib.tri_attn_bwd(*([p] * 5), p, None, p, p, p, p, p, p, p, 1, 32, 4, 32, 0, 0, p, 16, None) == 3
    assert lib.tri_attn_launch_count() == n0
    assert b"TRI_OK" in lib.tri_status_string(0)
    assert b"UNSUPPORTED" in lib.tri_status_string(2)


def test_overlapping_outputs_are_rejected_before_any_launch(lib):
    """include/tri_attn.h: outputs (and the workspace) must not overlap inputs or each other -> TRI_ERR_INVALID_ARG."""
    n0 = lib.tri_attn_launch_count()
    B, N, H, d = 1, 32, 4, 32
    U = B * N * H * N * d * 4
    base = 1 << 30
    a = [ctypes.c_void_p(base + i * (U + 4096)) for i in range(16)]  # fake, disjoint, aligned device addresses
    ws = ctypes.c_void_p(base + 20 * (U + 4096))
    wsb = 1 << 24
    # O aliases Q
    assert lib.tri_attn_fwd(a[0], a[1], a[2], a[3], a[4], None, a[0], a[6], B, N, H, d, 0, 0, ws, wsb, None) == 1
    # LSE inside V
    assert lib.tri_attn_fwd(a[0], a[1], a[2], a[3], a[4], None, a[5], ctypes.c_void_p(a[2].value + 64), B, N, H, d, 0, 0, ws, wsb, None) == 1
    # workspace overlaps K
    assert lib.tri_attn_fwd(a[0], a[1], a[2], a[3], a[4], None, a[5], a[6], B, N, H, d, 0, 0, a[1], wsb, None) == 1
    # backward: dK aliases dQ; dG aliases dO
    args = [a[0], a[1], a[2], a[3], a[4], a[5], None, a[6], a[7]]
    assert lib.tri_attn_bwd(*args, a[8], a[8], a[10], a[11], a[12], B, N, H, d, 0, 0, ws, wsb, None) == 1
    assert lib.tri_attn_bwd(*args, a[8], a[9], a[10], a[0], a[12], B, N, H, d, 0, 0, ws, wsb, None) == 1
    assert lib.tri_attn_launch_count() == n0


def test_tensor_core_path_query(lib):
    assert lib.tri_attn_uses_tensor_cores(2, 768, 4, 32, 0, 1) == 1
    assert lib.tri_attn_uses_tensor_cores(1, 200, 4, 32, 0, 1) == 1   # N % 8 == 0 is enough (partial tiles are masked)
    assert lib.tri_attn_uses_tensor_cores(1, 204, 4, 32, 0, 1) == 0   # N % 8 != 0: CUDA-core kernels
    assert lib.tri_attn_uses_tensor_cores(1, 120, 4, 32, 0, 1) == 0   # N < 128: CUDA-core kernels
    assert lib.tri_attn_uses_tensor_cores(1, 128, 4, 64, 0, 1) == 0   # d != 32
    assert lib.tri_attn_uses_tensor_cores(1, 128, 4, 32, 0, 0) == 0   # fp32 (reading A14)


@pytest.mark.parametrize("dtype", [0, 1])
@pytest.mark.parametrize("variant", [0, 1])
def test_workspace_is_quadratic_not_cubic(lib, variant, dtype):
    B, H, d = 1, 4, 32
    for N in (128, 384, 768, 1024):
        for fn in (lib.tri_attn_fwd_workspace_bytes, lib.tri_attn_bwd_workspace_bytes):
            w = fn(B, N, H, d, variant, dtype)
            assert w >= 256
            # O(N^2 H) with a small constant: per (b,h,q,k) element dA 2d = 64 B, D 4 B, bias^T 2 B, <= 8 dBias planes 32 B
            assert w <= 128 * B * H * N * N + (1 << 20), (N, w)
            assert w < B * H * N * N * N * 2 or N <= 128                # far below the bf16 map
    assert lib.tri_attn_fwd_workspace_bytes(0, 1, 1, 32, 0, 0) == 0


def test_binding_refuses_cpu_tensors(lib):
    import torch

    from paper_2506_20686_b200 import TriAttnError, tri_attn_fwd

    x = torch.zeros(1, 4, 1, 4, 32)
    with pytest.raises(TriAttnError):
        tri_attn_fwd(x, x, x, x, torch.zeros(1, 1, 4, 4))


def test_rows_and_peer_entry_points_validate_before_any_launch(lib):
    """The newer entry points (rows, no-alloc, peer reduce-scatter) reject bad arguments without a GPU and without a launch."""
    n0 = lib.tri_attn_launch_count()
    p = ctypes.c_void_p(4096)
    # rows: unsupported dtype / head dim / N not a multiple of 8 -> workspace 0 and TRI_ERR_UNSUPPORTED; bad R -> invalid
    assert lib.tri_attn_rows_fwd_workspace_bytes(1, 8, 128, 2, 32, 0) == 0
    assert lib.tri_attn_rows_fwd_workspace_bytes(1, 8, 132, 2, 32, 1) == 0
    assert lib.tri_attn_rows_fwd_workspace_bytes(1, 1, 128, 2, 32, 1) > 0          # any R >= 1
    assert lib.tri_attn_rows_bwd_workspace_bytes(1, 8, 16384, 1, 32, 1) == 0       # backward stops at N = 8192 ...
    assert lib.tri_attn_rows_fwd_workspace_bytes(1, 8, 16384, 1, 32, 1) > 0        # ... the forward at 16384
    assert lib.tri_attn_rows_fwd(p, p, p, p, p, None, p, p, 1, 0, 128, 2, 32, 1, p, 1 << 20, None) == 1
    assert lib.tri_attn_rows_fwd(p, p, p, p, p, None, p, p, 1, 8, 128, 2, 64, 1, p, 1 << 20, None) == 2
    assert lib.tri_attn_rows_bwd(*([p] * 6), None, *([p] * 7), 1, 8, 128, 2, 32, 1, None, 0, None) == 3
    # peer reduce-scatter
    arr = (ctypes.c_void_p * 3)(4096, 8192, 12288)
    ptrs = ctypes.cast(arr, ctypes.c_void_p)
    assert lib.tri_attn_dbias_reduce_scatter(None, 3, 0, p, 1, 2, 384, None) == 1
    assert lib.tri_attn_dbias_reduce_scatter(ptrs, 3, 3, p, 1, 2, 384, None) == 1      # rank outside the group
    assert lib.tri_attn_dbias_reduce_scatter(ptrs, 3, 0, p, 1, 2, 400, None) == 2      # N % P != 0
    assert lib.tri_attn_dbias_reduce_scatter(ptrs, 17, 0, p, 1, 2, 17 * 16, None) == 2  # more than 16 peers
    assert lib.tri_attn_bias_all_gather(None, 3, p, 1, 2, 384, 1, None) == 1
    assert lib.tri_attn_bias_all_gather(ptrs, 3, p, 1, 2, 400, 1, None) == 2           # N % P != 0
    assert lib.tri_attn_bias_all_gather(ptrs, 3, p, 1, 2, 384, 7, None) == 1           # bad dtype
    arr_bad = (ctypes.c_void_p * 3)(4096, 8200, 12288)
    assert lib.tri_attn_dbias_reduce_scatter(ctypes.cast(arr_bad, ctypes.c_void_p), 3, 0, p, 1, 2, 384, None) == 1  # misaligned peer
    assert lib.tri_attn_launch_count() == n0
