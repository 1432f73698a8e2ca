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
