"""tri_attn_fwd_noalloc (include/tri_attn.h): the forward with its scratch in the library's built-in device array, for
callers that cannot allocate.  Collected last on purpose (the suite runs with pytest -x).  The GPU test compares the
new entry point with the existing workspace path (tri_attn_fwd) on calls made one after another, so that each call finds
the previous call's contents in the shared array; it passes alone in a fresh process and after the other tests."""
import ctypes
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import parity_util as pu  # noqa: E402
import tri_inputs  # noqa: E402
from tri_inputs import ENDING, STARTING  # noqa: E402


@pytest.fixture(scope="module")
def tri():
    import paper_2506_20686_b200 as t
    from paper_2506_20686_b200 import build as b

    b.build()
    t.load()
    return t


def test_noalloc_rejects_problems_beyond_the_built_in_scratch(tri):
    """No GPU needed: the size check comes before any CUDA call.  bf16 d=32 N=2048 H=4 needs 67 MB of fp32 bias planes."""
    lib = tri.load()
    assert tri.noalloc_scratch_bytes() == 32 << 20
    assert tri.fwd_workspace_bytes(1, 2048, 4, 32, STARTING, tri.BF16) > tri.noalloc_scratch_bytes()
    p = ctypes.c_void_p(4096)
    n0 = tri.launch_count()
    assert lib.tri_attn_fwd_noalloc(p, p, p, p, p, None, p, p, 1, 2048, 4, 32, STARTING, tri.BF16, None) == 5
    assert b"TOO_LARGE" in lib.tri_status_string(5)
    # bad arguments keep tri_attn_fwd's codes, before any launch
    assert lib.tri_attn_fwd_noalloc(None, p, p, p, p, None, p, p, 1, 128, 4, 32, STARTING, tri.BF16, None) == 1
    assert lib.tri_attn_fwd_noalloc(p, p, p, p, p, None, p, p, 1, 128, 4, 48, STARTING, tri.BF16, None) == 2
    assert tri.launch_count() == n0


@pytest.mark.gpu
def test_noalloc_forward_matches_the_workspace_path_on_calls_in_a_row(tri):
    import torch

    cases = [
        tri_inputs.small_config(2, 256, 2, 32, "bf16", STARTING, 1.5, "random:9", seed=801),   # tensor-core path, mask words
        tri_inputs.small_config(1, 384, 3, 32, "bf16", ENDING, 1.0, "none", seed=802),         # other planes, no mask
        tri_inputs.small_config(2, 200, 2, 32, "bf16", STARTING, 1.0, "none", seed=803),       # partial tiles: synthesised mask
        tri_inputs.small_config(2, 40, 3, 16, "f32", ENDING, 1.0, "lengths:33,40", seed=804),  # CUDA-core path
    ]
    probs = []
    for cfg in cases:
        x = tri_inputs.make_inputs(cfg)
        g = pu.gpu_inputs(x, cfg.dtype)
        O_ref, LSE_ref = tri.tri_attn_fwd(g["Q"], g["K"], g["V"], g["G"], g["bias"], g["mask"], cfg.variant)
        probs.append((cfg, g, O_ref, LSE_ref, torch.empty_like(O_ref), torch.empty_like(LSE_ref)))
    torch.cuda.synchronize()
    # two rounds over the cases, back to back on one stream: every call starts from the previous call's scratch contents
    for rnd in range(2):
        for cfg, g, O_ref, LSE_ref, O, LSE in probs:
            O.fill_(float("nan"))
            LSE.fill_(float("nan"))
            before = torch.cuda.memory_allocated()
            tri.tri_attn_fwd_noalloc(g["Q"], g["K"], g["V"], g["G"], g["bias"], g["mask"], cfg.variant, O, LSE)
            assert torch.cuda.memory_allocated() == before
            torch.cuda.synchronize()
            tol = pu.TOL[cfg.dtype]
            eo = pu.rel_err(O.float().cpu().numpy(), O_ref.float().cpu().numpy())
            el = pu.rel_err(LSE.cpu().numpy(), LSE_ref.cpu().numpy())
            assert eo <= tol and el <= tol, (rnd, cfg.name, eo, el)
            # same kernels, same order of operations: in fact bitwise equal
            assert torch.equal(O.view(torch.uint8), O_ref.view(torch.uint8)), (rnd, cfg.name)
            assert np.array_equal(LSE.cpu().numpy(), LSE_ref.cpu().numpy()), (rnd, cfg.name)


@pytest.mark.gpu
def test_noalloc_size_limit_through_the_binding(tri):
    """cfg4's forward scratch (19 MB) fits; a problem beyond 32 MiB raises a clear error without touching the GPU."""
    import torch

    assert tri.fwd_workspace_bytes(2, 768, 4, 32, STARTING, tri.BF16) <= tri.noalloc_scratch_bytes()
    B, N, H, d = 3, 1024, 4, 32  # 3 x 4 x 1024 x 1024 x 4 B = 50 MB of bias planes
    assert tri.fwd_workspace_bytes(B, N, H, d, STARTING, tri.BF16) > tri.noalloc_scratch_bytes()
    q = torch.zeros((B, N, H, N, d), dtype=torch.bfloat16, device="cuda")
    bias = torch.zeros((B, H, N, N), dtype=torch.bfloat16, device="cuda")
    lse = torch.empty((B, N, H, N), dtype=torch.float32, device="cuda")
    with pytest.raises(tri.TriAttnError, match="TOO_LARGE"):
        tri.tri_attn_fwd_noalloc(q, q, q, q, bias, None, STARTING, torch.empty_like(q), lse)
