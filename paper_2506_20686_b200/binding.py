"""ctypes binding of libtri_attn.so (include/tri_attn.h).  Argument marshalling only: every step of
the path runs in the library's CUDA kernels.  PyTorch is used for device memory and streams.

There is no CPU path and no fallback: if the shared library is missing, import of this module's
functions raises; if a call returns a non-zero tri_status, TriAttnError is raised.
"""
from __future__ import annotations

import ctypes
import os

import torch

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libtri_attn.so")

STARTING, ENDING = 0, 1
F32, BF16 = 0, 1

_lib = None

_vp, _sz, _i = ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int

SIGNATURES = {
    "tri_attn_fwd_workspace_bytes": (_sz, [_i] * 6),
    "tri_attn_bwd_workspace_bytes": (_sz, [_i] * 6),
    "tri_attn_fwd": (_i, [_vp] * 8 + [_i] * 6 + [_vp, _sz, _vp]),
    "tri_attn_bwd": (_i, [_vp] * 14 + [_i] * 6 + [_vp, _sz, _vp]),
    "tri_attn_rows_fwd_workspace_bytes": (_sz, [_i] * 6),
    "tri_attn_rows_bwd_workspace_bytes": (_sz, [_i] * 6),
    "tri_attn_rows_fwd": (_i, [_vp] * 8 + [_i] * 6 + [_vp, _sz, _vp]),
    "tri_attn_rows_bwd": (_i, [_vp] * 14 + [_i] * 6 + [_vp, _sz, _vp]),
    "tri_attn_noalloc_scratch_bytes": (_sz, []),
    "tri_attn_fwd_noalloc": (_i, [_vp] * 8 + [_i] * 6 + [_vp]),
    "tri_attn_dbias_reduce_scatter": (_i, [_vp, _i, _i, _vp, _i, _i, _i, _vp]),
    "tri_attn_bias_all_gather": (_i, [_vp, _i, _vp, _i, _i, _i, _i, _vp]),
    "tri_attn_step_host_arena_bytes": (_sz, [_i] * 6),
    "tri_attn_step_host": (_i, [_vp] * 14 + [_i] * 6 + [_vp, _sz, _vp]),
    "tri_attn_uses_tensor_cores": (_i, [_i] * 6),
    "tri_attn_launch_count": (ctypes.c_ulonglong, []),
    "tri_attn_profile_begin": (None, []),
    "tri_attn_profile_end": (_i, [ctypes.c_char_p, _sz]),
    "tri_status_string": (ctypes.c_char_p, [_i]),
    "tri_attn_last_cuda_error": (ctypes.c_char_p, []),
}


class TriAttnError(RuntimeError):
    pass


def load():
    """dlopen the in-tree library (built by paper_2506_20686_b200/build.py).  Fails loudly."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise TriAttnError(f"{LIB_PATH} not built: run `python -m paper_2506_20686_b200.build` "
                               "or __graft_entry__.build(); there is no fallback path")
        lib = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


def _check(status: int):
    if status != 0:
        lib = load()
        msg = lib.tri_status_string(status).decode()
        if status == 4:
            msg += " [" + lib.tri_attn_last_cuda_error().decode() + "]"
        raise TriAttnError(msg)


def _dtype_code(t: torch.Tensor) -> int:
    if t.dtype == torch.float32:
        return F32
    if t.dtype == torch.bfloat16:
        return BF16
    raise TriAttnError(f"unsupported dtype {t.dtype}")


def _ptr(t):
    return None if t is None else t.data_ptr()


def _dims(Q):
    B, N, H, N2, d = Q.shape
    if N != N2:
        raise TriAttnError("Q must be [B,N,H,N,d]")
    return B, N, H, d


def _chk(t, shape, dtype, name, device=None):
    if t is None:
        return
    if tuple(t.shape) != tuple(shape) or t.dtype != dtype or not t.is_contiguous():
        raise TriAttnError(f"{name}: expected contiguous {tuple(shape)} {dtype}, got {tuple(t.shape)} {t.dtype}")
    if device is not None and t.device != device:
        raise TriAttnError(f"{name}: wrong device {t.device}")


def fwd_workspace_bytes(B, N, H, d, variant, dtype_code) -> int:
    return int(load().tri_attn_fwd_workspace_bytes(B, N, H, d, variant, dtype_code))


def bwd_workspace_bytes(B, N, H, d, variant, dtype_code) -> int:
    return int(load().tri_attn_bwd_workspace_bytes(B, N, H, d, variant, dtype_code))


def uses_tensor_cores(B, N, H, d, variant, dtype_code) -> bool:
    return bool(load().tri_attn_uses_tensor_cores(B, N, H, d, variant, dtype_code))


def launch_count() -> int:
    return int(load().tri_attn_launch_count())


def profile_begin() -> None:
    """Start bracketing every kernel the library launches with CUDA events (bench roofline leg)."""
    load().tri_attn_profile_begin()


def profile_end() -> dict:
    """Stop, synchronise the events and return {kernel_name: (launches, total_ms)}."""
    buf = ctypes.create_string_buffer(1 << 14)
    n = load().tri_attn_profile_end(buf, len(buf))
    if n < 0:
        raise TriAttnError("tri_attn_profile_end: CUDA error")
    out = {}
    for line in buf.value.decode().splitlines():
        name, cnt, ms = line.split()
        out[name] = (int(cnt), float(ms))
    return out


def _workspace(nbytes, device, workspace):
    if workspace is None:
        workspace = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=device)
    return workspace


def tri_attn_fwd(Q, K, V, G, bias, mask=None, variant=STARTING, O=None, LSE=None, workspace=None):
    """O, LSE = forward.  All tensors CUDA, contiguous (see include/tri_attn.h for layouts)."""
    lib = load()
    if not Q.is_cuda:
        raise TriAttnError("tri_attn_fwd needs CUDA tensors (there is no CPU path)")
    B, N, H, d = _dims(Q)
    dt, dev = Q.dtype, Q.device
    for t, n in ((K, "K"), (V, "V"), (G, "G")):
        _chk(t, Q.shape, dt, n, dev)
    _chk(Q, Q.shape, dt, "Q", dev)
    _chk(bias, (B, H, N, N), dt, "bias", dev)
    _chk(mask, (B, N, N), torch.uint8, "mask", dev)
    if O is None:
        O = torch.empty_like(Q)
    if LSE is None:
        LSE = torch.empty((B, N, H, N), dtype=torch.float32, device=dev)
    _chk(O, Q.shape, dt, "O", dev)
    _chk(LSE, (B, N, H, N), torch.float32, "LSE", dev)
    code = _dtype_code(Q)
    need = fwd_workspace_bytes(B, N, H, d, variant, code)
    ws = _workspace(need, dev, workspace)
    with torch.cuda.device(dev):
        stream = torch.cuda.current_stream().cuda_stream
        _check(lib.tri_attn_fwd(_ptr(Q), _ptr(K), _ptr(V), _ptr(G), _ptr(bias), _ptr(mask), _ptr(O), _ptr(LSE),
                                B, N, H, d, variant, code, _ptr(ws), ws.numel(), stream))
    return O, LSE


def tri_attn_bwd(dO, Q, K, V, G, bias, mask, O, LSE, variant=STARTING, out=None, workspace=None):
    """dQ, dK, dV, dG, dBias = backward.  `out` may carry preallocated (dQ,dK,dV,dG,dBias)."""
    lib = load()
    if not Q.is_cuda:
        raise TriAttnError("tri_attn_bwd needs CUDA tensors (there is no CPU path)")
    B, N, H, d = _dims(Q)
    dt, dev = Q.dtype, Q.device
    for t, n in ((dO, "dO"), (Q, "Q"), (K, "K"), (V, "V"), (G, "G"), (O, "O")):
        _chk(t, Q.shape, dt, n, dev)
    _chk(bias, (B, H, N, N), dt, "bias", dev)
    _chk(mask, (B, N, N), torch.uint8, "mask", dev)
    _chk(LSE, (B, N, H, N), torch.float32, "LSE", dev)
    if out is None:
        out = tuple(torch.empty_like(Q) for _ in range(4)) + (
            torch.empty((B, H, N, N), dtype=torch.float32, device=dev),)
    dQ, dK, dV, dG, dBias = out
    for t, n in ((dQ, "dQ"), (dK, "dK"), (dV, "dV"), (dG, "dG")):
        _chk(t, Q.shape, dt, n, dev)
    _chk(dBias, (B, H, N, N), torch.float32, "dBias", dev)
    code = _dtype_code(Q)
    need = bwd_workspace_bytes(B, N, H, d, variant, code)
    ws = _workspace(need, dev, workspace)
    with torch.cuda.device(dev):
        stream = torch.cuda.current_stream().cuda_stream
        _check(lib.tri_attn_bwd(_ptr(dO), _ptr(Q), _ptr(K), _ptr(V), _ptr(G), _ptr(bias), _ptr(mask), _ptr(O),
                                _ptr(LSE), _ptr(dQ), _ptr(dK), _ptr(dV), _ptr(dG), _ptr(dBias),
                                B, N, H, d, variant, code, _ptr(ws), ws.numel(), stream))
    return dQ, dK, dV, dG, dBias


def rows_fwd_workspace_bytes(B, R, N, H, d, dtype_code) -> int:
    return int(load().tri_attn_rows_fwd_workspace_bytes(B, R, N, H, d, dtype_code))


def rows_bwd_workspace_bytes(B, R, N, H, d, dtype_code) -> int:
    return int(load().tri_attn_rows_bwd_workspace_bytes(B, R, N, H, d, dtype_code))


def tri_attn_rows_fwd(Q, K, V, G, bias, mask=None, O=None, LSE=None, workspace=None):
    """O, LSE = forward with a decoupled row count: Q,K,V,G [B,R,H,N,d], bias [B,H,N,N], mask [B,R,N] (starting node)."""
    lib = load()
    if not Q.is_cuda:
        raise TriAttnError("tri_attn_rows_fwd needs CUDA tensors (there is no CPU path)")
    B, R, H, N, d = Q.shape
    dt, dev = Q.dtype, Q.device
    for t, n in ((Q, "Q"), (K, "K"), (V, "V"), (G, "G")):
        _chk(t, Q.shape, dt, n, dev)
    _chk(bias, (B, H, N, N), dt, "bias", dev)
    _chk(mask, (B, R, N), torch.uint8, "mask", dev)
    if O is None:
        O = torch.empty_like(Q)
    if LSE is None:
        LSE = torch.empty((B, R, H, N), dtype=torch.float32, device=dev)
    _chk(O, Q.shape, dt, "O", dev)
    _chk(LSE, (B, R, H, N), torch.float32, "LSE", dev)
    code = _dtype_code(Q)
    need = rows_fwd_workspace_bytes(B, R, N, H, d, code)
    ws = _workspace(need, dev, workspace)
    with torch.cuda.device(dev):
        stream = torch.cuda.current_stream().cuda_stream
        _check(lib.tri_attn_rows_fwd(_ptr(Q), _ptr(K), _ptr(V), _ptr(G), _ptr(bias), _ptr(mask), _ptr(O), _ptr(LSE),
                                     B, R, N, H, d, code, _ptr(ws), ws.numel(), stream))
    return O, LSE


def tri_attn_rows_bwd(dO, Q, K, V, G, bias, mask, O, LSE, out=None, workspace=None):
    """dQ, dK, dV, dG, dBias = backward of tri_attn_rows_fwd; dBias [B,H,N,N] fp32 sums over the R rows."""
    lib = load()
    if not Q.is_cuda:
        raise TriAttnError("tri_attn_rows_bwd needs CUDA tensors (there is no CPU path)")
    B, R, H, N, d = Q.shape
    dt, dev = Q.dtype, Q.device
    for t, n in ((dO, "dO"), (Q, "Q"), (K, "K"), (V, "V"), (G, "G"), (O, "O")):
        _chk(t, Q.shape, dt, n, dev)
    _chk(bias, (B, H, N, N), dt, "bias", dev)
    _chk(mask, (B, R, N), torch.uint8, "mask", dev)
    _chk(LSE, (B, R, H, N), torch.float32, "LSE", dev)
    if out is None:
        out = tuple(torch.empty_like(Q) for _ in range(4)) + (
            torch.empty((B, H, N, N), dtype=torch.float32, device=dev),)
    dQ, dK, dV, dG, dBias = out
    for t, n in ((dQ, "dQ"), (dK, "dK"), (dV, "dV"), (dG, "dG")):
        _chk(t, Q.shape, dt, n, dev)
    _chk(dBias, (B, H, N, N), torch.float32, "dBias", dev)
    code = _dtype_code(Q)
    need = rows_bwd_workspace_bytes(B, R, N, H, d, code)
    ws = _workspace(need, dev, workspace)
    with torch.cuda.device(dev):
        stream = torch.cuda.current_stream().cuda_stream
        _check(lib.tri_attn_rows_bwd(_ptr(dO), _ptr(Q), _ptr(K), _ptr(V), _ptr(G), _ptr(bias), _ptr(mask), _ptr(O),
                                     _ptr(LSE), _ptr(dQ), _ptr(dK), _ptr(dV), _ptr(dG), _ptr(dBias),
                                     B, R, N, H, d, code, _ptr(ws), ws.numel(), stream))
    return dQ, dK, dV, dG, dBias


def noalloc_scratch_bytes() -> int:
    """Size of the library's built-in scratch array: the limit of tri_attn_fwd_noalloc."""
    return int(load().tri_attn_noalloc_scratch_bytes())


def tri_attn_fwd_noalloc(Q, K, V, G, bias, mask, variant, O, LSE):
    """Forward into the caller's O, LSE with the scratch in the library's built-in device array: nothing is allocated,
    here or in the library (every tensor, outputs included, comes from the caller).  See include/tri_attn.h for the
    size limit and for why overlapping calls race."""
    lib = load()
    if not Q.is_cuda:
        raise TriAttnError("tri_attn_fwd_noalloc needs CUDA tensors (there is no CPU path)")
    B, N, H, d = _dims(Q)
    dt, dev = Q.dtype, Q.device
    for t, n in ((Q, "Q"), (K, "K"), (V, "V"), (G, "G"), (O, "O")):
        _chk(t, Q.shape, dt, n, dev)
    _chk(bias, (B, H, N, N), dt, "bias", dev)
    _chk(mask, (B, N, N), torch.uint8, "mask", dev)
    _chk(LSE, (B, N, H, N), torch.float32, "LSE", dev)
    if O is None or LSE is None:
        raise TriAttnError("tri_attn_fwd_noalloc: O and LSE must be preallocated by the caller")
    with torch.cuda.device(dev):
        stream = torch.cuda.current_stream().cuda_stream
        _check(lib.tri_attn_fwd_noalloc(_ptr(Q), _ptr(K), _ptr(V), _ptr(G), _ptr(bias), _ptr(mask), _ptr(O), _ptr(LSE),
                                        B, N, H, d, variant, _dtype_code(Q), stream))
    return O, LSE


def tri_attn_bias_all_gather(peer_ptrs, B, H, N, dtype, out=None, device=None):
    """bias [B,H,N,N] assembled from the P ranks' shards [B,H,N/P,N] (device pointers in rank order), by pulling."""
    lib = load()
    P = len(peer_ptrs)
    if P == 0 or N % P:
        raise TriAttnError(f"N={N} is not a multiple of the group size {P}")
    dev = torch.device("cuda", torch.cuda.current_device()) if device is None else device
    if out is None:
        out = torch.empty((B, H, N, N), dtype=dtype, device=dev)
    _chk(out, (B, H, N, N), dtype, "out", dev)
    arr = (ctypes.c_void_p * P)(*[int(p) for p in peer_ptrs])
    with torch.cuda.device(dev):
        stream = torch.cuda.current_stream().cuda_stream
        _check(lib.tri_attn_bias_all_gather(ctypes.cast(arr, ctypes.c_void_p), P, _ptr(out), B, H, N, _dtype_code(out), stream))
    return out


def tri_attn_dbias_reduce_scatter(peer_ptrs, rank, B, H, N, out=None, device=None):
    """out[b,h,l,k] = sum over the ranks (ascending) of their partial dBias lines rank*N/P + l.  peer_ptrs: the P device
    pointers (ints) of the ranks' [B,H,N,N] fp32 partial dBias buffers, in rank order (see include/tri_attn.h)."""
    lib = load()
    P = len(peer_ptrs)
    if P == 0 or N % P:
        raise TriAttnError(f"N={N} is not a multiple of the group size {P}")
    dev = torch.device("cuda", torch.cuda.current_device()) if device is None else device
    if out is None:
        out = torch.empty((B, H, N // P, N), dtype=torch.float32, device=dev)
    _chk(out, (B, H, N // P, N), torch.float32, "out", dev)
    arr = (ctypes.c_void_p * P)(*[int(p) for p in peer_ptrs])
    with torch.cuda.device(dev):
        stream = torch.cuda.current_stream().cuda_stream
        _check(lib.tri_attn_dbias_reduce_scatter(ctypes.cast(arr, ctypes.c_void_p), P, rank, _ptr(out), B, H, N, stream))
    return out


def step_host_arena_bytes(B, N, H, d, variant, dtype_code) -> int:
    return int(load().tri_attn_step_host_arena_bytes(B, N, H, d, variant, dtype_code))


def tri_attn_step_host(hin: dict, hout: dict, variant, arena):
    """End-to-end step on HOST (pinned) tensors.  hin: Q,K,V,G,bias,mask(optional),dO; hout: O,LSE,dQ,dK,dV,dG,
    dBias (all CPU tensors).  `arena` is a CUDA uint8 tensor of step_host_arena_bytes().  Asynchronous on the
    current stream of arena's device."""
    lib = load()
    Q = hin["Q"]
    B, N, H, d = _dims(Q)
    code = _dtype_code(Q)
    for k in ("Q", "K", "V", "G", "dO"):
        _chk(hin[k], Q.shape, Q.dtype, k)
        assert not hin[k].is_cuda
    _chk(hin["bias"], (B, H, N, N), Q.dtype, "bias")
    _chk(hin.get("mask"), (B, N, N), torch.uint8, "mask")
    for k in ("O", "dQ", "dK", "dV", "dG"):
        _chk(hout[k], Q.shape, Q.dtype, k)
    _chk(hout["LSE"], (B, N, H, N), torch.float32, "LSE")
    _chk(hout["dBias"], (B, H, N, N), torch.float32, "dBias")
    with torch.cuda.device(arena.device):
        stream = torch.cuda.current_stream().cuda_stream
        _check(lib.tri_attn_step_host(
            _ptr(hin["Q"]), _ptr(hin["K"]), _ptr(hin["V"]), _ptr(hin["G"]), _ptr(hin["bias"]), _ptr(hin.get("mask")),
            _ptr(hin["dO"]), _ptr(hout["O"]), _ptr(hout["LSE"]), _ptr(hout["dQ"]), _ptr(hout["dK"]),
            _ptr(hout["dV"]), _ptr(hout["dG"]), _ptr(hout["dBias"]),
            B, N, H, d, variant, code, _ptr(arena), arena.numel(), stream))
