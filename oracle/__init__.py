"""CPU fp64 oracle for triangle attention with pair bias -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin numpy/ctypes wrapper around ``tri_attn_oracle.c`` (plain C, fp64, the definition of
PAPER.md Table I P:L504-514 written out; see that file's header for the citations and layouts).
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tri_attn_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

STARTING, ENDING = 0, 1


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (-O2 -fopenmp) next to its source."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.tri_oracle_num_threads.restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(_load().tri_oracle_num_threads())


def _d(x):
    return np.ascontiguousarray(x, dtype=np.float64)


def _p(x):
    return None if x is None else x.ctypes.data_as(ctypes.c_void_p)


def _m(mask):
    return None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)


def fwd_start_general(Q, K, V, G, bias, mask=None, return_P=False):
    """Starting-node forward on decoupled shapes.  Q,G:[B,R,H,Nq,d] K,V:[B,R,H,Nk,d]
    bias:[B,H,Nq,Nk] mask:[B,R,Nk] (keep flags).  Returns O, LSE (and P [B,R,H,Nq,Nk])."""
    Q, K, V, G, bias, mask = _d(Q), _d(K), _d(V), _d(G), _d(bias), _m(mask)
    B, R, H, Nq, d = Q.shape
    Nk = K.shape[3]
    assert K.shape == (B, R, H, Nk, d) and V.shape == K.shape and G.shape == Q.shape
    assert bias.shape == (B, H, Nq, Nk) and (mask is None or mask.shape == (B, R, Nk))
    O = np.empty_like(Q)
    LSE = np.empty((B, R, H, Nq), np.float64)
    P = np.empty((B, R, H, Nq, Nk), np.float64) if return_P else None
    rc = _load().tri_oracle_fwd_start(_p(Q), _p(K), _p(V), _p(G), _p(bias), _p(mask), B, R, H, Nq,
                                      Nk, d, _p(O), _p(LSE), _p(P))
    assert rc == 0
    return (O, LSE, P) if return_P else (O, LSE)


def bwd_start_general(dO, Q, K, V, G, bias, mask=None):
    """Starting-node backward on decoupled shapes.  Returns dQ, dK, dV, dG, dBias."""
    dO, Q, K, V, G, bias, mask = _d(dO), _d(Q), _d(K), _d(V), _d(G), _d(bias), _m(mask)
    B, R, H, Nq, d = Q.shape
    Nk = K.shape[3]
    assert dO.shape == Q.shape
    dQ, dG = np.empty_like(Q), np.empty_like(Q)
    dK, dV = np.empty_like(K), np.empty_like(K)
    dBias = np.empty((B, H, Nq, Nk), np.float64)
    rc = _load().tri_oracle_bwd_start(_p(dO), _p(Q), _p(K), _p(V), _p(G), _p(bias), _p(mask), B, R,
                                      H, Nq, Nk, d, _p(dQ), _p(dK), _p(dV), _p(dG), _p(dBias))
    assert rc == 0
    return dQ, dK, dV, dG, dBias


def fwd(Q, K, V, G, bias, mask=None, variant=STARTING, return_P=False):
    """The paper's square operator.  All of Q,K,V,G: [B,N,H,N,d]; bias [B,H,N,N]; mask [B,N,N]."""
    if variant == STARTING:
        return fwd_start_general(Q, K, V, G, bias, mask, return_P)
    Q, K, V, G, bias, mask = _d(Q), _d(K), _d(V), _d(G), _d(bias), _m(mask)
    B, N, H, N2, d = Q.shape
    assert N == N2 and K.shape == Q.shape and bias.shape == (B, H, N, N)
    O = np.empty_like(Q)
    LSE = np.empty((B, N, H, N), np.float64)
    P = np.empty((B, N, H, N, N), np.float64) if return_P else None
    rc = _load().tri_oracle_fwd_end(_p(Q), _p(K), _p(V), _p(G), _p(bias), _p(mask), B, N, H, d,
                                    _p(O), _p(LSE), _p(P))
    assert rc == 0
    return (O, LSE, P) if return_P else (O, LSE)


def bwd(dO, Q, K, V, G, bias, mask=None, variant=STARTING):
    if variant == STARTING:
        return bwd_start_general(dO, Q, K, V, G, bias, mask)
    dO, Q, K, V, G, bias, mask = _d(dO), _d(Q), _d(K), _d(V), _d(G), _d(bias), _m(mask)
    B, N, H, _, d = Q.shape
    dQ, dK, dV, dG = (np.empty_like(Q) for _ in range(4))
    dBias = np.empty((B, H, N, N), np.float64)
    rc = _load().tri_oracle_bwd_end(_p(dO), _p(Q), _p(K), _p(V), _p(G), _p(bias), _p(mask), B, N, H,
                                    d, _p(dQ), _p(dK), _p(dV), _p(dG), _p(dBias))
    assert rc == 0
    return dQ, dK, dV, dG, dBias
