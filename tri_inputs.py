"""Seeded synthetic inputs for triangle attention (shared by the oracle-side tests and the CUDA side).

This module holds NONE of the method's arithmetic: it only draws random tensors with the shapes,
value distributions and mask structure of BASELINE.json's five configs (stand-ins for the paper's
PDB workload, which is not available), and rounds them to the storage dtype once
(SURVEY.md Sec. 8(c) reading A13) so the oracle and the GPU see bit-identical values.

Generation order: Q, K, V, G, bias, dO, then mask.  RNG: numpy Philox
(counter-based) keyed by the config's seed; float32 standard normals; bias multiplied by sigma
(reading A12: "N(0,s)" means std s).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

STARTING, ENDING = 0, 1


@dataclass(frozen=True)
class Config:
    name: str
    B: int
    N: int
    H: int
    d: int
    dtype: str  # "f32" | "bf16"
    variant: int
    sigma_bias: float
    mask: str  # "none" | "tail:<n>" | "lengths:<l0>,<l1>,..." | "random:<n>"
    seed: int


# BASELINE.json configs[0..4] (CFG1..CFG5 in SURVEY.md, 1-based).  CFG3 is run for both variants.
CONFIGS = {
    "cfg1": Config("cfg1", 1, 32, 4, 32, "f32", STARTING, 1.0, "none", 0),
    "cfg2": Config("cfg2", 1, 128, 4, 32, "bf16", STARTING, 2.0, "tail:13", 1),
    "cfg3s": Config("cfg3s", 1, 384, 4, 32, "bf16", STARTING, 1.0, "none", 2),
    "cfg3e": Config("cfg3e", 1, 384, 4, 32, "bf16", ENDING, 1.0, "none", 2),
    "cfg4": Config("cfg4", 2, 768, 4, 32, "bf16", STARTING, 1.0, "lengths:700,768", 3),
    "cfg5": Config("cfg5", 1, 1024, 4, 32, "bf16", ENDING, 3.0, "random:64", 4),
}


def round_bf16(x: np.ndarray) -> np.ndarray:
    """Round float32 to the nearest bfloat16 (ties to even); result stays float32."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = ((u >> 16) & 1) + np.uint32(0x7FFF)
    return ((u + r) & np.uint32(0xFFFF0000)).view(np.float32)


def bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 values that are exactly representable in bf16 -> their uint16 bit patterns."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    assert not np.any(u & np.uint32(0xFFFF)), "value is not bf16-representable"
    return (u >> 16).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (b.astype(np.uint32) << 16).view(np.float32)


def key_keep(cfg: Config, rng: np.random.Generator) -> np.ndarray | None:
    """keep(b,k) flags of the key-padding mask (reading A5), or None."""
    B, N = cfg.B, cfg.N
    if cfg.mask == "none":
        return None
    keep = np.ones((B, N), np.uint8)
    kind, arg = cfg.mask.split(":")
    if kind == "tail":
        keep[:, N - int(arg):] = 0
    elif kind == "lengths":
        for b, L in enumerate(int(a) for a in arg.split(",")):
            keep[b, L:] = 0
    elif kind == "random":
        for b in range(B):
            keep[b, rng.permutation(N)[: int(arg)]] = 0
    else:
        raise ValueError(cfg.mask)
    return keep


def expand_mask(keep: np.ndarray | None, N: int, variant: int) -> np.ndarray | None:
    """Broadcast keep(b,k) to the ABI's [B,N,N] mask: starting mask[b,i,k], ending mask[b,k,j]."""
    if keep is None:
        return None
    B = keep.shape[0]
    if variant == STARTING:
        return np.ascontiguousarray(np.broadcast_to(keep[:, None, :], (B, N, N)))
    return np.ascontiguousarray(np.broadcast_to(keep[:, :, None], (B, N, N)))


def make_inputs(cfg: Config) -> dict:
    """Returns float32 arrays (already rounded to cfg.dtype) Q,K,V,G,dO [B,N,H,N,d], bias [B,H,N,N],
    mask [B,N,N] u8 or None."""
    rng = np.random.Generator(np.random.Philox(cfg.seed))
    B, N, H, d = cfg.B, cfg.N, cfg.H, cfg.d
    shp = (B, N, H, N, d)
    out = {}
    for name in ("Q", "K", "V", "G"):
        out[name] = rng.standard_normal(shp, dtype=np.float32)
    out["bias"] = rng.standard_normal((B, H, N, N), dtype=np.float32) * np.float32(cfg.sigma_bias)
    out["dO"] = rng.standard_normal(shp, dtype=np.float32)
    out["mask"] = expand_mask(key_keep(cfg, rng), N, cfg.variant)
    if cfg.dtype == "bf16":
        for name in ("Q", "K", "V", "G", "bias", "dO"):
            out[name] = round_bf16(out[name])
    return out


def small_config(B, N, H, d, dtype="f32", variant=STARTING, sigma_bias=1.0, mask="none", seed=0):
    return Config(f"custom_B{B}_N{N}_H{H}_d{d}_{dtype}_v{variant}", B, N, H, d, dtype, variant,
                  sigma_bias, mask, seed)
