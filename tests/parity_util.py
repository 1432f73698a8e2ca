"""Helpers of the GPU parity tests: run the CUDA path through the C-ABI binding on seeded inputs,
run the fp64 oracle on the same (already rounded) values, compare with the north_star error metric
(SURVEY.md Sec. 8(c) A15): max|X_gpu - X_ref| / max|X_ref| per output tensor, +-inf must match exactly.

No arithmetic of the method lives here: only data movement (dtype views, the axis swap T that maps
the ending-node variant onto the oracle's general starting-node routine, row / query sub-sampling).
"""
from __future__ import annotations

import numpy as np

import tri_inputs

TOL = {"f32": 1e-4, "bf16": 2e-2}  # BASELINE.json north_star
OUT_NAMES = ("O", "LSE", "dQ", "dK", "dV", "dG", "dBias")


def to_torch(x: np.ndarray, dtype: str, device="cuda"):
    import torch

    t = torch.from_numpy(np.ascontiguousarray(x))
    if dtype == "bf16" and t.dtype == torch.float32:
        t = t.to(torch.bfloat16)  # exact: values are already bf16-representable
    return t.to(device)


def gpu_inputs(x: dict, dtype: str):
    g = {k: to_torch(x[k], dtype) for k in ("Q", "K", "V", "G", "bias", "dO")}
    g["mask"] = None if x["mask"] is None else to_torch(x["mask"], "u8")
    return g


def run_gpu(x: dict, dtype: str, variant: int):
    """Forward + backward through the C-ABI (python binding).  Returns dict of float64 numpy arrays."""
    import torch

    import paper_2506_20686_b200 as tri

    g = gpu_inputs(x, dtype)
    O, LSE = tri.tri_attn_fwd(g["Q"], g["K"], g["V"], g["G"], g["bias"], g["mask"], variant)
    dQ, dK, dV, dG, dBias = tri.tri_attn_bwd(g["dO"], g["Q"], g["K"], g["V"], g["G"], g["bias"], g["mask"], O, LSE,
                                             variant)
    torch.cuda.synchronize()
    out = dict(O=O, LSE=LSE, dQ=dQ, dK=dK, dV=dV, dG=dG, dBias=dBias)
    return {k: v.float().cpu().numpy().astype(np.float64) for k, v in out.items()}, out


def run_oracle(oracle, x: dict, variant: int):
    O, LSE = oracle.fwd(x["Q"], x["K"], x["V"], x["G"], x["bias"], x["mask"], variant)
    dQ, dK, dV, dG, dBias = oracle.bwd(x["dO"], x["Q"], x["K"], x["V"], x["G"], x["bias"], x["mask"], variant)
    return dict(O=O, LSE=LSE, dQ=dQ, dK=dK, dV=dV, dG=dG, dBias=dBias)


def rel_err(got: np.ndarray, ref: np.ndarray) -> float:
    """A15.  Non-finite reference entries (LSE = -inf of fully masked rows) must match exactly."""
    got = np.asarray(got, np.float64)
    ref = np.asarray(ref, np.float64)
    assert got.shape == ref.shape, (got.shape, ref.shape)
    fin = np.isfinite(ref)
    if not fin.all():
        assert np.array_equal(got[~fin], ref[~fin]), "non-finite entries differ"
    assert np.isfinite(got[fin]).all(), "GPU produced non-finite values where the oracle is finite"
    if not fin.any():
        return 0.0
    den = np.max(np.abs(ref[fin]))
    num = np.max(np.abs(got[fin] - ref[fin]))
    return float(num / den) if den > 0 else float(num)


def assert_close(got: dict, ref: dict, tol: float, names=OUT_NAMES, what=""):
    errs = {k: rel_err(got[k], ref[k]) for k in names}
    bad = {k: e for k, e in errs.items() if not e <= tol}
    assert not bad, f"{what}: rel. error above {tol}: {bad} (all: {errs})"
    return errs


# ---- the axis swap T (ending(X) == T(starting(T(X))), pinned for the oracle in test_oracle_pins) ----
def T5(x):
    return None if x is None else np.ascontiguousarray(x.transpose(0, 3, 2, 1, 4))


def T_last2(x):
    return None if x is None else np.ascontiguousarray(np.swapaxes(x, -1, -2))


def T_lse(x):
    return np.ascontiguousarray(x.transpose(0, 3, 2, 1))


def to_starting(x: dict, variant: int) -> dict:
    """Inputs of either variant expressed as a starting-node problem (pure transposes)."""
    if variant == tri_inputs.STARTING:
        return dict(x)
    y = {k: T5(x[k]) for k in ("Q", "K", "V", "G", "dO")}
    y["bias"] = T_last2(x["bias"])
    y["mask"] = T_last2(x["mask"])
    return y


def outputs_to_starting(o: dict, variant: int) -> dict:
    if variant == tri_inputs.STARTING:
        return dict(o)
    y = {k: T5(o[k]) for k in ("O", "dQ", "dK", "dV", "dG") if k in o}
    if "LSE" in o:
        y["LSE"] = T_lse(o["LSE"])
    if "dBias" in o:
        y["dBias"] = T_last2(o["dBias"])
    return y


def oracle_rows(oracle, xs: dict, rows, with_dbias=False):
    """Oracle on a subset of broadcast rows r of a STARTING-form problem: exact O, LSE, dQ, dK, dV, dG of
    those rows (rows are independent given the bias plane); with_dbias adds those rows' partial sum of dBias."""
    rows = np.asarray(rows)
    sub = {k: xs[k][:, rows] for k in ("Q", "K", "V", "G", "dO")}
    m = None if xs["mask"] is None else xs["mask"][:, rows]
    O, LSE = oracle.fwd_start_general(sub["Q"], sub["K"], sub["V"], sub["G"], xs["bias"], m)
    dQ, dK, dV, dG, dBias = oracle.bwd_start_general(sub["dO"], sub["Q"], sub["K"], sub["V"], sub["G"], xs["bias"], m)
    out = dict(O=O, LSE=LSE, dQ=dQ, dK=dK, dV=dV, dG=dG)
    if with_dbias:
        out["dBias"] = dBias
    return out


def oracle_dbias_queries(oracle, xs: dict, queries):
    """Oracle dBias[b,h,q,:] for a subset of queries q of a STARTING-form problem, summed over ALL rows r
    (exact: a query's softmax row needs every key but no other query)."""
    q = np.asarray(queries)
    sub = {k: xs[k][:, :, :, q] for k in ("Q", "G", "dO")}
    _, _, _, _, dBias = oracle.bwd_start_general(sub["dO"], sub["Q"], xs["K"], xs["V"], sub["G"],
                                                 xs["bias"][:, :, q], xs["mask"])
    return dBias
