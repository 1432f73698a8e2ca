"""EvoSP-3D row sharding (paper_2506_20686_b200/evosp.py; Sec. IV-B) on CPU with the gloo
backend, world_size 2: the collectives' host logic (bias all-gather, dBias reduce-scatter, all_to_all axis
rotation) composed HERE, in the test, with the fp64 oracle as the per-rank compute, against the oracle on
the unsharded problem.  (The product's compute is CUDA-only; tests/test_parity_gpu.py checks that its row
shards reproduce the unsharded kernels.)"""
import os
import socket
import sys

import numpy as np
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _problem():
    sys.path.insert(0, ROOT)
    import tri_inputs

    cfg = tri_inputs.small_config(2, 12, 2, 4, "f32", tri_inputs.STARTING, 1.0, "random:3", seed=909)
    x = tri_inputs.make_inputs(cfg)
    return cfg, {k: (None if v is None else np.asarray(v, np.float64 if k != "mask" else np.uint8)) for k, v in x.items()}


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    import oracle
    from paper_2506_20686_b200 import evosp

    oracle.build()
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    cfg, x = _problem()
    N = cfg.N
    r0, n = evosp.shard_rows(N, world, rank)
    rows = slice(r0, r0 + n)
    T = lambda a: torch.from_numpy(np.ascontiguousarray(a))
    # ---- starting node: local rows, bias lines of the own shard gathered, dBias reduce-scattered
    bias = evosp.gather_bias(T(x["bias"][:, :, rows, :])).numpy()
    assert np.array_equal(bias, x["bias"])
    loc = {k: np.ascontiguousarray(x[k][:, rows]) for k in ("Q", "K", "V", "G", "dO", "mask")}
    O, LSE = oracle.fwd_start_general(loc["Q"], loc["K"], loc["V"], loc["G"], bias, loc["mask"])
    dQ, dK, dV, dG, dBp = oracle.bwd_start_general(loc["dO"], loc["Q"], loc["K"], loc["V"], loc["G"], bias, loc["mask"])
    dB = evosp.scatter_dbias(T(dBp)).numpy()
    # ---- ending node by rotation: X^T shards, starting-form compute, rotate the results back
    xe = {k: evosp.rotate(T(loc[k])).numpy() for k in ("Q", "K", "V", "G", "dO")}
    me = evosp.rotate(T(loc["mask"]), row_dim=1, col_dim=2).numpy()
    # ending bias[b,h,k,i] plays starting bias^T; this rank owns the lines i of its shard: columns -> lines
    bias_e = evosp.gather_bias(T(np.ascontiguousarray(np.swapaxes(x["bias"], -1, -2)[:, :, rows, :]))).numpy()
    Oe, LSEe = oracle.fwd_start_general(xe["Q"], xe["K"], xe["V"], xe["G"], bias_e, me)
    ge = oracle.bwd_start_general(xe["dO"], xe["Q"], xe["K"], xe["V"], xe["G"], bias_e, me)
    back = [evosp.rotate(T(a)).numpy() for a in (Oe,) + tuple(ge[:4])]
    lse_back = evosp.rotate(T(LSEe), row_dim=1, col_dim=3).numpy()  # [B,n,H,N] -> rows and positions swapped
    dBe = evosp.scatter_dbias(T(ge[4])).numpy()
    out[rank] = dict(r0=r0, n=n, O=O, LSE=LSE, dQ=dQ, dK=dK, dV=dV, dG=dG, dBias=dB,
                     eO=back[0], edQ=back[1], edK=back[2], edV=back[3], edG=back[4], eLSE=lse_back, edBias=dBe)
    dist.destroy_process_group()


def test_row_sharded_attention_matches_unsharded_oracle_gloo(oracle):
    world = 2
    port = _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = [out[r] for r in range(world)]
    sys.path.insert(0, ROOT)
    import tri_inputs

    cfg, x = _problem()
    args = (x["Q"], x["K"], x["V"], x["G"], x["bias"], x["mask"])
    for variant, pre in ((tri_inputs.STARTING, ""), (tri_inputs.ENDING, "e")):
        O, LSE = oracle.fwd(*args, variant)
        dQ, dK, dV, dG, dBias = oracle.bwd(x["dO"], *args, variant)
        ref = dict(O=O, LSE=LSE, dQ=dQ, dK=dK, dV=dV, dG=dG)
        for r in res:
            rows = slice(r["r0"], r["r0"] + r["n"])
            for k, full in ref.items():
                np.testing.assert_allclose(r[pre + k], full[:, rows], rtol=1e-12, atol=1e-13, err_msg=f"{pre}{k}")
            # dBias comes back in the sharding the bias went in with: starting -> query lines j of the shard;
            # ending -> lines i of the shard of bias^T, i.e. columns of dBias[b,h,k,i]
            want = dBias[:, :, rows, :] if variant == tri_inputs.STARTING else np.swapaxes(dBias, -1, -2)[:, :, rows, :]
            np.testing.assert_allclose(r[pre + "dBias"], want, rtol=1e-11, atol=1e-12, err_msg=pre + "dBias")


def test_shard_rows_rejects_uneven_splits():
    import pytest

    sys.path.insert(0, ROOT)
    from paper_2506_20686_b200 import evosp

    assert [evosp.shard_rows(768, 4, r) for r in range(4)] == [(0, 192), (192, 192), (384, 192), (576, 192)]
    with pytest.raises(ValueError):
        evosp.shard_rows(770, 4, 0)
    with pytest.raises(ValueError):
        evosp.shard_rows(768, 4, 4)
