"""Host-side logic of the multi-GPU bench path, exercised on CPU with the gloo backend (world_size 2):
rank -> batch assignment (weak scaling, no data-path collective), max-over-ranks timing, whole-job
aggregation, and the reference arm's contract (rank 0 prints, other ranks exit 0 silently)."""
import json
import os
import socket
import subprocess
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    import bench
    import tri_inputs

    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    cfg = tri_inputs.CONFIGS["cfg2"]
    rcfg = bench.rank_config(cfg, rank)
    x = tri_inputs.make_inputs(rcfg)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, torch.device("cpu"), world)  # rank 1 is the slow one
    val = bench.aggregate_value(cfg, world, ms)
    out[rank] = (rcfg.seed, float(x["Q"].ravel()[0]), x["Q"].shape, ms, val)
    dist.destroy_process_group()


def test_rank_sharding_and_max_over_ranks_gloo():
    world = 2
    port = _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        r0, r1 = out[0], out[1]
    sys.path.insert(0, ROOT)
    import bench
    import tri_inputs

    cfg = tri_inputs.CONFIGS["cfg2"]
    assert r0[0] == cfg.seed and r1[0] == cfg.seed + 1000  # every rank its own batch ...
    assert r0[1] != r1[1] and r0[2] == r1[2]  # ... different data, same shapes (weak scaling)
    assert r0[3] == r1[3] == 15.0  # the job's time is the slowest rank's
    assert r0[4] == r1[4] == bench.model_flop(cfg) * 2 / 15e-3 / 1e12  # whole-job aggregate


def test_reference_arm_prints_one_line_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       capture_output=True, text=True, env=env, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""  # non-zero ranks: no work, no output


def test_model_flop_matches_survey_table():
    sys.path.insert(0, ROOT)
    import bench
    import tri_inputs

    assert abs(bench.model_flop(tri_inputs.CONFIGS["cfg4"]) - 1.6235e12) / 1.6235e12 < 1e-4
    assert abs(bench.model_flop(tri_inputs.CONFIGS["cfg3s"]) - 1.0147e11) / 1.0147e11 < 1e-4
    line = json.loads(json.dumps({"metric": bench.METRIC, "unit": bench.UNIT}))
    assert line["unit"] == "TFLOP/s"
