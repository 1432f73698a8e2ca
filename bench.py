"""bench.py -- triangle-attention fwd+bwd TFLOP/s on synthetic AF3-crop pair tensors (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4] [--impl ours|reference]

One "step" = one pass of the whole hot path: tri_attn_fwd followed by
tri_attn_bwd through the C-ABI on one batch of synthetic input.  Default workload = BASELINE.json
configs[3] ("cfg4": B=2, N=768, H=4, d=32, bf16, starting node, ragged key mask 700/768), the N=768
configuration the metric is quoted on; it fits one GPU.  Model FLOP = 14*B*H*N^3*d (fwd 2 + bwd 5
matmuls of 2*N^2*d each per (b,row,h)).

Prints ONE JSON line (rank 0).  `value` = model TFLOP/s with inputs resident in HBM; `e2e` = the same
metric through tri_attn_step_host with pinned HOST buffers (H2D + D2H inside the timed region);
`roofline` = the dominant kernel's EXECUTED tensor FLOP per launch (KERNEL_FLOP_UNITS: every matmul the
kernel really issues, recomputation included) / its CUDA-event duration against the measured bf16 peak,
with the MUFU (exp) co-roofline beside it; per-kernel times come from a second, separately profiled loop
(no events inside the headline timed region); `also` = the N=384 half of the metric (cfg3s / cfg3e);
`cpu_baseline` = the fp64 oracle timed on this box's host cores on a bounded sample of the workload.
Multi-GPU (torchrun): rows are independent problems -> each rank runs its own batch, no data-path
collective (weak scaling); time = max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import tri_inputs  # noqa: E402

METRIC = "triangle-attn fwd+bwd TFLOP/s"
UNIT = "TFLOP/s"
SPEC_BF16_TFLOPS = 2250.0  # nominal dense bf16 (context only)
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}


def model_flop(cfg, rows=None) -> float:
    """14*B*H*N^3*d for the full problem; `rows` = number of (b,row) slices if a sample."""
    per_slice = 14.0 * cfg.H * cfg.N * cfg.N * cfg.d
    n = cfg.B * cfg.N if rows is None else rows
    return per_slice * n


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {k: float(d[k]) for k in FALLBACK_PEAKS if k in d} | {"source": "measured"}
    return dict(FALLBACK_PEAKS, source="fallback")


# ------------------------------------------------------------------------------------------------
# clocks sampling (nvidia-smi in the background during the timed region)
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "20"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self) -> dict:
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.f.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1])); pw.append(float(parts[2]))
            except ValueError:
                continue
            for n, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        self.f.close()
        os.unlink(self.f.name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
# the oracle leg (cpu_baseline of our arm, and the whole of --impl reference)
# ------------------------------------------------------------------------------------------------
def oracle_sample_inputs(cfg, rows_per_batch: int):
    """`rows_per_batch` broadcast rows of the workload (rows are independent given the bias plane), same
    distributions / rounding / mask recipe as tri_inputs.make_inputs, expressed in starting-node form."""
    rng = np.random.Generator(np.random.Philox(cfg.seed + 77))
    B, N, H, d, R = cfg.B, cfg.N, cfg.H, cfg.d, rows_per_batch
    x = {k: rng.standard_normal((B, R, H, N, d), dtype=np.float32) for k in ("Q", "K", "V", "G", "dO")}
    x["bias"] = rng.standard_normal((B, H, N, N), dtype=np.float32) * np.float32(cfg.sigma_bias)
    keep = tri_inputs.key_keep(cfg, rng)
    x["mask"] = None if keep is None else np.ascontiguousarray(np.broadcast_to(keep[:, None, :], (B, R, N)))
    if cfg.dtype == "bf16":
        for k in ("Q", "K", "V", "G", "dO", "bias"):
            x[k] = tri_inputs.round_bf16(x[k])
    return x


def time_oracle(cfg, rows_per_batch: int, reps: int = 1):
    """Seconds per pass of the fp64 oracle (fwd + bwd) over the sample; returns (sec, flop, threads)."""
    import oracle

    oracle.build()
    x = oracle_sample_inputs(cfg, rows_per_batch)
    x64 = {k: (None if v is None else (v if v.dtype == np.uint8 else v.astype(np.float64))) for k, v in x.items()}
    best = float("inf")
    for _ in range(reps):
        t0 = time.perf_counter()
        oracle.fwd_start_general(x64["Q"], x64["K"], x64["V"], x64["G"], x64["bias"], x64["mask"])
        oracle.bwd_start_general(x64["dO"], x64["Q"], x64["K"], x64["V"], x64["G"], x64["bias"], x64["mask"])
        best = min(best, time.perf_counter() - t0)
    return best, model_flop(cfg, rows=cfg.B * rows_per_batch), oracle.num_threads()


def oracle_rows_for_budget(cfg, seconds: float) -> int:
    """Pick a row count so one oracle pass takes about `seconds` (calibrated on an 8-row pass)."""
    t8, _, _ = time_oracle(cfg, 8)
    return int(max(1, min(cfg.N, 8 * seconds / max(t8, 1e-4))))


def run_reference(args, cfg):
    """--impl reference: the oracle, as it stands, on the host cores; each step = a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    total_budget = 120.0  # seconds for warmup+steps
    per_step = total_budget / max(1, args.steps + args.warmup)
    R = oracle_rows_for_budget(cfg, min(per_step, 20.0))
    for _ in range(args.warmup):
        time_oracle(cfg, R)
    t, fl, thr = 0.0, 0.0, 1
    for _ in range(args.steps):
        s, f, thr = time_oracle(cfg, R)
        t += s
        fl += f
    val = fl / t / 1e12
    sample = f"{R} of {cfg.N} broadcast rows per batch element (B={cfg.B}), full key range, fwd+bwd, fp64"
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": thr, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def workload_name(cfg) -> str:
    v = "starting" if cfg.variant == tri_inputs.STARTING else "ending"
    return (f"{cfg.name}: triangle attention {v} node, {cfg.dtype}, B={cfg.B} N={cfg.N} H={cfg.H} d={cfg.d}, "
            f"bias sigma={cfg.sigma_bias}, mask={cfg.mask}, seed={cfg.seed}")


# ------------------------------------------------------------------------------------------------
# multi-rank host logic (device-agnostic: tested with the gloo backend on CPU, world_size 2)
# ------------------------------------------------------------------------------------------------
def rank_config(cfg, rank: int):
    """Weak scaling: every rank draws its OWN batch of the workload (rows are independent problems,
    no data-path collective): same shapes, seed offset by the rank."""
    return tri_inputs.Config(**{**cfg.__dict__, "seed": cfg.seed + 1000 * rank})


def max_over_ranks(ms: float, device, world: int) -> float:
    """The job's step time is the slowest rank's (all-reduce MAX of the device-measured milliseconds)."""
    if world == 1:
        return ms
    import torch
    import torch.distributed as dist

    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(cfg, world: int, ms_step: float) -> float:
    """Whole-job model TFLOP/s: all ranks' FLOP over the max-over-ranks step time."""
    return model_flop(cfg) * world / (ms_step * 1e-3) / 1e12


# ------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------
# executed tensor FLOP per logit-pass of each kernel, in units of B*H*N^3*d (2 per matmul)
KERNEL_FLOP_UNITS = (("fwd", 4.0), ("dkdv", 8.0), ("dqdb", 6.0), ("dq_", 6.0), ("dbias_kernel", 4.0))
# one exp per logit and kernel pass: 16 MUFU.EX2 / clk / SM
KERNEL_EXP_PASSES = (("fwd", 1.0), ("dkdv", 1.0), ("dqdb", 1.0), ("dq_", 1.0), ("dbias_kernel", 1.0))
# bench.py never reads a stored DRAM-traffic number: `traffic` is null here and the ncu --set full summary of the
# same commit (dram__bytes_read.sum + dram__bytes_write.sum per launch) is named in `traffic_source`
TRAFFIC_SOURCE = "profiles/r2_ncu_full_cfg4.md"


def exp_floor_ms(name: str, cfg, sm_mhz: float) -> float | None:
    """MUFU co-roofline: B*H*N^3 exps per pass at 148 SMs x 16 / clk."""
    for key, passes in KERNEL_EXP_PASSES:
        if key in name:
            return passes * cfg.B * cfg.H * cfg.N ** 3 / (148 * 16 * sm_mhz * 1e6) * 1e3
    return None


def kernel_flop(name: str, cfg) -> float | None:
    base = float(cfg.B) * cfg.H * cfg.N ** 3 * cfg.d
    for key, units in KERNEL_FLOP_UNITS:
        if key in name:
            return units * base
    return None


# kernels tri_attn_bwd launches on its library-owned side streams (csrc/sm100_bwd.cu), concurrent with caller-stream kernels
SIDE_STREAM_KERNELS = ("transpose_bf16_kernel", "sm100_dkdv_kernel(side)", "sm100_dbias_reduce_kernel")


class DeviceProblem:
    """One workload resident in HBM: inputs, outputs, workspace, and a step() = fwd + bwd through the C-ABI binding."""

    def __init__(self, tri, cfg, rank, dev, keep_host=False):
        import torch

        x = tri_inputs.make_inputs(rank_config(cfg, rank))
        tdt = torch.bfloat16 if cfg.dtype == "bf16" else torch.float32
        names = ("Q", "K", "V", "G", "bias", "dO")
        host = {k: torch.from_numpy(x[k]).to(tdt) for k in names}
        host["mask"] = None if x["mask"] is None else torch.from_numpy(x["mask"])
        if keep_host:
            host = {k: (None if v is None else v.pin_memory()) for k, v in host.items()}
        self.host = host if keep_host else None
        self.g = {k: (None if v is None else v.to(dev)) for k, v in host.items()}
        B, N, H, d = cfg.B, cfg.N, cfg.H, cfg.d
        self.cfg, self.tri = cfg, tri
        self.code = tri.BF16 if cfg.dtype == "bf16" else tri.F32
        self.O = torch.empty_like(self.g["Q"])
        self.LSE = torch.empty((B, N, H, N), dtype=torch.float32, device=dev)
        self.grads = tuple(torch.empty_like(self.g["Q"]) for _ in range(4)) + (
            torch.empty((B, H, N, N), dtype=torch.float32, device=dev),)
        self.ws_bytes = max(tri.fwd_workspace_bytes(B, N, H, d, cfg.variant, self.code),
                            tri.bwd_workspace_bytes(B, N, H, d, cfg.variant, self.code))
        self.ws = torch.empty(self.ws_bytes, dtype=torch.uint8, device=dev)

    def fwd(self):
        g, cfg, tri = self.g, self.cfg, self.tri
        tri.tri_attn_fwd(g["Q"], g["K"], g["V"], g["G"], g["bias"], g["mask"], cfg.variant, O=self.O, LSE=self.LSE,
                         workspace=self.ws)

    def bwd(self):
        g, cfg, tri = self.g, self.cfg, self.tri
        tri.tri_attn_bwd(g["dO"], g["Q"], g["K"], g["V"], g["G"], g["bias"], g["mask"], self.O, self.LSE, cfg.variant,
                         out=self.grads, workspace=self.ws)

    def step(self):
        self.fwd()
        self.bwd()


def time_steps(prob, steps, warmup, barrier):
    """W untimed steps, then K steps between two CUDA events on the launching stream (no other events inside)."""
    import torch

    for _ in range(warmup):
        prob.step()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        prob.step()
    e1.record()
    barrier()
    return e0.elapsed_time(e1) / steps


def run_ours(args, cfg):
    import torch
    import torch.distributed as dist

    import paper_2506_20686_b200 as tri

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU path; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    if not os.path.exists(tri.binding.LIB_PATH):  # fresh checkout: compile the library in-tree first (a build step, not a fallback)
        from paper_2506_20686_b200 import build as _build

        if rank == 0:
            _build.build()
        if world > 1:
            dist.barrier()
    tri.load()
    peaks = load_peaks()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- inputs: seeded synthetic, rounded to bf16 once; each rank draws its own batch (weak scaling)
    prob = DeviceProblem(tri, cfg, rank, dev, keep_host=True)
    B, N, H, d = cfg.B, cfg.N, cfg.H, cfg.d
    for _ in range(args.warmup):
        prob.step()
    torch.cuda.synchronize()
    torch.cuda.reset_peak_memory_stats()

    # ---- timed region: K steps between two CUDA events, nothing else recorded inside
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    l0 = tri.launch_count()
    ms_step = time_steps(prob, args.steps, 0, barrier)
    launches = tri.launch_count() - l0
    clocks = sampler.stop() if sampler else None
    peak_bytes = torch.cuda.max_memory_allocated()
    ms_step = max_over_ranks(ms_step, dev, world)
    flop_all = model_flop(cfg) * world
    value = aggregate_value(cfg, world, ms_step)

    # ---- forward and backward on their own (outside the timed region; SURVEY Sec. 8(d) bench protocol)
    def phase_ms(fn, n):
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(n):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / n

    n_ph = max(3, min(args.steps, 20))
    phases = {"fwd_ms": phase_ms(prob.fwd, n_ph), "bwd_ms": phase_ms(prob.bwd, n_ph), "iterations": n_ph}
    phases["fwd_tflops"] = 4.0 / 14.0 * model_flop(cfg) / (phases["fwd_ms"] * 1e-3) / 1e12
    phases["bwd_tflops"] = 10.0 / 14.0 * model_flop(cfg) / (phases["bwd_ms"] * 1e-3) / 1e12

    # ---- per-kernel times: a second, separately profiled loop (events around every launch inside the library)
    prof_steps = max(3, min(args.steps, 10))
    tri.profile_begin()
    for _ in range(prof_steps):
        prob.step()
    torch.cuda.synchronize()
    prof = tri.profile_end()

    # ---- the N=384 half of the metric (cfg3s / cfg3e), same protocol, rank 0's batch only
    also = {}
    if rank == 0 and cfg.name == "cfg4":
        for name in ("cfg3s", "cfg3e"):
            c3 = tri_inputs.CONFIGS[name]
            p3 = DeviceProblem(tri, c3, 0, dev)
            ms3 = time_steps(p3, max(20, args.steps), 5, torch.cuda.synchronize)
            v3 = model_flop(c3) / (ms3 * 1e-3) / 1e12
            also[name] = {"workload": workload_name(c3), "value": v3, "unit": UNIT, "ms_per_step": ms3,
                          "pct_of_peak": {"spec_2250": 100 * v3 / SPEC_BF16_TFLOPS, "measured_burst": 100 * v3 / peaks["bf16_tflops"]},
                          "l2": "inputs + outputs (10 x 75 MB) exceed the 126 MB L2; no flush"}
            del p3
        torch.cuda.empty_cache()

    # ---- e2e: the same step through tri_attn_step_host on pinned HOST buffers (H2D + D2H inside)
    host = prob.host
    ws_bytes = prob.ws_bytes
    code = prob.code
    hout = {k: torch.empty_like(host["Q"]).pin_memory() for k in ("O", "dQ", "dK", "dV", "dG")}
    hout["LSE"] = torch.empty((B, N, H, N), dtype=torch.float32).pin_memory()
    hout["dBias"] = torch.empty((B, H, N, N), dtype=torch.float32).pin_memory()
    del prob
    torch.cuda.empty_cache()
    arena = torch.empty(tri.step_host_arena_bytes(B, N, H, d, cfg.variant, code), dtype=torch.uint8, device=dev)
    hin = dict(host)
    e2e_steps = max(2, min(args.steps, 5))
    tri.tri_attn_step_host(hin, hout, cfg.variant, arena)  # warm-up
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(e2e_steps):
        tri.tri_attn_step_host(hin, hout, cfg.variant, arena)
    e1.record()
    barrier()
    ms_e2e = e0.elapsed_time(e1) / e2e_steps
    ms_e2e = max_over_ranks(ms_e2e, dev, world)
    h2d = sum(v.numel() * v.element_size() for v in hin.values() if v is not None)
    d2h = sum(v.numel() * v.element_size() for v in hout.values())
    if world > 1:
        dist.destroy_process_group()
    if rank != 0:
        return

    # ---- roofline of the dominant kernel (times from the profiled loop)
    # share = fraction of the summed brackets of the kernels on the caller's stream (the step's critical path); kernels the
    # backward runs on its side streams overlap those, their brackets include the time they share the GPU: share = null
    tot = sum(ms for k, (_, ms) in prof.items() if k not in SIDE_STREAM_KERNELS) or 1.0
    kernels = {k: {"launches": n, "ms_per_launch": ms / n, "share": None if k in SIDE_STREAM_KERNELS else ms / tot,
                   "stream": "side (concurrent)" if k in SIDE_STREAM_KERNELS else "caller"} for k, (n, ms) in prof.items()}
    dom = max((k for k in prof if k not in SIDE_STREAM_KERNELS), key=lambda k: prof[k][1])
    dn, dms = prof[dom]
    dflop = kernel_flop(dom, cfg)
    sustained = args.steps * ms_step > 500.0  # a long step loop sits under the power cap
    peak = peaks["bf16_tflops_sustained" if sustained else "bf16_tflops"]
    sm_mhz = (clocks or {}).get("sm_mhz") or 1965.0
    if dflop is not None:
        ach = dflop / (dms / dn * 1e-3) / 1e12
        bound = "tensor" if "simt" not in dom else "alu"
        if bound == "alu":
            # fp32 CUDA-core kernels: 148 SMs x 128 FMA lanes x 2 flop x max SM clock
            peak = 148 * 128 * 2 * 1.965e9 / 1e12
        roof = {"kernel": dom, "bound": bound, "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                "traffic": None, "traffic_source": TRAFFIC_SOURCE,
                "peak_source": peaks["source"] + (" sustained" if sustained else " burst") if bound == "tensor"
                else "derived: 148 SM x 128 lanes x 2 x 1.965 GHz", "flop_per_launch": dflop, "flop_kind": "executed",
                "ms_per_launch": dms / dn}
        fl = exp_floor_ms(dom, cfg, sm_mhz)
        if fl is not None:
            roof["mufu_co_roofline"] = {"exp_floor_ms": fl, "frac": fl / (dms / dn),
                                        "note": "one ex2 per logit and pass at 148 SM x 16/clk"}
        # second co-bound: HBM.  Algorithmic bytes of the whole step = 15 U (fwd: Q,K,V,G in, O out;
        # bwd: Q,K,V,G,O,dO in, dQ,dK,dV,dG out) + bias x 2, LSE x 2, dBias, mask; of the dominant kernel = 5 U.
        es = 2 if cfg.dtype == "bf16" else 4
        U = B * N * H * N * d * es
        step_bytes = 15 * U + 2 * B * H * N * N * es + 2 * B * N * H * N * 4 + B * H * N * N * 4 + (B * N * N if host["mask"] is not None else 0)
        roof["hbm_co_roofline"] = {"step_algorithmic_gb": step_bytes / 1e9, "step_achieved_gbs": step_bytes / (ms_step * 1e-3) / 1e9,
                                   "kernel_algorithmic_gb": 5 * U / 1e9, "kernel_achieved_gbs": 5 * U / (dms / dn * 1e-3) / 1e9,
                                   "peak_gbs": peaks["hbm_gbs"], "step_frac": step_bytes / (ms_step * 1e-3) / 1e9 / peaks["hbm_gbs"],
                                   "hbm_floor_ms": step_bytes / peaks["hbm_gbs"] / 1e6}
    else:
        U = B * N * H * N * d * (2 if cfg.dtype == "bf16" else 4)
        bytes_ = 4 * U + B * N * H * N * 4  # preprocess: read dO,O,G, write dG + D
        ach = bytes_ / (dms / dn * 1e-3) / 1e9
        roof = {"kernel": dom, "bound": "hbm", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "frac": ach / peaks["hbm_gbs"], "traffic": None, "traffic_source": TRAFFIC_SOURCE, "peak_source": peaks["source"]}

    # ---- oracle on the host cores, bounded sample (~15 s)
    R = oracle_rows_for_budget(cfg, 15.0 / 1.0)
    sec, fl, thr = time_oracle(cfg, R)
    cpu = {"value": fl / sec / 1e12, "unit": UNIT, "cores": thr, "kind": "oracle",
           "sample": f"{R} of {N} broadcast rows per batch element (B={B}), full key range, fwd+bwd fp64, {sec:.1f} s"}

    U_bytes = B * N * H * N * d * (2 if cfg.dtype == "bf16" else 4)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": cfg.dtype,
        "data": "synthetic",
        "config": {"workload": workload_name(cfg), "per_gpu_batch": B, "l2": "inputs (10 x %.0f MB) exceed the 126 MB L2; no flush" % (U_bytes / 1e6),
                   "model_flop_per_step_per_gpu": model_flop(cfg)},
        "pct_of_peak": {"spec_2250": 100 * value / world / SPEC_BF16_TFLOPS,
                        "measured_burst": 100 * value / world / peaks["bf16_tflops"],
                        "measured_sustained": 100 * value / world / peaks["bf16_tflops_sustained"], "peaks": peaks["source"]},
        "memory": {"peak_gb": peak_bytes / 1e9, "io_tensors_gb": (10 * U_bytes + 3 * B * H * N * N * 4) / 1e9,
                   "workspace_bytes": ws_bytes, "avoided_map_gb_bf16": B * H * N ** 3 * 2 / 1e9},
        "kernels": kernels, "kernels_source": f"separate profiled loop of {prof_steps} steps after the timed region (CUDA events around every launch, "
                                             "on the stream it is launched on); the backward runs kernels on library-owned side streams beside "
                                             "main-stream ones -- transpose / pack_mask / bias_planes beside sm100_bwd_pre_kernel, "
                                             "sm100_dkdv_kernel(side) beside sm100_dqdb_kernel on the SMs its clusters leave empty, "
                                             "sm100_dbias_reduce_kernel beside the rest of sm100_dkdv_kernel -- so their event brackets include "
                                             "the time they share the GPU; `share` is taken over the caller-stream kernels only",
        "phases": phases, "roofline": roof, "also": also, "cpu_baseline": cpu,
        "e2e": {"value": flop_all / (ms_e2e * 1e-3) / 1e12, "unit": UNIT, "ms_per_step": ms_e2e,
                "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps},
        "gpu_launches": int(launches), "clocks": clocks,
    }
    print(json.dumps(line))


def run_evosp(args, cfg):
    """--sp: EvoSP-3D strong scaling of ONE batch: the broadcast rows are
    sharded over the ranks, the step is bias all-gather -> rows forward -> rows backward -> dBias reduce-scatter
    (paper_2506_20686_b200/evosp.py).  Not the driver's default line (that one is weak scaling without collectives)."""
    import torch
    import torch.distributed as dist

    import paper_2506_20686_b200 as tri
    from paper_2506_20686_b200 import evosp

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU path)")
    if cfg.variant != tri_inputs.STARTING:
        raise SystemExit("bench.py --sp: starting-node workloads only (rotate() the operands for the ending node)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if not dist.is_initialized():
        if "RANK" in os.environ and "MASTER_ADDR" in os.environ:  # torchrun (also with one rank): its rendezvous
            dist.init_process_group("nccl", device_id=dev)
        else:  # plain `python bench.py --sp`: a single-rank group of our own
            dist.init_process_group("nccl", init_method="tcp://127.0.0.1:29517", rank=0, world_size=1, device_id=dev)
    tri.load()
    r0, n = evosp.shard_rows(cfg.N, world, rank)
    x = tri_inputs.make_inputs(cfg)  # the same batch on every rank; each keeps its rows
    tdt = torch.bfloat16
    g = {k: torch.from_numpy(x[k][:, r0:r0 + n].copy()).to(tdt).to(dev) for k in ("Q", "K", "V", "G", "dO")}
    bias_shard = torch.from_numpy(x["bias"][:, :, r0:r0 + n].copy()).to(tdt).to(dev)
    mask = None if x["mask"] is None else torch.from_numpy(x["mask"][:, r0:r0 + n].copy()).to(dev)
    op = evosp.RowShardedTriAttention(peer_reduce=args.peer_reduce)

    def step():
        op.forward(g["Q"], g["K"], g["V"], g["G"], bias_shard, mask)
        op.backward(g["dO"])

    for _ in range(args.warmup):
        step()
    dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    dist.barrier()
    torch.cuda.synchronize()
    ms = max_over_ranks(e0.elapsed_time(e1) / args.steps, dev, world)
    if rank == 0:
        print(json.dumps({
            "metric": "triangle-attn fwd+bwd TFLOP/s", "value": model_flop(cfg) / (ms * 1e-3) / 1e12, "unit": "TFLOP/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": cfg.dtype, "data": "synthetic",
            "config": {"workload": workload_name(cfg), "parallelism": f"sp{world}: {n} of {cfg.N} rows per rank, "
                       "bias all-gather + dBias reduce-scatter inside the step"
                       + (" (reduce-scatter: one kernel over peer memory)" if args.peer_reduce else " (NCCL)")}}))
    dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4", choices=sorted(tri_inputs.CONFIGS))
    ap.add_argument("--sp", action="store_true", help="EvoSP-3D row sharding of one batch (strong scaling)")
    ap.add_argument("--peer-reduce", action="store_true",
                    help="with --sp: dBias reduce-scatter by the peer-memory kernel (torch symmetric memory) instead of NCCL")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    cfg = tri_inputs.CONFIGS[args.workload]
    if args.impl == "reference":
        run_reference(args, cfg)
    elif args.sp:
        run_evosp(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
