#!/usr/bin/env python
"""Benchmark of the Chebyshev-filter hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--assembly 0|1] [--impl reference]

One "step" = one pass of the whole hot path over one batch of synthetic input: the degree-m Chebyshev filter
(cell extraction, per-cell contraction, non-local projectors, assembly, fused recurrence; m times) applied to
all N vectors of the chosen BASELINE.json config in chunks of B columns.  Prints ONE JSON line.

N > 1 (torchrun): the path shards over the vectors (the paper's band parallelisation): every rank
holds a replica of the operator and filters its own N columns; there is no data-path collective (weak scaling).
`--impl reference` times the CPU oracle (oracle/, NumPy FP64) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "chebyshev_filter_vector_applies_per_s"
UNIT = "vector-applies/s"
DEFAULT_CONFIG = 2          # BASELINE.json configs[1]

# dram__bytes_read.sum + dram__bytes_write.sum per launch of the contraction kernel, from the `ncu --set full`
# capture summarised in profiles/ (file named in the value); None until a capture exists for that key.
NCU_TRAFFIC_BYTES_PER_LAUNCH = {
    (2, 0): 1.661e9,        # profiles/r01_v4_config2_config3.md: 1.334 GB read + 0.327 GB written per launch
    (3, 0): 14.54e9,        # same file: 11.68 GB read + 2.86 GB written per launch
}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=DEFAULT_CONFIG, choices=[1, 2, 3, 4, 5, 6],
                    help="BASELINE.json config 1..5; 6 = extra p=7 workload (config 2's box at FE degree 7)")
    ap.add_argument("--assembly", type=int, default=0, choices=[0, 1],
                    help="0 deterministic coloured assembly, 1 atomic assembly")
    ap.add_argument("--variant", type=int, default=0, choices=[0, 1, 2, 3],
                    help="contraction kernel: 0 default (persistent single launch), 1 generic, 2 one launch per colour, "
                         "3 FP32 storage with 3xTF32 products (opt-in, looser accuracy)")
    ap.add_argument("--block-width", type=int, default=0,
                    help="override the chunk width B of the config (block-width sweep, the shape of the paper's Fig. 2a); "
                         "N becomes one chunk of that width")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cpu-sample-cols", type=int, default=0, help="columns of the oracle sample (0 = auto)")
    return ap.parse_args()


def workload_name(spec):
    return (f"config{spec.config}: periodic {spec.n}^3 cells p={spec.p} ({(spec.n * spec.p) ** 3} dofs), "
            f"N={spec.N} vectors in chunks of B={spec.B}, m={spec.m}, FP{spec.precision}")


# ------------------------------------------------------------------------------------------------------------
# clocks
# ------------------------------------------------------------------------------------------------------------
class ClockSampler:
    """Samples SM clock and throttle reasons of one GPU with NVML while the timed region runs."""

    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
               0x80: "hw_power_brake_slowdown"}

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self._nv = None

    def _run(self):
        nv = self._nv
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM))
                mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self._h)
                for bit, name in self.REASONS.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(0.02)

    def start(self):
        if self._nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


# ------------------------------------------------------------------------------------------------------------
# CPU oracle leg
# ------------------------------------------------------------------------------------------------------------
def cpu_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 1) for p in threadpool_info() if p.get("user_api") == "blas"]
        return max(n) if n else 1
    except Exception:
        return os.cpu_count() or 1


def oracle_setup(spec):
    """Oracle operator of the config + bounds; the (untimed) setup both CPU legs share."""
    from oracle import chfsi_oracle as orc
    from workloads.generate import load_bounds, make_workload
    wl = make_workload(spec.config)
    op = orc.operator_from_workload(wl)
    a0, a, b = load_bounds(spec.bounds_key, "B")
    return orc, wl, op, (a0, a, b)


def oracle_sample_cols(spec, requested):
    if requested > 0:
        return requested
    # ~10-30 s of CPU work: the oracle streams all cell matrices once per degree (memory-bound at few columns)
    gflop_per_vec_apply = spec.n ** 3 * 2 * ((spec.p + 1) ** 3) ** 2 * 1e-9
    budget_gflop = 400.0
    return int(max(1, min(spec.B, budget_gflop / (gflop_per_vec_apply * spec.m))))


def time_oracle(orc, op, wl, spec, bounds, ncols, steps, warmup):
    from workloads.generate import SEED_X, random_block
    a0, a, b = bounds
    X = random_block(wl.n_dofs, range(ncols), spec.seed_base + SEED_X)
    for _ in range(warmup):
        orc.chebyshev_filter(op, X, spec.m, a, b, a0)
    t0 = time.perf_counter()
    for _ in range(steps):
        orc.chebyshev_filter(op, X, spec.m, a, b, a0)
    dt = time.perf_counter() - t0
    return ncols * spec.m * steps / dt, dt / steps


def run_reference(args, spec):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    orc, wl, op, bounds = oracle_setup(spec)
    ncols = oracle_sample_cols(spec, args.cpu_sample_cols)
    value, s_per_step = time_oracle(orc, op, wl, spec, bounds, ncols, args.steps, args.warmup)
    sample = f"columns 0..{ncols - 1} of the first chunk, full degree m={spec.m}, per step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": s_per_step * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(spec), "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cpu_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------------------
# the CUDA path
# ------------------------------------------------------------------------------------------------------------
def run_b200(args, spec):
    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_2203_07820_b200 import Operator, measure_fp64_peak
    from paper_2203_07820_b200.sharding import aggregate_max
    from workloads.generate import SEED_X, load_bounds, make_workload

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    wl = make_workload(spec.config)
    a0, a, b = load_bounds(spec.bounds_key, "B")
    op = Operator.from_workload(wl, precision=spec.precision, assembly=args.assembly)
    op.set_kernel_variant(args.variant)
    info = op.info
    N, B, m = spec.N, spec.B, spec.m
    dtype = op.dtype

    # synthetic N(0,1) block, generated on the host with a per-rank seed (band-parallel shard), pinned
    rng = np.random.default_rng([spec.seed_base + SEED_X, rank])
    X_host = torch.from_numpy(rng.standard_normal((wl.n_dofs, N)).astype(np.float64 if spec.precision == 64 else np.float32))
    try:
        X_host = X_host.pin_memory()
    except Exception:
        pass
    X0 = X_host.to("cuda")
    X = torch.empty_like(X0)
    ws = op.workspace(min(B, N))
    peaks = measure_fp64_peak()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        X.copy_(X0)                      # device-resident input of this step (counted in the timed region)
        op.chebyshev_filter_chunked(X, B, m, a, b, a0, workspace=ws)

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(torch.cuda.current_device())
    op.set_profiling(True)
    launches0 = op.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.start()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    clocks = sampler.stop()
    ms_local = e0.elapsed_time(e1)
    launches = op.launch_count() - launches0 + args.steps     # + the X <- X0 copy kernel of each step
    prof = op.get_profile()
    op.set_profiling(False)
    ms_total = aggregate_max(ms_local, world)
    ms_per_step = ms_total / args.steps
    value = world * N * m / (ms_per_step * 1e-3)
    flops_va = info["flops_per_vector_apply"]

    # roofline of the dominant kernel (per-cell contraction incl. gather, 3d rows, assembly, recurrence)
    elt = 8 if spec.precision == 64 else 4
    contr_flops_per_apply = (info["n_cells"] * 2.0 * info["m_cell"] ** 2 + 2.0 * info["m_cell"] * info["nnz_cell_proj"])
    n_apply = prof["applies"]
    cols_total = N * m * args.steps                           # column-applies covered by the profile
    contr_tflops = contr_flops_per_apply * cols_total / (prof["contraction_ms"] * 1e-3) * 1e-12 if prof["contraction_ms"] > 0 else None
    if spec.precision == 32 and args.variant == 3:
        peak, bound, peak_note = 277.3 / 3.0, "tensor", \
            "mma.sync m16n8k8 TF32 rate measured on B200 (277.3 TFLOP/s, round-1 microbenchmark) / 3 passes per FP32 product"
    elif spec.precision == 64 or args.variant == 0:
        # the FP32 variant stores matrices and vectors in FP32 and contracts them on the same FP64 tensor pipe
        peak, bound, peak_note = peaks["dmma_tflops"], "tensor", \
            "FP64 mma.sync m8n8k4 (DMMA) rate measured in this run by chfsi_measure_fp64_peak; MEASURED_PEAKS.json has no FP64 figure"
    else:
        peak, bound, peak_note = 2 * 37.2, "alu", "FP32 FFMA: 148 SMs x 128 lanes x 2 x 1.965 GHz (B200_PROFILING.md unit counts)"
    key = (spec.config, args.assembly)
    roofline = {
        "kernel": ({0: "k_apply_dmma_p<double>", 1: "k_apply_generic<double>", 2: "k_apply_dmma"}[args.variant]
                   if spec.precision == 64 else {0: "k_apply_dmma_p<float>", 3: "k_apply_tf32_p"}.get(args.variant, "k_apply_generic<float>")),
        "bound": bound, "achieved": contr_tflops, "peak": peak, "unit": "TFLOP/s",
        "frac": (contr_tflops / peak) if contr_tflops else None,
        "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH.get(key),
        "peak_source": peak_note,
        "launches": prof["contraction_launches"],
        "avg_launch_ms": prof["contraction_ms"] / max(1, prof["contraction_launches"]),
        "flops_per_launch": contr_flops_per_apply * cols_total / max(1, prof["contraction_launches"]),
        "share_of_step": prof["contraction_ms"] / ms_local,
        "projector_ms_share": prof["projector_ms"] / ms_local,
        "fp64_dfma_peak": peaks["dfma_tflops"] if peaks else None,
    }

    # end to end through the host-buffer entry point: H2D of every chunk, filter, D2H of the result
    e2e = None
    if not args.no_e2e:
        Xh = X_host.clone()
        try:
            Xh = Xh.pin_memory()
        except Exception:
            pass
        n_e2e = max(1, min(args.steps, 3))
        op.chebyshev_filter_host(Xh, B, m, a, b, a0)          # warm-up (allocations, first touch)
        Xh.copy_(X_host)
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            op.chebyshev_filter_host(Xh, B, m, a, b, a0)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt = aggregate_max(dt, world)
        nbytes = wl.n_dofs * N * elt
        e2e = {"value": world * N * m * n_e2e / dt, "unit": UNIT, "h2d_bytes_per_step": nbytes,
               "d2h_bytes_per_step": nbytes, "steps": n_e2e, "timer": "host wall clock around chfsi_chebyshev_filter_host"}

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        orc, owl, oop, bounds = oracle_setup(spec)
        ncols = oracle_sample_cols(spec, args.cpu_sample_cols)
        v, _ = time_oracle(orc, oop, owl, spec, bounds, ncols, 1, 0)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": cpu_threads(), "kind": "oracle",
                        "sample": f"columns 0..{ncols - 1} of the first chunk, full degree m={spec.m}, one pass"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None,
            "dtype": ("f64" if spec.precision == 64 else
                      "f32 (3xTF32 products, f32 accumulate)" if args.variant == 3 else
                      "f64 accumulate on f32-stored matrices and vectors"),
            "data": "synthetic",
            "config": {"workload": workload_name(spec), "assembly": "coloured" if args.assembly == 0 else "atomic",
                       "n_colors": info["n_colors"], "bounds": {"a0": a0, "a": a, "b": b},
                       "parallelism": f"band-parallel x{world} (operator replicated, no collective)",
                       "l2": "inputs larger than L2 (cell matrices %.2f GB + vector blocks %.2f GB vs 126 MB)"
                             % (info["matrix_bytes"] / 1e9, 2 * wl.n_dofs * min(B, N) * elt / 1e9)},
            "tflops": value * flops_va * 1e-12,
            "flops_per_vector_apply": flops_va,
            "roofline": roofline, "e2e": e2e, "cpu_baseline": cpu_baseline,
            "gpu_launches": launches, "clocks": clocks,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    from workloads.generate import CONFIGS
    spec = CONFIGS[args.config]
    if args.block_width > 0:
        import dataclasses
        spec = dataclasses.replace(spec, B=args.block_width, N=args.block_width)
    if args.impl == "reference":
        run_reference(args, spec)
    else:
        run_b200(args, spec)


if __name__ == "__main__":
    main()
