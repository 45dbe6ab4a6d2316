#!/usr/bin/env python
"""Benchmark of the Chebyshev-filter hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--assembly 0|1] [--variant V] [--impl reference]
    python bench.py --all-configs            one JSON line per BASELINE.json config (profiles/r02_all_configs.md)
    python bench.py --rr                     Rayleigh-Ritz products S, H^, Y Z on config 3's rows (Alg. 2 steps 1 and 3)
    python bench.py --kpoint                 k-point variant (complex Hermitian H~^k) on config 3's mesh, 512 complex vectors

One "step" = one pass of the whole hot path over one batch of synthetic input: the degree-m Chebyshev filter
(cell extraction, per-cell product, non-local projectors, assembly, fused recurrence; m times) applied to
all N vectors of the chosen BASELINE.json config in chunks of B columns.  Prints ONE JSON line.  The default workload
is the largest single-GPU configuration, config 5 (1,728,000 dofs = the paper's Mo6x6x6 count, 4,000 vectors, m = 40).

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
DEFAULT_CONFIG = 5          # the largest single-GPU configuration of BASELINE.json (the metric names no config)

# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the `ncu --set full` captures
# summarised in profiles/ (one capture per (config, kernel); re-captured whenever that kernel changes); None = no capture.
NCU_TRAFFIC_BYTES_PER_LAUNCH = {
    (2, "k_apply_dmma_p<double>"): 1.661e9,    # profiles/r01_v4_config2_config3.md: 1.334 GB read + 0.327 GB written
    (3, "k_apply_dmma_p<double>"): 14.54e9,    # same file: 11.68 GB read + 2.86 GB written
    (5, "k_apply_sf<double>"): 27.24e9,        # profiles/r02_sf_kernel.md: 18.48 GB read + 8.76 GB written
    (3, "k_apply_sf<double>"): 8.82e9,         # same file: 5.97 GB read + 2.84 GB written
    (5, "k_apply_sf_ws<double>"): 27.22e9,     # profiles/r02c_ws_kernel.md: 18.48 GB read + 8.74 GB written
    (3, "k_apply_sf_ws<double>"): 8.80e9,      # same file: 5.97 GB read + 2.83 GB written
    (2, "k_apply_sf_ws<double>"): 0.943e9,     # profiles/r02d_final.md: 0.661 GB read + 0.282 GB written
    (4, "k_apply_sf_ws<float>"): 8.80e9,       # same file: 5.97 GB read + 2.83 GB written (32-column tiles of FP32 rows)
}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=DEFAULT_CONFIG, choices=[1, 2, 3, 4, 5, 6],
                    help="BASELINE.json config 1..5; 6 = extra p=7 workload (config 2's box at FE degree 7)")
    ap.add_argument("--assembly", type=int, default=0, choices=[0, 1],
                    help="0 deterministic coloured assembly, 1 atomic assembly")
    ap.add_argument("--variant", type=int, default=0, choices=[0, 1, 2, 3, 4, 5, 6],
                    help="kernel of the per-cell product: 0 automatic (warp-specialised sum-factorised for p <= 6, else dense persistent), "
                         "1 generic, 2 dense one launch per colour, 3 FP32 storage with 3xTF32 products (looser accuracy), "
                         "4 dense persistent DMMA kernel, 5 sum-factorised, 6 sum-factorised warp-specialised")
    ap.add_argument("--all-configs", action="store_true", help="one JSON line per BASELINE.json config (1..5)")
    ap.add_argument("--rr", action="store_true",
                    help="Rayleigh-Ritz products (S = Y^T Y, H^ = Y^T H~ Y, Y Z) at N = 1024 on config 3's rows")
    ap.add_argument("--partition", action="store_true",
                    help="cell-partitioned filter (paper's domain decomposition, PAPER.md:649): the mesh of --config (default 3) is "
                         "split over the --gpus ranks, boundary rows summed by NCCL all-reduce once per H~ application (strong scaling)")
    ap.add_argument("--boundary-fp32", action="store_true", help="with --partition: FP32 boundary payload (PAPER.md:536)")
    ap.add_argument("--soak", type=float, default=0.0,
                    help="soak run of SECONDS per case on config 2's operator: degree-9 filters repeated at several block widths, "
                         "FP64 and FP32 storage, every result compared bit for bit with the first one (flag-ordered assembly, "
                         "buffer hand-over of the persistent kernels); prints one JSON line")
    ap.add_argument("--kpoint", action="store_true",
                    help="k-point variant (chfsi_create_k) on config 3's mesh: 512 complex vectors in chunks of 128, m = 30")
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


def oracle_sample(spec, requested_cols, seconds):
    """(columns, degree) of the oracle's bounded sample: about `seconds` of CPU work per pass.  The oracle streams every cell
    matrix once per H~ application (memory-bound at few columns: ~3 GB/s through its per-cell NumPy products), so the cost of a
    pass is set by the number of applications; on the large configs the sample is a filter of LOWER DEGREE on a few columns
    of the first chunk (the metric counts vector-applications, whatever the degree)."""
    stream_s = spec.n ** 3 * ((spec.p + 1) ** 3) ** 2 * 8 / 3.0e9 + 0.02            # one pass over the cell matrices
    gflop_per_vec_apply = spec.n ** 3 * 2 * ((spec.p + 1) ** 3) ** 2 * 1e-9
    # columns: as many as cost about one more stream pass at ~15 GFLOP/s (about 20 at p = 6), never more than the chunk
    ncols = requested_cols if requested_cols > 0 else int(max(1, min(spec.B, stream_s * 15.0 / gflop_per_vec_apply)))
    apply_s = stream_s + ncols * gflop_per_vec_apply / 15.0
    return ncols, int(max(2, min(spec.m, seconds / apply_s)))


def time_oracle(orc, op, wl, spec, bounds, ncols, m_s, steps, warmup):
    from workloads.generate import SEED_X, random_block
    a0, a, b = bounds
    X = random_block(wl.n_dofs, range(ncols), spec.seed_base + SEED_X)
    for _ in range(warmup):
        orc.chebyshev_filter(op, X, m_s, a, b, a0)
    t0 = time.perf_counter()
    for _ in range(steps):
        orc.chebyshev_filter(op, X, m_s, a, b, a0)
    dt = time.perf_counter() - t0
    return ncols * m_s * steps / dt, dt / steps


def run_reference(args, spec):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    orc, wl, op, bounds = oracle_setup(spec)
    # ~8 s per step: the driver's --steps K --warmup W run of this arm has to end within a few minutes
    ncols, m_s = oracle_sample(spec, args.cpu_sample_cols, 8.0)
    value, s_per_step = time_oracle(orc, op, wl, spec, bounds, ncols, m_s, args.steps, args.warmup)
    sample = (f"columns 0..{ncols - 1} of the first chunk, degree {m_s}" + (" (full)" if m_s == spec.m else f" of m={spec.m}") +
              ", per step")
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
KERNEL_NAMES = {
    (64, 1): "k_apply_generic<double>", (64, 2): "k_apply_dmma", (64, 4): "k_apply_dmma_p<double>", (64, 5): "k_apply_sf<double>",
    (64, 6): "k_apply_sf_ws<double>", (32, 6): "k_apply_sf_ws<float>",
    (32, 1): "k_apply_generic<float>", (32, 3): "k_apply_tf32_p", (32, 4): "k_apply_dmma_p<float>", (32, 5): "k_apply_sf<float>",
}


def dominant_kernel(precision, variant, info):
    """Name of the kernel the automatic choice (variant 0) resolves to for this operator (include/chfsi.h)."""
    if variant == 0:
        variant = 6 if info["sf_flops_per_vector_apply"] > 0 else 4
    if variant in (5, 6) and not info["sf_flops_per_vector_apply"] > 0:
        variant = 4
    return KERNEL_NAMES.get((precision, variant), "k_apply_generic"), variant


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
    if world > 1 and not dist.is_initialized():
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    wl = make_workload(spec.config)
    a0, a, b = load_bounds(spec.bounds_key, "B")
    op = Operator.from_workload(wl, precision=spec.precision, assembly=args.assembly)
    op.set_kernel_variant(args.variant)
    info = op.info
    N, B, m = spec.N, spec.B, spec.m
    dtype = op.dtype
    elt = 8 if spec.precision == 64 else 4
    kernel, eff_variant = dominant_kernel(spec.precision, args.variant, info)

    # synthetic N(0,1) block resident in HBM, one seeded stream per rank (band-parallel shard), generated on the device
    gen = torch.Generator(device="cuda")
    gen.manual_seed(1000003 * (spec.seed_base + SEED_X) + rank)
    X0 = torch.empty((wl.n_dofs, N), dtype=dtype, device="cuda")
    for j0 in range(0, N, 256):
        j1 = min(N, j0 + 256)
        X0[:, j0:j1] = torch.randn((wl.n_dofs, j1 - j0), dtype=dtype, device="cuda", generator=gen)
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

    # roofline of the dominant kernel (per-cell product incl. gather, projector term, assembly, recurrence)
    cols_total = N * m * args.steps                           # column-applies covered by the profile
    sf = eff_variant in (5, 6)
    if sf:
        # the sum-factorised kernel: EXECUTED flops; DMMA and DFMA share one FP64 pipe on B200
        kflops_per_col = info["sf_flops_per_vector_apply"]
        peak, bound = peaks["dmma_tflops"], "alu"
        peak_note = ("FP64 pipe rate measured in this run by chfsi_measure_fp64_peak (mma.sync m8n8k4 f64; plain DFMA measures "
                     "the same and the two share the pipe: a mixed stream never exceeds it, DESIGN.md Sec. 5); "
                     "MEASURED_PEAKS.json has no FP64 figure")
    else:
        kflops_per_col = info["n_cells"] * 2.0 * info["m_cell"] ** 2 + 2.0 * info["m_cell"] * info["nnz_cell_proj"]
        if spec.precision == 32 and eff_variant == 3:
            peak, bound, peak_note = 277.3 / 3.0, "tensor", \
                "mma.sync m16n8k8 TF32 rate measured on B200 (277.3 TFLOP/s, round-1 microbenchmark) / 3 passes per FP32 product"
        elif eff_variant in (2, 4):
            peak, bound, peak_note = peaks["dmma_tflops"], "tensor", \
                "FP64 mma.sync m8n8k4 (DMMA) rate measured in this run by chfsi_measure_fp64_peak; MEASURED_PEAKS.json has no FP64 figure"
        else:
            peak = peaks["dfma_tflops"] * (2.0 if spec.precision == 32 else 1.0)
            bound, peak_note = "alu", "plain FMA loop: DFMA rate measured in this run (x2 for FP32 FFMA, B200_PROFILING.md unit counts)"
    k_tflops = kflops_per_col * cols_total / (prof["contraction_ms"] * 1e-3) * 1e-12 if prof["contraction_ms"] > 0 else None
    roofline = {
        "kernel": kernel, "bound": bound, "achieved": k_tflops, "peak": peak, "unit": "TFLOP/s",
        "frac": (k_tflops / peak) if k_tflops else None,
        "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH.get((spec.config, kernel)) if args.assembly == 0 else None,
        "flops_counted": "executed (sum-factorised kernel)" if sf else "algorithmic 2 (M_cell + N_psp) M_cell per cell and column",
        "peak_source": peak_note,
        "launches": prof["contraction_launches"],
        "avg_launch_ms": prof["contraction_ms"] / max(1, prof["contraction_launches"]),
        "flops_per_launch": kflops_per_col * cols_total / max(1, prof["contraction_launches"]),
        "share_of_step": prof["contraction_ms"] / ms_local,
        "projector_ms_share": prof["projector_ms"] / ms_local,
        "fp64_dfma_peak": peaks["dfma_tflops"] if peaks else None,
        "dense_equivalent_tflops": (info["n_cells"] * 2.0 * info["m_cell"] ** 2 + 2.0 * info["m_cell"] * info["nnz_cell_proj"])
        * cols_total / (prof["contraction_ms"] * 1e-3) * 1e-12 if prof["contraction_ms"] > 0 else None,
    }

    # end to end through the host-buffer entry point: H2D of every chunk, filter, D2H of the result, pinned host memory.
    # One pinned buffer, filtered in place step after step (the cost of a step does not depend on the values).
    e2e = None
    if not args.no_e2e:
        del X
        torch.cuda.empty_cache()
        Xh = torch.empty((wl.n_dofs, N), dtype=dtype, pin_memory=True)
        Xh.copy_(X0)
        del X0
        torch.cuda.empty_cache()
        n_e2e = max(1, min(args.steps, 10))
        op.chebyshev_filter_host(Xh, B, m, a, b, a0)          # warm-up (staging allocations, first touch)
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            op.chebyshev_filter_host(Xh, B, m, a, b, a0)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt = aggregate_max(dt, world)
        nbytes = wl.n_dofs * N * elt
        e2e = {"value": world * N * m * n_e2e / dt, "unit": UNIT, "h2d_bytes_per_step": nbytes,
               "d2h_bytes_per_step": nbytes, "steps": n_e2e, "timer": "host wall clock around chfsi_chebyshev_filter_host",
               "fraction_of_device_resident": world * N * m * n_e2e / dt / value}
        del Xh

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        orc, owl, oop, bounds = oracle_setup(spec)
        ncols, m_s = oracle_sample(spec, args.cpu_sample_cols, 20.0)
        v, _ = time_oracle(orc, oop, owl, spec, bounds, ncols, m_s, 1, 0)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": cpu_threads(), "kind": "oracle",
                        "sample": f"columns 0..{ncols - 1} of the first chunk, degree {m_s}" +
                                  (" (full)" if m_s == spec.m else f" of m={spec.m}") + ", one pass"}

    line = None
    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None,
            "dtype": ("f64" if spec.precision == 64 else
                      "f32 (3xTF32 products, f32 accumulate)" if eff_variant == 3 else
                      "f64 arithmetic on f32-stored vectors"),
            "data": "synthetic",
            "config": {"workload": workload_name(spec), "assembly": "coloured" if args.assembly == 0 else "atomic",
                       "kernel": kernel, "n_colors": info["n_colors"], "bounds": {"a0": a0, "a": a, "b": b},
                       "parallelism": f"band-parallel x{world} (operator replicated, no collective)",
                       "l2": "inputs larger than L2 (vector blocks %.2f GB + operator data %.2f GB vs 126 MB)"
                             % (2 * wl.n_dofs * min(B, N) * elt / 1e9,
                                (info["sf_field_bytes"] if sf else info["matrix_bytes"]) / 1e9)},
            "tflops": value * (info["sf_flops_per_vector_apply"] if sf else flops_va) * 1e-12,
            "tflops_counted": "executed" if sf else "algorithmic",
            "dense_equivalent_tflops": value * flops_va * 1e-12,
            "flops_per_vector_apply": info["sf_flops_per_vector_apply"] if sf else flops_va,
            "roofline": roofline, "e2e": e2e, "cpu_baseline": cpu_baseline,
            "gpu_launches": launches, "clocks": clocks,
        }
        print(json.dumps(line), flush=True)
    op.close()
    return line


def run_rr(args):
    """Rayleigh-Ritz products of Algorithm 2 at N = 1024 columns on config 3's 884,736 rows:
    S = Y^T Y (k_xty), H^ = Y^T (H~ Y) (apply + k_xty per chunk), Out = Y Z (k_xz).  One JSON line."""
    import torch

    from paper_2203_07820_b200 import Operator, measure_fp64_peak
    from workloads.generate import CONFIGS, make_workload
    spec = CONFIGS[3]
    wl = make_workload(3)
    op = Operator.from_workload(wl)
    info = op.info
    N, B = 1024, 256
    gen = torch.Generator(device="cuda")
    gen.manual_seed(77)
    Y = torch.randn((wl.n_dofs, N), dtype=torch.float64, device="cuda", generator=gen)
    Z = torch.randn((N, N), dtype=torch.float64, device="cuda", generator=gen)
    Out = torch.empty_like(Y)
    ws = op.workspace(B)
    peaks = measure_fp64_peak()
    sampler = ClockSampler(torch.cuda.current_device())

    def timed(fn):
        for _ in range(args.warmup):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / args.steps

    sampler.start()
    l0 = op.launch_count()
    ms_s = timed(lambda: op.overlap_matrix(Y))
    ms_h = timed(lambda: op.projected_hamiltonian(Y, B=B, workspace=ws))
    ms_z = timed(lambda: op.subspace_transform(Y, Z, Out=Out))
    # the paper's mixed-precision blocking (Eq. 38-39): diagonal blocks of 256 columns FP64, N_fr = 128 of 1024
    blk, n_oc = 256, N - 128
    ms_sm = timed(lambda: op.overlap_matrix_mixed(Y, blk))
    ms_hm = timed(lambda: op.projected_hamiltonian_mixed(Y, n_oc, B=B, workspace=ws))
    ms_zm = timed(lambda: op.subspace_transform_mixed(Y, Z, Out=Out))
    Zu = Z.triu()                                             # Z = L^-T of step 3b is upper triangular: zero panels are skipped
    ms_zu = timed(lambda: op.subspace_transform(Y, Zu, Out=Out))
    ms_zum = timed(lambda: op.subspace_transform_mixed(Y, Zu, Out=Out))
    Sd = op.overlap_matrix(Y)
    ms_ch = timed(lambda: op.cholesky_inverse(Sd))
    # DHM step of an SCF iteration (chfsi_update_potential, Alg. 1 step 4): host wall clock incl. the H2D copy of the samples
    import numpy as _np
    veff_new = _np.ascontiguousarray(wl.veff_q * 0.99)

    def timed_host(fn, n=5):
        fn()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(n):
            fn()
        torch.cuda.synchronize()
        return (time.perf_counter() - t0) / n * 1e3

    ms_dhm_sf = timed_host(lambda: op.update_potential(veff_new))
    op.set_kernel_variant(4)
    ms_dhm_dense = timed_host(lambda: (op.update_potential(veff_new), op.apply_H(Y[:, :32])))
    op.set_kernel_variant(args.variant)
    launches = op.launch_count() - l0
    clocks = sampler.stop()
    gemm = 2.0 * wl.n_dofs * N * N                            # flops of one tall product
    gemm_low = 1.0 * wl.n_dofs * N * (N + 1)                  # ... of the lower triangle of a Hermitian one (S, H^: PAPER.md:558)
    kernel, _ = dominant_kernel(64, args.variant, info)
    apply_flops = (info["sf_flops_per_vector_apply"] if "sf" in kernel else info["flops_per_vector_apply"]) * N
    peak = peaks["dmma_tflops"]
    parts = {
        # S and H^: lower triangle only; flops = those of the triangle (whole tiles that cross the diagonal are executed on top)
        "overlap_S": {"kernel": "k_xty (lower triangle) + k_mirror_lower", "ms": ms_s, "tflops": gemm_low / ms_s * 1e-9,
                      "frac": gemm_low / ms_s * 1e-9 / peak},
        "projected_H": {"kernel": kernel + " + k_xty (lower triangle)", "ms": ms_h, "tflops": (gemm_low + apply_flops) / ms_h * 1e-9,
                        "frac": (gemm_low + apply_flops) / ms_h * 1e-9 / peak},
        "transform_YZ": {"kernel": "k_xz", "ms": ms_z, "tflops": gemm / ms_z * 1e-9, "frac": gemm / ms_z * 1e-9 / peak},
        # mixed precision: same algorithmic flops; speed-up over the FP64 product of the same step
        "overlap_S_mixed": {"kernel": "k_umma<xty> (tcgen05 kind::tf32, 3xTF32) + k_xty (FP64 diagonal blocks)", "ms": ms_sm,
                            "tflops": gemm_low / ms_sm * 1e-9, "speedup_vs_fp64": ms_s / ms_sm},
        "projected_H_mixed": {"kernel": kernel + " + k_umma<xty> (tcgen05) + k_xty (fr-fr block)", "ms": ms_hm,
                              "tflops": (gemm_low + apply_flops) / ms_hm * 1e-9, "speedup_vs_fp64": ms_h / ms_hm},
        "transform_mixed": {"kernel": "k_umma<xz> (tcgen05 kind::tf32, 3xTF32 off-diagonal + FP64 diagonal)", "ms": ms_zm,
                            "tflops": gemm / ms_zm * 1e-9, "speedup_vs_fp64": ms_z / ms_zm},
        "transform_YZ_upper": {"kernel": "k_xz, upper-triangular Z (detected on the device)", "ms": ms_zu,
                               "tflops": gemm_low / ms_zu * 1e-9, "frac": gemm_low / ms_zu * 1e-9 / peak},
        "transform_mixed_upper": {"kernel": "k_umma<xz>, upper-triangular Z", "ms": ms_zum, "tflops": gemm_low / ms_zum * 1e-9,
                                  "speedup_vs_fp64": ms_zu / ms_zum},
        "cholesky_inverse": {"kernel": "k_chol_* / k_trinv_row (N = 1024)", "ms": ms_ch},
        "update_potential": {"kernel": "k_sf_fields (default: quadrature-point fields only; 17 MB of samples H2D)", "ms": ms_dhm_sf},
        "update_potential_dense": {"kernel": "k_sf_fields + k_cell_matrix (lazy rebuild of the 3.9 GB of dense cell matrices, "
                                             "variant 4) + one 32-column apply", "ms": ms_dhm_dense},
    }
    total_ms = ms_s + ms_h + ms_z
    line = {
        "metric": "rayleigh_ritz_products_fp64_tflops", "value": (2 * gemm_low + gemm + apply_flops) / total_ms * 1e-9, "unit": "TFLOP/s",
        "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": total_ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"Rayleigh-Ritz products of Alg. 2 (S, H^, Y Z) on config 3's mesh: {wl.n_dofs} rows, N = {N} columns, "
                               f"H~Y in chunks of {B}", "l2": "blocks of 7.2 GB vs 126 MB L2"},
        "roofline": {"kernel": "k_xz", "bound": "tensor", "achieved": parts["transform_YZ"]["tflops"], "peak": peak,
                     "unit": "TFLOP/s", "frac": parts["transform_YZ"]["frac"], "traffic": None,
                     "peak_source": "FP64 mma.sync m8n8k4 (DMMA) rate measured in this run by chfsi_measure_fp64_peak"},
        "parts": parts, "gpu_launches": launches, "clocks": clocks,
    }
    print(json.dumps(line), flush=True)
    op.close()


def run_kpoint(args):
    """Chebyshev filter of the k-point variant (Eq. 30 k-terms PAPER.md:309-311; the paper's best CF speed-up is on its
    k-point benchmark, Table 5) on config 3's mesh and potential: 512 complex vectors (= 1,024 real columns, the
    same bytes as config 3) in chunks of 128, m = 30.  One JSON line; value counts COMPLEX vector-applies."""
    import torch

    from paper_2203_07820_b200 import Operator, measure_fp64_peak
    from workloads.generate import CONFIGS, load_bounds, make_workload
    spec = CONFIGS[3]
    kvec = [0.05, 0.03, -0.04]
    wl = make_workload(3, kvec=kvec)
    a0, a, b = load_bounds(spec.bounds_key, "B")
    b = 1.05 * b + 1.0                                  # the k-terms widen the spectrum slightly
    op = Operator.from_workload(wl)
    info = op.info
    N, B, m = 512, 128, spec.m
    gen = torch.Generator(device="cuda")
    gen.manual_seed(4242)
    X0 = torch.view_as_complex(torch.randn((wl.n_dofs, N, 2), dtype=torch.float64, device="cuda", generator=gen))
    X = torch.empty_like(X0)
    ws = op.workspace(B)
    peaks = measure_fp64_peak()

    def step():
        X.copy_(X0)
        op.chebyshev_filter_chunked(X, B, m, a, b, a0, workspace=ws)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(torch.cuda.current_device())
    op.set_profiling(True)
    l0 = op.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.start()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    prof = op.get_profile()
    launches = op.launch_count() - l0 + args.steps
    value = N * m * args.steps / (ms * 1e-3)
    flops_col = 2.0 * info["sf_flops_per_vector_apply"]           # a complex column = two real columns (+ 12 flop per Gauss point)
    k_tflops = flops_col * N * m * args.steps / (prof["contraction_ms"] * 1e-3) * 1e-12
    line = {
        "metric": "chebyshev_filter_complex_vector_applies_per_s", "value": value, "unit": "complex vector-applies/s",
        "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64 (complex)", "data": "synthetic",
        "config": {"workload": f"k-point variant on config 3's mesh: {wl.n_dofs} dofs, N={N} complex vectors in chunks of B={B}, "
                               f"m={m}, k={kvec}", "kernel": "k_apply_sf_ws<double, k-point> + k_proj_back",
                   "l2": "inputs larger than L2"},
        "real_equivalent_vector_applies_per_s": 2.0 * value,
        "roofline": {"kernel": "k_apply_sf_ws<double, k-point> (+ k_proj_back)", "bound": "alu", "achieved": k_tflops,
                     "peak": peaks["dmma_tflops"], "unit": "TFLOP/s", "frac": k_tflops / peaks["dmma_tflops"], "traffic": None,
                     "flops_counted": "executed: 2 x the real sum-factorised count per complex column",
                     "share_of_step": prof["contraction_ms"] / ms, "projector_ms_share": prof["projector_ms"] / ms},
        "gpu_launches": launches, "clocks": clocks,
    }
    print(json.dumps(line), flush=True)
    op.close()


def run_partition(args, spec):
    """Strong scaling over cells: every rank holds a slab of the mesh (partition.py) and the rows of its dofs for ALL N vectors;
    per H~ application one all-reduce of the projector coefficients and one of the shared rows.  N = 1 measures the same
    sequence (phased, accumulating apply in scaled blocks; shared-row fix-up) without any exchange."""
    import torch
    import torch.distributed as dist

    from paper_2203_07820_b200.partition import PartitionedOperator, SingleComm, TorchComm
    from paper_2203_07820_b200.sharding import aggregate_max
    from workloads.generate import load_bounds, make_workload
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    if world > 1 and not dist.is_initialized():
        dist.init_process_group("nccl", device_id=torch.device("cuda", torch.cuda.current_device()))
    wl = make_workload(spec.config)
    a0, a, b = load_bounds(spec.bounds_key, "B")
    part = PartitionedOperator(wl, comm=TorchComm() if world > 1 else SingleComm(), precision=spec.precision,
                               boundary_fp32=args.boundary_fp32)
    N, B, m = spec.N, spec.B, spec.m
    gen = torch.Generator(device="cuda")
    gen.manual_seed(99)                                      # same seed on every rank; only the timing matters here
    X0 = torch.randn((part.n_local_dofs, N), dtype=part.dtype, device="cuda", generator=gen)
    X = torch.empty_like(X0)
    ws = part.op.workspace(min(B, N))

    def step():
        X.copy_(X0)
        part.chebyshev_filter_chunked(X, B, m, a, b, a0, workspace=ws)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(torch.cuda.current_device())
    l0 = part.op.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.start()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    clocks = sampler.stop()
    ms = aggregate_max(e0.elapsed_time(e1), world) / args.steps
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": N * m / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": "f64" if spec.precision == 64 else "f64 arithmetic on f32-stored vectors", "data": "synthetic",
            "config": {"workload": workload_name(spec), "parallelism": f"cell partition x{world} (slabs), all-reduce of the "
                       f"projector coefficients and of the shared rows per H~ application, payload "
                       f"{'FP32' if args.boundary_fp32 else 'block precision'}",
                       "shared_dofs": int(part.n_shared), "local_dofs_rank0": int(part.n_local_dofs),
                       "l2": "inputs larger than L2"},
            "gpu_launches": part.op.launch_count() - l0 + args.steps, "clocks": clocks}), flush=True)
    part.close()
    if dist.is_initialized():
        dist.destroy_process_group()


def run_soak(args):
    import torch

    from paper_2203_07820_b200 import Operator
    from workloads.generate import load_bounds, make_workload
    wl = make_workload(2)
    a0, a, b = load_bounds("2", "B")
    cases, total_filters, total_launches = [], 0, 0
    for precision in (64, 32):
        op = Operator.from_workload(wl, precision=precision)
        for B in (256, 200, 72, 32, 16):
            gen = torch.Generator(device="cuda")
            gen.manual_seed(7 + B)
            X0 = torch.randn((wl.n_dofs, B), dtype=op.dtype, device="cuda", generator=gen)
            ws = op.workspace(B)
            ref, n, l0, t0 = None, 0, op.launch_count(), time.perf_counter()
            while time.perf_counter() - t0 < args.soak:
                for _ in range(20):
                    X = X0.clone()
                    op.chebyshev_filter(X, 9, a, b, a0, workspace=ws)
                    if ref is None:
                        ref = X
                    elif not torch.equal(X, ref):
                        raise RuntimeError(f"soak: result differs from the first run (precision {precision}, B = {B}, filter {n})")
                    n += 1
                torch.cuda.synchronize()
            cases.append({"precision": precision, "B": B, "filters": n})
            total_filters += n
            total_launches += op.launch_count() - l0
        op.close()
    print(json.dumps({"soak": "bit-identical throughout, no hang", "seconds_per_case": args.soak, "filters": total_filters,
                      "kernel_launches": total_launches, "cases": cases}), flush=True)


def main():
    args = parse_args()
    from workloads.generate import CONFIGS
    if args.soak > 0:
        run_soak(args)
        return
    if args.partition:
        run_partition(args, CONFIGS[args.config if args.config != DEFAULT_CONFIG else 3])
        return
    if args.rr:
        run_rr(args)
        return
    if args.kpoint:
        run_kpoint(args)
        return
    if args.all_configs:
        for c in (1, 2, 3, 4, 5):
            if args.impl == "reference":
                run_reference(args, CONFIGS[c])
            else:
                run_b200(args, CONFIGS[c])
        return
    spec = CONFIGS[args.config]
    if args.block_width > 0:
        import dataclasses
        spec = dataclasses.replace(spec, B=args.block_width, N=args.block_width)
    if args.impl == "reference":
        run_reference(args, spec)
    else:
        run_b200(args, spec)
        import torch.distributed as dist
        if dist.is_initialized():
            dist.destroy_process_group()


if __name__ == "__main__":
    main()
