"""Writes workloads/bounds.json: the filter scalars (a0, a, b) of every BASELINE.json config, computed ONCE
with the oracle's apply_H and passed identically to the oracle and to the CUDA path (reading U7).
TEST INFRASTRUCTURE: calls only `oracle/` and the seeded input generator.

    python -m oracle.make_bounds [config ...]        (default: 1 2 3 5; config 4 shares config 3's operator)

Recipe A (BASELINE.json config 1, literally): b = 20-step Lanczos upper bound lambda_max(T_20) + |f_20| from a
    seeded start vector; a0 = theta_min and a = theta_max of a Rayleigh-Ritz (Algorithm 2) on
    a seeded random 30-vector start.
Recipe B (ChFSI-realistic): same b; a0 = lambda_min(T_20); a = mean(V_eff) + 1/2 (6 pi^2 N / Omega)^(2/3), the
    free-electron estimate of the upper edge of the wanted spectrum for N states in the volume Omega,
    clipped into (a0, b).
"""
from __future__ import annotations

import json
import os
import sys
import time

import numpy as np

from oracle import chfsi_oracle as orc
from workloads.generate import CONFIGS, SEED_LANCZOS, SEED_RR, make_workload

OUT = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "workloads", "bounds.json")


def bounds_for(config: int):
    spec = CONFIGS[config]
    wl = make_workload(config)
    op = orc.operator_from_workload(wl)
    v0 = np.random.default_rng(spec.seed_base + SEED_LANCZOS).standard_normal(wl.n_dofs)
    b, lmin = orc.lanczos_upper_bound(op, v0, 20)
    V0 = np.random.default_rng(spec.seed_base + SEED_RR).standard_normal((wl.n_dofs, 30))
    Q, _ = np.linalg.qr(V0)
    theta = orc.rayleigh_ritz(op, Q)
    rec_a = {"a0": float(theta[0]), "a": float(theta[-1]), "b": float(b)}
    omega = wl.L ** 3
    a_fe = float(np.mean(wl.veff_q)) + 0.5 * (6 * np.pi ** 2 * spec.N / omega) ** (2.0 / 3.0)
    a_b = min(max(a_fe, lmin + 1e-3 * (b - lmin)), lmin + 0.5 * (b - lmin))
    rec_b = {"a0": float(lmin), "a": float(a_b), "b": float(b)}
    return {"A": rec_a, "B": rec_b}


def main(argv):
    configs = [int(x) for x in argv] or [1, 2, 3, 5]
    table = {}
    if os.path.exists(OUT):
        with open(OUT) as f:
            table = json.load(f)
    for c in configs:
        t = time.time()
        table[CONFIGS[c].bounds_key] = bounds_for(c)
        print(f"config {c}: {table[CONFIGS[c].bounds_key]}  ({time.time() - t:.1f} s)", flush=True)
        with open(OUT, "w") as f:
            json.dump(table, f, indent=1, sort_keys=True)
            f.write("\n")


if __name__ == "__main__":
    main(sys.argv[1:])
