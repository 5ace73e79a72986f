#!/usr/bin/env python
"""bench.py — throughput of the SU(Nc) heatbath + overrelaxation hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload su3_48] [--precision fp64]
                    [--storage full|recon12] [--kernel auto|generic] [--impl ours|reference]

One STEP = one pass of the whole hot path over the lattice: su_sweep(beta, 1 heatbath,
4 overrelaxation) = 40 staple+update kernels, then su_reunitarize, su_plaquette (8-byte D2H) and
su_polyakov (16-byte D2H). Metric (BASELINE.json): link updates per second; GFLOPS by the stated
per-update formula and effective HBM GB/s ride along in the same line.

Default workload = BASELINE.json configs[2], the headline case: SU(3) 48^4, beta 6.0, hot start seed 7,
lattice resident in HBM (3.06 GB fp64: far above the 126 MB L2, so no L2 flush is needed between steps).
N > 1 (torchrun): the path is specified for one GPU (north_star); ranks run independent replicas
(Markov chains with seed + rank), no data-path collective -> "scaling": "weak".

--impl reference times the CPU oracle (oracle/, as it stands) on the host cores on a bounded sample.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

WORKLOADS = {  # BASELINE.json configs, in order
    "su2_8": dict(Nc=2, L=8, beta=2.3, start="hot", seed=1),
    "su3_16": dict(Nc=3, L=16, beta=6.0, start="cold", seed=3),
    "su3_48": dict(Nc=3, L=48, beta=6.0, start="hot", seed=7),
    "su4_24": dict(Nc=4, L=24, beta=11.0, start="hot", seed=11),
    "su6_16": dict(Nc=6, L=16, beta=25.0, start="cold", seed=5),
}
N_HB, N_OR = 1, 4
METRIC = "link_updates_per_s"
UNIT = "link updates/s"


# ---- the stated per-update formulas -------------
def reals_per_link(Nc, recon12):
    return 4 if Nc == 2 else (12 if recon12 else 2 * Nc * Nc)


def flops_per_update(Nc, kind, recon12=False, mean_attempts=1.05):
    """real add/mul = 1, FMA = 2, div/sqrt/log/sin/cos = 1, integer/Philox = 0."""
    if Nc == 2:                       # quaternion path: 12 products of 28 + 5 adds of 4, then the update
        return 356 + (68 if kind == "or" else 71)
    mm = 8 * Nc ** 3 - 2 * Nc ** 2
    n_sub = Nc * (Nc - 1) // 2
    base = 13 * mm + 10 * Nc * Nc
    per_sub = (23 + 56 * Nc) if kind == "or" else (57 + 13 * mean_attempts + 56 * Nc)
    return base + n_sub * per_sub + (19 * 42 if recon12 else 0)


def algorithmic_bytes_per_update(Nc, precision, recon12):
    """9 link transfers (8 reads + 1 write) per update when every neighbour re-use is captured."""
    return 9 * reals_per_link(Nc, recon12) * (8 if precision == "fp64" else 4)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_traffic(tag):
    """DRAM bytes per launch of the dominant kernel from the committed ncu --set full summary, or None."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        return json.load(open(p)).get(tag)
    except Exception:
        return None
