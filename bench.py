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
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        with open(p) as f:
            for line in f.read().splitlines()[1:]:
                t, b = line.split(",")[:2]
                if t == tag:
                    return float(b)
    except Exception:
        pass
    return None


def ncu_l2_bytes(tag):
    """L2 -> SM bytes per launch of the dominant kernel (ncu l1tex__m_xbar2l1tex_read_bytes.sum, committed), or None."""
    p = os.path.join(ROOT, "profiles", "l2_traffic.csv")
    try:
        with open(p) as f:
            for line in f.read().splitlines()[1:]:
                t, b = line.split(",")[:2]
                if t == tag:
                    return float(b)
    except Exception:
        pass
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons every 200 ms while the timed region runs (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.rows, self.proc, self.thread = [], None, None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200", "-i", str(gpu_index)],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        inside = [r for t, r in self.rows if t0 <= t <= t1] or [r for _, r in self.rows]
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in inside:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except Exception:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def sustained_copy(torch, device_index, seconds=0.6, nbytes=1 << 30):
    """What a pure-DRAM kernel keeps on THIS box for as long as a timed step runs: device-to-device copies of 1 GiB
    (cudaMemcpyAsync through torch's copy_, read + write = 2 GiB of traffic each), back to back for `seconds`, CUDA events
    around all of them, clocks and power sampled meanwhile. MEASURED_PEAKS.json's figure is the best of ten single
    copies (a burst); the update kernels are timed inside a 0.3 - 0.6 s run at the board's power cap, so this is the
    denominator of the same regime (measurement item 7)."""
    dev = torch.device("cuda", device_index)
    a = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    b = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    a.zero_()
    for _ in range(3):
        b.copy_(a)
    torch.cuda.synchronize(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(); b.copy_(a); e1.record(); torch.cuda.synchronize(dev)
    one_ms = max(e0.elapsed_time(e1), 1e-3)
    n = max(10, int(seconds * 1e3 / one_ms))
    sampler = ClockSampler(device_index)
    t0 = time.perf_counter()
    e0.record()
    for _ in range(n):
        b.copy_(a)
    e1.record()
    torch.cuda.synchronize(dev)
    t1 = time.perf_counter()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop(t0, t1)
    del a, b
    torch.cuda.empty_cache()
    return {"gbs": 2.0 * nbytes * n / (ms * 1e-3) / 1e9, "single_copy_gbs": 2.0 * nbytes / (one_ms * 1e-3) / 1e9, "copies": n,
            "bytes_per_copy": nbytes, "seconds": ms * 1e-3, "clocks": clocks,
            "how": "torch copy_ (cudaMemcpyAsync D2D) of 1 GiB, back to back, CUDA events, read + write bytes"}


def rank_seed(wl, rank):
    """N > 1 runs independent replicas: rank r's Markov chain is seeded seed + r."""
    return wl["seed"] + rank


def max_over_ranks(dist, ms, device):
    """The job's time is the slowest rank's device time (one all-reduce MAX of a double; gloo on CPU in tests)."""
    if dist is None:
        return float(ms)
    import torch
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(world, updates_per_rank_step, ms, steps):
    """value = the units ALL ranks processed / the max-over-ranks time"""
    return world * updates_per_rank_step / (ms / steps * 1e-3)


OPTIONS = {}          # --option name=value: su_set_option knobs applied to every lattice of the run


def make_lattice(su, wl, precision, recon12, kernel, rank, device):
    lat = su.Lattice(wl["Nc"], (wl["L"],) * 4, precision, recon12=recon12, kernel=kernel, device=device)
    for k, v in OPTIONS.items():
        lat.set_option(k, v)
    if wl["Nc"] > 2 and REUNIT_MODE == "on-store":
        lat.set_option("reunit_on_store", 1)
    if wl["start"] == "hot":
        lat.init_hot(rank_seed(wl, rank))
    else:
        lat.init_cold(rank_seed(wl, rank))
    return lat


REUNIT_MODE = "on-store"      # --reunit: "on-store" (su_set_option reunit_on_store: inside the sweep's last pass) or "separate"


def one_step(lat, beta, reunit):
    """the whole hot path once: 40 update sub-steps, reunitarisation (Nc >= 3: in the last pass of the sweep where the
    kernels can do it on store, else / with --reunit separate by su_reunitarize), both reductions (24 bytes D2H)"""
    lat.sweep(beta, N_HB, N_OR)
    if reunit and REUNIT_MODE == "separate":
        lat.reunitarize()
    return lat.plaquette(), lat.polyakov()


def time_resident(torch, dist, lat, wl, steps, warmup, sample_clocks, gpu_index):
    """K steps with the lattice resident in HBM; CUDA events on the launching stream; max over ranks."""
    reunit = wl["Nc"] > 2
    for _ in range(warmup):
        one_step(lat, wl["beta"], reunit)
    # L2-resident lattices are launch-bound: the per-kind kernel times (roofline) come from a short pass of plain
    # launches, the timed steps then replay each sweep as ONE CUDA graph (su_set_graph_mode; the two cannot be combined)
    graph = lat.links_bytes < 96e6 and not lat.slab
    tim = None
    if graph:
        lat.set_timing(True)
        for _ in range(min(steps, 5)):
            one_step(lat, wl["beta"], reunit)
        tim = lat.timing()
        lat.set_timing(False)
        lat.set_graph_mode(True)
        for _ in range(3):
            one_step(lat, wl["beta"], reunit)
    else:
        lat.set_timing(True)
    n0 = lat.launch_count()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(gpu_index) if sample_clocks else None
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.perf_counter()
    ev0.record(lat.stream)
    for _ in range(steps):
        plaq, poly = one_step(lat, wl["beta"], reunit)
    ev1.record(lat.stream)
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    if dist is not None:
        dist.barrier()
    ms = ev0.elapsed_time(ev1)
    clocks = sampler.stop(t0, t1) if sampler else None
    if not graph:
        tim = lat.timing()
        lat.set_timing(False)
    launches = lat.launch_count() - n0
    att, exh = lat.counters()
    return dict(ms=ms, wall_ms=(t1 - t0) * 1e3, clocks=clocks, timing=tim, launches=launches, plaquette=plaq,
                polyakov=[poly.real, poly.imag], kp_exhausted=exh, graph=graph)


def time_e2e(torch, dist, lat, wl, steps):
    """Same step through the C ABI with HOST buffers: every step copies the configuration in from pinned
    host memory (su_import_links, canonical doubles), runs the hot path, and copies the new configuration
    back out (su_export_links) plus the 24 bytes of observables."""
    import numpy as np
    reunit = wl["Nc"] > 2
    n_doubles = 4 * lat.V * 2 * lat.Nc * lat.Nc
    pinned = torch.empty(n_doubles, dtype=torch.float64, pin_memory=True)
    host = pinned.numpy().view(np.complex128).reshape(lat.dims[::-1] + (4, lat.Nc, lat.Nc))
    lat.export_links(out=host)
    for _ in range(1):
        lat.import_links(host); one_step(lat, wl["beta"], reunit); lat.export_links(out=host)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.perf_counter()
    ev0.record(lat.stream)
    for _ in range(steps):
        lat.import_links(host)
        one_step(lat, wl["beta"], reunit)
        lat.export_links(out=host)
    ev1.record(lat.stream)
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    if dist is not None:
        dist.barrier()
    ms = max(ev0.elapsed_time(ev1), (t1 - t0) * 1e3)       # host-side copies count: take the longer clock
    return dict(ms=ms, steps=steps, h2d=n_doubles * 8, d2h=n_doubles * 8 + 24)


# ---- the CPU oracle, timed as it stands (cpu_baseline leg and --impl reference) -----------------------
def oracle_substep_rate(wl, precision, recon12, L, budget_s):
    """Time oracle sub-steps of the 1 HB + 4 OR schedule on an L^4 lattice with the workload's group,
    coupling and start; returns (link updates/s over a 1+4 mix, threads, description, seconds spent)."""
    import oracle
    t_start = time.perf_counter()
    O = oracle.OracleLattice(wl["Nc"], (L,) * 4, precision, recon12)
    (O.init_hot if wl["start"] == "hot" else O.init_cold)(wl["seed"])
    half = O.V // 2
    t_kind = {}
    for kind in (0, 1):
        n, t = 0, 0.0
        while n < 8 and (n == 0 or t < budget_s / 2):
            t0 = time.perf_counter()
            O.substep(wl["beta"], kind, 0, n // 4 % 2, n % 4)
            t += time.perf_counter() - t0
            n += 1
        t_kind[kind] = (t / n, n)
    t_mix = N_HB * t_kind[0][0] + N_OR * t_kind[1][0]            # per (parity, mu): 1 HB + 4 OR sub-steps
    rate = (N_HB + N_OR) * half / t_mix
    desc = (f"SU({wl['Nc']}) {L}^4 {precision}{' recon12' if recon12 else ''} beta {wl['beta']} {wl['start']} start: "
            f"{t_kind[0][1]} heatbath + {t_kind[1][1]} overrelaxation sub-steps ({half} link updates each), "
            f"combined 1:4 as in the sweep")
    threads = oracle.num_threads()
    O.close()
    return rate, threads, desc, time.perf_counter() - t_start


def cpu_baseline(wl, precision, recon12, budget_s=20.0):
    import oracle
    # probe on 8^4 to pick the largest lattice (<= the workload's) whose sub-steps fit the budget
    r0, threads, _, _ = oracle_substep_rate(wl, precision, recon12, 8, 0.5)
    L = wl["L"]
    while L > 8 and (L ** 4 / 2) * 10 / r0 > budget_s * 3:        # ~10 sub-steps + init
        L = {48: 32, 32: 24, 24: 16, 16: 12, 12: 8}.get(L, 8)
    rate, threads, desc, spent = oracle_substep_rate(wl, precision, recon12, L, budget_s)
    return {"value": rate, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc,
            "host_cpus": os.cpu_count(), "seconds": round(spent, 2)}


def run_reference(args, wl, rank):
    """--impl reference: the oracle on the host cores, one bounded sample (sub-steps of the sweep) per step."""
    if rank != 0:
        return 0
    import oracle
    precision, recon12 = args.precision, args.storage == "recon12"
    r0, threads, _, _ = oracle_substep_rate(wl, precision, recon12, 8, 0.5)
    budget_step = 150.0 / max(1, args.steps + args.warmup)
    L = wl["L"]
    while L > 8 and (L ** 4 / 2) / r0 > budget_step:
        L = {48: 32, 32: 24, 24: 16, 16: 12, 12: 8}.get(L, 8)
    O = oracle.OracleLattice(wl["Nc"], (L,) * 4, precision, recon12)
    (O.init_hot if wl["start"] == "hot" else O.init_cold)(wl["seed"])
    half = O.V // 2
    sched = [(0 if p < N_HB else 1, parity, mu) for p in range(N_HB + N_OR) for parity in range(2) for mu in range(4)]
    i = 0
    for _ in range(args.warmup):
        kind, parity, mu = sched[i % 40]; O.substep(wl["beta"], kind, 0, parity, mu); i += 1
    t0 = time.perf_counter()
    for _ in range(args.steps):
        kind, parity, mu = sched[i % 40]; O.substep(wl["beta"], kind, 0, parity, mu); i += 1
    dt = time.perf_counter() - t0
    value = args.steps * half / dt
    sample = (f"SU({wl['Nc']}) {L}^4 {precision} beta {wl['beta']} {wl['start']} start; each step = one (parity, mu) "
              f"sub-step of the 1 HB + 4 OR schedule ({half} link updates), schedule order, on {threads} OpenMP threads")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64" if precision == "fp64" else "f32", "data": "synthetic",
            "config": {"workload": args.workload, "Nc": wl["Nc"], "lattice": f"{wl['L']}^4", "beta": wl["beta"],
                       "sweep": "1 heatbath + 4 overrelaxation", "storage": args.storage, "sample_lattice": f"{L}^4"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def run_nc_scan(args, torch, su, local):
    """One JSON line per (Nc, kernel, lattice, precision): ms per iteration, the paper's iteration:
    1 heatbath + 1 overrelaxation + reunitarisation (Nc >= 3) + plaquette, cold start, CUDA-graph replay of the sweep."""
    rows = []
    for L in (8, 16):
        for precision in ("fp32", "fp64"):
            # the paper's range: Nc <= 32 in single, <= 16 in double precision at 8^4; 16^4 up to Nc = 8
            nc_max = 8 if L == 16 else (32 if precision == "fp32" else 16)
            for Nc in range(2, nc_max + 1):
                for kernel in (("specialised", "generic") if Nc <= 4 else ("generic",)):
                    lat = su.Lattice(Nc, (L,) * 4, precision, kernel=kernel, device=local, graph=True)
                    lat.init_cold(1)

                    def it():
                        lat.sweep(6.2, 1, 1)
                        if Nc > 2:
                            lat.reunitarize()
                        return lat.plaquette()

                    for _ in range(5):
                        it()
                    torch.cuda.synchronize()
                    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    n = max(5, args.steps)
                    ev0.record(lat.stream)
                    for _ in range(n):
                        plaq = it()
                    ev1.record(lat.stream)
                    torch.cuda.synchronize()
                    ms = ev0.elapsed_time(ev1) / n
                    rows.append({"scan": "nc", "Nc": Nc, "kernel": kernel, "lattice": f"{L}^4", "precision": precision,
                                 "beta": 6.2, "iteration": "1 HB + 1 OR + reunitarise + plaquette", "ms_per_iteration": ms,
                                 "link_updates_per_s": 2 * 4 * L ** 4 / (ms * 1e-3), "plaquette": plaq})
                    print(json.dumps(rows[-1]), flush=True)
                    lat.close()
    return 0


CONFIG_RUNS = [   # BASELINE.json configs, as stated there: (tag, workload, sweeps, [(precision, recon12, kernel)], oracle sweeps)
    ("C1", "su2_8", 20, [("fp64", False, "auto")], 20),
    ("C2", "su3_16", 200, [("fp64", False, "auto"), ("fp64", True, "auto"), ("fp32", False, "auto"), ("fp32", True, "auto")], 200),
    ("C3", "su3_48", 100, [("fp64", False, "auto"), ("fp64", True, "auto"), ("fp32", False, "auto"), ("fp32", True, "auto")], 2),
    ("C4", "su4_24", 100, [("fp64", False, "auto"), ("fp64", False, "generic"), ("fp32", False, "auto"), ("fp32", False, "generic")], 5),
    ("C5", "su6_16", 50, [("fp64", False, "auto")], 50),
]


def run_config_table(args, torch, su, local, peak):
    """--config-table: every BASELINE.json config run as stated there (sweep counts, reunitarisation per sweep for
    Nc >= 3, plaquette (and Polyakov loop) per sweep), GPU and oracle side by side. One JSON line per (config, variant)
    and a markdown table at the end (committed under profiles/ and quoted in BASELINE.md section 3). The oracle runs the
    whole chain where that takes seconds to a minute (C1, C2, C5: the plaquette histories are compared sweep by
    sweep) and a bounded number of sweeps otherwise (C3: 2, C4: 5), always the first variant of the config."""
    import numpy as np
    import oracle
    rows = []
    for tag, wname, n_sweeps, variants, n_oracle in CONFIG_RUNS:
        if args.workload != "su3_48" and args.workload != wname:
            continue
        wl = WORKLOADS[wname]
        Nc, V = wl["Nc"], wl["L"] ** 4
        reunit = Nc > 2
        warm = 20 if tag == "C3" else 0
        o_hist, o_rate, o_threads = None, None, None
        for vi, (precision, r12, kernel) in enumerate(variants):
            lat = su.Lattice(Nc, (wl["L"],) * 4, precision, recon12=r12, kernel=kernel, device=local)
            for k, v in OPTIONS.items():
                lat.set_option(k, v)
            (lat.init_hot if wl["start"] == "hot" else lat.init_cold)(wl["seed"])
            if lat.links_bytes < 96e6:
                lat.set_graph_mode(True)
            for _ in range(warm):
                lat.sweep(wl["beta"], N_HB, N_OR)
                if reunit:
                    lat.reunitarize()
            torch.cuda.synchronize()
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            hist, poly = [], []
            t_meas = 0.0
            ev0.record(lat.stream)
            for _ in range(n_sweeps):
                lat.sweep(wl["beta"], N_HB, N_OR)
                if reunit:
                    lat.reunitarize()
                hist.append(lat.plaquette())
                if tag == "C5":
                    poly.append(abs(lat.polyakov()))
            ev1.record(lat.stream)
            torch.cuda.synchronize()
            ms = ev0.elapsed_time(ev1) / n_sweeps                     # per sweep, measurements included
            # per-kind kernel times from a short pass of plain launches
            lat.set_graph_mode(False)
            lat.set_timing(True)
            for _ in range(3):
                lat.sweep(wl["beta"], N_HB, N_OR)
            tim = lat.timing()
            lat.set_timing(False)
            or_ms, hb_ms = tim["or_ms"] / tim["or_launches"], tim["hb_ms"] / tim["hb_launches"]
            bpu = algorithmic_bytes_per_update(Nc, precision, r12)
            gbs = bpu * (V // 2) / (or_ms * 1e-3) / 1e9
            tf = flops_per_update(Nc, "or", r12) * (V // 2) / (or_ms * 1e-3) / 1e12
            flops_sweep = 4 * V * (N_HB * flops_per_update(Nc, "hb", r12) + N_OR * flops_per_update(Nc, "or", r12))
            if vi == 0:                                              # the oracle beside it, same start
                O = oracle.OracleLattice(Nc, (wl["L"],) * 4, precision, r12)
                (O.init_hot if wl["start"] == "hot" else O.init_cold)(wl["seed"])
                o_hist = []
                t0 = time.perf_counter()
                for i in range(n_oracle):
                    O.sweep(wl["beta"], N_HB, N_OR)
                    if reunit:
                        O.reunitarize()
                    o_hist.append(O.plaquette())
                    if time.perf_counter() - t0 > 150.0:
                        break
                o_rate = len(o_hist) * (N_HB + N_OR) * 4 * V / (time.perf_counter() - t0)
                o_threads = oracle.num_threads()
                O.close()
            n_cmp = min(len(o_hist), len(hist)) if vi == 0 and warm == 0 else 0
            row = {"config": tag, "workload": wname, "Nc": Nc, "lattice": f"{wl['L']}^4", "precision": precision,
                   "storage": "12-real" if r12 else ("4-real" if Nc == 2 else f"{2 * Nc * Nc}-real"), "kernel": kernel,
                   "beta": wl["beta"], "start": f"{wl['start']} seed {wl['seed']}", "sweeps": n_sweeps, "warmup_sweeps": warm,
                   "ms_per_sweep": ms, "link_updates_per_s": (N_HB + N_OR) * 4 * V / (ms * 1e-3),
                   "gflops": flops_sweep / (ms * 1e-3) / 1e9, "or_substep_ms": or_ms, "hb_substep_ms": hb_ms,
                   "or_hbm_frac_measured_peak": gbs / peak[0], "or_hbm_frac_8TBs": gbs / 8000.0,
                   "or_alu_frac": tf / FMA_PEAKS[precision], "plaquette_last": hist[-1],
                   "plaquette_mean_last_half": float(np.mean(hist[len(hist) // 2:])),
                   "polyakov_abs_last": poly[-1] if poly else None,
                   "oracle_link_updates_per_s": o_rate if vi == 0 else None, "oracle_threads": o_threads if vi == 0 else None,
                   "oracle_sweeps": len(o_hist) if vi == 0 else None,
                   "max_abs_dP_first_3_sweeps": float(np.abs(np.array(hist[:3]) - np.array(o_hist[:3])).max()) if n_cmp >= 3 else None,
                   "oracle_plaquette_mean_last_half": float(np.mean(o_hist[len(o_hist) // 2:])) if vi == 0 and n_cmp == len(hist) else None,
                   "graph_replay": lat.links_bytes < 96e6}
            rows.append(row)
            print(json.dumps(row), flush=True)
            lat.close()
    print("\n| config | group, lattice | precision, storage, kernel | ms / sweep | G link updates/s | TFLOP/s | OR sub-step ms | HB sub-step ms | "
          "OR frac of HBM (measured / 8 TB/s) | OR frac of FMA peak | oracle M updates/s (threads) | plaquette (GPU; oracle) |")
    print("|---|---|---|---:|---:|---:|---:|---:|---:|---:|---:|---|")
    for r in rows:
        orc = f"{r['oracle_link_updates_per_s'] / 1e6:.2f} ({r['oracle_threads']}; {r['oracle_sweeps']} sweeps)" if r["oracle_link_updates_per_s"] else ""
        pl = f"{r['plaquette_mean_last_half']:.5f}"
        if r["oracle_plaquette_mean_last_half"] is not None:
            pl += f"; {r['oracle_plaquette_mean_last_half']:.5f}"
        if r["max_abs_dP_first_3_sweeps"] is not None:
            pl += f" (first 3 sweeps agree to {r['max_abs_dP_first_3_sweeps']:.1e})"
        print(f"| {r['config']} | SU({r['Nc']}) {r['lattice']} | {r['precision']}, {r['storage']}, {r['kernel']} | {r['ms_per_sweep']:.3f} | "
              f"{r['link_updates_per_s'] / 1e9:.3f} | {r['gflops'] / 1e3:.2f} | {r['or_substep_ms']:.4f} | {r['hb_substep_ms']:.4f} | "
              f"{r['or_hbm_frac_measured_peak']:.2f} / {r['or_hbm_frac_8TBs']:.2f} | {r['or_alu_frac']:.2f} | {orc} | {pl} |")
    return 0


def run_slabs(args, wl, torch, dist, rank, world, local, warmup, recon12):
    """--parallel slabs: ONE lattice, rank r owns the time slices [r Lt/N, (r+1) Lt/N). Step =
    40 sub-steps (each followed by the stream-ordered rank ordering) + reunitarise + plaquette (all-reduce). The
    Polyakov loop crosses slabs and is not part of this mode's step. Strong scaling: total work fixed."""
    from paper_1112_4533_b200.slab import DistributedLattice
    D = DistributedLattice(wl["Nc"], (wl["L"],) * 4, args.precision, recon12, args.kernel, device=local)
    (D.init_hot if wl["start"] == "hot" else D.init_cold)(wl["seed"])
    reunit = wl["Nc"] > 2

    def step():
        D.sweep(wl["beta"], N_HB, N_OR)
        if reunit:
            D.reunitarize()
        return D.plaquette()

    for _ in range(warmup):
        step()
    n0 = D.lat.launch_count()
    dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.perf_counter()
    ev0.record(D.lat.stream)
    for _ in range(args.steps):
        plaq = step()
    ev1.record(D.lat.stream)
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    dist.barrier()
    ms = max_over_ranks(dist, ev0.elapsed_time(ev1), "cuda")
    clocks = sampler.stop(t0, t1)
    launches = D.lat.launch_count() - n0
    updates_step = (N_HB + N_OR) * 4 * wl["L"] ** 4                  # the whole lattice, once
    # per-kind sub-step times of THIS rank's slab (two more sweeps, events at the heatbath / overrelaxation boundary)
    from paper_1112_4533_b200.slab import schedule
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    hb_ms = or_ms = 0.0
    for _ in range(2):
        evs[0].record(D.lat.stream)
        for i, (kind, pass_, parity, mu) in enumerate(schedule(N_HB, N_OR)):
            if i == 8 * N_HB:
                evs[1].record(D.lat.stream)
            D.lat.substep(wl["beta"], kind, pass_, parity, mu)
            D._order()
        evs[2].record(D.lat.stream)
        torch.cuda.synchronize()
        hb_ms += evs[0].elapsed_time(evs[1]) / (8 * N_HB) / 2
        or_ms += evs[1].elapsed_time(evs[2]) / (8 * N_OR) / 2
        D.sweep_counter += 1
        D.lat.set_rng(D.seed, D.sweep_counter)
    V_loc = wl["L"] ** 4 // world
    bpu = algorithmic_bytes_per_update(wl["Nc"], args.precision, recon12)
    ach = bpu * (V_loc // 2) / (or_ms * 1e-3) / 1e9
    tf = flops_per_update(wl["Nc"], "or", recon12) * (V_loc // 2) / (or_ms * 1e-3) / 1e12
    peak = measured_peaks()
    roof = {"bound": "hbm", "kernel": "staple + overrelaxation update of one slab, one (parity, mu) sub-step incl. the rank ordering (rank 0)",
            "achieved": ach, "peak": peak[0], "unit": "GB/s", "frac": ach / peak[0], "peak_source": peak[1],
            "alu": {"achieved_tflops": tf, "peak_tflops": FMA_PEAKS.get(args.precision),
                    "frac": tf / FMA_PEAKS[args.precision] if FMA_PEAKS.get(args.precision) else None},
            "avg_launch_ms": or_ms, "hb_avg_launch_ms": hb_ms, "bytes_per_link_update": bpu,
            "algorithmic_bytes_per_launch": bpu * (V_loc // 2), "traffic": None}
    if rank == 0:
        line = {"metric": METRIC, "value": whole_job_rate(1, updates_step, ms, args.steps), "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
                "scaling": "strong", "vs_baseline": None, "dtype": "f64" if args.precision == "fp64" else "f32",
                "data": "synthetic",
                "config": {"workload": args.workload, "Nc": wl["Nc"], "lattice": f"{wl['L']}^4", "beta": wl["beta"],
                           "start": f"{wl['start']} (Philox seed {wl['seed']})", "sweep": "1 heatbath + 4 overrelaxation",
                           "step": "40 x (su_substep + rank ordering) + su_reunitarize + su_plaquette (all-reduce)",
                           "storage": args.storage, "kernel": args.kernel,
                           "parallelism": f"{world} t-slabs of {wl['L'] // world} time slices, halo push fused into the "
                                          "update kernel (peer memory), ordering by a 1-element all-reduce",
                           "l2": "inputs larger than L2 (no flush)"},
                "roofline": roof, "cpu_baseline": None, "e2e": None, "gpu_launches": launches, "clocks": clocks,
                "plaquette": plaq}
        print(json.dumps(line), flush=True)
    D.close()
    dist.barrier()
    dist.destroy_process_group()
    return 0


FMA_PEAKS = {}        # precision -> measured TFLOP/s of the FMA pipe (su_measure_fma_peak), filled once per run
L2_PEAK = {}          # {"gbs", "bytes_per_clk"} of the L2 -> SM read path (su_measure_l2_peak), filled once per run


def variant_numbers(wl, precision, recon12, res, steps, n_ranks, peak):
    """Turn one timed run into the metric, GFLOPS and the roofline object of its dominant (OR) kernel.
    Two roofs are evaluated for the overrelaxation sub-step: HBM (9 R s bytes per update, against the
    measured copy bandwidth) and ALU (the stated flop count per update against the FMA rate measured in this run by
    su_measure_fma_peak: 64 FP64 / 128 FP32 FMAs per clock and SM at the clock of a short burst); `bound` names the
    roof the kernel sits closer to (the larger fraction), both fractions are reported."""
    Nc, V = wl["Nc"], wl["L"] ** 4
    updates_step = (N_HB + N_OR) * 4 * V
    t_step = res["ms"] / steps * 1e-3
    value = whole_job_rate(n_ranks, updates_step, res["ms"], steps)
    flops_step = 4 * V * (N_HB * flops_per_update(Nc, "hb", recon12) + N_OR * flops_per_update(Nc, "or", recon12))
    bpu = algorithmic_bytes_per_update(Nc, precision, recon12)
    tim = res["timing"]
    roof = None
    if tim["or_launches"]:
        or_ms = tim["or_ms"] / tim["or_launches"]
        hb_ms = tim["hb_ms"] / tim["hb_launches"] if tim["hb_launches"] else None
        ach = bpu * (V // 2) / (or_ms * 1e-3) / 1e9
        f_or = flops_per_update(Nc, "or", recon12)
        tf = f_or * (V // 2) / (or_ms * 1e-3) / 1e12
        alu_peak = FMA_PEAKS.get(precision)
        frac_hbm, frac_alu = ach / peak[0], (tf / alu_peak if alu_peak else None)
        alu_bound = frac_alu is not None and frac_alu > frac_hbm
        roof = {"bound": "alu" if alu_bound else "hbm",
                "kernel": "staple + overrelaxation update, one (parity, mu) sub-step (32 of the 40 update sub-steps per sweep)",
                "achieved": tf if alu_bound else ach, "peak": alu_peak if alu_bound else peak[0],
                "unit": "TFLOP/s" if alu_bound else "GB/s", "frac": frac_alu if alu_bound else frac_hbm,
                "peak_source": "measured in this run (su_measure_fma_peak, burst clock)" if alu_bound else peak[1],
                "hbm": {"achieved_gbs": ach, "peak_gbs": peak[0], "frac": frac_hbm, "frac_of_8TBs": ach / 8000.0,
                        "bytes_per_link_update": bpu, "algorithmic_bytes_per_launch": bpu * (V // 2)},
                "alu": {"achieved_tflops": tf, "peak_tflops": alu_peak, "frac": frac_alu, "flops_per_link_update": f_or},
                "frac_of_8TBs": ach / 8000.0, "algorithmic_bytes_per_launch": bpu * (V // 2),
                "bytes_per_link_update": bpu, "avg_launch_ms": or_ms, "hb_avg_launch_ms": hb_ms,
                "hb_achieved": (bpu * (V // 2) / (hb_ms * 1e-3) / 1e9) if hb_ms else None,
                "hb_alu_frac": (flops_per_update(Nc, "hb", recon12) * (V // 2) / (hb_ms * 1e-3) / 1e12 / alu_peak) if hb_ms and alu_peak else None,
                "update_kernels_share_of_step": ((or_ms * N_OR * 8 + (hb_ms or 0.0) * N_HB * 8) / (res["ms"] / steps)),
                "traffic": ncu_traffic(f"su{Nc}_{precision}_{'recon12' if recon12 else 'full'}_or"),
                "traffic_source": "profiles/traffic.csv (round-3 ncu capture of this kernel, profiles/r03a_traffic_and_sustained_copy.md; not re-measured in this run)"}
        # Third figure: the L2 -> SM read path. A link update issues 19 link loads (18 staple links + the own link) and L1
        # serves < 10 % of them, so ~19 R s bytes per update cross the L2 fabric, 2.1 x the 9 R s that must cross HBM. The
        # path delivers 11 kB per SM clock chip-wide (su_measure_l2_peak, = 94 % of the 11.8 kB / clock ncu states), and the
        # kernel uses 0.5 - 0.6 of that: reported so that the reader can rule this roof out (profiles/r02g).
        loaded = 19 * reals_per_link(Nc, recon12) * (8 if precision == "fp64" else 4) * (V // 2)
        xbar = ncu_l2_bytes(f"su{Nc}_{precision}_{'recon12' if recon12 else 'full'}_or")
        if L2_PEAK.get("gbs"):
            l2_bytes = xbar if xbar else loaded
            l2_ach = l2_bytes / (or_ms * 1e-3) / 1e9
            sm_mhz = (res.get("clocks") or {}).get("sm_mhz")
            run_peak = L2_PEAK["bytes_per_clk"] * sm_mhz * 1e6 / 1e9 if sm_mhz and L2_PEAK.get("bytes_per_clk") else None
            roof["l2"] = {"achieved_gbs": l2_ach, "peak_gbs_burst_clock": L2_PEAK["gbs"], "frac_of_burst_peak": l2_ach / L2_PEAK["gbs"],
                          "peak_bytes_per_sm_clock": L2_PEAK.get("bytes_per_clk"), "sm_mhz_in_run": sm_mhz,
                          "peak_gbs_at_run_clock": run_peak, "frac_at_run_clock": (l2_ach / run_peak) if run_peak else None,
                          "bytes_per_launch": l2_bytes, "link_loads_issued_bytes_per_launch": loaded,
                          "bytes_source": ("profiles/l2_traffic.csv (ncu l1tex__m_xbar2l1tex_read_bytes.sum of this kernel, committed)"
                                           if xbar else "19 link loads per update, no L1 hits assumed"),
                          "peak_source": "measured in this run (su_measure_l2_peak: 24 MB L2-resident buffer, ld.global.cg)"}
    return {"value": value, "ms_per_step": res["ms"] / steps, "gflops": n_ranks * flops_step / t_step / 1e9,
            "effective_gbs": n_ranks * bpu * updates_step / t_step / 1e9, "roofline": roof}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="su3_48", choices=sorted(WORKLOADS))
    ap.add_argument("--precision", default="fp64", choices=["fp32", "fp64"])
    ap.add_argument("--storage", default="full", choices=["full", "recon12"])
    ap.add_argument("--kernel", default="auto", choices=["auto", "specialised", "generic"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--parallel", default="auto", choices=["auto", "replicas", "slabs"],
                    help="N > 1: ONE lattice cut into N t-slabs with halo pushes over peer memory (the default when N > 1: "
                         "the path that shards, strong scaling; DESIGN.md 9) or independent replicas (weak scaling, on request)")
    ap.add_argument("--nc-scan", action="store_true",
                    help="the paper's Nc-scaling study (PAPER.md:295-303, Figs 11-12): time per iteration (1 heatbath + 1 "
                         "overrelaxation + reunitarise + plaquette) vs Nc at 8^4 and 16^4, beta 6.2, generic and specialised")
    ap.add_argument("--option", action="append", default=[], metavar="NAME=VALUE",
                    help="su_set_option knob for every lattice of the run (e.g. fuse=2); recorded in config.options")
    ap.add_argument("--reunit", default="on-store", choices=["on-store", "separate"],
                    help="Nc >= 3 reunitarise once per step: inside the sweep's last pass (su_set_option reunit_on_store; the "
                         "default) or by a separate su_reunitarize call")
    ap.add_argument("--config-table", action="store_true",
                    help="run the five BASELINE.json configs as stated there (sweep counts, histories), GPU and oracle side by "
                         "side; JSON lines plus a markdown table (BASELINE.md section 3). --workload X restricts it to one config")
    ap.add_argument("--no-variants", action="store_true", help="skip the extra fp32 / 12-real runs")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=3)
    args = ap.parse_args()
    wl = WORKLOADS[args.workload]
    global REUNIT_MODE
    REUNIT_MODE = args.reunit
    for kv in args.option:
        k, v = kv.split("=", 1)
        OPTIONS[k] = int(v)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        return run_reference(args, wl, rank)

    import torch
    import paper_1112_4533_b200 as su          # raises if libsugauge.so is missing: no fallback
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    warmup = max(args.warmup, 3)
    peak = measured_peaks()
    recon12 = args.storage == "recon12"
    if args.nc_scan:
        return run_nc_scan(args, torch, su, local)
    if args.parallel == "auto":
        args.parallel = "slabs" if world > 1 else "replicas"
    for prec in {args.precision, "fp32", "fp64"}:
        FMA_PEAKS[prec] = su.measure_fma_peak(prec, local)[0]
    g, _, bpc = su.measure_l2_peak(local)
    L2_PEAK.update({"gbs": g, "bytes_per_clk": bpc})
    if args.config_table:
        return run_config_table(args, torch, su, local, peak)
    if args.parallel == "slabs":
        if dist is None:                          # a single rank still goes through the slab path (one slab, self-peered)
            import torch.distributed as dist
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29533")
            dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", local))
        return run_slabs(args, wl, torch, dist, rank, world, local, warmup, recon12)

    def timed(precision, r12, kernel, steps, wu, clocks):
        lat = make_lattice(su, wl, precision, r12, kernel, rank, local)
        res = time_resident(torch, dist, lat, wl, steps, wu, clocks, local)
        res["ms"] = max_over_ranks(dist, res["ms"], "cuda")     # max over ranks of the device time
        return lat, res

    lat, res = timed(args.precision, recon12, args.kernel, args.steps, warmup, True)
    main_num = variant_numbers(wl, args.precision, recon12, res, args.steps, world, peak)
    e2e = None
    if not args.no_e2e:
        r = time_e2e(torch, dist, lat, wl, max(1, args.e2e_steps))
        r["ms"] = max_over_ranks(dist, r["ms"], "cuda")
        e2e = {"value": whole_job_rate(world, (N_HB + N_OR) * 4 * wl["L"] ** 4, r["ms"], r["steps"]), "unit": UNIT,
               "h2d_bytes_per_step": r["h2d"], "d2h_bytes_per_step": r["d2h"], "ms_per_step": r["ms"] / r["steps"],
               "steps": r["steps"], "what": "su_import_links(pinned host, canonical doubles) + step + su_export_links"}
    lat.close()
    del lat

    variants = []
    if not args.no_variants and wl["Nc"] <= 4:
        combos = [(p, s) for p in ("fp64", "fp32") for s in ((False, True) if wl["Nc"] == 3 else (False,))]
        for p, r12 in combos:
            if (p, r12) == (args.precision, recon12):
                continue
            k = max(3, min(args.steps, 10))
            l2, r2 = timed(p, r12, args.kernel, k, 3, False)
            n = variant_numbers(wl, p, r12, r2, k, world, peak)
            variants.append({"precision": p, "storage": "recon12" if r12 else "full", "steps": k, "value": n["value"],
                             "ms_per_step": n["ms_per_step"], "gflops": n["gflops"],
                             "roofline_frac": n["roofline"]["frac"] if n["roofline"] else None,
                             "or_launch_ms": n["roofline"]["avg_launch_ms"] if n["roofline"] else None,
                             "hb_launch_ms": n["roofline"]["hb_avg_launch_ms"] if n["roofline"] else None})
            l2.close()
            del l2

    if rank == 0 and main_num["roofline"] is not None:
        sc = sustained_copy(torch, local)
        roof = main_num["roofline"]
        roof["hbm"]["sustained_copy_gbs"] = sc["gbs"]
        roof["hbm"]["frac_of_sustained_copy"] = roof["hbm"]["achieved_gbs"] / sc["gbs"]
        roof["sustained_copy"] = sc

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(wl, args.precision, recon12)

    if rank == 0:
        line = {"metric": METRIC, "value": main_num["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": warmup, "ms_per_step": main_num["ms_per_step"], "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64" if args.precision == "fp64" else "f32", "data": "synthetic",
                "config": {"workload": args.workload, "Nc": wl["Nc"], "lattice": f"{wl['L']}^4", "beta": wl["beta"],
                           "start": f"{wl['start']} (Philox seed {wl['seed']} + rank)", "sweep": "1 heatbath + 4 overrelaxation",
                           "step": ("su_sweep(1,4) + su_reunitarize + su_plaquette + su_polyakov" if REUNIT_MODE == "separate"
                                    else "su_sweep(1,4) with reunitarisation in its last pass (reunit_on_store) + su_plaquette + su_polyakov")
                                   if wl["Nc"] > 2 else "su_sweep(1,4) + su_plaquette + su_polyakov",
                           "storage": args.storage, "kernel": args.kernel, "options": dict(OPTIONS), "library": su.LIB_PATH,
                           "graph_replay": bool(res.get("graph")),
                           "lattice_bytes": su.lattice_bytes(wl["Nc"], (wl["L"],) * 4, args.precision, recon12),
                           "l2": "inputs larger than L2 (no flush)" if su.lattice_bytes(wl["Nc"], (wl["L"],) * 4, args.precision, recon12) > 3 * 126e6
                                 else "lattice fits in L2: L2-resident by design, HBM fraction not meaningful",
                           "parallelism": "single GPU" if world == 1 else f"{world} independent replicas (no collective)"},
                "gflops": main_num["gflops"], "effective_hbm_gbs": main_num["effective_gbs"],
                "flop_formula": "13*mm+10Nc^2 + n_sub*(23+56Nc) [OR] / n_sub*(57+13*1.05+56Nc) [HB], mm=8Nc^3-2Nc^2 (DESIGN.md)",
                "fma_peaks_tflops": dict(FMA_PEAKS), "l2_peak": dict(L2_PEAK),
                "roofline": main_num["roofline"], "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": res["launches"],
                "clocks": res["clocks"], "plaquette": res["plaquette"], "polyakov": res["polyakov"],
                "kp_exhausted": res["kp_exhausted"], "variants": variants}
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
