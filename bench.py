#!/usr/bin/env python
"""bench.py -- MLUPS of the coupled fp64 ACM LB step (BASELINE.json metric) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl acm|reference] [--config 3] [--inplace]

A "step" is one pass of the whole hot path (phase-field kernel + hydrodynamic kernel) over the
whole grid of the workload.  The path does not shard (north_star: one GPU, no collectives):
with N > 1 every rank runs an independent replica ("replicas only") and `value` is the
number of lattice updates all ranks did divided by the slowest rank's device time.

One JSON line is printed by rank 0.  `--impl reference` times the CPU oracle (oracle/) instead,
on a bounded sample of the same workload (this tier's reference arm).
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "MLUPS of coupled fp64 ACM step at 256^3; achieved HBM GB/s vs B200 peak"
UNIT = "MLUPS"


def bytes_per_cell(Qh, Qg, esz=8):
    """Algorithmic bytes per cell update by the paper's counting rule:
    phase: Qh+3+1 loads, Qh+1 stores; hydro: Qg+3+1 loads, Qg+3 stores."""
    return esz * (2 * Qh + 5), esz * (2 * Qg + 7)


def bytes_per_cell_moments(esz=8):
    """The same rule for the moment representation (ACM_OPT_MOMENTS), whatever the lattices: the phase-field
    kernel reads A, b (4), phi, the velocity its last collision used (3) and the current velocity (3) and writes A, b,
    phi; the hydrodynamic kernel reads A, b, T (10), phi, the velocity (3) and writes A, b, T and the velocity."""
    return esz * (11 + 5), esz * (14 + 13)


def workload(config, size=None):
    from paper_2012_06144_b200 import inputs
    if config == 1:
        p, phi, u = inputs.config1() if size is None else inputs.config1(n=size)
        name = f"config1: {p.nx}^3 periodic static droplet, D3Q15+D3Q19"
    elif config == 2:
        p, phi, u = inputs.config2()
        name = "config2: 128x512x128 rising bubble, walls y, gravity, D3Q15+D3Q19"
    elif config == 3:
        p, phi, u = inputs.config3() if size is None else inputs.scaled_config3(size)
        name = f"config3: {p.nx}^3 periodic, seeded bubbles + velocity noise, D3Q15+D3Q19"
    elif config == 4:
        p, phi, u = inputs.config4()
        name = "config4: 512^3 periodic, 512 seeded bubbles, D3Q15+D3Q19"
    elif config == 5:
        p, phi, u = inputs.config5() if size is None else inputs.scaled_config3(size, 27, 27)
        name = f"config5: {p.nx}^3 periodic, seeded bubbles + velocity noise, D3Q27+D3Q27"
    elif config == 7:
        p, phi, u = inputs.disc2d() if size is None else inputs.disc2d(n=size, count=4, r_min=size / 16, r_max=size / 8)
        name = f"2-D instance: {p.nx}^2 periodic, seeded discs + velocity noise, D2Q9+D2Q9 (P:360)"
    elif config == 8:
        # beyond what the population storage holds on one B200 (768^3 x 632 B = 286 GB): moment representation only (149 GB)
        p, phi, u = inputs.config4(n=768, count=1728)
        name = "768^3 periodic (453 M cells), 1728 seeded bubbles, D3Q15+D3Q19: the density of config 4 on the largest cube of 256-multiples that fits 180 GB in moment representation"
    elif config == 6:
        p, phi, u = inputs.paper_benchmark() if size is None else inputs.paper_benchmark(n=size)
        name = f"paper benchmark P:283: {p.nx}^3 periodic, one bubble R={p.nx // 4}, D3Q15 SRT + D3Q27 MRT"
    else:
        raise SystemExit(f"unknown config {config}")
    return p, phi, u, name


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (torch copy, best of 10)"
    except Exception:
        return 6650.0, "fallback 6.65 TB/s (B200_PROFILING.md)"


class ClockSampler:
    """Samples SM clocks and throttle reasons with NVML while the timed region runs."""

    BAD = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20}
    NOTE = {"sw_power_cap": 0x4, "hw_power_brake": 0x80, "sync_boost": 0x10, "display_clock": 0x100}

    def __init__(self, index):
        self.samples, self.reasons, self.max_mhz, self._stop = [], set(), None, threading.Event()
        self.power, self.mem = [], []
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
                    self.mem.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_MEM))
                except Exception:
                    pass
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in {**self.BAD, **self.NOTE}.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(0.02)

    def __enter__(self):
        if self.nv:
            self._thread = threading.Thread(target=self._loop, daemon=True)
            self._thread.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thread:
            self._thread.join()

    def summary(self):
        s, pw, mm = sorted(self.samples), sorted(self.power), sorted(self.mem)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz,
                "sm_mhz_first_last": [self.samples[0], self.samples[-1]] if s else None,
                "mem_mhz": mm[len(mm) // 2] if mm else None,
                "power_w": pw[len(pw) // 2] if pw else None, "power_w_max": pw[-1] if pw else None,
                "reasons": sorted(self.reasons), "samples": len(s)}


def oracle_sample(config, budget_s, steps=None, threads=0):
    """Times the oracle as it stands on the host cores, on a bounded sample of the workload:
    the same recipe on a smaller cube.  Returns (mlups, cores, description, steps, seconds)."""
    from oracle import Oracle, oracle as om
    all_cores = om.set_threads(0)
    cores = om.set_threads(threads) if threads else all_cores
    try:
        # calibrate on 24^3
        base = config if config in (1, 3, 5, 6, 7) else 3
        sz = (lambda n: int(round(n ** 1.5))) if base == 7 else (lambda n: n)      # 2-D: the same number of cells as n^3
        p, phi, u, _ = workload(base, size=sz(24))
        o = Oracle.from_params(p)
        o.init(phi, u)
        o.step(1)
        t = time.perf_counter()
        o.step(2)
        per_cell = (time.perf_counter() - t) / (2 * p.ncells)
        del o
        if steps is None:
            n, steps = 64, max(2, min(20, int(budget_s / (per_cell * 64 ** 3))))
            while n > 24 and per_cell * n ** 3 * steps > 1.5 * budget_s:
                n -= 8
        else:
            n = 64
            while n > 16 and per_cell * n ** 3 * steps > budget_s:
                n -= 8
        p, phi, u, name = workload(base, size=sz(n))
        o = Oracle.from_params(p)
        o.init(phi, u)
        t = time.perf_counter()
        o.step(steps)
        dt = time.perf_counter() - t
    finally:
        om.set_threads(all_cores)
    return p.ncells * steps / dt / 1e6, cores, f"{name} ({steps} steps; same recipe as the benchmark workload)", steps, dt


def oracle_full_size(config, p, phi, u, steps=3, max_cells=1 << 24):
    """The oracle on the REAL input of the workload for a few steps (256^3 x 3 steps), all cores."""
    if p.ncells > max_cells:
        return None
    from oracle import Oracle, oracle as om
    cores = om.set_threads(0)
    o = Oracle.from_params(p)
    o.init(phi, u)
    t = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t
    return {"value": p.ncells * steps / dt / 1e6, "unit": UNIT, "cores": cores, "steps": steps, "seconds": dt,
            "sample": f"the benchmark input itself, {p.nx}x{p.ny}x{p.nz}, {steps} steps"}


def cpu_baseline(config, p, phi, u):
    """cpu_baseline object: the oracle as it stands on the box's host cores (reported, not a target)."""
    v, cores, sample, _, _ = oracle_sample(config, budget_s=10.0)
    out = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
    v1, c1, s1, _, dt1 = oracle_sample(config, budget_s=4.0, threads=1)
    out["single_thread"] = {"value": v1, "unit": UNIT, "cores": c1, "seconds": dt1, "sample": s1}
    full = oracle_full_size(config, p, phi, u)
    if full is not None:
        out["full_size"] = full
    return out


def run_reference(args, rank, world):
    if rank != 0:
        return
    os.environ.setdefault("OMP_NUM_THREADS", str(os.cpu_count() or 1))
    K, W = args.steps, args.warmup
    mlups, cores, sample, steps, dt = oracle_sample(args.config, budget_s=150.0, steps=K + W)
    # the warm-up share is inside the same run; the rate is per step, so it is unaffected
    _, _, _, name = workload_name_only(args.config)
    out = {"impl": "reference", "metric": METRIC, "value": mlups, "unit": UNIT, "n_gpus": args.gpus, "steps": K,
           "warmup": W, "ms_per_step": dt / steps * 1e3, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": name, "note": "CPU oracle on a bounded sample of the workload"},
           "cpu_baseline": {"value": mlups, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
           "e2e": {"value": mlups, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def workload_name_only(config):
    names = {1: "config1: 32^3 periodic static droplet, D3Q15+D3Q19",
             2: "config2: 128x512x128 rising bubble, walls y, gravity, D3Q15+D3Q19",
             3: "config3: 256^3 periodic, seeded bubbles + velocity noise, D3Q15+D3Q19",
             4: "config4: 512^3 periodic, 512 seeded bubbles, D3Q15+D3Q19",
             5: "config5: 256^3 periodic, seeded bubbles + velocity noise, D3Q27+D3Q27",
             6: "paper benchmark P:283: 260^3 periodic, one bubble R=65, D3Q15 SRT + D3Q27 MRT",
             7: "2-D instance: 4096^2 periodic, seeded discs + velocity noise, D2Q9+D2Q9 (P:360)"}
    return None, None, None, names[config]


def dist_backend():
    """"nccl" (one rank per GPU).  ACM_DIST_BACKEND=gloo lets the multi-rank flow be exercised on a box with fewer
    GPUs than ranks (tests/test_gpu_bench_flow.py): the ranks then share GPUs and only host tensors are reduced."""
    return os.environ.get("ACM_DIST_BACKEND", "nccl")


def pick_device(local_rank):
    import torch
    n = torch.cuda.device_count()
    if dist_backend() == "nccl" and local_rank >= n:
        raise SystemExit(f"bench.py: local rank {local_rank} has no GPU ({n} visible)")
    local_rank = local_rank % n
    torch.cuda.set_device(local_rank)
    return local_rank, torch.device("cuda", local_rank)


def copy_bandwidth(dev, n=1 << 28, repeats=10):
    """Device-to-device copy of n fp64 values (read + write bytes, best of `repeats`, CUDA events): the box's copy
    bandwidth re-measured in this run; the roofline's denominator stays MEASURED_PEAKS.json's."""
    import torch
    a = torch.empty(n, dtype=torch.float64, device=dev).normal_()
    b = torch.empty_like(a)
    b.copy_(a)
    best = float("inf")
    for _ in range(repeats):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        b.copy_(a)
        e1.record()
        torch.cuda.synchronize(dev)
        best = min(best, e0.elapsed_time(e1))
    del a, b
    torch.cuda.empty_cache()
    return 2 * n * 8 / (best * 1e-3) / 1e9


NOMINAL_HBM_GBS = 8000.0      # vendor figure for context (B200_PROFILING.md: 7.7 TB/s HGX, 8 TB/s DGX)
REPEATS = 5


def traffic_row(kernel, config, precision):
    """DRAM bytes per launch of that kernel from the committed ncu --set full capture (profiles/traffic.csv) and the
    commit of the build it was captured from."""
    tpath = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(tpath):
        import csv
        for row in csv.DictReader(open(tpath)):
            if (row["kernel"], row["config"], row["precision"]) == (kernel, str(config), precision):
                return float(row["dram_bytes_per_launch"]), row.get("commit") or None
    return None, None


def measure(args, config, precision, dev, local_rank, world, K, W, with_e2e=True, moments=False):
    """Device-resident throughput of one workload: W warm-up steps, then REPEATS back-to-back intervals of exactly K
    steps each (no per-kernel instrumentation inside them), each bracketed by CUDA events on the launching stream,
    max over ranks per interval, median over the intervals; then a separate pass of K steps with per-kernel events
    (acm_profile) for the kernel split; then the end-to-end run through acm_run_host."""
    import torch
    from paper_2012_06144_b200 import replicas
    from paper_2012_06144_b200.binding import ACM

    p, phi, u, name = workload(config)
    esz = 8 if precision == "f64" else 4
    np_dtype = "float64" if precision == "f64" else "float32"
    phi_h = torch.from_numpy(phi.astype(np_dtype)).pin_memory()
    u_h = torch.from_numpy(u.astype(np_dtype)).pin_memory()
    sim = ACM.from_params(p, precision=precision, device=dev, inplace=args.inplace, unfused=args.unfused, moments=moments)
    if moments and args.moment_kernels is not None:
        sim.set_moment_kernels(*args.moment_kernels)
    if args.cpt:
        sim.set_cells_per_thread(*args.cpt)
    if args.block:
        sim.set_block(*args.block)
    if args.graph is not None:
        sim.set_graph(args.graph)
    sim.init(phi_h.to(dev), u_h.to(dev))
    N = p.ncells
    b_phase, b_hydro = bytes_per_cell_moments(esz) if moments else bytes_per_cell(p.stencil_phase, p.stencil_hydro, esz)

    sim.step(W)
    replicas.barrier(dev)
    launches0 = sim.launch_count
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(REPEATS + 1)]
    with ClockSampler(local_rank) as clk:
        ev[0].record()
        for r in range(REPEATS):
            sim.step(K)
            ev[r + 1].record()
        replicas.barrier(dev)
    launches = (sim.launch_count - launches0) // REPEATS
    graph_replays = sim.graph_replays
    intervals = sorted(replicas.max_over_ranks(ev[r].elapsed_time(ev[r + 1]), dev) for r in range(REPEATS))
    ms = intervals[REPEATS // 2]
    value = replicas.aggregate_mlups(N, K, ms, world)

    # per-kernel split: a separate, instrumented pass (events from a pool created before the first kernel)
    sim.profile(True)
    sim.step(K)
    phase_ms, hydro_ms, nprof = sim.profile_read()
    sim.profile(False)
    phase_ms, hydro_ms = phase_ms / max(nprof, 1), hydro_ms / max(nprof, 1)
    mass = sim.phi_mass()

    res = {"p": p, "phi": phi, "u": u, "name": name, "N": N, "esz": esz, "value": value, "ms": ms, "intervals": intervals,
           "value_min": replicas.aggregate_mlups(N, K, intervals[-1], world), "value_max": replicas.aggregate_mlups(N, K, intervals[0], world),
           "phase_ms": phase_ms, "hydro_ms": hydro_ms, "launches": launches, "graph_replays": graph_replays, "mass": mass, "clocks": clk.summary(),
           "b_phase": b_phase, "b_hydro": b_hydro, "moments": moments}

    if with_e2e:
        # end to end through the C ABI with host buffers (pinned), copies inside the timed region
        po, uo, pro = (torch.empty_like(phi_h).pin_memory(), torch.empty_like(u_h).pin_memory(), torch.empty_like(phi_h).pin_memory())
        sim.run_host(phi_h, u_h, 2, po, uo, pro)            # warm the path
        replicas.barrier(dev)
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0.record()
        sim.run_host(phi_h, u_h, K, po, uo, pro)
        t1.record()
        replicas.barrier(dev)
        ms_e2e = replicas.max_over_ranks(t0.elapsed_time(t1), dev)
        res["e2e"] = replicas.aggregate_mlups(N, K, ms_e2e, world)
        res["finite"] = bool(torch.isfinite(po).all() and torch.isfinite(uo).all())
    del sim
    torch.cuda.empty_cache()
    return res


def roofline_of(args, config, precision, r, K):
    peak, peak_src = measured_peaks()
    hydro = r["hydro_ms"] >= r["phase_ms"]
    dom = "hydro_kernel" if hydro else "phase_kernel"     # unfused: the three kernels of that LB step
    if r.get("moments"):
        dom = dom.replace("_kernel", "_mom_kernel")      # rows of profiles/traffic.csv: the kernels of the moment representation
    dom_ms = r["hydro_ms"] if hydro else r["phase_ms"]
    dom_bytes = (r["b_hydro"] if hydro else r["b_phase"]) * r["N"]
    achieved = dom_bytes / (dom_ms * 1e-3) / 1e9
    step_gbs = (r["b_phase"] + r["b_hydro"]) * r["N"] * K / (r["ms"] * 1e-3) / 1e9
    traffic, commit = traffic_row(dom, config, precision)
    roof = {"bound": "hbm", "kernel": dom if not args.unfused else
            dom.replace("_kernel", "") + " step as three kernels (stream, update, collide); bytes = the fused kernel's algorithmic count",
            "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic, "traffic_commit": commit,
            "peak_source": peak_src + " -- a plain copy: a lower bound of what HBM delivers, fractions above 1 are possible",
            "peak_is_lower_bound": achieved > peak, "frac_of_nominal": achieved / NOMINAL_HBM_GBS, "peak_nominal": NOMINAL_HBM_GBS,
            "algorithmic_bytes_per_launch": dom_bytes, "kernel_ms": dom_ms,
            "kernel_share_of_step": dom_ms / (r["phase_ms"] + r["hydro_ms"])}
    return roof, step_gbs, peak


def run_acm(args, rank, local_rank, world):
    import torch
    from paper_2012_06144_b200 import replicas

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU fallback")
    local_rank, dev = pick_device(local_rank)
    replicas.init(dist_backend(), dev)

    K, W = args.steps, max(args.warmup, 20)      # never fewer than 20 warm-up steps
    precision = args.precision
    if args.config == 8 and not args.moments:
        raise SystemExit("bench.py: --config 8 (768^3) needs --moments: the population storage would take 286 GB")
    r = measure(args, args.config, precision, dev, local_rank, world, K, W, moments=args.moments, with_e2e=args.config != 8)
    copy_now = copy_bandwidth(dev) if world == 1 else None
    extras = []
    if args.config == 3 and precision == "f64" and world == 1 and not (args.no_extras or args.inplace or args.unfused or args.cpt or args.block or args.moments):
        # the fp32 instance of config 5 (BASELINE.json configs[4]) in the same run: device-resident throughput only
        x = measure(args, 5, "f32", dev, local_rank, world, K, W, with_e2e=False)
        roof, step_gbs, peak = roofline_of(args, 5, "f32", x, K)
        extras.append({"workload": x["name"], "dtype": "f32", "value": x["value"], "value_min": x["value_min"], "value_max": x["value_max"],
                       "unit": UNIT, "ms_per_step": x["ms"] / K, "phase_ms": x["phase_ms"], "hydro_ms": x["hydro_ms"],
                       "bytes_per_cell": {"phase": x["b_phase"], "hydro": x["b_hydro"]}, "step_algorithmic_GBps": step_gbs,
                       "step_frac_of_peak": step_gbs / peak, "roofline": roof})
        # the headline workload in moment representation (ACM_OPT_MOMENTS: same time step, the state stored as the 4 + 10
        # coefficients of the post-collision populations; beyond the paper's byte contract, so never the headline)
        for cfg in (3, 5):
            x = measure(args, cfg, "f64", dev, local_rank, world, K, W, with_e2e=False, moments=True)
            roof, step_gbs, peak = roofline_of(args, cfg, "f64", x, K)
            extras.append({"workload": x["name"] + ", moment representation (ACM_OPT_MOMENTS)", "dtype": "f64", "value": x["value"],
                           "value_min": x["value_min"], "value_max": x["value_max"], "unit": UNIT, "ms_per_step": x["ms"] / K,
                           "phase_ms": x["phase_ms"], "hydro_ms": x["hydro_ms"], "bytes_per_cell": {"phase": x["b_phase"], "hydro": x["b_hydro"]},
                           "step_algorithmic_GBps": step_gbs, "step_frac_of_peak": step_gbs / peak, "roofline": roof,
                           "workspace_bytes_per_cell": 8 * (2 * (4 + 10) + 2 + 6), "clocks": x["clocks"]})

    if rank == 0:
        p, N, esz, ms = r["p"], r["N"], r["esz"], r["ms"]
        roof, step_gbs, peak = roofline_of(args, args.config, precision, r, K)
        if copy_now:
            roof["copy_GBps_this_run"] = copy_now
            roof["frac_of_copy_this_run"] = roof["achieved"] / copy_now
        out = {
            "metric": METRIC, "value": r["value"], "value_min": r["value_min"], "value_max": r["value_max"], "unit": UNIT, "n_gpus": world,
            "steps": K, "warmup": W, "repeats": REPEATS, "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak",
            # BASELINE.md holds the paper's number only for its own benchmark (config 6: 550 MLUPS, P100)
            "vs_baseline": (r["value"] / (211.0 if args.unfused else 550.0) if args.config == 6 and world == 1 and precision == "f64" else None),
            "dtype": precision, "data": "synthetic",
            "config": {"workload": r["name"], "grid": [p.nx, p.ny, p.nz], "stencils": [p.stencil_phase, p.stencil_hydro], "phase_collision": "SRT" if p.phase_srt else "MRT", "streaming": "in-place AA" if args.inplace else "moment representation, two grids of coefficients" if args.moments else "two-grid pull",
                       "algorithm": "Algorithm 1: six unfused kernels (comparison)" if args.unfused else "Algorithm 2: two fused kernels",
                       "parallelism": "replicas only" if world > 1 else "single GPU",
                       "timing": f"median of {REPEATS} back-to-back intervals of {K} steps (CUDA events, no per-kernel instrumentation inside); "
                                 f"value_min / value_max = slowest / fastest interval; kernel split from a separate instrumented pass",
                       "interval_ms": r["intervals"],
                       "l2": f"inputs larger than L2: {((2 * 14 + 8) if args.moments else (2 * (p.stencil_phase + p.stencil_hydro) + 5)) * N * esz / 1e9:.1f} GB "
                             "of state streamed every step vs 126 MB L2",
                       "bytes_per_cell": {"phase": r["b_phase"], "hydro": r["b_hydro"]},
                       "step_algorithmic_GBps": step_gbs, "step_frac_of_peak": step_gbs / peak, "step_frac_of_nominal": step_gbs / NOMINAL_HBM_GBS,
                       "phase_ms": r["phase_ms"], "hydro_ms": r["hydro_ms"], "cuda_graph_replays": r["graph_replays"],
                       "sum_phi": r["mass"], "finite": r.get("finite")},
            "clocks": r["clocks"],
            "e2e": {"value": r.get("e2e"), "unit": UNIT, "h2d_bytes_per_step": 4 * N * esz / K,
                    "d2h_bytes_per_step": 5 * N * esz / K, "steps": K,
                    "what": "acm_run_host: pinned host phi,u -> device, init, K steps, fields, phi,u,p -> host"},
            "gpu_launches": r["launches"],
            "roofline": roof,
        }
        if extras:
            out["also"] = extras
        if not args.no_cpu_baseline and world == 1:
            out["cpu_baseline"] = cpu_baseline(args.config, p, r["phi"], r["u"])
        print(json.dumps(out), flush=True)
    replicas.shutdown()


def run_decomposed(args, rank, local_rank, world):
    """--decompose: ONE global domain cut into z-slabs, one per rank (outside north_star, which
    is a single GPU).  Weak scaling: every rank owns a full copy of the workload's grid, the global domain is
    their stack along z (the workloads are periodic in z, so the stacked field is continuous); the ranks
    exchange halo planes every step (slab.py).  Not the default: `--gpus N` alone runs replicas."""
    import torch
    from paper_2012_06144_b200 import replicas
    from paper_2012_06144_b200.slab import PeerSlabRunner, SlabRunner, pad_planes

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU fallback")
    local_rank, dev = pick_device(local_rank)
    replicas.init(dist_backend(), dev)
    K, W = args.steps, max(args.warmup, 20)
    p, phi, u, name = workload(args.config)
    if p.wall_flags & 4:
        raise SystemExit("--decompose stacks the workload along z: it must be periodic in z")
    precision = args.precision
    esz = 8 if precision == "f64" else 4
    np_dtype = "float64" if precision == "f64" else "float32"
    phi_h = torch.from_numpy(phi.astype(np_dtype)).pin_memory()
    u_h = torch.from_numpy(u.astype(np_dtype)).pin_memory()
    pg = p.replace(nz=p.nz * world)
    if args.peer:       # the kernels read the neighbours' boundary planes directly (CUDA IPC / NVLink peer memory)
        run = (PeerSlabRunner.local(pg, 1, precision=precision, device=dev) if world == 1
               else PeerSlabRunner.distributed(pg, rank, world, precision=precision, device=dev))
    else:
        run = SlabRunner.distributed(pg, rank, world, precision=precision, device=dev, overlap=not args.no_overlap)
    slab = run.slabs[0]

    def load():
        slab.init(pad_planes(phi_h.to(dev, non_blocking=True), 0, p.nz), pad_planes(u_h.to(dev, non_blocking=True), 0, p.nz))
        run.refresh_halos()

    load()
    run.step(W)
    replicas.barrier(dev)
    launches0 = slab.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local_rank) as clk:
        e0.record()
        run.step(K)
        run.sync_halos()
        e1.record()
        replicas.barrier(dev)
    ms = replicas.max_over_ranks(e0.elapsed_time(e1), dev)
    launches = slab.launch_count - launches0
    N = p.ncells
    value = replicas.aggregate_mlups(N, K, ms, world)
    mass = slab.phi_mass()
    # evidence that every rank drove its own GPU and, in peer mode, that the neighbours' memory is reachable
    # (NCCL_DEBUG is left as the caller set it: NCCL_DEBUG=INFO shows the communicator and the transports)
    import torch.distributed as dist
    props = torch.cuda.get_device_properties(dev)
    nbrs = sorted({(rank - 1) % world, (rank + 1) % world} - {rank})
    mine = {"rank": rank, "device": local_rank, "name": props.name, "uuid": str(getattr(props, "uuid", "")),
            "launches": launches, "peak_alloc_GB": torch.cuda.max_memory_allocated(dev) / 1e9,
            "peer_access": {str(n): bool(torch.cuda.can_device_access_peer(local_rank, n % torch.cuda.device_count()))
                            for n in nbrs if n % torch.cuda.device_count() != local_rank}}
    ranks_info = [mine]
    if world > 1:
        ranks_info = [None] * world
        dist.all_gather_object(ranks_info, mine)
    # end to end: host -> device, init, halos, K steps, fields -> host
    po, uo = torch.empty_like(phi_h).pin_memory(), torch.empty_like(u_h).pin_memory()
    replicas.barrier(dev)
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record()
    load()
    run.step(K)
    c, uu, _ = run.fields(False)
    po.copy_(c, non_blocking=True)
    uo.copy_(uu, non_blocking=True)
    t1.record()
    replicas.barrier(dev)
    ms_e2e = replicas.max_over_ranks(t0.elapsed_time(t1), dev)
    if rank == 0:
        peak, peak_src = measured_peaks()
        b_phase, b_hydro = bytes_per_cell(p.stencil_phase, p.stencil_hydro, esz)
        step_gbs = (b_phase + b_hydro) * N * K / (ms * 1e-3) / 1e9      # N = cells of ONE rank: already the per-GPU rate
        out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms / K,
               "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": precision, "data": "synthetic",
               "config": {"workload": name + f", stacked {world}x along z and decomposed into {world} z-slabs",
                          "grid": [pg.nx, pg.ny, pg.nz], "stencils": [p.stencil_phase, p.stencil_hydro],
                          "parallelism": f"slab decomposition, {world} rank(s), " +
                                         ("peer mode: kernels read the neighbours' planes directly, one signal per kernel" if args.peer else
                                          "halo exchange " + ("overlapped on a second stream" if run.comm is not None else "in stream order")),
                          "l2": "inputs larger than L2 (per rank as in the single-GPU run)",
                          "bytes_per_cell": {"phase": b_phase, "hydro": b_hydro}, "sum_phi_rank0": mass,
                          "ranks": ranks_info, "gpus_active": len({r["uuid"] or r["device"] for r in ranks_info}),
                          "nccl": {"version": ".".join(str(v) for v in torch.cuda.nccl.version()) if world > 1 else None,
                                   "NCCL_DEBUG": os.environ.get("NCCL_DEBUG")}},
               "clocks": clk.summary(),
               "e2e": {"value": replicas.aggregate_mlups(N, K, ms_e2e, world), "unit": UNIT, "h2d_bytes_per_step": 4 * N * esz / K,
                       "d2h_bytes_per_step": 4 * N * esz / K, "steps": K,
                       "what": "per rank: pinned host phi,u -> device, init, halo exchange, K steps, phi,u -> host"},
               "gpu_launches": launches,
               "roofline": {"bound": "hbm", "kernel": "phase + hydro kernels of one rank (whole step, slab schedule)",
                            "achieved": step_gbs, "peak": peak, "unit": "GB/s", "frac": step_gbs / peak, "frac_of_nominal": step_gbs / NOMINAL_HBM_GBS,
                            "traffic": None, "peak_source": peak_src}}
        print(json.dumps(out), flush=True)
    replicas.shutdown()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="acm", choices=["acm", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"])
    ap.add_argument("--block", type=int, nargs=3, default=None)
    ap.add_argument("--cpt", type=int, nargs=2, default=None, metavar=("PHASE", "HYDRO"),
                    help="cells per thread of the phase / hydro kernel: 1, 2, or 0 = the library's default")
    ap.add_argument("--graph", type=int, default=None, choices=[-1, 0, 1], help="CUDA graphs in acm_step: -1 automatic (small grids), 0 never, 1 always")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the extra fp32 config-5 measurement of the default run")
    ap.add_argument("--inplace", action="store_true", help="in-place AA streaming (one grid per population set)")
    ap.add_argument("--moments", action="store_true", help="moment representation of the state (ACM_OPT_MOMENTS)")
    ap.add_argument("--moment-kernels", type=int, nargs=2, default=None, metavar=("MODE", "ZCHUNK"),
                    help="with --moments: acm_set_moment_kernels (mode -1 automatic | 0 direct | 1 tiled; planes per block, 0 = automatic)")
    ap.add_argument("--unfused", action="store_true", help="Algorithm 1 (six kernels per step) as a measured comparison")
    ap.add_argument("--decompose", action="store_true", help="one global domain in z-slabs with halo exchange instead of replicas")
    ap.add_argument("--peer", action="store_true", help="with --decompose: peer mode (no halo copies; kernels read neighbour memory)")
    ap.add_argument("--no-overlap", action="store_true", help="with --decompose: exchange in stream order (no second stream)")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    elif args.decompose:
        run_decomposed(args, rank, local_rank, world)
    else:
        run_acm(args, rank, local_rank, world)


if __name__ == "__main__":
    main()
