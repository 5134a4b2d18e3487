#!/usr/bin/env python
"""bench.py -- throughput of the GPUMCD hot path on B200 (one JSON line on stdout).

    python bench.py --gpus N --steps K --warmup W            # the CUDA library (this repo)
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle, timed as it stands
    python bench.py --paper-tables [--steps K]               # PAPER.md Tab. IV-VI measured here (markdown)
    python bench.py --ablation [--steps K]                   # Tab. VI / L180 / L352 ablation on configs 2-5 (JSON)

A "step" is one gpumcd_run of the whole hot path (source, photon and electron transport with all
secondaries, tally, finalize) over one batch of synthetic histories.  BASELINE.json quotes its metric on
no single configuration, so the workload at N = 1 is the largest single-GPU one, config 5 (18 MV spectrum,
10x10 cm^2 field, 1e8 histories, 256x256x128 CT-like phantom at 0.2 cm); the same figures for all five
configurations are in the line's `per_config` block.  --config selects another headline.

Metric: coupled photon-electron histories/s (value) and condensed-history steps/s (ch_steps_per_s).
Multi-GPU (--gpus N under torchrun): every rank simulates its own disjoint history range (weak
scaling) and the dose grids are summed with one all-reduce per step.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# thread-instructions one condensed-history step needs at minimum, and the
# issue peak = 148 SMs x 4 schedulers x 32 lanes x 1 inst/clk x max SM clock.
ALG_INST_PER_CH_STEP = 330.0
N_SM, N_SCHED, LANES = 148, 4, 32


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return d, "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """Samples SM clock and throttle reasons while the timed region runs (NVML every 20 ms; falls back to
    `nvidia-smi -lms 200` when the NVML binding is unavailable)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc, self.thread = index, [], None, None
        self.sm, self.smax, self.reasons, self._stop = [], [], set(), threading.Event()

    def _nvml_loop(self, nv, h):
        names = {"hw_slowdown": nv.nvmlClocksThrottleReasonHwSlowdown,
                 "hw_thermal_slowdown": nv.nvmlClocksThrottleReasonHwThermalSlowdown,
                 "sw_thermal_slowdown": nv.nvmlClocksThrottleReasonSwThermalSlowdown,
                 "sw_power_cap": nv.nvmlClocksThrottleReasonSwPowerCap}
        smax = float(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
        while not self._stop.is_set():
            try:
                self.sm.append(float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)))
                self.smax.append(smax)
                mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for n, bit in names.items():
                    if mask & bit:
                        self.reasons.add(n)
            except Exception:
                pass
            self._stop.wait(0.02)

    def start(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            # NVML enumerates physical devices: map the CUDA ordinal through CUDA_VISIBLE_DEVICES when it lists indices
            vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
            idx = self.index
            if vis and all(x.strip().isdigit() for x in vis.split(",")):
                idx = int(vis.split(",")[self.index])
            h = nv.nvmlDeviceGetHandleByIndex(idx)
            self.thread = threading.Thread(target=self._nvml_loop, args=(nv, h), daemon=True)
            self.thread.start()
            return
        except Exception:
            self.thread = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        self._stop.set()
        if self.thread:
            self.thread.join(timeout=1)
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except subprocess.TimeoutExpired:
                self.proc.kill()
        sm, smax, reasons = list(self.sm), list(self.smax), set(self.reasons)
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                smax.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_rate(w, seconds: float, threads: int = 0):
    """Time the oracle, as it stands, on a bounded sample of workload ``w`` sized for ~``seconds``."""
    import oracle
    n = max(2000, min(20000, w.n_histories))
    oracle.run_workload(w, n, n_threads=threads)                  # first call: builds / loads the library, warms up
    while True:
        t0 = time.perf_counter()
        r = oracle.run_workload(w, n, n_threads=threads)
        dt = time.perf_counter() - t0
        if dt >= 0.5 * seconds or n >= w.n_histories:
            return n, dt, r.counters
        n = int(min(w.n_histories, max(2 * n, n * seconds / max(dt, 1e-3))))


def reference_arm(args):
    """The base contract's reference arm for this tier: the CPU oracle on the box's host cores."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    from paper_1101_1245_b200.inputs import make_config
    w = make_config(args.config)
    cores = os.cpu_count() or 1
    n = args.ref_histories
    for _ in range(args.warmup):
        oracle.run_workload(w, max(n // 10, 1000))
    t0 = time.perf_counter()
    steps_ch = 0
    for k in range(args.steps):
        r = oracle.run(w.density, w.material, w.voxel_cm, w.tables, w.source, n, seed=w.seed + k)
        steps_ch += r.counters["ch_steps"]
    dt = time.perf_counter() - t0
    value = args.steps * n / dt
    line = {
        "impl": "reference", "metric": "coupled photon-electron histories/s", "value": value, "unit": "histories/s",
        "ch_steps_per_s": steps_ch / dt, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "histories_per_step": n, "note": "bounded sample of the workload per step"},
        "cpu_baseline": {"value": value, "unit": "histories/s", "cores": cores, "kind": "oracle",
                         "sample": f"{n} histories of {w.name} per step, {args.steps} steps"},
        "e2e": {"value": value, "unit": "histories/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


PAPER_TAB4 = {(1, 1): 0.118, (2, 1): 0.147, (3, 1): 0.162, (1, 0): 0.269, (2, 0): 0.275, (3, 0): 0.366}  # s, GTX480


def time_gpu(g, torch, w, n, reps, **opts):
    """Median device time (ms) of gpumcd_run over ``reps`` runs after three warm-up runs, L2 flushed in between."""
    dev = torch.device("cuda:0")
    rho = torch.from_numpy(w.density).to(dev)
    mat = torch.from_numpy(w.material).to(dev)
    dose = torch.empty(rho.shape, dtype=torch.float32, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    ts = []
    with g.gpumcd_create(rho, mat, w.voxel_cm, w.tables, g.gpumcd_default_options(**opts)) as ctx:
        g.gpumcd_set_source(ctx, w.source)
        for k in range(reps + 3):
            flush.fill_(k)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            a.record()
            g.gpumcd_run(ctx, n, w.seed + k, dose)
            b.record()
            torch.cuda.synchronize()
            if k >= 3:
                ts.append(a.elapsed_time(b))
        c = g.gpumcd_get_counters(ctx)
    return float(np.median(ts)), c


def s_gpu(g, torch, ev, w, n, nb=40, **opts):
    dev = torch.device("cuda:0")
    rho = torch.from_numpy(w.density).to(dev)
    mat = torch.from_numpy(w.material).to(dev)
    dose = torch.empty(rho.shape, dtype=torch.float32, device=dev)
    sig = torch.empty(rho.shape, dtype=torch.float32, device=dev)
    with g.gpumcd_create(rho, mat, w.voxel_cm, w.tables, g.gpumcd_default_options(**opts)) as ctx:
        g.gpumcd_set_source(ctx, w.source)
        g.gpumcd_run_uncertainty(ctx, n, nb, w.seed, dose, sig)
        torch.cuda.synchronize()
    return ev.relative_uncertainty(dose.cpu().numpy().astype(np.float64), sig.cpu().numpy().astype(np.float64), 0.2)


def paper_tables(args):
    """--paper-tables: PAPER.md Tab. IV, V and VI measured here (markdown on stdout instead of the JSON line).
    Tab. V's reference systems (EGSnrc, DPM) are not available: the reference is the CPU oracle (this file's
    cpu_baseline leg), timed on a bounded share of the histories.  Tab. VI's base scheme is scheduler 0."""
    import torch

    import oracle
    import paper_1101_1245_b200 as g
    from paper_1101_1245_b200 import evaluation as ev
    from paper_1101_1245_b200.inputs import ELECTRON, PHOTON, make_paper_geometry

    assert torch.cuda.is_available(), "needs a CUDA device"
    cores = os.cpu_count() or 1
    rows4, rows5, rows6 = [], [], []
    for particle, pname in ((ELECTRON, "electrons"), (PHOTON, "photons")):
        for geom in (1, 2, 3):
            w = make_paper_geometry(geom, particle)
            n = w.n_histories
            t1, c = time_gpu(g, torch, w, n, args.steps)
            t0, _ = time_gpu(g, torch, w, n, args.steps, scheduler=0)
            ta, _ = time_gpu(g, torch, w, n, args.steps, cta_threads=512)
            tb, _ = time_gpu(g, torch, w, n, args.steps, cta_threads=1024)
            tm, cm = time_gpu(g, torch, w, n, args.steps, hom_tol=0.1)
            s = s_gpu(g, torch, ev, w, n)
            eps = ev.efficiency(s, t1 * 1e-3)
            s_m = s_gpu(g, torch, ev, w, n, hom_tol=0.1)      # R32: the one-point deposit adds variance per step
            eps_m = ev.efficiency(s_m, tm * 1e-3)
            # the oracle on a bounded sample; s scales as 1/sqrt(N) (L334), time as N
            n_o = max(2000, int(n * args.oracle_fraction))
            tw = time.perf_counter()
            e, sq, _ = oracle.run_moments(w.density, w.material, w.voxel_cm, w.tables, w.source, n_o, w.seed)
            t_o = (time.perf_counter() - tw) * n / n_o
            mass = w.density.astype(np.float64) * w.voxel_cm ** 3
            s_o = ev.relative_uncertainty(e / n_o / mass, oracle.uncertainty_from_moments(e, sq, n_o) / mass, 0.2)
            s_o *= np.sqrt(n_o / n)
            eps_o = ev.efficiency(s_o, t_o)
            rows4.append(f"| {pname} | Geom{geom} | {n:.0e} | {t1:.3f} | {n / t1 / 1e3:.1f} | {c['ch_steps'] / t1 / 1e6:.1f} | "
                         f"{PAPER_TAB4[(geom, particle)] * 1e3:.0f} |")
            rows5.append(f"| {pname} | Geom{geom} | {t_o:.1f} | {t_o / (t1 * 1e-3):.0f} | {s * 100:.3f} | {s_o * 100:.3f} | "
                         f"{eps:.3g} | {eps_o:.3g} | {eps / eps_o:.0f} |")
            rows6.append(f"| {pname} | Geom{geom} | {t0:.3f} | {t0 / t1:.2f} | {t0 / ta:.2f} | {t0 / tb:.2f} | "
                         f"{t0 / tm:.2f} ({tm:.3f} ms, {c['ch_steps'] / cm['ch_steps']:.2f} x fewer steps) | "
                         f"{s_m * 100:.3f} ({s * 100:.3f}) | {eps_m / eps:.2f} |")
    print("## Tab. IV analogue: absolute times of `gpumcd_run` (device time, CUDA events, median of "
          f"{args.steps}, L2 flushed between runs)\n")
    print("| particles | geometry | histories | ms | M histories/s | G CH steps/s | paper, GTX480, ms (context) |")
    print("|---|---|---|---|---|---|---|")
    print("\n".join(rows4))
    print(f"\n## Tab. V analogue: against the CPU oracle on {cores} host cores (timed on "
          f"{args.oracle_fraction:.0%} of the histories and scaled; a deliberately plain program, not EGSnrc or DPM)\n")
    print("| particles | geometry | T_oracle, s (scaled) | A = T_oracle / T | s, % (Eq. 12, device, 40 batches) | "
          "s, % (oracle, history by history, scaled by sqrt(N)) | eps (Eq. 11), 1/s | eps oracle | A_eps |")
    print("|---|---|---|---|---|---|---|---|---|")
    print("\n".join(rows5))
    print("\n## Tab. VI analogue: scheduling strategies against the paper's base scheme (scheduler 0)\n")
    print("| particles | geometry | T_base = scheduler 0, ms | A, scheduler 1 (default CTA size) | A, 512 threads/SM | "
          "A, 1024 threads/SM | A, scheduler 1 + multi-voxel steps (hom_tol 0.1, another step algorithm: DESIGN.md R32) | "
          "s, % with multi-voxel steps (Eq. 4 steps) at equal N | efficiency gain of multi-voxel steps, eps_m / eps (Eq. 11) |")
    print("|---|---|---|---|---|---|---|---|---|")
    print("\n".join(rows6))



def ablation(args):
    """--ablation: the paper's divergence-reduction ablation (Tab. VI; compaction interval N, L180; pool, L182;
    "grouping particles", L352) restated for this scheduler, on configs 2-5 at full size: scheduler 0 (the paper's
    base scheme, with its wave size and bank factor d, L166) against scheduler 1, CTA size, tally mode, the
    high-water marks that set how much work of one type a warp does before it picks up the other type, the
    drain threshold, the stack capacity, and multi-voxel steps.  One JSON object on stdout; ms = median device
    time of gpumcd_run over --steps runs after 3 warm-up runs, L2 flushed in between."""
    import torch

    import paper_1101_1245_b200 as g
    from paper_1101_1245_b200.inputs import make_config
    assert torch.cuda.is_available(), "needs a CUDA device"
    variants = [("default", {}),
                ("scheduler0", {"scheduler": 0}), ("scheduler0_wave2^18", {"scheduler": 0, "wave_size": 1 << 18}),
                ("scheduler0_wave2^22_d4", {"scheduler": 0, "wave_size": 1 << 22, "bank_factor": 4}),
                ("cta1024", {"cta_threads": 1024}),
                ("tally_warp", {"tally_mode": 1}), ("tally_fixed", {"tally_mode": 2}),
                ("round1_marks80_160_stack1024", {"bank_high_g": 80, "bank_high_e": 160, "warp_stack": 1024, "steps_per_refill": 1}),
                ("marks80_160", {"bank_high_g": 80, "bank_high_e": 160}), ("marks24_40", {"bank_high_g": 24, "bank_high_e": 40}),
                ("marks320_640", {"bank_high_g": 320, "bank_high_e": 640}), ("marks1000_2000", {"bank_high_g": 1000, "bank_high_e": 2000}),
                ("low24", {"bank_low": 24}), ("low32", {"bank_low": 32}),
                ("stack256", {"warp_stack": 256}), ("stack1024", {"warp_stack": 1024}), ("stack2048", {"warp_stack": 2048}),
                ("stack4096", {"warp_stack": 4096}), ("stack16384", {"warp_stack": 16384}),
                ("cta512", {"cta_threads": 512}),
                ("steps_per_refill1", {"steps_per_refill": 1}), ("steps_per_refill2", {"steps_per_refill": 2}),
                ("steps_per_refill4", {"steps_per_refill": 4}), ("steps_per_refill8", {"steps_per_refill": 8}),
                ("hom_tol0.1", {"hom_tol": 0.1})]
    small = ("default", "scheduler0", "tally_warp", "tally_fixed")   # config 1 (1e5 histories): these only
    out = {"what": "ms per gpumcd_run (median of %d, device time), full history counts" % args.steps, "configs": {}}
    for c in (1, 2, 3, 4, 5):
        w = make_config(c)
        row = {}
        for name, o in variants:
            if c == 1 and name not in small:
                continue
            if c == 5 and o.get("scheduler") == 0 and o.get("wave_size", 1 << 20) > (1 << 20):
                continue                      # 4 queues x 2^22 x 4 x 48 B does not leave room for the rest
            print(f"ablation: {w.name} {name}", file=sys.stderr, flush=True)
            t, cnt = time_gpu(g, torch, w, w.n_histories, args.steps, **o)
            row[name] = {"ms": round(t, 4), "ch_steps": cnt["ch_steps"], "bank_high_water": cnt["bank_high_water"]}
        out["configs"][w.name] = row
    print(json.dumps(out))
    return 0


def load_traffic_table():
    """profiles/ncu_traffic.csv: DRAM bytes per launch of k_persistent from the kept `ncu --set full` captures
    (dram__bytes_read.sum + dram__bytes_write.sum), one row per workload, written next to each ncu summary."""
    out = {}
    path = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if os.path.exists(path):
        for line in open(path):
            f = [x.strip() for x in line.split(",")]
            if len(f) >= 4 and not line.startswith("#") and f[0] != "workload":
                out[f[0]] = {"read": float(f[1]), "write": float(f[2]), "capture": f[3]}
    return out


# algorithmic DRAM bytes of one run: first touch of the packed phantom (4 B / voxel), the tally zeroed, read and
# written back (2 x 8 B / voxel) and the dose written (4 B / voxel); DESIGN.md 7 "Rooflines"
def algorithmic_dram_bytes(w):
    return int(w.density.size) * (4 + 16 + 4)


def measure(g, torch, dist, w, n, opts, steps, warmup, dev, rank, world, flush, e2e=True, probe=True):
    """Time `steps` runs of workload `w` (device time by CUDA events on the launching stream, L2 flushed in between),
    then the same through the host entry points.  Returns the figures of one bench line."""
    from paper_1101_1245_b200.sharding import combine_dose
    rho = torch.from_numpy(w.density).to(dev)
    mat = torch.from_numpy(w.material).to(dev)
    dose = torch.empty(rho.shape, dtype=torch.float32, device=dev)
    opt = g.gpumcd_default_options(**opts)
    ctx = g.gpumcd_create(rho, mat, w.voxel_cm, w.tables, opt)
    g.gpumcd_set_source(ctx, w.source)
    g.gpumcd_set_history_offset(ctx, rank * n)       # disjoint history ranges per rank
    g.gpumcd_set_profiling(ctx, True)

    def step(seed):
        g.gpumcd_run(ctx, n, seed, dose)
        if dist:
            combine_dose(dose, n, world * n, dist)    # "the resulting dose arrays are summed" (L188)

    for k in range(warmup):
        step(w.seed + k)
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    ch_steps = flights = launches = 0
    ms_e = 0.0
    n_e = 0
    wall0 = time.perf_counter()
    for k in range(steps):
        g.gpumcd_release_l2(ctx)                       # (l2_persist: every timed step starts from a cold L2 too)
        flush.fill_(k & 0xFF)                          # evict the phantom / tally / tables from L2
        torch.cuda.synchronize()
        ev[k][0].record()
        step(w.seed + 100 + k)
        ev[k][1].record()
        torch.cuda.synchronize()
        c = g.gpumcd_get_counters(ctx)
        p = g.gpumcd_get_profile(ctx)
        ch_steps += c["ch_steps"]
        flights += c["photon_flights"]
        launches += p["launches"]
        ms_e += p["ms_electron"] + p["ms_photon"]
        n_e += p["n_electron"] + p["n_photon"]
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    wall = time.perf_counter() - wall0
    t_ms = sum(a.elapsed_time(b) for a, b in ev)
    if dist:
        tt = torch.tensor([t_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        t_ms = float(tt.item())
        agg = torch.tensor([ch_steps, flights], dtype=torch.float64, device=dev)
        dist.all_reduce(agg)
        ch_steps, flights = (float(x) for x in agg.tolist())
    t_s = t_ms * 1e-3
    out = {"workload": w.name, "histories_per_step_per_gpu": n, "ms_per_step": t_ms / steps,
           "value": world * steps * n / t_s, "ch_steps_per_s": ch_steps / t_s, "photon_flights_per_s": flights / t_s,
           "gpu_launches": int(launches), "wall_s_timed_region": wall,
           "bank_high_water": int(c["bank_high_water"])}

    # ---- roofline of the dominant kernel (the transport kernel): issue-rate bound
    peaks, peak_kind = measured_peaks()
    peak_inst = N_SM * N_SCHED * LANES * peaks.get("sm_max_mhz", 1965.0) * 1e6
    local_ch = ch_steps / world
    achieved = ALG_INST_PER_CH_STEP * local_ch / (ms_e * 1e-3) if ms_e > 0 else None
    traffic = load_traffic_table().get(w.name) if n == w.n_histories else None
    out["roofline"] = {"bound": "alu", "kernel": "k_persistent (transport + tally + finalize)" if opt.scheduler == 1 else "transport passes",
                       "achieved": achieved, "peak": peak_inst,
                       "unit": "thread-inst/s", "frac": (achieved / peak_inst) if achieved else None,
                       "traffic": (traffic["read"] + traffic["write"]) if traffic else None,
                       "traffic_source": traffic["capture"] if traffic else None,
                       "algorithmic_dram_bytes": algorithmic_dram_bytes(w),
                       "peak_source": f"148 SMs x 4 x 32 x sm_max_mhz ({peak_kind})",
                       "kernel_ms_per_step": ms_e / steps, "kernel_launches_per_step": n_e / steps,
                       "kernel_share_of_step": ms_e / t_ms if t_ms else None,
                       "alg_inst_per_ch_step": ALG_INST_PER_CH_STEP}

    # ---- secondary rooflines (BASELINE.json north_star): the tally against the measured atomic rate of the L2
    # (gpumcd_probe_tally: the same grid, the field's footprint, nothing but atomic adds of the tally's type), and the
    # DRAM traffic of the ncu capture against the measured HBM copy bandwidth
    if probe:
        tally_peak = g.gpumcd_probe_tally(ctx, 200_000_000)
        tally_rate = local_ch / t_s
        out["roofline_tally"] = {"bound": "l2_atomic", "achieved": tally_rate, "peak": tally_peak,
                                 "unit": ("u64" if opt.tally_mode == 2 else "fp64") + " atomic adds/s",
                                 "frac": tally_rate / tally_peak, "tally_mode": int(opt.tally_mode),
                                 "what": "one add per condensed-history step against gpumcd_probe_tally under this field"}
    out["roofline_hbm"] = None
    if traffic and ms_e > 0:
        gbs = (traffic["read"] + traffic["write"]) / (ms_e / max(n_e, 1) * 1e-3) / 1e9
        out["roofline_hbm"] = {"bound": "hbm", "achieved": gbs, "peak": peaks.get("hbm_gbs"), "unit": "GB/s",
                               "frac": gbs / peaks.get("hbm_gbs"),
                               "what": f"ncu DRAM bytes per launch / kernel time ({peak_kind} copy bandwidth)"}

    # ---- end to end through the host entry points: every step copies that step's inputs (the phantom volumes,
    # from pinned host memory) to the device and the resulting dose grid back to the host
    out["e2e"] = None
    if e2e:
        rho_h = torch.from_numpy(w.density).pin_memory()
        mat_h = torch.from_numpy(w.material).pin_memory()
        dose_h = torch.empty(rho.shape, dtype=torch.float32).pin_memory()
        rho_np, mat_np, dose_np = rho_h.numpy(), mat_h.numpy(), dose_h.numpy()

        def e2e_step(seed):
            g.gpumcd_set_phantom_host(ctx, rho_np, mat_np)
            g.gpumcd_set_source(ctx, w.source)
            g.gpumcd_run_host(ctx, n, seed, dose_np)          # returns after the device-to-host copy

        g.gpumcd_set_profiling(ctx, False)
        for k in range(warmup):
            e2e_step(w.seed + 300 + k)
        if dist:
            dist.barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for k in range(steps):
            e2e_step(w.seed + 400 + k)
        torch.cuda.synchronize()
        e2e_t = (time.perf_counter() - t0) / steps
        if dist:
            tt = torch.tensor([e2e_t], dtype=torch.float64, device=dev)
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            e2e_t = float(tt.item())
        blob_bytes = 4 * (w.tables.photon.size + w.tables.electron.size + w.tables.ms_a.size + 2 * w.tables.n_energy)
        out["e2e"] = {"value": world * n / e2e_t, "unit": "histories/s",
                      "h2d_bytes_per_step": int(rho.numel() * 5 + blob_bytes), "d2h_bytes_per_step": int(rho.numel() * 4),
                      "ms_per_step": e2e_t * 1e3,
                      "what": "gpumcd_set_phantom_host + gpumcd_set_source + gpumcd_run_host per step, wall clock, pinned host buffers"}
    out["options"] = {"scheduler": int(opt.scheduler), "hom_tol": float(opt.hom_tol), "wave_size": int(opt.wave_size),
                      "tally_mode": int(opt.tally_mode), "cta_threads": int(opt.cta_threads) or 512,
                      "steps_per_refill": int(opt.steps_per_refill) or 4, "warp_stack": int(opt.warp_stack)}
    g.gpumcd_destroy(ctx)
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5,
                    help="the headline workload (default 5: the largest single-GPU configuration of BASELINE.json)")
    ap.add_argument("--no-per-config", action="store_true",
                    help="skip the per_config block (the other four configurations, measured the same way)")
    ap.add_argument("--histories", type=int, default=0, help="override histories per step (0 = the config's)")
    ap.add_argument("--scheduler", type=int, default=-1)
    ap.add_argument("--wave", type=int, default=0, help="override wave_size (0 = library default)")
    ap.add_argument("--cta-threads", type=int, default=0, help="override cta_threads (0 = the library's choice)")
    ap.add_argument("--tally-mode", type=int, default=-1, help="override tally_mode (-1 = the library's default)")
    ap.add_argument("--warp-stack", type=int, default=0, help="override warp_stack (0 = library default)")
    ap.add_argument("--l2-persist", type=int, default=-1, help="override l2_persist (-1 = library default)")
    ap.add_argument("--opt", action="append", default=[], help="any other gpumcd_options field, name=value (repeatable)")
    ap.add_argument("--hom-tol", type=float, default=0.0,
                    help="multi-voxel electron steps (gpumcd_options.hom_tol; 0 = Eq. 4 as printed, the default)")
    ap.add_argument("--ref-histories", type=int, default=200_000)
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--paper-tables", action="store_true", help="print PAPER.md Tab. IV-VI measured here (markdown)")
    ap.add_argument("--ablation", action="store_true",
                    help="scheduling / tally ablation of PAPER.md Tab. VI and L180, L352 on configs 2-5 (JSON on stdout)")
    ap.add_argument("--oracle-fraction", type=float, default=0.02,
                    help="--paper-tables: share of the histories the oracle is timed on")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return reference_arm(args)
    if args.paper_tables:
        return paper_tables(args)
    if args.ablation:
        return ablation(args)

    import torch

    import paper_1101_1245_b200 as g
    from paper_1101_1245_b200 import build as cuda_build
    from paper_1101_1245_b200.inputs import make_config

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    if rank == 0:
        cuda_build.build()
    if dist:
        dist.barrier()
    g.load_library()

    opts = {}
    if args.scheduler >= 0:
        opts["scheduler"] = args.scheduler
    if args.wave > 0:
        opts["wave_size"] = args.wave
    if args.cta_threads > 0:
        opts["cta_threads"] = args.cta_threads
    if args.hom_tol > 0:
        opts["hom_tol"] = args.hom_tol
    if args.tally_mode >= 0:
        opts["tally_mode"] = args.tally_mode
    if args.warp_stack > 0:
        opts["warp_stack"] = args.warp_stack
    if args.l2_persist >= 0:
        opts["l2_persist"] = args.l2_persist
    for kv in args.opt:
        k, v = kv.split("=")
        opts[k] = float(v) if "." in v else int(v)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    w = make_config(args.config)
    n = args.histories or w.n_histories
    sampler = ClockSampler(local)
    sampler.start()
    head = measure(g, torch, dist, w, n, opts, args.steps, args.warmup, dev, rank, world, flush, e2e=not args.no_e2e)
    per_config = {}
    if not args.no_per_config and not args.histories:
        for c in (1, 2, 3, 4, 5):
            if c == args.config:
                per_config[f"cfg{c}"] = {k: head[k] for k in ("workload", "histories_per_step_per_gpu", "ms_per_step", "value",
                                                               "ch_steps_per_s", "photon_flights_per_s", "roofline",
                                                               "roofline_tally", "roofline_hbm", "e2e")}
                continue
            wc = make_config(c)
            m = measure(g, torch, dist, wc, wc.n_histories, opts, args.steps, args.warmup, dev, rank, world, flush,
                        e2e=not args.no_e2e)
            per_config[f"cfg{c}"] = {k: m[k] for k in ("workload", "histories_per_step_per_gpu", "ms_per_step", "value",
                                                        "ch_steps_per_s", "photon_flights_per_s", "roofline",
                                                        "roofline_tally", "roofline_hbm", "e2e")}
            del wc
    clocks = sampler.stop()

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        ns, dt, oc = oracle_rate(w, args.cpu_seconds)
        cpu = {"value": ns / dt, "unit": "histories/s", "cores": os.cpu_count(), "kind": "oracle",
               "ch_steps_per_s": oc["ch_steps"] / dt,
               "sample": f"first {ns} histories of {w.name}, OpenMP over all host cores, {dt:.1f} s"}

    if rank == 0:
        o = head["options"]
        line = {
            "metric": "coupled photon-electron histories/s", "value": head["value"], "unit": "histories/s",
            "ch_steps_per_s": head["ch_steps_per_s"], "photon_flights_per_s": head["photon_flights_per_s"],
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": head["ms_per_step"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "histories_per_step_per_gpu": n, "scheduler": o["scheduler"], "hom_tol": o["hom_tol"],
                       "wave_size": o["wave_size"], "cta_threads": o["cta_threads"],
                       "l2": "flushed between timed steps (512 MiB write)",
                       "tally": {0: "fp64 atomics", 1: "warp-aggregated fp64 atomics", 2: "64-bit fixed-point atomics"}[o["tally_mode"]],
                       "parallelism": f"histories x{world}"},
            "clocks": clocks, "e2e": head["e2e"], "gpu_launches": head["gpu_launches"], "roofline": head["roofline"],
            "roofline_tally": head.get("roofline_tally"), "roofline_hbm": head["roofline_hbm"], "cpu_baseline": cpu,
            "wall_s_timed_region": head["wall_s_timed_region"], "bank_high_water": head["bank_high_water"],
            "per_config": per_config or None,
        }
        print(json.dumps(line))
    if dist:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
