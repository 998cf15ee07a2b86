#!/usr/bin/env python
"""bench.py -- the measurement contract.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--impl ours|reference]

One STEP = one pass of the whole hot path over one batch of
synthetic markers in random order: bind -> bin (counting sort by cell) -> zero grids -> tile
deposit of charge (+ parallel current).  Default workload: BASELINE.json configs[3] (the config
the >= 50 % HBM-roofline target is quoted on; 2^26 markers, 256x512x128 cells, N_L = 4, rho and
j_par), which fits one B200.

Prints ONE JSON line (rank 0).  `value` = Larmor points/s of the whole job with the markers
already resident in HBM; `e2e` = the same through orb_deposit_host with HOST (pinned) marker
arrays and host grids, copies inside the timed region; `roofline` = algorithmic bytes of the
deposit kernel / its CUDA-event duration against MEASURED_PEAKS.json; `cpu_baseline` = the
CPU oracle, as it stands, on a bounded sample of the same workload.

`--impl reference` times the oracle (single thread, host cores) on the same workload, each
step a bounded sample; rank 0 only.
"""
from __future__ import annotations

import argparse
import dataclasses
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_1908_02219_b200 import replicas as R  # noqa: E402
from paper_1908_02219_b200 import workloads as W  # noqa: E402

METRIC = "gyro-averaged Larmor points deposited/sec and achieved HBM GB/s (% of roofline)"
UNIT = "Larmor points/s"
HBM_FALLBACK_GBS = 6650.0      # /opt/skills/guides/B200_PROFILING.md fallback
HBM_NOMINAL_GBS = 8000.0       # the "~8 TB/s" north_star quotes
L2_BYTES = 126 << 20
# fp64 roof of the scatter arithmetic: measured DFMA/DMMA rate of this pool's
# B200 (profiles/r01_microbench.md: 17.9 TFMA/s = 61.7 of 64 lanes/clk/SM at 1965 MHz); nominal
# 148 SM x 64 lanes x 2 flop x 1.965 GHz = 37.2 TFLOP/s.
FP64_MEASURED_TFLOPS = 35.8    # fallback if the live probe (orb_probe_dfma) fails
FP64_NOMINAL_TFLOPS = 37.2

TRAFFIC_JSON = os.path.join(ROOT, "profiles", "r02_traffic.json")


def ncu_traffic(workload: str, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel, from the
    committed `ncu --set full` capture (profiles/r02_traffic.json, written by
    `python -m paper_1908_02219_b200.profile_traffic`).  Keyed by workload AND by the hash of the
    kernel sources: a capture of other sources is stale and reads as null, with the reason."""
    from paper_1908_02219_b200 import profile_traffic as PT
    try:
        with open(TRAFFIC_JSON) as f:
            db = json.load(f)
    except Exception:  # noqa: BLE001
        return None, "no capture committed (profiles/r02_traffic.json missing)"
    e = db.get("entries", {}).get(workload)
    if not e:
        return None, "no ncu capture of workload %s" % workload
    if e.get("kernel_source_sha16") != PT.kernel_source_hash():
        return None, "stale: kernel sources changed since the capture (%s)" % e.get("captured", "?")
    if kernel not in e.get("kernel", ""):
        return None, "capture is of %s, not %s" % (e.get("kernel"), kernel)
    return int(e["dram_bytes"]), "profiles/r02_traffic.json (%s)" % e.get("source", "")


def measured_hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    REASONS = {
        0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap",
        0x8: "hw_slowdown", 0x10: "sync_boost", 0x20: "sw_thermal_slowdown",
        0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting",
    }

    def __init__(self, index=0, period_s=0.004):
        self.index, self.period = index, period_s
        self.samples, self.reasons, self.sm_max = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:  # noqa: BLE001
            self.err = repr(e)

    def _loop(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                bits = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                for b, name in self.REASONS.items():
                    if bits & b and name != "gpu_idle":
                        self.reasons.add(name)
            except Exception:  # noqa: BLE001
                pass
            self._stop.wait(self.period)

    def start(self):
        if self.ok:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()

    def stop(self):
        if self._thr:
            self._stop.set()
            self._thr.join()

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.sm_max,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def pick_config(name: str, rank: int):
    cfg = W.CONFIGS[name]
    return dataclasses.replace(cfg, seed=R.replica_seed(cfg.seed, rank))


def describe(cfg):
    return ("%s: grid %dx%dx%d cells, %d markers fp64 SoA, %s N_L%s, rho_star=1/%d, q=%g, %s, %s order"
            % (cfg.name, cfg.ns, cfg.ntheta, cfg.nphi, cfg.n_markers,
               "adaptive" if cfg.adaptive else "fixed",
               ("=%d..%d" % (cfg.n_fixed, cfg.n_max)) if cfg.adaptive else ("=%d" % cfg.n_fixed),
               round(1 / cfg.rho_star), cfg.q, "rho+jpar" if cfg.current else "rho only", cfg.order))


def config_json(cfgs, world, workload=None, extra=None):
    if not isinstance(cfgs, (list, tuple)):
        cfgs = [cfgs]
    c = {"workload": " + ".join(describe(x) for x in cfgs) if len(cfgs) > 1 else describe(cfgs[0]),
         "step": "per species: bind + bin + tile deposit; grids zeroed once",
         "l2_policy": "inputs (%.2f GB markers) larger than the 126 MB L2; no flush needed"
                      % (sum(x.n_markers for x in cfgs) * 48 / 1e9),
         "parallelism": "replicas x%d (no sharding, no collective)" % world if world > 1 else "1 GPU"}
    if workload:
        c["name"] = workload
    if extra:
        c.update(extra)
    return c


def oracle_sample(cfg, m, n_sample):
    """Times the oracle, single-threaded and as it stands, on the first n_sample markers."""
    import oracle as O
    og = O.geom(cfg.ns, cfg.ntheta, cfg.nphi, r0=cfg.r0, a=cfg.a, b0=cfg.b0, rho_star=cfg.rho_star,
                q=cfg.q)
    op = (O.policy_adaptive(cfg.n_fixed, cfg.n_max, cfg.rho_ref) if cfg.adaptive
          else O.policy_fixed(cfg.n_fixed))
    O.lib()
    arrs = [np.ascontiguousarray(m[f][:n_sample]) for f in W.FIELDS]
    shape = O.grid_shape(og)
    rho = np.zeros(shape)
    jpar = np.zeros(shape) if cfg.current else None
    t0 = time.perf_counter()
    _, _, npts = O.deposit(og, op, *arrs, current=cfg.current, rho=rho, jpar=jpar)
    dt = time.perf_counter() - t0
    return npts, dt


# ------------------------------------------------------------------------------------------
def run_reference(args):
    rank, _, world = R.env_rank()
    if rank != 0:
        return 0
    cfg = pick_config(W.WORKLOADS[args.workload][0], 0)
    n_sample = min(args.ref_sample, cfg.n_markers)
    m = W.generate(W.scaled(cfg, n_sample))
    for _ in range(args.warmup):
        oracle_sample(cfg, m, n_sample)
    pts, secs = 0, 0.0
    for _ in range(args.steps):
        n, dt = oracle_sample(cfg, m, n_sample)
        pts += n
        secs += dt
    value = pts / secs
    sample = "first %d markers of %s per step (%d Larmor points), single thread" % (
        n_sample, cfg.name, pts // max(args.steps, 1))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": config_json(cfg, 1, args.workload, {"step": "oracle_deposit on a bounded sample"}),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0, "host_cores": os.cpu_count(),
    }
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------
class Species:
    """One marker species of the workload: pinned host arrays, device copies, its grid handle."""

    def __init__(self, cfg, dev, local_rank, B, torch, binning):
        self.cfg = cfg
        n = cfg.n_markers
        self.host = {f: torch.empty(n, dtype=torch.float64, pin_memory=True) for f in W.FIELDS}
        self.m = {f: self.host[f].numpy() for f in W.FIELDS}
        W.generate(cfg, out=self.m)
        self.d = {f: self.host[f].to(dev, non_blocking=True) for f in W.FIELDS}
        self.g = B.grid_for(cfg, device=local_rank)
        self.pol = B.policy_for(cfg)
        self.bind_flags = (B.ORB_MARKERS_SORTED if cfg.order == "sorted"
                           else B.ORB_MARKERS_TILE_BINS if binning == "tile" else 0)

    def bind(self):
        d, cfg = self.d, self.cfg
        self.g.markers_bind(d["s"], d["theta"], d["phi"], d["vpar"] if cfg.current else None, d["mu"],
                            d["w"], flags=self.bind_flags)


def deposit_kernel_name(cfg):
    """The tile kernel orb_deposit picks for this N_L policy (csrc/orb_api.cu)."""
    if cfg.adaptive or cfg.n_fixed > 4:
        return "k_deposit_tile"
    return "k_deposit_ws<" if cfg.n_fixed == 1 else "k_deposit_ws2"


def run_ours(args):
    import torch

    from paper_1908_02219_b200 import binding as B
    from paper_1908_02219_b200 import build as build_mod

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path is the only path (no CPU fallback)")
    rank, local_rank, world = R.init()
    if world != args.gpus and world > 1:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%d" % (args.gpus, world))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if rank == 0:
        build_mod.build()
    R.barrier()
    B.lib()

    # fp64 roof of this device, measured live (outside any timed region)
    try:
        fp64_peak, fp64_src = B.probe_dfma(local_rank), "measured live (orb_probe_dfma: 8 DFMA chains/thread)"
    except Exception:  # noqa: BLE001
        fp64_peak, fp64_src = FP64_MEASURED_TFLOPS, "profiles/r01_microbench.md"

    # inputs: generated on the host into pinned memory (they are the e2e leg's source)
    cfgs = [pick_config(name, rank) for name in W.WORKLOADS[args.workload]]
    species = [Species(c, dev, local_rank, B, torch, args.binning) for c in cfgs]
    torch.cuda.synchronize()
    cfg = cfgs[0]                     # grid shape and outputs are common to the species
    current = any(c.current for c in cfgs)
    shape = species[0].g.shape()
    rho = torch.zeros(shape, dtype=torch.float64, device=dev)
    jpar = torch.zeros(shape, dtype=torch.float64, device=dev) if current else None
    stream = torch.cuda.current_stream()
    st = stream.cuda_stream
    NS = len(species)

    def step(evs=None):
        for i, sp in enumerate(species):
            sp.bind()
            if evs:
                evs[4 * i + 0].record(stream)
            sp.g.markers_bin(st)
            if evs:
                evs[4 * i + 1].record(stream)
            if i == 0:
                sp.g.grid_zero(rho, jpar, st)
            if evs:
                evs[4 * i + 2].record(stream)
            sp.g.deposit(rho, jpar if sp.cfg.current else None, sp.pol, st)
            if evs:
                evs[4 * i + 3].record(stream)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    npts_sp = [sp.g.last_points() for sp in species]
    npts_step = sum(npts_sp)
    fallback_step = sum(sp.g.last_fallback_points() for sp in species)

    K = args.steps
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4 * NS)] for _ in range(K)]
    e_start, e_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(index=local_rank)
    launches0 = sum(sp.g.launch_count() for sp in species)
    R.barrier()
    torch.cuda.synchronize()
    sampler.start()
    e_start.record(stream)
    for k in range(K):
        step(evs[k])
    e_end.record(stream)
    torch.cuda.synchronize()
    R.barrier()
    sampler.stop()
    launches = sum(sp.g.launch_count() for sp in species) - launches0
    total_ms = e_start.elapsed_time(e_end)
    bin_ms = sum(e[4 * i].elapsed_time(e[4 * i + 1]) for e in evs for i in range(NS)) / K
    zero_ms = sum(e[1].elapsed_time(e[2]) for e in evs) / K
    dep_sp = [[e[4 * i + 2].elapsed_time(e[4 * i + 3]) for e in evs] for i in range(NS)]
    dep_ms_all = [sum(dep_sp[i][k] for i in range(NS)) for k in range(K)]
    dep_ms = sum(dep_ms_all) / K
    assert sum(sp.g.last_points() for sp in species) == npts_step

    # result sanity inside the bench: charge conservation (P1) of the last step
    q_sum = float(rho.sum().item())
    w_sum = sum(float(sp.d["w"].sum().item()) * sp.cfg.q for sp in species)
    w_abs = sum(float(sp.d["w"].abs().sum().item()) * abs(sp.cfg.q) for sp in species)
    conservation = abs(q_sum - w_sum) / w_abs

    job_ms, job_pts = R.combine(total_ms, float(npts_step) * K, device=dev)
    value = job_pts / (job_ms * 1e-3)

    # ---- NEXT-1 leg: get fields + gyroaverage of n_grids fields on the binned markers
    gather = None
    if not args.no_gather:
        nf = 2 if current else 1
        gen = torch.Generator(device=dev)
        gen.manual_seed(1234 + rank)
        fields = [torch.randn(shape, dtype=torch.float64, device=dev, generator=gen) for _ in range(nf)]
        g_ms, g_pts, g_fb = 0.0, 0, 0
        for sp in species:
            outs = [torch.empty(sp.cfg.n_markers, dtype=torch.float64, device=dev) for _ in range(nf)]
            ge = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
            for _ in range(3):
                sp.g.gather(fields, outs, sp.pol, st)
            ge[0].record(stream)
            for _ in range(K):
                sp.g.gather(fields, outs, sp.pol, st)
            ge[1].record(stream)
            torch.cuda.synchronize()
            g_ms += ge[0].elapsed_time(ge[1]) / K
            g_pts += sp.g.last_points()
            g_fb += sp.g.last_fallback_points()
            del outs
        # what the method must move: s, theta*, phi, mu in and nf results out per marker; every
        # node of every field read once
        g_bytes = sum(c.n_markers for c in cfgs) * 8 * (4 + nf) + nf * cfg.nodes * 8
        gather = {"ms": g_ms, "fields": nf, "points": g_pts, "fallback_points": g_fb,
                  "algorithmic_bytes": g_bytes}
        del fields
        torch.cuda.empty_cache()

    # ---- NEXT-2 leg: incremental re-binning of the slack bins after a synthetic push, and
    # NEXT-3 leg: the materialised-ring-data / cell-owner path on the same markers (single species)
    rebin = ring = None
    if not args.no_next_legs and NS == 1:
        sp = species[0]
        ev = lambda: torch.cuda.Event(enable_timing=True)  # noqa: E731
        if args.binning == "tile" and sp.bind_flags == B.ORB_MARKERS_TILE_BINS:
            rebin = {"what": "orb_markers_rebin after a seeded fraction of the markers jumped 24 "
                             "theta* cells (1.5 tiles); refresh = orb_markers_refresh (records <- bound arrays)",
                     "build_ms": bin_ms, "cases": []}
            gen = torch.Generator(device=dev)
            gen.manual_seed(99 + rank)
            theta0 = sp.d["theta"].clone()
            for frac in (0.0, 0.01, 0.1, 0.5):
                sel = torch.rand(sp.cfg.n_markers, device=dev, generator=gen) < frac
                sp.d["theta"][sel] += 24.0 * (W.TWO_PI / sp.cfg.ntheta)
                e0, e1, e2 = ev(), ev(), ev()
                e0.record(stream)
                sp.g.markers_refresh(st)
                e1.record(stream)
                sp.g.markers_rebin(st)
                e2.record(stream)
                torch.cuda.synchronize()
                moved, left = sp.g.last_moved()
                rebin["cases"].append({"moved_fraction": frac, "moved": moved, "left_in_place": left,
                                       "refresh_ms": e0.elapsed_time(e1), "rebin_ms": e1.elapsed_time(e2)})
            e0, e1 = ev(), ev()
            sp.g.grid_zero(rho, jpar, st)
            e0.record(stream)
            sp.g.deposit(rho, jpar if sp.cfg.current else None, sp.pol, st)
            e1.record(stream)
            torch.cuda.synchronize()
            rebin["deposit_after_rebin_ms"] = e0.elapsed_time(e1)
            w_now = float(rho.sum().item())
            rebin["charge_conservation_rel"] = abs(w_now - w_sum) / w_abs
            sp.d["theta"].copy_(theta0)
            del theta0
            sp.bind()
            sp.g.markers_bin(st)
        try:
            nl_cap = sp.cfg.n_max if sp.cfg.adaptive else sp.cfg.n_fixed
            sp.g.ring_reserve(sp.cfg.n_markers, min(npts_step + 1024, sp.cfg.n_markers * nl_cap))
            pol_ring = B.policy_for(sp.cfg, flags=B.ORB_DEPOSIT_ALGO_RING_DATA)
            ts = []
            for _ in range(3):
                sp.g.grid_zero(rho, jpar, st)
                e0, e1 = ev(), ev()
                e0.record(stream)
                sp.g.deposit(rho, jpar if sp.cfg.current else None, pol_ring, st)
                e1.record(stream)
                torch.cuda.synchronize()
                ts.append(e0.elapsed_time(e1))
            ring = {"what": "ORB_DEPOSIT_ALGO_RING_DATA: build Larmor ring data in HBM, bucket-sort the "
                            "points by cell, cell-owner loop (PAPER.md:73-75); no marker binning needed",
                    "ms": min(ts), "value": npts_step / (min(ts) * 1e-3), "unit": UNIT,
                    "charge_conservation_rel": abs(float(rho.sum().item()) - w_sum) / w_abs,
                    "compare_with_step_ms": job_ms / K}
            sp.g.ring_reserve(0, 0)
        except B.OrbError as e:  # noqa: PERF203
            ring = {"unavailable": str(e)}
        torch.cuda.empty_cache()

    # ---- e2e: HOST marker arrays -> orb_deposit_host -> HOST grids, every step
    E = max(1, min(args.e2e_steps, K))
    rho_h = [torch.empty(shape, dtype=torch.float64, pin_memory=True) for _ in species]
    jpar_h = [torch.empty(shape, dtype=torch.float64, pin_memory=True) if sp.cfg.current else None
              for sp in species]
    for sp in species:
        sp.d = None
    torch.cuda.empty_cache()

    def e2e_step():
        pts = up = down = 0
        for i, sp in enumerate(species):
            m, c = sp.m, sp.cfg
            a, b, cdown = sp.g.deposit_host(m["s"], m["theta"], m["phi"], m["vpar"] if c.current else None,
                                            m["mu"], m["w"], rho_h[i].numpy(),
                                            jpar_h[i].numpy() if c.current else None, sp.pol)
            pts, up, down = pts + a, up + b, down + cdown
            if i > 0:      # species add into the same grids: summed on the host
                rho_h[0].add_(rho_h[i])
                if c.current and jpar_h[0] is not None:
                    jpar_h[0].add_(jpar_h[i])
        return pts, up, down

    e2e_step()
    torch.cuda.synchronize()
    launches_e0 = sum(sp.g.launch_count() for sp in species)
    R.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(E):
        npts_e, up, down = e2e_step()
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    R.barrier()
    launches_e = sum(sp.g.launch_count() for sp in species) - launches_e0
    e2e_job_ms, e2e_job_pts = R.combine(e2e_ms, float(npts_e) * E, device=dev)
    e2e_value = e2e_job_pts / (e2e_job_ms * 1e-3)
    e2e_conservation = abs(float(rho_h[0].sum().item()) - w_sum) / w_abs
    for sp in species:
        sp.g.destroy()

    line = None
    if rank == 0:
        peak, peak_src = measured_hbm_peak()
        n_grids = 2 if current else 1
        alg_bytes = sum(c.n_markers * 8 * (6 if c.current else 5) for c in cfgs) + n_grids * cfg.nodes * 16
        achieved = alg_bytes / (dep_ms * 1e-3) / 1e9
        flops = sum(2.0 * 64.0 * (2 if c.current else 1) * n for c, n in zip(cfgs, npts_sp))
        # the dominant kernel: the deposit kernel of the species that takes longest
        dom = max(range(NS), key=lambda i: sum(dep_sp[i]))
        kernel = deposit_kernel_name(cfgs[dom])
        traffic, traffic_src = ncu_traffic(args.workload, kernel)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K,
            "warmup": args.warmup, "ms_per_step": job_ms / K, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_json(cfgs, world, args.workload, {
                "binning": "slack tile bins, one pass (ORB_MARKERS_TILE_BINS)" if args.binning == "tile"
                else "dense counting sort by cell (count, scan, scatter)"}),
            "points_per_step": npts_step,
            "fallback_points_per_step": fallback_step,
            "phases_ms": {"bin": bin_ms, "zero": zero_ms, "deposit": dep_ms,
                          "deposit_min": min(dep_ms_all), "deposit_max": max(dep_ms_all),
                          "deposit_per_species": [sum(x) / K for x in dep_sp]},
            "deposit_only": {"value": npts_step / (dep_ms * 1e-3), "unit": UNIT,
                             "note": "tile deposit kernel(s) on already-binned markers"},
            "step_hbm": {"achieved": alg_bytes * K / (total_ms * 1e-3) / 1e9, "unit": "GB/s",
                         "frac": alg_bytes * K / (total_ms * 1e-3) / 1e9 / peak,
                         "note": "same algorithmic bytes over the whole step (bin + zero + deposit)"},
            "roofline": {"bound": "hbm", "kernel": kernel, "achieved": achieved,
                         "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                         "algorithmic_bytes": alg_bytes, "kernel_ms": dep_ms,
                         "frac_of_nominal_8TBs": achieved / HBM_NOMINAL_GBS,
                         "note": "contract metric of BASELINE.json; the roof that actually binds "
                                 "this path is the fp64 pipe: see roofline_alu (DESIGN.md 6)"},
            "roofline_alu": {"bound": "alu", "pipe": "fp64", "kernel": kernel,
                             "achieved": flops / (dep_ms * 1e-3) / 1e12, "peak": fp64_peak,
                             "peak_source": fp64_src,
                             "unit": "TFLOP/s",
                             "frac": flops / (dep_ms * 1e-3) / 1e12 / fp64_peak,
                             "frac_of_nominal": flops / (dep_ms * 1e-3) / 1e12 / FP64_NOMINAL_TFLOPS,
                             "algorithmic_flops": flops,
                             "note": "scatter only: 64 nodes x n_grids FMA per Larmor point; the "
                                     "geometry (sincos, sqrt, atan2) is not counted"},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": up,
                    "d2h_bytes_per_step": down, "steps": E, "ms_per_step": e2e_job_ms / E,
                    "api": "orb_deposit_host (pinned host SoA in, host grids out)",
                    "gpu_launches": launches_e},
            "gpu_launches": launches,
            "clocks": sampler.summary(),
            "checks": {"charge_conservation_rel": conservation,
                       "e2e_charge_conservation_rel": e2e_conservation},
        }
        if rebin:
            line["rebin"] = rebin
        if ring:
            line["ring_data"] = ring
        if gather:
            g_ach = gather["algorithmic_bytes"] / (gather["ms"] * 1e-3) / 1e9
            line["gather"] = {
                "what": "NEXT-1 get fields + gyroaverage (orb_gather) of %d field(s) on the binned "
                        "markers" % gather["fields"],
                "value": gather["points"] / (gather["ms"] * 1e-3), "unit": UNIT,
                "ms": gather["ms"], "fallback_points": gather["fallback_points"],
                "roofline": {"bound": "hbm", "kernel": "k_gather_tile", "achieved": g_ach, "peak": peak,
                             "unit": "GB/s", "frac": g_ach / peak, "traffic": None,
                             "algorithmic_bytes": gather["algorithmic_bytes"],
                             "note": "4 marker fields in + 1 result out per marker and field, every "
                                     "node of every field read once"}}
        if world == 1 and not args.no_cpu_baseline:
            n_sample = min(args.cpu_sample, cfg.n_markers)
            npts_o, secs = oracle_sample(cfg, species[0].m, n_sample)
            line["cpu_baseline"] = {
                "value": npts_o / secs, "unit": UNIT, "cores": 1, "kind": "oracle",
                "sample": "first %d markers of %s (%d Larmor points, %.1f s), single thread; host has %d cores"
                          % (n_sample, cfg.name, npts_o, secs, os.cpu_count() or 0)}
        else:
            line["cpu_baseline"] = None
        print(json.dumps(line), flush=True)
    R.finalize()
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3", choices=sorted(W.WORKLOADS))
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--cpu-sample", type=int, default=1 << 21,
                    help="markers of the workload the cpu_baseline leg times the oracle on")
    ap.add_argument("--ref-sample", type=int, default=1 << 18,
                    help="markers per step of the --impl reference arm")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--binning", default="tile", choices=["tile", "dense"],
                    help="marker binning of the step: slack tile bins built in one pass "
                         "(ORB_MARKERS_TILE_BINS) or the dense counting sort by cell")
    ap.add_argument("--no-next-legs", action="store_true",
                    help="skip the incremental re-binning (NEXT-2) and ring-data (NEXT-3) legs")
    ap.add_argument("--no-gather", action="store_true", help="skip the orb_gather (NEXT-1) leg")
    args = ap.parse_args(argv)
    if args.warmup < 3 and args.impl == "ours":
        print("bench.py: note: fewer than 3 warm-up steps requested", file=sys.stderr)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
