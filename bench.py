#!/usr/bin/env python
"""bench.py — throughput of the whole PIC hot path (sort + gather + push + deposit + Yee + guards)
on BASELINE.json's headline workload, one JSON line on stdout (rank 0).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C2] [--impl ours|reference]

* A "step" is one `pic_step(1)`: every row of SURVEY.md §8(a) once, the sort at its cadence
  (every 4th step). Workload at N=1: C2 (128^3 cells, 8 ppc, order 3, fp64).
* `value`   = particles * K / device time of K steps with the state resident in HBM (CUDA events on
  the stream the library launches on; barrier + synchronize on both sides; max over ranks).
* `e2e`     = the same job through the C ABI with HOST (pinned) buffers: pic_create, pic_add_species
  (H2D), K steps, pic_get_particles + pic_get_fields (D2H), all inside the timed region.
* `roofline`= the dominant kernel's algorithmic bytes / flops per launch (DESIGN.md "Byte and flop
  model") over its average launch duration measured by the library's per-kernel CUDA events.
* `roofline.peak` = measured: HBM from MEASURED_PEAKS.json, the fp64 pipe and shared-memory bandwidth by
  the library's own probes (pic_probe_peaks) in this run, before the timed region.
* `cpu_baseline` = the oracle (oracle/, as it stands) timed on this box's host cores on a bounded sample of
  the same workload: its OpenMP variant (the paper's CPU scheme; pinned to the serial
  oracle by T12) on all cores, and the canonical serial oracle on one. `--impl reference` times only that.
* N>1 (torchrun): the path does not shard: every rank runs
  an independent replica of the workload, no data-path collective; value = N * particles * K / max time.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import workloads as W  # noqa: E402

METRIC = "particle-steps/s (sort+gather+push+deposit+Yee)"
UNIT = "particle-steps/s"
ATTRS = ("x", "y", "z", "ux", "uy", "uz", "w")


# ----------------------------------------------------------------------------- byte / flop model
def model(cfg, deposit_split=True):
    """Algorithmic bytes and flops per particle-step."""
    P = 8 if cfg.dtype == "f64" else 4
    n = cfg.order
    npart = cfg.n_particles
    ncell = cfg.n_cells[0] * cfg.n_cells[1] * cfg.n_cells[2]
    ppc = npart / ncell
    si = cfg.sort_interval
    step = 13 * P + 6 * P / ppc + 9 * P / ppc + 30 * P / ppc
    if si > 0:
        step += (3 * P + 4 + 8 + 2 * (7 * P + 8)) / si
    # per kernel, per particle (inputs read once, outputs written once, fields once per cell)
    push_b = 12 * P + 6 * P / ppc                 # x,u in; x_new,u out; E,B once per cell
    dep_b = 10 * P + 4 + 6 * P / ppc              # x_old,x_new,w,cell in; wrapped x out; J RMW per cell
    fused_b = 13 * P + 12 * P / ppc
    # flops: gather 6 comps x nested tensor product, shapes, Boris, Esirkepov (counted in DESIGN.md)
    m = n + 1
    gather_f = 6 * 2 * (m ** 3 + m ** 2 + m) + 6 * (8 if n == 3 else 5 if n == 2 else 2) * 2
    boris_f = 110
    nw = n + 2
    dep_f = 3 * (nw * nw * 8 + nw * nw * (nw - 1) * 3) + 6 * (10 if n == 3 else 6 if n == 2 else 2) * 2 + 60
    # the gather's shared-memory reads in k_push_tile: every stencil value of every component, once per particle
    push_smem_b = 6 * m ** 3 * P
    return dict(P=P, ppc=ppc, step_bytes=step, push_bytes=push_b, deposit_bytes=dep_b, fused_bytes=fused_b,
                push_flops=gather_f + boris_f, deposit_flops=dep_f, push_smem_bytes=push_smem_b)


# ----------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples SM clock and throttle reasons of one GPU while the timed region runs (NVML)."""

    def __init__(self, index, uuid=None):
        self.index = index
        self.samples = []
        self.reasons = set()
        self.sm_max = None
        self._stop = threading.Event()
        self._t = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            try:
                self.h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + str(uuid)).encode()) if uuid else None
            except Exception:
                self.h = None
            if self.h is None:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4),
            "hw_power_brake": getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.02)

    def __enter__(self):
        if self.nv is not None:
            self._t = threading.Thread(target=self._loop, daemon=True)
            self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._t is not None:
            self._t.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.sm_max,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ----------------------------------------------------------------------------- distributed plumbing
def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def init_dist(backend):
    """Process group for the barrier and the max-over-ranks of the timing; no data-path collective."""
    rank, local, world = dist_env()
    if world == 1:
        return None
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29511")
    if not dist.is_initialized():
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return dist


def barrier(dist):
    if dist is not None:
        dist.barrier()


def max_over_ranks(dist, value, device="cpu"):
    """Max of a scalar over all ranks (the contract's timing rule)."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate(n_particles_per_rank, world, steps, ms_max):
    """Whole-job throughput of `world` independent replicas: all ranks' particle-steps / slowest rank's time."""
    return n_particles_per_rank * world * steps / (ms_max * 1e-3)


# ----------------------------------------------------------------------------- the oracle arm
def _sample_cfg(cfg_full, n):
    """The same recipe on an n^3 box (clipped to the configured grid): the bounded sample the oracle is timed on."""
    shape = tuple(min(n, c) for c in cfg_full.n_cells)
    if shape == tuple(cfg_full.n_cells):
        return cfg_full
    return W.scaled(cfg_full, shape, z_first=0, ramp_cells=0, laser=False)


def time_oracle(cfg_full, steps, warmup, budget_s, threads):
    """The oracle as it stands on a bounded sample of the workload: the largest box of the same recipe whose
    warmup+steps oracle steps fit the budget (the configured box itself if that fits). threads = 1: the
    canonical serial oracle; otherwise its OpenMP variant on that many threads (0 = all OpenMP offers).
    Returns dict(value, sample, ms_per_step, cores, particles)."""
    import oracle
    cal = _sample_cfg(cfg_full, 16)
    o = _make_oracle(oracle, cal)
    used = 1
    t0 = time.perf_counter()
    if threads == 1:
        o.step(1)
    else:
        used = o.step_omp(1, threads)
    t_cal = (time.perf_counter() - t0) / max(cal.n_particles, 1)
    o.close()
    chosen = None
    for n in (256, 128, 96, 64, 48, 40, 32, 24, 16, 8):
        if n > max(cfg_full.n_cells) and n != 8:
            continue
        cfg = _sample_cfg(cfg_full, n)
        # the calibration box is small (threads idle, caches warm): leave a factor of two
        if cfg.n_particles * t_cal * (steps + warmup) * 2.0 <= budget_s or n == 8:
            chosen = cfg
            break
    o = _make_oracle(oracle, chosen)
    run = (lambda k: o.step(k)) if threads == 1 else (lambda k: o.step_omp(k, threads))
    if warmup:
        run(warmup)
    t0 = time.perf_counter()
    run(steps)
    dt = time.perf_counter() - t0
    o.close()
    whole = tuple(chosen.n_cells) == tuple(cfg_full.n_cells)
    sample = "%s %s (%d particles), %d oracle steps after %d warm-up, %s" % (
        cfg_full.name, "at its configured size" if whole else "recipe on a %dx%dx%d box" % tuple(chosen.n_cells),
        chosen.n_particles, steps, warmup,
        "serial oracle, 1 thread" if threads == 1 else "OpenMP variant of the oracle, %d threads" % used)
    return dict(value=chosen.n_particles * steps / dt, sample=sample, ms_per_step=dt / steps * 1e3, cores=used,
                particles=chosen.n_particles)


def _make_oracle(oracle, cfg):
    species, E, B = W.generate(cfg)
    o = oracle.Oracle(cfg.n_cells, cfg.dx, cfg.dt, cfg.order, dtype=cfg.np_dtype, periodic=cfg.periodic,
                      tile=cfg.tile, sort_interval=cfg.sort_interval)
    for spec, arrs in species:
        o.add_species(*[arrs[k] for k in ATTRS], spec.charge, spec.mass)
    if E is not None:
        o.set_fields(E, B)
    return o


def run_reference(args):
    """The reference arm of this tier is the oracle: its OpenMP variant on all host cores, on a bounded
    sample of the same workload (the line says which), K steps after W warm-up steps."""
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    cfg = W.CONFIGS[args.config]
    r = time_oracle(cfg, args.steps, args.warmup, budget_s=150.0, threads=0)
    cd = config_dict(cfg, world, args)
    cd["timed_sample"] = r["sample"]                 # what this arm ran: a bounded sample of the workload above
    cd["particles_timed"] = r["particles"]
    line = {
        "impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": r["ms_per_step"],
        "ms_per_step_is_for": ("%d particles: the workload at its configured size" % r["particles"]) if r["particles"] == cfg.n_particles
        else "%d particles (the timed sample), not the configured %d" % (r["particles"], cfg.n_particles),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": cfg.dtype, "data": "synthetic", "config": cd,
        "cpu_baseline": {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"]},
        "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def config_dict(cfg, world, args):
    return {
        "workload": "%s: %dx%dx%d Yee cells, %s, order-%d shape, %s, sort every %d steps, tile %s" % (
            cfg.name, *cfg.n_cells, " + ".join("%d ppc %s" % (s.ppc, s.name) for s in cfg.species), cfg.order,
            cfg.dtype, cfg.sort_interval, "x".join(str(t) for t in cfg.tile)),
        "particles_per_gpu": cfg.n_particles,
        "cells_per_gpu": cfg.n_cells[0] * cfg.n_cells[1] * cfg.n_cells[2],
        "parallelism": "replicas x%d (no sharding, no collective)" % world,
        "l2": "inputs larger than L2 (particle state %.2f GB per buffer vs 126 MB L2)" % (
            cfg.n_particles * (7 * (8 if cfg.dtype == "f64" else 4) + 8) / 1e9),
        "deposit_mode": args.deposit_mode,
        "variant": {"pusher": args.pusher, "gather_mode": args.gather_mode, "solver": args.solver,
                    "deterministic": bool(args.deterministic), "cuda_graph": not args.no_graph,
                    "box_staging": args.box_staging},
    }


# ----------------------------------------------------------------------------- our arm
def pinned_like(arr):
    import torch
    t = torch.from_numpy(arr).pin_memory()
    return t, t.numpy()


def run_ours(args):
    import torch
    import paper_2101_12149_b200 as pic

    rank, local, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the library has no CPU fallback)")
    torch.cuda.set_device(local)
    dist = init_dist("nccl")
    dev = torch.device("cuda", local)
    cfg = W.CONFIGS[args.config]
    # Fig. 1-style sweeps: same recipe, other sort cadence /
    # bin size / temperature. The default run leaves the configuration untouched.
    over = {}
    if args.sort_interval is not None:
        over["sort_interval"] = args.sort_interval
    if args.tile is not None:
        over["tile"] = tuple(int(v) for v in args.tile.split(","))
    if over or args.sigma is not None:
        cfg = W.scaled(cfg, cfg.n_cells, name=cfg.name, **over)
        if args.sigma is not None:
            for sp in cfg.species:
                sp.sigma = args.sigma
    if rank != 0:
        cfg = W.scaled(cfg, cfg.n_cells, name=cfg.name, seed=cfg.seed + 7919 * rank)   # replicas draw their own inputs
    species, E0, B0 = W.generate(cfg)
    np_dt = cfg.np_dtype
    P = np.dtype(np_dt).itemsize
    n_part = cfg.n_particles
    n_cell = cfg.n_cells[0] * cfg.n_cells[1] * cfg.n_cells[2]
    stream = torch.cuda.current_stream()
    kw = dict(dtype=np_dt, periodic=cfg.periodic, tile=cfg.tile, sort_interval=cfg.sort_interval,
              deposit_mode=args.deposit_mode, sort_key_mode=args.sort_key_mode, stream=stream.cuda_stream,
              pusher=args.pusher, gather_mode=args.gather_mode, solver=args.solver, deterministic=args.deterministic, cuda_graph=not args.no_graph,
              box_staging=args.box_staging)

    # ---------------- leg 1: state resident in HBM
    sim = pic.Sim(cfg.n_cells, cfg.dx, cfg.dt, cfg.order, **kw)
    for spec, arrs in species:
        d = [torch.from_numpy(arrs[k]).to(dev) for k in ATTRS]
        sim.add_species(*d, spec.charge, spec.mass)
        del d
    if E0 is not None:
        sim.set_fields(E0, B0)
    # on-chip ceilings measured in this run (roofline against measured ceilings)
    probes = pic.pic_probe_peaks(stream.cuda_stream, 0.0 if args.skip_probe else 0.2)
    sim.step(args.warmup)
    sim.synchronize()
    d0 = sim.diagnostics()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier(dist)
    torch.cuda.synchronize()
    with ClockSampler(local, getattr(torch.cuda.get_device_properties(local), "uuid", None)) as clk:
        ev0.record(stream)
        sim.step(args.steps)
        ev1.record(stream)
        torch.cuda.synchronize()
    barrier(dist)
    ms = ev0.elapsed_time(ev1)
    d1 = sim.diagnostics()
    # per-kernel device times: the same K steps again with the library's CUDA-event timers on (one span per
    # launch; this pass launches kernel by kernel, the timed region above replays captured graphs)
    sim.enable_phase_timing(True)
    sim.phase_times(reset=True)
    sim.step(args.steps)
    sim.synchronize()
    phases = sim.phase_times(reset=True)
    sim.enable_phase_timing(False)
    # SURVEY.md 8(d) timing protocol: best and median of 5 repetitions of the K steps (the contract's `value`
    # above is the first of them; these four more run after it and are reported beside it, never instead)
    rep_ms = [ms]
    for _ in range(4):
        ev0.record(stream)
        sim.step(args.steps)
        ev1.record(stream)
        torch.cuda.synchronize()
        rep_ms.append(ev0.elapsed_time(ev1))
    repeats = {"n": len(rep_ms), "ms_per_step": [t / max(args.steps, 1) for t in rep_ms],
               "best_ms_per_step": min(rep_ms) / max(args.steps, 1),
               "median_ms_per_step": float(np.median(rep_ms)) / max(args.steps, 1)}
    launches = int(d1["step_launches"] - d0["step_launches"])
    ms_max = max_over_ranks(dist, ms, dev)
    value = aggregate(n_part, world, args.steps, ms_max)
    energy = d1["field_E"] + d1["field_B"] + d1["kinetic"]
    if not math.isfinite(energy):
        raise SystemExit("non-finite energy after the timed region")
    sim.close()
    del sim
    torch.cuda.empty_cache()

    # ---------------- leg 2: end to end through the C ABI with host buffers
    e2e = None
    if not args.skip_e2e:
        host_in = []
        keep = []
        for spec, arrs in species:
            row = []
            for k in ATTRS:
                t, a = pinned_like(arrs[k])
                keep.append(t)
                row.append(a)
            host_in.append((spec, row))
        if E0 is not None:
            hostE = [pinned_like(np.ascontiguousarray(a))[1] for a in E0]
            hostB = [pinned_like(np.ascontiguousarray(a))[1] for a in B0]
        outs = []
        for spec, row in host_in:
            o = [pinned_like(np.empty(len(row[0]), dtype=np_dt)) for _ in ATTRS]
            oid = pinned_like(np.empty(len(row[0]), dtype=np.int64))
            outs.append(([a for _, a in o], oid[1], [t for t, _ in o] + [oid[0]]))
        fshape = (cfg.n_cells[2], cfg.n_cells[1], cfg.n_cells[0])
        f_out = [[pinned_like(np.empty(fshape, dtype=np_dt)) for _ in range(3)] for _ in range(2)]
        fE = [a for _, a in f_out[0]]
        fB = [a for _, a in f_out[1]]
        h2d = sum(len(row[0]) * 7 * P for _, row in host_in) + (6 * n_cell * P if E0 is not None else 0)
        d2h = sum(len(row[0]) * (7 * P + 8) for _, row in host_in) + 6 * n_cell * P
        e2e_ms = []
        for rep in range(3):          # first repetition warms the allocator / page tables; the faster of the next two is
                                      # reported (a single run now and then catches a slow cudaFree / page-table episode
                                      # on the host: 148 ms instead of 115 ms once in this round's runs)
            barrier(dist)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            ev0.record(stream)
            s2 = pic.Sim(cfg.n_cells, cfg.dx, cfg.dt, cfg.order, **kw)
            for spec, row in host_in:
                s2.add_species(*row, spec.charge, spec.mass)
            if E0 is not None:
                s2.set_fields(hostE, hostB)
            s2.step(args.steps)
            for si, (arrs_o, ids_o, _) in enumerate(outs):
                pic.pic_get_particles(s2._h, si, len(ids_o), *arrs_o, ids_o, np_dt)
            pic.pic_get_fields(s2._h, fE, fB, None, np_dt, n_cell)
            ev1.record(stream)
            torch.cuda.synchronize()
            wall = (time.perf_counter() - t0) * 1e3
            e2e_ms.append(max(ev0.elapsed_time(ev1), wall))
            s2.close()
            barrier(dist)
        e2e_max = max_over_ranks(dist, min(e2e_ms[1:]), dev)
        e2e = {"value": aggregate(n_part, world, args.steps, e2e_max), "unit": UNIT,
               "h2d_bytes_per_step": h2d / args.steps, "d2h_bytes_per_step": d2h / args.steps,
               "ms_total": e2e_max, "ms_total_all_repetitions": e2e_ms,
               "what": "pic_create + pic_add_species(host, pinned) + pic_step(K) + pic_get_particles + pic_get_fields(host)"}
        del keep, outs, f_out

    if rank != 0:
        return 0

    # ---------------- rooflines of the particle kernels, from the per-kernel device timers
    m = model(cfg)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    hbm_src = "hbm: measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "hbm: fallback 6650 GB/s (B200_PROFILING.md)"
    clocks = clk.summary()
    f64 = cfg.dtype == "f64"
    # fp64: the DFMA probe for vector kernels, the DMMA probe for the tensor-pipe deposition (same pipe);
    # fp32: the FFMA probe. Shared memory: the 64-bit load probe.
    alu_vec = probes["fp64_fma_tflops"] if f64 else probes["fp32_fma_tflops"]
    alu_mma = probes["fp64_mma_tflops"] if f64 else probes["fp32_fma_tflops"]
    smem_peak = probes["smem_tbs"]
    per_launch = {k: (v[0] / v[1] if v[1] else 0.0) for k, v in phases.items()}
    n_species = len(cfg.species)
    units = n_part / n_species                      # particles one launch processes
    mode = args.deposit_mode
    mma = f64 and mode in (0, 4, 5)
    if phases["deposit"][1] == 0:                   # one kernel does the whole particle step
        nm = "k_fused_mma (gather + push + deposit, tensor pipe)" if mode == 5 else "k_particles_global (gather + push + deposit)"
        kern = {"push": (nm, m["fused_bytes"], m["push_flops"] + m["deposit_flops"], alu_mma if mode == 5 else alu_vec,
                         m["push_smem_bytes"] if mode == 5 else 0)}
    else:
        dep_name = "k_deposit_mma (Esirkepov, fp64 tensor pipe)" if mma else "k_deposit_tile / k_deposit_coop (Esirkepov, lane groups)"
        kern = {"push": ("k_push_tile (gather + Boris push)", m["push_bytes"], m["push_flops"], alu_vec, m["push_smem_bytes"]),
                "deposit": (dep_name, m["deposit_bytes"], m["deposit_flops"], alu_mma if mma else alu_vec, 0)}
    traffic_file = {}
    try:
        traffic_file = json.load(open(os.path.join(ROOT, "profiles", "traffic_%s.json" % cfg.name)))
    except Exception:
        pass
    per_kernel = {}
    for key, (name, bpp, fpp, alu_peak, smem_b) in kern.items():
        dur = per_launch[key] * 1e-3
        if dur <= 0:
            continue
        e = {"kernel": name, "ms_per_launch": per_launch[key], "launches_timed": phases[key][1],
             "bytes_per_particle": bpp, "flops_per_particle": fpp,
             "hbm_gbs": bpp * units / dur / 1e9, "alu_tflops": fpp * units / dur / 1e12, "alu_peak_tflops": alu_peak}
        e["hbm_frac"] = e["hbm_gbs"] / hbm_peak
        e["alu_frac"] = e["alu_tflops"] / alu_peak if alu_peak > 0 else None
        if smem_b:
            # the roof that actually binds the gather: every stencil value of every
            # component is one shared-memory read per particle
            e["smem"] = {"achieved": smem_b * units / dur / 1e12, "peak": smem_peak, "unit": "TB/s",
                         "frac": (smem_b * units / dur / 1e12) / smem_peak if smem_peak > 0 else None,
                         "bytes_per_particle": smem_b}
        tk = [k for k in traffic_file.get("dram_bytes_per_launch", {}) if k in name]
        if tk and mode == 0:
            e["traffic"] = float(traffic_file["dram_bytes_per_launch"][tk[0]])
            e["shared_wavefront_frac_ncu"] = traffic_file.get("shared_wavefront_frac_of_peak", {}).get(tk[0])
        per_kernel[key] = e
    dom = max(per_kernel, key=lambda k: per_kernel[k]["ms_per_launch"] * per_kernel[k]["launches_timed"])
    d = per_kernel[dom]
    if (d["alu_frac"] or 0) >= d["hbm_frac"]:
        roof = {"bound": "alu", "achieved": d["alu_tflops"], "peak": d["alu_peak_tflops"], "unit": "TFLOP/s", "frac": d["alu_frac"]}
    else:
        roof = {"bound": "hbm", "achieved": d["hbm_gbs"], "peak": hbm_peak, "unit": "GB/s", "frac": d["hbm_frac"]}
    traffic = args.traffic if args.traffic is not None else d.get("traffic")
    roof.update({
        "kernel": d["kernel"], "ms_per_launch": d["ms_per_launch"], "launches_timed": d["launches_timed"],
        "traffic": traffic,
        "traffic_source": "--traffic" if args.traffic is not None else (traffic_file.get("source") if traffic is not None else None),
        "hbm_gbs": d["hbm_gbs"], "hbm_frac": d["hbm_frac"], "alu_tflops": d["alu_tflops"], "alu_frac": d["alu_frac"],
        "bytes_per_particle": d["bytes_per_particle"], "flops_per_particle": d["flops_per_particle"],
        "peak_source": hbm_src + "; alu and shared memory: measured in this run by pic_probe_peaks "
                       "(%s)" % ("probes skipped" if args.skip_probe else "0.2 s per probe, best launch"),
        "measured_peaks": probes,
        "kernels": per_kernel,
        "phase_ms_per_step": {k: v[0] / args.steps for k, v in phases.items()},
    })
    if "smem" in d:
        roof["smem"] = d["smem"]
    step_gbs = m["step_bytes"] * n_part * args.steps / (ms * 1e-3) / 1e9

    cpu = None
    if not args.skip_cpu and world == 1:
        par = time_oracle(cfg, 2, 0, budget_s=25.0, threads=0)
        ser = time_oracle(cfg, 2, 0, budget_s=8.0, threads=1)
        cpu = {"value": par["value"], "unit": UNIT, "cores": par["cores"], "kind": "oracle", "sample": par["sample"],
               "serial": {"value": ser["value"], "unit": UNIT, "cores": 1, "sample": ser["sample"]}}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": cfg.dtype, "data": "synthetic", "config": config_dict(cfg, world, args),
        "hbm_model": {"bytes_per_particle_step": m["step_bytes"], "achieved_gbs": step_gbs, "peak_gbs": hbm_peak,
                      "frac": step_gbs / hbm_peak},
        "roofline": roof, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clocks, "repeats": repeats,
        "check": {"total_energy_J": energy, "deactivated": d1["deactivated"], "pool_chunks": d1["pool_chunks"]},
    }
    print(json.dumps(line), flush=True)
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=8)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C2", choices=sorted(W.CONFIGS))
    ap.add_argument("--deposit-mode", type=int, default=0, help="PIC_DEPOSIT_* (0 auto, 1 global, 2 cooperative, 3 tile, 4 tile + fp64 tensor pipe, 5 one fused kernel)")
    ap.add_argument("--sort-interval", type=int, default=None, help="sweeps: sort every N steps (0 = only never)")
    ap.add_argument("--tile", default=None, help="sweeps: cells per sort bin, e.g. 4,4,4")
    ap.add_argument("--sort-key-mode", type=int, default=0, help="sweeps: 0 cell key inside the tile, 1 tile only")
    ap.add_argument("--sigma", type=float, default=None, help="sweeps: thermal momentum spread u/c of every species")
    ap.add_argument("--pusher", type=int, default=0, help="variants: PIC_PUSHER_* (0 Boris, 1 Vay)")
    ap.add_argument("--gather-mode", type=int, default=0, help="variants: PIC_GATHER_* (0 uniform, 1 Galerkin)")
    ap.add_argument("--solver", type=int, default=0, help="variants: PIC_SOLVER_* (0 Yee, 1 CKC)")
    ap.add_argument("--deterministic", action="store_true", help="variants: pic_options.deterministic (integer reductions into J)")
    ap.add_argument("--no-graph", action="store_true", help="variants: launch every kernel of a step separately (pic_options.cuda_graph = 0)")
    ap.add_argument("--box-staging", type=int, default=0, help="variants: PIC_STAGE_* (0 auto = TMA in fp64, 1 element-wise cp.async, 2 TMA)")
    ap.add_argument("--skip-e2e", action="store_true", help="profiling runs: device-resident leg only")
    ap.add_argument("--skip-cpu", action="store_true", help="profiling runs: do not time the oracle")
    ap.add_argument("--skip-probe", action="store_true", help="profiling runs: one launch per on-chip probe instead of 0.2 s")
    ap.add_argument("--traffic", type=float, default=None,
                    help="dram bytes per launch of the dominant kernel from the committed ncu capture (profiles/)")
    args = ap.parse_args(argv)
    if args.steps < 1 or args.warmup < 0:
        ap.error("steps >= 1, warmup >= 0")
    _, _, world = dist_env()
    if world != args.gpus and world > 1:
        ap.error("--gpus %d but WORLD_SIZE=%d" % (args.gpus, world))
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
