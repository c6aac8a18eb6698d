#!/usr/bin/env python
"""bench.py -- particle-steps/s of the Langevin droplet step (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl lv|reference]

A "step" is one pass of the whole hot path (hash, sort, offsets + scatter,
pair force, fused update: SURVEY.md sec. 8(a) rows A1-A7) over all N particles of
the workload, i.e. one simulation time step.  Workload: BASELINE.json
configs[2] ("C3": N = 250 000, three NP types, LJ + Coulomb, gravity,
centrifugal, shrinking interface), the configuration with the N = 2.5e5 the
metric is quoted on; inputs are seeded and synthetic (workloads.py).

Own arm (--impl lv, default):
  value       whole-job particle-steps/s, state resident in HBM, K timed steps of
              the product path (lv_step(1) = one CUDA-graph replay of the whole
              step), device time from a CUDA event pair on the library's stream
              around every step, L2 flushed (256 MiB memset) between timed
              steps, max over ranks.
  stage_ms_per_step / roofline
              the K steps that follow are launched kernel by kernel with an event
              after every stage (lv_stage_timing; ~2.5 us of event overhead per
              stage, hence not the headline): the breakdown, and the pair-force
              kernel's average duration for the roofline -- algorithmic FP32
              flops per launch / that duration, against the FP32 FMA peak
              derived in DESIGN.md.
  resident    the same K steps as one lv_step(K) graph replay without flushes
              (how a simulation actually runs: the 8 MB state stays in L2).
  e2e         set_state(host) + lv_step(1) + get_state(host) per step through
              the C ABI with pinned host buffers, copies inside the timed region.
  cpu_baseline  the fp64 oracle, as it stands, on the host cores (rank 0, N=1).
Multi-GPU: independent replicas, one per rank, no data-path collective
(DESIGN.md "Multi-GPU: replicas only"); value = sum of units / slowest rank.

Reference arm (--impl reference): the oracle timed on the host cores on the
same workload; rank 0 only.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2501_04456_b200 import replicas, tuning, workloads  # noqa: E402

METRIC = "particle-steps/sec at N=2.5e5"
UNIT = "particle-steps/s"
FLUSH_BYTES = 256 << 20            # > 126 MB L2
# Algorithmic FP32 flops of one ordered in-range pair (DESIGN.md "Roofline of
# the pair-force kernel"): 3 sub + (1 mul + 2 fma = 5) + 1 compare for the
# distance test, 1 rcp + 2 mul + 1 fma (2) + 2 mul + 3 fma (6) for LJ and the
# accumulation = 22.  Charged pairs add 4 (rsqrt, mul, fma); not counted here,
# so the figure is a lower bound.
FLOP_PER_PAIR = 22.0
# "algorithmic flops = the in-range ordered pairs x ~33 (distance test +
# force)".  roofline.frac uses THIS figure and the FMA peak measured in the same run; the
# 22-flop count and the nominal peak are kept as secondary keys.
FLOP_PER_PAIR_SURVEY = 33.0
FP32_LANES_PER_SM = 128
KERNEL_OF_PATH = {"list": "k_pair_force_rows", "cells": "k_pair_force_s", "tile": "k_pair_force_t",
                  "packed": "k_pair_force_s", "queued": "k_pair_force_q", "simple": "k_pair_force"}


def source_hash():
    """Content hash of the CUDA sources + the header: ncu figures are only quoted for the
    kernels they were captured on."""
    import hashlib
    h = hashlib.sha256()
    base = os.path.join(ROOT, "paper_2501_04456_b200", "csrc")
    for f in sorted(os.listdir(base)):
        with open(os.path.join(base, f), "rb") as fh:
            h.update(f.encode() + b"\0" + fh.read())
    with open(os.path.join(ROOT, "include", "lv.h"), "rb") as fh:
        h.update(fh.read())
    return h.hexdigest()[:16]


def ncu_record(kernel, workload, start_step, path):
    """The entry of profiles/ncu_kernels.json (written by `python -m paper_2501_04456_b200.ncu_summary`
    from a committed ncu command) for this kernel / workload / step / force path, or None.
    `stale` says whether the sources have changed since the capture."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_kernels.json")) as f:
            recs = json.load(f)
    except Exception:
        return None
    for r in recs:
        if (r.get("kernel") == kernel and r.get("workload") == workload
                and int(r.get("start_step", -1)) == int(start_step) and r.get("path") == path):
            r = dict(r)
            r["stale"] = r.get("source_hash") != source_hash()
            return r
    return None


def peaks():
    p = {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback (B200_PROFILING.md)"}
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            m = json.load(f)
        p.update(hbm_gbs=float(m["hbm_gbs"]), sm_max_mhz=float(m["sm_max_mhz"]),
                 source="MEASURED_PEAKS.json")
    except Exception:
        pass
    return p


class ClockSampler(threading.Thread):
    """SM clock and throttle reasons during the timed region (NVML)."""

    def __init__(self, index, period=0.02):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.sm, self.reasons, self.max_mhz = [], set(), None
        self._stop_evt = threading.Event()
        try:
            import pynvml as nv
            nv.nvmlInit()
            self.nv = nv
            self.h = nv.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake",
        }
        while not self._stop_evt.is_set():
            try:
                self.sm.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop_evt.wait(self.period)

    def finish(self):
        self._stop_evt.set()
        self.join(timeout=2.0)
        return {"sm_mhz": float(np.median(self.sm)) if self.sm else None,
                "sm_max_mhz": float(self.max_mhz) if self.max_mhz else None,
                "samples": len(self.sm), "reasons": sorted(self.reasons)}


def visible_gpu_index(local_rank):
    cvd = os.environ.get("CUDA_VISIBLE_DEVICES")
    if cvd:
        try:
            return int(cvd.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


# ----------------------------------------------------------------- own arm
def timed_steps(sim, torch, flush, k):
    """k steps with stage events, L2 flushed between steps.
    -> (stage ms sums, step ms sum)."""
    sim.stage_timing(k)
    with torch.cuda.stream(sim.stream):
        for _ in range(k):
            if flush is not None:
                flush.zero_()
            sim.step(1)
    stages, tot, n = sim.read_stage_timing()
    assert n == k
    sim.stage_timing(0)
    return stages, tot


def timed_steps_product(sim, torch, flush, k):
    """k steps through the product path -- lv_step(1) = one CUDA-graph replay of the whole
    step -- L2 flushed between steps, one CUDA event pair per step on the library's stream
    (the flush is outside the pairs).  -> step ms sum."""
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(k)]
    with torch.cuda.stream(sim.stream):
        for e0, e1 in ev:
            if flush is not None:
                flush.zero_()
            e0.record()
            sim.step(1)
            e1.record()
    sim.synchronize()
    return sum(e0.elapsed_time(e1) for e0, e1 in ev)


def inrange_pairs(sim):
    """In-range ordered pairs of the current state (lv_compute_forces: always the cells, does
    not disturb a list run)."""
    sim.compute_forces()
    _, cnt = sim.get_forces()
    return float(cnt.astype(np.int64).sum())


def force_path_of(args):
    if args.force_kernel in (None, 2):
        return "cells" if args.no_list else "list"
    return {0: "simple", 1: "queued", 3: "packed", 4: "tile"}[args.force_kernel]


def make_sim(binding, w, args, device, cpc=None, use_list=None):
    """The product path: the workload's tuned grids and -- unless --no-list -- the automatic
    skin neighbour list (lv_set_neighbour_list(skin <= 0, -1))."""
    options = {}
    if args.force_kernel is not None:
        options[binding.OPT_FORCE_KERNEL] = args.force_kernel
    if args.tile_substreams is not None:
        options[binding.OPT_TILE_SUBSTREAMS] = args.tile_substreams
    if cpc is None:
        cpc = args.cells_per_cut if args.cells_per_cut else tuning.cells_per_cut(w)
    if use_list is None:
        use_list = not args.no_list and args.force_kernel in (None, 2)
    nl = (args.skin, -1) if use_list else None      # from_workload's own default is (0, -1) too
    return binding.Simulation.from_workload(w, cells_per_cut=cpc, device=device, options=options or None,
                                            neighbour_list=nl), cpc, use_list


def measure_point(sim, torch, flush, n, steps, warmup, peak_tflops):
    """Flushed product-path time of `steps` steps from the current state, then the stage pass
    over the next `steps` steps and the roofline figures of the pair-force stage."""
    timed_steps_product(sim, torch, flush, max(warmup, 1))
    tot = timed_steps_product(sim, torch, flush, steps)
    p0 = inrange_pairs(sim)
    stages, stot = timed_steps(sim, torch, flush, steps)
    p1 = inrange_pairs(sim)
    pairs = 0.5 * (p0 + p1)
    fm = stages["pair_force"] / steps
    return {"ms_per_step": tot / steps, "value": float(n) * steps / (tot * 1e-3), "unit": UNIT,
            "stage_ms_per_step": {k: v / steps for k, v in stages.items()},
            "kernel_ms": fm, "in_range_ordered_pairs": pairs,
            "frac": FLOP_PER_PAIR_SURVEY * pairs / (fm * 1e-3) * 1e-12 / peak_tflops if fm > 0 else None}


def list_info(sim, use_list):
    if not use_list:
        return None
    st = sim.list_stats()
    return {"rebuilds": st["rebuilds"], "fallback_steps": st["fallback_steps"],
            "entries_used": st["entries_used"], "pool_entries": st["pool_entries"]}


def run_lv(args):
    import torch
    from paper_2501_04456_b200 import binding

    rank, local_rank, world = replicas.env_rank_world()
    if args.gpus != world:
        if world == 1 and args.gpus > 1:
            raise SystemExit("bench.py --gpus N>1 must be launched with torch.distributed.run "
                             "(one rank per GPU)")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the library has no CPU path")
    torch.cuda.set_device(local_rank)
    device = f"cuda:{local_rank}"
    if world > 1:
        replicas.init("nccl")
    binding.load()
    pk = peaks()
    solo = rank == 0 and world == 1

    base = workloads.make_workload(args.workload, state=False)
    w = workloads.make_workload(args.workload, seed=replicas.replica_seed(base.seed, rank))
    n = w.n
    sim, cpc, use_list = make_sim(binding, w, args, device)
    path = force_path_of(args)
    if args.start_step > 0:
        sim.step(args.start_step)
        sim.get_state()                      # synchronises; raises on a non-finite state
    flush = torch.empty(FLUSH_BYTES, dtype=torch.uint8, device=device)
    n_sms = torch.cuda.get_device_properties(device).multi_processor_count
    fma_tflops = sim.measure_fp32_peak()     # the roofline's denominator: measured in this run
    nominal_tflops = n_sms * FP32_LANES_PER_SM * 2 * pk["sm_max_mhz"] * 1e6 * 1e-12

    # ---- timed region: K steps of the product path (graph replay), events on the
    # library's stream around every step --------------------------------------
    timed_steps_product(sim, torch, flush, max(args.warmup, 3))
    l0 = list_info(sim, use_list)
    sampler = ClockSampler(visible_gpu_index(local_rank))
    replicas.barrier()
    torch.cuda.synchronize()
    sampler.start()
    t_wall0 = time.perf_counter()
    tot_ms = timed_steps_product(sim, torch, flush, args.steps)
    torch.cuda.synchronize()
    wall_s = time.perf_counter() - t_wall0
    clocks = sampler.finish()
    replicas.barrier()
    l1 = list_info(sim, use_list)
    # ---- stage pass: the next K steps launched kernel by kernel with an event after every
    # stage (lv_stage_timing); the event records cost ~2.5 us per stage, so this pass is
    # the breakdown and the source of the pair-force kernel time, not the headline
    pairs0 = inrange_pairs(sim)
    stages, stage_tot_ms = timed_steps(sim, torch, flush, args.steps)
    pairs1 = inrange_pairs(sim)
    launches_per_step = sim.launches_per_step()

    ms_max, units = replicas.reduce_timing(tot_ms, float(n) * args.steps, device=device)
    value = units / (ms_max * 1e-3)

    # ---- a longer window without flushes: lv_step(K') as graph replays, the state (and, at this
    # size, the list) L2-resident -- how a simulation actually runs; K' >= 500 so that the
    # rebuilds of the list are averaged over
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    kres = max(args.steps, args.resident_steps)
    sim.step(max(args.warmup, 3))
    sim.synchronize()
    l2 = list_info(sim, use_list)
    e0.record(sim.stream)
    sim.step(kres)
    e1.record(sim.stream)
    e1.synchronize()
    res_ms = e0.elapsed_time(e1)
    l3 = list_info(sim, use_list)
    res_max, _ = replicas.reduce_timing(res_ms, 0.0, device=device)

    # ---- variant (not the headline): the paper's literal scheme, cells rebuilt every step ----
    variants = {}
    if solo and use_list and not args.no_variants:
        vs, _, _ = make_sim(binding, w, args, device, cpc=cpc, use_list=False)
        if args.start_step > 0:
            vs.step(args.start_step)
        v = measure_point(vs, torch, flush, n, args.steps, max(args.warmup, 3), fma_tflops)
        vs.step(max(args.warmup, 3))
        vs.synchronize()
        e0.record(vs.stream)
        vs.step(kres)
        e1.record(vs.stream)
        e1.synchronize()
        v["resident_ms_per_step"] = e0.elapsed_time(e1) / kres
        v["what"] = ("lv_set_neighbour_list off: cell hash, sort, offsets and the cell-walk force kernel "
                     "(k_pair_force_s) every step, as PAPER.md:62-69 does")
        variants["cells_every_step"] = v
        vs.close()

    # ---- variant: many small droplets at once (NEXT-3 batched replicas; the paper's own
    # sizes, Table 1: 10^4 NPs, fill a fraction of a B200) -- R handles on R streams
    if solo and not args.no_variants and args.small_replicas > 0:
        ks = 1000
        sr = {}
        for R_, batched in ((1, False), (args.small_replicas, False), (args.small_replicas, True)):
            rs = replicas.ReplicaSet(lambda seed: workloads.make_workload("P1", seed=seed), R_,
                                     base_seed=1234, device=device, batched=batched, steps_per_launch=10)
            rs.step(100)
            rs.synchronize()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            rs.step(ks)
            rs.synchronize()
            dt_ = time.perf_counter() - t0
            sr[("%d_one_graph" % R_) if batched else str(R_)] = {
                "ms_per_step_of_all": dt_ / ks * 1e3, "value": rs.n_particles * ks / dt_, "unit": UNIT}
            npart = rs.workloads[0].n
            rs.close()
        variants["small_replicas"] = {
            "what": "independent P1 droplets (Table 1 row 1 shape, N = %d each) on one GPU, each replica "
                    "bit-identical to its solo run (test_replica_set_equals_solo_runs): R handles on R streams "
                    "driven from the host, and lv_batch = ONE CUDA graph with 10 steps of every replica as "
                    "parallel branches; wall clock over %d resident steps, no L2 flush" % (npart, ks),
            "replicas": sr,
            "speedup": sr["%d_one_graph" % args.small_replicas]["value"] / sr["1"]["value"],
        }

    # ---- NEXT-1 rows: the paper's observables on the device (synchronous calls) -------
    observables = {}
    if solo and not args.no_variants:
        nb = 100
        drb = 5.0 / nb                                  # g(r) to r = 5 sigma, as in the long-run tests
        sim.observe_rdf(drb, nb); sim.observe_radial(w.R0 / 100.0, 128)      # warm
        t0 = time.perf_counter()
        for _ in range(5):
            hh, _ = sim.observe_rdf(drb, nb)
        t_rdf = (time.perf_counter() - t0) / 5
        t0 = time.perf_counter()
        for _ in range(5):
            sim.observe_radial(w.R0 / 100.0, 128)
        t_rad = (time.perf_counter() - t0) / 5
        t0 = time.perf_counter()
        for _ in range(5):
            cl = sim.observe_clusters(1.5, want_labels=False)
        t_cl = (time.perf_counter() - t0) / 5
        pal = [0x00ff8040, 0x004080ff, 0x0040ff80, 0x00c0c0c0]
        eye = 2.6 * w.R0
        sim.render(eye, 900.0 * eye / (2.2 * w.R0), 0.4, 0.3, 1920, 1080, pal, on_device=True)
        sim.synchronize()
        t0 = time.perf_counter()
        for _ in range(5):
            sim.render(eye, 900.0 * eye / (2.2 * w.R0), 0.4, 0.3, 1920, 1080, pal, on_device=True)
        sim.synchronize()
        t_view = (time.perf_counter() - t0) / 5
        observables = {
            "view": {"ms": t_view * 1e3, "width": 1920, "height": 1080,
                     "how": "lv_render: 1920x1080 perspective splat of all NPs into a device buffer, wall clock"},
            "clusters": {"ms": t_cl * 1e3, "bond_factor": 1.5, "n_clusters": cl["n_clusters"],
                         "largest": cl["largest"],
                         "how": "lv_observe_clusters: cell rebuild + union-find + statistics, wall clock"},
            "rdf": {"ms": t_rdf * 1e3, "bins": nb, "dr": drb, "ordered_pairs": int(hh.sum()),
                    "how": "lv_observe_rdf: cell rebuild + pair walk + D2H of the histogram, wall clock"},
            "radial": {"ms": t_rad * 1e3, "bins": 128,
                       "how": "lv_observe_radial: one pass over the NPs + D2H, wall clock"},
        }

    # ---- e2e: host buffers through the C ABI, copies inside the timed region
    hp = torch.empty((n, 3), dtype=torch.float32).pin_memory()
    hv = torch.empty((n, 3), dtype=torch.float32).pin_memory()
    ht = torch.empty((n,), dtype=torch.int32).pin_memory()
    R, st = sim.get_state_ptrs(hp.data_ptr(), hv.data_ptr(), ht.data_ptr(), 0)
    ke = args.e2e_steps if args.e2e_steps > 0 else args.steps

    def e2e_loop(k, st):
        for _ in range(k):
            sim.set_state_ptrs(hp.data_ptr(), hv.data_ptr(), ht.data_ptr(), st, 0)
            sim.step(1)
            _, st = sim.get_state_ptrs(hp.data_ptr(), hv.data_ptr(), ht.data_ptr(), 0)
        return st

    st = e2e_loop(3, st)
    replicas.barrier()
    torch.cuda.synchronize()
    e0.record(sim.stream)
    t0 = time.perf_counter()
    st = e2e_loop(ke, st)
    e1.record(sim.stream)
    e1.synchronize()
    e2e_wall_ms = (time.perf_counter() - t0) * 1e3
    e2e_ms = max(e0.elapsed_time(e1), e2e_wall_ms)
    replicas.barrier()
    e2e_max, e2e_units = replicas.reduce_timing(e2e_ms, float(n) * ke, device=device)

    # ---- roofline of the dominant kernel (pair force) ----------------------
    force_ms = stages["pair_force"] / args.steps
    pairs = 0.5 * (pairs0 + pairs1)
    kernel = KERNEL_OF_PATH[path]
    achieved = FLOP_PER_PAIR_SURVEY * pairs / (force_ms * 1e-3) * 1e-12
    rec = ncu_record(kernel, w.name, args.start_step, path)
    usable = rec is not None and not rec["stale"]
    roofline = {
        "kernel": kernel, "bound": "alu",
        "achieved": achieved, "peak": fma_tflops, "unit": "TFLOP/s",
        "frac": achieved / fma_tflops,
        "flop_per_pair": FLOP_PER_PAIR_SURVEY,
        "peak_source": "FMA microkernel of this run (lv_measure_fp32_peak): %.1f TFLOP/s; nominal %d SMs x 128 "
                       "FP32 lanes x 2 x %.0f MHz = %.1f TFLOP/s" % (fma_tflops, n_sms, pk["sm_max_mhz"], nominal_tflops),
        "algorithmic_flops_per_launch": FLOP_PER_PAIR_SURVEY * pairs,
        "in_range_ordered_pairs": pairs,
        # secondary conventions: DESIGN.md's own count of 22 flop per pair, and the nominal peak
        "frac_at_22_flop_per_pair": FLOP_PER_PAIR * pairs / (force_ms * 1e-3) * 1e-12 / fma_tflops,
        "frac_of_nominal_peak": achieved / nominal_tflops,
        # from the committed ncu capture of this kernel on this workload / step / path
        # (profiles/ncu_kernels.json); null when there is none or the sources have changed since
        "traffic": rec["dram_bytes"] if usable else None,
        "executed_fp32_frac": rec["executed_fp32_frac"] if usable else None,
        "ncu": ({"report": rec["report"], "duration_us": rec["duration_us"], "issue_active_pct": rec["issue_active_pct"],
                 "l1_data_pipe_pct": rec["l1_data_pipe_pct"], "lts_bytes": rec["lts_bytes"],
                 "source_hash": rec["source_hash"], "stale": rec["stale"]} if rec is not None else None),
        # the same kernel against the HBM roofline: its measured DRAM traffic (the list is streamed
        # once per launch) over the kernel time, of the measured copy bandwidth
        "hbm": ({"achieved": rec["dram_bytes"] / (force_ms * 1e-3) * 1e-9, "peak": pk["hbm_gbs"], "unit": "GB/s",
                 "frac": rec["dram_bytes"] / (force_ms * 1e-3) * 1e-9 / pk["hbm_gbs"],
                 "peak_source": pk["source"]} if usable else None),
        "kernel_ms": force_ms,
        "share_of_step": stages["pair_force"] / tot_ms,          # against the graph-replayed (headline) step
        "share_of_stage_pass": stages["pair_force"] / stage_tot_ms,   # that pass carries event overhead
        "kernel_ms_source": "stage-event pass over the K steps that follow the headline region "
                            "(same workload, kernels launched one by one with an event after each stage)",
        "hbm_algorithmic_gbs": 32.0 * n / (force_ms * 1e-3) * 1e-9,
        "hbm_peak_gbs": pk["hbm_gbs"],
    }

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": config_of(w, args.start_step, extra={
            "cells_per_cut": list(cpc) if cpc else [1] * w.n_types,
            "force_path": path, "force_kernel": kernel,
            "neighbour_list": ("automatic skin and pool (lv_set_neighbour_list(<= 0, -1)): cells + list rebuilt on the "
                               "device when an NP has moved skin/2, cell kernel when the pool is too small")
            if use_list else "off: cells rebuilt every step",
            "replicas": world, "parallelism": "independent replicas, no collective",
            "l2": "flushed between timed steps (256 MiB memset on the same stream)",
            "timing": "lv_step(1) = one CUDA-graph replay per step; a CUDA event pair on the library's stream "
                      "around every step (the flush outside it); sum over K"}),
        "clocks": clocks,
        "gpu_launches": launches_per_step * args.steps,
        "launches_per_step": launches_per_step,
        "list": ({"rebuilds_in_timed_region": l1["rebuilds"] - l0["rebuilds"],
                  "fallback_steps_in_timed_region": l1["fallback_steps"] - l0["fallback_steps"],
                  "entries_used": l1["entries_used"], "pool_entries": l1["pool_entries"]} if use_list else None),
        "stage_ms_per_step": {k: v / args.steps for k, v in stages.items()},
        "stage_pass_ms_per_step": stage_tot_ms / args.steps,
        "wall_s_timed_region": wall_s,
        "roofline": roofline,
        "variants": variants,
        "observables": observables,
        "resident": {"value": float(n) * kres * world / (res_max * 1e-3), "unit": UNIT,
                     "ms_per_step": res_max / kres, "steps": kres,
                     "rebuilds": (l3["rebuilds"] - l2["rebuilds"]) if use_list else None,
                     "how": "lv_step(K') as CUDA-graph replays, no L2 flush, events around the K' steps"},
        "e2e": {"value": e2e_units / (e2e_max * 1e-3), "unit": UNIT, "steps": ke,
                "h2d_bytes_per_step": 28 * n, "d2h_bytes_per_step": 28 * n + 16,
                "ms_per_step": e2e_max / ke,
                "how": "lv_set_state(host pinned) + lv_step(1) + lv_get_state(host pinned) per step "
                       "(the first step after lv_set_state runs on the cell kernel: no list is built for one step)"},
    }

    # ---- further points of the schedule (not the headline) -----------------
    if solo and args.snapshots:
        snaps = []
        for target in args.snapshots:
            _, _, _, _, cur = sim.get_state()
            if target < cur:
                continue
            sim.step(target - cur)
            _, _, _, Rn, cur = sim.get_state()
            m = measure_point(sim, torch, flush, n, args.snapshot_steps, 10, fma_tflops)
            m.update(step=cur, R=Rn, list=list_info(sim, use_list))
            m["roofline_frac"] = m.pop("frac")
            m["pair_force_ms"] = m["kernel_ms"]
            snaps.append(m)
        out["snapshots"] = snaps

    # ---- the whole shrinking schedule in one call (reading R26: up to step 17 800 for C3) ----
    if solo and args.schedule_steps > 0:
        ss, _, _ = make_sim(binding, w, args, device, cpc=cpc, use_list=use_list)
        ss.step(10)
        ss.synchronize()
        e0.record(ss.stream)
        ss.step(args.schedule_steps - 10)
        e1.record(ss.stream)
        e1.synchronize()
        sch_ms = e0.elapsed_time(e1)
        _, _, _, Rend, cur = ss.get_state()
        out["schedule_mean"] = {"steps": args.schedule_steps, "ms_per_step": sch_ms / (args.schedule_steps - 10),
                                "value": float(n) * (args.schedule_steps - 10) / (sch_ms * 1e-3), "unit": UNIT,
                                "end_step": cur, "end_R": Rend, "status": ss.status(), "list": list_info(ss, use_list),
                                "how": "one lv_step(S) from the initial state, device time, no flush"}
        ss.close()

    # ---- the other BASELINE configs, one short point each (default path, tuned grids) --------
    if solo and args.other_workloads:
        others = {}
        for name in args.other_workloads:
            if name == w.name:
                continue
            wo = workloads.make_workload(name)
            so, cpo, ulo = make_sim(binding, wo, args, device)
            m = measure_point(so, torch, flush, wo.n, args.other_steps, 10, fma_tflops)
            m.update(n_particles=wo.n, cells_per_cut=list(cpo), force_path=path, list=list_info(so, ulo))
            others[name] = m
            so.close()
        out["workloads"] = others

    # ---- oracle beside it (rank 0, N = 1 only) -----------------------------
    if solo and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(args.workload, args.cpu_seconds)
    sim.close()
    if rank == 0:
        print(json.dumps(out))


def config_of(w, start_step, extra=None):
    """The same workload keys in both arms (the driver compares them)."""
    c = {"workload": f"{w.name} (BASELINE.json configs[{int(w.name[1]) - 1}]): N={w.n}, {w.n_types} types"
                     if w.name[0] == "C" and w.name[1:].isdigit() else w.name,
         "n_particles": w.n, "start_step": start_step}
    if extra:
        c.update(extra)
    return c



# ------------------------------------------------------------ oracle timing
def cpu_baseline(name, budget_s):
    """The oracle as it stands on the host cores: full-size steps of the same
    workload from its initial state until ~budget_s of work is done."""
    import oracle
    w = workloads.make_workload(name)
    p = oracle.params_from_workload(w)
    x, v = w.pos.astype(np.float64), w.vel.astype(np.float64)
    t0 = time.perf_counter()
    x, v, bad = oracle.step(p, x, v, w.type, step0=0, nsteps=1)
    t1 = time.perf_counter() - t0
    m = int(max(1, min(50, budget_s / max(t1, 1e-3))))
    t0 = time.perf_counter()
    x, v, bad = oracle.step(p, x, v, w.type, step0=1, nsteps=m)
    dt = time.perf_counter() - t0
    out = {"value": w.n * m / dt, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle",
           "sample": f"{m} full-size steps (N={w.n}) of {w.name} from its initial state, "
                     f"fp64, OpenMP over particles, {dt:.1f} s",
           "ms_per_step": dt / m * 1e3}
    # the same oracle on ONE core ("single-thread and OpenMP-all-cores"): a child
    # process with OMP_NUM_THREADS=1 -- the thread count of an OpenMP runtime is fixed at start
    try:
        import subprocess
        env = dict(os.environ, OMP_NUM_THREADS="1")
        r = subprocess.run([sys.executable, os.path.abspath(__file__), "--oracle-single-thread", "--workload", name],
                           env=env, capture_output=True, text=True, timeout=300)
        out["single_thread"] = json.loads(r.stdout.strip().splitlines()[-1])
    except Exception as e:              # a reported baseline: never fails the bench
        out["single_thread"] = {"error": repr(e)[:200]}
    return out


def oracle_single_thread(name):
    """Child of cpu_baseline (OMP_NUM_THREADS=1): two full-size oracle steps on one core."""
    import oracle
    w = workloads.make_workload(name)
    p = oracle.params_from_workload(w)
    x, v = w.pos.astype(np.float64), w.vel.astype(np.float64)
    t0 = time.perf_counter()
    x, v, bad = oracle.step(p, x, v, w.type, step0=0, nsteps=2)
    dt = time.perf_counter() - t0
    print(json.dumps({"value": w.n * 2 / dt, "unit": UNIT, "cores": oracle.max_threads(),
                      "ms_per_step": dt / 2 * 1e3, "sample": f"2 full-size steps (N={w.n}) of {w.name}, fp64"}))


def run_reference(args):
    rank, _, world = replicas.env_rank_world()
    if rank != 0:
        return
    import oracle
    w = workloads.make_workload(args.workload)
    n = w.n
    p = oracle.params_from_workload(w)
    x, v = w.pos.astype(np.float64), w.vel.astype(np.float64)
    t0 = time.perf_counter()
    x, v, _ = oracle.step(p, x, v, w.type, step0=0, nsteps=1)
    t1 = time.perf_counter() - t0
    total = args.steps + args.warmup
    sample = f"full-size steps (N={n})"
    if t1 * total > args.reference_budget_s:
        # bounded sample: a scaled-down copy of the workload at the same volume
        # fractions (workloads.make_workload(name, n)), so a step costs the same per particle
        n = max(2048, int(n * args.reference_budget_s / (t1 * total)))
        w = workloads.make_workload(args.workload, n)
        p = oracle.params_from_workload(w)
        x, v = w.pos.astype(np.float64), w.vel.astype(np.float64)
        sample = f"scaled-down copy with N={n} at the same volume fractions"
        done = 0
    else:
        done = 1
    step = done
    for _ in range(max(args.warmup - done, 0)):
        x, v, _ = oracle.step(p, x, v, w.type, step0=step, nsteps=1)
        step += 1
    t0 = time.perf_counter()
    x, v, bad = oracle.step(p, x, v, w.type, step0=step, nsteps=args.steps)
    dt = time.perf_counter() - t0
    value = n * args.steps / dt
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": config_of(workloads.make_workload(args.workload, state=False), 0, extra={"sample": sample, "sample_n_particles": n}),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.max_threads(),
                         "kind": "oracle", "sample": f"{args.steps} {sample} of {w.name}, fp64"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=500)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--impl", default="lv", choices=["lv", "reference"])
    ap.add_argument("--workload", default="C3")
    ap.add_argument("--start-step", type=int, default=0)
    ap.add_argument("--cells-per-cut", type=int, nargs="*", default=None)
    ap.add_argument("--force-kernel", type=int, default=None,
                    help="lv_set_option(LV_OPT_FORCE_KERNEL): 0 simple, 1 queued, 2 segments (default), 3 packed f32x2, "
                         "4 tile (shared candidate stream); anything but 2 switches the neighbour list off")
    ap.add_argument("--tile-substreams", type=int, default=None)
    ap.add_argument("--no-list", action="store_true",
                    help="headline without the skin neighbour list: cells rebuilt every step, cell-walk force kernel")
    ap.add_argument("--skin", type=float, default=0.0, help="skin of the neighbour list (<= 0: automatic)")
    ap.add_argument("--resident-steps", type=int, default=500)
    ap.add_argument("--schedule-steps", type=int, default=-1,
                    help="steps of the whole-schedule run (-1: 17800 for C3, else 0 = skip)")
    ap.add_argument("--other-workloads", nargs="*", default=["C1", "C2", "C4", "C5"])
    ap.add_argument("--other-steps", type=int, default=20)
    ap.add_argument("--oracle-single-thread", action="store_true", help=argparse.SUPPRESS)
    ap.add_argument("--no-variants", action="store_true", help="skip the variants and the observables")
    ap.add_argument("--small-replicas", type=int, default=16,
                    help="size of the concurrent small-droplet replica set of the variants leg (0: skip)")
    ap.add_argument("--e2e-steps", type=int, default=0)
    ap.add_argument("--snapshots", type=int, nargs="*", default=[10000, 17000])
    ap.add_argument("--snapshot-steps", type=int, default=100)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--reference-budget-s", type=float, default=150.0)
    args = ap.parse_args()
    if args.schedule_steps < 0:
        args.schedule_steps = 17800 if (args.workload == "C3" and args.start_step == 0) else 0
    if args.oracle_single_thread:
        oracle_single_thread(args.workload)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_lv(args)


if __name__ == "__main__":
    main()
