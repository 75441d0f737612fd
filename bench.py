#!/usr/bin/env python
"""bench.py -- throughput of the full hydrodynamic update on B200 (BASELINE.json metric: fp64 cell
updates/s per HD step on 1 B200; achieved HBM GB/s vs peak).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl ours|reference]

A "step" is one pass of the whole hot path (ghost fill, dt reduction, source sub-steps, X/Y/Z sweeps,
orbital advection where on, new velocities) over the whole synthetic mesh.  Prints ONE JSON line.
  value      cells * K / device time of fargo_step(K) (CUDA events on the context's stream, max over ranks),
             inputs resident in HBM, one CUDA-graph replay per step;
  e2e        same metric through the public API with pinned HOST buffers: every step does
             fargo_set_fields (H2D) + fargo_step(1) + fargo_get_fields (D2H) inside the timed region;
  roofline   the launcher with the largest share of the step, timed live with per-launch CUDA events
             (fargo_profile) in a second region of K steps: algorithmic bytes / mean launch duration
             against the measured copy bandwidth of MEASURED_PEAKS.json;
  kernels    the same for every launcher (share of the step, GB/s), step_roofline for the whole update;
  cpu_baseline  the CPU oracle, as it stands, single thread, on a bounded sample of the same recipe.
With --gpus N > 1 (torchrun) every rank runs an independent replica of the workload ("replicas only",
DESIGN.md section 8(e)): no data-path collective; value = N * cells * K / max-over-ranks time.
--impl reference times the CPU oracle (there is no reference implementation to install: the reference
is a paper), on rank 0 only.
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

from paper_1602_02359_b200 import workloads as W  # noqa: E402

METRIC = "fp64 cell updates/s per HD step"
UNIT = "cell updates/s"


# ---------------------------------------------------------------------------------- workloads -------
def make_workload(name: str):
    """(workload, bounded oracle sample of the same recipe, description of the sample)."""
    if name.startswith("noise"):
        n = int(name[5:])
        sample = W.noise_box(shape3=(n, min(n, 64), min(n, 64)))
        return W.noise_box(n), sample, "same recipe on a %dx%dx%d slab" % (n, min(n, 64), min(n, 64))
    if name.startswith("mhd"):   # NEXT-4: the config-5 box threaded by a magnetic field (MOC + constrained transport)
        n = int(name[3:])
        return W.mhd_box(n), W.mhd_box(shape3=(n, min(n, 32), min(n, 32))), "same recipe on a %dx%dx%d slab" % (n, min(n, 32), min(n, 32))
    if name == "disk3d":
        return W.disk3d(), W.disk3d(1536, 32, 16), "same recipe on 1536x32x16 (full rings, fewer r and theta cells)"
    if name == "disk3dvisc":   # config 4 with a kinematic viscosity: the 3-D viscous stress of NEXT-1 (Eqs. B3, B6)
        import dataclasses
        full, small = W.disk3d(), W.disk3d(1536, 32, 16)
        for w in (full, small):
            w.params = dataclasses.replace(w.params, nu=1e-5)
            w.name += "_nu1e-5"
        return full, small, "same recipe on 1536x32x16 (full rings, fewer r and theta cells)"
    if name == "sheet3d":   # NEXT-1: shearing sheet (Eqs. 28-30, Tab. 2), adiabatic, orbital advection on
        return W.sheet3d(), W.sheet3d(1024, 32, 16), "same recipe on 1024x32x16 (full rows, fewer y and z cells)"
    if name == "disk3dlive":   # NEXT-2: config 4 with its planet live (RK5 + gas force by direct summation)
        return W.disk3d_live(), W.disk3d_live(1536, 32, 16), "same recipe on 1536x32x16 (full rings, fewer r and theta cells)"
    if name == "disk2d":
        return W.disk2d(), W.disk2d(), "the whole 768x256 mesh"
    if name == "sound":
        return W.sound_wave(), W.sound_wave(), "the whole 32^3 mesh"
    if name == "sod":
        return W.sod(), W.sod(), "the whole 512x4x4 mesh"
    raise SystemExit("unknown workload " + name)


# roofline.traffic and the fp64-pipe figure are READ from the tracked raw ncu export of this workload
# (profiles/ncu_raw_<workload>_<kernel source hash>.csv, see paper_1602_02359_b200/profiling.py); when the export was
# captured on other kernel sources than the ones built here, traffic is null and the line says "stale".
CONFIG_OF = {"mhd128": "5 with a magnetic field (NEXT-4 workload)", "mhd256": "5 with a magnetic field (NEXT-4 workload)", "mhd512": "5 with a magnetic field (NEXT-4 workload)", "sheet3d": "none (NEXT-1 workload)", "disk3dlive": "4 with a live planet (NEXT-2 workload)", "disk3dvisc": 4, "noise64": 5, "noise128": 5, "noise256": 5, "noise512": 5, "disk3d": 4, "disk2d": 3, "sound": 1, "sod": 2}


def algorithmic_reals(w):
    """Reals (read + written) per ACTIVE cell that each launcher must move if every array it touches
    crosses HBM exactly once, and the fused-plan total of SURVEY.md 8(d.3)."""
    nd = sum(1 for n in (w.mesh.nx, w.mesh.ny, w.mesh.nz) if n > 1)
    adi = w.eos == W.ADIABATIC
    pot = w.geometry != W.CARTESIAN and (w.params.gm_star != 0 or w.params.planet_mass != 0)
    nq = (1 if adi else 0) + 2 * nd
    visc = w.params.nu > 0
    k = {
        "vmean": 1,
        "dt": (2 if adi else 1) + nd,
        "source": ((2 if adi else 1) + nd + (1 if pot else 0)) + (nd + (1 if adi else 0)),
        "source_a": (2 + nd + (1 if pot else 0)) + nd,
        "source_b": (1 + (1 if adi else 0) + nd) + (nd + (1 if adi else 0)),
        "source_bc": (2 + nd) + (nd + 1),
        # 7d: tensor kernel (rho, v -> components) + force kernel (rho, v, components -> v)
        # 3-D, wrapped X: one pass, the tensor is never stored (rho, v -> v); else tensor kernel + force kernel
        "source_d": ((1 + 3) + 3 if w.mesh.bc[0][0] == W.PERIODIC else ((1 + 3) + 6) + ((1 + 3 + 6) + 3)) if nd == 3
        else (3 + 3) + (3 + 3 + 2),
        "first_sweep": (1 + (1 if adi else 0) + nd) + (1 + nq),
        "sweep": (1 + nq + 1) + (1 + nq),
        "orbital": (1 + nq) + (1 + nq),
        "newvel": (1 + 2 * nd) + nd,
        "potential": 1,     # live planets: Phi rewritten every update
        "planets": 1,       # gas force: rho read once per planet (ring served by L1 for the further ones)
        "newvel_dt": (1 + 2 * nd + (1 if adi else 0)) + nd,
        # NEXT-4 (3-D): B joins the dt pass; pressure: rho, B, v_b -> v_b; emf (three kernels): rho, two v and two B
        # components each -> eps and two star values; tension: rho, B, 6 star values, v -> v; ct: eps, B -> B
        "mhd_pressure": (1 + 3 + 3) + 3, "mhd_emf": 3 * (1 + 2 + 2) + 9, "mhd_tension": (1 + 3 + 6 + 3) + 3, "mhd_ct": (3 + 3) + 3,
    }
    if getattr(w, "bfield", None):
        k["dt"] += 3
    if not adi:
        k["source_bc"] = 0
    else:
        k["source_b"] = 0
    if not visc:
        k["source_d"] = 0
    # fused plan of SURVEY.md 8(d.3): dt, one source pass, one pass per direction, orbital, Eq. 51 folded
    state_r = (2 if adi else 1) + nd                                  # rho, e (adiabatic), velocities
    fused = state_r                                                   # dt
    fused += (state_r + (1 if pot else 0)) + (nd + (1 if adi else 0))   # source: state (+ phi) -> e', v'
    npass = nd + (1 if w.params.fargo_on else 0)
    for p in range(npass):
        reads = state_r if p == 0 else (1 + nq + 1)                   # first pass forms the momenta on the fly
        writes = (1 + nq) if p < npass - 1 else (1 + (1 if adi else 0) + nd)   # last pass ends with Eq. 51
        fused += reads + writes
    return k, fused


# ---------------------------------------------------------------------------------- clocks ----------
class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md, clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.lines, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 8:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (copy, read+write bytes)"
    except Exception:
        return 6650.0, "fallback of B200_PROFILING.md (MEASURED_PEAKS.json absent)"


# ---------------------------------------------------------------------------------- ranks -----------
def rank_barrier(world: int):
    """Barrier over the process group (no-op for one process)."""
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def rank_max(ms: float, world: int, device: str) -> float:
    """Max over ranks of a device-measured time: the slowest replica defines the job's time."""
    if world == 1:
        return ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(cells_per_rank: int, steps: int, world: int, ms: float) -> float:
    """Replicas only: every rank updates its own mesh, value = all cells / max time."""
    return world * cells_per_rank * steps / (ms * 1e-3)


# ---------------------------------------------------------------------------------- reference arm ---
def oracle_rate(sample, steps, warmup):
    from oracle.binding import Oracle
    o = Oracle(sample.mesh, sample.geometry, sample.eos, sample.params)
    o.set_fields(*sample.fields())
    if sample.planets:
        o.set_planets(**sample.planets)
    if sample.bfield:
        o.set_bfield(**sample.bfield)
    o.step(warmup)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    return sample.mesh.ncells * steps / dt, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w, sample, desc = make_workload(args.workload)
    steps = max(1, min(args.steps, max(1, int(40e6 // sample.mesh.ncells))))   # bound the whole run to minutes
    warm = min(args.warmup, 1)
    rate, dt = oracle_rate(sample, steps, warm)
    out = {
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / steps * (w.mesh.ncells / sample.mesh.ncells),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "baseline_config": CONFIG_OF[args.workload],
                   "note": "CPU oracle (plain C++, one thread) timed on %d step(s) of a bounded sample; ms_per_step is "
                           "scaled to the full mesh" % steps},
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out))


# ---------------------------------------------------------------------------------- our arm ---------
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1602_02359_b200 import Fargo

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        rank_barrier(world)
        torch.cuda.synchronize()

    def max_over_ranks(ms):
        return rank_max(ms, world, "cuda")

    w, sample, sample_desc = make_workload(args.workload)
    prec = 32 if args.fp32 else 64
    g = Fargo(w.mesh, w.geometry, w.eos, w.params, precision=prec, mhd=w.bfield is not None)
    es = 8 if prec == 64 else 4
    ncell = w.mesh.ncells
    tdt = torch.float64 if prec == 64 else torch.float32
    host_in = [None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to(tdt).pin_memory() for a in w.fields()]
    g.set_fields(*host_in)
    if w.planets:
        g.set_planets(**w.planets)
    if w.bfield:
        g.set_bfield(**w.bfield)
    K, Wm = args.steps, max(args.warmup, 3)

    # ---- region 1: device-resident throughput (graph replay) ----
    g.step(Wm)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    l0 = g.kernel_launches()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0 = g.time()[2]
    e0.record(g.stream)
    g.step(K)
    e1.record(g.stream)
    barrier()
    clocks = sampler.stop()
    if g.time()[2] - n0 != K:   # t_stop reached: later updates are no-ops and must not be counted as cell updates
        raise SystemExit("only %d of %d updates ran inside the timed region (t_stop reached): use fewer steps" % (g.time()[2] - n0, K))
    ms = max_over_ranks(e0.elapsed_time(e1))
    launches = g.kernel_launches() - l0
    value = whole_job_rate(ncell, K, world, ms)

    # ---- region 2: per-launcher CUDA-event timing (plain launches) ----
    g.profile(True)
    e2, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e2.record(g.stream)
    g.step(K)
    e3.record(g.stream)
    rep = g.profile_report()
    g.profile(False)
    ms_prof = e2.elapsed_time(e3)
    reals, fused_reals = algorithmic_reals(w)
    if "newvel_dt" in rep:
        reals["dt"] = 0   # only the one-block finish is left of the dt pass: its bytes moved into newvel_dt
    peak, peak_src = measured_peak()
    total_ms = sum(v[1] for v in rep.values())
    kernels = {}
    first_sweep = next((n for n in ("sweep_x", "sweep_y", "sweep_z") if n in rep), None)
    for name, (nk, tms) in rep.items():
        key = "first_sweep" if name == first_sweep else ("sweep" if name.startswith("sweep") else name)
        r = reals.get(key, 0)
        calls = K * ((3 if w.bfield else 2) if name == "bc" else 1)
        per_launch_ms = tms / calls
        gbs = (r * es * ncell / (per_launch_ms * 1e-3) / 1e9) if r else None
        kernels[name] = {"share": tms / total_ms, "ms_per_launch": per_launch_ms, "kernels": nk // calls,
                         "algorithmic_bytes_per_cell": r * es, "achieved_gbs": gbs,
                         "frac": (gbs / peak) if gbs else None}
    dom = max((n for n in kernels if kernels[n]["achieved_gbs"]), key=lambda n: kernels[n]["share"])
    from paper_1602_02359_b200 import profiling as P
    ncu, ncu_file, ncu_stale = P.ncu_table(args.workload + ("_fp32" if prec == 32 else ""))
    for name, e in ncu.items():   # per launch, beside the live timing of the same launcher
        if name in kernels and e["launches"]:
            per = max(1, kernels[name]["kernels"]) * ((3 if w.bfield else 2) if name == "bc" else 1)   # kernels of this launcher per update
            upd = e["launches"] / per
            kernels[name]["ncu_dram_bytes_per_cell"] = None if ncu_stale else e["dram_bytes"] / upd / ncell
            kernels[name]["ncu_fp64_pipe_pct"] = None if (ncu_stale or not e["fp64"]) else sum(e["fp64"]) / len(e["fp64"])
            # thread-level instructions per cell and update, and instructions issued per cycle and SM (of 4)
            kernels[name]["ncu_inst_per_cell"] = None if (ncu_stale or not e["inst"]) else 32.0 * e["inst"] / upd / ncell
            kernels[name]["ncu_ipc_per_sm"] = None if (ncu_stale or not e["ipc"]) else sum(e["ipc"]) / len(e["ipc"])
    dom_ncu = kernels[dom].get("ncu_dram_bytes_per_cell")
    roofline = {"bound": "hbm", "kernel": dom, "achieved": kernels[dom]["achieved_gbs"], "peak": peak, "unit": "GB/s",
                "frac": kernels[dom]["frac"],
                "traffic": dom_ncu * ncell if dom_ncu else None,
                "traffic_source": ("%s (ncu --set full --clock-control none of this command; dram__bytes_read.sum + "
                                   "dram__bytes_write.sum per launch)" % ncu_file) if ncu_file else "no tracked ncu export for this workload",
                "traffic_note": ("stale: %s was captured on other kernel sources than %s" % (ncu_file, P.kernel_source_hash()))
                if ncu_stale else None,
                "kernel_source_hash": P.kernel_source_hash(),
                "peak_source": peak_src,
                "fp64_pipe_pct_ncu": kernels[dom].get("ncu_fp64_pipe_pct"),
                "algorithmic_bytes_per_launch": kernels[dom]["algorithmic_bytes_per_cell"] * ncell,
                "ms_per_launch": kernels[dom]["ms_per_launch"], "share_of_step": kernels[dom]["share"]}
    step_gbs = fused_reals * es * ncell / (ms / K * 1e-3) / 1e9
    as_built = sum(reals["first_sweep" if n == first_sweep else ("sweep" if n.startswith("sweep") else n)] * es
                   for n in rep if n in reals or n.startswith("sweep"))
    built_gbs = as_built * ncell / (ms / K * 1e-3) / 1e9
    # DRAM bytes per cell and update that ncu counted (tracked export, same kernel sources), summed over the launchers
    ncu_step = None
    if ncu and not ncu_stale:
        ncu_step = sum(k.get("ncu_dram_bytes_per_cell") or 0.0 for n, k in kernels.items()) or None
    step_roofline = {"algorithmic_bytes_per_cell_fused_plan": fused_reals * es,
                     "algorithmic_bytes_per_cell_as_built": as_built,
                     "achieved_gbs_vs_fused_plan": step_gbs, "frac_of_measured_peak": step_gbs / peak,
                     "frac_of_nominal_8TBs": step_gbs / 8000.0,
                     "achieved_gbs_as_built": built_gbs, "frac_of_measured_peak_as_built": built_gbs / peak,
                     "frac_of_nominal_8TBs_as_built": built_gbs / 8000.0,
                     "ncu_dram_bytes_per_cell_update": ncu_step,
                     "frac_of_nominal_8TBs_ncu_dram": (ncu_step * ncell / (ms / K * 1e-3) / 1e9 / 8000.0) if ncu_step else None,
                     # the bound the update actually reaches: instructions per cell and update
                     "ncu_inst_per_cell_update": (sum(k.get("ncu_inst_per_cell") or 0.0 for k in kernels.values()) or None)
                     if (ncu and not ncu_stale) else None,
                     "ms_per_step_profiled": ms_prof / K}

    # ---- region 3: end to end through the public API with pinned host buffers ----
    ke = max(1, min(K, args.e2e_steps))
    if args.no_e2e:
        ke = 0
    e2e = None
    if ke > 0:
        host_out = [None if a is None else torch.empty_like(a).pin_memory() for a in host_in]
        cur = host_in
        g.set_fields(*cur); g.step(1); g.get_fields(host_out)   # warm the path once
        barrier()
        e4, e5 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e4.record(g.stream)
        for _ in range(ke):
            g.set_fields(*cur)
            g.step(1)
            g.get_fields(host_out)
            cur = host_out
        e5.record(g.stream)
        barrier()
        ms_e2e = max_over_ranks(e4.elapsed_time(e5))
        nfield = sum(1 for a in host_in if a is not None)
        e2e = {"value": whole_job_rate(ncell, ke, world, ms_e2e), "unit": UNIT, "h2d_bytes_per_step": nfield * ncell * es,
               "d2h_bytes_per_step": nfield * ncell * es, "steps": ke, "ms_per_step": ms_e2e / ke}

    # ---- CPU baseline: the oracle as it stands, one thread, bounded sample (rank 0, N = 1) ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        nst = max(1, int(20e6 // sample.mesh.ncells))
        rate, _ = oracle_rate(sample, nst, 0)
        cpu = {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": "%s, %d step(s), single thread, %d host cores present" % (sample_desc, nst, os.cpu_count())}

    if rank == 0:
        out = {
            "metric": METRIC if prec == 64 else METRIC.replace("fp64", "fp32"), "value": value, "unit": UNIT,
            "n_gpus": world, "steps": K, "warmup": Wm, "ms_per_step": ms / K, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64" if prec == 64 else "f32", "data": "synthetic",
            "config": {"workload": w.name, "baseline_config": CONFIG_OF[args.workload], "cells": ncell,
                       "state_bytes": 5 * ncell * es, "l2": "inputs larger than L2" if 5 * ncell * es > 4 * 126e6
                       else "working set fits L2: launch/latency-bound, HBM fraction not meaningful",
                       "parallelism": "replicas x%d" % world if world > 1 else "1 GPU, whole mesh resident in HBM",
                       "launch": "one CUDA graph replay per step"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
            "step_roofline": step_roofline, "kernels": kernels, "cpu_baseline": cpu,
        }
        print(json.dumps(out))
    g.close()
    if world > 1:
        dist.destroy_process_group()


def run_local_slabs(args):
    """Cost of the Y-slab decomposition on ONE device: the same workload as N slabs, halos
    passed buffer to buffer, dt reduced over the slabs, plain launches (no graph), against nothing but itself --
    compare with the default line of the same workload.  Device-resident, CUDA events on the slabs' stream."""
    import torch
    from paper_1602_02359_b200.slabs import SlabRun
    torch.cuda.set_device(0)
    w, _, _ = make_workload(args.workload)
    s = SlabRun(w.mesh, w.geometry, w.eos, w.params, nslabs=args.local_slabs, precision=32 if args.fp32 else 64)
    s.set_fields(*w.fields())
    K, Wm = args.steps, max(args.warmup, 3)
    s.step(Wm)
    s.synchronize()
    l0 = sum(c.kernel_launches() for c in s.ctx.values())
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(s.stream)
    s.step(K)
    e1.record(s.stream)
    s.synchronize()
    ms = e0.elapsed_time(e1)
    halo = sum(2 * (c.halo_bytes(0, 1) + c.halo_bytes(1, 1)) * len([p for p in (c.mesh_bc_y) if p == 3]) for c in s.ctx.values())
    print(json.dumps({
        "metric": METRIC, "value": w.mesh.ncells * K / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": K, "warmup": Wm,
        "ms_per_step": ms / K, "higher_is_better": True, "dtype": "f32" if args.fp32 else "f64", "data": "synthetic",
        "config": {"workload": w.name, "local_slabs": args.local_slabs, "rows": [list(r) for r in s.rows.values()],
                   "launch": "plain launches, five phases per update and slab, halos device to device on one stream",
                   "halo_bytes_copied_per_update": halo},
        "gpu_launches": sum(c.kernel_launches() for c in s.ctx.values()) - l0}))


def run_dist_slabs(args):
    """NEXT-3 over torch.distributed (NCCL): ONE mesh split into one Y-slab per rank, halos by batch_isend_irecv, dt by
    all_reduce(MIN) on the device.  Strong scaling (the total work is fixed).  Opt-in (--slabs): the contract line stays
    the replica run, because this box has one GPU and the NCCL transport has only been run at world size 1 on it
    (the routing itself is covered by the gloo tests at world size 2 and 3)."""
    import torch
    import torch.distributed as dist
    from paper_1602_02359_b200.slabs import SlabRun
    rank, world, local = (int(os.environ.get(k, d)) for k, d in (("RANK", "0"), ("WORLD_SIZE", "1"), ("LOCAL_RANK", "0")))
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1"); os.environ.setdefault("MASTER_PORT", "29517")
    os.environ.setdefault("RANK", "0"); os.environ.setdefault("WORLD_SIZE", "1")
    torch.cuda.set_device(local)
    dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    w, _, _ = make_workload(args.workload)
    s = SlabRun(w.mesh, w.geometry, w.eos, w.params, group=dist.group.WORLD, precision=32 if args.fp32 else 64)
    s.set_fields(*w.fields())
    K, Wm = args.steps, max(args.warmup, 3)
    s.step(Wm)
    s.synchronize()
    rank_barrier(world)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(s.stream)
    s.step(K)
    e1.record(s.stream)
    s.synchronize()
    rank_barrier(world)
    ms = rank_max(e0.elapsed_time(e1), world, "cuda")
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": w.mesh.ncells * K / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K,
            "warmup": Wm, "ms_per_step": ms / K, "higher_is_better": True, "scaling": "strong",
            "dtype": "f32" if args.fp32 else "f64", "data": "synthetic",
            "config": {"workload": w.name, "parallelism": "%d Y-slabs, one per GPU, NCCL halos + all_reduce(MIN) of dt" % world,
                       "rows_of_rank0": list(s.rows[0])}}))
    dist.destroy_process_group()


def self_launch(n: int, argv, backend_env=None) -> int:
    """`python bench.py --gpus N` started without torchrun: start N ranks of this same command line under
    torch.distributed.run on this node (one process per GPU) and pass their exit code on."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(n), "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + list(argv)
    env = dict(os.environ)
    env.update(backend_env or {})
    return subprocess.call(cmd, env=env)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="noise512", choices=sorted(CONFIG_OF))
    ap.add_argument("--fp32", action="store_true", help="the optional fp32 build (config 5)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer region (short runs under ncu)")
    ap.add_argument("--slabs", action="store_true",
                    help="NEXT-3, under torchrun: one mesh split into one Y-slab per rank over NCCL (strong scaling) "
                         "instead of independent replicas")
    ap.add_argument("--local-slabs", type=int, default=0,
                    help="NEXT-3: advance the workload as N Y-slabs on THIS GPU (slabs.SlabRun, local transport) and "
                         "print what the decomposition costs on one device; not the contract line")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.local_slabs == 0:
        sys.exit(self_launch(args.gpus, sys.argv[1:]))
    if args.impl == "reference":
        run_reference(args)
    elif args.local_slabs > 0:
        run_local_slabs(args)
    elif args.slabs:
        run_dist_slabs(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
