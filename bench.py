#!/usr/bin/env python
"""bench.py -- throughput of the fused split-step Schroedinger-Poisson step on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload t512|cfg2|cfg3|cfg4|cfg5] [--impl reference]

One "step" is one kick-drift-kick step of the whole hot path (all rows of SURVEY.md 8(a)).  The timed
region is ONE wdm_step(K, dt) call (the user's call) bracketed by CUDA events on the context's stream,
after W warm-up steps.  Default workload: T512 = 512^3 complex64 soliton + 65536-mode halo, the
configuration BASELINE.json's north_star quotes its HBM-roofline target on (psi alone is 1.07 GB, 8x the
126 MB L2, so no L2 flush is needed between steps).  Prints ONE JSON line (rank 0).

Multi-GPU: the path does not shard: --gpus N runs N independent replicas, one process
per GPU under torchrun, no data-path collective; value = all ranks' cells / max-over-ranks time.

--impl reference times the CPU oracle (oracle/, as it stands) on the host cores on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import wdm_workloads as wl  # noqa: E402

METRIC = "SPE grid cell-updates/sec per KDK step"
UNIT = "cell-updates/s"

# algorithmic HBM bytes per cell per launch of each kernel, in units of the complex size c (DESIGN.md
# "Kernels": one read + one write of the field per axis sweep; reals are c/2)
ALG_BYTES_PER_CELL_C = {
    "psi_sweep_z_kick": 2.5, "psi_sweep_y": 2.0, "psi_sweep_x_rho_r2c": 2.5,
    "poisson_y_fwd": 1.0, "poisson_z_green": 1.0, "poisson_y_inv": 1.0, "poisson_x_c2r": 1.0,
}
# The CPU oracle is timed on ONE sample, in the reference arm and in the cpu_baseline leg alike: the soliton + halo
# recipe of the bench workload at 256^3 (float64, 0.3 s per KDK step on 16 host cores; 512^3 would need 6.5 GB and
# 3 s per step).
REF_SAMPLE_N = 256
# algorithmic HBM bytes per particle of the particle kernels (pos, vel read + write in the push,
# pos read in the deposit; the gathered Phi nodes and the deposited rho_p nodes go through L2)
PARTICLE_BYTES = {"particle_gather_kick_drift": 48, "particle_cic_deposit": 12}


def make_workload(name: str):
    if name == "t512":
        return wl.t512()
    if name == "cfg2":
        return wl.config2()
    if name == "cfg3":
        return wl.config3()
    if name == "cfg4":
        return wl.config4()
    if name == "cfg5":
        return wl.config5()
    if name.startswith("sample"):          # soliton + halo at a reduced grid (reference arm / cpu_baseline)
        n = int(name[6:])
        w = wl.config2(N=n, nmodes=4096 if n < 512 else 65536, name=f"sample{n}_c64_soliton_halo", seed=4)
        w.dt = (w.L / n) ** 2 / 6.0
        return w
    raise SystemExit(f"unknown workload {name}")


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """Polls SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._t = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {
            nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
            nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
            nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake",
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, nm in names.items():
                    if r & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(0.01)

    def __enter__(self):
        if self.nv:
            self._t = threading.Thread(target=self._run, daemon=True)
            self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._t:
            self._t.join()

    def summary(self):
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def max_over_ranks(x: float, dist, device) -> float:
    """MAX all-reduce of a per-rank scalar (the only collective of the bench: timing, never data)."""
    if dist is None:
        return x
    import torch
    t = torch.tensor([x], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(cells_per_rank: int, steps: int, world: int, ms_max: float) -> float:
    """whole-job throughput of `world` independent replicas: all ranks' cell updates / slowest rank's time"""
    return world * cells_per_rank * steps / (ms_max * 1e-3)


def oracle_rate(sample_name: str, steps: int, warmup: int):
    """cells/s of the CPU oracle on the named sample: `warmup` untimed then `steps` timed KDK steps."""
    import oracle
    w = make_workload(sample_name)
    o = oracle.Oracle(w.N, w.L, w.hbar_over_m, w.G)
    o.set_psi(w.psi)
    if w.pos is not None:
        o.set_particles(w.pos, w.vel, w.mass)
    dt = w.dt if w.dt is not None else (w.L / w.N) ** 2 / 6.0
    o.step(warmup, dt)                      # also pays the first potential refresh
    t0 = time.perf_counter()
    o.step(steps, dt)
    el = time.perf_counter() - t0
    return w, (w.N ** 3) * steps / el, el, oracle.threads()


def run_reference(args, rank, world):
    if rank != 0:
        return
    n_ref = REF_SAMPLE_N
    w, rate, el, thr = oracle_rate(f"sample{n_ref}", args.steps, args.warmup)
    sample = (f"float64 CPU oracle, soliton+halo workload at {n_ref}^3 instead of 512^3 "
              f"({args.steps} timed KDK steps, {el:.1f} s)")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * el / max(1, args.steps),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "t512_c64_soliton_halo", "sample": sample},
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": thr, "kind": "oracle", "sample": sample},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def run_dist(args, rank, world, local, dist, torch):
    """One box sharded over the ranks.  NOT the north_star path: a separate line, scaling "strong"."""
    import paper_2606_25026_b200.dist as wd
    K, W = args.steps, max(3, args.warmup)
    w = make_workload(args.workload)
    N, xl = w.N, w.N // world
    sim = wd.DistSim(N, w.L, w.hbar_over_m, w.G, w.dtype, rank, world)
    slab = torch.from_numpy(w.psi[rank * xl:(rank + 1) * xl])
    dt = w.dt if w.dt is not None else (w.L / N) ** 2 / 6.0

    def run(prog):
        if dist is not None:
            sim.run(prog)
        else:
            wd.run_emulated([sim], [prog])

    run(sim.prog_set_psi(slab))
    run(sim.prog_step(W, dt))
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
        torch.cuda.synchronize()
    stream = torch.cuda.current_stream()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clk:
        e0.record(stream)
        run(sim.prog_step(K, dt))
        e1.record(stream)
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()
    ms = max_over_ranks(e0.elapsed_time(e1), dist, "cuda")
    csize = 8 if w.dtype == "c64" else 16
    xbytes = (2 * xl * xl * N + 2 * xl * (-(-(N // 2 + 1) // world)) * N) * csize * (world - 1)     # sent per rank per step
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": N ** 3 * K / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": "f32" if w.dtype == "c64" else "f64", "data": "synthetic",
            "config": {"workload": w.name, "N": N, "mode": "slab-decomposed (wdm_dist.h), pure SPE",
                       "parallelism": f"x-slabs over {world} rank(s), 4 all-to-all exchanges per step",
                       "exchange": "NCCL all_to_all_single" if dist is not None else "local copy (single process)",
                       "exchange_bytes_sent_per_rank_per_step": xbytes,
                       "note": "with one rank the exchanges are local copies: this is the cost of the decomposition "
                               "machinery (pack / unpack passes), not a scaling measurement"},
            "gpu_launches": sim.launched_phases, "clocks": clk.summary()}))
    sim.close()


def coupled_record(wdm, torch, K, W):
    """cfg5: ONE wdm_step(K, dt) between CUDA events after W warm-up steps; cell- and particle-updates/s, per-kernel means."""
    w = wl.config5()
    N, npart = w.N, len(w.pos)
    sim = wdm.Sim(N, w.L, w.hbar_over_m, w.G, w.dtype, max_particles=npart)
    sim.set_psi(torch.from_numpy(w.psi).pin_memory())
    sim.set_particles(w.pos, w.vel, w.mass)
    sim.step(0, 0.0)
    dt = wl.cfl_dt(w, float(sim.potential().abs().max()))
    stream = torch.cuda.current_stream()
    sim.step(W, dt)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    sim.step(K, dt)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    wdm.wdm_set_profiling(sim.h, True)
    kp = min(K, 64)
    sim.step(kp, dt)
    stats = wdm.wdm_kernel_stats(sim.h)
    wdm.wdm_set_profiling(sim.h, False)
    sim.close()
    peak, _ = peaks()
    rec = {"workload": w.name, "N": N, "particles": npart, "steps": K, "ms_per_step": ms / K,
           "cell_updates_per_s": N ** 3 * K / (ms * 1e-3), "particle_updates_per_s": npart * K / (ms * 1e-3),
           "alg_bytes_per_step": 12 * 8 * N ** 3 + 60 * npart,
           "frac_of_hbm_peak": (12 * 8 * N ** 3 + 60 * npart) / (ms / K * 1e-3) / 1e9 / peak,
           "note": "12c per cell (rho_p cleared and read) + 60 B per particle, SURVEY 8(d); 256^3 sits near the 126 MB L2",
           "kernels_avg_ms": {k: t / c for k, (c, t) in stats.items() if c},
           "kernel_launches_per_step": {k: c / kp for k, (c, t) in stats.items() if c}}
    return rec


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="t512")
    ap.add_argument("--impl", default="wdm")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip e2e / per-kernel / particle legs (used under ncu)")
    ap.add_argument("--dist", action="store_true",
                    help="slab-decomposed step (include/wdm_dist.h): ONE box sharded over the ranks, NCCL all-to-all "
                         "between phases (strong scaling); with one rank the exchange is a local copy")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import paper_2606_25026_b200 as wdm   # raises if libwdm.so is missing: there is no fallback

    torch.cuda.set_device(local)
    dist = None
    if world > 1 or (args.dist and "RANK" in os.environ):      # (--dist under torchrun: NCCL also with a single rank)
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if args.dist:
        run_dist(args, rank, world, local, dist, torch)
        if dist is not None:
            dist.destroy_process_group()
        return

    K, W = args.steps, max(3, args.warmup)
    w = make_workload(args.workload)
    N = w.N
    npart = 0 if w.pos is None else len(w.pos)
    sim = wdm.Sim(N, w.L, w.hbar_over_m, w.G, w.dtype, max_particles=npart)
    psi_host = torch.from_numpy(w.psi).pin_memory()
    sim.set_psi(psi_host)
    if npart:
        sim.set_particles(w.pos, w.vel, w.mass)
    dt = w.dt
    if dt is None:                                     # CFL from the initial potential (reading G17)
        sim.step(0, 0.0)
        dt = wl.cfl_dt(w, float(sim.potential().abs().max()))
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    # ---- warm-up, then the timed region: ONE wdm_step(K, dt)
    sim.step(W, dt)
    barrier()
    l0 = wdm.wdm_launch_count(sim.h)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clk:
        barrier()
        e0.record(stream)
        sim.step(K, dt)
        e1.record(stream)
        barrier()
    ms = e0.elapsed_time(e1)
    launches = wdm.wdm_launch_count(sim.h) - l0
    ms = max_over_ranks(ms, dist, "cuda")
    value = aggregate_value(N ** 3, K, world, ms)

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if w.dtype == "c64" else "f64", "data": "synthetic",
        "config": {"workload": w.name, "N": N, "grid_dtype": "complex64" if w.dtype == "c64" else "complex128",
                   "particles": npart, "dt": dt, "timed_call": f"wdm_step({K}, dt)",
                   "l2": "inputs larger than L2 (psi alone is %.2f GB vs 126 MB L2), no flush" % (N ** 3 * 8 / 1e9)
                         if N >= 512 else "working set near/below L2: L2-resident, launch-bound regime",
                   "parallelism": "replicas only (no sharding, no collective)" if world > 1 else "single GPU"},
        "gpu_launches": launches, "clocks": clk.summary(),
    }
    if npart:
        out["particle_updates_per_s"] = world * npart * K / (ms * 1e-3)

    if not args.no_extras:
        csize = 8 if w.dtype == "c64" else 16
        # ---- per-kernel CUDA-event timing on the context's stream (profiled pass, not the headline number)
        wdm.wdm_set_profiling(sim.h, True)
        kp = min(K, 20)
        sim.step(kp, dt)
        stats = wdm.wdm_kernel_stats(sim.h)
        wdm.wdm_set_profiling(sim.h, False)
        total_ms = sum(t for _, t in stats.values())
        kern = {k: {"launches": c, "avg_ms": t / c, "share": t / total_ms} for k, (c, t) in stats.items() if c}
        dom = max((k for k in kern if k in ALG_BYTES_PER_CELL_C), key=lambda k: kern[k]["launches"] * kern[k]["avg_ms"])
        peak, how = peaks()
        alg = ALG_BYTES_PER_CELL_C[dom] * csize * N ** 3
        achieved = alg / (kern[dom]["avg_ms"] * 1e-3) / 1e9
        traffic = None
        tp = os.path.join(ROOT, "profiles", "traffic.json")
        if os.path.exists(tp):
            traffic = json.load(open(tp)).get(w.name, {}).get(dom)
        out["roofline"] = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                           "frac": achieved / peak, "traffic": traffic, "peak_source": how,
                           "alg_bytes_per_launch": alg,
                           "whole_step": {"alg_bytes_per_step": 11 * csize * N ** 3,
                                          "achieved": 11 * csize * N ** 3 / (ms / K * 1e-3) / 1e9,
                                          "frac": 11 * csize * N ** 3 / (ms / K * 1e-3) / 1e9 / peak,
                                          "frac_of_nominal_8TBs": 11 * csize * N ** 3 / (ms / K * 1e-3) / 1e9 / 8000.0,
                                          "note": "11c per cell = SURVEY 8(d) count for the seven sweeps of a step"}}
        out["kernels"] = kern
        if npart:
            # particle kernels against their own HBM count; the rho_p clear (one real per cell, "particle_mesh_clear")
            # and rho_p's read inside the density sweep are per-cell costs of the coupled step (96 B/cell instead of 88)
            rsize = csize // 2
            pk = {}
            for name, b in PARTICLE_BYTES.items():
                if name in kern:
                    g = b * (rsize // 4) * npart / (kern[name]["avg_ms"] * 1e-3) / 1e9
                    pk[name] = {"avg_ms": kern[name]["avg_ms"], "launches_per_step": kern[name]["launches"] / kp,
                                "alg_bytes_per_particle": b * (rsize // 4), "achieved_GBs": g, "frac": g / peak}
            for name in ("particle_mesh_clear", "particle_cell_sort"):
                if name in kern:
                    pk[name] = {"avg_ms": kern[name]["avg_ms"], "launches_per_step": kern[name]["launches"] / kp}
            if "particle_mesh_clear" in pk:
                pk["particle_mesh_clear"]["note"] = "zeroes only the (y, 16 z-cell) columns the last deposit flagged"
            pk["ms_per_step_all_particle_kernels"] = sum(kern[k]["avg_ms"] * kern[k]["launches"] for k in kern if k.startswith("particle_")) / kp
            pk["share_of_step"] = sum(kern[k]["share"] for k in kern if k.startswith("particle_"))
            out["particles"] = pk

        # ---- end to end through the C ABI with HOST buffers: copy in + K steps + copy out, wall clock
        out_host = torch.empty_like(psi_host).pin_memory()
        ke = K
        barrier()
        t0 = time.perf_counter()
        wdm.wdm_run_host(sim.h, psi_host, ke, dt, out_host)     # synchronises before returning
        el = time.perf_counter() - t0
        el = max_over_ranks(el, dist, "cuda")
        nbytes = psi_host.numel() * psi_host.element_size()
        out["e2e"] = {"value": world * N ** 3 * ke / el, "unit": UNIT, "h2d_bytes_per_step": nbytes / ke,
                      "d2h_bytes_per_step": nbytes / ke, "call": f"wdm_run_host(psi_in, {ke}, dt, psi_out)",
                      "note": "state stays on the device between steps; one H2D of psi and one D2H per call"}

        # ---- CPU oracle on the host cores, bounded sample (rank 0, N = 1 only)
        if rank == 0 and world == 1 and not args.no_cpu_baseline:
            n_ref, CPU_STEPS = REF_SAMPLE_N, 40         # about 13 s on 16 host cores (bounded sample: 10-30 s of CPU work)
            ws, rate, el, thr = oracle_rate(f"sample{n_ref}", CPU_STEPS, 1)
            out["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": thr, "kind": "oracle",
                                   "sample": f"float64 CPU oracle, soliton+halo at {n_ref}^3, {CPU_STEPS} timed KDK steps ({el:.1f} s)"}
    sim.close()
    # ---- the coupled run of BASELINE.json's metric ("+ particle updates/s"): config 5 (256^3 complex64 soliton + halo,
    # 2^20 disc particles), same timing rules, as a sub-record of the default line (rank 0, N = 1)
    if rank == 0 and world == 1 and not args.no_extras and args.workload == "t512":
        del sim
        torch.cuda.empty_cache()
        out["coupled"] = coupled_record(wdm, torch, K, W)
    if rank == 0:
        print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
