#!/usr/bin/env python
"""bench.py -- timesteps/s of the RUMD hot path on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--inner M] [--workload ka8000|lj864|lj1m|charged|kaNNNN]
                    [--sweep] [--impl reference]

A bench "step" is a block of M (= --inner, default 1000) consecutive MD time steps issued by ONE
rumd_run_steps call; every MD time step is one pass of the whole hot path (rebuild decision, list build when
needed, pair forces, integrate + wrap).  value = MD time steps per second (whole job: sum over ranks; each
rank runs its own replica: replicas only).  See DESIGN.md "Measurement".
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_1506_05094_b200 import workloads as W  # noqa: E402

SM_COUNT = 148
FP32_LANES_PER_SM = 128


def make_workload(name: str):
    if name == "ka8000":
        return W.ka_lattice(8000), "configs[1]: Kob-Andersen 80:20 LJ, N=8000, density 1.2, NVT T=0.8, dt=0.0025"
    if name == "lj864":
        return W.lj_fcc(6), "configs[0]: LJ fcc N=864, density 0.8442, NVE dt=0.005"
    if name == "lj1m":
        return W.lj_fcc(64), "configs[3]: LJ fcc N=1048576, density 0.8442, NVE dt=0.005"
    if name == "charged":
        return W.charged_sc(32), "configs[4]: charged LJ N=32768, density 0.5, SF Coulomb rc=4, NVT T=1, dt=0.002"
    if name.startswith("ka"):
        n = int(name[2:])
        return W.ka_lattice(n), "configs[2]: Kob-Andersen sweep, N=%d, density 1.2, NVT T=0.8" % n
    raise SystemExit("unknown workload " + name)


# ------------------------------------------------------------------------------------------------ clocks


class ClockSampler:
    """nvidia-smi clock / throttle-reason samples DURING the timed region (B200_PROFILING.md clocks line)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def mark(self) -> int:
        return len(self.lines)

    def stop(self, first: int = 0) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        lines = self.lines[first:] or self.lines[-1:]
        for ln in lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                smax.append(float(f[1]))
                pw.append(float(f[2]))
            except ValueError:
                continue
            for k, nm in enumerate(names):
                if f[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------ peaks


def measured_peaks() -> dict:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


def fp32_peak_tflops(sm_mhz: float) -> float:
    """FP32 FMA peak derived from unit counts and clock: 148 SMs x 128 lanes x 2 flop x f."""
    return SM_COUNT * FP32_LANES_PER_SM * 2 * sm_mhz * 1e6 / 1e12


# ------------------------------------------------------------------------------------------------ ranks


def max_over_ranks(value: float, world: int, device="cpu") -> float:
    """Max of a per-rank scalar over all ranks (torch.distributed must be initialised when world > 1)."""
    if world <= 1:
        return float(value)
    import torch

    t = torch.tensor([value], dtype=torch.float64, device=device)
    torch.distributed.all_reduce(t, op=torch.distributed.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank: float, seconds_local: float, world: int, device="cpu") -> float:
    """Replicas only: every rank processes units_per_rank; the job's rate is the units all
    ranks processed divided by the slowest rank's time."""
    return world * units_per_rank / max_over_ranks(seconds_local, world, device)


# ------------------------------------------------------------------------------------------------ GPU arm

# DRAM bytes (read + write) per MD time step of the dominant kernel, from the committed ncu --set full captures
# (profiles/r01_persist_c1_ncu.md: 4.70 MB per 200-step k_persist launch at C1; profiles/r01_force_lj1m_ncu.md:
# 376.8 MB per k_force launch at C3).  Workloads without a capture report traffic = null.
NCU_DRAM_BYTES_PER_TIMESTEP = {"ka8000": 4.70e6 / 200, "lj1m": 376.8e6}

FLOP_PER_LISTED_PAIR_LJ = 42.0       # SURVEY.md 8(d) / DESIGN.md "Roofline": 21 always + 30 x 0.712 inside rc
FLOP_PER_LISTED_PAIR_COUL = 50.0     # + the Coulomb term


def count_listed(s):
    """Listed pairs of the current state (the unit of the flop convention).  With the "none" method there is no
    list: the count is taken from a list built once with the N^2 method at the same skin."""
    from paper_1506_05094_b200 import rumd

    t = s.get_tuning()
    none = t.method == rumd.NB_NONE
    if none:
        s.set_tuning(method=rumd.NB_N2)
    s.compute_forces()
    cnt, _ = s.export_nblist()
    if none:
        s.set_tuning(method=rumd.NB_NONE)
        s.compute_forces()
    return int(cnt.sum())


def equilibrate(s, wl, steps):
    """Untimed: leave the lattice start (hot transient, frequent rebuilds; SURVEY 8(d) C2 note)."""
    done = 0
    while done < steps:
        n = min(500, steps - done)
        s.run_steps(n)
        th = s.get_thermo(grow=True)
        if th is None:       # list overflow -> capacity doubled; repeat from the last good state
            continue
        done += n


def run_gpu(args, rank, world, local_rank):
    import torch

    from paper_1506_05094_b200 import rumd

    torch.cuda.set_device(local_rank)
    dev = "cuda:%d" % local_rank
    wl, desc = make_workload(args.workload)
    s = rumd.from_workload(wl, device=dev)
    N = wl.N
    inner = args.inner
    equilibrate(s, wl, args.equil)
    tune_info = {}
    if args.autotune:
        t, tps = s.autotune(steps_per_trial=args.tune_steps)
        tune_info = {"autotuned": True, "trial_tps": tps}
    tun = s.get_tuning().as_dict()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    # ---- device-resident arm: inputs already in HBM, K blocks of `inner` time steps
    sampler = ClockSampler(local_rank)
    sampler.start()
    for _ in range(args.warmup):
        s.run_steps(inner)
    th0 = s.get_thermo()
    stream = s.stream
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    l0 = s.launch_count()
    barrier()
    mark = sampler.mark()
    with torch.cuda.stream(stream):
        for a, b in ev:
            flush.fill_(1)                   # L2 flush between timed iterations (same stream, not timed)
            a.record(stream)
            s.run_steps(inner)
            b.record(stream)
    barrier()
    clocks = sampler.stop(mark)
    l1 = s.launch_count()
    ms = sum(a.elapsed_time(b) for a, b in ev)
    th1 = s.get_thermo()
    ms = max_over_ranks(ms, world, dev)
    tsteps = args.steps * inner
    tps = world * tsteps / (ms * 1e-3)

    # ---- end-to-end arm: host buffers through the C ABI, H2D + D2H inside the timed region
    h_r = torch.empty((N, 4), dtype=torch.float32).pin_memory()
    h_v = torch.empty((N, 4), dtype=torch.float32).pin_memory()
    h_f = torch.empty((N, 4), dtype=torch.float32).pin_memory()
    h_w = torch.empty((N,), dtype=torch.float32).pin_memory()
    h_im = torch.empty((N, 4), dtype=torch.int32).pin_memory()
    h_id = torch.empty((N,), dtype=torch.int32).pin_memory()
    s.download_state(h_r, h_v, None, None, h_im, h_id)
    s.h_r.copy_(h_r), s.h_v.copy_(h_v), s.h_image.copy_(h_im), s.h_id.copy_(h_id)
    h2d = (16 + 16 + 16 + 4) * N
    d2h = (16 + 16 + 16 + 4 + 16 + 4) * N + 120
    e2e_times = []
    for it in range(args.warmup + args.steps):
        barrier()
        t0 = time.perf_counter()
        s.upload_state()                                  # H2D of r, v, image, id (pinned host memory)
        s.run_steps(inner)
        s.download_state(h_r, h_v, h_f, h_w, h_im, h_id)  # D2H of the whole state + forces; synchronizes
        th = s.get_thermo()                               # D2H of the thermo scalars
        dt_ = time.perf_counter() - t0
        s.h_r.copy_(h_r), s.h_v.copy_(h_v), s.h_image.copy_(h_im), s.h_id.copy_(h_id)
        if it >= args.warmup:
            e2e_times.append(dt_)
    e2e_tps = whole_job_rate(tsteps, sum(e2e_times), world, dev)

    out = None
    if rank == 0:
        # ---- roofline of the dominant kernel (pair force), timed live with CUDA events on the library's stream
        listed = count_listed(s)
        us = s.time_force(reps=200)
        coul = bool((wl.pot[..., 4] > 0).any())
        flop = (FLOP_PER_LISTED_PAIR_COUL if coul else FLOP_PER_LISTED_PAIR_LJ) * listed
        peaks = measured_peaks()
        sm_mhz = clocks.get("sm_mhz") or peaks["sm_max_mhz"]
        peak_tf = fp32_peak_tflops(peaks["sm_max_mhz"])
        ach_tf = flop / (us * 1e-6) / 1e12
        alg_bytes = 4.0 * listed + (16 + 4 + 20) * N
        s.profile_step()          # first call pays CUDA's lazy loading of the un-fused kernels
        prof = s.profile_step()
        flop_pp = flop / listed
        force_kernel = {"kernel": "k_force (stand-alone, current tuning)", "us_per_launch": us, "achieved": ach_tf,
                        "frac": ach_tf / peak_tf, "hbm_equiv_gbs": alg_bytes / (us * 1e-6) / 1e9,
                        "hbm_peak_gbs": peaks["hbm_gbs"], "unfused_step_ms": prof}
        if tun["persistent"]:
            # the dominant kernel IS the whole run: one k_persist launch = `inner` time steps; its duration is the
            # CUDA-event time of the timed region itself
            us_launch = 1e3 * ms / args.steps
            ach = flop * inner / (us_launch * 1e-6) / 1e12
            phases = s.profile_persistent(inner)
            roof = {"kernel": "k_persist (one launch = %d time steps: rebuilds + forces + integration)" % inner,
                    "bound": "alu", "achieved": ach, "peak": peak_tf, "unit": "TFLOP/s", "frac": ach / peak_tf,
                    "traffic": (NCU_DRAM_BYTES_PER_TIMESTEP[args.workload] * inner
                                if args.workload in NCU_DRAM_BYTES_PER_TIMESTEP else None),
                    "traffic_source": "ncu dram__bytes_read.sum + dram__bytes_write.sum, profiles/r01_*_ncu.md",
                    "algorithmic_bytes": alg_bytes * inner,
                    "us_per_launch": us_launch, "phases_us_per_timestep": phases}
        else:
            roof = {"kernel": "k_force", "bound": "alu", "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s",
                    "frac": ach_tf / peak_tf, "traffic": None, "us_per_launch": us,
                    "force_share_of_step": us * 1e-3 / (ms / tsteps)}
        roof.update({"peak_source": "derived: 148 SMs x 128 FP32 lanes x 2 x %.0f MHz (max SM clock, %s)" % (
                         peaks["sm_max_mhz"], peaks["source"]),
                     "frac_at_observed_clock": roof["achieved"] / fp32_peak_tflops(sm_mhz),
                     "listed_pairs": listed, "flop_per_listed_pair": flop_pp, "force_kernel": force_kernel})
        out = {
            "metric": "timesteps/s", "value": tps, "unit": "timesteps/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "particle_steps_per_s": tps * N, "us_per_timestep": 1e3 * ms / tsteps,
            "config": {"workload": desc, "N": N, "md_timesteps_per_step": inner, "equilibration_steps": args.equil,
                       "tuning": tun, **tune_info,
                       "l2": "256 MiB L2 flush between timed iterations (outside the event pairs)",
                       "parallelism": "replicas x%d" % world,
                       "rebuilds_in_window": th1["n_rebuilds"] - th0["n_rebuilds"], "max_nbrs": th1["max_nbrs"],
                       "mean_nbrs": listed / N},
            "clocks": clocks,
            "e2e": {"value": e2e_tps, "unit": "timesteps/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
            "gpu_launches": int(l1 - l0),
            "roofline": roof,
            "thermo": {k: th1[k] for k in ("U", "K", "H", "xi")},
        }
    s.close()
    return out


# ------------------------------------------------------------------------------------------------ N sweep

SWEEP = ["lj864", "ka512", "ka1000", "ka2048", "ka4096", "ka8000", "ka8192", "ka16384", "ka32768", "ka65536",
         "ka131072", "charged", "lj1m"]


def run_sweep(args, names):
    """BASELINE.json metric "timesteps/s and particle-steps/s vs N": device-resident arm only, one entry per
    workload, each autotuned (configs[2]) after equilibration.  Not part of the default run."""
    import torch

    from paper_1506_05094_b200 import rumd

    peaks = measured_peaks()
    peak_tf = fp32_peak_tflops(peaks["sm_max_mhz"])
    out = []
    for name in names:
        wl, desc = make_workload(name)
        s = rumd.from_workload(wl)
        N = wl.N
        equilibrate(s, wl, args.equil if N < 500000 else 500)
        info = {}
        if args.autotune:
            t, tps_trial = s.autotune(steps_per_trial=args.tune_steps if N < 500000 else 60)
            info["trial_tps"] = tps_trial
        inner = max(50, min(args.inner, int(2e8 / N)))
        for _ in range(3):
            s.run_steps(inner)
        th0 = s.get_thermo()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(5)]
        with torch.cuda.stream(s.stream):
            for a, b in ev:
                a.record(s.stream)
                s.run_steps(inner)
                b.record(s.stream)
        torch.cuda.synchronize()
        ms = sum(a.elapsed_time(b) for a, b in ev)
        th1 = s.get_thermo()
        tps = 5 * inner / (ms * 1e-3)
        listed = count_listed(s)
        us = s.time_force(reps=50)
        coul = bool((wl.pot[..., 4] > 0).any())
        flop = (FLOP_PER_LISTED_PAIR_COUL if coul else FLOP_PER_LISTED_PAIR_LJ) * listed
        tun = s.get_tuning().as_dict()
        phases = s.profile_persistent(inner) if tun["persistent"] else None
        out.append({"workload": name, "N": N, "timesteps_per_s": tps, "particle_steps_per_s": tps * N,
                    "us_per_timestep": 1e3 * ms / (5 * inner), "tuning": tun, **info,
                    "rebuild_interval": 5 * inner / max(1, th1["n_rebuilds"] - th0["n_rebuilds"]),
                    "mean_nbrs": listed / N, "whole_step_frac_fp32": flop / (1e-3 * ms / (5 * inner)) / 1e12 / peak_tf,
                    "force_kernel_us": us, "force_kernel_frac_fp32": flop / (us * 1e-6) / 1e12 / peak_tf,
                    "phases_us_per_timestep": phases})
        print("sweep %s: %.0f timesteps/s" % (name, tps), file=sys.stderr, flush=True)
        s.close()
    return out


# ------------------------------------------------------------------------------------------------ ensembles

ENSEMBLES = [("ka512", 444), ("ka1000", 444), ("ka2048", 444)]


def run_ensembles(args, specs):
    """SURVEY 8(f)-2 / P:63: R independent replicas of a small system advanced by one launch (one thread block per
    replica).  Reports replica-time-steps per second (R x steps / time) and particle-steps per second."""
    import torch

    from paper_1506_05094_b200 import rumd

    out = []
    for name, R in specs:
        wl, desc = make_workload(name)
        v = np.stack([W.maxwell_boltzmann(np.random.default_rng(W.SEED0 + 7000 + q), wl.m.astype(np.float64),
                                          float(wl.T0)).astype(np.float32) for q in range(R)])
        best = None
        for tp in (2, 4, 8):
            s = rumd.System(np.stack([wl.r] * R), v, wl.m, wl.types, wl.box, wl.pot, skin_for_capacity=0.6)
            s.set_integrator(wl.integrator, wl.dt, wl.T0, wl.tau)
            s.set_tuning(method=rumd.NB_N2, tp=tp, pb=256 // tp, skin=0.45)
            s.run_steps(args.equil)
            s.get_thermo_replicas()
            n = max(200, min(2000, int(4e8 / (R * wl.N))))
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(s.stream)
            s.run_steps(n)
            b.record(s.stream)
            torch.cuda.synchronize()
            ms = a.elapsed_time(b)
            s.get_thermo_replicas()
            rate = R * n / (ms * 1e-3)
            if best is None or rate > best["replica_timesteps_per_s"]:
                best = {"workload": name, "N": wl.N, "replicas": R, "tp": tp, "replica_timesteps_per_s": rate,
                        "particle_steps_per_s": rate * wl.N, "us_per_batch_step": 1e3 * ms / n}
            s.close()
        out.append(best)
        print("ensemble %s x%d: %.0f replica-timesteps/s" % (name, R, best["replica_timesteps_per_s"]), file=sys.stderr,
              flush=True)
    return out


# ------------------------------------------------------------------------------------------------ oracle arm


def oracle_sample(wl, nsteps):
    """Time the fp64 oracle, as it stands, for nsteps whole time steps of this workload on the host cores."""
    import oracle

    t0 = time.perf_counter()
    o = oracle.run(wl.r.astype(np.float64), wl.v.astype(np.float64), wl.m.astype(np.float64),
                   np.zeros((wl.N, 3), np.int32), wl.types, wl.box.astype(np.float64), wl.pot, float(wl.skin),
                   float(wl.dt), int(nsteps), mode=wl.integrator, T0=wl.T0, tau=wl.tau, use_cell=wl.N >= 4096,
                   want_log=False)
    dt_ = time.perf_counter() - t0
    return nsteps / dt_, dt_, o["n_builds"], oracle.num_threads()


def cpu_baseline(wl, target_s=12.0):
    tps0, dt0, _, cores = oracle_sample(wl, 4)
    n = int(max(8, min(20000, target_s * tps0)))
    tps, dt_, nb, cores = oracle_sample(wl, n)
    return {"value": tps, "unit": "timesteps/s", "cores": cores, "kind": "oracle",
            "sample": "%d time steps of the same workload from its t=0 state (%d list builds), %.1f s, fp64, "
                      "OpenMP over particles" % (n, nb, dt_)}


def run_reference(args, rank, world):
    """--impl reference: the oracle on the host cores, same config/metric; each bench step is a bounded
    sample (inner_ref time steps)."""
    if rank != 0:
        return None
    wl, desc = make_workload(args.workload)
    tps0, _, _, cores = oracle_sample(wl, 2)
    # whole run (warmup + steps) bounded to ~60 s
    inner_ref = int(max(1, min(args.inner, 60.0 * tps0 / max(1, args.steps + args.warmup))))
    times = []
    nb = 0
    for it in range(args.warmup + args.steps):
        tps, dt_, b, cores = oracle_sample(wl, inner_ref)
        if it >= args.warmup:
            times.append(dt_)
            nb += b
    total = sum(times)
    val = args.steps * inner_ref / total
    sample = "%d bench steps x %d time steps of the workload from t=0 (%d list builds)" % (args.steps, inner_ref, nb)
    return {"impl": "reference", "metric": "timesteps/s", "value": val, "unit": "timesteps/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "particle_steps_per_s": val * wl.N,
            "config": {"workload": desc, "N": wl.N, "md_timesteps_per_step": inner_ref},
            "cpu_baseline": {"value": val, "unit": "timesteps/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "timesteps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


# ------------------------------------------------------------------------------------------------ main


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--inner", type=int, default=1000, help="MD time steps per bench step")
    ap.add_argument("--equil", type=int, default=2000, help="untimed equilibration steps (configs[1])")
    ap.add_argument("--workload", default="ka8000")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-autotune", dest="autotune", action="store_false")
    ap.add_argument("--tune-steps", type=int, default=300)
    ap.add_argument("--no-cpu-baseline", dest="cpu", action="store_false")
    ap.add_argument("--sweep", nargs="*", default=None, metavar="WORKLOAD",
                    help="also time the N sweep (all of configs[0..4] when no names are given) -> key 'sweep'")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        out = run_reference(args, rank, world)
        if out is not None:
            print(json.dumps(out), flush=True)
        return 0

    import torch

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; librumd_b200 has no CPU fallback")
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        torch.cuda.set_device(local_rank)
        torch.distributed.init_process_group("nccl", device_id=torch.device("cuda:%d" % local_rank))
    out = run_gpu(args, rank, world, local_rank)
    if rank == 0:
        if args.cpu and world == 1:
            wl, _ = make_workload(args.workload)
            out["cpu_baseline"] = cpu_baseline(wl)
        else:
            out["cpu_baseline"] = None
        if args.sweep is not None and world == 1:
            out["sweep"] = run_sweep(args, args.sweep or SWEEP)
            if not args.sweep:
                out["ensembles"] = run_ensembles(args, ENSEMBLES)
        print(json.dumps(out), flush=True)
    if world > 1:
        torch.distributed.barrier()
        torch.distributed.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
