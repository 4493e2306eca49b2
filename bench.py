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

# ncu --set full captures of the dominant kernels (dram__bytes_read.sum + dram__bytes_write.sum per launch) live
# under profiles/ and are named here; `roofline.traffic` carries a number only when bench.py is pointed at one that
# was taken on the same workload and commit (it is a profiler measurement, never re-measured inside a timed run).
TRAFFIC_PROFILES = {"ka8000": "profiles/r02_persist_c1_ncu.md", "lj1m": "profiles/r02_persist_lj1m_ncu.md",
                    "ka65536": "profiles/r02_ka65536_ncu.md", "ka1000": "profiles/r02_persist_ka1000_ncu.md",
                    "charged": "profiles/r02_charged_ncu.md"}

# The paper's parameter file (P:382 step 8): tunings found by rumd_autotune on "NVIDIA B200", keyed by GPU name, N,
# box, potentials, integrator; a hit costs no trial run, a miss tunes and appends.
TUNING_CACHE = os.path.join(ROOT, "paper_1506_05094_b200", "tuning_b200.jsonl")

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
    s.build_nblist()          # a fresh list of the current positions (the one in flight is a few steps old)
    s.compute_forces()
    cnt, _ = s.export_nblist()
    if none:
        s.set_tuning(method=rumd.NB_NONE)
        s.compute_forces()
    return int(cnt.sum())


def equilibrate(s, wl, steps):
    """Untimed: leave the lattice start (hot transient, frequent rebuilds; SURVEY 8(d) C2 note).  A block that
    overflowed the list ran with truncated rows (missing forces): it is repeated from the state held before it.
    That state is kept in the System's pinned host buffers, because the in-workspace snapshot does not survive
    the re-bind that doubles the capacity."""
    done = 0
    while done < steps:
        n = min(500, steps - done)
        s.download_state(s.h_r, s.h_v, None, None, s.h_image, s.h_id)
        s.run_steps(n)
        th = s.get_thermo(grow=True)
        if th is None:       # list overflow -> workspace re-bound with doubled capacity: redo the block
            s.upload_state()
            continue
        done += n


def roofline_of(s, wl, name, tun, ms_per_timestep, inner, peaks, fp32_measured, sm_mhz):
    """Roofline entries of one workload: the stand-alone pair-force kernel (timed alone: rumd_time_force replays
    200 launches from a graph between two CUDA events on the library's stream) and the whole time step.
    achieved = algorithmic flop (42 / 50 per LISTED pair) x live listed pairs / duration."""
    N = wl.N
    listed = count_listed(s)
    us = s.time_force(reps=200 if N < 500000 else 50)
    coul = bool((wl.pot[..., 4] > 0).any())
    flop_pp = FLOP_PER_LISTED_PAIR_COUL if coul else FLOP_PER_LISTED_PAIR_LJ
    flop = flop_pp * listed
    peak_tf = fp32_peak_tflops(peaks["sm_max_mhz"])
    ach_force = flop / (us * 1e-6) / 1e12
    ach_step = flop / (ms_per_timestep * 1e-3) / 1e12
    alg_bytes = 4.0 * listed + (16 + 4 + 20) * N
    return {
        "listed_pairs": listed, "mean_nbrs": listed / N, "flop_per_listed_pair": flop_pp,
        "force_kernel": {"kernel": "k_force (stand-alone, current tuning)", "us_per_launch": us,
                         "achieved": ach_force, "unit": "TFLOP/s", "frac": ach_force / peak_tf,
                         "frac_of_measured_fp32": ach_force / fp32_measured if fp32_measured else None,
                         "hbm_equiv_gbs": alg_bytes / (us * 1e-6) / 1e9,
                         "hbm_frac": alg_bytes / (us * 1e-6) / 1e9 / peaks["hbm_gbs"]},
        "whole_step": {"us_per_timestep": ms_per_timestep * 1e3, "achieved": ach_step, "frac": ach_step / peak_tf,
                       "frac_of_measured_fp32": ach_step / fp32_measured if fp32_measured else None,
                       "frac_at_observed_clock": ach_step / fp32_peak_tflops(sm_mhz)},
        "algorithmic_bytes_per_timestep": alg_bytes,
    }


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
    if args.set_tuning:
        kv = dict(item.split("=") for item in args.set_tuning.split(","))
        s.set_tuning(**{k: (float(v) if k == "skin" else int(v)) for k, v in kv.items()})
        tune_info = {"autotuned": False, "tuning_fixed_by": "--set-tuning " + args.set_tuning}
    elif args.autotune:
        t, tps = s.autotune(steps_per_trial=args.tune_steps, cache_path=TUNING_CACHE if args.tuning_cache else None)
        tune_info = {"autotuned": True, "tuning_from_cache": bool(s.tuning_from_cache), "trial_tps": tps}
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
    # the equilibrated state the timed region ran on, in ORIGINAL particle order: input of the cpu_baseline leg
    eq_state = s.state() if rank == 0 else None
    eq_thermo = th1

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
        peaks = measured_peaks()
        fp32_measured = s.measure_fp32_peak(5)
        sm_mhz = clocks.get("sm_mhz") or peaks["sm_max_mhz"]
        peak_tf = fp32_peak_tflops(peaks["sm_max_mhz"])
        rl = roofline_of(s, wl, args.workload, tun, ms / tsteps, inner, peaks, fp32_measured, sm_mhz)
        if tun["persistent"]:
            # the dominant kernel IS the whole run: one k_persist launch = `inner` time steps; its duration is the
            # CUDA-event time of the timed region itself
            us_launch = 1e3 * ms / args.steps
            phases = s.profile_persistent(inner)
            roof = {"kernel": "k_persist (one launch = %d time steps: rebuilds + forces + integration)" % inner,
                    "bound": "alu", "achieved": rl["whole_step"]["achieved"], "peak": peak_tf, "unit": "TFLOP/s",
                    "frac": rl["whole_step"]["frac"], "us_per_launch": us_launch, "phases_us_per_timestep": phases,
                    "algorithmic_bytes": rl["algorithmic_bytes_per_timestep"] * inner}
        else:
            fk = rl["force_kernel"]
            roof = {"kernel": "k_force", "bound": "alu", "achieved": fk["achieved"], "peak": peak_tf,
                    "unit": "TFLOP/s", "frac": fk["frac"], "us_per_launch": fk["us_per_launch"],
                    "force_share_of_step": fk["us_per_launch"] * 1e-3 / (ms / tsteps)}
        roof.update({
            "traffic": None,
            "traffic_source": "ncu --set full capture (dram__bytes_read.sum + dram__bytes_write.sum): %s" %
                              TRAFFIC_PROFILES.get(args.workload, "none for this workload"),
            "peak_source": "derived: 148 SMs x 128 FP32 lanes x 2 x %.0f MHz (max SM clock, %s)" % (
                peaks["sm_max_mhz"], peaks["source"]),
            "peak_measured_ffma": fp32_measured,
            "frac_of_measured_fp32": roof["achieved"] / fp32_measured if fp32_measured else None,
            "frac_at_observed_clock": roof["achieved"] / fp32_peak_tflops(sm_mhz),
            "regime": "N = %d: %s" % (N, "latency / dependency chain (SURVEY 8(d)): no throughput roofline applies; "
                                      "see sweep[] for N >= 65536" if N < 30000 else "FP32 ALU"),
            "listed_pairs": rl["listed_pairs"], "flop_per_listed_pair": rl["flop_per_listed_pair"],
            "force_kernel": rl["force_kernel"], "hbm_peak_gbs": peaks["hbm_gbs"]})
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
                       "mean_nbrs": rl["mean_nbrs"],
                       "nvt_note": "Nose-Hoover discretisation and tau = 0.2 are readings (the paper prints "
                                   "neither, P:54, P:78): NVT parity against the paper is unpinned"},
            "clocks": clocks,
            "e2e": {"value": e2e_tps, "unit": "timesteps/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
            "gpu_launches": int(l1 - l0),
            "roofline": roof,
            "thermo": {k: th1[k] for k in ("U", "K", "H", "xi")},
        }
        out["_eq_state"] = (eq_state, eq_thermo)
        out["_headline_row"] = sweep_row(args.workload, N, tps, ms / tsteps, tun, rl, th1["n_rebuilds"] - th0["n_rebuilds"],
                                         tsteps, tune_info)
        if tun["persistent"]:
            add_phases(out["_headline_row"], phases, rl, peaks, args.phases)
    s.close()
    return out


def add_phases(row, phases, rl, peaks, keep_all):
    """In-kernel phase timers of k_persist (block 0's SM-cycle counters, rumd_profile_persistent), per time step: the
    force + integrate phase is the production path's pair-force work (no energies, warm L2, no launch), so its
    fraction of the FP32 peak is reported beside the stand-alone kernel's."""
    us = phases["force_integrate_us"]
    ach = rl["flop_per_listed_pair"] * rl["listed_pairs"] / (us * 1e-6) / 1e12
    row.update({"force_phase_us": us, "force_phase_frac_fp32": ach / fp32_peak_tflops(peaks["sm_max_mhz"]),
                "rebuild_us_per_timestep": phases["rebuild_us"], "barrier_us_per_timestep": phases["barrier_us"]})
    if keep_all:
        row["phases_us_per_timestep"] = phases


def sweep_row(name, N, tps, ms_per_timestep, tun, rl, rebuilds, tsteps, info):
    fk, ws = rl["force_kernel"], rl["whole_step"]
    return {"workload": name, "N": N, "timesteps_per_s": tps, "particle_steps_per_s": tps * N,
            "us_per_timestep": 1e3 * ms_per_timestep,
            "tuning": {k: tun[k] for k in ("method", "tp", "skin", "build_tp", "persistent", "tile")},
            "tuning_from_cache": info.get("tuning_from_cache"),
            "rebuild_interval": tsteps / max(1, rebuilds), "mean_nbrs": rl["mean_nbrs"],
            "k_force_us": fk["us_per_launch"], "k_force_frac_fp32": fk["frac"],
            "k_force_frac_of_measured_fp32": fk["frac_of_measured_fp32"], "k_force_hbm_frac": fk["hbm_frac"],
            "whole_step_frac_fp32": ws["frac"], "whole_step_frac_of_measured_fp32": ws["frac_of_measured_fp32"]}


# ------------------------------------------------------------------------------------------------ N sweep

# BASELINE.json metric "timesteps/s and particle-steps/s vs N; % FP32/HBM roofline": rows emitted by the DEFAULT run
# beside the configs[1] headline (which is itself the N = 8000 row).  --sweep-all adds every size of configs[0..4].
SWEEP_DEFAULT = ["ka1000", "ka65536", "ka131072", "charged", "lj1m"]
SWEEP_ALL = ["lj864", "ka512", "ka1000", "ka2048", "ka4096", "ka8192", "ka16384", "ka32768", "ka65536", "ka131072",
             "charged", "lj1m"]


def run_sweep(args, names, fp32_measured):
    """Device-resident arm only, one row per workload: equilibrated, tuned (tuning file first), timed with
    CUDA events on the library's stream, then the stand-alone force kernel and the roofline fractions."""
    import torch

    from paper_1506_05094_b200 import rumd

    peaks = measured_peaks()
    out = []
    for name in names:
        t_row = time.perf_counter()
        wl, desc = make_workload(name)
        s = rumd.from_workload(wl)
        N = wl.N
        equilibrate(s, wl, args.equil if N < 500000 else 500)
        info = {}
        if args.autotune:
            t, tps_trial = s.autotune(steps_per_trial=args.tune_steps if N < 500000 else 60,
                                      cache_path=TUNING_CACHE if args.tuning_cache else None)
            info = {"tuning_from_cache": bool(s.tuning_from_cache), "trial_tps": tps_trial}
        inner = max(50, min(args.inner, int(2e8 / N)))
        for _ in range(3):
            s.run_steps(inner)
        th0 = s.get_thermo()
        reps = 5
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
        with torch.cuda.stream(s.stream):
            for a, b in ev:
                a.record(s.stream)
                s.run_steps(inner)
                b.record(s.stream)
        torch.cuda.synchronize()
        ms = sum(a.elapsed_time(b) for a, b in ev)
        th1 = s.get_thermo()
        tps = reps * inner / (ms * 1e-3)
        tun = s.get_tuning().as_dict()
        rl = roofline_of(s, wl, name, tun, ms / (reps * inner), inner, peaks, fp32_measured, peaks["sm_max_mhz"])
        row = sweep_row(name, N, tps, ms / (reps * inner), tun, rl, th1["n_rebuilds"] - th0["n_rebuilds"], reps * inner, info)
        if tun["persistent"]:
            add_phases(row, s.profile_persistent(inner), rl, peaks, args.phases)
        row["wall_s"] = time.perf_counter() - t_row
        out.append(row)
        print("sweep %s: %.0f timesteps/s, k_force %.1f us = %.3f of FP32" % (name, tps, row["k_force_us"],
                                                                              row["k_force_frac_fp32"]),
              file=sys.stderr, flush=True)
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


def cpu_model() -> str:
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_sample(wl, nsteps, state=None, threads=None):
    """Time the fp64 oracle, as it stands, for nsteps whole time steps of this workload on the host cores.
    state: (r, v, image, xi, eta) to start from (fp32-representable values); default the workload's t = 0."""
    import oracle

    if threads is not None:
        oracle.set_num_threads(threads)
    r, v, image, xi, eta = state if state is not None else (wl.r, wl.v, np.zeros((wl.N, 3), np.int32), 0.0, 0.0)
    t0 = time.perf_counter()
    o = oracle.run(np.asarray(r, np.float64), np.asarray(v, np.float64), wl.m.astype(np.float64),
                   np.asarray(image, np.int32), wl.types, wl.box.astype(np.float64), wl.pot, float(wl.skin),
                   float(wl.dt), int(nsteps), mode=wl.integrator, T0=wl.T0, tau=wl.tau, xi=xi, eta=eta,
                   use_cell=wl.N >= 4096, want_log=False)
    dt_ = time.perf_counter() - t0
    return nsteps / dt_, dt_, o, oracle.num_threads()


def cpu_baseline(wl, state, target_s=12.0, one_core_s=5.0):
    """The oracle on the SAME equilibrated state the GPU arm was timed on (downloaded, original particle order),
    all host cores, plus a 1-core figure."""
    import oracle

    all_cores = oracle.num_threads()
    oracle_sample(wl, 2, state)                       # first call: library load, thread pool
    tps0, _, _, cores = oracle_sample(wl, 24, state)
    n = int(max(8, min(20000, target_s * tps0)))
    tps, dt_, o, cores = oracle_sample(wl, n, state)
    oracle.set_num_threads(1)
    tps1_0, _, _, _ = oracle_sample(wl, 2, state)
    n1 = int(max(2, min(5000, one_core_s * tps1_0)))
    tps1, dt1, _, _ = oracle_sample(wl, n1, state)
    oracle.set_num_threads(all_cores)
    return {"value": tps, "unit": "timesteps/s", "cores": cores, "kind": "oracle", "cpu_model": cpu_model(),
            "one_core": {"value": tps1, "unit": "timesteps/s", "cores": 1,
                         "sample": "%d time steps, %.1f s" % (n1, dt1)},
            "same_state_as_gpu_arm": True,
            "sample": "%d time steps of the same workload from the equilibrated state the GPU arm was timed on "
                      "(%d list builds), %.1f s, fp64, skin %.2f, OpenMP over particles" % (n, o["n_builds"], dt_,
                                                                                           float(wl.skin))}


def run_reference(args, rank, world):
    """--impl reference: the oracle on the host cores, same config/metric.  Like the GPU arm it first leaves the
    lattice start (args.equil untimed steps, run by the oracle itself: nothing of the CUDA path is on this arm),
    then each bench step is a bounded sample (inner_ref time steps) continuing from that state."""
    if rank != 0:
        return None
    wl, desc = make_workload(args.workload)
    tps0, _, _, cores = oracle_sample(wl, 2)
    equil = int(min(args.equil, max(0, 45.0 * tps0)))          # bounded: at most ~45 s of equilibration
    st = None
    if equil > 0:
        _, _, o, _ = oracle_sample(wl, equil)
        st = (o["r"], o["v"], o["image"], o["xi"], o["eta"])
    tps0, _, _, cores = oracle_sample(wl, 2, st)
    # timed part (warmup + steps) bounded to ~60 s
    inner_ref = int(max(1, min(args.inner, 60.0 * tps0 / max(1, args.steps + args.warmup))))
    times = []
    nb = 0
    for it in range(args.warmup + args.steps):
        tps, dt_, o, cores = oracle_sample(wl, inner_ref, st)
        st = (o["r"], o["v"], o["image"], o["xi"], o["eta"])
        if it >= args.warmup:
            times.append(dt_)
            nb += o["n_builds"]
    total = sum(times)
    val = args.steps * inner_ref / total
    sample = ("%d bench steps x %d time steps, continuing from the state after %d untimed equilibration steps of "
              "the oracle (%d list builds in the timed part)" % (args.steps, inner_ref, equil, nb))
    return {"impl": "reference", "metric": "timesteps/s", "value": val, "unit": "timesteps/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "particle_steps_per_s": val * wl.N,
            "config": {"workload": desc, "N": wl.N, "md_timesteps_per_step": inner_ref, "equilibration_steps": equil},
            "cpu_baseline": {"value": val, "unit": "timesteps/s", "cores": cores, "kind": "oracle",
                             "cpu_model": cpu_model(), "sample": sample},
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
    ap.add_argument("--no-tuning-cache", dest="tuning_cache", action="store_false",
                    help="tune from scratch instead of reading / appending paper_1506_05094_b200/tuning_b200.jsonl")
    ap.add_argument("--tune-steps", type=int, default=300)
    ap.add_argument("--set-tuning", default=None, metavar="K=V,...",
                    help="fix the headline workload's tuning instead of autotuning it, e.g. method=3,tile=6,tp=1,pb=256,skin=0.25")
    ap.add_argument("--no-cpu-baseline", dest="cpu", action="store_false")
    ap.add_argument("--no-sweep", dest="sweep_default", action="store_false",
                    help="skip the N sweep rows of the default run")
    ap.add_argument("--sweep", nargs="*", default=None, metavar="WORKLOAD",
                    help="sweep these workloads (no names: every size of configs[0..4]) instead of the default rows")
    ap.add_argument("--phases", action="store_true", help="add in-kernel phase timings to the sweep rows")
    ap.add_argument("--ensembles", action="store_true", help="also time the batched ensembles")
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
        eq_state, eq_thermo = out.pop("_eq_state")
        headline_row = out.pop("_headline_row")
        if args.cpu and world == 1:
            wl, _ = make_workload(args.workload)
            st = (eq_state["r"], eq_state["v"], eq_state["image"], eq_thermo["xi"], eq_thermo["eta"])
            out["cpu_baseline"] = cpu_baseline(wl, st)
        else:
            out["cpu_baseline"] = None
        if world == 1 and (args.sweep is not None or args.sweep_default):
            names = SWEEP_DEFAULT if args.sweep is None else (args.sweep or SWEEP_ALL)
            rows = run_sweep(args, [n for n in names if n != args.workload], out["roofline"]["peak_measured_ffma"])
            out["sweep"] = sorted(rows + [headline_row], key=lambda r: (r["N"], r["workload"]))
            if args.ensembles:
                out["ensembles"] = run_ensembles(args, ENSEMBLES)
        print(json.dumps(out), flush=True)
    if world > 1:
        torch.distributed.barrier()
        torch.distributed.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
