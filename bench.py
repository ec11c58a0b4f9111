#!/usr/bin/env python
"""bench.py -- particle-turns/s and turns/min of the space-charge tracking hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W]            # our CUDA path (libsc_track)
    python bench.py --impl reference [--steps K] [--warmup W]      # the CPU oracle, as it stands

A "step" is one whole turn: every table row of BASELINE.json configs[2] (1e6 macroparticles, 6D
Gaussian bunch, 2377 rows = 216 segments of ~10 elements + one RF kick, a space-charge node with a
128x128 grid and a 256-bin line-density histogram at every segment end).  Inputs are seeded and
synthetic (workloads/); they stand in for the J-PARC MR lattice of the paper, which is not
available.  Prints ONE JSON line (rank 0).  For N > 1 (torchrun, one rank per GPU) every rank tracks
its own bunch (the MR holds 8) -- replicas, no data-path collective, weak scaling.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "particle_turns_per_s"
UNIT = "particle-turns/s"
NAMES = ("x", "px", "y", "py", "sigma", "psigma")


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cfg", type=int, default=3, help="BASELINE.json config number (3 = headline)")
    ap.add_argument("--particles", type=int, default=0, help="override the config's particle count")
    ap.add_argument("--grid", type=int, default=0, help="override the grid size (cfg 4 sweep)")
    ap.add_argument("--deposit", default="fixed", choices=["fixed", "f64"])
    ap.add_argument("--boundary", default="open", choices=["open", "pipe"],
                    help="open: Hockney free-space solve (headline); pipe: the paper's conducting-pipe solver, eqs. 15-27")
    ap.add_argument("--interp", default="bilinear", choices=["bilinear", "bicubic"],
                    help="bilinear: gather of the node field (headline); bicubic: the paper's Bezier surface of the potential, eqs. 28-29")
    ap.add_argument("--chromatic", action="store_true",
                    help="track the thick quadrupoles by eq. 6 per particle (SC_CQUAD rows) instead of the on-momentum matrix")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-sample-particles", type=int, default=1_000_000)
    ap.add_argument("--ref-sample-particles", type=int, default=0,
                    help="--impl reference: macroparticles per step (0 = the config's own count: the same workload)")
    ap.add_argument("--hbm-particles", type=int, default=10_000_000,
                    help="second roofline leg (roofline_hbm): the same lattice and beam recipe with this many macroparticles, "
                         "streaming from HBM; 0 to skip")
    return ap.parse_args()


def workload_name(wl, args):
    g = wl.grids[0]
    return (f"cfg{args.cfg}: {wl.n} macroparticles ({'6D' if wl.particles['sigma'] is not None else '4D'}), "
            f"{wl.n_rows} table rows/turn, {wl.n_sc} SC nodes/turn, {g['nx']}x{g['ny']} grid, "
            f"{g['nbins']}-bin lambda histogram")


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_traffic():
    """(dram__bytes_read.sum + dram__bytes_write.sum per k_push launch, source file) from the committed summary of the
    latest `ncu --set full` capture of THIS round's build (profiles/r02*_k_push_full.md: a line
    `dram_bytes_per_launch: <bytes>`; cold caches, ncu flushes L2 between replays), or (None, why)."""
    import glob
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "r02*_k_push_full.md")), reverse=True):
        try:
            with open(path) as f:
                for line in f:
                    if line.startswith("dram_bytes_per_launch:"):
                        return float(line.split(":")[1].split()[0]), os.path.relpath(path, ROOT)
        except Exception:
            continue
    return None, "no ncu --set full summary of this build under profiles/"


BASE_SEED = {1: 1, 2: 2, 3: 3, 4: 3, 5: 5}


def rank_seed(cfg: int, rank: int):
    """Replicas: every rank tracks its own bunch -- rank 0 the config's seed, rank r that seed + 1000 r."""
    return BASE_SEED[cfg] + 1000 * rank if rank else None


def max_over_ranks(value: float, world: int, device) -> float:
    """The slowest rank's time (device-timed milliseconds): what the whole job waited for."""
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_rate(n_per_rank: int, steps: int, world: int, ms_max: float) -> float:
    """Whole-job particle-turns/s: the units all ranks processed over the slowest rank's time."""
    return world * n_per_rank * steps / (ms_max * 1e-3)


class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap,power.draw"

    def __init__(self, index: int):
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(index)], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except Exception:
            self.proc.kill()
            out = ""
        sm, mx, reasons, pw = [], [], set(), []
        for line in out.strip().splitlines():
            f = [t.strip() for t in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[6]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm), "power_w_max": max(pw) if pw else None}


def cpu_oracle_rate(args, n: int, deposit_mode: int, turns: int = 1):
    """The oracle as it stands (single thread), one bounded sample of the same workload."""
    from oracle import ref as orc
    from workloads import make_config
    wl = apply_variants(make_config(args.cfg, n=n, grid_n=args.grid or None, deposit_mode=deposit_mode), args)
    orc.lib()
    t0 = time.perf_counter()
    orc.track_workload(wl, n_turns=turns)
    dt = time.perf_counter() - t0
    return wl.n * turns / dt, dt, wl


def config_dict(wl, args, world: int):
    """The `config` object of the JSON line: what both arms run (the reference arm the same workload on the host)."""
    g = wl.grids[0]
    mode = 1 if args.deposit == "fixed" else 0
    return {"workload": workload_name(wl, args),
            "deposit": f"{args.deposit}" + (f" (int64, s={g['fixed_bits']})" if mode else " (fp64 atomics)"),
            "poisson": "open boundary (Hockney)" if args.boundary == "open" else "conducting pipe (eqs. 15-27)",
            "quadrupoles": "eq. 6 per particle (chromatic)" if args.chromatic else "on-momentum matrix",
            "interpolation": "bicubic potential, eqs. 28-29" if args.interp == "bicubic" else "bilinear field gather",
            "parallelism": "replicas" if world > 1 else "single GPU"}


def apply_variants(wl, args):
    """--boundary / --interp / --chromatic act on the workload description, identically for both arms."""
    for g in wl.grids:
        g["boundary"] = 1 if args.boundary == "pipe" else 0
        g["interp"] = 1 if args.interp == "bicubic" else 0
    if args.chromatic:
        from workloads import CQUAD, QUAD
        wl.kind = wl.kind.copy()
        wl.kind[wl.kind == QUAD] = CQUAD
    return wl


def run_reference(args):
    """--impl reference: the oracle (plain single-threaded C, oracle/) on the host cores, as it stands; each step is one
    turn of the SAME workload (all of the config's macroparticles unless --ref-sample-particles bounds the sample)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import ref as orc
    from workloads import make_config
    mode = 1 if args.deposit == "fixed" else 0
    n_full = args.particles or {1: 10_000, 2: 100_000, 3: 1_000_000, 4: 1_000_000, 5: 10_000_000}[args.cfg]
    wl = apply_variants(make_config(args.cfg, n=args.ref_sample_particles or n_full, grid_n=args.grid or None, deposit_mode=mode), args)
    p = wl.particles
    for _ in range(args.warmup):
        p, _w = orc.track(wl.kind, wl.ipar, wl.par, wl.grids, wl.beam, p, n_turns=1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        p, _w = orc.track(wl.kind, wl.ipar, wl.par, wl.grids, wl.beam, p, n_turns=1)
    dt = time.perf_counter() - t0
    value = wl.n * args.steps / dt
    sample = (f"{wl.n} of {n_full} macroparticles, same lattice/grid/histogram, {args.steps} turns after {args.warmup} warm-up turns, "
              f"1 thread (host has {os.cpu_count()} logical cores)")
    cfg = config_dict(wl, args, 1)
    if wl.n != n_full:
        cfg["workload"] = cfg["workload"].replace(f"{wl.n} macroparticles", f"{n_full} macroparticles")
        cfg["sample"] = sample
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "turns_per_min": 60.0 * args.steps / dt * (wl.n / n_full),
        "config": cfg,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def push_bytes_per_launch(ncoord: int, n: int, n_push: int, n_psigma_stores: int) -> float:
    """Mean bytes one k_push launch of a turn must move (8 B per coordinate read and per coordinate
    written): all ncoord coordinates are read; all are written back except psigma (6D) on the launches without an RF
    row or a longitudinal kick, which cannot change it (k_push.cuh skips that store)."""
    reads = ncoord * n_push
    writes = ncoord * n_push if ncoord == 4 else 5 * n_push + n_psigma_stores
    return 8.0 * n * (reads + writes) / max(n_push, 1)


def solve_floor_us(nx: int, ny: int, pass_gbs: float) -> dict:
    """Work count of one open-boundary field solve from SURVEY.md 8(d), row "Poisson P+F": flops of the forward and inverse
    transforms on the doubled grid, and four passes (each a read and a write) over the nx x (ny+1) complex half spectrum,
    charged at pass_gbs (the measured copy bandwidth: the passes run out of the L2, which is no slower)."""
    import math
    flop = 2.0 * (nx * 2.5 * 2 * ny * math.log2(2 * ny) + (ny + 1) * 5.0 * 2 * nx * math.log2(2 * nx))
    pass_bytes = 4.0 * 2 * nx * (ny + 1) * 16
    t_flop, t_pass = flop / 37e12 * 1e6, pass_bytes / (pass_gbs * 1e9) * 1e6
    return {"flop": flop, "pass_bytes": pass_bytes, "floor_us": max(t_flop, t_pass), "floor_flop_us": t_flop, "floor_pass_us": t_pass}


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2010_11540_b200 as sc
    from workloads import make_config

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the CUDA path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    mode = 1 if args.deposit == "fixed" else 0
    # every rank tracks its own bunch: same lattice, its own seed (replicas only)
    wl = apply_variants(make_config(args.cfg, n=args.particles or None, grid_n=args.grid or None, deposit_mode=mode,
                                    seed=rank_seed(args.cfg, rank)), args)
    sixd = wl.particles["sigma"] is not None
    ncoord = 6 if sixd else 4
    t = sc.Tracker.from_workload(wl)
    # pinned host copies of the inputs (for the end-to-end leg) and device-resident ones
    host = {k: (None if wl.particles[k] is None else torch.from_numpy(wl.particles[k]).pin_memory()) for k in NAMES}
    host_np = {k: (None if v is None else v.numpy()) for k, v in host.items()}
    t.sc_load_particles(host_np)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    flush_buf = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")

    def flush_l2():
        with torch.cuda.stream(t.stream):
            flush_buf.zero_()

    # ---------------- device-resident throughput: W warm-up turns, then exactly K timed turns
    for _ in range(max(args.warmup, 0)):
        t.sc_track(1)
    barrier()
    clocks = ClockSampler(local)
    l0 = t.sc_kernel_launches()
    evs = []
    barrier()
    for _ in range(args.steps):
        flush_l2()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(t.stream)
        t.sc_track(1)
        e1.record(t.stream)
        evs.append((e0, e1))
    barrier()
    launches = t.sc_kernel_launches() - l0
    ms = sum(a.elapsed_time(b) for a, b in evs)
    clk = clocks.stop()
    ms_max = max_over_ranks(ms, world, "cuda")
    value = aggregate_rate(wl.n, args.steps, world, ms_max)

    # ---------------- roofline of the dominant kernel (k_push) and where a node's time goes
    # sc_profile_replay: one turn's launches captured into a CUDA graph in four modes (whole turn / k_push launches only /
    # field-solve launches only / every kernel empty) and replayed back to back between ONE CUDA-event pair on the
    # tracker's stream: kernel durations as they are inside the timed turns, free of launch latency.
    reps = 5
    rp = {name: t.sc_profile_replay(mode, reps) for name, mode in
          (("turn", sc.SC_REPLAY_TURN), ("push", sc.SC_REPLAY_PUSH), ("poisson", sc.SC_REPLAY_POISSON), ("empty", sc.SC_REPLAY_EMPTY))}
    n_push = rp["push"]["n_kernels"]
    nodes = max(rp["turn"]["n_nodes"], 1)
    push_ms = rp["push"]["turn_ms"] / n_push
    cp = t.sc_profile_copy(reps)
    prof = [t.sc_profile_turn() for _ in range(3)][1:]
    push_ms_pairs = statistics.mean(p["push_ms"] / p["n_push"] for p in prof)
    pois_ms = statistics.mean(p["poisson_ms"] / max(p["n_poisson"], 1) for p in prof)
    # bytes a k_push launch must move: every coordinate read, every coordinate written back except psigma on the launches
    # that cannot change it (6D: no RF row and no longitudinal kick in the launch; sc_profile_replay counts the others)
    n_ps = rp["push"]["n_psigma_stores"]
    bytes_per_launch = push_bytes_per_launch(ncoord, wl.n, n_push, n_ps)
    peak, peak_src = measured_peak()
    achieved = bytes_per_launch / (push_ms * 1e-3) / 1e9
    # the plain copy kernel moves read + write of every coordinate: scale its time to the bytes a k_push launch moves
    copy_like_ms = cp["copy_ms"] * bytes_per_launch / cp["bytes"]
    turn_ms = ms_max / args.steps
    turn_bytes = n_push * bytes_per_launch
    g0 = wl.grids[0]
    solve_floor = solve_floor_us(g0["nx"], g0["ny"], peak)
    traffic, traffic_src = ncu_traffic()
    mom_after = t.sc_moments()
    split = {"unit": "us per SC node, inside a CUDA graph", "turn": 1e3 * rp["turn"]["turn_ms"] / nodes,
             "push_only": 1e3 * rp["push"]["turn_ms"] / nodes, "poisson_only": 1e3 * rp["poisson"]["turn_ms"] / nodes,
             "empty_kernels": 1e3 * rp["empty"]["turn_ms"] / nodes,
             "kernels_per_turn": rp["turn"]["n_kernels"], "k_push_launches_per_turn": n_push, "nodes_per_turn": nodes,
             "n_outside_per_deposit_push_replay": rp["push"]["n_outside"], "n_outside_last_node_tracked": float(mom_after[31]),
             "note": "poisson_only and empty_kernels still launch the turn's k_push kernels as no-ops (wait for the predecessor, "
                     "return); push_only launches no field-solve kernels, its kicks read the last solved fields"}
    roofline = {"bound": "hbm", "regime": "L2-resident, latency-limited" if 8 * ncoord * wl.n < 100e6 else "streams from HBM",
                "kernel": "k_push (kick + segment maps + deposit)", "achieved": achieved, "peak": peak,
                "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
                "limiter": "latency: at 1e6 macroparticles the 48 MB particle set is L2-resident, achieved is an EFFECTIVE bandwidth "
                           "(algorithmic bytes / time), not DRAM utilisation; roofline_hbm below is the streaming (HBM-bound) point",
                "traffic": traffic, "traffic_source": traffic_src,
                "algorithmic_bytes_per_launch": bytes_per_launch, "avg_launch_ms": push_ms,
                "bytes_accounting": f"8 B x n x ({ncoord} reads + {ncoord} writes), minus the psigma store on the "
                                    f"{n_push - n_ps} of {n_push} launches per turn that cannot change psigma; mean over the turn's launches",
                "launches_per_turn": n_push, "launches_per_turn_storing_psigma": n_ps,
                "push_share_of_turn": n_push * push_ms / turn_ms,
                "copy_kernel_ms": cp["copy_ms"], "copy_kernel_bytes": cp["bytes"],
                "frac_of_copy_kernel": copy_like_ms / push_ms,
                "avg_launch_ms_event_pairs": push_ms_pairs, "frac_event_pairs": bytes_per_launch / (push_ms_pairs * 1e-3) / 1e9 / peak,
                "poisson_group_ms_event_pairs": pois_ms,
                "split": split,
                "how": "sc_profile_replay(SC_REPLAY_PUSH): the k_push launches of one turn (same arguments and particle count) replayed "
                       "back to back from a CUDA graph, 5 replays between one CUDA-event pair on the tracker's stream; copy_kernel_ms: a plain "
                       "copy of the same arrays (sc_profile_copy); the *_event_pairs figures put an event pair around every plain launch "
                       "instead (launch latency included)"}
    roofline_hbm = None
    if args.hbm_particles > 0 and rank == 0 and args.cfg in (3, 4):
        # the streaming point: the same lattice and beam recipe with 1e7 macroparticles (480 MB, far beyond L2)
        wl2 = apply_variants(make_config(args.cfg, n=args.hbm_particles, grid_n=args.grid or None, deposit_mode=mode), args)
        t2 = sc.Tracker.from_workload(wl2)
        t2.sc_load_particles(wl2.particles)
        t2.sc_track(1)
        r2 = t2.sc_profile_replay(sc.SC_REPLAY_PUSH, 2)
        rt2 = t2.sc_profile_replay(sc.SC_REPLAY_TURN, 2)
        c2 = t2.sc_profile_copy(5)
        l2 = r2["turn_ms"] / r2["n_kernels"]
        b2 = push_bytes_per_launch(ncoord, wl2.n, r2["n_kernels"], r2["n_psigma_stores"])
        roofline_hbm = {"bound": "hbm", "kernel": "k_push", "workload": f"{workload_name(wl2, args)} (streams from HBM)",
                        "achieved": b2 / (l2 * 1e-3) / 1e9, "peak": peak, "unit": "GB/s", "frac": b2 / (l2 * 1e-3) / 1e9 / peak,
                        "avg_launch_ms": l2, "algorithmic_bytes_per_launch": b2, "copy_kernel_ms": c2["copy_ms"],
                        "copy_kernel_frac_of_peak": c2["bytes"] / (c2["copy_ms"] * 1e-3) / 1e9 / peak,
                        "frac_of_copy_kernel": c2["copy_ms"] * b2 / c2["bytes"] / l2, "turn_ms": rt2["turn_ms"],
                        "roofline_turn_frac": r2["n_kernels"] * b2 / (rt2["turn_ms"] * 1e-3) / 1e9 / peak,
                        "particle_turns_per_s": wl2.n / (rt2["turn_ms"] * 1e-3)}
        t2.close()
        del t2

    # ---------------- end to end through the C ABI with HOST buffers (pinned): load -> 1 turn -> moments
    e2e_steps = max(3, min(args.steps, 10))
    for _ in range(2):
        t.sc_load_particles(host_np); t.sc_track(1); t.sc_moments()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        t.sc_load_particles(host_np)
        t.sc_track(1)
        mom = t.sc_moments()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_max = max_over_ranks(e2e_s, world, "cuda")
    e2e = {"value": world * wl.n * e2e_steps / e2e_max, "unit": UNIT, "h2d_bytes_per_step": 8 * ncoord * wl.n,
           "d2h_bytes_per_step": 8 * sc.SC_N_MOMENTS + 64, "steps": e2e_steps,
           "what": "per step: sc_load_particles(pinned host arrays) + sc_track(1) + sc_moments() read back"}

    # the other end-to-end shape: the caller wants the PARTICLES back, not only their moments (48 MB D2H per step at cfg3)
    import ctypes as C
    back = {k: (None if host[k] is None else torch.empty_like(host[k]).pin_memory()) for k in NAMES}
    back_ptrs = [C.c_void_p(0 if back[k] is None else back[k].data_ptr()) for k in NAMES]

    def step_with_particles_back():
        t.sc_load_particles(host_np)
        t.sc_track(1)
        rc = t.lib.sc_get_particles(t.h, *back_ptrs, 0)        # synchronises; pinned host destinations
        if rc:
            raise RuntimeError("sc_get_particles failed: %d" % rc)

    step_with_particles_back()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        step_with_particles_back()
    torch.cuda.synchronize()
    e2e_p_max = max_over_ranks(time.perf_counter() - t0, world, "cuda")
    e2e["particles_back"] = {"value": world * wl.n * e2e_steps / e2e_p_max, "unit": UNIT, "h2d_bytes_per_step": 8 * ncoord * wl.n,
                             "d2h_bytes_per_step": 8 * ncoord * wl.n, "steps": e2e_steps,
                             "what": "per step: sc_load_particles(pinned host arrays) + sc_track(1) + sc_get_particles into pinned host arrays"}

    line = None
    if rank == 0:
        g = wl.grids[0]
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "turns_per_min": 60.0 * args.steps / (ms_max * 1e-3),
            "config": {**config_dict(wl, args, world),
                       "l2": "256 MiB written between timed steps (L2 flushed); within a turn the 48 MB particle set is re-read 217x",
                       "emittance_x_after": float(mom[28]),
                       "n_outside_last_node_after_timed_turns": float(mom_after[31]), "non_finite_after_timed_turns": float(mom_after[32])},
            "clocks": clk, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "roofline_hbm": roofline_hbm,
            "frac_of_copy_kernel": roofline["frac_of_copy_kernel"],
            "roofline_turn": {"bound": "hbm", "what": "every k_push launch of a turn (the bytes all of them must move) over the whole timed turn, "
                                                      "field solves and graph overhead included",
                              "achieved": turn_bytes / (turn_ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                              "frac": turn_bytes / (turn_ms * 1e-3) / 1e9 / peak, "bytes_per_turn": turn_bytes, "ms_per_turn": turn_ms},
            "roofline_solve": {"bound": "latency/L2 (no roofline stage, SURVEY.md 8(d) row Poisson P+F)", "kernel": "field solve (1 or 3 launches per node)",
                               "us_per_node": split["poisson_only"], "floor_us": solve_floor["floor_us"], "frac": solve_floor["floor_us"] / split["poisson_only"],
                               **solve_floor,
                               "note": "us_per_node is the solve-only graph replay (it also carries the empty k_push launches of the turn); the floor "
                                       "is the larger of the fp64 work at the nominal 37 TFLOP/s and four read+write passes over the Hermitian half spectrum "
                                       "at the measured copy bandwidth, both with all 148 SMs busy; dependent stages, barriers and launch latency are "
                                       "not in it, and they are what bounds a 128 x 128 solve"},
        }
    t.close()
    if world > 1:
        dist.destroy_process_group()
    return line


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    line = run_ours(args)
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    if args.gpus == 1 and not args.no_cpu_baseline:
        mode = 1 if args.deposit == "fixed" else 0
        n = min(args.cpu_sample_particles, args.particles or 10 ** 9)
        rate, dt, swl = cpu_oracle_rate(args, n, mode)
        line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"1 turn of the same workload with {swl.n} macroparticles ({dt:.1f} s, single thread; "
                                          f"host has {os.cpu_count()} logical cores)"}
    print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
