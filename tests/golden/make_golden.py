#!/usr/bin/env python
"""Writes the stored expected values under tests/golden/ that are too slow to recompute inside the GPU test run.

    python tests/golden/make_golden.py long_cfg2 | long_cfg3 | long_cfg3_paper | cfg5_full | all | long_cfg2_twin | long_cfg3_twin | long_cfg3_paper_twin | cfg5_full_twin
    python tests/golden/make_golden.py long_cfg3_twins K      # one more member (K = 1, 2, ...) of long_cfg3's twin ensemble

It calls ONLY the oracle (oracle/) and the seeded input generators (workloads/); nothing here comes from the CUDA path.
Each output file records the command, the recipe and the oracle's wall time.

  long_cfg2  BASELINE.json configs[1] literally: 1e5 macroparticles (4D waterbag), 128x128, 100 turns, fp64 deposit.
             Stored: rms emittances every 10 turns, and mean / rms of the per-particle tunes of the first 4096
             particles (turn-averaged phase advance in Floquet-normalised coordinates).
  long_cfg3  configs[2] decimated to 1e5 macroparticles (bunch charge kept at 2e13: same space-charge regime),
             200 turns, fixed-point deposit (last paragraph).  Same statistics, three planes.
  long_cfg3_paper   the same 6D run (cfg3 lattice, RF, 256-bin line density, 1e5 macroparticles, 200 turns, fixed-point deposit)
             with the bunch charge lowered to 2.3e12: the paper's tune-shift regime (-0.3; PAPER.md:352-354
             prints -0.45), where the motion is regular and north_star's 1e-3 on the long-run statistics can hold.
             long_cfg3_paper_twin adds the run from initial coordinates moved by one unit in the last place: its deviation
             shows whether this regime is chaotic.
  cfg5_full  configs[4] at its full 1e7 macroparticles, one turn, fixed-point deposit, 256x256: the six coordinates of
             1024 sampled particles and the oracle's moments.
"""
import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

from oracle import ref as orc  # noqa: E402
from workloads import make_config  # noqa: E402
from workloads.configs import CFG3_TWISS  # noqa: E402

N_TAGGED = 4096


def tunes(q, p, beta, alpha):
    """q, p: [turns, particles] -> per-particle turn-averaged phase advance / 2 pi."""
    phi = np.arctan2(-(beta * p + alpha * q), q)
    d = np.mod(np.diff(phi, axis=0), 2 * np.pi)
    return d.mean(axis=0) / (2 * np.pi)


N_REAL_PAPER_REGIME = 2.3e12   # cfg3's bunch charge scaled to the paper's tune-shift regime (-0.3; -0.45)


def long_run(cfg, n, turns, mode, planes, name, twin=False, member=0, n_real=None):
    """twin=True: the same run from initial coordinates moved by one unit in the last place (random signs): how far the
    oracle's OWN statistics move under a rounding-level change -- the floor below which no two implementations of a
    chaotic system can be asked to agree (stored as "twin" next to the unperturbed run's values)."""
    wl = make_config(cfg, n=n, deposit_mode=mode)
    if n_real is not None:
        wl.beam["n_real"] = float(n_real)
    p = {k: (None if v is None else v.copy()) for k, v in wl.particles.items()}
    if twin:
        rng = np.random.Generator(np.random.PCG64(77 + 1000 * member))   # member 0: the first twin; 1, 2, ...: the ensemble
        for k, v in p.items():
            if v is not None:
                p[k] = v * (1.0 + 2.0 ** -52 * rng.choice([-1.0, 1.0], size=v.shape))
    snaps = {k: [] for k in ("x", "px", "y", "py")}
    emit = {}
    t0 = time.time()
    for turn in range(1, turns + 1):
        p, _w = orc.track(wl.kind, wl.ipar, wl.par, wl.grids, wl.beam, p, n_turns=1)
        for k in snaps:
            snaps[k].append(p[k][:N_TAGGED].copy())
        if turn % 10 == 0 or turn == turns:
            m = orc.moments(p)
            emit[str(turn)] = [float(m[28]), float(m[29]), float(m[30])]
            print(name, "turn", turn, emit[str(turn)], f"{time.time() - t0:.0f} s", flush=True)
    out = dict(command=f"python tests/golden/make_golden.py {name}", cfg=cfg, n=n, turns=turns, deposit_mode=mode,
               n_tagged=N_TAGGED, emittances=emit, oracle_seconds=time.time() - t0, tunes={})
    if n_real is not None:
        out["n_real"] = float(n_real)
    for (a, b, (beta, alpha)) in planes:
        tq = tunes(np.stack(snaps[a]), np.stack(snaps[b]), beta, alpha)
        out["tunes"][a] = dict(mean=float(tq.mean()), rms_spread=float(tq.std()), beta=beta, alpha=alpha)
    m = orc.moments(p)
    out["moments_final"] = [float(v) for v in m]
    path = os.path.join(HERE, f"{name}.json")
    if twin:                                  # merge into the unperturbed run's file
        with open(path) as f:
            base = json.load(f)
        rec = dict(command=f"python tests/golden/make_golden.py {name}_twin" + (f"s {member}" if member else ""), emittances=out["emittances"],
                   tunes=out["tunes"], oracle_seconds=out["oracle_seconds"],
                   what="same run, every initial coordinate moved by one unit in the last place (random sign)")
        if member:
            # an ensemble of further twins (independent sign patterns): the spread of a chaotic run's statistics under
            # rounding-level changes, from which the GPU test's bound is taken.  Written to its own file (several members
            # run at the same time); `long_cfg3_merge` folds the member files into long_cfg3.json["twins"].
            with open(os.path.join(HERE, f"{name}.twin{member}.json"), "w") as f:
                json.dump(rec, f, indent=1)
            return
        base["twin"] = rec
        out = base
    with open(path, "w") as f:
        json.dump(out, f, indent=1)


def cfg5_full(twin=False):
    """twin=True: the same turn from initial coordinates moved by 1e-13 relative (random signs) -- the level at which
    two correct implementations agree after a node (FFT summation order, fused multiply-adds); the stored sample then
    shows how far cfg5's violent dynamics (80 % of the charge in a spike two cells wide) carry such a difference in one
    turn."""
    wl = make_config(5)
    if twin:
        rng = np.random.Generator(np.random.PCG64(78))
        for k, v in wl.particles.items():
            wl.particles[k] = v * (1.0 + 1e-13 * rng.choice([-1.0, 1.0], size=v.shape))
    t0 = time.time()
    want, works = orc.track_workload(wl, n_turns=1)
    dt = time.time() - t0
    rng = np.random.Generator(np.random.PCG64(2010_11540))
    idx = np.sort(rng.choice(wl.n, 1024, replace=False))
    if twin:
        path = os.path.join(HERE, "cfg5_full.json")
        with open(path) as f:
            base = json.load(f)
        base["twin"] = dict(command="python tests/golden/make_golden.py cfg5_full_twin", oracle_seconds=dt,
                            what="same turn, every initial coordinate moved by 1e-13 relative (random sign)",
                            particles={k: [float(v) for v in want[k][idx]] for k in want})
        with open(path, "w") as f:
            json.dump(base, f, indent=1)
        print("cfg5_full twin", dt, "s", flush=True)
        return
    m = orc.moments(want)
    out = dict(command="python tests/golden/make_golden.py cfg5_full", cfg=5, n=wl.n, turns=1, oracle_seconds=dt,
               n_inside_last_node=int(works[0].n_inside), index=[int(i) for i in idx],
               rms={k: float(np.sqrt(np.mean(want[k] ** 2))) for k in want},
               particles={k: [float(v) for v in want[k][idx]] for k in want},
               moments=[float(v) for v in m])
    with open(os.path.join(HERE, "cfg5_full.json"), "w") as f:
        json.dump(out, f, indent=1)
    print("cfg5_full", dt, "s", flush=True)


def main():
    what = sys.argv[1] if len(sys.argv) > 1 else "all"
    if what in ("long_cfg2", "all"):
        bx, by = 4e-3 / 0.10365e-3, 2e-3 / 0.47027e-3       # matched, alpha = 0 at the QF centre (workloads/configs.py)
        long_run(2, 100_000, 100, 0, (("x", "px", (bx, 0.0)), ("y", "py", (by, 0.0))), "long_cfg2")
    if what in ("long_cfg3", "all"):
        long_run(3, 100_000, 200, 1, (("x", "px", CFG3_TWISS[0]), ("y", "py", CFG3_TWISS[1])), "long_cfg3")
    if what == "long_cfg2_twin":
        bx, by = 4e-3 / 0.10365e-3, 2e-3 / 0.47027e-3
        long_run(2, 100_000, 100, 0, (("x", "px", (bx, 0.0)), ("y", "py", (by, 0.0))), "long_cfg2", twin=True)
    if what == "long_cfg3_twin":
        long_run(3, 100_000, 200, 1, (("x", "px", CFG3_TWISS[0]), ("y", "py", CFG3_TWISS[1])), "long_cfg3", twin=True)
    if what == "long_cfg3_paper":
        long_run(3, 100_000, 200, 1, (("x", "px", CFG3_TWISS[0]), ("y", "py", CFG3_TWISS[1])), "long_cfg3_paper", n_real=N_REAL_PAPER_REGIME)
    if what == "long_cfg3_paper_twin":
        long_run(3, 100_000, 200, 1, (("x", "px", CFG3_TWISS[0]), ("y", "py", CFG3_TWISS[1])), "long_cfg3_paper", twin=True, n_real=N_REAL_PAPER_REGIME)
    if what == "long_cfg3_twins":
        long_run(3, 100_000, 200, 1, (("x", "px", CFG3_TWISS[0]), ("y", "py", CFG3_TWISS[1])), "long_cfg3", twin=True, member=int(sys.argv[2]))
    if what == "long_cfg3_merge":
        import glob
        path = os.path.join(HERE, "long_cfg3.json")
        with open(path) as f:
            base = json.load(f)
        base["twins"] = []
        for mf in sorted(glob.glob(os.path.join(HERE, "long_cfg3.twin*.json"))):
            with open(mf) as f:
                base["twins"].append(json.load(f))
        with open(path, "w") as f:
            json.dump(base, f, indent=1)
        print("merged", len(base["twins"]), "ensemble members")
    if what in ("cfg5_full", "all"):
        cfg5_full()
    if what == "cfg5_full_twin":
        cfg5_full(twin=True)


if __name__ == "__main__":
    main()
