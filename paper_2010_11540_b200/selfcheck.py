"""Self-check of an installed libsc_track on this machine's GPU: a few small tracking runs through every kernel variant.

    python -m paper_2010_11540_b200.selfcheck [--particles N] [--turns T]

No oracle is involved (that comparison is tests/): the runs only have to complete without a CUDA error and keep their
invariants (particle count, nothing non-finite, deterministic deposit reproducible run to run -- which a race in the
deposit, the flush or the field solve would break).  It is the workload for

    compute-sanitizer --tool memcheck  python -m paper_2010_11540_b200.selfcheck
    compute-sanitizer --tool racecheck python -m paper_2010_11540_b200.selfcheck

and, where compute-sanitizer is not available (it is closed on the B200 pool this was developed on, profiles/r02_sanitizer.md),
for the library's own checked build, whose kernels test every index they form before using it:

    python -m paper_2010_11540_b200.build --check && python -m paper_2010_11540_b200.selfcheck --check
"""
from __future__ import annotations

import argparse
import sys

import numpy as np


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--particles", type=int, default=20_000)
    ap.add_argument("--turns", type=int, default=1)
    ap.add_argument("--check", action="store_true", help="run the checked build (libsc_track_check.so, device-side index assertions)")
    args = ap.parse_args()
    if args.check:
        import os
        from . import build as b
        if not os.path.exists(b.LIB_CHECK):
            b.build(check=True)
        os.environ["SC_TRACK_LIB"] = b.LIB_CHECK
        from . import binding
        binding.LIB_PATH = b.LIB_CHECK
    import paper_2010_11540_b200 as sc
    from workloads import CQUAD, QUAD, make_config

    cases = [
        ("cfg3 128^2 fixed-point deposit, open boundary (field-window kernel, one-cluster field solve)", dict(cfg=3, mode=1), {}, 0),
        ("same, three-launch warp-per-transform field solve", dict(cfg=3, mode=1), {}, sc.SC_FLAG_WARP_FFT_POISSON),
        ("same, plain launches without programmatic dependent launch", dict(cfg=3, mode=1), {}, sc.SC_FLAG_NO_PDL),
        ("same, gather through the L1 and block FFTs", dict(cfg=3, mode=1), {}, sc.SC_FLAG_NO_FIELD_WINDOW | sc.SC_FLAG_BLOCK_FFT_POISSON),
        ("same, fused single-launch field solve", dict(cfg=3, mode=1), {}, sc.SC_FLAG_FUSED_POISSON),
        ("cfg3 128^2 fp64-atomic deposit, conducting pipe, longitudinal kick", dict(cfg=3, mode=0), dict(boundary=1, long_kick=1), 0),
        ("cfg4 256^2 fixed-point deposit (windowed deposit, L2 atomics outside the window)", dict(cfg=4, mode=1, grid=256), {}, 0),
        ("cfg4 64^2 fp64-atomic deposit", dict(cfg=4, mode=0, grid=64), {}, 0),
        ("cfg3 bicubic potential interpolation (eqs. 28-29), pipe", dict(cfg=3, mode=1), dict(interp=1, boundary=1), 0),
        ("cfg3 chromatic quadrupoles (heavy instantiation)", dict(cfg=3, mode=1, chromatic=True), {}, 0),
        ("cfg1 4D coasting beam, 64^2, particles leaving the grid", dict(cfg=1, mode=1, n=10_000), {}, 0),
        ("cfg5 spike + ring on 256^2", dict(cfg=5, mode=1), {}, 0),
    ]
    for name, c, gpatch, flags in cases:
        wl = make_config(c["cfg"], n=c.get("n", args.particles), grid_n=c.get("grid"), deposit_mode=c["mode"])
        wl.grids[0].update(gpatch)
        if c.get("chromatic"):
            wl.kind = wl.kind.copy()
            wl.kind[wl.kind == QUAD] = CQUAD
        outs = []
        for rep in range(2 if c["mode"] == 1 else 1):
            t = sc.Tracker.from_workload(wl, flags=flags)
            t.sc_load_particles(wl.particles)
            t.sc_step(7)                       # plain launches, stop inside a turn (kick pending)
            t.sc_step(wl.n_rows - 7)           # ... to the end of the turn
            t.sc_track(args.turns)             # whole turns by graph replay
            m = t.sc_moments()
            outs.append(t.sc_get_particles())
            t.close()
            assert m[0] == wl.n and m[32] == 0, (name, m[0], m[32])
        if len(outs) == 2:
            for k, v in outs[0].items():
                assert v is None or np.array_equal(v, outs[1][k]), (name, k, "fixed-point run not reproducible")
        print(f"ok  {name}: eps_x {m[28]:.6e} eps_y {m[29]:.6e} outside {int(m[31])}", flush=True)
    print("selfcheck ok")
    return 0


if __name__ == "__main__":
    sys.exit(main())
