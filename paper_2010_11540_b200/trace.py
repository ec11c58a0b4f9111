"""Where the time of one space-charge node goes: global-timer stamps at the phase boundaries of k_push and of the one-cluster
field solve, from the tracing build of the library (-DSC_TRACE: thread 0 of every CTA stores %globaltimer at each boundary).

    python -m paper_2010_11540_b200.build --trace && python -m paper_2010_11540_b200.trace [--particles N]

Tracks two turns of the bench configuration (cfg3), then all rows but the last of a third (so that the last launches are a
k_push with a deposit and its field solve), and prints the stamps of those two kernels relative to the first k_push CTA's start
(32 ns resolution).  The stamps cost a few hundred nanoseconds per node; the timed numbers come from the plain build (bench.py).
"""
from __future__ import annotations

import argparse
import ctypes as C
import os
import sys

import numpy as np


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--particles", type=int, default=1_000_000)
    ap.add_argument("--flags", type=int, default=0)
    args = ap.parse_args()
    from . import build as b
    if not os.path.exists(b.LIB_TRACE):
        b.build(trace=True)
    from . import binding
    binding.LIB_PATH = b.LIB_TRACE
    import paper_2010_11540_b200 as sc
    from workloads import make_config

    wl = make_config(3, n=args.particles, deposit_mode=1)
    t = sc.Tracker.from_workload(wl, flags=args.flags)
    t.sc_load_particles(wl.particles)
    t.sc_track(2)
    t.sc_step(wl.n_rows - 1)
    lib = binding.load_library()
    lib.sc_debug_trace.argtypes = [C.c_void_p, C.POINTER(C.c_uint64), C.c_int32]
    n_slots = 512 + 160 * 8
    out = (C.c_uint64 * n_slots)()
    if lib.sc_debug_trace(t.h, out, n_slots):
        raise RuntimeError("sc_debug_trace failed (not a tracing build?)")
    push = np.array(out[512:512 + 148 * 8], dtype=np.int64).reshape(148, 8)
    pois = np.array(out[:256], dtype=np.int64).reshape(16, 16)
    t0 = push[:, 0].min()
    d = push[:, [0, 1, 2, 5, 4, 6]] - t0
    print(f"k_push, {args.particles} macroparticles, 148 CTAs; ns after the first CTA's start (mean / min / max over the CTAs)")
    for k, name in enumerate(("CTA start", "private grid zeroed, waiting for the field solve", "field solve complete (griddepcontrol.wait returned)",
                              "field window staged (first warp's first kick can start)", "piece loop done, all warps", "flush done")):
        print(f"  {name:58s} {d[:, k].mean():9.0f} {d[:, k].min():9d} {d[:, k].max():9d}")
    names = {0: "first instruction", 13: "barriers armed", 1: "predecessor complete (griddepcontrol.wait returned)", 14: "loads issued", 2: "rows forward: transform starts",
             3: "rows forward done", 4: "row spectra sent", 5: "column inputs complete", 6: "columns done (forward, multiply, inverse)", 7: "potential sent",
             8: "row inputs complete", 9: "rows inverse done", 10: "halo rows in", 12: "fields computed", 11: "potential and fields stored"}
    print("k_poisson_cluster, 16 CTAs; ns after the first k_push CTA's start (mean / min / max over the CTAs)")
    for k in (0, 13, 1, 14, 2, 3, 4, 5, 6, 7, 8, 9, 10, 12, 11):
        v = pois[:, k] - t0
        print(f"  {names[k]:58s} {v.mean():9.0f} {v.min():9d} {v.max():9d}")
    loop, flush = push[:, 4] - push[:, 2], push[:, 6] - push[:, 4]
    print(f"per CTA: piece loop {loop.mean():.0f} ({loop.min()}..{loop.max()}) ns, flush {flush.mean():.0f} ({flush.min()}..{flush.max()}) ns, "
          f"loop + flush {(loop + flush).mean():.0f} ({(loop + flush).min()}..{(loop + flush).max()}) ns, correlation(loop, flush) {np.corrcoef(loop, flush)[0, 1]:.2f}")
    t.close()
    return 0


if __name__ == "__main__":
    sys.exit(main())
