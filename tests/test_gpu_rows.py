"""GPU parity on a lattice that exercises every row kind and every interpreter op of k_push: fused and unfused
drift+multipole pairs, normal and skew multipoles of orders 0-6, explicit LINMAP rows, QUAD and CQUAD, RF with a
phase, two different grids (one open, one pipe, different sizes and deposit modes), a segment longer than one
launch's program slots (split into pieces: kick with the first, deposit with the last), and back-to-back SC nodes."""
import numpy as np
import pytest

from workloads import CQUAD, DRIFT, LINMAP, MULT, QUAD, RF, SCNODE, make_beam_spec, make_grid, rows_to_arrays
from workloads.configs import Workload

pytestmark = pytest.mark.gpu
NAMES = ("x", "px", "y", "py", "sigma", "psigma")


@pytest.fixture(scope="module")
def sc():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    import paper_2010_11540_b200 as sc
    sc.load_library()
    return sc


def rel_err(a, b):
    return float(np.abs(a - b).max() / max(np.sqrt(np.mean(b * b)), 1e-300))


def kitchen_sink(n, seed=77):
    th = 0.3
    rot = [np.cos(th), 2.0 * np.sin(th), -0.5 * np.sin(th), np.cos(th)]          # det 1
    rows = []
    for c in range(6):
        s = 1.0 if c % 2 == 0 else -1.0
        rows += [(QUAD, 0, [s * 0.11, 1.2]), (DRIFT, 0, [0.7]), (MULT, 2, [s * 0.04, 0.0]),      # fused DM2
                 (DRIFT, 0, [0.3]), (MULT, 1, [0.002, 0.001]),                                    # skew quad: unfused
                 (MULT, 0, [1e-5, -2e-5]), (DRIFT, 0, [0.4]), (MULT, 3, [s * 0.8, 0.0]),         # dipole kick; fused DM3
                 (MULT, 4, [30.0, -10.0]), (MULT, 6, [2.0e5, 1.0e5]),                             # general orders
                 (LINMAP, 0, rot + [1.0, 0.5, 0.0, 1.0] + [0.5]), (DRIFT, 0, [0.6]),
                 (SCNODE, c % 2, [4.0]),
                 (CQUAD, 0, [-s * 0.09, 0.8]), (DRIFT, 0, [1.1]), (MULT, 1, [s * 0.01, 0.0]),    # fused DM1
                 (DRIFT, 0, [0.2]), (MULT, 0, [0.0, 0.0]),                                        # fused DM0
                 (SCNODE, (c + 1) % 2, [2.0]), (SCNODE, c % 2, [0.5])]                            # back-to-back nodes
        if c == 3:                                                                                # > 160 slots: pieces
            rows += [(LINMAP, 0, rot + [1.0, 0.1, 0.0, 1.0] + [0.1])] * 40 + [(DRIFT, 0, [0.05]), (MULT, 5, [1.0e3, 0.0])] * 30
            rows += [(SCNODE, 1, [3.0])]
    rows += [(RF, 0, [150.0e3, 4.0, 0.2]), (RF, 0, [40.0e3, 8.0, -0.1])]
    kind, ipar, par = rows_to_arrays(rows)
    C = 60.0
    grids = [make_grid(64, 0.03, nbins=64, smin=-C / 8, smax=C / 8, deposit_mode=1, fixed_bits=17),
             dict(make_grid(32, 0.035, ny=128, half_y=0.03, nbins=100, smin=-C / 8, smax=C / 8, deposit_mode=0), boundary=1,
                  long_kick=1)]
    rng = np.random.Generator(np.random.PCG64(seed))
    g = rng.standard_normal((n, 6))
    parts = dict(x=4e-3 * g[:, 0], px=4e-4 * g[:, 1], y=3e-3 * g[:, 2], py=5e-4 * g[:, 3], sigma=2.0 * g[:, 4],
                 psigma=3e-3 * g[:, 5])
    parts = {k: np.ascontiguousarray(v) for k, v in parts.items()}
    beam = make_beam_spec(n_real=4.0e11, circumference=C)
    return Workload(name="sink", kind=kind, ipar=ipar, par=par, grids=grids, beam=beam, particles=parts, n_turns=2,
                    notes={})


@pytest.mark.parametrize("n,turns", [(7_001, 1), (3_000, 3)])
def test_every_row_kind_two_grids_and_pieces(sc, orc, n, turns):
    wl = kitchen_sink(n)
    want, _ = orc.track_workload(wl, n_turns=turns)
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    t.sc_track(turns)
    got = t.sc_get_particles()
    tol = (1e-10 if turns == 1 else 1e-9) + 16 * 2.0 ** -17 / n
    for k in NAMES:
        assert rel_err(got[k], want[k]) < tol, (k, rel_err(got[k], want[k]))
    t.close()


def test_stepping_through_the_sink_matches_whole_turns(sc, orc):
    """sc_step in odd row counts (stops inside pieces, on nodes, between back-to-back nodes) == one sc_track."""
    wl = kitchen_sink(2_000)
    a = sc.Tracker.from_workload(wl)
    a.sc_load_particles(wl.particles)
    a.sc_track(1)
    pa = a.sc_get_particles()
    b = sc.Tracker.from_workload(wl)
    b.sc_load_particles(wl.particles)
    done = 0
    for step in (13, 1, 6, 1, 1, 37, 60, 29):
        b.sc_step(step)
        done += step
    b.sc_step(wl.n_rows - done)
    b.sc_track(0)                                   # the last node's kick
    pb = b.sc_get_particles()
    for k in NAMES:
        assert rel_err(pb[k], pa[k]) < 1e-12, k       # fp64 grid on grid 1: summation order differs run to run
    a.close(); b.close()
