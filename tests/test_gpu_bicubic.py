"""GPU parity of row N4: the paper's bicubic interpolation of the potential with the analytic gradient (eqs. 28-29,
PAPER.md:297-310; grid.interp = SC_INTERP_BICUBIC) against the oracle's orc_gather_bicubic, per particle."""
import numpy as np
import pytest

from workloads import SCNODE, make_config

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


@pytest.mark.parametrize("boundary,long_kick,grid_n", [(0, 0, 128), (1, 1, 128), (0, 1, 64), (1, 0, 256)])
def test_bicubic_kick_one_turn(sc, orc, boundary, long_kick, grid_n):
    """cfg3 decimated, fp64 deposit (no fixed-point allowance): all six coordinates within 1e-10 after one turn."""
    wl = make_config(4, n=20_011, grid_n=grid_n, deposit_mode=0)
    wl.grids[0].update(interp=1, boundary=boundary, long_kick=long_kick)
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    t.sc_track(1)
    got = t.sc_get_particles()
    want, _ = orc.track_workload(wl, n_turns=1)
    for k in NAMES:
        assert rel_err(got[k], want[k]) < 1e-10, (k, rel_err(got[k], want[k]))
    # it is a different kick from the bilinear one (the test would pass vacuously otherwise)
    wl.grids[0]["interp"] = 0
    other, _ = orc.track_workload(wl, n_turns=1)
    assert rel_err(other["px"], want["px"]) > 1e-6
    t.close()


def test_bicubic_edge_cells_and_outside(sc, orc):
    """cfg1 puts a quarter of its particles outside the grid and some in the edge cells on the way, where the stencil is
    extrapolated: 4D coasting beam, 64x64, three turns."""
    wl = make_config(1, deposit_mode=0)
    wl.grids[0]["interp"] = 1
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    t.sc_track(3)
    got = t.sc_get_particles()
    want, works = orc.track_workload(wl, n_turns=3)
    assert wl.n - works[0].n_inside > 0          # particles leave the grid: they crossed the edge cells on the way
    for k in ("x", "px", "y", "py"):
        assert rel_err(got[k], want[k]) < 1e-9, (k, rel_err(got[k], want[k]))
    t.close()


def test_bicubic_chromatic_rows_share_the_heavy_kernel(sc, orc):
    """interp = bicubic together with CQUAD rows (both live in the heavy k_push instantiation), fp64 deposit: 1e-10."""
    from workloads import CQUAD, QUAD
    wl = make_config(3, n=10_007, deposit_mode=0)
    wl.kind = wl.kind.copy()
    wl.kind[wl.kind == QUAD] = CQUAD
    wl.grids[0]["interp"] = 1
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    t.sc_track(1)
    got = t.sc_get_particles()
    want, _ = orc.track_workload(wl, n_turns=1)
    for k in NAMES:
        assert rel_err(got[k], want[k]) < 1e-10, (k, rel_err(got[k], want[k]))
    t.close()
