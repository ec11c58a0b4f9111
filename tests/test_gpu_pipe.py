"""GPU parity of the paper's conducting-pipe Poisson solver (grid.boundary = SC_BOUNDARY_PIPE, eqs. 15-27) against the
oracle: node grids element by element, tracking over turns, at small and at bench size."""
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


def grid_err(a, b):
    return float(np.abs(a - b).max() / np.abs(b).max())


def pipe_config(cfg, **kw):
    wl = make_config(cfg, **kw)
    for g in wl.grids:
        g["boundary"] = 1
    return wl


@pytest.mark.parametrize("cfg,n,mode,grid_n", [(1, 10_000, 0, None), (1, 10_000, 1, None), (2, 20_000, 0, None),
                                               (3, 30_011, 1, None), (4, 20_000, 1, 256), (4, 20_000, 0, 32)])
def test_pipe_first_node_grids(sc, orc, cfg, n, mode, grid_n):
    wl = pipe_config(cfg, n=n, deposit_mode=mode, grid_n=grid_n)
    first = int(np.argmax(wl.kind == SCNODE)) + 1
    _, works = orc.track_workload(wl, stop_after_rows=first)
    w = works[0]
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    t.sc_step(first)
    if mode == 1:
        assert np.array_equal(t.sc_get_grid(sc.SC_GRID_RHO_I64).ravel(), w.Qi)
    else:
        assert grid_err(t.sc_get_grid(sc.SC_GRID_RHO_F64).ravel(), w.Q) < 1e-10
    phi = t.sc_get_grid(sc.SC_GRID_PHI)
    assert grid_err(phi.ravel(), w.u) < 1e-10
    assert np.abs(phi[0, :]).max() < 1e-12 * np.abs(w.u).max()          # u = 0 on the wall nodes
    assert np.abs(phi[:, 0]).max() < 1e-12 * np.abs(w.u).max()
    assert grid_err(t.sc_get_grid(sc.SC_GRID_EX).ravel(), w.Ex) < 1e-10
    assert grid_err(t.sc_get_grid(sc.SC_GRID_EY).ravel(), w.Ey) < 1e-10
    # and it is not the open-boundary answer
    wo = make_config(cfg, n=n, deposit_mode=mode, grid_n=grid_n)
    _, works_open = orc.track_workload(wo, stop_after_rows=first)
    assert grid_err(phi.ravel(), works_open[0].u) > 1e-3
    t.close()


@pytest.mark.parametrize("cfg,n,turns,tol,mode", [(1, 10_000, 1, 1e-10, 0), (1, 10_000, 10, 1e-8, 0),
                                                  (2, 5_000, 10, 1e-8, 0), (3, 20_000, 1, 1e-10, 1)])
def test_pipe_tracking_parity(sc, orc, cfg, n, turns, tol, mode):
    wl = pipe_config(cfg, n=n, deposit_mode=mode)
    want, _ = orc.track_workload(wl, n_turns=turns)
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    t.sc_track(turns)
    got = t.sc_get_particles()
    if mode == 1:
        tol = tol + 16.0 * 2.0 ** -wl.grids[0]["fixed_bits"] / n
    for k in NAMES:
        if want.get(k) is None:
            continue
        assert rel_err(got[k], want[k]) < tol, (k, rel_err(got[k], want[k]))
    t.close()


def test_pipe_full_size_first_node(sc, orc):
    """cfg3 at 1e6 macroparticles, 128 x 128, the launch configuration bench.py times, pipe boundary."""
    wl = pipe_config(3, deposit_mode=1)
    first = int(np.argmax(wl.kind == SCNODE)) + 1
    _, works = orc.track_workload(wl, stop_after_rows=first)
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    t.sc_step(first)
    assert np.array_equal(t.sc_get_grid(sc.SC_GRID_RHO_I64).ravel(), works[0].Qi)
    assert grid_err(t.sc_get_grid(sc.SC_GRID_PHI).ravel(), works[0].u) < 1e-10
    assert grid_err(t.sc_get_grid(sc.SC_GRID_EX).ravel(), works[0].Ex) < 1e-10
    assert grid_err(t.sc_get_grid(sc.SC_GRID_EY).ravel(), works[0].Ey) < 1e-10
    t.sc_track(2)
    m = t.sc_moments()
    assert m[0] == wl.n and m[32] == 0
    t.close()


@pytest.mark.parametrize("boundary,n,turns,tol,mode", [(1, 20_000, 1, 1e-10, 1), (1, 6_000, 5, 1e-9, 0), (0, 20_000, 1, 1e-10, 0)])
def test_longitudinal_kick_parity(sc, orc, boundary, n, turns, tol, mode):
    """N2 (eq. 13): grid.long_kick = 1 -- psigma is kicked too; all six coordinates against the oracle."""
    wl = make_config(3, n=n, deposit_mode=mode)
    for g in wl.grids:
        g["boundary"] = boundary
        g["long_kick"] = 1
    want, _ = orc.track_workload(wl, n_turns=turns)
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    t.sc_track(turns)
    got = t.sc_get_particles()
    if mode == 1:
        tol = tol + 16.0 * 2.0 ** -wl.grids[0]["fixed_bits"] / n
    for k in NAMES:
        assert rel_err(got[k], want[k]) < tol, (k, rel_err(got[k], want[k]))
    t.close()
    # the longitudinal kick is really there: psigma differs from the run without it by far more than the tolerance
    wl0 = make_config(3, n=n, deposit_mode=mode)
    for g in wl0.grids:
        g["boundary"] = boundary
    base, _ = orc.track_workload(wl0, n_turns=turns)
    d = np.abs(base["psigma"] - want["psigma"]).max() / np.sqrt(np.mean(want["psigma"] ** 2))
    assert d > 1e3 * tol


def test_long_kick_needs_a_histogram(sc):
    wl = make_config(1, n=100)
    bad = dict(wl.grids[0], long_kick=1)                 # coasting beam: no lambda(sigma) to differentiate
    with pytest.raises(sc.ScError) as e:
        sc.Tracker(wl.kind, wl.ipar, wl.par, [bad], wl.beam, 100)
    assert e.value.code == -1
