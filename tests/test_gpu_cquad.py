"""GPU parity of the chromatic thick quadrupole row (N3: eq. 6 per particle, SC_CQUAD) against the oracle."""
import numpy as np
import pytest

from workloads import CQUAD, QUAD, make_config

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


def chromatic(wl):
    """cfg3 with every thick quadrupole tracked by eq. 6 as printed instead of its on-momentum matrix."""
    wl.kind = wl.kind.copy()
    wl.kind[wl.kind == QUAD] = CQUAD
    return wl


@pytest.mark.parametrize("n,turns,tol,mode", [(20_000, 1, 1e-10, 0), (20_000, 1, 1e-10, 1), (4_000, 10, 1e-8, 0)])
def test_cquad_tracking_parity(sc, orc, n, turns, tol, mode):
    wl = chromatic(make_config(3, n=n, deposit_mode=mode))
    assert (wl.kind == CQUAD).sum() == 216
    want, _ = orc.track_workload(wl, n_turns=turns)
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    t.sc_track(turns)
    got = t.sc_get_particles()
    if mode == 1:
        tol = tol + 16.0 * 2.0 ** -wl.grids[0]["fixed_bits"] / n
    for k in NAMES:
        assert rel_err(got[k], want[k]) < tol, (k, rel_err(got[k], want[k]))
    # chromatic tracking is not the linear tracking: off-momentum particles end up elsewhere
    lin, _ = orc.track_workload(make_config(3, n=n, deposit_mode=mode), n_turns=turns)
    assert rel_err(lin["x"], want["x"]) > 1e-4
    t.close()


def test_cquad_4d_beam_and_zero_strength(sc, orc):
    """4D coasting beam (psigma = 0: the chromatic map reduces to the matrix) and a k1 = 0 row (a drift)."""
    from workloads import DRIFT, SCNODE, rows_to_arrays
    wl = make_config(1, n=5_000)
    rows = [(CQUAD, 0, [0.3, 0.5]), (DRIFT, 0, [2.0]), (CQUAD, 0, [-0.3, 0.5]), (CQUAD, 0, [0.0, 2.0]), (SCNODE, 0, [5.0])] * 8
    wl.kind, wl.ipar, wl.par = rows_to_arrays(rows)
    want, _ = orc.track_workload(wl, n_turns=2)
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    t.sc_track(2)
    got = t.sc_get_particles()
    for k in ("x", "px", "y", "py"):
        assert rel_err(got[k], want[k]) < 1e-10, k
    t.close()


def test_thick_sextupole_row(sc, orc):
    """SC_SEXT (eq. 8) in a FODO ring with space charge: against the oracle's five-map composition."""
    from workloads import DRIFT, QUAD, SCNODE, SEXT, rows_to_arrays
    wl = make_config(2, n=8_000)
    f = 0.25
    cell = [(QUAD, 0, [f, 0.4]), (DRIFT, 0, [1.0]), (SEXT, 0, [3.0, 0.3]), (DRIFT, 0, [1.0]), (SCNODE, 0, [2.7]),
            (QUAD, 0, [-f, 0.4]), (DRIFT, 0, [1.0]), (SEXT, 0, [-3.0, 0.3]), (DRIFT, 0, [1.0]), (SCNODE, 0, [2.7])]
    wl.kind, wl.ipar, wl.par = rows_to_arrays(cell * 12)
    want, _ = orc.track_workload(wl, n_turns=3)
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    t.sc_track(3)
    got = t.sc_get_particles()
    for k in ("x", "px", "y", "py"):
        assert rel_err(got[k], want[k]) < 1e-9, (k, rel_err(got[k], want[k]))
    t.close()


def test_exact_drift_row(sc, orc):
    """SC_XDRIFT everywhere cfg3 has a DRIFT: against the oracle's straight-line drift, 6D, with space charge."""
    from workloads import DRIFT, XDRIFT
    n = 20_000
    wl = make_config(3, n=n, deposit_mode=0)
    wl.kind = wl.kind.copy()
    wl.kind[wl.kind == DRIFT] = XDRIFT
    want, _ = orc.track_workload(wl, n_turns=1)
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    t.sc_track(1)
    got = t.sc_get_particles()
    for k in NAMES:
        assert rel_err(got[k], want[k]) < 1e-10, (k, rel_err(got[k], want[k]))
    lin, _ = orc.track_workload(make_config(3, n=n, deposit_mode=0), n_turns=1)
    assert np.abs(lin["sigma"] - want["sigma"]).max() > 1e-6          # not the H0 drift
    t.close()


def test_exact_sector_bend_row(sc, orc):
    """SC_SBEND in a small ring of FODO cells with bends (dispersion mixes psigma into x), exact drifts, space charge
    and an RF kick, 6D beam: all six coordinates against the oracle after two turns."""
    from workloads import DRIFT, QUAD, RF, SBEND, SCNODE, XDRIFT, rows_to_arrays
    n = 10_000
    wl = make_config(3, n=n, deposit_mode=1)
    ncell, lb = 16, 2.0
    h = 2.0 * np.pi / (2 * ncell * lb)                   # the bends close the ring: 2 per cell
    cell = [(QUAD, 0, [0.12, 0.5]), (XDRIFT, 0, [0.8]), (SBEND, 0, [lb, h]), (DRIFT, 0, [0.8]), (SCNODE, 0, [4.1]),
            (QUAD, 0, [-0.12, 0.5]), (XDRIFT, 0, [0.8]), (SBEND, 0, [lb, h]), (SBEND, 0, [0.0, h]), (DRIFT, 0, [0.8]),
            (SCNODE, 0, [4.1])]
    rows = cell * ncell + [(RF, 0, [100.0e3, 4.0, 0.0])]
    wl.kind, wl.ipar, wl.par = rows_to_arrays(rows)
    wl.beam["circumference"] = ncell * 2 * (0.5 + 0.8 + lb + 0.8)
    half = wl.beam["circumference"] / 8
    wl.grids[0].update(smin=-half, smax=half)
    wl.particles["sigma"] = np.ascontiguousarray(wl.particles["sigma"] * (half / 60.0))
    want, works = orc.track_workload(wl, n_turns=2)
    assert works[0].n_inside > 0.9 * n
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    t.sc_track(2)
    got = t.sc_get_particles()
    tol = 1e-9 + 16 * 2.0 ** -19 / n
    for k in NAMES:
        assert rel_err(got[k], want[k]) < tol, (k, rel_err(got[k], want[k]))
    t.close()
