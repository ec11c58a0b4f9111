"""Pins of the ORACLE's driver loop and moments.  CPU only."""
import numpy as np
import pytest

from workloads import SCNODE, make_config, rng_normal


def test_moments_against_numpy_covariance(orc):
    rng = np.random.Generator(np.random.PCG64(9))
    n = 5000
    A = rng_normal(rng, 36).reshape(6, 6)
    z = rng_normal(rng, 6 * n).reshape(n, 6) @ A.T * 1e-3 + np.arange(6) * 1e-2
    names = ("x", "px", "y", "py", "sigma", "psigma")
    p = {k: np.ascontiguousarray(z[:, i]) for i, k in enumerate(names)}
    m = orc.moments(p)
    cov = np.cov(z.T, bias=True)
    assert m[0] == n
    assert m[1:7] == pytest.approx(z.mean(axis=0), rel=1e-12)
    k = 7
    for a in range(6):
        for c in range(a, 6):
            assert m[k] == pytest.approx(cov[a, c], rel=1e-10)
            k += 1
    for pl in range(3):
        assert m[28 + pl] == pytest.approx(np.sqrt(np.linalg.det(cov[2 * pl:2 * pl + 2, 2 * pl:2 * pl + 2])), rel=1e-10)
    # 4D beam: longitudinal slots are zero
    p4 = dict(p, sigma=None, psigma=None)
    m4 = orc.moments(p4)
    assert m4[5] == 0 and m4[6] == 0 and m4[30] == 0 and m4[28] == pytest.approx(m[28], rel=1e-14)


def test_track_is_the_row_by_row_composition(orc):
    """orc_track == calling the exported per-row functions one after the other (cfg1, one cell)."""
    wl = make_config(1, n=2000)
    b = orc.beam_struct(wl.beam)
    out, works = orc.track(wl.kind[:5], wl.ipar[:5], wl.par[:5], wl.grids, wl.beam, wl.particles, n_turns=1)
    p = {k: (None if v is None else v.copy()) for k, v in wl.particles.items()}
    orc.mult(p, 1, wl.par[0, 0], 0.0)
    orc.drift(p, 10.0, b.gamma0)
    orc.mult(p, 1, wl.par[2, 0], 0.0)
    orc.drift(p, 10.0, b.gamma0)
    w = orc.scnode(p, wl.grids[0], wl.beam, 20.0)
    for k in ("x", "px", "y", "py"):
        assert np.array_equal(out[k], p[k])
    assert np.array_equal(works[0].Q, w.Q) and w.n_inside == works[0].n_inside
    # the literal cfg1 beam is mismatched: a sizeable fraction is outside the +-5 sigma grid
    assert 0 < wl.n - w.n_inside < wl.n // 2


def test_stop_after_rows_stops_after_the_deposit(orc):
    wl = make_config(1, n=1000, deposit_mode=1)
    first_sc = int(np.argmax(wl.kind == SCNODE))
    full, _ = orc.track_workload(wl, stop_after_rows=first_sc)          # rows before the node
    part, works = orc.track_workload(wl, stop_after_rows=first_sc + 1)  # + deposit, no kick
    for k in ("x", "px", "y", "py"):
        assert np.array_equal(full[k], part[k])
    Qi, n_in = orc.deposit_fixed(part["x"], part["y"], wl.grids[0])
    assert np.array_equal(works[0].Qi.reshape(Qi.shape), Qi)
    assert int(Qi.sum()) == n_in << 38
    # crossing a turn boundary: n_rows + 3 rows = one turn then 3 rows
    a, _ = orc.track_workload(wl, stop_after_rows=wl.n_rows + 3)
    t1, _ = orc.track_workload(wl, n_turns=1)
    wl2 = make_config(1, n=1000, deposit_mode=1)
    wl2.particles = t1
    b, _ = orc.track_workload(wl2, stop_after_rows=3)
    for k in ("x", "px", "y", "py"):
        assert np.array_equal(a[k], b[k])


def test_bunched_beam_kick_scales_with_local_line_density(orc):
    """eq. 12: kick proportional to lambda(z): two particles at the same (x,y) but
    different sigma receive kicks in the ratio of the line density at their positions."""
    wl = make_config(3, n=20000)
    g = wl.grids[0]
    p = {k: v.copy() for k, v in wl.particles.items()}
    p["x"][:2] = 1e-3
    p["y"][:2] = 0.5e-3
    p["px"][:2] = 0
    p["py"][:2] = 0
    p["sigma"][0], p["sigma"][1] = 0.0, 20.0
    cnt = orc.lambda_hist(p["sigma"], g)
    l0 = orc.lambda_at(0.0, g, cnt, wl.beam["n_real"], wl.n)
    l1 = orc.lambda_at(20.0, g, cnt, wl.beam["n_real"], wl.n)
    orc.scnode(p, g, wl.beam, 7.0)
    assert p["px"][0] / p["px"][1] == pytest.approx(l0 / l1, rel=1e-12)
    assert p["px"][0] > 0 and p["py"][0] > 0          # defocusing: pushed away from the axis
    # Gaussian bunch: lambda(0)/lambda(20 m) = exp(20^2/(2 15^2)) within histogram noise
    assert l0 / l1 == pytest.approx(np.exp(400 / 450), rel=0.15)
    # integral of lambda over the bucket = n_real
    ds = (g["smax"] - g["smin"]) / g["nbins"]
    assert cnt.sum() * wl.beam["n_real"] / wl.n == pytest.approx(wl.beam["n_real"], rel=1e-3)
    assert ds == pytest.approx(1567.5 / 9 / 256)
