"""Pins of the oracle's longitudinal space-charge kick (N2; eq. 13) and of the pieces it adds:
the slope of the piecewise-linear line density, the bilinear gather of the potential, and the kick itself on
prescribed smooth fields where the answer has a closed form."""
import numpy as np
import pytest

from workloads import make_beam_spec, make_grid


def bunch_grid(n=64, half=0.02, nbins=32, smin=-8.0, smax=8.0, **kw):
    g = make_grid(n, half, nbins=nbins, smin=smin, smax=smax)
    g.update(kw)
    return g


def test_lambda_slope_is_the_derivative_of_lambda_at(orc):
    g = bunch_grid()
    rng = np.random.Generator(np.random.PCG64(5))
    cnt = rng.integers(0, 500, g["nbins"]).astype(np.int64)
    n, n_real = int(cnt.sum()), 3.0e12
    ds = (g["smax"] - g["smin"]) / g["nbins"]
    h = 1e-4 * ds
    for s in rng.uniform(g["smin"] + 0.01 * ds, g["smax"] - 0.01 * ds, 200):
        c = (s - g["smin"]) / ds - 0.5
        if abs(c - round(c)) < 1e-3:                       # slope jumps at the bin centres
            continue
        fd = (orc.lambda_at(s + h, g, cnt, n_real, n) - orc.lambda_at(s - h, g, cnt, n_real, n)) / (2 * h)
        assert orc.lambda_slope(s, g, cnt, n_real, n) == pytest.approx(fd, rel=1e-6, abs=1e-9 * n_real / (n * ds * ds))
    # hand values: between the centres of bins 3 and 4; before the first centre (left neighbour counts as 0); outside
    scale = n_real / (n * ds)
    s34 = g["smin"] + 4.0 * ds
    assert orc.lambda_slope(s34, g, cnt, n_real, n) == pytest.approx(scale * (cnt[4] - cnt[3]) / ds, rel=1e-13)
    assert orc.lambda_slope(g["smin"] + 0.25 * ds, g, cnt, n_real, n) == pytest.approx(scale * cnt[0] / ds, rel=1e-13)
    assert orc.lambda_slope(g["smax"] - 0.25 * ds, g, cnt, n_real, n) == pytest.approx(-scale * cnt[-1] / ds, rel=1e-13)
    assert orc.lambda_slope(g["smin"] - 1e-9, g, cnt, n_real, n) == 0.0
    assert orc.lambda_slope(g["smax"], g, cnt, n_real, n) == 0.0


def test_gather_scalar_is_bilinear(orc):
    g = bunch_grid(16, 0.015)
    dx = 0.03 / 15
    xs = g["xmin"] + dx * np.arange(16)
    X, Y = np.meshgrid(xs, xs)
    u = 2.0 + 3.0 * X - 5.0 * Y + 7.0e2 * X * Y            # bilinear functions are reproduced exactly
    rng = np.random.Generator(np.random.PCG64(6))
    for x, y in rng.uniform(-0.0149, 0.0149, (100, 2)):
        inside, v = orc.gather_scalar(u, g, x, y)
        assert inside and v == pytest.approx(2.0 + 3.0 * x - 5.0 * y + 7.0e2 * x * y, rel=1e-12)
    assert orc.gather_scalar(u, g, xs[3], xs[7]) == (True, pytest.approx(u[7, 3], rel=1e-14))
    assert orc.gather_scalar(u, g, 0.0151, 0.0)[0] is False


def smooth_case(orc, long_kick):
    """Prescribed fields on a 128^2 grid: u = U0 cos(kx x) cos(ky y) (E = -grad u by orc.field), a Gaussian line
    density sampled as integer counts; test particles well inside."""
    g = bunch_grid(128, 0.02, nbins=1024, smin=-40.0, smax=40.0, long_kick=int(long_kick))
    beam = make_beam_spec(n_real=2.0e13, circumference=1567.5)
    n = 200
    dx = 0.04 / 127
    xs = g["xmin"] + dx * np.arange(128)
    X, Y = np.meshgrid(xs, xs)
    kx, ky, U0 = 90.0, 60.0, 0.3
    w = orc.Work(g)
    w.u[:] = (U0 * np.cos(kx * X) * np.cos(ky * Y)).ravel()
    Ex, Ey = orc.field(w.u.reshape(128, 128), g)
    w.Ex[:], w.Ey[:] = Ex.ravel(), Ey.ravel()
    ds = 80.0 / 1024
    centres = g["smin"] + ds * (np.arange(1024) + 0.5)
    sig_z, ntot = 9.0, 4.0e9
    w.cnt[:] = np.rint(ntot * ds * np.exp(-0.5 * (centres / sig_z) ** 2) / (np.sqrt(2 * np.pi) * sig_z)).astype(np.int64)
    rng = np.random.Generator(np.random.PCG64(7))
    p = dict(x=rng.uniform(-0.012, 0.012, n), y=rng.uniform(-0.012, 0.012, n), px=np.zeros(n), py=np.zeros(n),
             sigma=rng.uniform(-20.0, 20.0, n), psigma=np.zeros(n))
    # the kick normalises lambda by the number of particles it is called with; make that the histogram's total
    scale_fix = n / float(w.cnt.sum())
    lam = lambda s: beam["n_real"] * np.exp(-0.5 * (s / sig_z) ** 2) / (np.sqrt(2 * np.pi) * sig_z) * (ntot / w.cnt.sum())
    dlam = lambda s: -s / sig_z ** 2 * lam(s)
    return g, beam, w, p, (kx, ky, U0), lam, dlam, scale_fix


def test_long_kick_closed_form_on_smooth_fields(orc):
    """psigma -= kappa L u(x,y) lambda'(sigma) and px += kappa L lambda(sigma) (-du/dx): against the analytic u,
    lambda and their derivatives, within the O(h^2) error of bilinear interpolation and central differences
    (< 2e-3 of the kick scale here) and the O(ds) error of the piecewise-constant slope of the histogram
    (ds/(2 sigma_z) / 0.6 = 0.7 % with 1024 bins)."""
    g, beam, w, p, (kx, ky, U0), lam, dlam, fix = smooth_case(orc, True)
    L = 7.25
    kappa = orc.beam_struct(beam).kappa
    x, y, s = p["x"].copy(), p["y"].copy(), p["sigma"].copy()
    orc.sc_kick(p, g, beam, L, w)
    u = U0 * np.cos(kx * x) * np.cos(ky * y)
    ex = U0 * kx * np.sin(kx * x) * np.cos(ky * y)
    ey = U0 * ky * np.cos(kx * x) * np.sin(ky * y)
    # orc normalises counts by n (= len(p)), the analytic lambda by the histogram total: undo with fix
    want_ps = -kappa * L * u * dlam(s) / fix
    want_px = kappa * L * lam(s) * ex / fix
    want_py = kappa * L * lam(s) * ey / fix
    assert np.abs(p["psigma"] - want_ps).max() < 1e-2 * np.abs(want_ps).max()
    assert np.abs(p["px"] - want_px).max() < 2e-3 * np.abs(want_px).max()
    assert np.abs(p["py"] - want_py).max() < 2e-3 * np.abs(want_py).max()
    assert np.array_equal(p["x"], x) and np.array_equal(p["sigma"], s)


def test_long_kick_off_leaves_psigma_alone_and_kicks_share_one_hamiltonian(orc):
    g, beam, w, p, _, _, _, _ = smooth_case(orc, False)
    ps0 = p["psigma"].copy()
    orc.sc_kick(p, g, beam, 7.25, w)
    assert np.array_equal(p["psigma"], ps0)
    # d(delta px)/d sigma = d(delta psigma)/dx (both = -d2H/dx dsigma): finite differences on the frozen fields
    g, beam, w, p, _, _, _, _ = smooth_case(orc, True)
    n = len(p["x"])
    def kick(dxv, dsv):
        q = {k: v.copy() for k, v in p.items()}
        q["x"] += dxv; q["sigma"] += dsv
        orc.sc_kick(q, g, beam, 7.25, w)
        return q["px"], q["psigma"]
    hx, hs = 2e-5, 0.05
    dpx_ds = (kick(0.0, hs)[0] - kick(0.0, -hs)[0]) / (2 * hs)
    dps_dx = (kick(hx, 0.0)[1] - kick(-hx, 0.0)[1]) / (2 * hx)
    scale = np.abs(dpx_ds).max()
    assert np.median(np.abs(dpx_ds - dps_dx)) < 2e-2 * scale      # O(h^2) + kinks of the piecewise-linear tables
    assert np.corrcoef(dpx_ds, dps_dx)[0, 1] > 0.999
