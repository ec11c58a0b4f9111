"""Pins of the oracle's N4 row: the paper's bicubic "Bezier surface" interpolation of the potential and its analytic
gradient (eqs. 28-29, section IV.C), in the reading A9 of DESIGN.md section 2 (control net = the
B-spline-to-Bezier conversion of the 4x4 stencil).  Nothing here retypes the oracle's formula: the pins are
  * what the mathematics fixes for any such surface (partition of unity, exact on linear potentials also in the edge
    cells, C^2 continuity across cell edges by one-sided limits, gradient = finite difference of the interpolant);
  * a library routine that evaluates the same spline (scipy.ndimage.map_coordinates, order 3, no prefilter);
  * the analytic field of a round Gaussian charge (convergence order 2 of the gathered field on the potential solved
    by the oracle's own, separately pinned, Poisson solver);
  * and a demonstration that eq. 28 READ LITERALLY (control points = node values) jumps between neighbouring cells,
    which is why that reading is rejected.
"""
import numpy as np
import pytest
from scipy import ndimage

from workloads import make_beam_spec, make_grid


def grid(nx=16, ny=12, hx=8e-3, hy=5e-3):
    return make_grid(nx, hx, ny=ny, half_y=hy)


def nodes(g):
    x = np.linspace(g["xmin"], g["xmax"], g["nx"])
    y = np.linspace(g["ymin"], g["ymax"], g["ny"])
    return x, y, (g["xmax"] - g["xmin"]) / (g["nx"] - 1), (g["ymax"] - g["ymin"]) / (g["ny"] - 1)


def test_partition_of_unity_and_zero_gradient(orc):
    g = grid()
    u = np.full((g["ny"], g["nx"]), 3.25)
    rng = np.random.default_rng(0)
    for _ in range(200):
        x = rng.uniform(g["xmin"], g["xmax"] * 0.999)
        y = rng.uniform(g["ymin"], g["ymax"] * 0.999)
        ins, v, ex, ey = orc.gather_bicubic(u, g, x, y)
        assert ins
        assert abs(v - 3.25) < 1e-14
        assert abs(ex) < 1e-10 and abs(ey) < 1e-10       # derivatives of the weights sum to zero (times 1/dx ~ 1e3)


def test_exact_on_linear_potentials_including_edge_cells(orc):
    g = grid()
    xs, ys, dx, dy = nodes(g)
    a, b, c = 0.7, -123.0, 456.0
    u = a + b * xs[None, :] + c * ys[:, None]
    pts = [(xs[0] + 0.3 * dx, ys[0] + 0.6 * dy), (xs[-1] - 0.2 * dx, ys[-1] - 0.9 * dy), (xs[0], ys[5]),
           (xs[3] + 0.5 * dx, ys[-1] - 1e-9), (xs[7] + 0.25 * dx, ys[6] + 0.75 * dy)]
    for x, y in pts:
        ins, v, ex, ey = orc.gather_bicubic(u, g, x, y)
        assert ins
        assert abs(v - (a + b * x + c * y)) < 1e-12
        assert abs(ex + b) < 1e-9 and abs(ey + c) < 1e-9


def test_outside_is_zero_and_flagged(orc):
    g = grid()
    u = np.random.default_rng(1).normal(size=(g["ny"], g["nx"]))
    for x, y in [(g["xmax"], 0.0), (g["xmin"] - 1e-6, 0.0), (0.0, g["ymax"]), (0.0, g["ymin"] - 1e-9)]:
        ins, v, ex, ey = orc.gather_bicubic(u, g, x, y)
        assert not ins and v == 0.0 and ex == 0.0 and ey == 0.0


def test_equals_library_cubic_bspline_in_the_interior(orc):
    """scipy.ndimage.map_coordinates(order=3, prefilter=False) evaluates the uniform cubic B-spline whose
    coefficients are the array itself -- the same surface, from a library."""
    g = grid(20, 18)
    xs, ys, dx, dy = nodes(g)
    rng = np.random.default_rng(2)
    u = rng.normal(size=(g["ny"], g["nx"]))
    px = rng.uniform(xs[2], xs[-3], 300)
    py = rng.uniform(ys[2], ys[-3], 300)
    want = ndimage.map_coordinates(u, [(py - ys[0]) / dy, (px - xs[0]) / dx], order=3, prefilter=False, mode="nearest")
    got = np.array([orc.gather_bicubic(u, g, x, y)[1] for x, y in zip(px, py)])
    assert np.abs(got - want).max() < 1e-13


def test_gradient_is_the_derivative_of_the_interpolant(orc):
    g = grid()
    xs, ys, dx, dy = nodes(g)
    rng = np.random.default_rng(3)
    u = rng.normal(size=(g["ny"], g["nx"]))
    for _ in range(100):
        ci, cj = rng.integers(0, g["nx"] - 1), rng.integers(0, g["ny"] - 1)
        x = xs[ci] + rng.uniform(0.1, 0.9) * dx
        y = ys[cj] + rng.uniform(0.1, 0.9) * dy
        _, v, ex, ey = orc.gather_bicubic(u, g, x, y)
        hx, hy = 1e-4 * dx, 1e-4 * dy
        fx = (orc.gather_bicubic(u, g, x + hx, y)[1] - orc.gather_bicubic(u, g, x - hx, y)[1]) / (2 * hx)
        fy = (orc.gather_bicubic(u, g, x, y + hy)[1] - orc.gather_bicubic(u, g, x, y - hy)[1]) / (2 * hy)
        scale = np.abs(u).max() / dx
        assert abs(ex + fx) < 1e-6 * scale and abs(ey + fy) < 1e-6 * scale * dx / dy


def test_c2_across_cell_edges(orc):
    """One-sided limits at interior cell edges: value, gradient and second derivative agree from both sides."""
    g = grid()
    xs, ys, dx, dy = nodes(g)
    rng = np.random.default_rng(4)
    u = rng.normal(size=(g["ny"], g["nx"]))
    eps = 1e-7
    for i in range(1, g["nx"] - 1):
        y = ys[4] + 0.37 * dy
        xl, xr = xs[i] - eps * dx, xs[i] + eps * dx
        _, vl, exl, eyl = orc.gather_bicubic(u, g, xl, y)
        _, vr, exr, eyr = orc.gather_bicubic(u, g, xr, y)
        assert abs(vl - vr) < 1e-5 and abs(exl - exr) * dx < 1e-5 and abs(eyl - eyr) * dy < 1e-5
        # second derivative from each side: finite difference of the ANALYTIC gradient inside that cell
        h = 1e-3 * dx
        d2l = (orc.gather_bicubic(u, g, xl, y)[2] - orc.gather_bicubic(u, g, xl - h, y)[2]) / h
        d2r = (orc.gather_bicubic(u, g, xr + h, y)[2] - orc.gather_bicubic(u, g, xr, y)[2]) / h
        assert abs(d2l - d2r) * dx * dx < 2e-2      # third derivative jumps (cubic pieces): O(h/dx) = 1e-3 slack
    for j in range(1, g["ny"] - 1):
        x = xs[5] + 0.61 * dx
        yl, yr = ys[j] - eps * dy, ys[j] + eps * dy
        _, vl, exl, eyl = orc.gather_bicubic(u, g, x, yl)
        _, vr, exr, eyr = orc.gather_bicubic(u, g, x, yr)
        assert abs(vl - vr) < 1e-5 and abs(exl - exr) * dx < 1e-5 and abs(eyl - eyr) * dy < 1e-5
        h = 1e-3 * dy
        d2l = (orc.gather_bicubic(u, g, x, yl)[3] - orc.gather_bicubic(u, g, x, yl - h)[3]) / h
        d2r = (orc.gather_bicubic(u, g, x, yr + h)[3] - orc.gather_bicubic(u, g, x, yr)[3]) / h
        assert abs(d2l - d2r) * dy * dy < 2e-2


def test_literal_eq28_is_discontinuous_hence_rejected():
    """Eq. 28 with the node values themselves as Bezier control points: at x -> x_i+ the surface equals u_{i-1},
    at x -> x_{i+1}- it equals u_{i+2}; the cell to the right starts at u_i.  One axis suffices."""
    u = np.array([0.0, 1.0, 4.0, 9.0, 16.0, 25.0])

    def literal(i, t):   # PAPER.md:303-306, one axis: sum_m u_{i+m-1} C(3,m) t^m (1-t)^(3-m)
        from math import comb
        return sum(u[i + m - 1] * comb(3, m) * t ** m * (1 - t) ** (3 - m) for m in range(4))

    assert literal(2, 1.0) == u[4] and literal(3, 0.0) == u[2]      # end of cell 2 vs start of cell 3: 16 vs 4
    assert literal(2, 0.0) == u[1]                                   # and not the node value u[2] either


@pytest.mark.parametrize("n", [64, 128])
def test_field_of_a_round_gaussian_converges_at_second_order(orc, n):
    """Potential of a round Gaussian charge solved by the oracle's (separately pinned) open-boundary solver, field by
    eqs. 28-29: error against (1 - exp(-r^2/2 sigma^2))/(2 pi r) is O(h^2) (the spline smooths with h^2 u''/6)."""
    sig = 3e-3
    errs = {}
    for nn in (n, 2 * n):
        g = make_grid(nn, 5 * sig)
        xs, ys, dx, dy = nodes(g)
        X, Y = np.meshgrid(xs, ys)
        Q = np.exp(-(X * X + Y * Y) / (2 * sig * sig))
        ntot = Q.sum()
        u = orc.poisson(Q, g, ntot)
        rng = np.random.default_rng(5)
        r = rng.uniform(0.3 * sig, 3.0 * sig, 400)
        th = rng.uniform(0, 2 * np.pi, 400)
        err = 0.0
        for x, y in zip(r * np.cos(th), r * np.sin(th)):
            _, _, ex, ey = orc.gather_bicubic(u, g, x, y)
            rr = np.hypot(x, y)
            er = (1 - np.exp(-rr * rr / (2 * sig * sig))) / (2 * np.pi * rr)
            err = max(err, np.hypot(ex - er * x / rr, ey - er * y / rr))
        errs[nn] = err * 2 * np.pi * sig
    ratio = errs[n] / errs[2 * n]
    assert errs[n] < (3e-2 if n == 64 else 8e-3)
    assert 3.0 < ratio < 5.5, (errs, ratio)


def test_kick_uses_the_bicubic_field_and_potential(orc):
    """orc_sc_kick with interp = 1: px += kappa lambda L (-du/dx) of the surface; psigma -= kappa L u lambda'."""
    g = make_grid(32, 10e-3, nbins=16, smin=-40.0, smax=40.0)
    g["interp"] = 1
    g["long_kick"] = 1
    xs, ys, dx, dy = nodes(g)
    rng = np.random.default_rng(6)
    n = 500
    p = dict(x=rng.uniform(-9e-3, 9e-3, n), px=np.zeros(n), y=rng.uniform(-9e-3, 9e-3, n), py=np.zeros(n),
             sigma=rng.normal(0, 12.0, n), psigma=np.zeros(n))
    beam = make_beam_spec(n_real=1e12, circumference=720.0)
    w = orc.Work(g)
    X, Y = np.meshgrid(xs, ys)
    w.u[:] = (np.cos(150.0 * X) * np.sin(90.0 * Y + 0.3)).ravel()
    w.cnt[:] = orc.lambda_hist(p["sigma"], g)
    q = {k: v.copy() for k, v in p.items()}
    orc.sc_kick(q, g, beam, 2.5, w)
    kappa = orc.beam_struct(beam).kappa
    for k in range(0, n, 7):
        _, uv, ex, ey = orc.gather_bicubic(w.u, g, p["x"][k], p["y"][k])
        lam = orc.lambda_at(p["sigma"][k], g, w.cnt, beam["n_real"], n)
        dl = orc.lambda_slope(p["sigma"][k], g, w.cnt, beam["n_real"], n)
        assert q["px"][k] == pytest.approx(kappa * lam * 2.5 * ex, rel=1e-12, abs=1e-30)
        assert q["py"][k] == pytest.approx(kappa * lam * 2.5 * ey, rel=1e-12, abs=1e-30)
        assert q["psigma"][k] == pytest.approx(-kappa * 2.5 * uv * dl, rel=1e-12, abs=1e-30)
