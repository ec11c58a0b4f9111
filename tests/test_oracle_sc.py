"""Pins of the ORACLE's space-charge node (section IV) against closed
forms, invariants, numerical quadrature, a different library's FFT and brute force.  CPU only."""
import math

import numpy as np
import pytest
from scipy.integrate import dblquad

from workloads import LINMAP, SCNODE, make_grid, rows_to_arrays, rng_normal, rng_uniform

M_P = 938.27208816e6
BEAM = dict(kinetic_eV=3e9, mass_eV=M_P, charge=1, line_density=1e11)


def nodes(g):
    xs = np.linspace(g["xmin"], g["xmax"], g["nx"])
    ys = np.linspace(g["ymin"], g["ymax"], g["ny"])
    return xs, ys


# ---------------------------------------------------------------- deposit (P3)
def test_deposit_single_particle_hand_weights(orc):
    """eq. 14 on a 4x3 grid with dx = 1, dy = 2; particle at (1.25, 3.0):
    cell i=1, j=1, fx = .25, fy = .5 -> weights .375 .125 .375 .125 typed by hand."""
    g = dict(nx=4, ny=3, xmin=0.0, xmax=3.0, ymin=0.0, ymax=4.0)
    Q, n_in = orc.deposit_f64(np.array([1.25]), np.array([3.0]), g)
    want = np.zeros((3, 4))
    want[1, 1], want[1, 2], want[2, 1], want[2, 2] = 0.375, 0.125, 0.375, 0.125
    assert n_in == 1 and np.array_equal(Q, want)
    gf = dict(g, deposit_mode=1, fixed_bits=4)
    Qi, _ = orc.deposit_fixed(np.array([1.25]), np.array([3.0]), gf)
    assert np.array_equal(Qi, (want * 256).astype(np.int64))


def test_deposit_edges_and_outside(orc):
    g = dict(nx=5, ny=5, xmin=-2.0, xmax=2.0, ymin=-2.0, ymax=2.0)
    x = np.array([-2.0, 2.0, 1.9999999, -2.0000001, 0.0, np.nan, 0.0])
    y = np.array([-2.0, 0.0, 1.9999999, 0.0, 2.0, 0.0, np.inf])
    Q, n_in = orc.deposit_f64(x, y, g)
    assert n_in == 2                       # lower edge inclusive, upper edge exclusive, NaN/inf outside
    assert Q[0, 0] == 1.0
    assert Q.sum() == pytest.approx(2.0, abs=1e-15)
    assert Q[4, 4] == pytest.approx(1.0, abs=1e-6)


def test_deposit_conserves_charge_and_first_moments(orc):
    rng = np.random.Generator(np.random.PCG64(11))
    n = 20000
    x = 3e-3 * rng_normal(rng, n)
    y = 2e-3 * rng_normal(rng, n)
    g = make_grid(64, 9e-3)               # +-3 sigma in x: some particles outside
    Q, n_in = orc.deposit_f64(x, y, g)
    xs, ys = nodes(g)
    inside = (x >= g["xmin"]) & (x < g["xmax"]) & (y >= g["ymin"]) & (y < g["ymax"])
    assert n_in == inside.sum() and n_in < n
    assert Q.sum() == pytest.approx(n_in, rel=1e-13)
    # CIC conserves the first moments of the deposited particles
    assert (Q * xs[None, :]).sum() == pytest.approx(x[inside].sum(), rel=1e-11)
    assert (Q * ys[:, None]).sum() == pytest.approx(y[inside].sum(), rel=1e-11)
    # fixed point: exact integer total, and close to the fp64 grid
    for s in (12, 19):
        gf = dict(g, deposit_mode=1, fixed_bits=s)
        Qi, n_in2 = orc.deposit_fixed(x, y, gf)
        assert n_in2 == n_in
        assert int(Qi.sum()) == n_in * (1 << (2 * s))
        assert abs(Qi * 2.0 ** (-2 * s) - Q).max() < 40 * 2.0 ** (-s)


def test_deposit_brute_force_tent_functions(orc):
    """Q[node] = sum_p tent((x_p - x_node)/dx) tent((y_p - y_node)/dy): the cloud-in-cell shape
    written as a dense (node x particle) product instead of a scatter."""
    rng = np.random.Generator(np.random.PCG64(5))
    g = dict(nx=8, ny=4, xmin=-1.0, xmax=2.5, ymin=0.0, ymax=1.5)
    x = -1.0 + 3.5 * rng_uniform(rng, 300) * 0.999
    y = 1.5 * rng_uniform(rng, 300) * 0.999
    Q, _ = orc.deposit_f64(x, y, g)
    xs, ys = nodes(g)
    tent = lambda t: np.clip(1 - np.abs(t), 0, None)
    Wx = tent((x[None, :] - xs[:, None]) / 0.5)
    Wy = tent((y[None, :] - ys[:, None]) / 0.5)
    assert Q == pytest.approx(Wy @ Wx.T, abs=1e-12)


# ---------------------------------------------------------------- lambda histogram
def test_lambda_histogram_and_interpolation(orc):
    g = dict(nx=4, ny=4, xmin=0, xmax=1, ymin=0, ymax=1, nbins=4, smin=-2.0, smax=2.0)
    s = np.array([-2.0, -1.5, -0.5, -0.25, 0.0, 1.999, 2.0, -2.1, 5.0])
    cnt = orc.lambda_hist(s, g)
    assert list(cnt) == [2, 2, 1, 1]
    assert np.array_equal(cnt, np.histogram(s[(s >= -2) & (s < 2)], bins=4, range=(-2, 2))[0])
    n, n_real = len(s), 9e12
    lam = n_real * cnt / (n * 1.0)          # per metre, bin width 1
    centres = np.array([-1.5, -0.5, 0.5, 1.5])
    for sig in (-1.5, -1.0, -0.2, 0.5, 1.2):
        assert orc.lambda_at(sig, g, cnt, n_real, n) == pytest.approx(np.interp(sig, centres, lam), rel=1e-14)
    # half bins at the ends interpolate towards empty neighbours; outside the range: 0
    assert orc.lambda_at(-1.75, g, cnt, n_real, n) == pytest.approx(0.75 * lam[0], rel=1e-14)
    assert orc.lambda_at(1.75, g, cnt, n_real, n) == pytest.approx(0.75 * lam[3], rel=1e-14)
    assert orc.lambda_at(2.0, g, cnt, n_real, n) == 0.0 and orc.lambda_at(-2.5, g, cnt, n_real, n) == 0.0
    # the histogram integrates to the number of real particles inside the range
    assert (lam * 1.0).sum() == pytest.approx(n_real * 6 / n, rel=1e-14)


# ---------------------------------------------------------------- FFT and Green's function (P9, A10)
@pytest.mark.parametrize("n", [2, 8, 64, 256])
def test_fft_against_naive_dft_and_numpy(orc, n):
    rng = np.random.Generator(np.random.PCG64(n))
    re, im = rng_normal(rng, n), rng_normal(rng, n)
    for inv in (False, True):
        got = orc.fft(re, im, inv)
        want = np.fft.ifft(re + 1j * im) if inv else np.fft.fft(re + 1j * im)
        assert abs(got - want).max() < 1e-13 * n
        assert abs(orc.dft_naive(re, im, inv) - want).max() < 1e-13 * n


def test_green_cell_against_quadrature(orc):
    dx, dy = 0.3, 0.2
    f = lambda yy, xx: -math.log(max(xx * xx + yy * yy, 1e-300)) / (4 * math.pi)
    for a, b in ((0, 0), (1, 0), (0, 1), (2, 3), (7, 5)):
        if (a, b) == (0, 0):     # integrable log singularity at the corner of each quadrant
            num = 4 * dblquad(f, 0, dx / 2, 0, dy / 2, epsabs=1e-13, epsrel=1e-11)[0]
        else:
            num = dblquad(f, a * dx - dx / 2, a * dx + dx / 2, b * dy - dy / 2, b * dy + dy / 2,
                          epsabs=1e-13, epsrel=1e-11)[0]
        assert orc.green_cell(a * dx, b * dy, dx, dy) == pytest.approx(num / (dx * dy), rel=2e-7 if (a, b) == (0, 0) else 1e-9)
    # far field -> point value -ln(r^2)/(4 pi), correction O((dx/r)^2)
    x, y = 40 * dx, 25 * dy
    assert orc.green_cell(x, y, dx, dy) == pytest.approx(-math.log(x * x + y * y) / (4 * math.pi), abs=1e-5)
    # symmetry
    assert orc.green_cell(-x, y, dx, dy) == pytest.approx(orc.green_cell(x, -y, dx, dy), rel=1e-13)


def test_poisson_fft_equals_direct_sum(orc):
    rng = np.random.Generator(np.random.PCG64(3))
    for nx, ny, hx, hy in ((16, 16, 1.0, 1.0), (32, 16, 2.0, 0.7), (32, 32, 15e-3, 15e-3)):
        g = make_grid(nx, hx, ny=ny, half_y=hy)
        Q = rng_uniform(rng, nx * ny).reshape(ny, nx)
        Q[rng_uniform(rng, nx * ny).reshape(ny, nx) < 0.5] = 0.0
        ud = orc.poisson(Q, g, 1000.0, direct=True)
        uf = orc.poisson(Q, g, 1000.0, direct=False)
        assert abs(ud - uf).max() < 1e-13 * abs(ud).max()


def test_poisson_direct_is_the_written_sum(orc):
    """u[j,i] = (1/N) sum G_cell((i-i')dx,(j-j')dy) Q[j',i'] evaluated with numpy on a 6x5 grid."""
    g = dict(nx=6, ny=5, xmin=0.0, xmax=2.5, ymin=-1.0, ymax=1.0)
    dx, dy = 0.5, 0.5
    rng = np.random.Generator(np.random.PCG64(8))
    Q = rng_uniform(rng, 30).reshape(5, 6)
    u = orc.poisson(Q, g, 7.0, direct=True)
    want = np.zeros((5, 6))
    for j in range(5):
        for i in range(6):
            want[j, i] = sum(orc.green_cell((i - ii) * dx, (j - jj) * dy, dx, dy) * Q[jj, ii]
                             for jj in range(5) for ii in range(6)) / 7.0
    assert u == pytest.approx(want, rel=1e-13)


# ---------------------------------------------------------------- field of round beams (P4, P5, P5b)
def _radial_field_error(orc, n, dens, er, half=15e-3, rmin=0.0, rmax=1e9):
    g = make_grid(n, half)
    xs, ys = nodes(g)
    X, Y = np.meshgrid(xs, ys)
    R = np.hypot(X, Y)
    dx = 2 * half / (n - 1)
    f = dens(R)
    Q = f * dx * dx                                   # charge per node for N = 1
    u = orc.poisson(Q, g, 1.0)
    Ex, Ey = orc.field(u, g)
    with np.errstate(invalid="ignore", divide="ignore"):
        Er = np.where(R > 0, (Ex * X + Ey * Y) / R, 0.0)
        Et = np.where(R > 0, (-Ex * Y + Ey * X) / R, 0.0)
    interior = (np.abs(X) < half - 2 * dx) & (np.abs(Y) < half - 2 * dx) & (R >= rmin) & (R <= rmax) & (R > 0)
    want = er(np.where(R > 0, R, 1.0))
    scale = abs(want[interior]).max()
    return abs(Er - want)[interior].max() / scale, abs(Et)[interior].max() / scale, Q.sum()


def test_field_of_round_gaussian_beam(orc):
    """E~_r = (1 - exp(-r^2/2 sigma^2))/(2 pi r)  (north_star closed form); O(h^2) convergence."""
    s = 3e-3
    dens = lambda R: np.exp(-R * R / (2 * s * s)) / (2 * math.pi * s * s)
    er = lambda R: (1 - np.exp(-R * R / (2 * s * s))) / (2 * math.pi * R)
    e64, t64, q64 = _radial_field_error(orc, 64, dens, er)
    e128, t128, q128 = _radial_field_error(orc, 128, dens, er)
    assert q64 == pytest.approx(1.0, abs=1e-5) and q128 == pytest.approx(1.0, abs=1e-5)
    assert e64 < 7e-3 and e128 < 1.8e-3               # 5.3e-3, 1.3e-3
    assert 3.0 < e64 / e128 < 5.0                     # second order
    assert t64 < 1e-3 and t128 < 3e-4                 # no azimuthal field


def test_field_of_uniform_round_beam(orc):
    """E~_r = r/(2 pi a^2) inside, 1/(2 pi r) outside (north_star closed form)."""
    a = 7e-3
    dens = lambda R: (R <= a) / (math.pi * a * a)
    er = lambda R: np.where(R <= a, R / (2 * math.pi * a * a), 1 / (2 * math.pi * R))
    e_in, _, q = _radial_field_error(orc, 128, dens, er, rmax=0.8 * a)
    e_out, _, _ = _radial_field_error(orc, 128, dens, er, rmin=1.2 * a)
    # the staircase disc holds q != 1 of the charge; the outside field scales with it
    assert e_in < 2e-2 and abs(e_out - abs(q - 1)) < 5e-3


def test_field_of_round_waterbag_beam(orc):
    """cfg2 shape: 4D waterbag projects to density (2/(pi a^2)) (1 - r^2/a^2); enclosed fraction
    2 (r/a)^2 - (r/a)^4 => E~_r = that/(2 pi r)."""
    a = 9e-3
    dens = lambda R: np.where(R <= a, 2 / (math.pi * a * a) * (1 - R * R / (a * a)), 0.0)
    er = lambda R: np.where(R <= a, 2 * (R / a) ** 2 - (R / a) ** 4, 1.0) / (2 * math.pi * R)
    e, t, q = _radial_field_error(orc, 128, dens, er)
    assert q == pytest.approx(1.0, abs=2e-3)
    assert e < 4e-3 and t < 5e-4


# ---------------------------------------------------------------- self-consistency and brute force (P7, P8)
def _kick(orc, x, y, g, L=1.0, direct=False):
    p = dict(x=np.array(x, np.float64), px=np.zeros(len(x)), y=np.array(y, np.float64), py=np.zeros(len(x)),
             sigma=None, psigma=None)
    w = orc.scnode(p, g, BEAM, L, direct)
    b = orc.beam_struct(BEAM)
    c = b.kappa * BEAM["line_density"] * L
    return p["px"] / c, p["py"] / c, w


def test_zero_self_force_and_momentum_conservation(orc):
    g = make_grid(64, 15e-3)
    dx = 30e-3 / 63
    ex, ey, _ = _kick(orc, [1.234e-3], [-2.345e-3], g)
    assert abs(ex[0]) < 1e-12 / dx and abs(ey[0]) < 1e-12 / dx     # scale of a one-cell field: 1/(2 pi dx)
    rng = np.random.Generator(np.random.PCG64(21))
    n = 5000
    x, y = 2e-3 * rng_normal(rng, n), 2e-3 * rng_normal(rng, n)
    ex, ey, w = _kick(orc, x, y, g)
    assert w.n_inside == n
    assert abs(ex.sum()) < 1e-12 * abs(ex).sum() and abs(ey.sum()) < 1e-12 * abs(ey).sum()


def test_grid_field_against_direct_pairwise_sum(orc):
    """E~(r_i) = (1/N) sum_j (r_i - r_j)/(2 pi |r_i - r_j|^2): direct 2D log-potential sum over
    particles separated by >= 8 cells (PIC resolves nothing below a cell; 0.6 % at 8)."""
    g = make_grid(128, 15e-3)
    dx = 30e-3 / 127
    rng = np.random.Generator(np.random.PCG64(4))
    pts = []
    while len(pts) < 12:
        c = (rng_uniform(rng, 2) - 0.5) * 24e-3
        if all(np.hypot(*(c - q)) >= 10 * dx for q in pts):
            pts.append(c)
    pts = np.array(pts)
    ex, ey, _ = _kick(orc, pts[:, 0], pts[:, 1], g)
    n = len(pts)
    for i in range(n):
        d = pts[i] - np.delete(pts, i, axis=0)
        r2 = (d * d).sum(axis=1)
        want = (d / (2 * math.pi * r2[:, None])).sum(axis=0) / n
        scale = np.hypot(*want)
        assert math.hypot(ex[i] - want[0], ey[i] - want[1]) < 0.012 * scale + 2e-3 / (2 * math.pi * 10 * dx) / n
    # direct-sum Poisson and FFT Poisson give the same kicks
    ex2, ey2, _ = _kick(orc, pts[:, 0], pts[:, 1], make_grid(32, 15e-3), direct=True)
    ex3, ey3, _ = _kick(orc, pts[:, 0], pts[:, 1], make_grid(32, 15e-3), direct=False)
    assert ex2 == pytest.approx(ex3, rel=1e-11, abs=1e-11 * abs(ex2).max())
    assert ey2 == pytest.approx(ey3, rel=1e-11, abs=1e-11 * abs(ey2).max())


def test_gather_is_bilinear_interpolation(orc):
    g = dict(nx=5, ny=4, xmin=0.0, xmax=4.0, ymin=0.0, ymax=3.0)
    xs, ys = nodes(g)
    X, Y = np.meshgrid(xs, ys)
    Ex, Ey = 2 + 3 * X - Y + 0.5 * X * Y, -1 + X + 2 * Y          # bilinear functions are reproduced exactly
    for x, y in ((0.3, 0.2), (3.9, 2.9), (2.0, 1.0), (0.0, 0.0)):
        ins, ex, ey = orc.gather(Ex, Ey, g, x, y)
        assert ins and ex == pytest.approx(2 + 3 * x - y + 0.5 * x * y, rel=1e-14) and ey == pytest.approx(-1 + x + 2 * y, rel=1e-14)
    assert orc.gather(Ex, Ey, g, 4.0, 1.0) == (False, 0.0, 0.0)
    assert orc.gather(Ex, Ey, g, -0.1, 1.0) == (False, 0.0, 0.0)


def test_field_is_central_difference_of_potential(orc):
    g = dict(nx=6, ny=5, xmin=0.0, xmax=2.5, ymin=0.0, ymax=4.0)
    xs, ys = nodes(g)
    X, Y = np.meshgrid(xs, ys)
    u = X ** 2 + 3 * Y ** 2 + X * Y                                   # quadratic: central differences exact inside
    Ex, Ey = orc.field(u, g)
    assert Ex[:, 1:-1] == pytest.approx(-(2 * X + Y)[:, 1:-1], rel=1e-13)
    assert Ey[1:-1, :] == pytest.approx(-(6 * Y + X)[1:-1, :], rel=1e-13)
    assert Ex[:, 0] == pytest.approx(-(u[:, 1] - u[:, 0]) / 0.5) and Ex[:, -1] == pytest.approx(-(u[:, -1] - u[:, -2]) / 0.5)
    assert Ey[0, :] == pytest.approx(-(u[1, :] - u[0, :]) / 1.0) and Ey[-1, :] == pytest.approx(-(u[-1, :] - u[-2, :]) / 1.0)


# ---------------------------------------------------------------- whole node scaling: eq. 30 (P6)
def test_small_amplitude_tune_shift_matches_eq30_form(orc):
    """Smooth-focusing ring (constant beta, round matched Gaussian coasting beam): the tune shift of a
    small-amplitude particle is  -r_c lambda C / (4 pi beta0^2 gamma0^3 eps)  -- eq. 30
    with N_ppb h / B_f -> lambda C.  Pins kappa, the lambda L scaling, the sign of the kick, the Poisson
    normalisation, the field and the gather end to end."""
    b = orc.beam_struct(BEAM)
    beta, nseg, nu0 = 10.0, 16, 3.21
    C_ = 2 * math.pi * beta * 3.0 * 0 + 160.0
    Lseg = C_ / nseg
    mu = 2 * math.pi * nu0 / nseg
    Mrot = [math.cos(mu), beta * math.sin(mu), -math.sin(mu) / beta, math.cos(mu)]
    sig = 3e-3
    eps = sig * sig / beta
    lam = 1e11
    want = -b.r_c * lam * C_ / (4 * math.pi * b.beta0 ** 2 * b.gamma0 ** 3 * eps)
    assert -0.04 < want < -0.02
    # the same thing without the first-order approximation: 16 x (rotation, thin defocusing kick with
    # the central gradient of a round Gaussian, E~_r -> r/(4 pi sigma^2))
    gk = b.kappa * lam * Lseg / (4 * math.pi * sig * sig)
    KR = np.array([[1, 0], [gk, 1]]) @ np.array([[Mrot[0], Mrot[1]], [Mrot[2], Mrot[3]]])
    frac = lambda M: math.acos(0.5 * np.trace(M)) / (2 * math.pi)     # fractional tune, nu0 = 3 + 0.21
    want_exact = frac(np.linalg.matrix_power(KR, nseg)) - (nu0 - 3)
    assert want_exact == pytest.approx(want, rel=0.03)      # eq. 30 is first order in the kick
    rows = [(LINMAP, 0, Mrot + Mrot + [Lseg]), (SCNODE, 0, [Lseg])] * nseg
    kind, ipar, par = rows_to_arrays(rows)
    rng = np.random.Generator(np.random.PCG64(17))
    n = 200_000
    d = 1e-6                                     # probe amplitude << sigma
    p = dict(x=sig * rng_normal(rng, n), px=sig / beta * rng_normal(rng, n), y=sig * rng_normal(rng, n),
             py=sig / beta * rng_normal(rng, n), sigma=None, psigma=None)
    probes = {"x": [d, -d, 0, 0, 0, 0, 0, 0], "px": [0, 0, d / beta, -d / beta, 0, 0, 0, 0],
              "y": [0, 0, 0, 0, d, -d, 0, 0], "py": [0, 0, 0, 0, 0, 0, d / beta, -d / beta]}
    for k in probes:
        p[k][:8] = probes[k]
    g = make_grid(128, 5 * sig)
    beam = dict(BEAM, line_density=lam)
    out, _ = orc.track(kind, ipar, par, [g], beam, p, n_turns=1)
    Mx = np.array([[(out["x"][0] - out["x"][1]) / (2 * d), (out["x"][2] - out["x"][3]) / (2 * d / beta)],
                   [(out["px"][0] - out["px"][1]) / (2 * d), (out["px"][2] - out["px"][3]) / (2 * d / beta)]])
    My = np.array([[(out["y"][4] - out["y"][5]) / (2 * d), (out["y"][6] - out["y"][7]) / (2 * d / beta)],
                   [(out["py"][4] - out["py"][5]) / (2 * d), (out["py"][6] - out["py"][7]) / (2 * d / beta)]])
    for M in (Mx, My):
        # (nu0 >> |want| keeps the injected beam matched: the envelope does not breathe)
        assert frac(M) - (nu0 - 3) == pytest.approx(want_exact, rel=0.03)
        assert frac(M) - (nu0 - 3) == pytest.approx(want, rel=0.05)
