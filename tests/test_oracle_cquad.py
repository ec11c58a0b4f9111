"""Pins of the oracle's chromatic thick quadrupole (N3: eq. 6 per particle)."""
import numpy as np
import pytest
from scipy.integrate import solve_ivp

GAMMA0 = 4.1973667744


def particles(n, seed, with_ps=True):
    rng = np.random.Generator(np.random.PCG64(seed))
    p = dict(x=3e-3 * rng.standard_normal(n), px=3e-4 * rng.standard_normal(n), y=3e-3 * rng.standard_normal(n),
             py=3e-4 * rng.standard_normal(n), sigma=10.0 * rng.standard_normal(n),
             psigma=(5e-3 * rng.standard_normal(n) if with_ps else np.zeros(n)))
    return p


@pytest.mark.parametrize("k1,L", [(0.115, 1.5), (-0.115, 1.5), (2.3, 0.4), (-0.02, 6.0)])
def test_cquad_against_ode_integration_of_h_approx(orc, k1, L):
    """Hamilton's equations of H_approx with e A_s/p0 = -k1 (x^2 - y^2)/2:
    x' = px (1 - ps), px' = -k1 x, y' = py (1 - ps), py' = +k1 y, sigma' = ps/gamma0^2 - (px^2 + py^2)/2, ps' = 0."""
    p = particles(12, 21)
    want = {k: v.copy() for k, v in p.items()}
    for i in range(12):
        ps = p["psigma"][i]
        def rhs(s, q):
            return [q[1] * (1 - ps), -k1 * q[0], q[3] * (1 - ps), k1 * q[2], ps / GAMMA0 ** 2 - 0.5 * (q[1] ** 2 + q[3] ** 2)]
        sol = solve_ivp(rhs, (0.0, L), [p["x"][i], p["px"][i], p["y"][i], p["py"][i], p["sigma"][i]], rtol=1e-13, atol=1e-18,
                        method="DOP853")
        for j, k in enumerate(("x", "px", "y", "py", "sigma")):
            want[k][i] = sol.y[j, -1]
    orc.cquad(p, k1, L, GAMMA0)
    for k in ("x", "px", "y", "py"):
        assert np.abs(p[k] - want[k]).max() < 1e-11 * np.abs(want[k]).max()
    assert np.abs(p["sigma"] - want["sigma"]).max() < 1e-12 * np.abs(want["sigma"]).max()
    assert np.array_equal(p["psigma"], want["psigma"])


def test_cquad_on_momentum_is_the_linear_quadrupole_map(orc):
    """At psigma = 0 eq. 6 is the matrix of the QUAD/LINMAP row (x, px, y, py); sigma differs by the
    -1/2 int (px^2 + py^2) term that the linear row leaves out (a second-order path length)."""
    for k1 in (0.115, -0.115):
        p = particles(50, 22, with_ps=False)
        q = {k: v.copy() for k, v in p.items()}
        orc.cquad(p, k1, 1.5, GAMMA0)
        orc.linmap(q, orc.quad_matrix(k1, 1.5), 1.5, GAMMA0)
        for k in ("x", "px", "y", "py"):
            assert np.abs(p[k] - q[k]).max() < 1e-14 * np.abs(q[k]).max()
        assert np.all(p["sigma"] <= q["sigma"]) and np.abs(p["sigma"] - q["sigma"]).max() < 1e-5


def test_cquad_is_symplectic_and_reduces_to_the_drift(orc):
    """6D Jacobian by central differences: J^T S J = S.  k1 -> 0: the H0 drift (eq. 7)."""
    base = particles(1, 23)
    names = ("x", "px", "y", "py", "sigma", "psigma")
    h = np.array([1e-6, 1e-7, 1e-6, 1e-7, 1e-3, 1e-6])
    J = np.zeros((6, 6))
    for c, nm in enumerate(names):
        out = []
        for sgn in (+1, -1):
            p = {k: v.copy() for k, v in base.items()}
            p[nm] = p[nm] + sgn * h[c]
            orc.cquad(p, 0.8, 1.2, GAMMA0)
            out.append(np.array([p[k][0] for k in names]))
        J[:, c] = (out[0] - out[1]) / (2 * h[c])
    S = np.zeros((6, 6))
    for k in range(3):
        S[2 * k, 2 * k + 1], S[2 * k + 1, 2 * k] = 1.0, -1.0
    assert np.abs(J.T @ S @ J - S).max() < 1e-7
    p = particles(40, 24)
    q = {k: v.copy() for k, v in p.items()}
    orc.cquad(p, 1e-13, 2.0, GAMMA0)
    orc.drift(q, 2.0, GAMMA0)
    for k in names:
        assert np.abs(p[k] - q[k]).max() <= 1e-11 * max(np.abs(q[k]).max(), 1e-300)
    p0 = particles(5, 25)
    q0 = {k: v.copy() for k, v in p0.items()}
    orc.cquad(p0, 0.0, 2.0, GAMMA0)
    orc.drift(q0, 2.0, GAMMA0)
    for k in names:
        assert np.array_equal(p0[k], q0[k])


def test_cquad_row_in_the_tracking_loop_and_chromaticity(orc):
    """A ring of CQUAD FODO cells: off-momentum particles see k1 (1 - ps): the tune drops with ps by the natural
    chromaticity, xi = -(1/4 pi) sum(beta k1 l) per cell in thin-lens terms -- checked in sign and size."""
    from workloads import CQUAD, DRIFT, rows_to_arrays, make_beam_spec
    kq, lq, ld = 0.6, 0.3, 2.0
    cell = [(CQUAD, 0, [kq, lq]), (DRIFT, 0, [ld]), (CQUAD, 0, [-kq, lq]), (DRIFT, 0, [ld])]
    kind, ipar, par = rows_to_arrays(cell)
    beam = make_beam_spec(line_density=0.0, circumference=2 * (lq + ld))
    def tune(ps):
        # one-cell matrix in x from two tiny displacements, cos(mu) = trace / 2
        cols = []
        for dx, dpx in ((1e-7, 0.0), (0.0, 1e-8)):
            p = dict(x=np.array([dx]), px=np.array([dpx]), y=np.zeros(1), py=np.zeros(1), sigma=np.zeros(1),
                     psigma=np.array([ps]))
            out, _ = orc.track(kind, ipar, par, [], beam, p, n_turns=1)
            cols.append([out["x"][0] / (dx or 1.0) if dx else out["x"][0] / dpx, out["px"][0] / (dx or 1.0) if dx else out["px"][0] / dpx])
        m11, m22 = cols[0][0], cols[1][1]
        return np.arccos(0.5 * (m11 + m22)) / (2 * np.pi)
    q0, qp, qm = tune(0.0), tune(1e-3), tune(-1e-3)
    xi = (qp - qm) / 2e-3
    assert 0.05 < q0 < 0.45
    assert xi < 0.0 and 0.3 * q0 < -xi < 3.0 * q0          # natural chromaticity of a FODO cell is about -tune


# ---------------------------------------------------------------- thick sextupole, eqs. 7-8
def _sext_ode(p, i, k2, L):
    ps = p["psigma"][i]
    def rhs(s, q):   # H_approx with V = k2 (x^3 - 3 x y^2)/6:  px' = -k2 (x^2 - y^2)/2, py' = k2 x y
        return [q[1] * (1 - ps), -0.5 * k2 * (q[0] ** 2 - q[2] ** 2), q[3] * (1 - ps), k2 * q[0] * q[2],
                ps / GAMMA0 ** 2 - 0.5 * (q[1] ** 2 + q[3] ** 2)]
    sol = solve_ivp(rhs, (0.0, L), [p["x"][i], p["px"][i], p["y"][i], p["py"][i], p["sigma"][i]], rtol=1e-13, atol=1e-18,
                    method="DOP853")
    return sol.y[:, -1]


def test_sext_converges_to_the_flow_of_h_approx(orc):
    """eq. 8 with a = (1 - 1/sqrt 3)/2, b = 1/2, c = 1/sqrt 3 (ref [7]: the kicks sit at the two Gauss points of the
    magnet) against the ODE of H_approx: as a splitting it is second order -- the one-step error falls like L^3 in the
    momenta and L^4 in the positions when L is halved (measured 8 and 16) -- with a small constant: several times
    closer to the flow than the drift-kick-drift leapfrog of the same cost class."""
    from workloads import DRIFT, MULT, rows_to_arrays, make_beam_spec
    k2 = 40.0
    beam = make_beam_spec(line_density=0.0, circumference=10.0)
    errs, leap = [], []
    for L in (0.8, 0.4):
        p = particles(8, 31)
        want = np.array([_sext_ode(p, i, k2, L) for i in range(8)])
        frog, _ = orc.track(*rows_to_arrays([(DRIFT, 0, [0.5 * L]), (MULT, 2, [k2 * L, 0.0]), (DRIFT, 0, [0.5 * L])]), [], beam, p,
                            n_turns=1)
        orc.sext(p, k2, L, GAMMA0)
        got = np.stack([p["x"], p["px"], p["y"], p["py"]], axis=1)
        lf = np.stack([frog["x"], frog["px"], frog["y"], frog["py"]], axis=1)
        scale = np.abs(want[:, :4]).max(axis=0)
        errs.append(np.abs(got - want[:, :4]).max(axis=0) / scale)
        leap.append(np.abs(lf - want[:, :4]).max(axis=0) / scale)
    errs, leap = np.array(errs), np.array(leap)
    assert errs[1].max() < 3e-4
    ratio = errs[0] / errs[1]
    assert np.all(ratio[[1, 3]] > 6.0) and np.all(ratio[[1, 3]] < 12.0)        # momenta: L^3
    assert np.all(ratio[[0, 2]] > 12.0) and np.all(ratio[[0, 2]] < 24.0)       # positions: L^4
    assert np.all(leap[1] > 2.0 * errs[1])


def test_sext_equals_its_five_rows_and_the_drift_at_zero_strength(orc):
    from workloads import DRIFT, MULT, SEXT, rows_to_arrays, make_beam_spec
    a, b, c = 0.5 * (1 - 1 / np.sqrt(3.0)), 0.5, 1 / np.sqrt(3.0)
    k2, L = 7.0, 0.6
    beam = make_beam_spec(line_density=0.0, circumference=10.0)
    p = particles(30, 32)
    five = [(DRIFT, 0, [a * L]), (MULT, 2, [k2 * (b * L), 0.0]), (DRIFT, 0, [c * L]), (MULT, 2, [k2 * (b * L), 0.0]),
            (DRIFT, 0, [a * L])]
    o5, _ = orc.track(*rows_to_arrays(five), [], beam, p, n_turns=1)
    o1, _ = orc.track(*rows_to_arrays([(SEXT, 0, [k2, L])]), [], beam, p, n_turns=1)
    for k in o1:
        assert np.array_equal(o1[k], o5[k])
    q = {k: v.copy() for k, v in p.items()}
    r = {k: v.copy() for k, v in p.items()}
    orc.sext(q, 0.0, L, orc.beam_struct(beam).gamma0)
    orc.drift(r, L, orc.beam_struct(beam).gamma0)
    for k in q:
        assert np.abs(q[k] - r[k]).max() <= 1e-15 * max(np.abs(r[k]).max(), 1e-300)


# ---------------------------------------------------------------- exact drift (section III.A at B = 0)
BETA0 = 0.9712051827


def test_xdrift_is_straight_line_kinematics_in_the_lab_frame(orc):
    """Independent route: build the particle's lab-frame velocity from (px, py, psigma), fly it to the plane z = L in
    Cartesian coordinates and time, then convert back with sigma = s - beta0 c t."""
    p = particles(200, 41)
    p["px"] *= 30.0; p["py"] *= 30.0                      # 10 mrad: far from the paraxial limit
    L = 3.7
    E0, m = 1.0 / np.sqrt(1.0 - BETA0 ** 2), 1.0           # units m c^2 = 1: E0 = gamma0
    p0 = BETA0 * E0
    E = E0 * (1.0 + BETA0 ** 2 * p["psigma"])              # psigma = (E - E0)/(beta0^2 E0)
    pt = np.sqrt(E ** 2 - m ** 2)                          # |P| c
    Px, Py = p0 * p["px"], p0 * p["py"]
    Pz = np.sqrt(pt ** 2 - Px ** 2 - Py ** 2)
    vx, vy, vz = Px / E, Py / E, Pz / E                    # velocity / c
    ct = L / vz
    want = dict(x=p["x"] + vx * ct, y=p["y"] + vy * ct, sigma=p["sigma"] + L - BETA0 * ct)
    q = {k: v.copy() for k, v in p.items()}
    orc.xdrift(q, L, BETA0)
    for k in ("x", "y", "sigma"):
        assert np.abs(q[k] - want[k]).max() < 1e-13 * max(np.abs(want[k]).max(), 1.0)
    for k in ("px", "py", "psigma"):
        assert np.array_equal(q[k], p[k])


def test_xdrift_against_the_exact_hamiltonian_and_the_h0_drift(orc):
    """Hamilton's equations of eq. 1 with h = 0, A_s = 0:  x' = px/pz, y' = py/pz, sigma' = 1 - (1 + beta0^2 ps)/pz,
    pz = sqrt((1+delta)^2 - px^2 - py^2); and the H0 drift of eq. 7 is its expansion to second order."""
    p = particles(10, 42)
    L = 2.0
    want = {k: v.copy() for k, v in p.items()}
    for i in range(10):
        ps, px, py = p["psigma"][i], p["px"][i], p["py"][i]
        pz = np.sqrt(1 + 2 * ps + BETA0 ** 2 * ps ** 2 - px ** 2 - py ** 2)
        sol = solve_ivp(lambda s, q: [px / pz, py / pz, 1 - (1 + BETA0 ** 2 * ps) / pz], (0.0, L),
                        [p["x"][i], p["y"][i], p["sigma"][i]], rtol=1e-13, atol=1e-18, method="DOP853")
        want["x"][i], want["y"][i], want["sigma"][i] = sol.y[:, -1]
    q = {k: v.copy() for k, v in p.items()}
    orc.xdrift(q, L, BETA0)
    for k in ("x", "y", "sigma"):
        assert np.abs(q[k] - want[k]).max() < 1e-12 * max(np.abs(want[k]).max(), 1.0)
    r = {k: v.copy() for k, v in p.items()}
    orc.drift(r, L, GAMMA0)
    # H_approx keeps H to second order: x differs by ~L px ps^2 (third order), sigma' by the next term of the expansion
    # of 1 - (1 + beta0^2 ps)/(1 + delta), -3 ps^2/(2 gamma0^2), which dominates at ps ~ 5e-3
    assert np.abs(q["x"] - r["x"]).max() < 5e-8 and np.abs(q["y"] - r["y"]).max() < 5e-8
    lead = -1.5 * L * p["psigma"] ** 2 / GAMMA0 ** 2
    assert np.abs((q["sigma"] - r["sigma"]) - lead).max() < 0.05 * np.abs(lead).max()
    assert np.abs(q["x"] - r["x"]).max() > 1e-12          # ... and they are not the same map


# ---------------------------------------------------------------- exact sector bend (section III.A, eqs. 2-5)
@pytest.mark.parametrize("L,h", [(2.0, 0.05), (5.85, 1.0 / 89.381), (1.0, -0.2)])
def test_sbend_against_the_exact_hamiltonian(orc, L, h):
    """Hamilton's equations of eq. 1 with curvature h and the sector dipole's e A_s/p0 = -(h x + h^2 x^2/2):
    x' = (1+hx) px/pz, px' = h (pz - 1 - h x), y' = (1+hx) py/pz, py' = 0, sigma' = 1 - (1+hx)(1 + beta0^2 ps)/pz."""
    p = particles(10, 51)
    want = {k: v.copy() for k, v in p.items()}
    for i in range(10):
        ps, py = p["psigma"][i], p["py"][i]
        d2 = 1 + 2 * ps + BETA0 ** 2 * ps ** 2
        def rhs(s, q):
            pz = np.sqrt(d2 - q[1] ** 2 - py ** 2)
            return [(1 + h * q[0]) * q[1] / pz, h * (pz - 1 - h * q[0]), (1 + h * q[0]) * py / pz,
                    1 - (1 + h * q[0]) * (1 + BETA0 ** 2 * ps) / pz]
        sol = solve_ivp(rhs, (0.0, L), [p["x"][i], p["px"][i], p["y"][i], p["sigma"][i]], rtol=1e-13, atol=1e-18, method="DOP853")
        want["x"][i], want["px"][i], want["y"][i], want["sigma"][i] = sol.y[:, -1]
    orc.sbend(p, L, h, BETA0)
    for k in ("x", "px", "y", "sigma"):
        assert np.abs(p[k] - want[k]).max() < 2e-11 * max(np.abs(want[k]).max(), 1e-3), k
    assert np.array_equal(p["py"], want["py"]) and np.array_equal(p["psigma"], want["psigma"])


def test_sbend_reference_orbit_matrix_dispersion_and_drift_limit(orc):
    L, h = 3.0, 0.1
    th, rho = L * h, 1.0 / h
    z = dict(x=np.zeros(1), px=np.zeros(1), y=np.zeros(1), py=np.zeros(1), sigma=np.zeros(1), psigma=np.zeros(1))
    orc.sbend(z, L, h, BETA0)
    for k in z:
        assert abs(z[k][0]) < 1e-15                         # the reference particle stays the reference particle
    e = 1e-7                                               # first order: the textbook sector-bend matrix and dispersion
    cols = {}
    for nm in ("x", "px", "psigma"):
        q = {k: np.zeros(1) for k in z}
        q[nm] = np.array([e])
        orc.sbend(q, L, h, BETA0)
        cols[nm] = (q["x"][0] / e, q["px"][0] / e)
    assert cols["x"] == pytest.approx((np.cos(th), -np.sin(th) / rho), rel=1e-6)
    assert cols["px"] == pytest.approx((rho * np.sin(th), np.cos(th)), rel=1e-6)
    # delta = psigma to first order: D = rho (1 - cos theta), D' = sin theta
    assert cols["psigma"] == pytest.approx((rho * (1 - np.cos(th)), np.sin(th)), rel=1e-5)
    p = particles(30, 52)
    q = {k: v.copy() for k, v in p.items()}
    orc.sbend(p, 2.0, 1e-7, BETA0)                          # a 1e7 m radius: the drift, up to h L^2 (x/rho, delta) ~ 1e-9
    orc.xdrift(q, 2.0, BETA0)                              # and the rounding of rho (1 - ...) ~ 1e-9
    for k in ("x", "y", "sigma"):
        assert np.abs(p[k] - q[k]).max() < 2e-8, k
    assert np.abs(p["px"] - q["px"]).max() < 1e-8              # h L delta = 2e-7 x 1e-2
    r = {k: v.copy() for k, v in q.items()}
    orc.sbend(r, 0.0, 0.3, BETA0)                          # zero length: identity
    for k in r:
        assert np.abs(r[k] - q[k]).max() < 1e-14 * max(np.abs(q[k]).max(), 1.0), k   # a few ulp of rho (1 + hx - 1)
