/*
 * sc_oracle.c -- ORACLE (test infrastructure, NOT the product).  See sc_oracle.h.
 *
 * Each function cites the PAPER.md passage (line, section, equation) it restates, or the
 * SURVEY.md 8(c) reading (A1..A18) taken where the paper is silent.  No blocking, fusion or
 * reordering beyond what the cited definition states: one table row at a time, one particle at
 * a time, in index order.
 */
#include "sc_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

#define ORC_PI 3.14159265358979323846264338327950288

/* ------------------------------------------------------------------------------------------
 * Reference particle.  gamma0 = 1 + T/m, beta0 = sqrt(1 - 1/gamma0^2), E0 = gamma0 m.
 * r_c = q^2 e^2 / (4 pi eps0 m c^2) = q^2 * (e/(4 pi eps0)) [V m] / (m c^2 [eV])   (A1: CODATA,
 * not the 1.547e-18 printed at PAPER.md:354).  kappa = 4 pi r_c/(beta0^2 gamma0^3) is the
 * prefactor e^2/(eps0 m gamma0^3 beta0^2 c^2) of eq. 11-12 for a potential
 * normalised as  laplace(u~) = -f, integral f = 1  (A4, A5).
 * ---------------------------------------------------------------------------------------- */
void orc_beam_init(orc_beam* b, double kinetic_eV, double mass_eV, int charge,
                   double line_density, double n_real, double circumference)
{
    const double e_charge = 1.602176634e-19;      /* C, exact (SI 2019)   */
    const double eps0 = 8.8541878128e-12;         /* F/m, CODATA 2018     */
    double k_e = e_charge / (4.0 * ORC_PI * eps0);  /* e/(4 pi eps0) in V m */
    b->gamma0 = 1.0 + kinetic_eV / mass_eV;
    b->beta0 = sqrt(1.0 - 1.0 / (b->gamma0 * b->gamma0));
    b->E0_eV = b->gamma0 * mass_eV;
    b->charge = charge;
    b->r_c = (double)charge * (double)charge * k_e / mass_eV;
    b->kappa = 4.0 * ORC_PI * b->r_c / (b->beta0 * b->beta0 * b->gamma0 * b->gamma0 * b->gamma0);
    b->line_density = line_density;
    b->n_real = n_real;
    b->circumference = circumference;
}

/* ------------------------------------------------------------------------------------------
 * DRIFT: the exact flow of H0 = (px^2+py^2)/2 (1 - psigma) + psigma^2/(2 gamma0^2)
 * (eq. 7; A3: the H0 drift is used for drift spaces):
 *   x'     = dH0/dpx     = px (1 - psigma)
 *   sigma' = dH0/dpsigma = psigma/gamma0^2 - (px^2+py^2)/2       (also PAPER.md:119)
 * px, py, psigma are constants of H0.
 * ---------------------------------------------------------------------------------------- */
void orc_drift(int64_t n, double* x, double* px, double* y, double* py, double* sg, double* ps,
               double L, double gamma0)
{
    for (int64_t i = 0; i < n; i++) {
        double p = ps ? ps[i] : 0.0;
        double d = 1.0 - p;
        x[i] = x[i] + L * d * px[i];
        y[i] = y[i] + L * d * py[i];
        if (sg) sg[i] = sg[i] + L * (p / (gamma0 * gamma0) - 0.5 * (px[i] * px[i] + py[i] * py[i]));
    }
}

/* ------------------------------------------------------------------------------------------
 * Thick quadrupole matrix: eq. 6 at psigma = 0, phi = sqrt(|k1|) L.
 * M = {m11,m12,m21,m22 of the x plane, then of the y plane}.  k1 > 0 focuses x (cos/sin) and
 * defocuses y (cosh/sinh); k1 < 0 swaps the planes; k1 = 0 is a drift of length L.
 * ---------------------------------------------------------------------------------------- */
void orc_quad_matrix(double k1, double L, double M[8])
{
    if (k1 == 0.0) {
        M[0] = 1; M[1] = L; M[2] = 0; M[3] = 1; M[4] = 1; M[5] = L; M[6] = 0; M[7] = 1;
        return;
    }
    double k = fabs(k1), rk = sqrt(k), phi = rk * L;
    double F[4] = { cos(phi), sin(phi) / rk, -rk * sin(phi), cos(phi) };
    double D[4] = { cosh(phi), sinh(phi) / rk, rk * sinh(phi), cosh(phi) };
    const double* X = k1 > 0 ? F : D;
    const double* Y = k1 > 0 ? D : F;
    for (int i = 0; i < 4; i++) { M[i] = X[i]; M[4 + i] = Y[i]; }
}

/* LINMAP: uncoupled 2x2 (+) 2x2 map; sigma advances by L psigma/gamma0^2 (SURVEY 8a row T2:
 * the on-momentum linear form of eq. 6; the -1/2 int(px^2+py^2) term of PAPER.md:119 belongs to
 * the chromatic variant N3 and is not part of this row). */
void orc_linmap(int64_t n, double* x, double* px, double* y, double* py, double* sg, double* ps,
                const double M[8], double L, double gamma0)
{
    for (int64_t i = 0; i < n; i++) {
        double x0 = x[i], p0 = px[i], y0 = y[i], q0 = py[i];
        x[i] = M[0] * x0 + M[1] * p0;
        px[i] = M[2] * x0 + M[3] * p0;
        y[i] = M[4] * y0 + M[5] * q0;
        py[i] = M[6] * y0 + M[7] * q0;
        if (sg) sg[i] = sg[i] + L * (ps[i] / (gamma0 * gamma0));
    }
}

/* ------------------------------------------------------------------------------------------
 * N3: thick quadrupole under H_approx, PER PARTICLE (eq. 6 as printed): the focusing
 * strength seen by a particle is k1 (1 - psigma), w = sqrt(|k1| (1 - psigma)),
 *   focusing plane:    q(L) = q0 cos wL + sqrt((1-ps)/|k1|) p0 sin wL,  p(L) = p0 cos wL - sqrt(|k1|/(1-ps)) q0 sin wL
 *   defocusing plane:  the same with cosh, sinh and a + sign in p(L)
 *   sigma(L) = sigma0 + psigma L/gamma0^2 - 1/2 int_0^L (px^2 + py^2) ds', psigma unchanged.
 * The integral is written out in closed form: with p(s) = p0 cos ws - r sin ws, r = q0 |k1|/w,
 *   int p^2 = L (p0^2 + r^2)/2 + (p0^2 - r^2) sin wL cos wL/(2w) - p0 r sin^2 wL / w,
 * and with p(s) = p0 cosh ws + r sinh ws,
 *   int p^2 = L (p0^2 - r^2)/2 + (p0^2 + r^2) sinh wL cosh wL/(2w) + p0 r sinh^2 wL / w.
 * k1 > 0 focuses x (sign convention of PAPER.md:99); k1 = 0 is the H0 drift (orc_drift).  4D beams: psigma = 0.
 * ---------------------------------------------------------------------------------------- */
void orc_cquad(int64_t n, double* x, double* px, double* y, double* py, double* sg, double* ps,
               double k1, double L, double gamma0)
{
    if (k1 == 0.0) { orc_drift(n, x, px, y, py, sg, ps, L, gamma0); return; }
    double ak = fabs(k1);
    for (int64_t i = 0; i < n; i++) {
        double psi = ps ? ps[i] : 0.0;
        double d = 1.0 - psi;
        double w = sqrt(ak * d);
        double c = cos(w * L), s = sin(w * L), ch = cosh(w * L), sh = sinh(w * L);
        double a = sqrt(d / ak), b = sqrt(ak / d);          /* the printed coefficients */
        /* f: focusing plane, g: defocusing plane */
        double f0 = k1 > 0.0 ? x[i] : y[i], pf0 = k1 > 0.0 ? px[i] : py[i];
        double g0 = k1 > 0.0 ? y[i] : x[i], pg0 = k1 > 0.0 ? py[i] : px[i];
        double f1 = f0 * c + a * pf0 * s;
        double pf1 = pf0 * c - b * f0 * s;
        double g1 = g0 * ch + a * pg0 * sh;
        double pg1 = pg0 * ch + b * g0 * sh;
        if (sg) {
            double rf = f0 * ak / w, rg = g0 * ak / w;
            double If = 0.5 * L * (pf0 * pf0 + rf * rf) + (pf0 * pf0 - rf * rf) * s * c / (2.0 * w) - pf0 * rf * s * s / w;
            double Ig = 0.5 * L * (pg0 * pg0 - rg * rg) + (pg0 * pg0 + rg * rg) * sh * ch / (2.0 * w) + pg0 * rg * sh * sh / w;
            sg[i] = sg[i] + L * (psi / (gamma0 * gamma0)) - 0.5 * (If + Ig);
        }
        if (k1 > 0.0) { x[i] = f1; px[i] = pf1; y[i] = g1; py[i] = pg1; }
        else { y[i] = f1; py[i] = pf1; x[i] = g1; px[i] = pg1; }
    }
}

/* ------------------------------------------------------------------------------------------
 * N3: EXACT drift -- section III.A's uniform-field solution for B = 0 ("for uniform fields such
 * as dipole magnets and drift spaces the equation of motion can be analytically solved so that we need not use
 * H_approx").  Eq. 2 is singular at B = 0 (A3) and eqs. 4-5 are garbled (A11), so the B = 0 case is restated from
 * what they solve, the force-free straight line, with eq. 3's momenta:
 *   P_z/p0 = pz = sqrt(1 + 2 ps + beta0^2 ps^2 - px^2 - py^2),  P_x/p0 = px,  P_y/p0 = py        (eq. 3)
 *   x(L) = x + L px/pz,  y(L) = y + L py/pz   (the particle reaches the plane s = L after a path L (1+delta)/pz)
 *   sigma(L) = sigma + L - beta0 c t'  (eq. 4),  c t' = path / beta,  beta0/beta = (1 + beta0^2 ps)/(1 + delta)
 *            = sigma + L (1 - (1 + beta0^2 ps)/pz);     px, py, psigma unchanged.
 * With (1+delta)^2 = 1 + 2 ps + beta0^2 ps^2 (eq. 3), i.e. psigma = (E - E0)/(beta0^2 E0).
 * ---------------------------------------------------------------------------------------- */
void orc_xdrift(int64_t n, double* x, double* px, double* y, double* py, double* sg, double* ps,
                double L, double beta0)
{
    for (int64_t i = 0; i < n; i++) {
        double psi = ps ? ps[i] : 0.0;
        double pz = sqrt(1.0 + 2.0 * psi + beta0 * beta0 * psi * psi - px[i] * px[i] - py[i] * py[i]);
        x[i] = x[i] + L * px[i] / pz;
        y[i] = y[i] + L * py[i] / pz;
        if (sg) sg[i] = sg[i] + L * (1.0 - (1.0 + beta0 * beta0 * psi) / pz);
    }
}

/* ------------------------------------------------------------------------------------------
 * N3: EXACT sector bend -- section III.A (eqs. 2-5, Fig. 2): uniform field B along y, reference orbit a
 * circle of radius rho = 1/h about the origin of the Cartesian frame (x~, z~), the particle enters at
 * (x~, z~) = (rho + x, 0) with momenta (eq. 3)  P_x~ = p0 px,  P_z~ = p0 pz,  pz = sqrt(1 + 2 ps + beta0^2 ps^2 - px^2 - py^2),
 * moves on a circle (eq. 2) and leaves through the plane z~ = x~ tan(L/rho) (eq. 5).  Eqs. 2, 4 are garbled as printed (A11:
 * a spurious 1/eB in P_x~(t), missing squares in x(s = L), a missing c in sigma), so the map is restated from that
 * geometry, lengths in units of rho, theta = L/rho:
 *   radius of the particle's circle   R = sqrt(px^2 + pz^2)            (p_perp/(eB) = rho p_perp/p0)
 *   its centre                        (cx, cz) = (1 + h x - pz, px)
 *   D = cx sin(theta) - cz cos(theta)                                  (distance of the centre from the exit plane, signed)
 *   x(L)  = rho (cx cos(theta) + cz sin(theta) + sqrt(R^2 - D^2) - 1)  (eq. 4, first line: radial position minus rho)
 *   px(L) = -D                                                         (eq. 4, second line: radial momentum / p0)
 *   angle turned on the own circle    phi = theta + asin(D/R) + atan2(px, pz)   (eq. 5 solved for t')
 *   y(L) = y + py rho phi,  py unchanged                               (no force along the field)
 *   sigma(L) = sigma + L - beta0 c t' = sigma + L - rho phi (1 + beta0^2 ps)   (eq. 4, third line; path = rho phi (1+delta))
 * h = 0 is the exact drift.  k0 = h: the field that bends the reference particle on the reference orbit.
 * ---------------------------------------------------------------------------------------- */
void orc_sbend(int64_t n, double* x, double* px, double* y, double* py, double* sg, double* ps,
               double L, double h, double beta0)
{
    if (h == 0.0) { orc_xdrift(n, x, px, y, py, sg, ps, L, beta0); return; }
    double rho = 1.0 / h, th = L * h, st = sin(th), ct = cos(th);
    for (int64_t i = 0; i < n; i++) {
        double psi = ps ? ps[i] : 0.0;
        double pz = sqrt(1.0 + 2.0 * psi + beta0 * beta0 * psi * psi - px[i] * px[i] - py[i] * py[i]);
        double R = sqrt(px[i] * px[i] + pz * pz);
        double cx = 1.0 + h * x[i] - pz, cz = px[i];
        double D = cx * st - cz * ct;
        double phi = th + asin(D / R) + atan2(px[i], pz);
        x[i] = rho * (cx * ct + cz * st + sqrt(R * R - D * D) - 1.0);
        px[i] = -D;
        y[i] = y[i] + py[i] * rho * phi;
        if (sg) sg[i] = sg[i] + L - rho * phi * (1.0 + beta0 * beta0 * psi);
    }
}

/* ------------------------------------------------------------------------------------------
 * N3: thick sextupole (eqs. 7-8): H_approx = H0 + V, V = k2 (x^3 - 3 x y^2)/6,
 *   e^{:H0 a L:} e^{:V b L:} e^{:H0 c L:} e^{:V b L:} e^{:H0 a L:},  a = (1 - 1/sqrt 3)/2, b = 1/2, c = 1/sqrt 3   (ref [7]).
 * e^{:H0 l:} is the drift of orc_drift, e^{:V l:} the thin kick px -= k2 l (x^2 - y^2)/2, py += k2 l x y of orc_mult.
 * Applied right to left on the state: H0 aL first (the composition is palindromic, so either reading is the same map).
 * ---------------------------------------------------------------------------------------- */
void orc_sext(int64_t n, double* x, double* px, double* y, double* py, double* sg, double* ps,
              double k2, double L, double gamma0)
{
    double a = 0.5 * (1.0 - 1.0 / sqrt(3.0)), b = 0.5, c = 1.0 / sqrt(3.0);
    orc_drift(n, x, px, y, py, sg, ps, a * L, gamma0);
    orc_mult(n, x, px, y, py, 2, k2 * (b * L), 0.0);
    orc_drift(n, x, px, y, py, sg, ps, c * L, gamma0);
    orc_mult(n, x, px, y, py, 2, k2 * (b * L), 0.0);
    orc_drift(n, x, px, y, py, sg, ps, a * L, gamma0);
}

/* ------------------------------------------------------------------------------------------
 * Thin multipole kick e^{:V:}: with e A_s/p0 = -Re[(kn + i ks)
 * (x+iy)^(n+1)/(n+1)!],  delta(px - i py) = -(knl + i ksl) (x + i y)^n / n!.
 *   n=1: px -= k1l x, py += k1l y   (V = k1 (x^2-y^2)/2)
 *   n=2: px -= k2l (x^2-y^2)/2, py += k2l x y   (V = k2 (x^3 - 3 x y^2)/6)
 * ---------------------------------------------------------------------------------------- */
void orc_mult(int64_t n, double* x, double* px, double* y, double* py,
              int order, double knl, double ksl)
{
    for (int64_t i = 0; i < n; i++) {
        double zr = 1.0, zi = 0.0;
        for (int k = 1; k <= order; k++) {
            double nr = (zr * x[i] - zi * y[i]) / (double)k;
            double ni = (zr * y[i] + zi * x[i]) / (double)k;
            zr = nr; zi = ni;
        }
        px[i] = px[i] - (knl * zr - ksl * zi);
        py[i] = py[i] + (knl * zi + ksl * zr);
    }
}

/* RF kick (PAPER.md:314 names the cavities; psigma is conjugate to sigma):
 * psigma -= amp sin(2 pi h sigma / C + phi0),  amp = q V/(beta0^2 E0). */
void orc_rf(int64_t n, double* sg, double* ps, double amp, double h, double circumference, double phi0)
{
    for (int64_t i = 0; i < n; i++)
        ps[i] = ps[i] - amp * sin(2.0 * ORC_PI * h * sg[i] / circumference + phi0);
}

/* ------------------------------------------------------------------------------------------
 * Cell lookup shared by deposit and gather (A7, A8, A18).  t = (x - xmin) * (1/dx); a particle
 * is inside iff 0 <= t < n-1 on both axes (so that node i+1 exists); i = floor(t), f = t - i.
 * ---------------------------------------------------------------------------------------- */
static int orc_locate(const orc_grid* g, double x, double y, int* i, int* j, double* fx, double* fy)
{
    double dx = (g->xmax - g->xmin) / (double)(g->nx - 1);
    double dy = (g->ymax - g->ymin) / (double)(g->ny - 1);
    double inv_dx = 1.0 / dx, inv_dy = 1.0 / dy;
    double tx = (x - g->xmin) * inv_dx;
    double ty = (y - g->ymin) * inv_dy;
    if (!(tx >= 0.0 && tx < (double)(g->nx - 1) && ty >= 0.0 && ty < (double)(g->ny - 1))) return 0;
    *i = (int)floor(tx);
    *j = (int)floor(ty);
    *fx = tx - (double)*i;
    *fy = ty - (double)*j;
    return 1;
}

/* Cloud-in-cell deposit, eq. 14, unit weight per particle (SURVEY note on
 * lambda: it multiplies the kick, eq. 12, not the deposit).  Q is nx*ny, index j*nx+i. */
int64_t orc_deposit_f64(int64_t n, const double* x, const double* y, const orc_grid* g, double* Q)
{
    int64_t n_in = 0;
    for (int64_t c = 0; c < (int64_t)g->nx * g->ny; c++) Q[c] = 0.0;
    for (int64_t p = 0; p < n; p++) {
        int i, j; double fx, fy;
        if (!orc_locate(g, x[p], y[p], &i, &j, &fx, &fy)) continue;
        n_in++;
        Q[(int64_t)j * g->nx + i] += (1.0 - fx) * (1.0 - fy);
        Q[(int64_t)j * g->nx + i + 1] += fx * (1.0 - fy);
        Q[(int64_t)(j + 1) * g->nx + i] += (1.0 - fx) * fy;
        Q[(int64_t)(j + 1) * g->nx + i + 1] += fx * fy;
    }
    return n_in;
}

/* Fixed-point variant of eq. 14: per-axis fractions quantised to s bits,
 * ax = llrint(fx 2^s) (round half to even), bx = 2^s - ax; the four integer products sum to
 * 2^(2s) exactly, so sum(Qi) = n_inside 2^(2s). */
int64_t orc_deposit_fixed(int64_t n, const double* x, const double* y, const orc_grid* g, int64_t* Qi)
{
    int64_t n_in = 0;
    int64_t S = (int64_t)1 << g->fixed_bits;
    for (int64_t c = 0; c < (int64_t)g->nx * g->ny; c++) Qi[c] = 0;
    for (int64_t p = 0; p < n; p++) {
        int i, j; double fx, fy;
        if (!orc_locate(g, x[p], y[p], &i, &j, &fx, &fy)) continue;
        n_in++;
        int64_t ax = llrint(fx * (double)S), ay = llrint(fy * (double)S);
        int64_t bx = S - ax, by = S - ay;
        Qi[(int64_t)j * g->nx + i] += bx * by;
        Qi[(int64_t)j * g->nx + i + 1] += ax * by;
        Qi[(int64_t)(j + 1) * g->nx + i] += bx * ay;
        Qi[(int64_t)(j + 1) * g->nx + i + 1] += ax * ay;
    }
    return n_in;
}

/* Line density ("sigma-distributions with 128 bins"; A6): integer counts of
 * sigma in nbins equal bins over [smin, smax); t = (sigma - smin) * (1/ds), bin = floor(t). */
void orc_lambda_hist(int64_t n, const double* sg, const orc_grid* g, int64_t* cnt)
{
    double ds = (g->smax - g->smin) / (double)g->nbins;
    double inv_ds = 1.0 / ds;
    for (int b = 0; b < g->nbins; b++) cnt[b] = 0;
    for (int64_t p = 0; p < n; p++) {
        double t = (sg[p] - g->smin) * inv_ds;
        if (!(t >= 0.0 && t < (double)g->nbins)) continue;
        cnt[(int)floor(t)]++;
    }
}

/* lambda(sigma) [1/m] = n_real cnt_b/(N ds) at bin centres, linear in between, bins outside the
 * range count as empty, 0 outside [smin, smax)  (A6). */
double orc_lambda_at(double sigma, const orc_grid* g, const int64_t* cnt, double n_real, int64_t n)
{
    double ds = (g->smax - g->smin) / (double)g->nbins;
    double inv_ds = 1.0 / ds;
    double t = (sigma - g->smin) * inv_ds;
    if (!(t >= 0.0 && t < (double)g->nbins)) return 0.0;
    double u = t - 0.5;
    double b0 = floor(u);
    double f = u - b0;
    int ib = (int)b0;
    double scale = n_real / ((double)n * ds);
    double l0 = (ib >= 0 && ib < g->nbins) ? scale * (double)cnt[ib] : 0.0;
    double l1 = (ib + 1 >= 0 && ib + 1 < g->nbins) ? scale * (double)cnt[ib + 1] : 0.0;
    return (1.0 - f) * l0 + f * l1;
}

/* d lambda / d sigma of the piecewise-linear lambda(sigma) above: (lambda_{b+1} - lambda_b)/ds between the
 * centres of bins b and b+1 (the same pair orc_lambda_at interpolates), 0 outside [smin, smax)
 * (eq. 13, needs "the derivative of lambda"; the paper does not say how it is taken). */
double orc_lambda_slope(double sigma, const orc_grid* g, const int64_t* cnt, double n_real, int64_t n)
{
    double ds = (g->smax - g->smin) / (double)g->nbins;
    double inv_ds = 1.0 / ds;
    double t = (sigma - g->smin) * inv_ds;
    if (!(t >= 0.0 && t < (double)g->nbins)) return 0.0;
    double u = t - 0.5;
    int ib = (int)floor(u);
    double scale = n_real / ((double)n * ds);
    double l0 = (ib >= 0 && ib < g->nbins) ? scale * (double)cnt[ib] : 0.0;
    double l1 = (ib + 1 >= 0 && ib + 1 < g->nbins) ? scale * (double)cnt[ib + 1] : 0.0;
    return (l1 - l0) * inv_ds;
}

/* ------------------------------------------------------------------------------------------
 * Open-boundary Green's function of  laplace(u) = -f  in 2D:  G(r) = -ln(r^2)/(4 pi), averaged
 * over the source cell (A10):  G_cell(x,y) = -(1/(4 pi dx dy)) int int ln(x'^2+y'^2) dx' dy'
 * over [x-dx/2, x+dx/2] x [y-dy/2, y+dy/2], with the antiderivative
 *   F(x,y) = x y ln(x^2+y^2) - 3 x y + x^2 atan(y/x) + y^2 atan(x/y)        (d2F/dxdy = ln(x^2+y^2))
 * evaluated in long double because the four-corner difference cancels ~5 digits far from 0.
 * ---------------------------------------------------------------------------------------- */
static long double orc_F(long double x, long double y)
{
    /* corners are at half-integer multiples of dx, dy: never zero */
    return x * y * logl(x * x + y * y) - 3.0L * x * y + x * x * atanl(y / x) + y * y * atanl(x / y);
}

double orc_green_cell(double x, double y, double dx, double dy)
{
    long double x1 = (long double)x - 0.5L * dx, x2 = (long double)x + 0.5L * dx;
    long double y1 = (long double)y - 0.5L * dy, y2 = (long double)y + 0.5L * dy;
    long double I = orc_F(x2, y2) - orc_F(x1, y2) - orc_F(x2, y1) + orc_F(x1, y1);
    return (double)(-I / (4.0L * (long double)ORC_PI * dx * dy));
}

/* table Gt[b*(nx+1)+a] = G_cell(a dx, b dy), a = 0..nx, b = 0..ny; cached per grid geometry */
typedef struct { int nx, ny; double dx, dy; double* Gt; double* Ghat_re; } orc_gcache;
static orc_gcache g_cache[16];
static int g_ncache = 0;

static orc_gcache* orc_green_table(const orc_grid* g)
{
    double dx = (g->xmax - g->xmin) / (double)(g->nx - 1);
    double dy = (g->ymax - g->ymin) / (double)(g->ny - 1);
    for (int c = 0; c < g_ncache; c++)
        if (g_cache[c].nx == g->nx && g_cache[c].ny == g->ny && g_cache[c].dx == dx && g_cache[c].dy == dy)
            return &g_cache[c];
    if (g_ncache == 16) { free(g_cache[0].Gt); free(g_cache[0].Ghat_re); g_cache[0] = g_cache[15]; g_ncache = 15; }
    orc_gcache* e = &g_cache[g_ncache++];
    e->nx = g->nx; e->ny = g->ny; e->dx = dx; e->dy = dy; e->Ghat_re = NULL;
    e->Gt = (double*)malloc(sizeof(double) * (size_t)(g->nx + 1) * (g->ny + 1));
    for (int b = 0; b <= g->ny; b++)
        for (int a = 0; a <= g->nx; a++)
            e->Gt[(size_t)b * (g->nx + 1) + a] = orc_green_cell(a * dx, b * dy, dx, dy);
    return e;
}

/* The DEFINITION of the open-boundary solve (north_star "open-boundary
 * Poisson"):  u~[i,j] = dx dy sum_{i',j'} G[i-i', j-j'] f[i',j'],  f = Q/(N dx dy)  (step 5e:
 * normalised to ALL N particles), i.e.  u~ = (1/N) sum G Q.   O(n^4); cells with Q = 0 add 0. */
void orc_poisson_direct(const orc_grid* g, const double* Q, double n_total, double* u)
{
    orc_gcache* e = orc_green_table(g);
    int nx = g->nx, ny = g->ny;
    for (int j = 0; j < ny; j++)
        for (int i = 0; i < nx; i++) {
            double s = 0.0;
            for (int jj = 0; jj < ny; jj++)
                for (int ii = 0; ii < nx; ii++) {
                    double q = Q[(size_t)jj * nx + ii];
                    if (q == 0.0) continue;
                    s += e->Gt[(size_t)abs(j - jj) * (nx + 1) + abs(i - ii)] * q;
                }
            u[(size_t)j * nx + i] = s / n_total;
        }
}

/* ---- own FFT: iterative radix-2 Cooley-Tukey, twiddles from cos/sin per stage entry -------- */
void orc_fft(int n, double* re, double* im, int inverse)
{
    for (int i = 1, j = 0; i < n; i++) {           /* bit reversal */
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { double t = re[i]; re[i] = re[j]; re[j] = t; t = im[i]; im[i] = im[j]; im[j] = t; }
    }
    for (int len = 2; len <= n; len <<= 1) {
        double sgn = inverse ? 1.0 : -1.0;
        for (int k = 0; k < len / 2; k++) {
            double ang = sgn * 2.0 * ORC_PI * (double)k / (double)len;
            double wr = cos(ang), wi = sin(ang);
            for (int s = 0; s < n; s += len) {
                int a = s + k, b = s + k + len / 2;
                double tr = re[b] * wr - im[b] * wi, ti = re[b] * wi + im[b] * wr;
                re[b] = re[a] - tr; im[b] = im[a] - ti;
                re[a] = re[a] + tr; im[a] = im[a] + ti;
            }
        }
    }
    if (inverse) for (int i = 0; i < n; i++) { re[i] /= (double)n; im[i] /= (double)n; }
}

/* eq. 21 / eq. 26 written out: the pin for orc_fft */
void orc_dft_naive(int n, const double* re, const double* im, double* ore, double* oim, int inverse)
{
    for (int p = 0; p < n; p++) {
        long double sr = 0, si = 0;
        for (int l = 0; l < n; l++) {
            long double ang = (inverse ? 2.0L : -2.0L) * (long double)ORC_PI * (long double)((long)p * l % n) / n;
            long double c = cosl(ang), s = sinl(ang);
            sr += re[l] * c - im[l] * s;
            si += re[l] * s + im[l] * c;
        }
        if (inverse) { sr /= n; si /= n; }
        ore[p] = (double)sr; oim[p] = (double)si;
    }
}

static void orc_fft2(int n0, int n1, double* re, double* im, int inverse)
{   /* array [n1][n0], n0 fastest */
    double* tr = (double*)malloc(sizeof(double) * (size_t)n1);
    double* ti = (double*)malloc(sizeof(double) * (size_t)n1);
    for (int r = 0; r < n1; r++) orc_fft(n0, re + (size_t)r * n0, im + (size_t)r * n0, inverse);
    for (int c = 0; c < n0; c++) {
        for (int r = 0; r < n1; r++) { tr[r] = re[(size_t)r * n0 + c]; ti[r] = im[(size_t)r * n0 + c]; }
        orc_fft(n1, tr, ti, inverse);
        for (int r = 0; r < n1; r++) { re[(size_t)r * n0 + c] = tr[r]; im[(size_t)r * n0 + c] = ti[r]; }
    }
    free(tr); free(ti);
}

/* Same sum as orc_poisson_direct evaluated as a circular convolution on the zero-padded
 * 2nx x 2ny (Hockney) grid, PAPER.md:213 ("we thus employ DFTs"), ref [1].  The periodic
 * extension of G uses distance min(a, 2nx-a); the one never-used wrap entry a = nx is set to
 * G(nx dx) so that the extension is even.  nx, ny powers of two. */
void orc_poisson_fft(const orc_grid* g, const double* Q, double n_total, double* u)
{
    orc_gcache* e = orc_green_table(g);
    int nx = g->nx, ny = g->ny, mx = 2 * nx, my = 2 * ny;
    size_t tot = (size_t)mx * my;
    double* wi = (double*)calloc(tot, sizeof(double));
    if (!e->Ghat_re) {
        double* gr = (double*)malloc(sizeof(double) * tot);
        for (int b = 0; b < my; b++)
            for (int a = 0; a < mx; a++) {
                int da = a <= nx ? a : mx - a, db = b <= ny ? b : my - b;
                gr[(size_t)b * mx + a] = e->Gt[(size_t)db * (nx + 1) + da];
            }
        orc_fft2(mx, my, gr, wi, 0);
        e->Ghat_re = gr;                           /* imaginary part is rounding noise: even extension */
        memset(wi, 0, sizeof(double) * tot);
    }
    double* wr = (double*)calloc(tot, sizeof(double));
    for (int j = 0; j < ny; j++)
        for (int i = 0; i < nx; i++) wr[(size_t)j * mx + i] = Q[(size_t)j * nx + i];
    orc_fft2(mx, my, wr, wi, 0);
    for (size_t k = 0; k < tot; k++) { wr[k] *= e->Ghat_re[k]; wi[k] *= e->Ghat_re[k]; }
    orc_fft2(mx, my, wr, wi, 1);
    for (int j = 0; j < ny; j++)
        for (int i = 0; i < nx; i++) u[(size_t)j * nx + i] = wr[(size_t)j * mx + i] / n_total;
    free(wr); free(wi);
}

/* The paper's own solver (section IV.B, eqs. 15-27): conducting rectangular pipe,
 * u = 0 on the wall (eq. 16), five-point Laplacian (eq. 17), odd extension V, F of u, f to
 * 2(m+1) points per axis (eq. 18), two DFTs, division by the symbol of eq. 25, two inverse DFTs
 * (eq. 27), written out in that order.
 * Readings (N1): the wall is node 0 and the virtual node n one spacing beyond the
 * last stored node (m = n-1 interior nodes per axis, 2(m+1) = 2n a power of two); charge deposited on
 * the wall node 0 is dropped (F_0 = 0 by eq. 18); sign and units as everywhere else (A4/A5):
 * laplace(u~) = -f with f = Q/(N dx dy), so V^ = +F^ / (4 (sin^2/dx^2 + sin^2/dy^2)); the (0,0)
 * mode, where eq. 25 divides by zero, has F^ = 0 by oddness and is set to 0 (A12). */
void orc_poisson_dirichlet(const orc_grid* g, const double* Q, double n_total, double* u)
{
    const double PI = 3.14159265358979323846;
    int nx = g->nx, ny = g->ny, Nx = 2 * nx, Ny = 2 * ny;      /* m+1 = n per axis */
    double dx = (g->xmax - g->xmin) / (double)(nx - 1);
    double dy = (g->ymax - g->ymin) / (double)(ny - 1);
    size_t tot = (size_t)Nx * Ny;
    double* Fr = (double*)calloc(tot, sizeof(double));
    double* Fi = (double*)calloc(tot, sizeof(double));
    /* eq. 18: F_{l,l'} = f_{l,l'} (1 <= l,l' <= m), odd about 0 and about m+1 in both indices */
    for (int lp = 1; lp < ny; lp++)
        for (int l = 1; l < nx; l++) {
            double f = Q[(size_t)lp * nx + l] / (n_total * dx * dy);
            Fr[(size_t)lp * Nx + l] = f;
            Fr[(size_t)lp * Nx + (Nx - l)] = -f;
            Fr[(size_t)(Ny - lp) * Nx + l] = -f;
            Fr[(size_t)(Ny - lp) * Nx + (Nx - l)] = f;
        }
    orc_fft2(Nx, Ny, Fr, Fi, 0);                               /* DFT_l', DFT_l (eq. 21) */
    for (int q = 0; q < Ny; q++)
        for (int p = 0; p < Nx; p++) {
            size_t k = (size_t)q * Nx + p;
            double sp = sin(PI * (double)p / (double)Nx), sq = sin(PI * (double)q / (double)Ny);
            double den = 4.0 * (sp * sp / (dx * dx) + sq * sq / (dy * dy));   /* eq. 25 */
            if (p == 0 && q == 0) { Fr[k] = 0.0; Fi[k] = 0.0; }
            else { Fr[k] = Fr[k] / den; Fi[k] = Fi[k] / den; }
        }
    orc_fft2(Nx, Ny, Fr, Fi, 1);                               /* iDFT_q, iDFT_p (eq. 26, 27) */
    for (int j = 0; j < ny; j++)
        for (int i = 0; i < nx; i++) u[(size_t)j * nx + i] = Fr[(size_t)j * Nx + i];
    free(Fr); free(Fi);
}

/* E~ = -grad u~ on the nodes (eq. 29) by central differences, one-sided on
 * the boundary nodes. */
void orc_field(const orc_grid* g, const double* u, double* Ex, double* Ey)
{
    int nx = g->nx, ny = g->ny;
    double dx = (g->xmax - g->xmin) / (double)(nx - 1);
    double dy = (g->ymax - g->ymin) / (double)(ny - 1);
    for (int j = 0; j < ny; j++)
        for (int i = 0; i < nx; i++) {
            size_t c = (size_t)j * nx + i;
            if (i == 0) Ex[c] = -(u[c + 1] - u[c]) / dx;
            else if (i == nx - 1) Ex[c] = -(u[c] - u[c - 1]) / dx;
            else Ex[c] = -(u[c + 1] - u[c - 1]) / (2.0 * dx);
            if (j == 0) Ey[c] = -(u[c + nx] - u[c]) / dy;
            else if (j == ny - 1) Ey[c] = -(u[c] - u[c - nx]) / dy;
            else Ey[c] = -(u[c + nx] - u[c - nx]) / (2.0 * dy);
        }
}

/* Bilinear gather with the SAME four weights as the deposit (the paper's own
 * interpolation, eq. 28, is the NEXT row N4). */
void orc_gather(const orc_grid* g, const double* Ex, const double* Ey, double x, double y,
                int* inside, double* ex, double* ey)
{
    int i, j; double fx, fy;
    *ex = 0.0; *ey = 0.0;
    *inside = orc_locate(g, x, y, &i, &j, &fx, &fy);
    if (!*inside) return;
    size_t c = (size_t)j * g->nx + i;
    double w00 = (1.0 - fx) * (1.0 - fy), w10 = fx * (1.0 - fy), w01 = (1.0 - fx) * fy, w11 = fx * fy;
    *ex = w00 * Ex[c] + w10 * Ex[c + 1] + w01 * Ex[c + g->nx] + w11 * Ex[c + g->nx + 1];
    *ey = w00 * Ey[c] + w10 * Ey[c + 1] + w01 * Ey[c + g->nx] + w11 * Ey[c + g->nx + 1];
}

/* Bilinear interpolation of a node scalar (the potential u~) with the deposit's weights. */
double orc_gather_scalar(const orc_grid* g, const double* u, double x, double y, int* inside)
{
    int i, j; double fx, fy;
    *inside = orc_locate(g, x, y, &i, &j, &fx, &fy);
    if (!*inside) return 0.0;
    size_t c = (size_t)j * g->nx + i;
    double w00 = (1.0 - fx) * (1.0 - fy), w10 = fx * (1.0 - fy), w01 = (1.0 - fx) * fy, w11 = fx * fy;
    return w00 * u[c] + w10 * u[c + 1] + w01 * u[c + g->nx] + w11 * u[c + g->nx + 1];
}

/* ------------------------------------------------------------------------------------------
 * N4: the paper's interpolation, eqs. 28-29 (section IV.C).
 *
 * Eq. 28 writes the potential at (x, y) inside the cell [x_i, x_i+1] x [y_j, y_j+1] as a bicubic BEZIER SURFACE
 *     u(x,y) = sum_{m=0..3} sum_{n=0..3} P_mn  C(3,m) t^m (1-t)^(3-m)  C(3,n) s^n (1-s)^(3-n),
 *     t = (x - x_i)/dx,  s = (y - y_j)/dy,
 * over the 4x4 stencil u_{i+m-1, j+n-1}, and eq. 29 takes E = -grad u of that surface analytically.
 * AS PRINTED the control points are the node values themselves, P_mn = u_{i+m-1,j+n-1}; a Bezier surface passes
 * through its corner control points, so that reading gives u(x_i, .) = u_{i-1, .} and u(x_i+1, .) = u_{i+2, .}:
 * a surface that jumps by two grid spacings between neighbouring cells (tests/test_oracle_bicubic.py shows the
 * jump).  Reading A9: the surface is the one cubic spline surface whose 4x4 stencil of
 * node values are its de Boor points, i.e. the uniform cubic B-spline; written in the paper's Bernstein form
 * its Bezier control points follow from the stencil by the textbook B-spline -> Bezier conversion, per axis
 *     P_0 = (U_0 + 4 U_1 + U_2)/6,  P_1 = (2 U_1 + U_2)/3,  P_2 = (U_1 + 2 U_2)/3,  P_3 = (U_1 + 4 U_2 + U_3)/6.
 * That surface is C^2 across cell edges, reproduces constants and linear potentials exactly and uses exactly the
 * stencil the paper names.  Stencil nodes beyond the grid edge (i-1 = -1, i+2 = nx; same in y) are linear
 * extrapolations u_{-1} = 2 u_0 - u_1, u_{nx} = 2 u_{nx-1} - u_{nx-2} (the paper is silent; this keeps linear
 * potentials exact in the edge cells).  Inside test and (i, j, t, s) are the deposit's (orc_locate).
 * ---------------------------------------------------------------------------------------- */
static double orc_node_ext(const orc_grid* g, const double* u, int i, int j)
{
    int nx = g->nx, ny = g->ny;
    if (i < 0) return 2.0 * orc_node_ext(g, u, 0, j) - orc_node_ext(g, u, 1, j);
    if (i > nx - 1) return 2.0 * orc_node_ext(g, u, nx - 1, j) - orc_node_ext(g, u, nx - 2, j);
    if (j < 0) return 2.0 * u[(size_t)0 * nx + i] - u[(size_t)1 * nx + i];
    if (j > ny - 1) return 2.0 * u[(size_t)(ny - 1) * nx + i] - u[(size_t)(ny - 2) * nx + i];
    return u[(size_t)j * nx + i];
}

/* Bernstein polynomial C(3,m) t^m (1-t)^(3-m) and its derivative with respect to t */
static void orc_bernstein3(double t, double B[4], double dB[4])
{
    static const double binom[4] = { 1.0, 3.0, 3.0, 1.0 };
    for (int m = 0; m < 4; m++) {
        double a = 1.0, b = 1.0;          /* t^m, (1-t)^(3-m) */
        for (int k = 0; k < m; k++) a *= t;
        for (int k = 0; k < 3 - m; k++) b *= (1.0 - t);
        double da = 0.0, db = 0.0;        /* d/dt t^m = m t^(m-1);  d/dt (1-t)^(3-m) = -(3-m)(1-t)^(2-m) */
        if (m > 0) { da = (double)m; for (int k = 0; k < m - 1; k++) da *= t; }
        if (3 - m > 0) { db = -(double)(3 - m); for (int k = 0; k < 2 - m; k++) db *= (1.0 - t); }
        B[m] = binom[m] * a * b;
        dB[m] = binom[m] * (da * b + a * db);
    }
}

void orc_gather_bicubic(const orc_grid* g, const double* u, double x, double y,
                        int* inside, double* uval, double* ex, double* ey)
{
    /* B-spline (de Boor points) -> Bezier control points, one axis */
    static const double conv[4][4] = { { 1.0 / 6.0, 4.0 / 6.0, 1.0 / 6.0, 0.0 },
                                       { 0.0, 2.0 / 3.0, 1.0 / 3.0, 0.0 },
                                       { 0.0, 1.0 / 3.0, 2.0 / 3.0, 0.0 },
                                       { 0.0, 1.0 / 6.0, 4.0 / 6.0, 1.0 / 6.0 } };
    int i, j; double t, s;
    *uval = 0.0; *ex = 0.0; *ey = 0.0;
    *inside = orc_locate(g, x, y, &i, &j, &t, &s);
    if (!*inside) return;
    double dx = (g->xmax - g->xmin) / (double)(g->nx - 1);
    double dy = (g->ymax - g->ymin) / (double)(g->ny - 1);
    double U[4][4], P[4][4];                  /* U[m][n] = u_{i+m-1, j+n-1} (eq. 28's stencil) */
    for (int m = 0; m < 4; m++)
        for (int n = 0; n < 4; n++) U[m][n] = orc_node_ext(g, u, i + m - 1, j + n - 1);
    for (int m = 0; m < 4; m++)
        for (int n = 0; n < 4; n++) {
            double acc = 0.0;
            for (int a = 0; a < 4; a++)
                for (int c = 0; c < 4; c++) acc += conv[m][a] * conv[n][c] * U[a][c];
            P[m][n] = acc;
        }
    double Bx[4], dBx[4], By[4], dBy[4];
    orc_bernstein3(t, Bx, dBx);
    orc_bernstein3(s, By, dBy);
    double val = 0.0, ddx = 0.0, ddy = 0.0;
    for (int m = 0; m < 4; m++)
        for (int n = 0; n < 4; n++) {
            val += P[m][n] * Bx[m] * By[n];           /* eq. 28 */
            ddx += P[m][n] * dBx[m] * By[n];
            ddy += P[m][n] * Bx[m] * dBy[n];
        }
    *uval = val;
    *ex = -ddx / dx;                                  /* eq. 29: dt/dx = 1/dx */
    *ey = -ddy / dy;
}

/* Gather + kick with the node's grids already in w (eq. 12, and eq. 13 when g->long_kick): px, py (and psigma)
 * of every inside particle; nothing else is touched.  Split out of orc_scnode so that it can be pinned on
 * prescribed fields. */
void orc_sc_kick(int64_t n, double* x, double* px, double* y, double* py, const double* sg, double* ps,
                 const orc_grid* g, const orc_beam* b, double L_sc, const orc_work* w)
{
    for (int64_t p = 0; p < n; p++) {
        int inside; double ex, ey, ubic = 0.0;
        if (g->interp == 1) orc_gather_bicubic(g, w->u, x[p], y[p], &inside, &ubic, &ex, &ey);   /* N4, eqs. 28-29 */
        else orc_gather(g, w->Ex, w->Ey, x[p], y[p], &inside, &ex, &ey);
        if (!inside) continue;
        double lam = g->nbins > 0 ? orc_lambda_at(sg[p], g, w->cnt, b->n_real, n) : b->line_density;
        px[p] = px[p] + b->kappa * lam * L_sc * ex;
        py[p] = py[p] + b->kappa * lam * L_sc * ey;
        /* N2, eq. 13: longitudinal kick  -K u(x,y) dlambda/dz L.  Reading:
         * both kicks are the flow of ONE kick Hamiltonian  kappa L lambda(sigma) u~(x,y)  (eq. 11's potential), so
         * the prefactor is eq. 12's (gamma0^3; eq. 13 prints gamma0^2) and  psigma -= kappa L u~ lambda'(sigma),
         * evaluated at the same pre-kick (x, y, sigma).  Bunched beams only. */
        if (g->long_kick && g->nbins > 0 && ps) {
            int in2;
            double up = g->interp == 1 ? ubic : orc_gather_scalar(g, w->u, x[p], y[p], &in2);
            double dl = orc_lambda_slope(sg[p], g, w->cnt, b->n_real, n);
            ps[p] = ps[p] - b->kappa * L_sc * up * dl;
        }
    }
}

/* One space-charge node (section IV): deposit -> lambda histogram ->
 * Poisson -> field -> gather -> kick  px += kappa lambda(sigma_i) L_sc E~x  (eq. 12,
 * PAPER.md:163-167; zero for particles outside the grid, A8). */
int orc_scnode(int64_t n, double* x, double* px, double* y, double* py, const double* sg, double* ps,
               const orc_grid* g, const orc_beam* b, double L_sc, int poisson_direct, orc_work* w)
{
    size_t nc = (size_t)g->nx * g->ny;
    if (g->fixed) {
        w->n_inside = orc_deposit_fixed(n, x, y, g, w->Qi);
        double scale = ldexp(1.0, -2 * g->fixed_bits);
        for (size_t c = 0; c < nc; c++) w->Q[c] = (double)w->Qi[c] * scale;
    } else {
        w->n_inside = orc_deposit_f64(n, x, y, g, w->Q);
    }
    if (g->nbins > 0) {
        if (!sg) return -1;
        orc_lambda_hist(n, sg, g, w->cnt);
    }
    if (g->boundary == 1) orc_poisson_dirichlet(g, w->Q, (double)n, w->u);
    else if (poisson_direct) orc_poisson_direct(g, w->Q, (double)n, w->u);
    else orc_poisson_fft(g, w->Q, (double)n, w->u);
    orc_field(g, w->u, w->Ex, w->Ey);
    if (L_sc < 0.0) return 0;                       /* orc_track stop: grids solved, kick not applied */
    orc_sc_kick(n, x, px, y, py, sg, ps, g, b, L_sc, w);
    return 0;
}

/* The per-turn loop: rows in table order, every turn. */
int orc_track(int64_t n, double* x, double* px, double* y, double* py, double* sg, double* ps,
              int64_t n_rows, const int32_t* kind, const int32_t* ipar, const double* par,
              int32_t n_grids, const orc_grid* grids, const orc_beam* b,
              int64_t n_turns, int64_t stop_after_rows, int poisson_direct, orc_work* works)
{
    int64_t done = 0;
    if (stop_after_rows == 0) return 0;
    for (int64_t t = 0; t < n_turns || stop_after_rows > 0; t++) {
        for (int64_t r = 0; r < n_rows; r++) {
            const double* p = par + 10 * r;
            int last = stop_after_rows >= 0 && done + 1 == stop_after_rows;
            switch (kind[r]) {
            case ORC_DRIFT: orc_drift(n, x, px, y, py, sg, ps, p[0], b->gamma0); break;
            case ORC_LINMAP: orc_linmap(n, x, px, y, py, sg, ps, p, p[8], b->gamma0); break;
            case ORC_QUAD: { double M[8]; orc_quad_matrix(p[0], p[1], M);
                             orc_linmap(n, x, px, y, py, sg, ps, M, p[1], b->gamma0); } break;
            case ORC_CQUAD: orc_cquad(n, x, px, y, py, sg, ps, p[0], p[1], b->gamma0); break;
            case ORC_XDRIFT: orc_xdrift(n, x, px, y, py, sg, ps, p[0], b->beta0); break;
            case ORC_SBEND: orc_sbend(n, x, px, y, py, sg, ps, p[0], p[1], b->beta0); break;
            case ORC_SEXT: orc_sext(n, x, px, y, py, sg, ps, p[0], p[1], b->gamma0); break;
            case ORC_MULT: orc_mult(n, x, px, y, py, ipar[r], p[0], p[1]); break;
            case ORC_RF:
                if (!sg || !ps) return -1;
                orc_rf(n, sg, ps, (double)b->charge * p[0] / (b->beta0 * b->beta0 * b->E0_eV),
                       p[1], b->circumference, p[2]);
                break;
            case ORC_SCNODE:
                if (ipar[r] < 0 || ipar[r] >= n_grids) return -1;
                if (orc_scnode(n, x, px, y, py, sg, ps, &grids[ipar[r]], b, last ? -1.0 : p[0],
                               poisson_direct, &works[ipar[r]])) return -1;
                break;
            default: return -1;
            }
            done++;
            if (stop_after_rows >= 0 && done == stop_after_rows) return 0;
        }
    }
    return 0;
}

/* Moments (beta from the rms of tracked particles): plain two-pass, long double.
 * eps_u = sqrt(<u^2><pu^2> - <u pu>^2) of the centred moments. */
void orc_moments(int64_t n, const double* x, const double* px, const double* y, const double* py,
                 const double* sg, const double* ps, double* out)
{
    const double* q[6] = { x, px, y, py, sg, ps };
    long double mean[6], C[6][6];
    for (int a = 0; a < 6; a++) {
        long double s = 0;
        if (q[a]) for (int64_t i = 0; i < n; i++) s += q[a][i];
        mean[a] = n > 0 ? s / n : 0;
    }
    for (int a = 0; a < 6; a++)
        for (int c = a; c < 6; c++) {
            long double s = 0;
            if (q[a] && q[c])
                for (int64_t i = 0; i < n; i++) s += ((long double)q[a][i] - mean[a]) * ((long double)q[c][i] - mean[c]);
            C[a][c] = n > 0 ? s / n : 0;
        }
    out[0] = (double)n;
    for (int a = 0; a < 6; a++) out[1 + a] = (double)mean[a];
    int k = 7;
    for (int a = 0; a < 6; a++) for (int c = a; c < 6; c++) out[k++] = (double)C[a][c];
    for (int pl = 0; pl < 3; pl++) {
        long double d = C[2 * pl][2 * pl] * C[2 * pl + 1][2 * pl + 1] - C[2 * pl][2 * pl + 1] * C[2 * pl][2 * pl + 1];
        out[28 + pl] = d > 0 ? (double)sqrtl(d) : 0.0;
    }
    out[31] = 0.0; out[32] = 0.0;
}
