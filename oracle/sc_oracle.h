/*
 * sc_oracle.h -- ORACLE (test infrastructure, NOT the product).
 *
 * Plain, slow, single-threaded fp64 CPU restatement of the per-turn hot path of the 2D
 * particle-in-cell space-charge tracker of arXiv 2010.11540 (Kurimoto), written from the paper
 * and the readings recorded in DESIGN.md / SURVEY.md section 8(c).  It shares no code
 * with the CUDA path (paper_2010_11540_b200/csrc) and neither includes the other.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * Build: gcc -O2 -ffp-contract=off -std=c99 (no FMA contraction, so that the index / fraction
 * arithmetic of the deposit is the literal sequence of IEEE operations written here).
 *
 * Variables: x, px, y, py, sigma = s - beta0 c t, psigma.  Arrays are SoA fp64.
 * sigma/psigma may be NULL: 4D coasting beam (psigma = 0, sigma not tracked).
 *
 * Every function has a pin in tests/test_oracle_*.py (closed form, invariant, brute force or a
 * value the paper prints); none is "parity unpinned".
 */
#ifndef SC_ORACLE_H
#define SC_ORACLE_H
#include <stdint.h>

/* lattice table row kinds (the oracle's own numbering is by name; values are passed from Python) */
enum { ORC_DRIFT = 0, ORC_LINMAP = 1, ORC_MULT = 2, ORC_RF = 3, ORC_SCNODE = 4, ORC_QUAD = 5, ORC_CQUAD = 6, ORC_SEXT = 7, ORC_XDRIFT = 8, ORC_SBEND = 9 };

typedef struct {
    int32_t nx, ny;            /* number of grid NODES per axis                 */
    double xmin, xmax, ymin, ymax; /* node coordinates of first/last node; dx=(xmax-xmin)/(nx-1) */
    int32_t nbins;             /* lambda(sigma) histogram bins; 0 => coasting beam              */
    double smin, smax;         /* histogram range [smin, smax)                                  */
    int32_t fixed;             /* 0: fp64 deposit, 1: int64 fixed-point deposit                 */
    int32_t fixed_bits;        /* s: per-axis fraction bits of the fixed-point weights          */
    int32_t boundary;          /* 0: open boundary (Hockney, north_star); 1: the paper's conducting
                                  rectangular pipe, u = 0 on the wall (eqs. 15-27)   */
    int32_t long_kick;         /* 1: also apply the longitudinal space-charge kick of eq. 13  */
    int32_t interp;            /* 0: bilinear gather of the node field (north_star); 1: the paper's bicubic
                                  "Bezier surface" of the POTENTIAL on the 4x4 stencil with the analytic gradient
                                  (eqs. 28-29; reading A9 in DESIGN.md)                          */
} orc_grid;

typedef struct {
    double gamma0, beta0, E0_eV;   /* reference particle                                        */
    double r_c;                    /* classical radius q^2 e^2/(4 pi eps0 m c^2) [m]            */
    double kappa;                  /* 4 pi r_c / (beta0^2 gamma0^3)   (eq. 11-12 prefactor)     */
    int32_t charge;
    double line_density;           /* coasting: particles per metre                             */
    double n_real;                 /* bunched: real particles per bunch                         */
    double circumference;          /* metres                                                    */
} orc_beam;

/* reference-particle constants from kinetic energy and rest mass (eV).  PAPER.md:51, eq. 11. */
void orc_beam_init(orc_beam* b, double kinetic_eV, double mass_eV, int charge,
                   double line_density, double n_real, double circumference);

/* ---- single-particle maps, applied to all n particles in index order (section III) */
void orc_drift(int64_t n, double* x, double* px, double* y, double* py, double* sg, double* ps,
               double L, double gamma0);
void orc_quad_matrix(double k1, double L, double M[8]);
void orc_linmap(int64_t n, double* x, double* px, double* y, double* py, double* sg, double* ps,
                const double M[8], double L, double gamma0);
/* eq. 6 as printed, per particle (chromatic thick quadrupole, N3) */
void orc_cquad(int64_t n, double* x, double* px, double* y, double* py, double* sg, double* ps,
               double k1, double L, double gamma0);
/* exact drift: the B -> 0 case of section III.A (eqs. 2-5), straight-line motion (N3) */
void orc_xdrift(int64_t n, double* x, double* px, double* y, double* py, double* sg, double* ps,
                double L, double beta0);
/* exact sector bend: section III.A (eqs. 2-5) restated from the circular motion it solves (N3) */
void orc_sbend(int64_t n, double* x, double* px, double* y, double* py, double* sg, double* ps,
               double L, double h, double beta0);
/* eq. 8: thick sextupole as the five-map symplectic composition (N3) */
void orc_sext(int64_t n, double* x, double* px, double* y, double* py, double* sg, double* ps,
              double k2, double L, double gamma0);
void orc_mult(int64_t n, double* x, double* px, double* y, double* py,
              int order, double knl, double ksl);
void orc_rf(int64_t n, double* sg, double* ps, double amp, double h, double circumference, double phi0);

/* ---- space-charge node pieces (section IV) */
int64_t orc_deposit_f64(int64_t n, const double* x, const double* y, const orc_grid* g, double* Q);
int64_t orc_deposit_fixed(int64_t n, const double* x, const double* y, const orc_grid* g, int64_t* Qi);
void orc_lambda_hist(int64_t n, const double* sg, const orc_grid* g, int64_t* cnt);
double orc_lambda_at(double sigma, const orc_grid* g, const int64_t* cnt, double n_real, int64_t n);
double orc_lambda_slope(double sigma, const orc_grid* g, const int64_t* cnt, double n_real, int64_t n);
double orc_gather_scalar(const orc_grid* g, const double* u, double x, double y, int* inside);
double orc_green_cell(double x, double y, double dx, double dy);
void orc_poisson_direct(const orc_grid* g, const double* Q, double n_total, double* u);
void orc_poisson_fft(const orc_grid* g, const double* Q, double n_total, double* u);
void orc_poisson_dirichlet(const orc_grid* g, const double* Q, double n_total, double* u);
void orc_field(const orc_grid* g, const double* u, double* Ex, double* Ey);
void orc_gather(const orc_grid* g, const double* Ex, const double* Ey, double x, double y,
                int* inside, double* ex, double* ey);

/* N4, eqs. 28-29: bicubic Bezier surface of the potential on the 4x4 stencil around the
   particle's cell and its analytic gradient.  *uval = u(x,y), *ex = -du/dx, *ey = -du/dy; all 0 outside the grid. */
void orc_gather_bicubic(const orc_grid* g, const double* u, double x, double y,
                        int* inside, double* uval, double* ex, double* ey);

/* own FFT, exported so that it can be pinned against the naive DFT */
void orc_fft(int n, double* re, double* im, int inverse);
void orc_dft_naive(int n, const double* re, const double* im, double* ore, double* oim, int inverse);

/* ---- whole SC node and whole tracking loop */
typedef struct {
    double* Q;  int64_t* Qi; double* u; double* Ex; double* Ey; int64_t* cnt; /* caller-allocated */
    int64_t n_inside;
} orc_work;

void orc_sc_kick(int64_t n, double* x, double* px, double* y, double* py, const double* sg, double* ps,
                 const orc_grid* g, const orc_beam* b, double L_sc, const orc_work* w);
int orc_scnode(int64_t n, double* x, double* px, double* y, double* py, const double* sg, double* ps,
               const orc_grid* g, const orc_beam* b, double L_sc, int poisson_direct, orc_work* w);

/* kind[i], ipar[i], par[10*i .. 10*i+9] describe row i (same meaning as include/sc_track.h but
   marshalled independently by the test harness).  stop_after_rows >= 0: stop after that many rows
   in total (a stop that lands on an SCNODE row stops after its deposit and field solve, before the
   kick), used to compare intermediate grids. */
int orc_track(int64_t n, double* x, double* px, double* y, double* py, double* sg, double* ps,
              int64_t n_rows, const int32_t* kind, const int32_t* ipar, const double* par,
              int32_t n_grids, const orc_grid* grids, const orc_beam* b,
              int64_t n_turns, int64_t stop_after_rows, int poisson_direct, orc_work* works);

/* out[33]: N, 6 means, 21 upper-triangular central second moments (row-major), eps_x, eps_y,
   eps_sigma, (slot 31, 32 unused by the oracle: set 0). */
void orc_moments(int64_t n, const double* x, const double* px, const double* y, const double* py,
                 const double* sg, const double* ps, double* out);

#endif
