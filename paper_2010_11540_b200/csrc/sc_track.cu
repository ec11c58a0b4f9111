// sc_track.cu -- host side of libsc_track (C ABI declared in include/sc_track.h).
// Product code: hand-written CUDA for sm_100a; no CPU fallback; shares nothing with oracle/.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <new>
#include <string>
#include <utility>
#include <vector>

#include "k_moments.cuh"
#include "k_poisson.cuh"
#include "k_poisson_fused.cuh"
#include "k_poisson_warp.cuh"
#include "k_poisson_cluster.cuh"
#include "k_push.cuh"
#include "sc_host.h"

using namespace sc;

#ifndef SC_EW_MAX
#define SC_EW_MAX 512     // largest grid (nodes per axis) whose kick is served from the shared-memory field window (A/B switch: with
                          // 128, grids of 256 and 512 nodes keep the larger accumulator-only deposit window and gather through the L1:
                          // measured 34.2 vs 24.0 us per launch at 256^2, 42.3 vs 37.3 at 512^2, cfg5 294 vs 229)
#endif

namespace {

thread_local std::string g_create_error = "";

struct PendingKick {
    int grid = -1;
    double L = 0.0;
    bool operator<(const PendingKick& o) const { return grid != o.grid ? grid < o.grid : L < o.L; }
    bool operator==(const PendingKick& o) const { return grid == o.grid && L == o.L; }
};

struct TurnGraph {
    cudaGraphExec_t exec = nullptr;
    PendingKick end;
    int64_t kernels = 0;
};

}  // namespace

struct sc_ctx {
    std::vector<sc_elem> rows;           // converted table (QUAD -> LINMAP, RF pre-scaled)
    std::vector<sc_grid> grids;
    std::vector<GridDev> gdev;
    sc_beam beam{};
    double gamma0 = 0, beta0 = 0, E0 = 0, r_c = 0, kappa = 0, circumference = 0;
    int64_t nmax = 0, n = 0;
    bool sixd = false, loaded = false;
    cudaStream_t stream = nullptr;
    bool use_graph = false, use_pdl = true, use_fused = false, use_ew = true, use_warp_fft = true, use_cluster = true;
    char* ws = nullptr;
    bool own_ws = false;
    int64_t ws_bytes = 0;
    // device pointers inside the workspace
    double* q[6] = {};
    unsigned long long* d_counters = nullptr;
    double* d_mom_partial = nullptr;
    double* d_mom_sums = nullptr;
    double* d_mom_cov = nullptr;
    int num_sms = 148;
    // tracking state
    int64_t pos = 0;                     // next row within the turn
    PendingKick pending;
    std::map<PendingKick, TurnGraph> graphs;
    int64_t launches = 0;
    int64_t ps_stores = 0;               // k_push launches so far that had to store psigma (6D and an RF row or a longitudinal kick in the launch)
    // sc_profile_turn: event pairs around every launch group
    bool profiling = false, skip_poisson = false, skip_push = false, noop = false;   // sc_profile_split's replays
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> ev_push, ev_poisson;
    std::string err;
};

namespace {

int fail(sc_ctx* c, int code, const std::string& msg) {
    if (c) c->err = msg; else g_create_error = msg;
    return code;
}

#define SC_CUDA(c, expr)                                                                          \
    do {                                                                                          \
        cudaError_t e_ = (expr);                                                                  \
        if (e_ != cudaSuccess)                                                                    \
            return fail((c), SC_ECUDA, std::string(#expr) + ": " + cudaGetErrorString(e_));       \
    } while (0)

}  // namespace

// used by the library's other translation units (sc_moments_static.cu): the message sc_last_error(NULL) returns
void sc::set_global_error(const std::string& msg) { g_create_error = msg; }

namespace {

size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }

// a pair of timing events, the first one recorded on the context's stream; on failure nothing is left behind
cudaError_t begin_event_pair(sc_ctx* c, cudaEvent_t* a, cudaEvent_t* b) {
    *a = *b = nullptr;
    cudaError_t e = cudaEventCreate(a);
    if (e == cudaSuccess) e = cudaEventCreate(b);
    if (e == cudaSuccess) e = cudaEventRecord(*a, c->stream);
    if (e != cudaSuccess) {
        if (*a) cudaEventDestroy(*a);
        if (*b) cudaEventDestroy(*b);
        *a = *b = nullptr;
    }
    return e;
}

bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }

// ---- workspace layout -----------------------------------------------------------------------
struct Layout {
    size_t off_q[6], off_counters, off_mom_partial, off_mom_sums, off_mom_cov;
    struct G { size_t rho, hist, rho_last, rhoi_last, hist_last, lam, A, BU, BV, phi, E, Ghat, twx, twy; };
    std::vector<G> g;
    size_t total;
};

constexpr int kMomBlocks = 592;   // 4 x 148
constexpr int kTraceSlots = 512 + 160 * 8;
#ifndef SC_DEP_W
#define SC_DEP_W 80
#endif
constexpr int kDepWindow = SC_DEP_W;          // private deposit window of grids up to 128 x 128, nodes per axis (multiple of 8); see launch_push
constexpr size_t kStageMinBytes = (size_t)96 << 20;   // particle sets beyond ~the L2 take the staged-load instantiation of k_push

Layout make_layout(int64_t n_elem, const sc_grid* grids, int32_t n_grids, int64_t nmax) {
    Layout L;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t r = o; o += align256(bytes); return r; };
    // particle arrays are copied in 16-byte units : even capacity
    for (int k = 0; k < 6; k++) L.off_q[k] = take((size_t)((nmax + 1) & ~(int64_t)1) * 8);
    L.off_counters = take((8 + kTraceSlots) * 8);   // 8 counters + the SC_TRACE builds' time stamps
    L.off_mom_partial = take((size_t)kMomBlocks * 21 * 8);
    L.off_mom_sums = take(8 * 8);
    L.off_mom_cov = take(21 * 8);
    for (int i = 0; i < n_grids; i++) {
        const sc_grid& s = grids[i];
        size_t nc = (size_t)s.nx * s.ny, nh = (size_t)(s.nx + 1) * s.ny, nb = (size_t)(s.nbins > 0 ? s.nbins : 1);
        Layout::G g;
        g.rho = take(nc * 8); g.hist = take(nb * 4); g.rho_last = take(nc * 8); g.rhoi_last = take(nc * 8);
        g.hist_last = take(nb * 8); g.lam = take((nb + 1) * 16);   // lambda pair table
        g.A = take(nh * 16); g.BU = take(2 * nh * 16); g.BV = g.BU + nh * 16;   // (U, V) as one block: the fused kernel's [j][kx][2]
        g.phi = take(nc * 8); g.E = take(nc * 16);
        g.Ghat = take((size_t)(s.nx + 1) * 2 * s.ny * 8);
        g.twx = take((size_t)s.nx * 16); g.twy = take((size_t)s.ny * 16);
        L.g.push_back(g);
    }
    L.total = o;
    return L;
}

int validate(const sc_elem* lat, int64_t n_elem, const sc_grid* grids, int32_t n_grids, int64_t nmax, std::string& why) {
    if (!lat || n_elem <= 0) { why = "empty lattice table"; return SC_EINVAL; }
    if (nmax <= 0) { why = "max_particles must be positive"; return SC_EINVAL; }
    if (n_grids < 0 || (n_grids > 0 && !grids)) { why = "bad grid array"; return SC_EINVAL; }
    for (int i = 0; i < n_grids; i++) {
        const sc_grid& g = grids[i];
        if (g.nx < 2 || g.ny < 2 || !(g.xmax > g.xmin) || !(g.ymax > g.ymin)) { why = "grid extent/size invalid"; return SC_EINVAL; }
        if (!is_pow2(g.nx) || !is_pow2(g.ny) || g.nx < 8 || g.ny < 8 || g.nx > 512 || g.ny > 512) {
            why = "grid nx, ny must be powers of two in 8..512 (hand-written radix-4/radix-2 FFTs)"; return SC_EUNSUPPORTED; }
        if (g.nbins < 0 || g.nbins > kMaxBins) { why = "nbins must be 0..4096"; return SC_EINVAL; }
        if (g.nbins > 0 && !(g.smax > g.smin)) { why = "lambda histogram range invalid"; return SC_EINVAL; }
        if (g.deposit_mode != SC_DEPOSIT_F64 && g.deposit_mode != SC_DEPOSIT_FIXED) { why = "deposit_mode must be 0 or 1"; return SC_EINVAL; }
        if (g.deposit_mode == SC_DEPOSIT_FIXED && (g.fixed_bits < 1 || g.fixed_bits > 20)) { why = "fixed_bits must be 1..20"; return SC_EINVAL; }
        // signed int64 accumulators: the worst case is every particle in one cell, N 2^(2s) < 2^63
        if (g.deposit_mode == SC_DEPOSIT_FIXED && std::ldexp((double)nmax, 2 * g.fixed_bits) >= 9223372036854775808.0) {
            why = "max_particles * 2^(2 fixed_bits) must stay below 2^63 (int64 accumulators)"; return SC_EINVAL; }
        if (g.long_kick != 0 && g.long_kick != 1) { why = "long_kick must be 0 or 1"; return SC_EINVAL; }
        if (g.long_kick && g.nbins <= 0) { why = "long_kick needs a lambda histogram (nbins > 0)"; return SC_EINVAL; }
        if (g.interp != SC_INTERP_BILINEAR && g.interp != SC_INTERP_BICUBIC) { why = "interp must be SC_INTERP_BILINEAR or SC_INTERP_BICUBIC"; return SC_EINVAL; }
        if (g.boundary != SC_BOUNDARY_OPEN && g.boundary != SC_BOUNDARY_PIPE) { why = "boundary must be SC_BOUNDARY_OPEN or SC_BOUNDARY_PIPE"; return SC_EINVAL; }
    }
    for (int64_t r = 0; r < n_elem; r++) {
        const sc_elem& e = lat[r];
        switch (e.kind) {
        case SC_DRIFT: case SC_LINMAP: case SC_RF: case SC_QUAD: case SC_CQUAD: case SC_SEXT: case SC_XDRIFT: case SC_SBEND: break;
        case SC_MULT: if (e.ipar < 0 || e.ipar > 20) { why = "MULT order must be 0..20"; return SC_EINVAL; } break;
        case SC_SCNODE: if (e.ipar < 0 || e.ipar >= n_grids) { why = "SCNODE refers to a grid that does not exist"; return SC_EINVAL; } break;
        default: why = "unknown row kind"; return SC_EINVAL;
        }
    }
    return SC_OK;
}

// ---- host precomputation ----------------------------------------------------------------------
// eq. 6 at psigma = 0
void quad_to_linmap(const sc_elem& q, sc_elem& out) {
    const double k1 = q.p[0], L = q.p[1];
    out = sc_elem{};
    out.kind = SC_LINMAP;
    double foc[4], def[4];
    if (k1 == 0.0) {
        foc[0] = 1; foc[1] = L; foc[2] = 0; foc[3] = 1;
        for (int i = 0; i < 4; i++) def[i] = foc[i];
    } else {
        const double w = std::sqrt(std::fabs(k1)), ph = w * L;
        const double c = std::cos(ph), s = std::sin(ph), ch = std::cosh(ph), sh = std::sinh(ph);
        foc[0] = c; foc[1] = s / w; foc[2] = -w * s; foc[3] = c;
        def[0] = ch; def[1] = sh / w; def[2] = w * sh; def[3] = ch;
    }
    const double* mx = k1 >= 0 ? foc : def;
    const double* my = k1 >= 0 ? def : foc;
    for (int i = 0; i < 4; i++) { out.p[i] = mx[i]; out.p[4 + i] = my[i]; }
    out.p[8] = L;
}

// host FFT in long double (only used once per grid at create time)
void host_fft(std::vector<long double>& re, std::vector<long double>& im, size_t off, size_t stride, int n) {
    const long double PI = 3.14159265358979323846264338327950288L;
    for (int i = 1, j = 0; i < n; i++) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { std::swap(re[off + i * stride], re[off + j * stride]); std::swap(im[off + i * stride], im[off + j * stride]); }
    }
    for (int len = 2; len <= n; len <<= 1) {
        for (int k = 0; k < len / 2; k++) {
            const long double ang = -2.0L * PI * k / len;
            const long double wr = cosl(ang), wi = sinl(ang);
            for (int s = 0; s < n; s += len) {
                const size_t a = off + (size_t)(s + k) * stride, b = off + (size_t)(s + k + len / 2) * stride;
                const long double tr = re[b] * wr - im[b] * wi, ti = re[b] * wi + im[b] * wr;
                re[b] = re[a] - tr; im[b] = im[a] - ti;
                re[a] += tr; im[a] += ti;
            }
        }
    }
}

// Cell-averaged 2D open-boundary Green's function of laplace(u) = -f:
//   G(x,y) = -(1/(4 pi dx dy)) * integral over the cell centred at (x,y) of ln(x'^2 + y'^2),
// closed form via the antiderivative  x y ln(x^2+y^2) - 3 x y + x^2 atan(y/x) + y^2 atan(x/y).
long double green_primitive(long double x, long double y) {
    return x * y * logl(x * x + y * y) - 3.0L * x * y + x * x * atanl(y / x) + y * y * atanl(x / y);
}

// Ghat[kx][ky] (kx = 0..nx, ky = 0..2ny-1): real 2D DFT of the even periodic extension of G on the
// doubled grid (distance min(a, 2nx - a); the unused wrap entry a = nx takes G(nx dx)).
void compute_ghat(const sc_grid& g, std::vector<double>& out) {
    const int nx = g.nx, ny = g.ny, Lx = 2 * nx, Ly = 2 * ny;
    const long double dx = ((long double)g.xmax - g.xmin) / (nx - 1), dy = ((long double)g.ymax - g.ymin) / (ny - 1);
    const double dxd = (g.xmax - g.xmin) / (double)(nx - 1), dyd = (g.ymax - g.ymin) / (double)(ny - 1);
    const long double PI = 3.14159265358979323846264338327950288L;
    std::vector<long double> tab((size_t)(nx + 1) * (ny + 1));
    for (int b = 0; b <= ny; b++)
        for (int a = 0; a <= nx; a++) {
            // node offsets use the same double dx, dy as the kernels' grid
            const long double x = (long double)a * dxd, y = (long double)b * dyd;
            const long double x1 = x - 0.5L * dxd, x2 = x + 0.5L * dxd, y1 = y - 0.5L * dyd, y2 = y + 0.5L * dyd;
            const long double I = green_primitive(x2, y2) - green_primitive(x1, y2) - green_primitive(x2, y1) + green_primitive(x1, y1);
            tab[(size_t)b * (nx + 1) + a] = -I / (4.0L * PI * dxd * dyd);
        }
    (void)dx; (void)dy;
    std::vector<long double> re((size_t)Lx * Ly), im((size_t)Lx * Ly, 0.0L);
    for (int b = 0; b < Ly; b++)
        for (int a = 0; a < Lx; a++) {
            const int da = a <= nx ? a : Lx - a, db = b <= ny ? b : Ly - b;
            re[(size_t)b * Lx + a] = tab[(size_t)db * (nx + 1) + da];
        }
    for (int b = 0; b < Ly; b++) host_fft(re, im, (size_t)b * Lx, 1, Lx);
    for (int a = 0; a < Lx; a++) host_fft(re, im, (size_t)a, Lx, Ly);
    out.resize((size_t)(nx + 1) * Ly);
    for (int kx = 0; kx <= nx; kx++)
        for (int ky = 0; ky < Ly; ky++) out[(size_t)kx * Ly + ky] = (double)re[(size_t)ky * Lx + kx];
}

// Conducting pipe (eqs. 15-27): with laplace(u~) = -f, f = Q/(N dx dy), the spectrum of the odd extension is
// multiplied by 1/(dx dy) / (4 (sin^2(pi p/2nx)/dx^2 + sin^2(pi q/2ny)/dy^2)) (eq. 25; the kernels apply the common
// 1/(Lx Ly N)); the (0,0) mode is empty by oddness and set to 0.  Same [kx][ky] layout as compute_ghat.
void compute_pipe_symbol(const sc_grid& g, std::vector<double>& out) {
    const int nx = g.nx, ny = g.ny, Ly = 2 * ny;
    const long double dx = (long double)((g.xmax - g.xmin) / (double)(nx - 1)), dy = (long double)((g.ymax - g.ymin) / (double)(ny - 1));
    const long double PI = 3.14159265358979323846264338327950288L;
    out.resize((size_t)(nx + 1) * Ly);
    for (int kx = 0; kx <= nx; kx++)
        for (int ky = 0; ky < Ly; ky++) {
            const long double sp = sinl(PI * kx / (2.0L * nx)), sq = sinl(PI * ky / (2.0L * ny));
            const long double den = 4.0L * (sp * sp / (dx * dx) + sq * sq / (dy * dy));
            out[(size_t)kx * Ly + ky] = (kx == 0 && ky == 0) ? 0.0 : (double)(1.0L / (den * dx * dy));
        }
}

void compute_twiddles(int L, std::vector<double2>& tw) {
    const long double PI = 3.14159265358979323846264338327950288L;
    tw.resize(L / 2);
    for (int k = 0; k < L / 2; k++) {
        const long double ang = -2.0L * PI * k / L;
        tw[k] = make_double2((double)cosl(ang), (double)sinl(ang));
    }
}

// head of the push kernel's dynamic shared memory (the lambda histogram, the work-queue counter, the flush's row bounds and an mbarrier, padded to 128 B); the grid window follows
size_t push_smem_head(int nh) { return ((((4 * (size_t)nh + 12 + 7) & ~(size_t)7) + 8) + 127) & ~(size_t)127; }

// shared-memory window of a deposit grid: the whole grid if it fits beside the histogram,
// else a centred window with the grid's aspect ratio (multiples of 8 nodes); particles outside it deposit with
// L2 atomics.  (A window fitted to the measured beam extent was tried and dropped: cfg3's beam covers most of
// the grid somewhere on the ring, so one window per grid saves nothing.)
size_t push_stage_bytes(int ew) { return ew == 2 ? 128 + (size_t)kPushWarps * 6 * kChunk * 8 + (size_t)kPushWarps * 8 : 0; }

void choose_window(GridDev& g, int max_bins_any, int ew) {
    // plain: 8 bytes per window node (deposit accumulators); EW: 24 (+ the node fields) and the lambda pair table
    // EW: + the lambda pair table, and with SC_STAGE the per-warp particle buffers and their mbarriers
    const size_t fixed = push_smem_head(max_bins_any) + (ew ? (size_t)(max_bins_any + 1) * 16 + push_stage_bytes(ew) : 0);
    const size_t cells = (kSmemBudget - fixed) / (ew ? 24 : 8);
    if ((size_t)g.nx * g.ny <= cells) { g.wi0 = 0; g.wj0 = 0; g.wnx = g.nx; g.wny = g.ny; return; }
    const double scale = std::sqrt((double)cells / ((double)g.nx * g.ny));
    int wx = ((int)(g.nx * scale)) & ~7, wy = ((int)(g.ny * scale)) & ~7;
    if (wx > g.nx) wx = g.nx;
    if (wy > g.ny) wy = g.ny;
    // a very oblong grid (512 x 8 beside 4096 bins and the staged particle buffers) would round its short axis down to 0 nodes:
    // keep at least 8 nodes (the smallest grid axis) on either axis and take the cells from the long one
    if (wx < 8) wx = 8;
    if (wy < 8) wy = 8;
    while ((size_t)wx * wy > cells && (wx > 8 || wy > 8)) { if (wx >= wy) wx -= 8; else wy -= 8; }
    g.wnx = wx; g.wny = wy; g.wi0 = (g.nx - wx) / 2; g.wj0 = (g.ny - wy) / 2;
}

size_t push_smem_bytes(const sc_ctx* c, const PushArgs& a, int dep, int ew) {
    const int nh = (dep && c->sixd) ? a.dg.nbins : 0;
    size_t b = push_smem_head(nh) + (dep ? (size_t)a.dg.wnx * a.dg.wny * 8 : 0);
    if (ew && a.do_kick) b += (size_t)a.kg.wnx * a.kg.wny * 16 + (size_t)(a.kg.nbins + 1) * 16;
    if (ew) b += push_stage_bytes(ew);
    return b;
}

// rows -> program slots (sc_device.cuh OP_*).  QUAD rows are already LINMAPs, RF rows pre-scaled.
double2 prog_hdr(int op, int ipar, double v) {
    const unsigned long long bits = (unsigned long long)(unsigned int)op | ((unsigned long long)(unsigned int)ipar << 32);
    double h;
    std::memcpy(&h, &bits, 8);
    return make_double2(h, v);
}

// Encode rows [r, s) (no SCNODE among them) into a->prog until the slots run out; returns the first row NOT
// encoded.  A DRIFT directly followed by a normal thin multipole of order <= 3 (or any order-0 kick) becomes one
// fused DMn op.  a == nullptr: dry run (only the return value).
int64_t encode_piece(const sc_ctx* c, int64_t r, int64_t s, PushArgs* a) {
    int n = 0;
    auto put = [&](double2 v) { if (a) a->prog[n] = v; n++; };
    const int cap = kMaxProgSlots - 1;            // keep one slot for OP_END
    while (r < s) {
        const sc_elem& e = c->rows[r];
        const bool fusable_next = e.kind == SC_DRIFT && r + 1 < s && c->rows[r + 1].kind == SC_MULT &&
                                  c->rows[r + 1].ipar <= 3 && (c->rows[r + 1].ipar == 0 || c->rows[r + 1].p[1] == 0.0);
        int need = 1;
        switch (e.kind) {
        case SC_DRIFT: need = fusable_next ? 2 : 1; break;
        case SC_LINMAP: need = 5; break;
        case SC_MULT: need = (e.ipar >= 1 && e.ipar <= 3 && e.p[1] == 0.0) ? 1 : 2; break;
        case SC_RF: need = 2; break;
        case SC_CQUAD: need = 2; break;
        case SC_SEXT: need = 5; break;
        case SC_XDRIFT: need = 1; break;
        case SC_SBEND: need = 3; break;
        default: need = 0; break;
        }
        if (n + need > cap) break;
        switch (e.kind) {
        case SC_DRIFT:
            if (fusable_next) {
                const sc_elem& m = c->rows[r + 1];
                put(prog_hdr(OP_DM0 + m.ipar, m.ipar, e.p[0]));
                put(make_double2(m.p[0], m.p[1]));
                r++;                                  // the multipole row is consumed too
            } else {
                put(prog_hdr(OP_DRIFT, 0, e.p[0]));
            }
            break;
        case SC_LINMAP:
            put(prog_hdr(OP_LINMAP, 0, e.p[8]));
            for (int k = 0; k < 4; k++) put(make_double2(e.p[2 * k], e.p[2 * k + 1]));
            break;
        case SC_MULT:
            if (e.ipar >= 1 && e.ipar <= 3 && e.p[1] == 0.0) {
                put(prog_hdr(OP_M0 + e.ipar, e.ipar, e.p[0]));
            } else if (e.ipar == 0) {
                put(prog_hdr(OP_M0, 0, e.p[0]));
                put(make_double2(e.p[1], 0.0));
            } else {
                put(prog_hdr(OP_MULTG, e.ipar, e.p[0]));
                put(make_double2(e.p[1], 0.0));
            }
            break;
        case SC_SEXT: {
            // eq. 8: drift aL, kick k2 bL, drift cL, kick k2 bL, drift aL -- two fused drift+sextupole ops and a drift
            const double sa = 0.5 * (1.0 - 1.0 / std::sqrt(3.0)), sb = 0.5, sc3 = 1.0 / std::sqrt(3.0);
            put(prog_hdr(OP_DM2, 2, sa * e.p[1])); put(make_double2(e.p[0] * (sb * e.p[1]), 0.0));
            put(prog_hdr(OP_DM2, 2, sc3 * e.p[1])); put(make_double2(e.p[0] * (sb * e.p[1]), 0.0));
            put(prog_hdr(OP_DRIFT, 0, sa * e.p[1]));
            break;
        }
        case SC_XDRIFT:
            put(prog_hdr(OP_XDRIFT, 0, e.p[0]));
            break;
        case SC_SBEND:
            put(prog_hdr(OP_SBEND, 0, e.p[0]));
            put(make_double2(e.p[1], 0.0));
            put(make_double2(std::sin(e.p[0] * e.p[1]), std::cos(e.p[0] * e.p[1])));
            break;
        case SC_CQUAD:
            put(prog_hdr(OP_CQUAD, 0, e.p[0]));
            put(make_double2(e.p[1], 0.0));
            break;
        case SC_RF:
            put(prog_hdr(OP_RF, 0, e.p[0]));
            put(make_double2(e.p[1], e.p[2]));
            break;
        default: break;
        }
        r++;
    }
    put(prog_hdr(OP_END, 0, 0.0));
    if (a) a->nslots = n;
    return r;
}

// Launch with the programmatic-stream-serialization attribute (PDL): the kernel may be scheduled while its
// predecessor in the stream is still running; it blocks in pdl_wait() until that one has completed.
template <typename... KArgs, typename... Args>
cudaError_t launch_k(const sc_ctx* c, void (*kern)(KArgs...), int blocks, int threads, size_t smem, Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)blocks); cfg.blockDim = dim3((unsigned)threads);
    cfg.dynamicSmemBytes = smem; cfg.stream = c->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = c->use_pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, std::forward<Args>(args)...);
}

// The same for a kernel that runs as ONE thread-block cluster of `blocks` CTAs (k_poisson_cluster.cuh).
template <typename... KArgs, typename... Args>
cudaError_t launch_cluster(const sc_ctx* c, void (*kern)(KArgs...), int blocks, int threads, size_t smem, Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)blocks); cfg.blockDim = dim3((unsigned)threads);
    cfg.dynamicSmemBytes = smem; cfg.stream = c->stream;
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)blocks; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = c->use_pdl ? 2 : 1;
    return cudaLaunchKernelEx(&cfg, kern, std::forward<Args>(args)...);
}

template <bool SIXD, int DEP>
cudaError_t launch_push_t(const sc_ctx* c, const PushArgs& a, size_t smem, int blocks, bool cq, int ew) {
    if (cq) return launch_k(c, k_push<SIXD, DEP, true, 0>, blocks, kPushThreadsCQ, smem, a);
    if (ew == 2) return launch_k(c, k_push<SIXD, DEP, false, 2>, blocks, kPushThreads, smem, a);
    if (ew == 1) return launch_k(c, k_push<SIXD, DEP, false, 1>, blocks, kPushThreads, smem, a);
    return launch_k(c, k_push<SIXD, DEP, false, 0>, blocks, kPushThreads, smem, a);
}

// opt in to 227 KB of dynamic shared memory for every push variant (once per process, outside capture)
cudaError_t configure_kernels() {
    cudaError_t e = cudaSuccess;
    auto set = [&](const void* f) {
        if (e == cudaSuccess) e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBudget);
    };
    set((const void*)k_push<true, 0>); set((const void*)k_push<true, 1>); set((const void*)k_push<true, 2>);
    set((const void*)k_push<false, 0>); set((const void*)k_push<false, 1>); set((const void*)k_push<false, 2>);
    set((const void*)k_push<true, 0, true>); set((const void*)k_push<true, 1, true>); set((const void*)k_push<true, 2, true>);
    set((const void*)k_push<false, 0, true>); set((const void*)k_push<false, 1, true>); set((const void*)k_push<false, 2, true>);
    set((const void*)k_push<true, 0, false, 1>); set((const void*)k_push<true, 1, false, 1>); set((const void*)k_push<true, 2, false, 1>);
    set((const void*)k_push<false, 0, false, 1>); set((const void*)k_push<false, 1, false, 1>); set((const void*)k_push<false, 2, false, 1>);
    set((const void*)k_push<true, 0, false, 2>); set((const void*)k_push<true, 1, false, 2>); set((const void*)k_push<true, 2, false, 2>);
    set((const void*)k_push<false, 0, false, 2>); set((const void*)k_push<false, 1, false, 2>); set((const void*)k_push<false, 2, false, 2>);
    auto setf = [&](const void* f, size_t bytes) {
        if (e == cudaSuccess) e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    };
    setf((const void*)k_poisson_fused<64, 64>, fused_smem_bytes<64, 64>());
    setf((const void*)k_poisson_fused<128, 128>, fused_smem_bytes<128, 128>());
    setf((const void*)k_poisson_fused<64, 128>, fused_smem_bytes<64, 128>());
    setf((const void*)k_poisson_fused<128, 64>, fused_smem_bytes<128, 64>());
    // one-cluster field solve: 16 CTAs is a non-portable cluster size
    setf((const void*)k_poisson_cluster, kPcSmemBytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute((const void*)k_poisson_cluster, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    return e;
}

// one push launch: [kick] rows [r0,r1) [deposit on grid dep_grid]
int launch_push(sc_ctx* c, int r0, int r1, const PendingKick& kick, int dep_grid) {
    PushArgs a{};
    for (int k = 0; k < 6; k++) a.q[k] = c->q[k];
    a.n = c->n;
    if (encode_piece(c, r0, r1, &a) != r1) return fail(c, SC_EINVAL, "internal: piece does not fit the program slots");
    a.inv_gamma2 = 1.0 / (c->gamma0 * c->gamma0);
    a.beta0_2 = c->beta0 * c->beta0;
    a.counters = c->d_counters;
    a.noop = c->noop || c->skip_push;
    a.do_kick = kick.grid >= 0;
    if (a.do_kick) {
        a.kg = c->gdev[kick.grid];
        a.kick_scale = c->kappa * kick.L;
        a.lam_const = c->beam.line_density;
    }
    int dep = 0;
    a.do_dep = dep_grid >= 0;
    if (a.do_dep) {
        a.dg = c->gdev[dep_grid];
        dep = a.dg.mode == SC_DEPOSIT_FIXED ? 2 : 1;
    }
    a.ps_changes = a.do_kick && a.kg.long_kick;
    for (int r = r0; r < r1; r++) a.ps_changes = a.ps_changes || c->rows[r].kind == SC_RF;
    if (c->sixd && a.ps_changes) c->ps_stores++;
    bool cq = false;
    for (int r = r0; r < r1; r++) cq = cq || c->rows[r].kind == SC_CQUAD || c->rows[r].kind == SC_XDRIFT || c->rows[r].kind == SC_SBEND;
    cq = cq || (a.do_kick && a.kg.interp == SC_INTERP_BICUBIC);      // the 16-load bicubic kick lives in the heavy instantiation too
    // field window in shared memory (EW): plain instantiation, a bilinear kick to serve, kick and deposit on the same grid.  The
    // window is ~96 x 96 nodes whatever the grid (24 bytes per node): the whole beam at 128 x 128, +-3 sigma of cfg3's beam at
    // 256 x 256, its core at 512 x 512; particles outside it gather through the L1 and deposit with L2 atomics
    int ew = (c->use_ew && !cq && a.do_kick && a.kg.nx <= SC_EW_MAX && a.kg.ny <= SC_EW_MAX && (!a.do_dep || dep_grid == kick.grid)) ? 1 : 0;
    // staged particle loads pay when the particles stream from HBM, not when they sit in L2 (k_push.cuh): by size of the set
    if (ew && (size_t)c->n * (c->sixd ? 6 : 4) * 8 > kStageMinBytes) ew = 2;
    if (ew) {
        int max_bins = 0;
        for (const auto& g : c->grids) if (g.nbins > max_bins) max_bins = g.nbins;
        choose_window(a.kg, max_bins, ew);
        if (a.do_dep) {
            a.dg.wi0 = a.kg.wi0; a.dg.wj0 = a.kg.wj0; a.dg.wnx = a.kg.wnx; a.dg.wny = a.kg.wny;
            // The private DEPOSIT window may be smaller than the field window: its cells are flushed with one L2 atomic each
            // by every CTA (the flush is bound by the L2's atomic throughput), while a particle outside it costs four L2 atomics
            // spread over the piece loop, when those units are idle.  Measured at cfg3 (128 x 128, beam sigma 8-14 nodes), per
            // node in the graph: 96 / 88 / 80 / 72 / 64 / 48 / 32 nodes per axis = 29.43 / 28.81 / 28.78 / 28.77 / 29.01 /
            // 29.96 / 39.70 us.  On 256 and 512 grids the window covers fewer sigma and shrinking it loses (256: 39.1 / 39.4 /
            // 40.7 / 41.2 us at 96 / 88 / 80 / 72): there it stays the field window.
            if (a.dg.nx <= 128 && a.dg.ny <= 128) {
                if (a.dg.wnx > kDepWindow) { a.dg.wi0 += (a.dg.wnx - kDepWindow) / 2; a.dg.wnx = kDepWindow; }
                if (a.dg.wny > kDepWindow) { a.dg.wj0 += (a.dg.wny - kDepWindow) / 2; a.dg.wny = kDepWindow; }
            }
        }
    }
    const size_t smem = push_smem_bytes(c, a, dep, ew);
    // one persistent CTA per SM; each owns a contiguous, even-sized particle range
    int blocks = (int)((c->n + 255) / 256);
    if (blocks > c->num_sms) blocks = c->num_sms;
    if (blocks < 1) blocks = 1;
    a.per_cta = (((c->n + blocks - 1) / blocks) + 1) & ~(long long)1;
    {
        // fp64 deposit mode: the CTA-private grid accumulates round(w 2^e); e leaves room for every particle of the CTA in one cell
        int e = 62;
        for (long long m = a.per_cta; m > 0; m >>= 1) e--;
        if (e > 52) e = 52;
        a.dep_scale = std::ldexp(1.0, e); a.dep_inv = std::ldexp(1.0, -e);
    }
    cudaError_t e;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    if (c->profiling && (e = begin_event_pair(c, &ev0, &ev1)) != cudaSuccess) return fail(c, SC_ECUDA, std::string("k_push timing events: ") + cudaGetErrorString(e));
    if (c->sixd) {
        if (dep == 0) e = launch_push_t<true, 0>(c, a, smem, blocks, cq, ew);
        else if (dep == 1) e = launch_push_t<true, 1>(c, a, smem, blocks, cq, ew);
        else e = launch_push_t<true, 2>(c, a, smem, blocks, cq, ew);
    } else {
        if (dep == 0) e = launch_push_t<false, 0>(c, a, smem, blocks, cq, ew);
        else if (dep == 1) e = launch_push_t<false, 1>(c, a, smem, blocks, cq, ew);
        else e = launch_push_t<false, 2>(c, a, smem, blocks, cq, ew);
    }
    if (c->profiling) {
        if (e == cudaSuccess) e = cudaEventRecord(ev1, c->stream);
        if (e == cudaSuccess) c->ev_push.emplace_back(ev0, ev1);
        else { cudaEventDestroy(ev0); cudaEventDestroy(ev1); }
    }
    if (e != cudaSuccess) return fail(c, SC_ECUDA, std::string("k_push launch: ") + cudaGetErrorString(e));
    c->launches++;
    return SC_OK;
}

int launch_poisson(sc_ctx* c, int grid) {
    if (c->skip_poisson) return SC_OK;
    PoissonArgs p{};
    p.g = c->gdev[grid];
    p.noop = c->noop;
    const int nx = p.g.nx, ny = p.g.ny;
    p.scale = 1.0 / ((double)(2 * nx) * (double)(2 * ny) * (double)c->n);
    p.lam_scale = p.g.nbins > 0 ? c->beam.n_real / ((double)c->n * p.g.ds) : 0.0;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    cudaError_t e;
    if (c->profiling && (e = begin_event_pair(c, &ev0, &ev1)) != cudaSuccess) return fail(c, SC_ECUDA, std::string("field-solve timing events: ") + cudaGetErrorString(e));
    const bool fused = c->use_fused && (nx == 64 || nx == 128) && (ny == 64 || ny == 128);
    if (fused) {
        // one launch: register transforms, two grid barriers (k_poisson_fused.cuh)
        const int blocks = (nx + 1 + kFusedGroups - 1) / kFusedGroups;
        if (nx == 64 && ny == 64) e = launch_k(c, k_poisson_fused<64, 64>, blocks, kFusedThreads, fused_smem_bytes<64, 64>(), p, c->d_counters);
        else if (nx == 128 && ny == 128) e = launch_k(c, k_poisson_fused<128, 128>, blocks, kFusedThreads, fused_smem_bytes<128, 128>(), p, c->d_counters);
        else if (nx == 64) e = launch_k(c, k_poisson_fused<64, 128>, blocks, kFusedThreads, fused_smem_bytes<64, 128>(), p, c->d_counters);
        else e = launch_k(c, k_poisson_fused<128, 64>, blocks, kFusedThreads, fused_smem_bytes<128, 64>(), p, c->d_counters);
        if (e == cudaSuccess) c->launches += 1;
    } else if (c->use_cluster && nx == kPcN && ny == kPcN) {
        // one launch of one 16-CTA cluster, hand-overs through distributed shared memory (k_poisson_cluster.cuh)
        e = launch_cluster(c, k_poisson_cluster, kPcCtas, kPcThreads, kPcSmemBytes, p, c->d_counters);
        if (e == cudaSuccess) c->launches += 1;
    } else if (c->use_warp_fft && (nx == 64 || nx == 128) && (ny == 64 || ny == 128)) {
        // three launches, one warp per transform (k_poisson_warp.cuh)
        const int b1 = (ny / 2 + kPwWarps - 1) / kPwWarps, b2 = (nx + 1 + kPwWarps - 1) / kPwWarps, b3 = (ny + kPwWarps - 1) / kPwWarps;
#define SC_PW(NX_, NY_)                                                                                                   \
        do {                                                                                                              \
            e = launch_k(c, k_pw_rows_fwd<NX_, NY_>, b1, kPwThreads, pw_smem_bytes<2 * NX_>(), p, c->d_counters);         \
            if (e == cudaSuccess) e = launch_k(c, k_pw_cols<NX_, NY_>, b2, kPwThreads, pw_smem_bytes<2 * NY_>(), p);      \
            if (e == cudaSuccess) e = launch_k(c, k_pw_rows_inv<NX_, NY_>, b3, kPwThreads, pw_smem_bytes<2 * NX_>(), p);  \
        } while (0)
        if (nx == 64 && ny == 64) SC_PW(64, 64);
        else if (nx == 128 && ny == 128) SC_PW(128, 128);
        else if (nx == 64) SC_PW(64, 128);
        else SC_PW(128, 64);
#undef SC_PW
        if (e == cudaSuccess) c->launches += 3;
    } else {
        const size_t smx = (size_t)(2 * (2 * nx) + nx) * sizeof(double2), smy = (size_t)(2 * (2 * ny) + ny) * sizeof(double2);
        e = launch_k(c, k_rows_fwd, ny / 2, nx, smx, p, c->d_counters);
        if (e == cudaSuccess) e = launch_k(c, k_cols, nx + 1, ny, smy, p);
        if (e == cudaSuccess) e = launch_k(c, k_rows_inv, ny, nx, smx, p);
        if (e == cudaSuccess) c->launches += 3;
    }
    if (c->profiling) {
        if (e == cudaSuccess) e = cudaEventRecord(ev1, c->stream);
        if (e == cudaSuccess) c->ev_poisson.emplace_back(ev0, ev1);
        else { cudaEventDestroy(ev0); cudaEventDestroy(ev1); }
    }
    if (e != cudaSuccess) return fail(c, SC_ECUDA, std::string("poisson launch: ") + cudaGetErrorString(e));
    return SC_OK;
}

// rows [a, b) of one turn (no wrap); honours and updates c->pending
int run_rows(sc_ctx* c, int64_t a, int64_t b) {
    int64_t start = a;
    while (start < b) {
        int64_t s = start;
        while (s < b && c->rows[s].kind != SC_SCNODE) s++;
        // pieces of at most kMaxProgSlots program slots; kick with the first piece, deposit with the last
        int64_t r = start;
        const int dep_grid = s < b ? c->rows[s].ipar : -1;
        do {
            const int64_t r1 = encode_piece(c, r, s, nullptr);
            const bool last = r1 == s;
            if (r1 > r || c->pending.grid >= 0 || (last && dep_grid >= 0)) {
                int rc = launch_push(c, (int)r, (int)r1, c->pending, last ? dep_grid : -1);
                if (rc) return rc;
                c->pending = PendingKick{};
            }
            r = r1;
        } while (r < s);
        if (s < b) {
            int rc = launch_poisson(c, dep_grid);
            if (rc) return rc;
            c->pending.grid = dep_grid;
            c->pending.L = c->rows[s].p[0];
            start = s + 1;
        } else {
            start = b;
        }
    }
    return SC_OK;
}

int flush_pending(sc_ctx* c) {
    if (c->pending.grid < 0) return SC_OK;
    int rc = launch_push(c, 0, 0, c->pending, -1);
    c->pending = PendingKick{};
    return rc;
}

void drop_graphs(sc_ctx* c) {
    for (auto& kv : c->graphs) if (kv.second.exec) cudaGraphExecDestroy(kv.second.exec);
    c->graphs.clear();
}

// one whole turn starting at row 0 with the current pending kick, via a cached CUDA graph
int run_turn_graph(sc_ctx* c) {
    const int64_t R = (int64_t)c->rows.size();
    auto it = c->graphs.find(c->pending);
    if (it == c->graphs.end()) {
        const PendingKick start = c->pending;
        const int64_t before = c->launches;
        SC_CUDA(c, cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
        int rc = run_rows(c, 0, R);
        cudaGraph_t graph = nullptr;
        cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
        if (rc || e != cudaSuccess) {                 // nothing ran: the tracking state is what it was before the capture
            if (graph) cudaGraphDestroy(graph);
            c->pending = start; c->launches = before;
            return rc ? rc : fail(c, SC_ECUDA, std::string("cudaStreamEndCapture: ") + cudaGetErrorString(e));
        }
        TurnGraph tg;
        tg.end = c->pending;
        tg.kernels = c->launches - before;
        c->launches = before;             // capture launched nothing
        e = cudaGraphInstantiate(&tg.exec, graph, 0);
        cudaGraphDestroy(graph);
        if (e != cudaSuccess) { c->pending = start; return fail(c, SC_ECUDA, std::string("cudaGraphInstantiate: ") + cudaGetErrorString(e)); }
        it = c->graphs.emplace(start, tg).first;
    }
    SC_CUDA(c, cudaGraphLaunch(it->second.exec, c->stream));
    c->launches += it->second.kernels;
    c->pending = it->second.end;
    return SC_OK;
}

int step_rows(sc_ctx* c, int64_t total) {
    const int64_t R = (int64_t)c->rows.size();
    while (total > 0) {
        if (c->pos == 0 && total >= R && c->use_graph) {
            int rc = run_turn_graph(c);
            if (rc) return rc;
            total -= R;
            continue;
        }
        const int64_t k = total < R - c->pos ? total : R - c->pos;
        int rc = run_rows(c, c->pos, c->pos + k);
        if (rc) return rc;
        c->pos = (c->pos + k) % R;
        total -= k;
    }
    return SC_OK;
}

}  // namespace

// ================================================================================== C ABI
extern "C" {

int sc_workspace_bytes(const sc_elem* lat, int64_t n_elem, const sc_grid* grids, int32_t n_grids,
                       int64_t max_particles, int64_t* bytes_out) {
    std::string why;
    int rc = validate(lat, n_elem, grids, n_grids, max_particles, why);
    if (rc) return fail(nullptr, rc, why);
    if (!bytes_out) return fail(nullptr, SC_EINVAL, "bytes_out is NULL");
    *bytes_out = (int64_t)make_layout(n_elem, grids, n_grids, max_particles).total;
    return SC_OK;
}

int sc_create(sc_ctx** out, const sc_elem* lat, int64_t n_elem, const sc_grid* grids, int32_t n_grids,
              const sc_beam* beam, int64_t max_particles, void* workspace, int64_t workspace_bytes,
              void* stream, uint64_t flags) {
    if (!out) return fail(nullptr, SC_EINVAL, "out is NULL");
    *out = nullptr;
    if (!beam) return fail(nullptr, SC_EINVAL, "beam is NULL");
    if (flags & ~(uint64_t)(SC_FLAG_NO_PDL | SC_FLAG_FUSED_POISSON | SC_FLAG_NO_FIELD_WINDOW | SC_FLAG_BLOCK_FFT_POISSON | SC_FLAG_WARP_FFT_POISSON)) return fail(nullptr, SC_EINVAL, "unknown flag bits");
    std::string why;
    int rc = validate(lat, n_elem, grids, n_grids, max_particles, why);
    if (rc) return fail(nullptr, rc, why);
    if (!(beam->kinetic_eV > 0) || !(beam->mass_eV > 0) || beam->charge == 0)
        return fail(nullptr, SC_EINVAL, "beam needs kinetic_eV > 0, mass_eV > 0, charge != 0");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
        return fail(nullptr, SC_ECUDA, "no CUDA device: libsc_track has no CPU fallback");

    sc_ctx* c = new (std::nothrow) sc_ctx();
    if (!c) return fail(nullptr, SC_ENOMEM, "out of host memory");
    auto bail = [&](int code, const std::string& msg) { g_create_error = msg; sc_destroy(c); return code; };

    c->beam = *beam;
    c->stream = (cudaStream_t)stream;
    c->use_graph = stream != nullptr;     // the legacy default stream cannot be captured
    c->use_pdl = !(flags & SC_FLAG_NO_PDL);
    c->use_fused = (flags & SC_FLAG_FUSED_POISSON) != 0;
    c->use_ew = !(flags & SC_FLAG_NO_FIELD_WINDOW);
    c->use_warp_fft = !(flags & SC_FLAG_BLOCK_FFT_POISSON);
    c->use_cluster = !(flags & (SC_FLAG_BLOCK_FFT_POISSON | SC_FLAG_WARP_FFT_POISSON));
    c->nmax = max_particles;
    c->grids.assign(grids, grids + n_grids);
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev);
    {
        cudaError_t ce = configure_kernels();
        if (ce != cudaSuccess) return bail(SC_ECUDA, std::string("cudaFuncSetAttribute(k_push): ") + cudaGetErrorString(ce));
    }
    if (c->use_cluster) {
        // can this device place one 16-CTA cluster of the field solve at all (a GPC with 16 SMs, no partitioning in the way)?
        // If not, 128 x 128 grids take the three-launch path like the other sizes.
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(kPcCtas); cfg.blockDim = dim3(kPcThreads); cfg.dynamicSmemBytes = kPcSmemBytes;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = kPcCtas; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        int n_clusters = 0;
        if (cudaOccupancyMaxActiveClusters(&n_clusters, (const void*)k_poisson_cluster, &cfg) != cudaSuccess || n_clusters < 1) {
            cudaGetLastError();
            c->use_cluster = false;
        }
    }

    // reference particle (eq. 11): r_c = q^2 e/(4 pi eps0) [V m] / (m c^2 [eV])
    {
        const double e_charge = 1.602176634e-19, eps0 = 8.8541878128e-12, pi = 3.14159265358979323846;
        c->gamma0 = 1.0 + beam->kinetic_eV / beam->mass_eV;
        c->beta0 = std::sqrt(1.0 - 1.0 / (c->gamma0 * c->gamma0));
        c->E0 = c->gamma0 * beam->mass_eV;
        c->r_c = (double)beam->charge * (double)beam->charge * (e_charge / (4.0 * pi * eps0)) / beam->mass_eV;
        c->kappa = 4.0 * pi * c->r_c / (c->beta0 * c->beta0 * c->gamma0 * c->gamma0 * c->gamma0);
    }
    // table: convert QUAD, sum lengths
    double length = 0.0;
    c->rows.assign(lat, lat + n_elem);
    for (auto& e : c->rows) {
        if (e.kind == SC_QUAD) { length += e.p[1]; sc_elem t; quad_to_linmap(e, t); e = t; }
        else if (e.kind == SC_SEXT) length += e.p[1];
        else if (e.kind == SC_XDRIFT) length += e.p[0];
        else if (e.kind == SC_SBEND) { length += e.p[0]; if (e.p[1] == 0.0) e.kind = SC_XDRIFT; }
        else if (e.kind == SC_CQUAD) { length += e.p[1]; if (e.p[0] == 0.0) { const double L = e.p[1]; e = sc_elem{}; e.kind = SC_DRIFT; e.p[0] = L; } }
        else if (e.kind == SC_DRIFT) length += e.p[0];
        else if (e.kind == SC_LINMAP) length += e.p[8];
    }
    c->circumference = beam->circumference > 0 ? beam->circumference : length;
    for (auto& e : c->rows)
        if (e.kind == SC_RF) {
            if (!(c->circumference > 0)) return bail(SC_EINVAL, "RF row needs a circumference");
            const double pi = 3.14159265358979323846;
            e.p[0] = (double)beam->charge * e.p[0] / (c->beta0 * c->beta0 * c->E0);
            e.p[1] = 2.0 * pi * e.p[1] / c->circumference;
        }

    // workspace
    Layout L = make_layout(n_elem, grids, n_grids, max_particles);
    if (workspace) {
        if (workspace_bytes < (int64_t)L.total) return bail(SC_ENOMEM, "workspace smaller than sc_workspace_bytes()");
        if (((uintptr_t)workspace & 255) != 0) return bail(SC_EINVAL, "workspace must be 256-byte aligned");
        c->ws = (char*)workspace;
    } else {
        cudaError_t e = cudaMalloc((void**)&c->ws, L.total);
        if (e != cudaSuccess) return bail(SC_ENOMEM, std::string("cudaMalloc workspace: ") + cudaGetErrorString(e));
        c->own_ws = true;
    }
    c->ws_bytes = (int64_t)L.total;
    for (int k = 0; k < 6; k++) c->q[k] = (double*)(c->ws + L.off_q[k]);
    c->d_counters = (unsigned long long*)(c->ws + L.off_counters);
    c->d_mom_partial = (double*)(c->ws + L.off_mom_partial);
    c->d_mom_sums = (double*)(c->ws + L.off_mom_sums);
    c->d_mom_cov = (double*)(c->ws + L.off_mom_cov);

    auto up = [&](void* dst, const void* src, size_t bytes) {
        return cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, c->stream);
    };
    cudaError_t e = cudaMemsetAsync(c->ws + L.off_counters, 0, L.total - L.off_counters, c->stream);
    if (e != cudaSuccess) return bail(SC_ECUDA, std::string("clear workspace: ") + cudaGetErrorString(e));

    int max_bins = 0;
    for (int i = 0; i < n_grids; i++) if (grids[i].nbins > max_bins) max_bins = grids[i].nbins;
    std::vector<std::vector<double>> ghats(n_grids);
    std::vector<std::vector<double2>> twxs(n_grids), twys(n_grids);
    for (int i = 0; i < n_grids; i++) {
        const sc_grid& s = grids[i];
        GridDev g{};
        g.nx = s.nx; g.ny = s.ny; g.xmin = s.xmin; g.ymin = s.ymin;
        g.dx = (s.xmax - s.xmin) / (double)(s.nx - 1);
        g.dy = (s.ymax - s.ymin) / (double)(s.ny - 1);
        g.inv_dx = 1.0 / g.dx; g.inv_dy = 1.0 / g.dy;
        g.nxm1 = (double)(s.nx - 1); g.nym1 = (double)(s.ny - 1);
        g.nbins = s.nbins; g.smin = s.smin; g.dnbins = (double)s.nbins;
        if (s.nbins > 0) { g.ds = (s.smax - s.smin) / (double)s.nbins; g.inv_ds = 1.0 / g.ds; }
        g.mode = s.deposit_mode; g.bits = s.fixed_bits; g.boundary = s.boundary; g.long_kick = s.long_kick; g.interp = s.interp;
        g.fixed_scale = std::ldexp(1.0, s.fixed_bits);
        g.fixed_inv = std::ldexp(1.0, -2 * s.fixed_bits);
        choose_window(g, max_bins, 0);
        const Layout::G& o = L.g[i];
        g.rho = (unsigned long long*)(c->ws + o.rho); g.hist = (unsigned int*)(c->ws + o.hist);
        g.rho_last = (double*)(c->ws + o.rho_last); g.rhoi_last = (long long*)(c->ws + o.rhoi_last);
        g.hist_last = (long long*)(c->ws + o.hist_last); g.lam = (double2*)(c->ws + o.lam);
        g.A = (double2*)(c->ws + o.A); g.BU = (double2*)(c->ws + o.BU); g.BV = (double2*)(c->ws + o.BV);
        g.phi = (double*)(c->ws + o.phi); g.E = (double2*)(c->ws + o.E);
        g.Ghat = (const double*)(c->ws + o.Ghat); g.twx = (const double2*)(c->ws + o.twx); g.twy = (const double2*)(c->ws + o.twy);
        // identical geometry => reuse the transform already computed
        int same = -1;
        for (int k = 0; k < i; k++)
            if (grids[k].nx == s.nx && grids[k].ny == s.ny && grids[k].xmax - grids[k].xmin == s.xmax - s.xmin &&
                grids[k].ymax - grids[k].ymin == s.ymax - s.ymin && grids[k].boundary == s.boundary) { same = k; break; }
        if (same >= 0) ghats[i] = ghats[same];
        else if (s.boundary == SC_BOUNDARY_PIPE) compute_pipe_symbol(s, ghats[i]);
        else compute_ghat(s, ghats[i]);
        compute_twiddles(2 * s.nx, twxs[i]);
        compute_twiddles(2 * s.ny, twys[i]);
        e = up((void*)g.Ghat, ghats[i].data(), ghats[i].size() * 8);
        if (e == cudaSuccess) e = up((void*)g.twx, twxs[i].data(), twxs[i].size() * 16);
        if (e == cudaSuccess) e = up((void*)g.twy, twys[i].data(), twys[i].size() * 16);
        if (e != cudaSuccess) return bail(SC_ECUDA, std::string("upload grid tables: ") + cudaGetErrorString(e));
        c->gdev.push_back(g);
    }
    e = cudaStreamSynchronize(c->stream);   // host staging vectors die at return
    if (e != cudaSuccess) return bail(SC_ECUDA, std::string("sc_create sync: ") + cudaGetErrorString(e));
    *out = c;
    return SC_OK;
}

int sc_load_particles(sc_ctx* c, const double* x, const double* px, const double* y, const double* py,
                      const double* sigma, const double* psigma, int64_t n, int32_t on_device) {
    if (!c) return SC_EINVAL;
    if (!x || !px || !y || !py) return fail(c, SC_EINVAL, "x, px, y, py must not be NULL");
    if ((sigma == nullptr) != (psigma == nullptr)) return fail(c, SC_EINVAL, "sigma and psigma must both be given or both be NULL");
    if (n <= 0 || n > c->nmax) return fail(c, SC_EINVAL, "n must be in 1..max_particles");
    const bool sixd = sigma != nullptr;
    if (!sixd) {
        for (const auto& e : c->rows) if (e.kind == SC_RF) return fail(c, SC_EINVAL, "RF rows need a 6D beam (sigma, psigma)");
        for (const auto& g : c->grids) if (g.nbins > 0) return fail(c, SC_EINVAL, "lambda histogram (nbins > 0) needs a 6D beam");
    }
    const double* src[6] = { x, px, y, py, sigma, psigma };
    const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    for (int k = 0; k < (sixd ? 6 : 4); k++)
        SC_CUDA(c, cudaMemcpyAsync(c->q[k], src[k], (size_t)n * 8, kind, c->stream));
    // accumulators must start clean (a previous sc_step may have stopped anywhere)
    for (const auto& g : c->gdev) {
        SC_CUDA(c, cudaMemsetAsync(g.rho, 0, (size_t)g.nx * g.ny * 8, c->stream));
        SC_CUDA(c, cudaMemsetAsync(g.hist, 0, (size_t)(g.nbins > 0 ? g.nbins : 1) * 4, c->stream));
    }
    SC_CUDA(c, cudaMemsetAsync(c->d_counters, 0, 64, c->stream));
    SC_CUDA(c, cudaStreamSynchronize(c->stream));   // inputs are copied: the caller may free or overwrite its arrays (host or device) on return
    if (n != c->n || sixd != c->sixd) drop_graphs(c);
    c->n = n; c->sixd = sixd; c->loaded = true;
    c->pos = 0; c->pending = PendingKick{};
    return SC_OK;
}

int sc_track(sc_ctx* c, int64_t n_turns) {
    if (!c) return SC_EINVAL;
    if (!c->loaded) return fail(c, SC_ESTATE, "sc_track before sc_load_particles");
    if (n_turns < 0) return fail(c, SC_EINVAL, "n_turns must be >= 0");
    int rc = step_rows(c, n_turns * (int64_t)c->rows.size());
    if (rc) return rc;
    if (c->pos == 0) return flush_pending(c);     // whole turns done: the last node's kick belongs to them
    return SC_OK;
}

int sc_step(sc_ctx* c, int64_t n_rows) {
    if (!c) return SC_EINVAL;
    if (!c->loaded) return fail(c, SC_ESTATE, "sc_step before sc_load_particles");
    if (n_rows < 0) return fail(c, SC_EINVAL, "n_rows must be >= 0");
    return step_rows(c, n_rows);
}

int sc_get_particles(sc_ctx* c, double* x, double* px, double* y, double* py, double* sigma, double* psigma,
                     int32_t on_device) {
    if (!c) return SC_EINVAL;
    if (!c->loaded) return fail(c, SC_ESTATE, "no particles loaded");
    double* dst[6] = { x, px, y, py, sigma, psigma };
    const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    for (int k = 0; k < (c->sixd ? 6 : 4); k++)
        if (dst[k]) SC_CUDA(c, cudaMemcpyAsync(dst[k], c->q[k], (size_t)c->n * 8, kind, c->stream));
    SC_CUDA(c, cudaStreamSynchronize(c->stream));
    return SC_OK;
}

int sc_get_grid(sc_ctx* c, int32_t grid_id, int32_t which, void* out, int64_t bytes) {
    if (!c) return SC_EINVAL;
    if (grid_id < 0 || grid_id >= (int)c->gdev.size() || !out) return fail(c, SC_EINVAL, "bad grid id or NULL output");
    const GridDev& g = c->gdev[grid_id];
    const size_t nc = (size_t)g.nx * g.ny;
    const void* src = nullptr;
    size_t need = nc * 8;
    switch (which) {
    case SC_GRID_RHO_F64: src = g.rho_last; break;
    case SC_GRID_RHO_I64:
        if (g.mode != SC_DEPOSIT_FIXED) return fail(c, SC_EINVAL, "RHO_I64 exists only in fixed-point mode");
        src = g.rhoi_last; break;
    case SC_GRID_PHI: src = g.phi; break;
    case SC_GRID_EX: case SC_GRID_EY: src = g.E; need = nc * 8; break;
    case SC_GRID_LAMBDA: src = g.hist_last; need = (size_t)g.nbins * 8; break;
    default: return fail(c, SC_EINVAL, "unknown grid selector");
    }
    if (bytes < (int64_t)need) return fail(c, SC_EINVAL, "output buffer too small");
    if (need == 0) return SC_OK;
    if (which == SC_GRID_EX || which == SC_GRID_EY) {
        // de-interleave (Ex,Ey): strided 2D copy, 8 bytes wide
        SC_CUDA(c, cudaMemcpy2DAsync(out, 8, (const char*)src + (which == SC_GRID_EY ? 8 : 0), 16, 8, nc,
                                     cudaMemcpyDeviceToHost, c->stream));
    } else {
        SC_CUDA(c, cudaMemcpyAsync(out, src, need, cudaMemcpyDeviceToHost, c->stream));
    }
    SC_CUDA(c, cudaStreamSynchronize(c->stream));
    return SC_OK;
}

int sc_moments(sc_ctx* c, double* out, int32_t n_out) {
    if (!c) return SC_EINVAL;
    if (!c->loaded) return fail(c, SC_ESTATE, "no particles loaded");
    if (!out || n_out < SC_N_MOMENTS) return fail(c, SC_EINVAL, "out must hold SC_N_MOMENTS doubles");
    const int nco = c->sixd ? 6 : 4;
    int blocks = (int)((c->n + kMomThreads - 1) / kMomThreads);
    if (blocks > kMomBlocks) blocks = kMomBlocks;
    k_mom_sum<<<blocks, kMomThreads, 0, c->stream>>>(nco, c->n, c->d_mom_partial, c->q[0], c->q[1], c->q[2], c->q[3], c->q[4], c->q[5]);
    k_mom_combine<<<1, 32, 0, c->stream>>>(c->d_mom_partial, blocks, 7, c->d_mom_sums);
    k_mom_cov<<<blocks, kMomThreads, 0, c->stream>>>(nco, c->n, c->d_mom_sums, c->d_mom_partial, c->q[0], c->q[1], c->q[2], c->q[3], c->q[4], c->q[5]);
    k_mom_combine<<<1, 32, 0, c->stream>>>(c->d_mom_partial, blocks, 21, c->d_mom_cov);
    SC_CUDA(c, cudaGetLastError());
    c->launches += 4;
    double sums[8], cov[21];
    unsigned long long counters[8];
    SC_CUDA(c, cudaMemcpyAsync(sums, c->d_mom_sums, 7 * 8, cudaMemcpyDeviceToHost, c->stream));
    SC_CUDA(c, cudaMemcpyAsync(cov, c->d_mom_cov, 21 * 8, cudaMemcpyDeviceToHost, c->stream));
    SC_CUDA(c, cudaMemcpyAsync(counters, c->d_counters, 64, cudaMemcpyDeviceToHost, c->stream));
    SC_CUDA(c, cudaStreamSynchronize(c->stream));
    const double n = (double)c->n;
    out[0] = n;
    for (int k = 0; k < 6; k++) out[1 + k] = sums[k] / n;
    for (int k = 0; k < 21; k++) out[7 + k] = cov[k] / n;
    // upper-triangular index of (r,c): diag of plane pl at (2pl,2pl), (2pl,2pl+1), (2pl+1,2pl+1)
    auto idx = [](int r, int cc) { return 7 + r * 6 - r * (r - 1) / 2 + (cc - r); };
    for (int pl = 0; pl < 3; pl++) {
        const double a = out[idx(2 * pl, 2 * pl)], b = out[idx(2 * pl, 2 * pl + 1)], d = out[idx(2 * pl + 1, 2 * pl + 1)];
        const double det = a * d - b * b;
        out[28 + pl] = det > 0 ? std::sqrt(det) : 0.0;
    }
    out[31] = (double)counters[1];
    out[32] = sums[6];
#ifdef SC_CHECK
    if (counters[6] != 0ull) return fail(c, SC_ECUDA, "checked build: " + std::to_string(counters[6]) + " device-side index assertions failed (SC_ASSERT)");
#endif
    if (counters[5] != 0ull) return fail(c, SC_ECUDA, "a grid barrier of the fused Poisson kernel timed out (its CTAs were not co-resident): results are invalid");
    return SC_OK;
}

int sc_profile_turn(sc_ctx* c, double* out, int32_t n_out) {
    if (!c) return SC_EINVAL;
    if (!c->loaded) return fail(c, SC_ESTATE, "sc_profile_turn before sc_load_particles");
    if (!out || n_out < 5) return fail(c, SC_EINVAL, "out must hold 5 doubles");
    if (c->pos != 0) return fail(c, SC_ESTATE, "sc_profile_turn must start at a turn boundary");
    cudaEvent_t t0, t1;
    cudaError_t e = begin_event_pair(c, &t0, &t1);
    if (e != cudaSuccess) return fail(c, SC_ECUDA, std::string("sc_profile_turn: timing events: ") + cudaGetErrorString(e));
    c->profiling = true;
    int rc = run_rows(c, 0, (int64_t)c->rows.size());
    if (!rc) rc = flush_pending(c);
    e = cudaEventRecord(t1, c->stream);
    c->profiling = false;
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    double push_ms = 0, pois_ms = 0;
    float ms = 0;
    for (auto& p : c->ev_push) { if (cudaEventElapsedTime(&ms, p.first, p.second) == cudaSuccess) push_ms += ms; cudaEventDestroy(p.first); cudaEventDestroy(p.second); }
    for (auto& p : c->ev_poisson) { if (cudaEventElapsedTime(&ms, p.first, p.second) == cudaSuccess) pois_ms += ms; cudaEventDestroy(p.first); cudaEventDestroy(p.second); }
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, t0, t1);
    out[0] = push_ms; out[1] = (double)c->ev_push.size(); out[2] = pois_ms; out[3] = (double)c->ev_poisson.size(); out[4] = ms;
    c->ev_push.clear(); c->ev_poisson.clear();
    cudaEventDestroy(t0); cudaEventDestroy(t1);
    if (rc) return rc;
    if (e != cudaSuccess) return fail(c, SC_ECUDA, std::string("sc_profile_turn: ") + cudaGetErrorString(e));
    return SC_OK;
}

int sc_profile_replay(sc_ctx* c, int32_t mode, int32_t reps, void* scratch, int64_t scratch_bytes, double* out, int32_t n_out) {
    if (!c) return SC_EINVAL;
    if (!c->loaded) return fail(c, SC_ESTATE, "sc_profile_replay before sc_load_particles");
    if (!out || n_out < 6 || reps < 1) return fail(c, SC_EINVAL, "out must hold 6 doubles, reps >= 1");
    if (mode < SC_REPLAY_TURN || mode > SC_REPLAY_EMPTY) return fail(c, SC_EINVAL, "unknown replay mode");
    if (c->pos != 0) return fail(c, SC_ESTATE, "sc_profile_replay must start at a turn boundary");
    if (!c->use_graph) return fail(c, SC_ESTATE, "sc_profile_replay needs a capturable stream");
    const int nco = c->sixd ? 6 : 4;
    const size_t bytes = (size_t)c->n * 8;
    if (!scratch || scratch_bytes < (int64_t)(bytes * nco)) return fail(c, SC_ENOMEM, "scratch must hold the particle backup (8 bytes x coordinates x n)");
    char* save = (char*)scratch;
    SC_CUDA(c, cudaStreamSynchronize(c->stream));
    for (int k = 0; k < nco; k++) SC_CUDA(c, cudaMemcpyAsync(save + k * bytes, c->q[k], bytes, cudaMemcpyDeviceToDevice, c->stream));
    const PendingKick saved_pending = c->pending;
    const int64_t saved_launches = c->launches;
    const int64_t saved_ps_stores = c->ps_stores;
    // one turn of launches in the requested mode, as one graph
    c->skip_poisson = mode == SC_REPLAY_PUSH;
    c->skip_push = mode == SC_REPLAY_POISSON;
    c->noop = mode == SC_REPLAY_EMPTY;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    cudaError_t e = cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal);
    int rc = SC_OK;
    if (e == cudaSuccess) {
        rc = run_rows(c, 0, (int64_t)c->rows.size());
        if (!rc) rc = flush_pending(c);
        e = cudaStreamEndCapture(c->stream, &graph);
    }
    c->skip_poisson = c->skip_push = c->noop = false;
    const int64_t n_kernels = c->launches - saved_launches;
    c->launches = saved_launches;
    const int64_t n_ps_stores = c->ps_stores - saved_ps_stores;
    c->pending = saved_pending;
    int64_t n_nodes = 0;
    for (const auto& r : c->rows) n_nodes += r.kind == SC_SCNODE;
    if (!rc && e == cudaSuccess) e = cudaGraphInstantiate(&exec, graph, 0);
    float ms = 0;
    unsigned long long counters[2] = { 0ull, 0ull };
    if (!rc && e == cudaSuccess) {
        cudaEvent_t t0 = nullptr, t1 = nullptr;
        e = cudaGraphLaunch(exec, c->stream);                  // warm-up replay
        if (e == cudaSuccess) e = cudaMemsetAsync(c->d_counters, 0, 8, c->stream);
        if (e == cudaSuccess) e = begin_event_pair(c, &t0, &t1);
        for (int r = 0; r < reps && e == cudaSuccess; r++) e = cudaGraphLaunch(exec, c->stream);
        if (e == cudaSuccess) e = cudaEventRecord(t1, c->stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(counters, c->d_counters, 16, cudaMemcpyDeviceToHost, c->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, t0, t1);
        if (t0) cudaEventDestroy(t0);
        if (t1) cudaEventDestroy(t1);
        c->launches += n_kernels * (reps + 1);
    }
    if (exec) cudaGraphExecDestroy(exec);
    if (graph) cudaGraphDestroy(graph);
    // put everything back: particles, accumulators (a push-only replay never cleared them), counters
    cudaError_t e2 = cudaSuccess;
    for (int k = 0; k < nco && e2 == cudaSuccess; k++) e2 = cudaMemcpyAsync(c->q[k], save + k * bytes, bytes, cudaMemcpyDeviceToDevice, c->stream);
    for (const auto& g : c->gdev) {
        if (e2 == cudaSuccess) e2 = cudaMemsetAsync(g.rho, 0, (size_t)g.nx * g.ny * 8, c->stream);
        if (e2 == cudaSuccess) e2 = cudaMemsetAsync(g.hist, 0, (size_t)(g.nbins > 0 ? g.nbins : 1) * 4, c->stream);
    }
    if (e2 == cudaSuccess) e2 = cudaMemsetAsync(c->d_counters, 0, 8, c->stream);
    if (e2 == cudaSuccess) e2 = cudaStreamSynchronize(c->stream);
    if (rc) return rc;
    if (e != cudaSuccess) return fail(c, SC_ECUDA, std::string("sc_profile_replay: ") + cudaGetErrorString(e));
    if (e2 != cudaSuccess) return fail(c, SC_ECUDA, std::string("sc_profile_replay (restore): ") + cudaGetErrorString(e2));
    out[0] = (double)ms / reps;
    out[1] = (double)n_kernels;
    out[2] = (double)n_nodes;
    // particles outside the grid per deposit: a push-only replay accumulates over all its deposits, a full turn keeps the last node's
    out[3] = mode == SC_REPLAY_PUSH ? (double)counters[0] / ((double)n_nodes * reps) : (mode == SC_REPLAY_TURN ? (double)counters[1] : 0.0);
    out[4] = (double)reps;
    out[5] = (double)c->n;
    if (n_out >= 7) out[6] = (double)n_ps_stores;
    return SC_OK;
}

int sc_profile_copy(sc_ctx* c, int32_t reps, void* scratch, int64_t scratch_bytes, double* out, int32_t n_out) {
    if (!c) return SC_EINVAL;
    if (!c->loaded) return fail(c, SC_ESTATE, "sc_profile_copy before sc_load_particles");
    if (!out || n_out < 2 || reps < 1) return fail(c, SC_EINVAL, "out must hold 2 doubles, reps >= 1");
    const int nco = c->sixd ? 6 : 4;
    const size_t bytes = (size_t)c->n * 8;
    if (!scratch || scratch_bytes < (int64_t)(bytes * nco) || ((uintptr_t)scratch & 15)) return fail(c, SC_ENOMEM, "scratch must hold 8 bytes x coordinates x n, 16-byte aligned");
    CopyArgs a{};
    for (int k = 0; k < nco; k++) { a.src[k] = c->q[k]; a.dst[k] = (double*)((char*)scratch + k * (((size_t)c->n + 1) / 2 * 16)); }
    if (scratch_bytes < (int64_t)((((size_t)c->n + 1) / 2 * 16) * nco)) return fail(c, SC_ENOMEM, "scratch too small for 16-byte padded arrays");
    a.nco = nco; a.n2 = (c->n + 1) / 2;
    cudaEvent_t t0 = nullptr, t1 = nullptr;
    cudaError_t e = cudaEventCreate(&t0);
    if (e == cudaSuccess) e = cudaEventCreate(&t1);
    if (e == cudaSuccess) {
        k_copy_soa<<<4 * c->num_sms, 512, 0, c->stream>>>(a);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaEventRecord(t0, c->stream);
    for (int r = 0; r < reps && e == cudaSuccess; r++) {
        k_copy_soa<<<4 * c->num_sms, 512, 0, c->stream>>>(a);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaEventRecord(t1, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    float ms = 0;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, t0, t1);
    if (t0) cudaEventDestroy(t0);
    if (t1) cudaEventDestroy(t1);
    if (e != cudaSuccess) return fail(c, SC_ECUDA, std::string("sc_profile_copy: ") + cudaGetErrorString(e));
    if (!(ms > 0.0f)) return fail(c, SC_ECUDA, "sc_profile_copy: the copies took no measurable time (did the kernel run?)");
    c->launches += reps + 1;
    out[0] = (double)ms / reps;
    out[1] = 16.0 * nco * (double)c->n;
    return SC_OK;
}

int sc_get_constants(const sc_ctx* c, double* out, int32_t n_out) {
    if (!c || !out || n_out < 6) return SC_EINVAL;
    out[0] = c->gamma0; out[1] = c->beta0; out[2] = c->E0; out[3] = c->r_c; out[4] = c->kappa; out[5] = c->circumference;
    return SC_OK;
}

int64_t sc_kernel_launches(const sc_ctx* c) { return c ? c->launches : 0; }

#ifdef SC_TRACE
// working builds only (-DSC_TRACE): the kernels' globaltimer stamps, slots 8.. of the counter block
int sc_debug_trace(sc_ctx* c, unsigned long long* out, int32_t n) {
    if (!c || !out || n > kTraceSlots) return SC_EINVAL;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return SC_ECUDA;
    return cudaMemcpy(out, c->d_counters + 8, (size_t)n * 8, cudaMemcpyDeviceToHost) == cudaSuccess ? SC_OK : SC_ECUDA;
}
#endif

int sc_abi_sizes(int32_t* out, int32_t n_out) {
    if (!out || n_out < 3) return SC_EINVAL;
    out[0] = (int32_t)sizeof(sc_elem); out[1] = (int32_t)sizeof(sc_grid); out[2] = (int32_t)sizeof(sc_beam);
    return SC_OK;
}

const char* sc_last_error(const sc_ctx* c) { return c ? c->err.c_str() : g_create_error.c_str(); }

void sc_destroy(sc_ctx* c) {
    if (!c) return;
    drop_graphs(c);
    if (c->own_ws && c->ws) cudaFree(c->ws);
    delete c;
}

}  // extern "C"
