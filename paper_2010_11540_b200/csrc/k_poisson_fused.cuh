// k_poisson_fused.cuh -- the whole space-charge field solve of one node in ONE launch (grids of 64 or 128 nodes per axis).
//
// Same mathematics as k_poisson.cuh (open boundary: Hockney convolution with the precomputed real transform of the
// cell-integrated Green's function on the doubled grid; pipe: the paper's odd extension and eq. 25, PAPER.md:204-289;
// node field by differences, eq. 29), same three stages
//     A  rows forward   (two real rows per complex transform, Hermitian half kept)
//     B  columns        (forward, x multiplier, inverse, crop, y-derivative)
//     C  rows inverse   (U + iV packed: potential and E~y from one transform; E~x by differences)
// but one kernel with two grid-wide barriers instead of three launches, and the transforms in REGISTERS:
//   * a transform of length L = 16 P (P = 8, 16) is done by a group of 16 lanes (half a warp): lane t holds the P
//     elements 16 n1 + t, does a P-point FFT in registers, multiplies by W_L^(t k1), exchanges through a padded
//     shared-memory tile, then lane k1 does a 16-point FFT in registers.  One exchange and two __syncwarp() per
//     transform instead of the 4 block-wide passes of the shared-memory Stockham version (1.15 us per 256-point
//     transform there, a pure barrier/latency chain);
//   * the ~4 MFLOP of a 128^2 solve are spread over ~33-65 small CTAs (one or two warps each) so that every
//     transform of a stage runs at the same time; the stages hand over through L2 ([kx][j] and [j][kx] arrays);
//   * grid barrier: one RED.release + ld.acquire spin per CTA on a counter in the workspace (self-resetting; a spin
//     limit turns a would-be hang into an error flag that sc_moments/sc_track report).  All CTAs are co-resident by
//     construction: the grid is at most one small CTA per SM and, under programmatic dependent launch, starts only
//     when every CTA of the preceding k_push has exited.
#pragma once
#include "sc_device.cuh"

namespace sc {

constexpr int kFusedGroups = SC_FUSED_GROUPS;       // 16-lane transform groups per CTA
constexpr int kFusedThreads = 16 * kFusedGroups;

__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 cmulf(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

// radix-4 butterfly, outputs in natural order: X_k = sum_n a_n w^(nk), w = -i (forward) / +i (inverse)
template <bool INV>
__device__ __forceinline__ void bfly4(double2& a0, double2& a1, double2& a2, double2& a3) {
    const double2 s02 = cadd(a0, a2), d02 = csub(a0, a2), s13 = cadd(a1, a3), d13 = csub(a1, a3);
    const double2 r = INV ? make_double2(-d13.y, d13.x) : make_double2(d13.y, -d13.x);
    a0 = cadd(s02, s13); a1 = cadd(d02, r); a2 = csub(s02, s13); a3 = csub(d02, r);
}

// multiply by exp(-+ 2 pi i m / 16) (upper sign forward), m a compile-time constant
template <bool INV, int M>
__device__ __forceinline__ double2 rot16(double2 a) {
    constexpr double C1 = 0.92387953251128673848, S1 = 0.38268343236508978178, R = 0.70710678118654752440;
    constexpr int m = M & 15;
    // forward twiddle (c, -s); inverse (c, +s)
    constexpr double c = m == 0 ? 1.0 : m == 1 ? C1 : m == 2 ? R : m == 3 ? S1 : m == 4 ? 0.0 : m == 5 ? -S1 : m == 6 ? -R : m == 7 ? -C1 :
                         m == 8 ? -1.0 : m == 9 ? -C1 : m == 10 ? -R : m == 11 ? -S1 : m == 12 ? 0.0 : m == 13 ? S1 : m == 14 ? R : C1;
    constexpr double s = m == 0 ? 0.0 : m == 1 ? S1 : m == 2 ? R : m == 3 ? C1 : m == 4 ? 1.0 : m == 5 ? C1 : m == 6 ? R : m == 7 ? S1 :
                         m == 8 ? 0.0 : m == 9 ? -S1 : m == 10 ? -R : m == 11 ? -C1 : m == 12 ? -1.0 : m == 13 ? -C1 : m == 14 ? -R : -S1;
    constexpr double wi = INV ? s : -s;
    if (m == 0) return a;
    if (m == 4) return INV ? make_double2(-a.y, a.x) : make_double2(a.y, -a.x);
    if (m == 8) return make_double2(-a.x, -a.y);
    if (m == 12) return INV ? make_double2(a.y, -a.x) : make_double2(-a.y, a.x);
    return make_double2(a.x * c - a.y * wi, a.x * wi + a.y * c);
}

// P-point FFT in registers, natural order in and out (P = 8, 16)
template <bool INV>
__device__ __forceinline__ void fft16_impl(double2 (&v)[16]) {
    // n = 4 n1 + n2, k = k1 + 4 k2:  4-point transforms over n1, twiddle W16^(n2 k1), 4-point transforms over n2
#pragma unroll
    for (int n2 = 0; n2 < 4; n2++) bfly4<INV>(v[n2], v[n2 + 4], v[n2 + 8], v[n2 + 12]);     // slot n2 + 4 k1
    v[1 + 4] = rot16<INV, 1>(v[1 + 4]); v[2 + 4] = rot16<INV, 2>(v[2 + 4]); v[3 + 4] = rot16<INV, 3>(v[3 + 4]);
    v[1 + 8] = rot16<INV, 2>(v[1 + 8]); v[2 + 8] = rot16<INV, 4>(v[2 + 8]); v[3 + 8] = rot16<INV, 6>(v[3 + 8]);
    v[1 + 12] = rot16<INV, 3>(v[1 + 12]); v[2 + 12] = rot16<INV, 6>(v[2 + 12]); v[3 + 12] = rot16<INV, 9>(v[3 + 12]);
#pragma unroll
    for (int k1 = 0; k1 < 4; k1++) bfly4<INV>(v[4 * k1], v[4 * k1 + 1], v[4 * k1 + 2], v[4 * k1 + 3]);   // slot 4 k1 + k2 = X[k1 + 4 k2]
    double2 o[16];
#pragma unroll
    for (int k1 = 0; k1 < 4; k1++)
#pragma unroll
        for (int k2 = 0; k2 < 4; k2++) o[k1 + 4 * k2] = v[4 * k1 + k2];
#pragma unroll
    for (int k = 0; k < 16; k++) v[k] = o[k];
}

template <bool INV>
__device__ __forceinline__ void fft8_impl(double2 (&v)[8]) {
    // n = 2 n1 + n2, k = k1 + 4 k2: 4-point transforms over n1 (slot n2 + 2 k1), twiddle W8^(n2 k1), 2-point over n2
    bfly4<INV>(v[0], v[2], v[4], v[6]);
    bfly4<INV>(v[1], v[3], v[5], v[7]);
    v[3] = rot16<INV, 2>(v[3]); v[5] = rot16<INV, 4>(v[5]); v[7] = rot16<INV, 6>(v[7]);
    double2 o[8];
#pragma unroll
    for (int k1 = 0; k1 < 4; k1++) { o[k1] = cadd(v[2 * k1], v[2 * k1 + 1]); o[k1 + 4] = csub(v[2 * k1], v[2 * k1 + 1]); }
#pragma unroll
    for (int k = 0; k < 8; k++) v[k] = o[k];
}
template <int P, bool INV>
__device__ __forceinline__ void fft_regs(double2 (&v)[P]) {
    static_assert(P == 8 || P == 16, "register transforms of 8 or 16 points");
    if constexpr (P == 16) fft16_impl<INV>(v); else fft8_impl<INV>(v);
}

// One transform of length L by a 16-lane group.  In: lane t holds v[n1] = x[16 n1 + t].  Out: natural order in the
// group's shared array out[0..L).  ex: the group's exchange tile (P rows of 17).  tw: exp(-2 pi i m/L), m < L.
// Both 16-lane groups of a warp must call it together (two __syncwarp()).
template <int L, bool INV>
__device__ __forceinline__ void fft_group(double2 (&v)[L / 16], double2* ex, double2* out, const double2* tw, int t) {
    constexpr int P = L / 16;
    fft_regs<P, INV>(v);
#pragma unroll
    for (int k1 = 1; k1 < P; k1++) {
        double2 w = tw[t * k1];                     // t k1 <= 15 (P - 1) < L
        if (INV) w.y = -w.y;
        v[k1] = cmulf(v[k1], w);
    }
#pragma unroll
    for (int k1 = 0; k1 < P; k1++) ex[k1 * 17 + t] = v[k1];
    __syncwarp();
    if (t < P) {
        double2 z[16];
#pragma unroll
        for (int n2 = 0; n2 < 16; n2++) z[n2] = ex[t * 17 + n2];
        fft_regs<16, INV>(z);
#pragma unroll
        for (int k2 = 0; k2 < 16; k2++) out[t + P * k2] = z[k2];
    }
    __syncwarp();
}

// grid-wide barrier (see the file header).  cnt counts arrivals since the launch began.
__device__ __forceinline__ void grid_barrier(unsigned int* cnt, unsigned int target, unsigned int* err) {
    __syncthreads();
    if (threadIdx.x == 0) {
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(cnt) : "memory");
        unsigned int v;
        int spins = 0;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(cnt) : "memory");
        } while (v < target && ++spins < (1 << 22));
        if (v < target) atomicOr(err, 1u);
    }
    __syncthreads();
}

#ifdef SC_TRACE
#define SC_STAMP(k_) do { if (threadIdx.x == 0) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); counters[8 + blockIdx.x * 8 + (k_)] = t_; } } while (0)
#else
#define SC_STAMP(k_) do { } while (0)
#endif

__device__ __forceinline__ double2 ldcg2(const double2* p) {
    double2 v;
    asm volatile("ld.global.cg.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p) : "memory");
    return v;
}

// grid = ceil((nx+1) / kFusedGroups) CTAs of kFusedThreads.  counters: [0] n_outside accumulating, [1] of the last node,
// [4] (u32) barrier arrivals, [5] (u32) error flag.  UV: stage B -> C hand-over, [j][kx][2] complex (U, V), kx = 0..nx.
template <int NX, int NY>
__global__ void __launch_bounds__(kFusedThreads) k_poisson_fused(const PoissonArgs p, unsigned long long* counters) {
    constexpr int LX = 2 * NX, LY = 2 * NY, PX = LX / 16, PY = LY / 16;
    constexpr int LMAX = LX > LY ? LX : LY, PMAX = LMAX / 16;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (p.noop) { pdl_launch_dependents(); pdl_wait(); return; }
    const GridDev& g = p.g;
    double2* const s_twx = reinterpret_cast<double2*>(smem_raw);             // LX
    double2* const s_twy = s_twx + LX;                                        // LY
    double2* const s_ex_all = s_twy + LY;                                     // groups x PMAX x 17
    double2* const s_out_all = s_ex_all + kFusedGroups * PMAX * 17;           // groups x LMAX
    double* const s_gh_all = reinterpret_cast<double*>(s_out_all + kFusedGroups * LMAX);   // groups x LY
    const int tid = threadIdx.x, t = tid & 15, grp = tid >> 4;
    double2* const ex = s_ex_all + grp * PMAX * 17;
    double2* const out = s_out_all + grp * LMAX;
    double* const gh = s_gh_all + grp * LY;
    unsigned int* const bar = reinterpret_cast<unsigned int*>(counters + 4);
    unsigned int* const err = reinterpret_cast<unsigned int*>(counters + 5);
    const bool pipe = g.boundary == SC_BOUNDARY_PIPE;
    const unsigned int G = gridDim.x;

    SC_STAMP(0);
    pdl_launch_dependents();
    // constant tables: before the wait.  Full-circle twiddles from the half-circle tables (tw[m + L/2] = -tw[m]).
    //  (constant trip counts, unrolled: the loads of a thread go out together, not one latency after the other)
    {
        constexpr int TX = (NX + kFusedThreads - 1) / kFusedThreads, TY = (NY + kFusedThreads - 1) / kFusedThreads;
        double2 wx[TX], wy[TY];
#pragma unroll
        for (int m = 0; m < TX; m++) { const int k = tid + m * kFusedThreads; wx[m] = k < NX ? __ldg(g.twx + k) : make_double2(0.0, 0.0); }
#pragma unroll
        for (int m = 0; m < TY; m++) { const int k = tid + m * kFusedThreads; wy[m] = k < NY ? __ldg(g.twy + k) : make_double2(0.0, 0.0); }
        // multiplier row of this group's first column (stage B)
        const int kx = blockIdx.x * kFusedGroups + grp;
        double gv[LY / 16];
        const double* src = g.Ghat + (size_t)(kx <= NX ? kx : 0) * LY;
#pragma unroll
        for (int m = 0; m < LY / 16; m++) gv[m] = __ldg(src + t + 16 * m);
#pragma unroll
        for (int m = 0; m < TX; m++) { const int k = tid + m * kFusedThreads; if (k < NX) { s_twx[k] = wx[m]; s_twx[k + NX] = make_double2(-wx[m].x, -wx[m].y); } }
#pragma unroll
        for (int m = 0; m < TY; m++) { const int k = tid + m * kFusedThreads; if (k < NY) { s_twy[k] = wy[m]; s_twy[k + NY] = make_double2(-wy[m].x, -wy[m].y); } }
#pragma unroll
        for (int m = 0; m < LY / 16; m++) gh[t + 16 * m] = gv[m] * p.scale;
    }
    SC_STAMP(1);
    pdl_wait();
    SC_STAMP(2);
    // sigma histogram -> lambda pair table: every CTA takes a slice of the bins, its loads go out before the grid's
    const int bins_per_cta = (g.nbins + (int)G - 1) / (int)G;
    const int bin_mine = blockIdx.x * bins_per_cta + tid;
    unsigned int hc_mine = 0u;
    const bool bin_ok = tid < bins_per_cta && bin_mine < g.nbins;
    if (bin_ok) hc_mine = g.hist[bin_mine];
    __syncthreads();

    // ---------------------------------------------------------------- stage A: rows forward
    {
        const bool lamjob = blockIdx.x == 0;
        unsigned long long n_out_now = 0ull;
        if (lamjob && tid == 0) n_out_now = counters[0];
        for (int w0 = blockIdx.x * kFusedGroups; w0 < NY / 2; w0 += G * kFusedGroups) {
            const int pr = w0 + grp;
            const bool valid = pr < NY / 2;
            const int j0 = 2 * pr, j1 = j0 + 1;
            double2 v[PX];
            unsigned long long raw0[PX / 2], raw1[PX / 2];
#pragma unroll
            for (int n1 = 0; n1 < PX / 2; n1++) {                        // n = 16 n1 + t < NX
                const int i = 16 * n1 + t;
                raw0[n1] = valid ? g.rho[(size_t)j0 * NX + i] : 0ull;
                raw1[n1] = valid ? g.rho[(size_t)j1 * NX + i] : 0ull;
            }
            unsigned long long m0[PX / 2], m1[PX / 2];
            if (pipe) {
#pragma unroll
                for (int n1 = 0; n1 < PX / 2; n1++) {                    // n = NX + 16 n1 + t: source LX - n = NX - 16 n1 - t
                    const int src = NX - 16 * n1 - t;
                    const bool ok = valid && src >= 1 && src < NX;
                    m0[n1] = ok ? g.rho[(size_t)j0 * NX + src] : 0ull;
                    m1[n1] = ok ? g.rho[(size_t)j1 * NX + src] : 0ull;
                }
                __syncwarp();                                            // mirrored loads before anybody zeroes
            }
#ifdef SC_TRACE_A
            if (raw0[0] == 0x123456789ull) counters[7] = 2;
            SC_STAMP(3);
#endif
            auto conv = [&](unsigned long long r) {
                return g.mode == SC_DEPOSIT_FIXED ? (double)(long long)r * g.fixed_inv : __longlong_as_double((long long)r);
            };
#pragma unroll
            for (int n1 = 0; n1 < PX / 2; n1++) {
                const int i = 16 * n1 + t;
                const double r0 = conv(raw0[n1]), r1 = conv(raw1[n1]);
                if (valid) {
                    const size_t c0 = (size_t)j0 * NX + i, c1 = (size_t)j1 * NX + i;
                    if (g.mode == SC_DEPOSIT_FIXED) { g.rhoi_last[c0] = (long long)raw0[n1]; g.rhoi_last[c1] = (long long)raw1[n1]; }
                    g.rho_last[c0] = r0; g.rho_last[c1] = r1;
                    g.rho[c0] = 0ull; g.rho[c1] = 0ull;
                }
                // eq. 18: the wall node 0 carries no charge in the odd extension
                v[n1] = (pipe && i == 0) ? make_double2(0.0, 0.0) : make_double2(r0, r1);
                v[n1 + PX / 2] = pipe ? make_double2(-conv(m0[n1]), -conv(m1[n1])) : make_double2(0.0, 0.0);
            }
#ifdef SC_TRACE_A
            if (v[0].x == 12345.678) counters[7] = 1; SC_STAMP(4);
#endif
            fft_group<LX, false>(v, ex, out, s_twx, t);
#ifdef SC_TRACE_A
            SC_STAMP(5);
#endif
            // unpack the two real rows: R0 = (Z[k] + conj Z[-k])/2, R1 = (Z[k] - conj Z[-k])/(2i); [kx][j] layout
            if (valid) {
                auto unpack = [&](int kx) {
                    const double2 zk = out[kx], zm = out[(LX - kx) & (LX - 1)];
                    double2* dst = g.A + (size_t)kx * NY + j0;
                    dst[0] = make_double2(0.5 * (zk.x + zm.x), 0.5 * (zk.y - zm.y));
                    dst[1] = make_double2(0.5 * (zk.y + zm.y), -0.5 * (zk.x - zm.x));
                };
#pragma unroll
                for (int m = 0; m < NX / 16; m++) unpack(t + 16 * m);
                if (t == 0) unpack(NX);
            }
            __syncwarp();
        }
        // line density of this node: lambda_b = n_real cnt_b / (N ds)
        if (bin_ok) {
            g.hist_last[bin_mine] = (long long)hc_mine;
            const double lb = p.lam_scale * (double)hc_mine;      // pair table: lambda_b is .y of entry b and .x of entry b+1
            g.lam[bin_mine].y = lb;
            g.lam[bin_mine + 1].x = lb;
            g.hist[bin_mine] = 0u;
        }
        for (int bin = blockIdx.x * bins_per_cta + kFusedThreads + tid; bin < (int)(blockIdx.x + 1) * bins_per_cta && bin < g.nbins; bin += kFusedThreads) {
            const unsigned int cnt = g.hist[bin];                 // more bins per CTA than threads (nbins > ~2000): the slow way
            g.hist_last[bin] = (long long)cnt;
            const double lb = p.lam_scale * (double)cnt;
            g.lam[bin].y = lb;
            g.lam[bin + 1].x = lb;
            g.hist[bin] = 0u;
        }
        if (lamjob && tid == 0) { counters[1] = n_out_now; counters[0] = 0ull; }
    }
#ifdef SC_TRACE_A
    SC_STAMP(6);
    grid_barrier(bar, G, err);
#else
    SC_STAMP(3);
    grid_barrier(bar, G, err);
    SC_STAMP(4);
#endif

    // ---------------------------------------------------------------- stage B: columns
    {
        const double hy = 0.5 * g.inv_dy;
        bool first = true;
        for (int w0 = blockIdx.x * kFusedGroups; w0 <= NX; w0 += G * kFusedGroups) {
            const int kx = w0 + grp;
            const bool valid = kx <= NX;
            if (!first) {
                const double* src = g.Ghat + (size_t)(valid ? kx : 0) * LY;
                double gv[LY / 16];
#pragma unroll
                for (int m = 0; m < LY / 16; m++) gv[m] = __ldg(src + t + 16 * m);
#pragma unroll
                for (int m = 0; m < LY / 16; m++) gh[t + 16 * m] = gv[m] * p.scale;
                __syncwarp();
            }
            first = false;
            double2 v[PY];
            const double2* col = g.A + (size_t)(valid ? kx : 0) * NY;
#pragma unroll
            for (int n1 = 0; n1 < PY / 2; n1++) {
                const int j = 16 * n1 + t;
                double2 a = ldcg2(col + j);
                if (pipe && j == 0) a = make_double2(0.0, 0.0);
                v[n1] = a;
                if (pipe) {
                    const int src = NY - 16 * n1 - t;               // j' = NY + 16 n1 + t mirrors to LY - j'
                    double2 m = make_double2(0.0, 0.0);
                    if (src >= 1 && src < NY) { m = ldcg2(col + src); m.x = -m.x; m.y = -m.y; }
                    v[n1 + PY / 2] = m;
                } else {
                    v[n1 + PY / 2] = make_double2(0.0, 0.0);
                }
            }
            fft_group<LY, false>(v, ex, out, s_twy, t);
#pragma unroll
            for (int n1 = 0; n1 < PY; n1++) {
                const int k = 16 * n1 + t;
                const double2 z = out[k];
                const double gs = gh[k];
                v[n1] = make_double2(z.x * gs, z.y * gs);
            }
            __syncwarp();                                           // out[] is rewritten by the inverse transform
            fft_group<LY, true>(v, ex, out, s_twy, t);
            if (valid) {
#pragma unroll
                for (int m = 0; m < NY / 16; m++) {
                    const int j = t + 16 * m;
                    const double2 uj = out[j];
                    const double2 up = out[j + 1], um = out[j > 0 ? j - 1 : 0];     // out[NY] exists (LY entries)
                    double2 d;
                    if (j == 0) d = make_double2(-(up.x - uj.x) * g.inv_dy, -(up.y - uj.y) * g.inv_dy);
                    else if (j == NY - 1) d = make_double2(-(uj.x - um.x) * g.inv_dy, -(uj.y - um.y) * g.inv_dy);
                    else d = make_double2(-(up.x - um.x) * hy, -(up.y - um.y) * hy);
                    double2* dst = g.BU + ((size_t)j * (NX + 1) + kx) * 2;
                    dst[0] = uj;
                    dst[1] = d;
                }
            }
            __syncwarp();
        }
    }
#ifndef SC_TRACE_A
    SC_STAMP(5);
#endif
    grid_barrier(bar, 2 * G, err);
#ifndef SC_TRACE_A
    SC_STAMP(6);
#endif

    // ---------------------------------------------------------------- stage C: rows inverse
    {
        for (int w0 = blockIdx.x * kFusedGroups; w0 < NY; w0 += G * kFusedGroups) {
            const int j = w0 + grp;
            const bool valid = j < NY;
            const double2* row = g.BU + (size_t)(valid ? j : 0) * (NX + 1) * 2;
            double2 v[PX];
#pragma unroll
            for (int n1 = 0; n1 < PX; n1++) {
                const int k = 16 * n1 + t;
                const int ks = k <= NX ? k : LX - k;
                double2 U = ldcg2(row + 2 * ks), V = ldcg2(row + 2 * ks + 1);
                if (k > NX) { U.y = -U.y; V.y = -V.y; }
                v[n1] = make_double2(U.x - V.y, U.y + V.x);          // U + i V
            }
            fft_group<LX, true>(v, ex, out, s_twx, t);
            if (valid) {
#pragma unroll
                for (int m = 0; m < NX / 16; m++) {
                    const int i = t + 16 * m;
                    const double2 zi = out[i];
                    const double up = out[i + 1].x, um = out[i > 0 ? i - 1 : 0].x;   // out[NX] exists (LX entries)
                    double exv;
                    if (i == 0) exv = -(up - zi.x) * g.inv_dx;
                    else if (i == NX - 1) exv = -(zi.x - um) * g.inv_dx;
                    else exv = -(up - um) * (0.5 * g.inv_dx);
                    g.phi[(size_t)j * NX + i] = zi.x;
                    g.E[(size_t)j * NX + i] = make_double2(exv, zi.y);
                }
            }
            __syncwarp();
        }
    }
    // last CTA out re-arms the barrier counter for the next launch
    __syncthreads();
    SC_STAMP(7);
    if (tid == 0) {
        const unsigned int old = atomicAdd(bar, 1u);
        if (old == 3u * G - 1u) *bar = 0u;
    }
}

template <int NX, int NY>
constexpr size_t fused_smem_bytes() {
    constexpr int LX = 2 * NX, LY = 2 * NY, LMAX = LX > LY ? LX : LY, PMAX = LMAX / 16;
    return (size_t)(LX + LY) * 16 + (size_t)kFusedGroups * PMAX * 17 * 16 + (size_t)kFusedGroups * LMAX * 16 + (size_t)kFusedGroups * LY * 8;
}

}  // namespace sc
