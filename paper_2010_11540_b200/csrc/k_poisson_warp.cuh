// k_poisson_warp.cuh -- the field solve for grids of 64 or 128 nodes per axis: the three launches of k_poisson.cuh
// (rows forward / columns / rows inverse; same mathematics, same hand-over arrays' meaning, same boundary options) with
// ONE WARP PER TRANSFORM instead of one 128-thread CTA per transform and four block-wide Stockham passes.
//
// A transform of length L = 32 P (P = 4, 8) lives in a warp's registers, P complex numbers per lane, element 32 n1 + t in
// lane t.  Index split  n = 32 n1 + 4 n2 + n3,  k = k1 + P k2 + 8P k3:
//     S1  P-point FFT over n1 in registers, twiddle W_L^(k1 t)
//     --  exchange through the warp's shared-memory tile (__syncwarp only) --
//     S2  8-point FFT over n2 in registers (lane = (k1, n3)), twiddle W_32^(n3 k2)
//     --  exchange --
//     S3  4-point FFTs over n3 (lane = pairs (k1, k2)), natural-order result in the warp's shared array.
// ~200 fp64 instructions per lane and transform, two warp-level exchanges, no block barrier inside a transform.
// Measured on B200: per-thread SERIAL instruction count decides these latency-chain kernels --
// 16 lanes x 16 points (k_poisson_fused.cuh) was slower than the 128-thread Stockham passes, 32 lanes x 8 points is faster.
// Global traffic stays coalesced: rows are loaded a warp-row at a time, and the two transposing stores (row spectra ->
// [kx][j], column results -> [j][kx]) are done by the whole CTA from shared memory so that every 128-byte line is written
// by consecutive lanes.
#pragma once
#include "k_poisson_fused.cuh"   // bfly4, rot16, fft8_impl, complex helpers

namespace sc {

#ifndef SC_PW_WARPS
#define SC_PW_WARPS 2
#endif
constexpr int kPwWarps = SC_PW_WARPS;          // transforms (warps) per CTA
constexpr int kPwThreads = 32 * kPwWarps;

template <int P, bool INV>
__device__ __forceinline__ void fft_small(double2 (&v)[P]) {
    static_assert(P == 4 || P == 8, "4 or 8 points per lane");
    if constexpr (P == 8) fft8_impl<INV>(v);
    else bfly4<INV>(v[0], v[1], v[2], v[3]);
}

// per-warp shared tiles: bufA holds the first exchange [P][33], later the natural-order result [L]; bufB the second [4P][9]
template <int L>
struct WarpTiles {
    static constexpr int P = L / 32;
    static constexpr int kA = (P * 33 > L) ? P * 33 : L;
    static constexpr int kB = 4 * P * 9;
    static constexpr int kTotal = kA + kB;     // complex numbers per warp
};

// In: lane t holds v[n1] = x[32 n1 + t].  Out: X[k] in natural order in bufA[0..L).  tw[m] = exp(-2 pi i m/L), m < L.
// All 32 lanes of the warp call it together.
template <int L, bool INV>
__device__ __forceinline__ void fft_warp(double2 (&v)[L / 32], double2* bufA, double2* bufB, const double2* tw, int t) {
    constexpr int P = L / 32;
    fft_small<P, INV>(v);                                   // S1: over n1 -> k1
#pragma unroll
    for (int k1 = 1; k1 < P; k1++) {
        double2 w = tw[k1 * t];
        if (INV) w.y = -w.y;
        v[k1] = cmulf(v[k1], w);
    }
#pragma unroll
    for (int k1 = 0; k1 < P; k1++) bufA[k1 * 33 + t] = v[k1];
    __syncwarp();
    if (t < 4 * P) {                                        // S2: lane = (k1, n3), 8-point FFT over n2
        const int k1 = t >> 2, n3 = t & 3;
        double2 z[8];
#pragma unroll
        for (int n2 = 0; n2 < 8; n2++) z[n2] = bufA[k1 * 33 + 4 * n2 + n3];
        fft8_impl<INV>(z);
#pragma unroll
        for (int k2 = 1; k2 < 8; k2++) {
            double2 w = tw[P * n3 * k2];                    // W_32^(n3 k2)
            if (INV) w.y = -w.y;
            z[k2] = cmulf(z[k2], w);
        }
#pragma unroll
        for (int k2 = 0; k2 < 8; k2++) bufB[t * 9 + k2] = z[k2];      // [(k1, n3)][k2]
    }
    __syncwarp();                                           // orders the reads of bufA above before the writes below, too
#pragma unroll
    for (int c = 0; c < P / 4; c++) {                       // S3: 4-point FFTs over n3 for the pairs (k1, k2)
        const int comb = t + 32 * c, k1 = comb % P, k2 = comb / P;
        double2 y0 = bufB[(4 * k1 + 0) * 9 + k2], y1 = bufB[(4 * k1 + 1) * 9 + k2], y2 = bufB[(4 * k1 + 2) * 9 + k2], y3 = bufB[(4 * k1 + 3) * 9 + k2];
        bfly4<INV>(y0, y1, y2, y3);
        const int k = k1 + P * k2;
        bufA[k] = y0; bufA[k + 8 * P] = y1; bufA[k + 16 * P] = y2; bufA[k + 24 * P] = y3;
    }
    __syncwarp();
}

template <int L>
__device__ __forceinline__ void stage_twiddles(double2* s_tw, const double2* tw_half) {
    // full circle from the half-circle table (tw[m + L/2] = -tw[m]); constant trip count so that the loads go out together
    constexpr int T = (L / 2 + kPwThreads - 1) / kPwThreads;
    double2 w[T];
#pragma unroll
    for (int m = 0; m < T; m++) { const int k = threadIdx.x + m * kPwThreads; w[m] = k < L / 2 ? __ldg(tw_half + k) : make_double2(0.0, 0.0); }
#pragma unroll
    for (int m = 0; m < T; m++) { const int k = threadIdx.x + m * kPwThreads; if (k < L / 2) { s_tw[k] = w[m]; s_tw[k + L / 2] = make_double2(-w[m].x, -w[m].y); } }
}

template <int L>
constexpr size_t pw_smem_bytes() { return (size_t)(L + kPwWarps * WarpTiles<L>::kTotal) * 16; }

// ---------------------------------------------------------------- rows forward: grid = ceil(NY/2 / kPwWarps)
template <int NX, int NY>
__global__ void __launch_bounds__(kPwThreads) k_pw_rows_fwd(const PoissonArgs p, unsigned long long* counters) {
    constexpr int LX = 2 * NX, P = LX / 32;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (p.noop) { pdl_launch_dependents(); pdl_wait(); return; }
    const GridDev& g = p.g;
    double2* const s_tw = reinterpret_cast<double2*>(smem_raw);
    const int tid = threadIdx.x, t = tid & 31, warp = tid >> 5;
    double2* const bufA = s_tw + LX + warp * WarpTiles<LX>::kTotal;
    double2* const bufB = bufA + WarpTiles<LX>::kA;
    const bool pipe = g.boundary == SC_BOUNDARY_PIPE;
    pdl_launch_dependents();
    stage_twiddles<LX>(s_tw, g.twx);
    pdl_wait();
    // sigma histogram -> lambda pair table: every CTA takes a slice of the bins, loads first
    const int G = gridDim.x;
    const int bins_per_cta = (g.nbins + G - 1) / G;
    unsigned long long n_out_now = 0ull;
    if (blockIdx.x == 0 && tid == 0) n_out_now = counters[0];
    const int pr = blockIdx.x * kPwWarps + warp;              // packed pair of rows
    const bool valid = pr < NY / 2;
    const int j0 = 2 * pr, j1 = j0 + 1;
    unsigned long long raw0[P / 2], raw1[P / 2], m0[P / 2], m1[P / 2];
#pragma unroll
    for (int n1 = 0; n1 < P / 2; n1++) {                      // n = 32 n1 + t < NX
        const int i = 32 * n1 + t;
        raw0[n1] = valid ? g.rho[(size_t)j0 * NX + i] : 0ull;
        raw1[n1] = valid ? g.rho[(size_t)j1 * NX + i] : 0ull;
        m0[n1] = 0ull; m1[n1] = 0ull;
    }
    if (pipe) {
#pragma unroll
        for (int n1 = 0; n1 < P / 2; n1++) {                  // n = NX + 32 n1 + t mirrors to LX - n = NX - 32 n1 - t (eq. 18)
            const int src = NX - 32 * n1 - t;
            const bool ok = valid && src >= 1 && src < NX;
            m0[n1] = ok ? g.rho[(size_t)j0 * NX + src] : 0ull;
            m1[n1] = ok ? g.rho[(size_t)j1 * NX + src] : 0ull;
        }
    }
    unsigned int hc[4] = { 0u, 0u, 0u, 0u };
#pragma unroll
    for (int q = 0; q < 4; q++) {                             // up to 4 bins per thread go out with the grid loads
        const int bin = blockIdx.x * bins_per_cta + tid + q * kPwThreads;
        if (tid + q * kPwThreads < bins_per_cta && bin < g.nbins) hc[q] = g.hist[bin];
    }
    __syncthreads();                                          // twiddles staged; mirrored loads issued before anybody zeroes
    auto conv = [&](unsigned long long r) {
        return g.mode == SC_DEPOSIT_FIXED ? (double)(long long)r * g.fixed_inv : __longlong_as_double((long long)r);
    };
    double2 v[P];
#pragma unroll
    for (int n1 = 0; n1 < P / 2; n1++) {
        const int i = 32 * n1 + t;
        const double r0 = conv(raw0[n1]), r1 = conv(raw1[n1]);
        if (valid) {
            const size_t c0 = (size_t)j0 * NX + i, c1 = (size_t)j1 * NX + i;
            if (g.mode == SC_DEPOSIT_FIXED) { g.rhoi_last[c0] = (long long)raw0[n1]; g.rhoi_last[c1] = (long long)raw1[n1]; }
            g.rho_last[c0] = r0; g.rho_last[c1] = r1;
            g.rho[c0] = 0ull; g.rho[c1] = 0ull;
        }
        v[n1] = (pipe && i == 0) ? make_double2(0.0, 0.0) : make_double2(r0, r1);     // the wall node carries no charge
        v[n1 + P / 2] = pipe ? make_double2(-conv(m0[n1]), -conv(m1[n1])) : make_double2(0.0, 0.0);
    }
    fft_warp<LX, false>(v, bufA, bufB, s_tw, t);
    // line density of this node: lambda_b = n_real cnt_b / (N ds); pair table: lambda_b is .y of entry b and .x of entry b+1
#pragma unroll
    for (int q = 0; q < 4; q++) {
        const int bin = blockIdx.x * bins_per_cta + tid + q * kPwThreads;
        if (tid + q * kPwThreads < bins_per_cta && bin < g.nbins) {
            g.hist_last[bin] = (long long)hc[q];
            const double lb = p.lam_scale * (double)hc[q];
            g.lam[bin].y = lb; g.lam[bin + 1].x = lb;
            g.hist[bin] = 0u;
        }
    }
    for (int bin = blockIdx.x * bins_per_cta + 4 * kPwThreads + tid; bin < (int)(blockIdx.x + 1) * bins_per_cta && bin < g.nbins; bin += kPwThreads) {
        const unsigned int cnt = g.hist[bin];                 // more than 4 bins per thread: the slow way
        g.hist_last[bin] = (long long)cnt;
        const double lb = p.lam_scale * (double)cnt;
        g.lam[bin].y = lb; g.lam[bin + 1].x = lb;
        g.hist[bin] = 0u;
    }
    if (blockIdx.x == 0 && tid == 0) { counters[1] = n_out_now; counters[0] = 0ull; }
    __syncthreads();                                          // every warp's spectrum is in its bufA
    // unpack the two real rows of every warp, R0 = (Z[k] + conj Z[-k])/2, R1 = (Z[k] - conj Z[-k])/(2i), and store A[kx][j]
    // with consecutive threads on consecutive rows of one kx: 2 kPwWarps x 16 contiguous bytes per kx
    constexpr int R = 2 * kPwWarps;
    const int jb = 2 * blockIdx.x * kPwWarps;
    for (int e = tid; e < (NX + 1) * R; e += kPwThreads) {
        const int kx = e / R, r = e % R;
        if (jb + r >= NY) continue;
        const double2* z = s_tw + LX + (r >> 1) * WarpTiles<LX>::kTotal;
        const double2 zk = z[kx], zm = z[(LX - kx) & (LX - 1)];
        g.A[(size_t)kx * NY + jb + r] = (r & 1) ? make_double2(0.5 * (zk.y + zm.y), -0.5 * (zk.x - zm.x))
                                                : make_double2(0.5 * (zk.x + zm.x), 0.5 * (zk.y - zm.y));
    }
}

// ---------------------------------------------------------------- columns: grid = ceil((NX+1) / kPwWarps)
template <int NX, int NY>
__global__ void __launch_bounds__(kPwThreads) k_pw_cols(const PoissonArgs p) {
    constexpr int LY = 2 * NY, P = LY / 32;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (p.noop) { pdl_launch_dependents(); pdl_wait(); return; }
    const GridDev& g = p.g;
    double2* const s_tw = reinterpret_cast<double2*>(smem_raw);
    const int tid = threadIdx.x, t = tid & 31, warp = tid >> 5;
    double2* const bufA = s_tw + LY + warp * WarpTiles<LY>::kTotal;
    double2* const bufB = bufA + WarpTiles<LY>::kA;
    const bool pipe = g.boundary == SC_BOUNDARY_PIPE;
    pdl_launch_dependents();
    stage_twiddles<LY>(s_tw, g.twy);
    const int kx = blockIdx.x * kPwWarps + warp;
    const bool valid = kx <= NX;
    // this column's multipliers are constant: fetch them before the wait, in the layout of the inverse transform's input
    double gs[P];
    {
        const double* gh = g.Ghat + (size_t)(valid ? kx : 0) * LY;
#pragma unroll
        for (int n1 = 0; n1 < P; n1++) gs[n1] = __ldg(gh + 32 * n1 + t) * p.scale;
    }
    pdl_wait();
    double2 v[P];
    const double2* col = g.A + (size_t)(valid ? kx : 0) * NY;
#pragma unroll
    for (int n1 = 0; n1 < P / 2; n1++) {
        const int j = 32 * n1 + t;
        double2 a = col[j];
        if (pipe && j == 0) a = make_double2(0.0, 0.0);
        v[n1] = a;
        double2 m = make_double2(0.0, 0.0);
        if (pipe) {
            const int src = NY - 32 * n1 - t;                 // j' = NY + 32 n1 + t mirrors to LY - j' (odd extension, eq. 18)
            if (src >= 1 && src < NY) { m = col[src]; m.x = -m.x; m.y = -m.y; }
        }
        v[n1 + P / 2] = m;
    }
    __syncthreads();                                          // twiddles staged
    fft_warp<LY, false>(v, bufA, bufB, s_tw, t);
#pragma unroll
    for (int n1 = 0; n1 < P; n1++) {
        const double2 z = bufA[32 * n1 + t];
        v[n1] = make_double2(z.x * gs[n1], z.y * gs[n1]);
    }
    __syncwarp();                                             // bufA is rewritten by the inverse transform
    fft_warp<LY, true>(v, bufA, bufB, s_tw, t);
    __syncthreads();                                          // every warp's column of the potential is in its bufA
    // store (U, V = -dU/dy) as [j][kx][2]: consecutive threads on consecutive 16-byte pieces of one j
    const double hy = 0.5 * g.inv_dy;
    const int kb = blockIdx.x * kPwWarps;
    for (int e = tid; e < NY * kPwWarps * 2; e += kPwThreads) {
        const int h = e & 1, c = (e >> 1) % kPwWarps, j = e / (2 * kPwWarps);
        if (kb + c > NX) continue;
        const double2* u = s_tw + LY + c * WarpTiles<LY>::kTotal;
        double2 val;
        if (h == 0) val = u[j];
        else if (j == 0) val = make_double2(-(u[1].x - u[0].x) * g.inv_dy, -(u[1].y - u[0].y) * g.inv_dy);
        else if (j == NY - 1) val = make_double2(-(u[j].x - u[j - 1].x) * g.inv_dy, -(u[j].y - u[j - 1].y) * g.inv_dy);
        else val = make_double2(-(u[j + 1].x - u[j - 1].x) * hy, -(u[j + 1].y - u[j - 1].y) * hy);
        g.BU[((size_t)j * (NX + 1) + kb + c) * 2 + h] = val;
    }
}

// ---------------------------------------------------------------- rows inverse: grid = ceil(NY / kPwWarps)
template <int NX, int NY>
__global__ void __launch_bounds__(kPwThreads) k_pw_rows_inv(const PoissonArgs p) {
    constexpr int LX = 2 * NX, P = LX / 32;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (p.noop) { pdl_launch_dependents(); pdl_wait(); return; }
    const GridDev& g = p.g;
    double2* const s_tw = reinterpret_cast<double2*>(smem_raw);
    const int tid = threadIdx.x, t = tid & 31, warp = tid >> 5;
    double2* const bufA = s_tw + LX + warp * WarpTiles<LX>::kTotal;
    double2* const bufB = bufA + WarpTiles<LX>::kA;
    pdl_launch_dependents();
    stage_twiddles<LX>(s_tw, g.twx);
    pdl_wait();
    const int j = blockIdx.x * kPwWarps + warp;
    const bool valid = j < NY;
    const double2* row = g.BU + (size_t)(valid ? j : 0) * (NX + 1) * 2;
    double2 v[P];
#pragma unroll
    for (int n1 = 0; n1 < P; n1++) {
        const int k = 32 * n1 + t;
        const int ks = k <= NX ? k : LX - k;                  // Hermitian half stored: the rest is the conjugate of LX - k
        double2 U = row[2 * ks], V = row[2 * ks + 1];
        if (k > NX) { U.y = -U.y; V.y = -V.y; }
        v[n1] = make_double2(U.x - V.y, U.y + V.x);           // U + i V: one inverse transform gives u~ (real) and E~y (imaginary)
    }
    __syncthreads();                                          // twiddles staged
    fft_warp<LX, true>(v, bufA, bufB, s_tw, t);
    if (valid) {
#pragma unroll
        for (int m = 0; m < NX / 32; m++) {
            const int i = t + 32 * m;
            const double2 zi = bufA[i];
            const double up = bufA[i + 1].x, um = bufA[i > 0 ? i - 1 : 0].x;       // bufA[NX] exists (LX entries)
            double exv;
            if (i == 0) exv = -(up - zi.x) * g.inv_dx;
            else if (i == NX - 1) exv = -(zi.x - um) * g.inv_dx;
            else exv = -(up - um) * (0.5 * g.inv_dx);
            g.phi[(size_t)j * NX + i] = zi.x;
            g.E[(size_t)j * NX + i] = make_double2(exv, zi.y);
        }
    }
}

}  // namespace sc
