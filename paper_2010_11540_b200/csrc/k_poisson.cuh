// k_poisson.cuh -- open-boundary Poisson solve on the doubled (Hockney) grid with hand-written
// shared-memory FFTs, plus the node field E~ = -grad u~ (eq. 29), in three launches:
//
//   k_rows_fwd : charge grid rows (zero-padded nx -> 2nx), two REAL rows packed into one complex
//                FFT, unpacked to the Hermitian half kx = 0..nx, stored transposed A[kx][j].
//                Also: converts/zeroes the accumulators, keeps a copy of Q for sc_get_grid, turns
//                the sigma histogram into lambda_b.
//   k_cols     : per kx: column FFT (ny -> 2ny zero-padded), multiply by the precomputed REAL
//                transform of the Green's function, inverse column FFT, crop to ny;
//                writes the potential BU[kx][j] and its y-derivative BV[kx][j] (central/one-sided
//                differences commute with the x transform).
//   k_rows_inv : per row j: pack the two Hermitian spectra as U + iV, ONE inverse complex FFT gives
//                u~ (real part) and E~y (imaginary part); E~x by differences along the row.
//
// With grid.boundary = SC_BOUNDARY_PIPE the same three kernels run the paper's own solver (eqs. 15-27): the rows and
// columns are extended ODD about the wall nodes instead of zero-padded, and the real multiplier is 1/(dx dy) over the
// symbol of eq. 25 instead of the Green's function transform (sc_track.cu: compute_pipe_symbol).
//
// The FFT is a radix-4 (+ one radix-2 pass for odd log2) Stockham autosort in shared memory (ping-pong buffers, twiddles staged in
// shared memory).  Lengths 16..1024.  The work is ~4 MFLOP at 128^2: latency-, not throughput-bound.
#pragma once
#include "sc_device.cuh"

namespace sc {

__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

// In-place-semantics Stockham FFT over L points held in buffer a (scratch b).  All threads of the
// CTA call it; returns the buffer holding the result.  INV: conjugated twiddles, no 1/L scaling.
// Radix-4 passes (half as many barriers as radix-2: the kernels are pure latency chains), then one
// radix-2 pass when log2(L) is odd.  tw[m] = exp(-2 pi i m / L), m < L/2.
template <bool INV>
__device__ double2* fft_smem(double2* a, double2* b, const double2* tw, int L) {
    const int half = L >> 1, quarter = L >> 2;
    int Ns = 1, lg = 0;                           // Ns = 2^lg: shifts, not integer divisions, on the way to the twiddles
    for (; Ns * 4 <= L; Ns <<= 2, lg += 2) {
        const int tstep = quarter >> lg;          // exp(-2 pi i k/(4 Ns)) = tw[k * L/(4 Ns)]
        for (int j = threadIdx.x; j < quarter; j += blockDim.x) {
            const int k = j & (Ns - 1);
            const int m1 = k * tstep;             // < L/4
            double2 w1 = tw[m1], w2 = tw[2 * m1];  // 2 m1 < L/2
            const int m3 = 3 * m1;                // < 3L/4: tw[m + L/2] = -tw[m]
            double2 w3 = tw[m3 < half ? m3 : m3 - half];
            if (m3 >= half) { w3.x = -w3.x; w3.y = -w3.y; }
            if (INV) { w1.y = -w1.y; w2.y = -w2.y; w3.y = -w3.y; }
            const double2 u0 = a[j];
            const double2 u1 = cmul(a[j + quarter], w1);
            const double2 u2 = cmul(a[j + half], w2);
            const double2 u3 = cmul(a[j + half + quarter], w3);
            const double2 s02 = make_double2(u0.x + u2.x, u0.y + u2.y), d02 = make_double2(u0.x - u2.x, u0.y - u2.y);
            const double2 s13 = make_double2(u1.x + u3.x, u1.y + u3.y), d13 = make_double2(u1.x - u3.x, u1.y - u3.y);
            // -i (u1 - u3) forward, +i (u1 - u3) inverse
            const double2 r = INV ? make_double2(-d13.y, d13.x) : make_double2(d13.y, -d13.x);
            const int j0 = ((j - k) << 2) + k;
            b[j0] = make_double2(s02.x + s13.x, s02.y + s13.y);
            b[j0 + Ns] = make_double2(d02.x + r.x, d02.y + r.y);
            b[j0 + 2 * Ns] = make_double2(s02.x - s13.x, s02.y - s13.y);
            b[j0 + 3 * Ns] = make_double2(d02.x - r.x, d02.y - r.y);
        }
        __syncthreads();
        double2* t = a; a = b; b = t;
    }
    if (Ns < L) {                                 // one radix-2 pass left (Ns == L/2)
        for (int j = threadIdx.x; j < half; j += blockDim.x) {
            const int k = j & (Ns - 1);
            double2 w = tw[k * (half >> lg)];
            if (INV) w.y = -w.y;
            const double2 u0 = a[j];
            const double2 u1 = cmul(a[j + half], w);
            const int j0 = ((j - k) << 1) + k;
            b[j0] = make_double2(u0.x + u1.x, u0.y + u1.y);
            b[j0 + Ns] = make_double2(u0.x - u1.x, u0.y - u1.y);
        }
        __syncthreads();
        double2* t = a; a = b; b = t;
    }
    return a;
}

// grid = ny/2 CTAs, block = nx threads.  smem: 2 * Lx + Lx/2 complex.
__global__ void k_rows_fwd(const PoissonArgs p, unsigned long long* counters) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (p.noop) { pdl_launch_dependents(); pdl_wait(); return; }
    const GridDev& g = p.g;
    const int nx = g.nx, ny = g.ny, Lx = 2 * nx;
    double2* a = reinterpret_cast<double2*>(smem_raw);
    double2* b = a + Lx;
    double2* tw = b + Lx;
    const int j0 = 2 * blockIdx.x, j1 = j0 + 1;
    const bool pipe = g.boundary == SC_BOUNDARY_PIPE;
    pdl_launch_dependents();
    for (int k = threadIdx.x; k < nx; k += blockDim.x) tw[k] = g.twx[k];   // constant table: before the wait
    pdl_wait();
    // CTA 0 also turns the sigma histogram into lambda_b: its first two loads per thread go out together with the
    // grid loads below instead of after them (the kernel is as long as its slowest CTA)
    const bool lamjob = blockIdx.x == 0;
    const int b0 = threadIdx.x, b1 = threadIdx.x + blockDim.x;
    unsigned int hc0 = 0u, hc1 = 0u;
    unsigned long long n_out_now = 0ull;
    if (lamjob) { if (b0 < g.nbins) hc0 = g.hist[b0]; if (b1 < g.nbins) hc1 = g.hist[b1]; if (threadIdx.x == 0) n_out_now = counters[0]; }
    for (int i = threadIdx.x; i < Lx; i += blockDim.x) {
        double r0 = 0.0, r1 = 0.0;
        if (i < nx) {
            const size_t c0 = (size_t)j0 * nx + i, c1 = (size_t)j1 * nx + i;
            const unsigned long long v0 = g.rho[c0], v1 = g.rho[c1];
            if (g.mode == SC_DEPOSIT_FIXED) {
                r0 = (double)(long long)v0 * g.fixed_inv;
                r1 = (double)(long long)v1 * g.fixed_inv;
                g.rhoi_last[c0] = (long long)v0;
                g.rhoi_last[c1] = (long long)v1;
            } else {
                r0 = __longlong_as_double((long long)v0);
                r1 = __longlong_as_double((long long)v1);
            }
            g.rho_last[c0] = r0;
            g.rho_last[c1] = r1;
            g.rho[c0] = 0ull;
            g.rho[c1] = 0ull;
            if (pipe) {
                // eq. 18: odd extension about the wall nodes 0 and nx (charge on the wall node is dropped)
                if (i == 0) { a[0] = make_double2(0.0, 0.0); a[nx] = make_double2(0.0, 0.0); }
                else { a[i] = make_double2(r0, r1); a[Lx - i] = make_double2(-r0, -r1); }
            } else {
                a[i] = make_double2(r0, r1);
            }
        } else if (!pipe) {
            a[i] = make_double2(0.0, 0.0);            // open boundary: zero padding (Hockney)
        }
    }
    if (lamjob) {            // line density of this node: lambda_b = n_real cnt_b / (N ds)
        for (int bin = threadIdx.x; bin < g.nbins; bin += blockDim.x) {
            const unsigned int cnt = bin == b0 ? hc0 : (bin == b1 ? hc1 : g.hist[bin]);
            g.hist_last[bin] = (long long)cnt;
            const double lb = p.lam_scale * (double)cnt;      // pair table: lambda_b is .y of entry b and .x of entry b+1
            g.lam[bin].y = lb;                                //   ([0].x = [nbins].y = 0, cleared at sc_create)
            g.lam[bin + 1].x = lb;
            g.hist[bin] = 0u;
        }
        if (threadIdx.x == 0) { counters[1] = n_out_now; counters[0] = 0ull; }
    }
    __syncthreads();
    double2* z = fft_smem<false>(a, b, tw, Lx);
    // unpack the two real rows: R0 = (Z[k] + conj Z[-k])/2, R1 = (Z[k] - conj Z[-k])/(2i)
    for (int kx = threadIdx.x; kx <= nx; kx += blockDim.x) {
        const double2 zk = z[kx];
        const double2 zm = z[(Lx - kx) & (Lx - 1)];
        const double2 r0 = make_double2(0.5 * (zk.x + zm.x), 0.5 * (zk.y - zm.y));
        const double2 r1 = make_double2(0.5 * (zk.y + zm.y), -0.5 * (zk.x - zm.x));
        g.A[(size_t)kx * ny + j0] = r0;
        g.A[(size_t)kx * ny + j1] = r1;
    }
}

// grid = nx+1 CTAs, block = ny threads.  smem: 2 * Ly + Ly/2 complex.
__global__ void __launch_bounds__(512, 2) k_cols(const PoissonArgs p) {   // 64 registers: two 512-thread CTAs per SM (at 72 registers only one fitted: ncu, profiles/r03_poisson_512.md)
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (p.noop) { pdl_launch_dependents(); pdl_wait(); return; }
    const GridDev& g = p.g;
    const int ny = g.ny, Ly = 2 * ny;
    double2* a = reinterpret_cast<double2*>(smem_raw);
    double2* b = a + Ly;
    double2* tw = b + Ly;
    const int kx = blockIdx.x;
    pdl_launch_dependents();
    for (int k = threadIdx.x; k < ny; k += blockDim.x) tw[k] = g.twy[k];
    // this column's multipliers are constant tables too: fetch them before the wait (blockDim.x == ny, two per thread)
    const double* gh = g.Ghat + (size_t)kx * Ly;
    const double gs0 = gh[threadIdx.x] * p.scale, gs1 = gh[threadIdx.x + ny] * p.scale;
    pdl_wait();
    const bool pipe = g.boundary == SC_BOUNDARY_PIPE;
    for (int j = threadIdx.x; j < Ly; j += blockDim.x) {
        double2 v = make_double2(0.0, 0.0);           // open boundary: zero padding; pipe: odd about 0 and ny (eq. 18)
        if (j < ny) { if (!(pipe && j == 0)) v = g.A[(size_t)kx * ny + j]; }
        else if (pipe && j > ny) { v = g.A[(size_t)kx * ny + (Ly - j)]; v.x = -v.x; v.y = -v.y; }
        a[j] = v;
    }
    __syncthreads();
    double2* z = fft_smem<false>(a, b, tw, Ly);
    double2* o = (z == a) ? b : a;
    {
        const double2 v0 = z[threadIdx.x], v1 = z[threadIdx.x + ny];
        z[threadIdx.x] = make_double2(v0.x * gs0, v0.y * gs0);
        z[threadIdx.x + ny] = make_double2(v1.x * gs1, v1.y * gs1);
    }
    __syncthreads();
    double2* u = fft_smem<true>(z, o, tw, Ly);
    for (int j = threadIdx.x; j < ny; j += blockDim.x) {
        const double2 uj = u[j];
        double2 d;
        // differences times 1/dy (a division is a ~200-cycle dependent chain here; the product differs from it by <= 1 ulp)
        const double hy = 0.5 * g.inv_dy;
        if (j == 0) { const double2 up = u[1]; d = make_double2(-(up.x - uj.x) * g.inv_dy, -(up.y - uj.y) * g.inv_dy); }
        else if (j == ny - 1) { const double2 um = u[j - 1]; d = make_double2(-(uj.x - um.x) * g.inv_dy, -(uj.y - um.y) * g.inv_dy); }
        else { const double2 up = u[j + 1], um = u[j - 1]; d = make_double2(-(up.x - um.x) * hy, -(up.y - um.y) * hy); }
        g.BU[(size_t)kx * ny + j] = uj;
        g.BV[(size_t)kx * ny + j] = d;
    }
}

// grid = ny CTAs, block = nx threads.  smem: 2 * Lx + Lx/2 complex.
__global__ void k_rows_inv(const PoissonArgs p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (p.noop) { pdl_launch_dependents(); pdl_wait(); return; }
    const GridDev& g = p.g;
    const int nx = g.nx, ny = g.ny, Lx = 2 * nx;
    double2* a = reinterpret_cast<double2*>(smem_raw);
    double2* b = a + Lx;
    double2* tw = b + Lx;
    const int j = blockIdx.x;
    pdl_launch_dependents();
    for (int k = threadIdx.x; k < nx; k += blockDim.x) tw[k] = g.twx[k];
    pdl_wait();
    {
        // blockDim.x == nx: every thread fills k = t (direct) and k = t + nx (k = nx direct, beyond it the conjugate
        // of Lx - k); the four global loads go out together
        const int k0 = threadIdx.x, k1 = threadIdx.x + nx;
        const int s1 = k1 <= nx ? k1 : Lx - k1;
        const double2 U0 = g.BU[(size_t)k0 * ny + j], V0 = g.BV[(size_t)k0 * ny + j];
        double2 U1 = g.BU[(size_t)s1 * ny + j], V1 = g.BV[(size_t)s1 * ny + j];
        if (k1 > nx) { U1.y = -U1.y; V1.y = -V1.y; }
        a[k0] = make_double2(U0.x - V0.y, U0.y + V0.x);     // U + i V
        a[k1] = make_double2(U1.x - V1.y, U1.y + V1.x);
    }
    __syncthreads();
    double2* z = fft_smem<true>(a, b, tw, Lx);
    for (int i = threadIdx.x; i < nx; i += blockDim.x) {
        const double ui = z[i].x;
        double ex;
        if (i == 0) ex = -(z[1].x - ui) * g.inv_dx;
        else if (i == nx - 1) ex = -(ui - z[i - 1].x) * g.inv_dx;
        else ex = -(z[i + 1].x - z[i - 1].x) * (0.5 * g.inv_dx);
        g.phi[(size_t)j * nx + i] = ui;
        g.E[(size_t)j * nx + i] = make_double2(ex, z[i].y);
    }
}

}  // namespace sc
