// k_push.cuh -- the fused per-segment particle kernel.
//
// One launch carries every particle, in registers, through
//   [pending space-charge kick: bilinear gather of (Ex,Ey) + lambda(sigma) interpolation, eq. 12]
//   -> the table rows of one lattice segment (DRIFT / LINMAP / MULT / RF; section III of the paper)
//   -> [cloud-in-cell deposit, eq. 14, + lambda histogram at the SC node that ends the segment].
// Particles are SoA fp64 in HBM: 6 loads + 6 stores of 8 B per particle per launch (96 B; 64 B for
// 4D beams) is the whole DRAM traffic; the element rows, the lambda table, the CTA-private charge
// grid and histogram live in shared memory.  One persistent CTA of 1024 threads per SM.
//
// Deposit (PAPER.md:175-200 uses block-private sub-histograms + atomics; so do we, but):
//   mode 1 (deterministic): int64 fixed point, each 64-bit cell updated with NATIVE 32-bit shared
//     atomics -- low word ATOMS.ADD returning the old value, carry folded into the high-word add --
//     because 64-bit shared atomics (integer or double) compile to a CAS loop on sm_100a;
//   mode 0: fp64 atomicAdd on shared memory (CAS loop), kept for the literal eq. 14 arithmetic.
//   Grids larger than shared memory keep a centred window in shared memory; particles outside the
//   window go straight to the global grid with native L2 atomics (RED.ADD.64 / RED.ADD.F64).
#pragma once
#include "sc_device.cuh"

namespace sc {

__device__ __forceinline__ bool locate(const GridDev& g, double x, double y, int& i, int& j, double& fx, double& fy) {
    // literal IEEE sequence (no contraction): t = (x - xmin) * (1/dx); inside iff 0 <= t < n-1
    double tx = __dmul_rn(__dsub_rn(x, g.xmin), g.inv_dx);
    double ty = __dmul_rn(__dsub_rn(y, g.ymin), g.inv_dy);
    if (!(tx >= 0.0 && tx < g.nxm1 && ty >= 0.0 && ty < g.nym1)) return false;
    i = (int)tx;
    j = (int)ty;
    fx = __dsub_rn(tx, (double)i);
    fy = __dsub_rn(ty, (double)j);
    return true;
}

__device__ __forceinline__ void smem_add_u64(unsigned int* cell32, unsigned long long w) {
    unsigned int lo = (unsigned int)w, hi = (unsigned int)(w >> 32);
    unsigned int old = atomicAdd(cell32, lo);
    hi += (old + lo < old) ? 1u : 0u;           // carry out of the low word, seen by exactly one adder
    if (hi) atomicAdd(cell32 + 1, hi);
}

template <bool SIXD, int DEP>   // DEP: 0 none, 1 fp64, 2 fixed
__global__ void __launch_bounds__(kPushThreads, 1) k_push(const PushArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // layout: [rows][lam (kick grid nbins doubles)][hist (dep nbins u32)][grid window (8 B cells)]
    sc_elem* s_rows = reinterpret_cast<sc_elem*>(smem_raw);
    double* s_lam = reinterpret_cast<double*>(smem_raw + sizeof(sc_elem) * kMaxSegRows);
    const int nlam = (a.do_kick && SIXD) ? a.kg.nbins : 0;
    unsigned int* s_hist = reinterpret_cast<unsigned int*>(s_lam + nlam);
    const int nh = (DEP && SIXD) ? a.dg.nbins : 0;
    unsigned long long* s_grid = reinterpret_cast<unsigned long long*>(
        smem_raw + ((sizeof(sc_elem) * kMaxSegRows + 8 * (size_t)nlam + 4 * (size_t)nh + 15) & ~(size_t)15));
    const int tid = threadIdx.x;
    const int nrows = a.r1 - a.r0;
    const int wcells = DEP ? a.dg.wnx * a.dg.wny : 0;

    // ---- stage the segment's rows, the lambda table; zero the private grid and histogram
    {
        const int nwords = nrows * (int)(sizeof(sc_elem) / 8);
        const double* src = reinterpret_cast<const double*>(a.rows + a.r0);
        double* dst = reinterpret_cast<double*>(s_rows);
        for (int w = tid; w < nwords; w += blockDim.x) dst[w] = src[w];
        for (int b = tid; b < nlam; b += blockDim.x) s_lam[b] = a.kg.lam[b];
        for (int b = tid; b < nh; b += blockDim.x) s_hist[b] = 0u;
        for (int c = tid; c < wcells; c += blockDim.x) s_grid[c] = 0ull;
    }
    __syncthreads();

    unsigned int n_out = 0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long p = (long long)blockIdx.x * blockDim.x + tid; p < a.n; p += stride) {
        double x = a.q[0][p], px = a.q[1][p], y = a.q[2][p], py = a.q[3][p];
        double sg = 0.0, ps = 0.0;
        if (SIXD) { sg = a.q[4][p]; ps = a.q[5][p]; }

        // ---- pending space-charge kick (eq. 12): px += kappa L lambda(sigma) E~x(x,y)
        if (a.do_kick) {
            int i, j; double fx, fy;
            if (locate(a.kg, x, y, i, j, fx, fy)) {
                const double2* e = a.kg.E + (size_t)j * a.kg.nx + i;
                double2 e00 = __ldg(e), e10 = __ldg(e + 1), e01 = __ldg(e + a.kg.nx), e11 = __ldg(e + a.kg.nx + 1);
                double gx = 1.0 - fx, gy = 1.0 - fy;
                double w00 = gx * gy, w10 = fx * gy, w01 = gx * fy, w11 = fx * fy;
                double ex = w00 * e00.x + w10 * e10.x + w01 * e01.x + w11 * e11.x;
                double ey = w00 * e00.y + w10 * e10.y + w01 * e01.y + w11 * e11.y;
                double lam = a.lam_const;
                if (SIXD && a.kg.nbins > 0) {
                    double t = __dmul_rn(__dsub_rn(sg, a.kg.smin), a.kg.inv_ds);
                    lam = 0.0;
                    if (t >= 0.0 && t < a.kg.dnbins) {
                        double u = t - 0.5;
                        double b0 = floor(u);
                        double f = u - b0;
                        int ib = (int)b0;
                        double l0 = ib >= 0 ? s_lam[ib] : 0.0;
                        double l1 = ib + 1 < a.kg.nbins ? s_lam[ib + 1] : 0.0;
                        lam = (1.0 - f) * l0 + f * l1;
                    }
                }
                double k = a.kick_scale * lam;
                px += k * ex;
                py += k * ey;
            }
        }

        // ---- single-particle maps of this segment, in table order
        for (int r = 0; r < nrows; r++) {
            const sc_elem& el = s_rows[r];
            const int kind = el.kind;
            if (kind == SC_DRIFT) {
                const double L = el.p[0];
                const double d = 1.0 - ps;
                if (SIXD) sg += L * (ps * a.inv_gamma2 - 0.5 * (px * px + py * py));
                x += L * d * px;
                y += L * d * py;
            } else if (kind == SC_LINMAP) {
                const double x0 = x, y0 = y;
                x = el.p[0] * x0 + el.p[1] * px;
                px = el.p[2] * x0 + el.p[3] * px;
                y = el.p[4] * y0 + el.p[5] * py;
                py = el.p[6] * y0 + el.p[7] * py;
                if (SIXD) sg += el.p[8] * (ps * a.inv_gamma2);
            } else if (kind == SC_MULT) {
                const int n = el.ipar;
                const double kn = el.p[0], ks = el.p[1];
                double zr, zi;
                if (n == 0) { zr = 1.0; zi = 0.0; }
                else if (n == 1) { zr = x; zi = y; }
                else if (n == 2) { zr = 0.5 * (x * x - y * y); zi = x * y; }
                else if (n == 3) { zr = x * (x * x - 3.0 * y * y) * (1.0 / 6.0); zi = y * (3.0 * x * x - y * y) * (1.0 / 6.0); }
                else {
                    zr = x; zi = y;
                    for (int k = 2; k <= n; k++) {
                        const double inv = 1.0 / (double)k;
                        const double nr = (zr * x - zi * y) * inv;
                        zi = (zr * y + zi * x) * inv;
                        zr = nr;
                    }
                }
                px -= kn * zr - ks * zi;
                py += kn * zi + ks * zr;
            } else if (kind == SC_RF) {
                if (SIXD) ps -= el.p[0] * sin(el.p[1] * sg + el.p[2]);   // p0 = qV/(beta0^2 E0), p1 = 2 pi h/C
            }
        }

        a.q[0][p] = x; a.q[1][p] = px; a.q[2][p] = y; a.q[3][p] = py;
        if (SIXD) { a.q[4][p] = sg; a.q[5][p] = ps; }

        // ---- deposit at the SC node that ends this segment (eq. 14) + lambda histogram
        if (DEP) {
            int i, j; double fx, fy;
            if (locate(a.dg, x, y, i, j, fx, fy)) {
                const int li = i - a.dg.wi0, lj = j - a.dg.wj0;
                const bool inw = li >= 0 && lj >= 0 && li + 1 < a.dg.wnx && lj + 1 < a.dg.wny;
                if (DEP == 2) {
                    const long long ax = __double2ll_rn(__dmul_rn(fx, a.dg.fixed_scale));
                    const long long ay = __double2ll_rn(__dmul_rn(fy, a.dg.fixed_scale));
                    const long long S = 1ll << a.dg.bits;
                    const long long bx = S - ax, by = S - ay;
                    if (inw) {
                        unsigned int* c = reinterpret_cast<unsigned int*>(s_grid + lj * a.dg.wnx + li);
                        smem_add_u64(c, (unsigned long long)(bx * by));
                        smem_add_u64(c + 2, (unsigned long long)(ax * by));
                        smem_add_u64(c + 2 * a.dg.wnx, (unsigned long long)(bx * ay));
                        smem_add_u64(c + 2 * a.dg.wnx + 2, (unsigned long long)(ax * ay));
                    } else {
                        unsigned long long* c = a.dg.rho + (size_t)j * a.dg.nx + i;
                        atomicAdd(c, (unsigned long long)(bx * by));
                        atomicAdd(c + 1, (unsigned long long)(ax * by));
                        atomicAdd(c + a.dg.nx, (unsigned long long)(bx * ay));
                        atomicAdd(c + a.dg.nx + 1, (unsigned long long)(ax * ay));
                    }
                } else {
                    const double gx = __dsub_rn(1.0, fx), gy = __dsub_rn(1.0, fy);
                    const double w00 = __dmul_rn(gx, gy), w10 = __dmul_rn(fx, gy), w01 = __dmul_rn(gx, fy), w11 = __dmul_rn(fx, fy);
                    if (inw) {
                        double* c = reinterpret_cast<double*>(s_grid) + lj * a.dg.wnx + li;
                        atomicAdd(c, w00); atomicAdd(c + 1, w10);
                        atomicAdd(c + a.dg.wnx, w01); atomicAdd(c + a.dg.wnx + 1, w11);
                    } else {
                        double* c = reinterpret_cast<double*>(a.dg.rho) + (size_t)j * a.dg.nx + i;
                        atomicAdd(c, w00); atomicAdd(c + 1, w10);
                        atomicAdd(c + a.dg.nx, w01); atomicAdd(c + a.dg.nx + 1, w11);
                    }
                }
            } else {
                n_out++;
            }
            if (SIXD && nh > 0) {
                double t = __dmul_rn(__dsub_rn(sg, a.dg.smin), a.dg.inv_ds);
                if (t >= 0.0 && t < a.dg.dnbins) atomicAdd(&s_hist[(int)t], 1u);
            }
        }
    }

    // ---- flush the CTA-private grid and histogram into the global accumulators (native L2 atomics)
    if (DEP) {
        __syncthreads();
        for (int c = tid; c < wcells; c += blockDim.x) {
            const unsigned long long v = s_grid[c];
            if (v != 0ull) {
                const int lj = c / a.dg.wnx, li = c - lj * a.dg.wnx;
                const size_t gc = (size_t)(a.dg.wj0 + lj) * a.dg.nx + a.dg.wi0 + li;
                if (DEP == 2) atomicAdd(a.dg.rho + gc, v);
                else atomicAdd(reinterpret_cast<double*>(a.dg.rho) + gc, __longlong_as_double((long long)v));
            }
        }
        for (int b = tid; b < nh; b += blockDim.x) {
            const unsigned int v = s_hist[b];
            if (v) atomicAdd(a.dg.hist + b, v);
        }
        n_out = __reduce_add_sync(0xffffffffu, n_out);
        if ((tid & 31) == 0 && n_out) atomicAdd(a.counters, (unsigned long long)n_out);
    }
}

}  // namespace sc
