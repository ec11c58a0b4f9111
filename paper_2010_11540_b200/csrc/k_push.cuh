// k_push.cuh -- the fused per-segment particle kernel.
//
// One launch carries every particle through
//   [pending space-charge kick: bilinear gather of (Ex,Ey) + lambda(sigma) interpolation, eq. 12]
//   -> the table rows of one lattice segment (DRIFT / LINMAP / MULT / RF; section III of the paper)
//   -> [cloud-in-cell deposit, eq. 14, + lambda histogram at the SC node that ends the segment].
// Particles are SoA fp64 in HBM: 6 loads + 6 stores of 8 B per particle per launch (96 B; 64 B for
// 4D beams) is the whole DRAM traffic.
//
// Data movement (Blackwell): one persistent CTA per SM owns a contiguous particle range and walks it
// in tiles.  A producer warp streams each tile HBM -> shared memory with 1D bulk-async copies (TMA,
// cp.async.bulk, completion on an mbarrier), double-buffered, and streams the updated tile back with
// bulk stores; the 8 consumer warps only ever touch shared memory and registers (four particles per
// thread, so every decoded table row is applied four times and the four dependency chains interleave:
// the kernel is bound by instruction latency, not by bandwidth, see profiles/).
// The segment's rows arrive PRE-DECODED by the host as 16-byte slots (sc_track.cu: encode_program)
// inside the kernel parameters, i.e. in the constant bank: a row costs one uniform load + a branch.
//
// Deposit (PAPER.md:175-200 uses block-private sub-histograms + atomics; so do we, but):
//   mode 1 (deterministic): int64 fixed point, each 64-bit cell updated with NATIVE 32-bit shared
//     atomics -- low word ATOMS.ADD returning the old value, carry folded into the high-word add --
//     because 64-bit shared atomics (integer or double) compile to a CAS loop on sm_100a;
//   mode 0: fp64 atomicAdd on shared memory (CAS loop), kept for the literal eq. 14 arithmetic.
//   Grids larger than shared memory keep a centred window in shared memory; particles outside the
//   window go straight to the global grid with L2 atomics (RED.ADD.64 / RED.ADD.F64).
//   Measured on B200 (profiles/r01_atomics_microbench.md): the shared-memory scheme costs ~4 us per
//   1e6 particles, direct L2 REDs 69-209 us, so the CTA-private grid of the paper still holds.
#pragma once
#include "sc_device.cuh"

namespace sc {

// ---- mbarrier / bulk-async-copy (TMA 1D) primitives -------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    const uint32_t addr = smem_u32(bar);
    uint32_t ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(addr), "r"(parity) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void bulk_load(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_store(void* dst_gmem, const void* src_smem, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                 ::"l"(dst_gmem), "r"(smem_u32(src_smem)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

// ---- cell lookup shared by gather and deposit --------------------------------------------------
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
__global__ void __launch_bounds__(kPushThreads, 1) k_push(const __grid_constant__ PushArgs a) {
    constexpr int NC = SIXD ? 6 : 4;
    constexpr int P = kPushP;
    extern __shared__ __align__(128) unsigned char smem_push[];
    // layout: [mbarriers][lam][hist][stage buffers][grid window]
    uint64_t* bar_full = reinterpret_cast<uint64_t*>(smem_push);            // [kStages]
    uint64_t* bar_done = bar_full + kStages;                                // [kStages]
    double* s_lam = reinterpret_cast<double*>(smem_push + 32);
    const int nlam = (a.do_kick && SIXD) ? a.kg.nbins : 0;
    unsigned int* s_hist = reinterpret_cast<unsigned int*>(s_lam + nlam);
    const int nh = (DEP && SIXD) ? a.dg.nbins : 0;
    const size_t head = (32 + 8 * (size_t)nlam + 4 * (size_t)nh + 15) & ~(size_t)15;
    double* s_stage = reinterpret_cast<double*>(smem_push + head);          // [kStages][NC][kTile]
    unsigned long long* s_grid = reinterpret_cast<unsigned long long*>(smem_push + head + sizeof(double) * kStages * NC * kTile);
    const int tid = threadIdx.x;
    const int nslots = a.nslots;
    const int wcells = DEP ? a.dg.wnx * a.dg.wny : 0;

    // ---- this CTA's particle range [p_lo, p_hi), an even number of particles per CTA (16-byte copies)
    const long long per = a.per_cta;
    const long long p_lo = (long long)blockIdx.x * per;
    const long long p_hi = p_lo + per < a.n ? p_lo + per : a.n;
    const int len = p_hi > p_lo ? (int)(p_hi - p_lo) : 0;
    const int ntiles = (len + kTile - 1) / kTile;
    // equal tiles (even size): no short last tile
    const int tsize = ntiles ? ((((len + ntiles - 1) / ntiles) + 1) & ~1) : 0;

    if (tid == 0) {
        for (int s = 0; s < kStages; s++) { mbar_init(&bar_full[s], 1); mbar_init(&bar_done[s], kPushConsumers); }
        fence_mbar_init();
    }
    __syncthreads();

    auto tile_count = [&](int t) { const int rem = len - t * tsize; return rem < tsize ? rem : tsize; };

    if (tid >= kPushConsumers) {
        // ================= producer warp: one elected lane drives the bulk-async copies =================
        if (tid == kPushConsumers && ntiles > 0) {
            auto issue_load = [&](int t) {
                const int s = t % kStages;
                const uint32_t bytes = (uint32_t)((tile_count(t) + 1) & ~1) * 8u;
                mbar_arrive_expect_tx(&bar_full[s], bytes * NC);
#pragma unroll
                for (int c = 0; c < NC; c++)
                    bulk_load(s_stage + ((size_t)s * NC + c) * kTile, a.q[c] + p_lo + (long long)t * tsize, bytes, &bar_full[s]);
            };
            for (int t = 0; t < kStages && t < ntiles; t++) issue_load(t);
            for (int t = 0; t < ntiles; t++) {
                const int s = t % kStages;
                mbar_wait(&bar_done[s], (uint32_t)((t / kStages) & 1));     // every consumer wrote its results back
                const uint32_t bytes = (uint32_t)((tile_count(t) + 1) & ~1) * 8u;
#pragma unroll
                for (int c = 0; c < NC; c++)
                    bulk_store(a.q[c] + p_lo + (long long)t * tsize, s_stage + ((size_t)s * NC + c) * kTile, bytes);
                bulk_commit();
                if (t + kStages < ntiles) { bulk_wait_read0(); issue_load(t + kStages); }
            }
            bulk_wait0();
        }
    } else {
        // ================= consumers =================
        // stage the lambda table; zero the private grid and histogram
        {
            for (int b = tid; b < nlam; b += kPushConsumers) s_lam[b] = a.kg.lam[b];
            for (int b = tid; b < nh; b += kPushConsumers) s_hist[b] = 0u;
            ulonglong2* g2 = reinterpret_cast<ulonglong2*>(s_grid);
            for (int c = tid; c < (wcells >> 1); c += kPushConsumers) g2[c] = make_ulonglong2(0ull, 0ull);
            if (tid == 0 && (wcells & 1)) s_grid[wcells - 1] = 0ull;
        }
        asm volatile("bar.sync 1, %0;" ::"n"(kPushConsumers) : "memory");

        unsigned int n_out = 0;
        for (int t = 0; t < ntiles; t++) {
            const int s = t % kStages;
            const int cnt = tile_count(t);
            double* st = s_stage + (size_t)s * NC * kTile;
            mbar_wait(&bar_full[s], (uint32_t)((t / kStages) & 1));

            double x[P], px[P], y[P], py[P], sg[P], ps[P];
            bool ok[P];
#pragma unroll
            for (int k = 0; k < P; k++) {
                const int o = tid + k * kPushConsumers;
                ok[k] = o < cnt;
                x[k] = ok[k] ? st[0 * kTile + o] : 0.0;
                px[k] = ok[k] ? st[1 * kTile + o] : 0.0;
                y[k] = ok[k] ? st[2 * kTile + o] : 0.0;
                py[k] = ok[k] ? st[3 * kTile + o] : 0.0;
                sg[k] = (SIXD && ok[k]) ? st[4 * kTile + o] : 0.0;
                ps[k] = (SIXD && ok[k]) ? st[5 * kTile + o] : 0.0;
            }

            // ---- pending space-charge kick (eq. 12): px += kappa L lambda(sigma) E~x(x,y)
            if (a.do_kick) {
                double fx[P], fy[P]; bool in[P];
                const double2* ep[P];
#pragma unroll
                for (int k = 0; k < P; k++) {
                    int i = 0, j = 0;
                    in[k] = ok[k] && locate(a.kg, x[k], y[k], i, j, fx[k], fy[k]);
                    ep[k] = a.kg.E + (in[k] ? j * a.kg.nx + i : 0);
                }
#pragma unroll
                for (int k = 0; k < P; k++) {
                    // the four node fields of this particle are in flight while lambda is interpolated
                    const double2 e00 = __ldg(ep[k]), e10 = __ldg(ep[k] + 1), e01 = __ldg(ep[k] + a.kg.nx), e11 = __ldg(ep[k] + a.kg.nx + 1);
                    double lam = a.lam_const;
                    if (SIXD && a.kg.nbins > 0) {
                        const double tt = __dmul_rn(__dsub_rn(sg[k], a.kg.smin), a.kg.inv_ds);
                        lam = 0.0;
                        if (tt >= 0.0 && tt < a.kg.dnbins) {
                            const double u = tt - 0.5;
                            const double b0 = floor(u);
                            const double f = u - b0;
                            const int ib = (int)b0;
                            const double l0 = ib >= 0 ? s_lam[ib] : 0.0;
                            const double l1 = ib + 1 < a.kg.nbins ? s_lam[ib + 1] : 0.0;
                            lam = (1.0 - f) * l0 + f * l1;
                        }
                    }
                    if (in[k]) {
                        const double gx = 1.0 - fx[k], gy = 1.0 - fy[k];
                        const double w00 = gx * gy, w10 = fx[k] * gy, w01 = gx * fy[k], w11 = fx[k] * fy[k];
                        const double ex = w00 * e00.x + w10 * e10.x + w01 * e01.x + w11 * e11.x;
                        const double ey = w00 * e00.y + w10 * e10.y + w01 * e01.y + w11 * e11.y;
                        const double kk = a.kick_scale * lam;
                        px[k] += kk * ex;
                        py[k] += kk * ey;
                    }
                }
            }

            // ---- single-particle maps of this segment, in table order (pre-decoded slots, constant bank)
            double dd[P], pg[P];             // 1 - psigma, psigma / gamma0^2: change only at an RF row
#pragma unroll
            for (int k = 0; k < P; k++) { dd[k] = 1.0 - ps[k]; pg[k] = ps[k] * a.inv_gamma2; }
            double2 h = a.prog[0];
            for (int pc = 0; pc < nslots;) {
                const int op = __double2loint(h.x);
                const double v = h.y;
                if (op == OP_DRIFT) {
                    pc += 1; h = a.prog[pc];
#pragma unroll
                    for (int k = 0; k < P; k++) {
                        const double tl = v * dd[k];
                        if (SIXD) sg[k] += v * (pg[k] - 0.5 * (px[k] * px[k] + py[k] * py[k]));
                        x[k] += tl * px[k];
                        y[k] += tl * py[k];
                    }
                } else if (op == OP_MULT2) {
                    pc += 1; h = a.prog[pc];
#pragma unroll
                    for (int k = 0; k < P; k++) {
                        px[k] -= v * (0.5 * (x[k] * x[k] - y[k] * y[k]));
                        py[k] += v * (x[k] * y[k]);
                    }
                } else if (op == OP_MULT3) {
                    pc += 1; h = a.prog[pc];
#pragma unroll
                    for (int k = 0; k < P; k++) {
                        const double xx = x[k] * x[k], yy = y[k] * y[k];
                        px[k] -= v * (x[k] * (xx - 3.0 * yy) * (1.0 / 6.0));
                        py[k] += v * (y[k] * (3.0 * xx - yy) * (1.0 / 6.0));
                    }
                } else if (op == OP_MULT1) {
                    pc += 1; h = a.prog[pc];
#pragma unroll
                    for (int k = 0; k < P; k++) { px[k] -= v * x[k]; py[k] += v * y[k]; }
                } else if (op == OP_KICK0) {
                    const double ks = a.prog[pc + 1].x;
                    pc += 2; h = a.prog[pc];
#pragma unroll
                    for (int k = 0; k < P; k++) { px[k] -= v; py[k] += ks; }
                } else if (op == OP_LINMAP) {
                    const double2 m0 = a.prog[pc + 1], m1 = a.prog[pc + 2], m2 = a.prog[pc + 3], m3 = a.prog[pc + 4];
                    pc += 5; h = a.prog[pc];
#pragma unroll
                    for (int k = 0; k < P; k++) {
                        const double x0 = x[k], y0 = y[k];
                        x[k] = m0.x * x0 + m0.y * px[k];
                        px[k] = m1.x * x0 + m1.y * px[k];
                        y[k] = m2.x * y0 + m2.y * py[k];
                        py[k] = m3.x * y0 + m3.y * py[k];
                        if (SIXD) sg[k] += v * pg[k];
                    }
                } else if (op == OP_MULTG) {
                    const int n = __double2hiint(h.x);
                    const double ks = a.prog[pc + 1].x;
                    pc += 2; h = a.prog[pc];
#pragma unroll
                    for (int k = 0; k < P; k++) {
                        double zr = x[k], zi = y[k];                    // n >= 1
                        for (int m = 2; m <= n; m++) {
                            const double inv = 1.0 / (double)m;
                            const double nr = (zr * x[k] - zi * y[k]) * inv;
                            zi = (zr * y[k] + zi * x[k]) * inv;
                            zr = nr;
                        }
                        px[k] -= v * zr - ks * zi;
                        py[k] += v * zi + ks * zr;
                    }
                } else if (op == OP_RF) {
                    const double2 kp = a.prog[pc + 1];             // 2 pi h/C, phi0;  v = q V/(beta0^2 E0)
                    pc += 2; h = a.prog[pc];
#pragma unroll
                    for (int k = 0; k < P; k++) {
                        if (SIXD) {
                            ps[k] -= v * sin(kp.x * sg[k] + kp.y);
                            dd[k] = 1.0 - ps[k];
                            pg[k] = ps[k] * a.inv_gamma2;
                        }
                    }
                } else {
                    pc = nslots;
                }
            }

            // ---- results back into the stage buffer; the producer streams it to HBM
#pragma unroll
            for (int k = 0; k < P; k++) {
                const int o = tid + k * kPushConsumers;
                if (ok[k]) {
                    st[0 * kTile + o] = x[k]; st[1 * kTile + o] = px[k]; st[2 * kTile + o] = y[k]; st[3 * kTile + o] = py[k];
                    if (SIXD) { st[4 * kTile + o] = sg[k]; st[5 * kTile + o] = ps[k]; }
                }
            }
            fence_async_smem();              // generic-proxy writes -> visible to the async (TMA) proxy
            mbar_arrive(&bar_done[s]);

            // ---- deposit at the SC node that ends this segment (eq. 14) + lambda histogram
            if (DEP) {
#pragma unroll
                for (int k = 0; k < P; k++) {
                    if (!ok[k]) continue;
                    int i, j; double fx, fy;
                    if (locate(a.dg, x[k], y[k], i, j, fx, fy)) {
                        const int li = i - a.dg.wi0, lj = j - a.dg.wj0;
                        const bool inw = li >= 0 && lj >= 0 && li + 1 < a.dg.wnx && lj + 1 < a.dg.wny;
                        if (DEP == 2) {
                            // ax, ay in [0, 2^s], s <= 20: 32 x 32 -> 64-bit products
                            const unsigned int ax = (unsigned int)__double2ll_rn(__dmul_rn(fx, a.dg.fixed_scale));
                            const unsigned int ay = (unsigned int)__double2ll_rn(__dmul_rn(fy, a.dg.fixed_scale));
                            const unsigned int S = 1u << a.dg.bits;
                            const unsigned int bx = S - ax, by = S - ay;
                            const unsigned long long w00 = (unsigned long long)bx * by, w10 = (unsigned long long)ax * by;
                            const unsigned long long w01 = (unsigned long long)bx * ay, w11 = (unsigned long long)ax * ay;
                            if (inw) {
                                unsigned int* c = reinterpret_cast<unsigned int*>(s_grid + lj * a.dg.wnx + li);
                                smem_add_u64(c, w00);
                                smem_add_u64(c + 2, w10);
                                smem_add_u64(c + 2 * a.dg.wnx, w01);
                                smem_add_u64(c + 2 * a.dg.wnx + 2, w11);
                            } else {
                                unsigned long long* c = a.dg.rho + (size_t)j * a.dg.nx + i;
                                atomicAdd(c, w00);
                                atomicAdd(c + 1, w10);
                                atomicAdd(c + a.dg.nx, w01);
                                atomicAdd(c + a.dg.nx + 1, w11);
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
                        const double tt = __dmul_rn(__dsub_rn(sg[k], a.dg.smin), a.dg.inv_ds);
                        if (tt >= 0.0 && tt < a.dg.dnbins) atomicAdd(&s_hist[(int)tt], 1u);
                    }
                }
            }
        }

        // ---- flush the CTA-private grid and histogram into the global accumulators (L2 atomics)
        if (DEP) {
            asm volatile("bar.sync 1, %0;" ::"n"(kPushConsumers) : "memory");
            if (ntiles > 0) {
                const int warp = tid >> 5, lane = tid & 31;
                for (int lj = warp; lj < a.dg.wny; lj += kPushConsumers / 32) {
                    const unsigned long long* row = s_grid + lj * a.dg.wnx;
                    unsigned long long* grow = a.dg.rho + (size_t)(a.dg.wj0 + lj) * a.dg.nx + a.dg.wi0;
                    for (int li = lane; li < a.dg.wnx; li += 32) {
                        const unsigned long long v = row[li];
                        if (v != 0ull) {
                            if (DEP == 2) atomicAdd(grow + li, v);
                            else atomicAdd(reinterpret_cast<double*>(grow) + li, __longlong_as_double((long long)v));
                        }
                    }
                }
                for (int b = tid; b < nh; b += kPushConsumers) {
                    const unsigned int v = s_hist[b];
                    if (v) atomicAdd(a.dg.hist + b, v);
                }
            }
            n_out = __reduce_add_sync(0xffffffffu, n_out);
            if ((tid & 31) == 0 && n_out) atomicAdd(a.counters, (unsigned long long)n_out);
        }
    }
}

}  // namespace sc
