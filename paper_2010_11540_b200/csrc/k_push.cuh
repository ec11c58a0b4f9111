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
// bulk stores; the 31 consumer warps only ever touch shared memory and registers.  The kernel is bound
// by instruction issue and latency, not by bandwidth (profiles/), hence one particle per thread at the
// maximum warp count the register file allows (1024 threads x 64 registers).
// The segment's rows arrive PRE-DECODED by the host as 16-byte slots (sc_track.cu: encode_piece)
// inside the kernel parameters, i.e. in the constant bank; "drift + thin multipole" pairs are fused
// into one slot pair so that a typical segment of ~10 rows costs ~6 dispatches.
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

// ---- mbarrier / bulk-async-copy (TMA 1D) primitives; all take 32-bit shared-memory addresses -----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    } while (!ok);
}
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void bulk_load(uint32_t dst_smem, const void* src_gmem, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst_smem), "l"(src_gmem), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void bulk_store(void* dst_gmem, uint32_t src_smem, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                 ::"l"(dst_gmem), "r"(src_smem), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

// ---- cell lookup shared by gather and deposit --------------------------------------------------
__device__ __forceinline__ bool locate(const GridDev& g, double x, double y, int& i, int& j, double& fx, double& fy) {
    // literal IEEE sequence (no contraction): t = (x - xmin) * (1/dx); inside iff 0 <= t < n-1
    const double tx = __dmul_rn(__dsub_rn(x, g.xmin), g.inv_dx);
    const double ty = __dmul_rn(__dsub_rn(y, g.ymin), g.inv_dy);
    i = __double2int_rz(tx);
    j = __double2int_rz(ty);
    fx = __dsub_rn(tx, (double)i);
    fy = __dsub_rn(ty, (double)j);
    return tx >= 0.0 && tx < g.nxm1 && ty >= 0.0 && ty < g.nym1;
}

__device__ __forceinline__ void smem_add_u64(unsigned int* cell32, unsigned long long w) {
    unsigned int lo = (unsigned int)w, hi = (unsigned int)(w >> 32);
    unsigned int old = atomicAdd(cell32, lo);
    hi += (old + lo < old) ? 1u : 0u;           // carry out of the low word, seen by exactly one adder
    if (hi) atomicAdd(cell32 + 1, hi);
}

// Tile geometry of one consumer group: its particle sub-range [0, glen) is cut into a first tile of f0 and
// further tiles of T particles (all even), f0 ~ T (g+1)/G: the groups run out of phase by T/G particles.
struct TileGeom {
    int n, T, f0, glen;
    __device__ __forceinline__ int off(int t) const { return t == 0 ? 0 : f0 + (t - 1) * T; }
    __device__ __forceinline__ int cnt(int t) const {
        const int o = off(t), sz = t == 0 ? f0 : T, rem = glen - o;
        return rem < sz ? rem : sz;
    }
};
__device__ __forceinline__ TileGeom tile_geom(int glen, int g) {
    TileGeom tg;
    tg.glen = glen;
    if (glen <= 0) { tg.n = 0; tg.T = 0; tg.f0 = 0; return tg; }
    const int cap0 = (kTile * (g + 1) / kPushGroups) & ~1;
    if (glen <= cap0) { tg.n = 1; tg.T = kTile; tg.f0 = (glen + 1) & ~1; return tg; }
    const int n = 1 + (glen - cap0 + kTile - 1) / kTile;
    const int den = (n - 1) * kPushGroups + (g + 1);
    int T = (((glen * kPushGroups + den - 1) / den) + 1) & ~1;
    if (T > kTile) T = kTile;
    int f0 = ((T * (g + 1) + kPushGroups - 1) / kPushGroups + 1) & ~1;
    if (f0 > cap0) f0 = cap0;
    tg.T = T; tg.f0 = f0;
    tg.n = 1 + (glen - f0 + T - 1) / T;
    return tg;
}

template <bool SIXD, int DEP>   // DEP: 0 none, 1 fp64, 2 fixed
__global__ void __launch_bounds__(kPushThreads, 1) k_push(const __grid_constant__ PushArgs a) {
    constexpr int NC = SIXD ? 6 : 4;
    constexpr int G = kPushGroups;
    extern __shared__ __align__(128) unsigned char smem_push[];
    // layout: [mbarriers: full[G][kStages], done[G][kStages]][lam (padded)][hist][stage buffers][grid window]
    const int nlam = (a.do_kick && SIXD && a.kg.nbins > 0) ? a.kg.nbins + 2 : 0;   // [0] = [n+1] = 0: no bounds tests
    const int nh = (DEP && SIXD) ? a.dg.nbins : 0;
    double* const s_lam = reinterpret_cast<double*>(smem_push + kPushBarBytes);
    unsigned int* const s_hist = reinterpret_cast<unsigned int*>(s_lam + nlam);
    const uint32_t head = ((uint32_t)kPushBarBytes + 8u * (uint32_t)nlam + 4u * (uint32_t)nh + 15u) & ~15u;
    double* const s_stage = reinterpret_cast<double*>(smem_push + head);          // [G][kStages][NC][kTile]
    unsigned long long* const s_grid = reinterpret_cast<unsigned long long*>(smem_push + head + sizeof(double) * G * kStages * NC * kTile);
    const uint32_t bar_full = smem_u32(smem_push);                 // + 8 (g kStages + s)
    const uint32_t bar_done = bar_full + 8 * G * kStages;
    const int tid = threadIdx.x;
    const int wcells = DEP ? a.dg.wnx * a.dg.wny : 0;

    // ---- this CTA's particle range [p_lo, p_hi), an even number of particles per CTA and per group (16-byte copies)
    const long long p_lo = (long long)blockIdx.x * a.per_cta;
    const long long p_hi = p_lo + a.per_cta < a.n ? p_lo + a.per_cta : a.n;
    const int len = p_hi > p_lo ? (int)(p_hi - p_lo) : 0;
    const int gper = (((len + G - 1) / G) + 1) & ~1;
    auto group_len = [&](int g) { const int r = len - g * gper; return r < 0 ? 0 : (r < gper ? r : gper); };

    if (tid == 0) {
        for (int s = 0; s < G * kStages; s++) { mbar_init(bar_full + 8 * s, 1); mbar_init(bar_done + 8 * s, kGroupThreads); }
        fence_mbar_init();
    }
    __syncthreads();

    if (tid >= kPushConsumers) {
        // ================= producer warp: one elected lane drives the bulk-async copies of all groups =================
        if (tid == kPushConsumers && len > 0) {
            const uint32_t stage0 = smem_u32(s_stage);
            TileGeom tg[G];
            int next[G];                          // next tile of group g whose results are to be stored
            int pending = 0;
#pragma unroll
            for (int g = 0; g < G; g++) { tg[g] = tile_geom(group_len(g), g); next[g] = 0; pending += tg[g].n; }
            auto issue_load = [&](int g, int t) {
                const int s = t & (kStages - 1);
                const uint32_t bytes = (uint32_t)((tg[g].cnt(t) + 1) & ~1) * 8u;
                const uint32_t bar = bar_full + 8 * (g * kStages + s);
                mbar_arrive_expect_tx(bar, bytes * NC);
#pragma unroll
                for (int c = 0; c < NC; c++)
                    bulk_load(stage0 + (uint32_t)(((g * kStages + s) * NC + c) * kTile * 8),
                              a.q[c] + p_lo + (long long)g * gper + tg[g].off(t), bytes, bar);
            };
            for (int t = 0; t < kStages; t++)
#pragma unroll
                for (int g = 0; g < G; g++) if (t < tg[g].n) issue_load(g, t);
            while (pending > 0) {
#pragma unroll
                for (int g = 0; g < G; g++) {
                    const int t = next[g];
                    if (t >= tg[g].n) continue;
                    const int s = t & (kStages - 1);
                    if (!mbar_test(bar_done + 8 * (g * kStages + s), (uint32_t)((t / kStages) & 1))) continue;
                    // every consumer of the group wrote its results back: stream the tile out, refill the buffer
                    const uint32_t bytes = (uint32_t)((tg[g].cnt(t) + 1) & ~1) * 8u;
#pragma unroll
                    for (int c = 0; c < NC; c++)
                        bulk_store(a.q[c] + p_lo + (long long)g * gper + tg[g].off(t),
                                   stage0 + (uint32_t)(((g * kStages + s) * NC + c) * kTile * 8), bytes);
                    bulk_commit();
                    if (t + kStages < tg[g].n) { bulk_wait_read0(); issue_load(g, t + kStages); }
                    next[g] = t + 1;
                    pending--;
                }
            }
            bulk_wait0();
        }
        return;
    }

    const int grp = tid / kGroupThreads;           // consumer group of this thread
    const int gt = tid - grp * kGroupThreads;      // thread index within the group
    const TileGeom geo = tile_geom(group_len(grp), grp);

    // ================= consumers =================
    // stage the lambda table (zero-padded at both ends); zero the private grid and histogram
    if (nlam) {
        for (int b = tid; b < nlam; b += kPushConsumers) s_lam[b] = (b >= 1 && b < nlam - 1) ? a.kg.lam[b - 1] : 0.0;
    }
    for (int b = tid; b < nh; b += kPushConsumers) s_hist[b] = 0u;
    {
        ulonglong2* g2 = reinterpret_cast<ulonglong2*>(s_grid);
        const int n2 = wcells >> 1;
        for (int c = tid; c < n2; c += kPushConsumers) g2[c] = make_ulonglong2(0ull, 0ull);
        if (tid == 0 && (wcells & 1)) s_grid[wcells - 1] = 0ull;
    }
    asm volatile("bar.sync 1, %0;" ::"n"(kPushConsumers) : "memory");

    unsigned int n_out = 0;
    for (int t = 0; t < geo.n; t++) {
        const int s = t & (kStages - 1);
        const int cnt = geo.cnt(t);
        double* const st = s_stage + (grp * kStages + s) * (NC * kTile);
        const bool ok = gt < cnt;
        const int o = ok ? gt : 0;           // idle lanes shadow particle 0 (never stored, never deposited)
        mbar_wait(bar_full + 8 * (grp * kStages + s), (uint32_t)((t / kStages) & 1));

        double x = st[0 * kTile + o], px = st[1 * kTile + o], y = st[2 * kTile + o], py = st[3 * kTile + o];
        double sg = 0.0, ps = 0.0;
        if (SIXD) { sg = st[4 * kTile + o]; ps = st[5 * kTile + o]; }

        // ---- pending space-charge kick (eq. 12): px += kappa L lambda(sigma) E~x(x,y)
        if (a.do_kick) {
            int i, j; double fx, fy;
            const bool in = locate(a.kg, x, y, i, j, fx, fy);
            const double2* ep = a.kg.E + (in ? j * a.kg.nx + i : 0);
            // the four node fields are in flight while lambda is interpolated
            const double2 e00 = __ldg(ep), e10 = __ldg(ep + 1), e01 = __ldg(ep + a.kg.nx), e11 = __ldg(ep + a.kg.nx + 1);
            double lam = a.lam_const;
            if (SIXD && nlam) {
                const double tt = __dmul_rn(__dsub_rn(sg, a.kg.smin), a.kg.inv_ds);
                // padded table: entry b+1 holds bin b; u = t - 0.5 + 1 indexes it without bounds tests
                const double u = tt + 0.5;
                const int ib = __double2int_rz(u);
                const bool inb = tt >= 0.0 && tt < a.kg.dnbins;
                const double f = u - (double)ib;
                const double* lp = s_lam + (inb ? ib : 0);
                const double l0 = lp[0], l1 = lp[1];
                lam = inb ? (1.0 - f) * l0 + f * l1 : 0.0;
            }
            const double gx = 1.0 - fx, gy = 1.0 - fy;
            const double w00 = gx * gy, w10 = fx * gy, w01 = gx * fy, w11 = fx * fy;
            const double ex = w00 * e00.x + w10 * e10.x + w01 * e01.x + w11 * e11.x;
            const double ey = w00 * e00.y + w10 * e10.y + w01 * e01.y + w11 * e11.y;
            const double kk = a.kick_scale * lam;
            if (in) { px += kk * ex; py += kk * ey; }
        }

        // ---- single-particle maps of this segment, in table order (pre-decoded slots, constant bank)
        double dd = 1.0 - ps, pg = ps * a.inv_gamma2;      // change only at an RF row
#define SC_DRIFT_BODY(L)                                                              \
        {                                                                             \
            const double tl_ = (L) * dd;                                              \
            if (SIXD) sg += (L) * (pg - 0.5 * (px * px + py * py));                   \
            x += tl_ * px;                                                            \
            y += tl_ * py;                                                            \
        }
#define SC_M1_BODY(K) { px -= (K) * x; py += (K) * y; }
#define SC_M2_BODY(K) { px -= (K) * (0.5 * (x * x - y * y)); py += (K) * (x * y); }
#define SC_M3_BODY(K)                                                                 \
        {                                                                             \
            const double xx_ = x * x, yy_ = y * y;                                    \
            px -= (K) * (x * (xx_ - 3.0 * yy_) * (1.0 / 6.0));                        \
            py += (K) * (y * (3.0 * xx_ - yy_) * (1.0 / 6.0));                        \
        }
        for (int pc = 0;;) {
            const double2 h = a.prog[pc];
            const int op = __double2loint(h.x);
            const double v = h.y;
            if (op <= OP_DM3) {                            // drift, then a thin kick of order op
                const double2 kq = a.prog[pc + 1];
                pc += 2;
                SC_DRIFT_BODY(v)
                if (op == OP_DM2) SC_M2_BODY(kq.x)
                else if (op == OP_DM3) SC_M3_BODY(kq.x)
                else if (op == OP_DM1) SC_M1_BODY(kq.x)
                else { px -= kq.x; py += kq.y; }
            } else if (op == OP_DRIFT) {
                pc += 1;
                SC_DRIFT_BODY(v)
            } else if (op <= OP_M3) {
                if (op == OP_M2) { pc += 1; SC_M2_BODY(v) }
                else if (op == OP_M3) { pc += 1; SC_M3_BODY(v) }
                else if (op == OP_M1) { pc += 1; SC_M1_BODY(v) }
                else { px -= v; py += a.prog[pc + 1].x; pc += 2; }
            } else if (op == OP_LINMAP) {
                const double2 m0 = a.prog[pc + 1], m1 = a.prog[pc + 2], m2 = a.prog[pc + 3], m3 = a.prog[pc + 4];
                pc += 5;
                const double x0 = x, y0 = y;
                x = m0.x * x0 + m0.y * px;
                px = m1.x * x0 + m1.y * px;
                y = m2.x * y0 + m2.y * py;
                py = m3.x * y0 + m3.y * py;
                if (SIXD) sg += v * pg;
            } else if (op == OP_MULTG) {
                const int n = __double2hiint(h.x);
                const double ks = a.prog[pc + 1].x;
                pc += 2;
                double zr = x, zi = y;                     // n >= 1
                for (int m = 2; m <= n; m++) {
                    const double inv = 1.0 / (double)m;
                    const double nr = (zr * x - zi * y) * inv;
                    zi = (zr * y + zi * x) * inv;
                    zr = nr;
                }
                px -= v * zr - ks * zi;
                py += v * zi + ks * zr;
            } else if (op == OP_RF) {
                const double2 kp = a.prog[pc + 1];         // 2 pi h/C, phi0;  v = q V/(beta0^2 E0)
                pc += 2;
                if (SIXD) {
                    ps -= v * sin(kp.x * sg + kp.y);
                    dd = 1.0 - ps;
                    pg = ps * a.inv_gamma2;
                }
            } else {
                break;                                     // OP_END
            }
        }
#undef SC_DRIFT_BODY
#undef SC_M1_BODY
#undef SC_M2_BODY
#undef SC_M3_BODY

        // ---- results back into the stage buffer; the producer streams it to HBM
        if (ok) {
            st[0 * kTile + o] = x; st[1 * kTile + o] = px; st[2 * kTile + o] = y; st[3 * kTile + o] = py;
            if (SIXD) { st[4 * kTile + o] = sg; st[5 * kTile + o] = ps; }
        }
        fence_async_smem();              // generic-proxy writes -> visible to the async (TMA) proxy
        mbar_arrive(bar_done + 8 * (grp * kStages + s));

        // ---- deposit at the SC node that ends this segment (eq. 14) + lambda histogram
        if (DEP && ok) {
            int i, j; double fx, fy;
            if (locate(a.dg, x, y, i, j, fx, fy)) {
                const int li = i - a.dg.wi0, lj = j - a.dg.wj0;
                const bool inw = (unsigned)li < (unsigned)(a.dg.wnx - 1) && (unsigned)lj < (unsigned)(a.dg.wny - 1);
                if (DEP == 2) {
                    // ax, ay in [0, 2^s], s <= 20: 32 x 32 -> 64-bit products
                    const unsigned int ax = (unsigned int)__double2int_rn(__dmul_rn(fx, a.dg.fixed_scale));
                    const unsigned int ay = (unsigned int)__double2int_rn(__dmul_rn(fy, a.dg.fixed_scale));
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
                const double tt = __dmul_rn(__dsub_rn(sg, a.dg.smin), a.dg.inv_ds);
                if (tt >= 0.0 && tt < a.dg.dnbins) atomicAdd(&s_hist[__double2int_rz(tt)], 1u);
            }
        }
    }

    // ---- flush the CTA-private grid and histogram into the global accumulators (L2 atomics)
    if (DEP) {
        asm volatile("bar.sync 1, %0;" ::"n"(kPushConsumers) : "memory");
        if (len > 0) {
            auto red = [&](unsigned long long* dst, unsigned long long v) {
                if (DEP == 2) atomicAdd(dst, v);
                else atomicAdd(reinterpret_cast<double*>(dst), __longlong_as_double((long long)v));
            };
            if (a.dg.wnx == a.dg.nx && a.dg.wny == a.dg.ny) {
                // whole grid in the window: cell index == global index, two cells per shared load
                const ulonglong2* g2 = reinterpret_cast<const ulonglong2*>(s_grid);
                const int n2 = wcells >> 1;
                for (int c = tid; c < n2; c += kPushConsumers) {
                    const ulonglong2 v = g2[c];
                    if (v.x) red(a.dg.rho + 2 * c, v.x);
                    if (v.y) red(a.dg.rho + 2 * c + 1, v.y);
                }
            } else {
                const int warp = tid >> 5, lane = tid & 31;
                for (int lj = warp; lj < a.dg.wny; lj += kPushConsumers / 32) {
                    const unsigned long long* row = s_grid + lj * a.dg.wnx;
                    unsigned long long* grow = a.dg.rho + (size_t)(a.dg.wj0 + lj) * a.dg.nx + a.dg.wi0;
                    for (int li = lane; li < a.dg.wnx; li += 32) {
                        const unsigned long long v = row[li];
                        if (v) red(grow + li, v);
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

}  // namespace sc
