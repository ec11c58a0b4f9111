// k_poisson_cluster.cuh -- the whole field solve of one SC node on a 128 x 128 grid in ONE launch of ONE thread-block
// cluster, the stages handing over through DISTRIBUTED SHARED MEMORY with mbarrier-counted asynchronous stores.
//
// Same mathematics as k_poisson.cuh / k_poisson_warp.cuh (open boundary: Hockney convolution with the precomputed real
// transform of the cell-integrated Green's function on the doubled grid; pipe: the paper's odd extension and eq. 25,
// PAPER.md:204-289; node field by differences, eq. 29):
//     A  128 rows forward      (one real row per 256-point complex transform, Hermitian half kx = 0..128 kept)
//     B  128 columns           (forward, x multiplier, inverse, crop to j < 128)
//     C  128 rows inverse      (Hermitian extension of U -> the potential, a real row)
//     D  E~x, E~y by differences of the potential (neighbour rows through shared memory / a one-row halo per CTA)
// What the three-launch paths pay for is the hand-over: arrays stored to L2, a kernel boundary (~1 us under programmatic
// dependent launch) and a cold first load per stage.  Here
//   * the cluster is 16 CTAs x 128 threads (non-portable cluster size, allowed on sm_100a): 128 GROUPS of 16 lanes, group
//     g owns row g in stages A and C and column g in stage B; every stage is one round of all groups;
//   * a 256-point transform is 16 points per lane: 16-point FFT in registers, twiddle, ONE exchange through a padded
//     shared-memory tile, 16-point FFT in registers.  Input layout (lane t holds 16 n1 + t) and output layout (lane t holds
//     t + 16 k2) are the same, so forward -> multiply -> inverse needs no reordering, and the twiddles W^(t k1) are 15
//     per-lane constants held in registers for all four transforms.  (One transform per 32-lane warp with 8 points per lane
//     needs two exchanges plus natural-order round trips: with 8 such warps per SM the shared-memory port, not the fp64
//     pipe, set the pace -- 13.4 us per node measured for that first cluster version against 9.0 us for the three-launch
//     path, whose warps have an SM almost to themselves.)
//   * hand-over: the producer writes each 16-byte result straight into the consumer group's input buffer in another CTA's
//     shared memory with st.async (SASS STAS), which counts bytes on an mbarrier in that CTA; the consumer waits for its own
//     buffer only.  No cluster-wide barrier between the stages (barrier.cluster with release semantics also waits for the
//     kernel's outstanding GLOBAL stores: ~0.8-1.2 us each in the first version) and no fence;
//   * columns kx = 0 and kx = 128 of the row spectra of real rows are real sequences: they share ONE complex column
//     transform (job 0), so that stage B is exactly 128 jobs.
#pragma once
#include "k_poisson_fused.cuh"   // fft16_impl, complex helpers

namespace sc {

constexpr int kPcN = 128;                       // nodes per axis
constexpr int kPcCtas = 16;                     // CTAs in the cluster
constexpr int kPcThreads = 128;                 // 4 warps = 8 groups of 16 lanes per CTA
constexpr int kPcGroups = kPcThreads / 16;
// shared memory per CTA, in 16-byte units: per group [exchange tile 16 x 17][column input 128][row input 129 + 1]
constexpr int kPcTile = 16 * 17, kPcCol = kPcTile, kPcRow = kPcTile + kPcN, kPcGroup = kPcTile + kPcN + kPcN + 2;
constexpr size_t kPcOffPhi = (size_t)kPcGroups * kPcGroup * 16;                 // (groups + 2 halo rows) x 128 doubles
constexpr size_t kPcOffGs2 = kPcOffPhi + (size_t)(kPcGroups + 2) * kPcN * 8;    // job 0's second multiplier row, 256 doubles
constexpr size_t kPcOffBar = kPcOffGs2 + 2 * kPcN * 8;                          // mbarriers: column inputs [4 warps], row inputs [4], halo
constexpr size_t kPcSmemBytes = kPcOffBar + 16 * 8;

#ifdef SC_TRACE
#define SC_STAMPC(k_) do { if (threadIdx.x == 0) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); counters[8 + blockIdx.x * 16 + (k_)] = t_; } } while (0)
#else
#define SC_STAMPC(k_) do { } while (0)
#endif

__device__ __forceinline__ unsigned cluster_ctarank() { unsigned r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ uint32_t mapa_shared(uint32_t addr, unsigned rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
// asynchronous 16- / 8-byte store into (another) CTA's shared memory; the bytes are counted on an mbarrier of that CTA
__device__ __forceinline__ void st_async2(uint32_t addr, double2 v, uint32_t mbar) {
    asm volatile("st.async.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1,%2}, [%3];" ::"r"(addr), "d"(v.x), "d"(v.y), "r"(mbar) : "memory");
}
__device__ __forceinline__ void st_async1(uint32_t addr, double v, uint32_t mbar) {
    asm volatile("st.async.shared::cluster.mbarrier::complete_tx::bytes.f64 [%0], %1, [%2];" ::"r"(addr), "d"(v), "r"(mbar) : "memory");
}
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }   // ordering comes from fence.mbarrier_init before and wait.acquire after
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ void pc_mbar_init(uint32_t bar, unsigned count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory"); }
__device__ __forceinline__ void pc_mbar_expect(uint32_t bar, unsigned bytes) { asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory"); }
__device__ __forceinline__ void pc_mbar_wait(uint32_t bar, unsigned parity) {
    asm volatile(
        "{\n.reg .pred p;\nWAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\nbra WAIT_%=;\nDONE_%=:\n}" ::"r"(bar), "r"(parity) : "memory");
}

// One 256-point transform by a group of 16 lanes.  In: lane t holds v[n1] = x[16 n1 + t].  Out: lane t holds v[k2] = X[t + 16 k2].
// tw[k1] = exp(-2 pi i t k1/256) in registers; ex: the group's exchange tile (16 rows of 17).  Both groups of a warp call it together.
template <bool INV>
__device__ __forceinline__ void fft256_group(double2 (&v)[16], double2* ex, const double2 (&tw)[16], int t) {
    fft16_impl<INV>(v);                                      // over n1 -> k1
#pragma unroll
    for (int k1 = 1; k1 < 16; k1++) {
        double2 w = tw[k1];
        if (INV) w.y = -w.y;
        v[k1] = cmulf(v[k1], w);
    }
#pragma unroll
    for (int k1 = 0; k1 < 16; k1++) ex[k1 * 17 + t] = v[k1];
    __syncwarp();
#pragma unroll
    for (int n2 = 0; n2 < 16; n2++) v[n2] = ex[t * 17 + n2];   // lane k1 gathers over n2
    __syncwarp();                                            // the tile is free again
    fft16_impl<INV>(v);                                      // over n2 -> k2
}

// grid = ONE cluster of 16 CTAs of 128 threads.  counters: [0] n_outside accumulating, [1] of the last node.
__global__ void __launch_bounds__(kPcThreads) k_poisson_cluster(const PoissonArgs p, unsigned long long* counters) {
    constexpr int N = kPcN, L = 2 * N;
    constexpr int TT = kPcCtas * kPcThreads, HB = (kMaxBins + TT - 1) / TT;      // histogram bins per thread
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (p.noop) { pdl_launch_dependents(); pdl_wait(); return; }
    const GridDev& g = p.g;
    const int tid = threadIdx.x, t = tid & 15, warp = tid >> 5, lg = tid >> 4;
    const unsigned rank = cluster_ctarank();
    const int gg = (int)rank * kPcGroups + lg;                   // this group's row (stages A, C, D) and column (stage B)
    double2* const s_c = reinterpret_cast<double2*>(smem_raw);
    double2* const ex = s_c + lg * kPcGroup;
    const double2* const col = ex + kPcCol;
    const double2* const row = ex + kPcRow;
    double* const s_phi = reinterpret_cast<double*>(smem_raw + kPcOffPhi);
    double* const s_gs2 = reinterpret_cast<double*>(smem_raw + kPcOffGs2);
    const uint32_t sa = (uint32_t)__cvta_generic_to_shared(smem_raw);
    const uint32_t bar0 = sa + (uint32_t)kPcOffBar;              // [0..3] column inputs per warp, [4..7] row inputs per warp, [8] halo rows
    const bool pipe = g.boundary == SC_BOUNDARY_PIPE;

    SC_STAMPC(0);
    pdl_launch_dependents();
    if (tid == 0) {
        // thread 0 arms all of this CTA's barriers (a warp's two groups share theirs) before it arrives at the cluster barrier:
        // no block-wide synchronisation, and the fence is issued while no load is outstanding (a fence waits for those too)
        for (int b = 0; b < 9; b++) pc_mbar_init(bar0 + 8u * b, 1);
        for (int w = 0; w < 4; w++) {
            pc_mbar_expect(bar0 + 8u * w, 2u * N * 16u);          // 128 producers x 16 bytes per column job
            pc_mbar_expect(bar0 + 8u * (4 + w), 2u * (N + 1) * 16u);
        }
        pc_mbar_expect(bar0 + 64u, (unsigned)((rank > 0) + (rank + 1 < kPcCtas)) * N * 8u);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
    cluster_arrive();                                            // "this CTA's barriers are armed": waited for before the first remote store
    SC_STAMPC(13);
    pdl_wait();                                                  // the deposit of the preceding k_push is final
    SC_STAMPC(1);
    // ---------------------------------------------------------------- every load of the kernel goes out now, untouched (no arithmetic
    // on the results yet: an in-order warp would stall on the first use): this row of the deposit, the histogram slice, the
    // constants
    unsigned long long raw[8], mr[8];
#pragma unroll
    for (int n1 = 0; n1 < 8; n1++) raw[n1] = g.rho[(size_t)gg * N + 16 * n1 + t];
#pragma unroll
    for (int n1 = 0; n1 < 8; n1++) {                             // pipe: n = N + 16 n1 + t mirrors to L - n = N - 16 n1 - t (eq. 18)
        const int src = N - 16 * n1 - t;
        mr[n1] = (pipe && src >= 1 && src < N) ? g.rho[(size_t)gg * N + src] : 0ull;
    }
    unsigned long long n_out_now = 0ull;
    if (gg == 0 && t == 0) n_out_now = counters[0];
    const int gtid = (int)rank * kPcThreads + tid;
    unsigned int hc[HB];
#pragma unroll
    for (int q = 0; q < HB; q++) { const int bin = gtid + q * TT; hc[q] = bin < g.nbins ? g.hist[bin] : 0u; }
    double2 tw[16];                                              // exp(-2 pi i t k1/256) from the half-circle table (sign applied below)
#pragma unroll
    for (int k1 = 1; k1 < 16; k1++) tw[k1] = __ldg(g.twx + ((t * k1) & (N - 1)));
    double gs[16], gs2[16];                                      // this column's multipliers in the transform's layout (scaled below)
#pragma unroll
    for (int k2 = 0; k2 < 16; k2++) gs[k2] = __ldg(g.Ghat + (size_t)gg * L + t + 16 * k2);
    if (gg == 0) {                                               // job 0 also carries column kx = N
#pragma unroll
        for (int k2 = 0; k2 < 16; k2++) gs2[k2] = __ldg(g.Ghat + (size_t)N * L + t + 16 * k2);
    }
    SC_STAMPC(14);
    tw[0] = make_double2(1.0, 0.0);
#pragma unroll
    for (int k1 = 1; k1 < 16; k1++) if (t * k1 >= N) tw[k1] = make_double2(-tw[k1].x, -tw[k1].y);

    // ---------------------------------------------------------------- stage A: row gg forward
    auto conv = [&](unsigned long long r) {
        return g.mode == SC_DEPOSIT_FIXED ? (double)(long long)r * g.fixed_inv : __longlong_as_double((long long)r);
    };
    double2 v[16];
#pragma unroll
    for (int n1 = 0; n1 < 8; n1++) {
        const int i = 16 * n1 + t;
        v[n1] = make_double2((pipe && i == 0) ? 0.0 : conv(raw[n1]), 0.0);   // the wall node carries no charge
        v[n1 + 8] = make_double2(pipe ? -conv(mr[n1]) : 0.0, 0.0);
    }
    SC_STAMPC(2);
    fft256_group<false>(v, ex, tw, t);
    SC_STAMPC(3);
    cluster_wait();                                              // every CTA of the cluster runs and has armed its barriers
    // A[kx][gg], kx = t + 16 k2 <= N, to the group that owns column kx; kx = 0 and kx = N (lane 0) are real: one entry (A[0], A[N])
#pragma unroll
    for (int k2 = 0; k2 < 8; k2++) {
        const int kx = t + 16 * k2;
        double2 val = v[k2];
        if (kx == 0) val = make_double2(v[0].x, v[8].x);
        const unsigned dr = (unsigned)(kx >> 3);
        const int dl = kx & 7;
        SC_ASSERT(counters, kx >= 0 && kx < N && dr < (unsigned)kPcCtas && (size_t)((dl * kPcGroup + kPcCol + gg) * 16 + 16) <= kPcOffPhi);
        st_async2(mapa_shared(sa + (uint32_t)((dl * kPcGroup + kPcCol + gg) * 16), dr), val, mapa_shared(bar0 + 8u * (dl >> 1), dr));
    }
    SC_STAMPC(4);
    // book-keeping off the critical path (the column inputs are still on their way): the node's deposit for sc_get_grid, the
    // accumulator cleared for the next deposit, and the line density lambda_b = n_real cnt_b / (N ds) as a pair table
    // (lambda_b is .y of entry b and .x of entry b+1)
#pragma unroll
    for (int n1 = 0; n1 < 8; n1++) {
        const size_t c = (size_t)gg * N + 16 * n1 + t;
        if (g.mode == SC_DEPOSIT_FIXED) g.rhoi_last[c] = (long long)raw[n1];
        g.rho_last[c] = conv(raw[n1]);
        g.rho[c] = 0ull;                                         // (every lane's loads of this row returned long ago)
    }
#pragma unroll
    for (int q = 0; q < HB; q++) {
        const int bin = gtid + q * TT;
        if (bin < g.nbins) {
            g.hist_last[bin] = (long long)hc[q];
            const double lb = p.lam_scale * (double)hc[q];
            g.lam[bin].y = lb; g.lam[bin + 1].x = lb;
            g.hist[bin] = 0u;
        }
    }
    if (gg == 0 && t == 0) { counters[1] = n_out_now; counters[0] = 0ull; }
#pragma unroll
    for (int k2 = 0; k2 < 16; k2++) gs[k2] *= p.scale;
    if (gg == 0) {
#pragma unroll
        for (int k2 = 0; k2 < 16; k2++) s_gs2[t + 16 * k2] = gs2[k2] * p.scale;     // read back by the same lane
    }

    // ---------------------------------------------------------------- stage B: column gg
    pc_mbar_wait(bar0 + 8u * warp, 0);
    SC_STAMPC(5);
#pragma unroll
    for (int n1 = 0; n1 < 8; n1++) {
        const int j = 16 * n1 + t;
        double2 a = col[j];
        if (pipe && j == 0) a = make_double2(0.0, 0.0);
        v[n1] = a;
        double2 mm = make_double2(0.0, 0.0);
        if (pipe) {
            const int src = N - 16 * n1 - t;                      // j' = N + 16 n1 + t mirrors to L - j' (odd extension, eq. 18)
            if (src >= 1 && src < N) { mm = col[src]; mm.x = -mm.x; mm.y = -mm.y; }
        }
        v[n1 + 8] = mm;
    }
    fft256_group<false>(v, ex, tw, t);
    if (gg == 0) {
        // two real columns in one transform: X0 = (Z[k] + conj Z[-k])/2, XN = (Z[k] - conj Z[-k])/(2i); each takes its own
        // (real, even) multiplier; repacked as G0 X0 + i GN XN, whose inverse is U0 + i UN with U0, UN real.  Z[-k] through the
        // group's (idle) exchange tile in natural order.
#pragma unroll
        for (int k2 = 0; k2 < 16; k2++) ex[t + 16 * k2] = v[k2];
    }
    __syncwarp();
    if (gg == 0) {
#pragma unroll
        for (int k2 = 0; k2 < 16; k2++) {
            const int k = t + 16 * k2;
            const double2 z = v[k2], zm = ex[(L - k) & (L - 1)];
            const double2 x0 = make_double2(0.5 * (z.x + zm.x), 0.5 * (z.y - zm.y));
            const double2 xn = make_double2(0.5 * (z.y + zm.y), -0.5 * (z.x - zm.x));
            const double g2 = s_gs2[k];
            v[k2] = make_double2(gs[k2] * x0.x - g2 * xn.y, gs[k2] * x0.y + g2 * xn.x);
        }
    } else {
#pragma unroll
        for (int k2 = 0; k2 < 16; k2++) v[k2] = make_double2(v[k2].x * gs[k2], v[k2].y * gs[k2]);
    }
    __syncwarp();                                                // the tile is rewritten by the inverse transform
    fft256_group<true>(v, ex, tw, t);
    SC_STAMPC(6);
    // U[gg][j], j = t + 16 n1 < N, to the group that owns row j
#pragma unroll
    for (int n1 = 0; n1 < 8; n1++) {
        const int j = t + 16 * n1;
        const unsigned dr = (unsigned)(j >> 3);
        const int dl = j & 7;
        const uint32_t dst = mapa_shared(sa + (uint32_t)((dl * kPcGroup + kPcRow) * 16), dr);
        const uint32_t db = mapa_shared(bar0 + 8u * (4 + (dl >> 1)), dr);
        SC_ASSERT(counters, j >= 0 && j < N && dr < (unsigned)kPcCtas && (size_t)((dl * kPcGroup + kPcRow + N) * 16 + 16) <= kPcOffPhi);
        if (gg == 0) { st_async2(dst, make_double2(v[n1].x, 0.0), db); st_async2(dst + (uint32_t)N * 16u, make_double2(v[n1].y, 0.0), db); }
        else st_async2(dst + (uint32_t)gg * 16u, v[n1], db);
    }
    SC_STAMPC(7);

    // ---------------------------------------------------------------- stage C: row gg inverse
    pc_mbar_wait(bar0 + 8u * (4 + warp), 0);
    SC_STAMPC(8);
#pragma unroll
    for (int n1 = 0; n1 < 16; n1++) {
        const int k = 16 * n1 + t;
        double2 U = row[k <= N ? k : L - k];                      // Hermitian half stored: the rest is the conjugate of L - k
        if (k > N) U.y = -U.y;
        v[n1] = U;
    }
    fft256_group<true>(v, ex, tw, t);
    SC_STAMPC(9);
    // ---------------------------------------------------------------- stage D: u~ row -> shared memory (+ halo rows of the neighbour CTAs), fields
    double* const prow = s_phi + (lg + 1) * N;
#pragma unroll
    for (int k2 = 0; k2 < 8; k2++) prow[t + 16 * k2] = v[k2].x;
    if (lg == 0 && rank > 0) {                                   // my first row is the row above the previous CTA's last
        const uint32_t dst = mapa_shared(sa + (uint32_t)(kPcOffPhi + (size_t)(kPcGroups + 1) * N * 8), rank - 1), db = mapa_shared(bar0 + 64u, rank - 1);
#pragma unroll
        for (int k2 = 0; k2 < 8; k2++) st_async1(dst + (uint32_t)(t + 16 * k2) * 8u, v[k2].x, db);
    }
    if (lg == kPcGroups - 1 && rank + 1 < kPcCtas) {             // my last row is the row below the next CTA's first
        const uint32_t dst = mapa_shared(sa + (uint32_t)kPcOffPhi, rank + 1), db = mapa_shared(bar0 + 64u, rank + 1);
#pragma unroll
        for (int k2 = 0; k2 < 8; k2++) st_async1(dst + (uint32_t)(t + 16 * k2) * 8u, v[k2].x, db);
    }
    __syncthreads();
    pc_mbar_wait(bar0 + 64u, 0);
    SC_STAMPC(10);
    {
        const double* const pm = prow - N;
        const double* const pp = prow + N;
        const double hx = 0.5 * g.inv_dx, hy = 0.5 * g.inv_dy;
        double exv[8], eyv[8];
        const double* const pu = gg == N - 1 ? prow : pp;         // one-sided differences on the first and last row / node
        const double* const pd = gg == 0 ? prow : pm;
        const double fy = (gg == 0 || gg == N - 1) ? g.inv_dy : hy;
#pragma unroll
        for (int k2 = 0; k2 < 8; k2++) {
            const int i = t + 16 * k2;
            const int il = i > 0 ? i - 1 : 0, ir = i < N - 1 ? i + 1 : N - 1;
            exv[k2] = -(prow[ir] - prow[il]) * ((i == 0 || i == N - 1) ? g.inv_dx : hx);
            eyv[k2] = -(pu[i] - pd[i]) * fy;
        }
        SC_STAMPC(12);
#pragma unroll
        for (int k2 = 0; k2 < 8; k2++) {
            const int i = t + 16 * k2;
            g.phi[(size_t)gg * N + i] = v[k2].x;
            g.E[(size_t)gg * N + i] = make_double2(exv[k2], eyv[k2]);
        }
    }
    SC_STAMPC(11);
}

}  // namespace sc
