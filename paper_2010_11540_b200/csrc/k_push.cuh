// k_push.cuh -- the fused per-segment particle kernel.
//
// One launch carries every particle through
//   [pending space-charge kick: bilinear gather of (Ex,Ey) + lambda(sigma) interpolation, eq. 12]
//   -> the table rows of one lattice segment (DRIFT / LINMAP / MULT / RF; section III of the paper)
//   -> [cloud-in-cell deposit, eq. 14, + lambda histogram at the SC node that ends the segment].
// Particles are SoA fp64 in HBM: 6 loads + 6 stores of 8 B per particle per launch (96 B; 64 B for
// 4D beams) is the whole algorithmic traffic.
//
// Shape (measured on B200, DESIGN.md section 5 and profiles/): at 1e6 particles a launch is ~6800 particles per SM
// and ~24 us long inside a graph (0.60 of the measured copy peak); it is bound by memory LATENCY (a chain of particle
// load -> field gather -> maps -> shared atomics per warp, the warps marching in lockstep), not by issue slots, fp64
// or bandwidth -- removing the segment's maps altogether saves 1.3 us.  Hence:
//  * one CTA of 32 warps per SM (the most the register file gives at 64 registers per thread), 2 particles per
//    lane per piece (16-byte loads and stores, 512 contiguous bytes per warp instruction), pieces of 64 particles
//    handed out from a CTA-wide queue so that the warps finish together;
//  * particles go HBM/L2 -> registers directly with L1::no_allocate loads.  A shared-memory staging pipeline
//    (TMA bulk copies + mbarriers, first with a producer warp, then one buffer per warp) was built, parity-green
//    and measured slower (36.3 vs 33.2 us): its 96 KB of buffers shrink the L1 to 28 KB, and the field gather,
//    which hits a ~120 KB L1 90 % of the time, then pays L2 latency on most accesses.
//  Tried and dropped, each measured: 4 particles per lane (fewer instructions, too few warps), per-warp equal
//  slices (+4 us), register prefetch of the next piece (spills), L1 warm-up of the field table (0), a 4x larger
//  per-cell field table read with 32-byte loads (L1 hit rate collapses, +5 us), cp.async prefetch of x, y into shared
//  slots (0), an interpreter fetching one op ahead (+0.6 us), rotated flush start per CTA (0).  Kept: a 1500-cycle
//  start-up stagger between four warp groups (-2 us).
// The segment's rows arrive PRE-DECODED by the host as 16-byte slots (sc_track.cu: encode_piece) inside the
// kernel parameters, i.e. in the constant bank; "drift + thin multipole" pairs are fused into one slot pair.
//
// Deposit (PAPER.md:175-200 uses block-private sub-histograms + atomics; so do we, but):
//   mode 1 (deterministic): int64 fixed point, each 64-bit cell updated with NATIVE 32-bit shared
//     atomics -- low word ATOMS.ADD returning the old value, carry folded into the high-word add --
//     because 64-bit shared atomics (integer or double) compile to a CAS loop on sm_100a;
//   mode 0 (eq. 14's double weights, summed in no particular order): 64-bit shared atomics being CAS loops, the CTA-private
//     grid accumulates the weights as integers too -- w 2^e rounded to nearest, e = 62 - ceil(log2(particles per CTA)) <= 52, so
//     that no cell can overflow; each deposit is then off by at most 2^-(e+1) (1e-15 at 1e6 particles, far inside the 1e-10
//     the summation order already costs) and the CTA's sum is exact -- and the flush adds the CTA's cell values to the global
//     double accumulators with the L2's native fp64 atomics, as particles outside the window do directly.
//   Grids larger than shared memory keep a centred window in shared memory; particles outside the
//   window go straight to the global grid with L2 atomics (RED.ADD.64 / RED.ADD.F64).
#pragma once
#include "sc_device.cuh"

#ifndef SC_SWIZZLE
#define SC_SWIZZLE 1       // A/B switch: 0 stores (low, high) in every cell of the private grid (low words on the 16 even banks only)
#endif
#ifndef SC_BULK_FLUSH
#define SC_BULK_FLUSH 0    // A/B switch: 1 flushes the private grid with TMA bulk reductions (cp.reduce.async.bulk .add.u64/.f64, SASS UBLKRED)
                           // instead of one RED per non-zero cell: measured 0.76 us per launch SLOWER at cfg3
#endif
#ifndef SC_F64_INT
#define SC_F64_INT 1       // A/B switch: 0 accumulates the fp64 deposit mode's private grid with shared-memory atomicAdd(double), a CAS loop on sm_100a
#endif
#if SC_BULK_FLUSH && SC_F64_INT
#error "SC_BULK_FLUSH adds the private grid's words as they are: build it with -DSC_F64_INT=0"
#endif
#ifndef SC_SKEW_NS
#define SC_SKEW_NS 750     // start-up stagger between the CTA's four warp groups, in units of 2 SM cycles; see k_push
#endif

namespace sc {

#ifdef SC_TRACE
#define SC_STAMPP(k_) do { if (threadIdx.x == 0) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); a.counters[8 + 512 + blockIdx.x * 8 + (k_)] = t_; } } while (0)
#else
#define SC_STAMPP(k_) do { } while (0)
#endif

// streaming 16-byte load: every particle coordinate is read once per launch, keep it out of L1
__device__ __forceinline__ double2 ld_stream2(const double* p) {
    double2 v;
    asm volatile("ld.global.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p) : "memory");
    return v;
}

// ---- mbarrier + TMA bulk copy (global -> shared), used to stage the field window of the EW instantiations
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
    asm volatile(
        "{\n.reg .pred p;\nWAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\nbra WAIT_%=;\nDONE_%=:\n}" ::"r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src, unsigned bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"((uint32_t)__cvta_generic_to_shared(dst_smem)), "l"(src), "r"(bytes), "r"((uint32_t)__cvta_generic_to_shared(bar)) : "memory");
}

// the same with 32-bit shared-window addresses (one register each; the staging path keeps them live across the piece loop)
__device__ __forceinline__ void mbar_expect_tx_sa(uint32_t bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait_sa(uint32_t bar, unsigned parity) {
    asm volatile(
        "{\n.reg .pred p;\nWAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\nbra WAIT_%=;\nDONE_%=:\n}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s_sa(uint32_t dst, const void* src, unsigned bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ double2 lds2_sa(uint32_t addr) {
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr) : "memory");
    return v;
}

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

// swizzled word index of the LOW 32-bit word of 64-bit cell c of the CTA-private grid; the high word is at idx ^ 1.
// Cells c and c + 16 share a bank pair; bit 4 of c decides which of the pair holds the low word, so the low-word
// atomics of a warp (random cells) spread over all 32 banks instead of the 16 even ones.
__device__ __forceinline__ int lo_word(int c) { return SC_SWIZZLE ? ((c << 1) | ((c >> 4) & 1)) : (c << 1); }

// EW ("field window"): the kick's node fields (E~x, E~y) of a window of the grid, and the lambda pair table, are staged in
// SHARED memory by TMA bulk copies at the start of the launch and gathered from there (4 LDS.128 per particle, a few
// wavefronts per warp instruction) instead of from the L1 (one tag look-up per lane: 32 wavefronts per warp
// instruction; ncu had the L1TEX pipe as the busiest unit of the round-1 kernel).  Window of the deposit and window of
// the fields are the same nodes, 24 bytes of shared memory per node: the whole grid up to ~96 x 96, a centred 96 x 96
// window of a 128 x 128 grid; particles outside it gather through the L1 and deposit with L2 atomics as before.
// EW = 2 ("staged") adds a per-warp shared-memory buffer into which every warp's NEXT piece of particles is prefetched by TMA bulk
// copies while the current piece is computed (affordable there: the gather no longer needs the L1).  Measured: 8 % faster when the
// particles stream from HBM (1e7: 212 vs 231 us per launch), 7 % SLOWER when they sit in L2 (1e6: 25.4 vs 23.8 us; the extra
// shared-memory traffic costs more than the hidden latency is worth), so the host picks it by the size of the particle set.
template <bool SIXD, int DEP, bool CQ = false, int EW = 0>   // DEP: 0 none, 1 fp64, 2 fixed; CQ ("heavy"): the piece holds a CQUAD, XDRIFT or SBEND row, or the kick
                                                 // interpolates the potential bicubically (eqs. 28-29): their sincos/exp/sqrt/asin and 16-load
                                                 // code costs registers; the plain instantiation is kept free of it and the heavy one runs
                                                 // 16 warps of up to 128 registers instead of 32 of 64
__global__ void __launch_bounds__(CQ ? kPushThreadsCQ : kPushThreads, 1) k_push(const __grid_constant__ PushArgs a) {
    constexpr int NT = CQ ? kPushThreadsCQ : kPushThreads, NW = NT / 32;
    extern __shared__ __align__(128) unsigned char smem_push[];
    if (a.noop) { pdl_wait(); return; }               // measurement: launch floor of the turn's graph
    SC_STAMPP(0);
    // No early trigger of the dependent launch here.  With the three-launch solvers their many small CTAs and the next k_push's
    // large ones compete for the draining SMs (round 1: 14.0 vs 8.55 ms per turn).  With the one-cluster solver it was tried
    // again (round 2): the 16-CTA cluster is not placed before this grid has drained anyway (it needs 16 free SMs of one GPC at
    // once: global-timer stamps show it starting after the last flush either way) and then spends 1.0 us in griddepcontrol.wait
    // that a launch after completion does not: 29.50 vs 29.39 us per node.
    // layout: [lambda histogram][work-queue counter, min row, max row][mbarrier][pad to 128][deposit window]
    //         [EW: field window (double2 per node)][EW: lambda pair table]
    const int nh = (DEP && SIXD) ? a.dg.nbins : 0;
    const bool use_lam = SIXD && a.do_kick && a.kg.nbins > 0;
    unsigned int* const s_hist = reinterpret_cast<unsigned int*>(smem_push);
    const uint32_t bar_off = (4u * (uint32_t)nh + 12u + 7u) & ~7u;
    uint64_t* const s_bar = reinterpret_cast<uint64_t*>(smem_push + bar_off);
    const uint32_t head = (bar_off + 8u + 127u) & ~127u;
    unsigned long long* const s_grid = reinterpret_cast<unsigned long long*>(smem_push + head);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wcells = DEP ? a.dg.wnx * a.dg.wny : 0;
    const int ewnx = EW ? a.kg.wnx : 0, ewcells = (EW && a.do_kick) ? a.kg.wnx * a.kg.wny : 0;
    double2* const s_E = reinterpret_cast<double2*>(s_grid + wcells);
    double2* const s_lam = s_E + ewcells;
    bool e_ready = !(EW && a.do_kick);
    // EW + SC_STAGE: [per-warp particle buffers: 6 coordinates x 64 doubles][per-warp mbarriers] behind the lambda table
    constexpr bool STAGE = EW == 2;
    constexpr int NCO = SIXD ? 6 : 4;
    const uint32_t st_area = ((uint32_t)__cvta_generic_to_shared(s_lam + ((EW && a.do_kick && use_lam) ? a.kg.nbins + 1 : 0)) + 127u) & ~127u;
    const uint32_t st = st_area + (uint32_t)warp * (6u * kChunk * 8u);                 // this warp's buffer (shared-window address)
#define SC_WBAR (st_area + (uint32_t)NW * (6u * kChunk * 8u) + (uint32_t)(threadIdx.x >> 5) * 8u)   // this warp's mbarrier

    // ---- this CTA's particle range [p_lo, p_hi) (an even number of particles per CTA: 16-byte accesses)
    const long long p_lo = (long long)blockIdx.x * a.per_cta;
    const long long p_hi = p_lo + a.per_cta < a.n ? p_lo + a.per_cta : a.n;
    const int len = p_hi > p_lo ? (int)(p_hi - p_lo) : 0;
    // Work is handed out from a CTA-wide queue (one shared counter, in particles): a warp takes its next piece of
    // 64 particles when it is done with the last one, so the warps finish together whatever the piece count
    // (a launch is only ~3 pieces per warp long).  No early trigger of the dependent kernel here: letting the
    // Poisson CTAs in before this grid has drained was measured to cost 60 %.
    int* const s_next = reinterpret_cast<int*>(smem_push + 4 * nh);
    if (tid == 0) { s_next[0] = 0; s_next[1] = 0x7fffffff; s_next[2] = -1; }   // queue head; min / max deposited window row
    if (EW && tid == 0) mbar_init(s_bar, 1);
    if (STAGE && lane == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(SC_WBAR) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }

    // zero the private grid and histogram: own shared memory, legal before the predecessor grid has finished
    for (int b = tid; b < nh; b += NT) s_hist[b] = 0u;
    if (DEP) {
        ulonglong2* g2 = reinterpret_cast<ulonglong2*>(s_grid);
        const int n2 = wcells >> 1;
        for (int c = tid; c < n2; c += NT) g2[c] = make_ulonglong2(0ull, 0ull);
        if (tid == 0 && (wcells & 1)) s_grid[wcells - 1] = 0ull;
    }
    SC_STAMPP(1);
    pdl_wait();                                       // fields, lambda, particles of the previous kernels are final
    SC_STAMPP(2);
    __syncthreads();
    if (EW && a.do_kick) {
        // field window: one TMA bulk copy per window row, and one for the lambda pair table; completion is counted in bytes
        // on the mbarrier.  The first piece's particle loads go out before anybody waits for these.
        const int wny = a.kg.wny;
        const unsigned lam_bytes = use_lam ? (unsigned)(a.kg.nbins + 1) * 16u : 0u;
        if (tid == 0) mbar_expect_tx(s_bar, (unsigned)(ewcells * 16) + lam_bytes);
        for (int r = tid; r < wny; r += NT)
            bulk_g2s(s_E + (size_t)r * ewnx, a.kg.E + (size_t)(a.kg.wj0 + r) * a.kg.nx + a.kg.wi0, (unsigned)(ewnx * 16), s_bar);
        if (use_lam && tid == NT - 1) bulk_g2s(s_lam, a.kg.lam, lam_bytes, s_bar);
    }

    // Per-warp clock stamps (profiles/r01c_k_push_timeline.md) show all 32 warps of all 148 CTAs marching in lockstep:
    // load (L2 burst, ~1.2 us) -> kick (~1.8 us) -> maps (fp64 pipe, ~1.7 us) -> store -> deposit, each phase using one
    // resource while the others idle.  Four warp groups (two warps per scheduler each) start 1500 cycles apart so
    // that their phases interleave; the work queue evens out the pieces.  Measured: 33.1 -> 30.7 us per launch at 1e6.
#if SC_SKEW_NS > 0
    if (len >= 2 * kChunk * NW) {   // only when every warp has pieces to interleave; busy-wait on the SM clock
                                            // (nanosleep was seen to cap at ~0.5 us whatever it is asked for)
        const long long t_go = clock64() + (long long)((warp >> 2) & 3) * (SC_SKEW_NS * 2);
        while (clock64() < t_go) { }
    }
#endif
    unsigned int n_out = 0;
    auto grab = [&]() {                               // next piece of the CTA's queue (offset in particles)
        int o = 0;
        if (lane == 0) o = atomicAdd(s_next, kChunk);
        return __shfl_sync(0xffffffffu, o, 0);
    };
    auto prefetch = [&](int off_) {                   // STAGE: this warp's piece at off_ -> its shared buffer, one bulk copy per coordinate
        if (off_ < len) {
            const int c_ = len - off_ < kChunk ? len - off_ : kChunk;
            const unsigned bytes = (unsigned)(((c_ + 1) & ~1) * 8);       // odd count: the pair's second slot is the allocation's padding
            if (lane == 0) mbar_expect_tx_sa(SC_WBAR, bytes * NCO);
            __syncwarp();
            if (lane < NCO) bulk_g2s_sa(st + (uint32_t)lane * (kChunk * 8u), a.q[lane] + p_lo + off_, bytes, SC_WBAR);
        }
    };
    int nxt = 0;
    unsigned ph = 0;
    if (STAGE) { nxt = grab(); prefetch(nxt); }
    for (;;) {
        const int off = STAGE ? nxt : grab();
        if (off >= len) break;
        const int cnt = len - off < kChunk ? len - off : kChunk;
        const long long base = p_lo + off;
        SC_ASSERT(a.counters, off >= 0 && (off & 1) == 0 && base + cnt <= a.n && cnt > 0);
        // ---- piece -> registers straight from HBM/L2 (16-byte loads, 512 contiguous bytes per warp instruction, not
        //      allocated in L1: the L1 is left to the field gather); lane l holds the pairs (64h + 2l, 64h + 2l + 1)
        double x[kPP], px[kPP], y[kPP], py[kPP], sg[kPP], ps[kPP];
#pragma unroll
        for (int h = 0; h < kPP / 2; h++) {
            const int i0 = h * 64 + 2 * lane;
            double2 t0 = make_double2(0.0, 0.0), t1 = t0, t2 = t0, t3 = t0, t4 = t0, t5 = t0;
            if (STAGE) {
                if (h == 0) { mbar_wait_sa(SC_WBAR, ph); ph ^= 1u; }   // this piece has landed in the warp's buffer
                if (i0 < cnt) {
                    const uint32_t sb = st + (uint32_t)(h * 32 + lane) * 16u;       // coordinate q at + q * 64 doubles
                    t0 = lds2_sa(sb); t2 = lds2_sa(sb + 2u * kChunk * 8u); t1 = lds2_sa(sb + kChunk * 8u); t3 = lds2_sa(sb + 3u * kChunk * 8u);
                    if (SIXD) { t4 = lds2_sa(sb + 4u * kChunk * 8u); t5 = lds2_sa(sb + 5u * kChunk * 8u); }
                }
            } else if (i0 < cnt) {                     // cnt odd: the pair's second slot is the allocation's padding
                t0 = ld_stream2(a.q[0] + base + i0); t2 = ld_stream2(a.q[2] + base + i0);
                if (SIXD) t4 = ld_stream2(a.q[4] + base + i0);
                t1 = ld_stream2(a.q[1] + base + i0); t3 = ld_stream2(a.q[3] + base + i0);
                if (SIXD) t5 = ld_stream2(a.q[5] + base + i0);
            }
            x[2 * h] = t0.x; x[2 * h + 1] = t0.y; px[2 * h] = t1.x; px[2 * h + 1] = t1.y;
            y[2 * h] = t2.x; y[2 * h + 1] = t2.y; py[2 * h] = t3.x; py[2 * h + 1] = t3.y;
            sg[2 * h] = t4.x; sg[2 * h + 1] = t4.y; ps[2 * h] = t5.x; ps[2 * h + 1] = t5.y;
        }
        if (cnt & 1) {                                // odd tail: the padding slot carries zeros (never stored, never deposited)
#pragma unroll
            for (int k = 0; k < kPP; k++)
                if ((k >> 1) * 64 + 2 * lane + (k & 1) >= cnt) { x[k] = px[k] = y[k] = py[k] = sg[k] = ps[k] = 0.0; }
        }

        // ---- pending space-charge kick (eq. 12): px += kappa L lambda(sigma) E~x(x,y)
        if (EW && !e_ready) { mbar_wait(s_bar, 0); e_ready = true; SC_STAMPP(5); }   // field window and lambda table staged
        if (CQ && a.do_kick && a.kg.interp) {
            // N4, eqs. 28-29: bicubic surface of the POTENTIAL on the 4x4 stencil around the particle's
            // cell -- the uniform cubic B-spline with the node values as de Boor points (reading A9) -- and its analytic
            // gradient; stencil nodes beyond the grid edge are linear extrapolations
#pragma unroll
            for (int k = 0; k < kPP; k++) {
                int i, j; double t, u;
                const bool in = locate(a.kg, x[k], y[k], i, j, t, u);
                if (!in) { i = 0; j = 0; }
                const int nx = a.kg.nx, ny = a.kg.ny;
                const double t2 = t * t, t3 = t2 * t, u2 = u * u, u3 = u2 * u, mt = 1.0 - t, mu = 1.0 - u;
                const double s6 = 1.0 / 6.0;
                const double bx[4] = { mt * mt * mt * s6, (3.0 * t3 - 6.0 * t2 + 4.0) * s6, (-3.0 * t3 + 3.0 * t2 + 3.0 * t + 1.0) * s6, t3 * s6 };
                const double gx[4] = { -0.5 * mt * mt, 1.5 * t2 - 2.0 * t, -1.5 * t2 + t + 0.5, 0.5 * t2 };
                const double by[4] = { mu * mu * mu * s6, (3.0 * u3 - 6.0 * u2 + 4.0) * s6, (-3.0 * u3 + 3.0 * u2 + 3.0 * u + 1.0) * s6, u3 * s6 };
                const double gy[4] = { -0.5 * mu * mu, 1.5 * u2 - 2.0 * u, -1.5 * u2 + u + 0.5, 0.5 * u2 };
                const int i0 = i > 0 ? i - 1 : 0, i3 = i + 2 < nx ? i + 2 : nx - 1;
                double rv[4], rd[4];
#pragma unroll
                for (int c = 0; c < 4; c++) {
                    int jj = j + c - 1;
                    jj = jj < 0 ? 0 : (jj > ny - 1 ? ny - 1 : jj);
                    const double* row = a.kg.phi + (size_t)jj * nx;
                    double U0 = __ldg(row + i0), U1 = __ldg(row + i), U2 = __ldg(row + i + 1), U3 = __ldg(row + i3);
                    if (i == 0) U0 = 2.0 * U1 - U2;
                    if (i + 2 > nx - 1) U3 = 2.0 * U2 - U1;
                    rv[c] = bx[0] * U0 + bx[1] * U1 + bx[2] * U2 + bx[3] * U3;
                    rd[c] = gx[0] * U0 + gx[1] * U1 + gx[2] * U2 + gx[3] * U3;
                }
                if (j == 0) { rv[0] = 2.0 * rv[1] - rv[2]; rd[0] = 2.0 * rd[1] - rd[2]; }
                if (j + 2 > ny - 1) { rv[3] = 2.0 * rv[2] - rv[1]; rd[3] = 2.0 * rd[2] - rd[1]; }
                const double uu = by[0] * rv[0] + by[1] * rv[1] + by[2] * rv[2] + by[3] * rv[3];
                const double ex = -(by[0] * rd[0] + by[1] * rd[1] + by[2] * rd[2] + by[3] * rd[3]) * a.kg.inv_dx;
                const double ey = -(gy[0] * rv[0] + gy[1] * rv[1] + gy[2] * rv[2] + gy[3] * rv[3]) * a.kg.inv_dy;
                double lam = a.lam_const, dlam = 0.0;
                if (use_lam) {
                    const double tt = __dmul_rn(__dsub_rn(sg[k], a.kg.smin), a.kg.inv_ds);
                    const double uq = tt + 0.5;
                    const int ib = __double2int_rz(uq);
                    const bool inb = tt >= 0.0 && tt < a.kg.dnbins;
                    const double f = uq - (double)ib;
                    const double2 l = __ldg(a.kg.lam + (inb ? ib : 0));
                    lam = inb ? (1.0 - f) * l.x + f * l.y : 0.0;
                    dlam = inb ? (l.y - l.x) * a.kg.inv_ds : 0.0;
                }
                const double kk = a.kick_scale * lam;
                if (in) { px[k] += kk * ex; py[k] += kk * ey; }
                if (SIXD && a.kg.long_kick && in) ps[k] -= a.kick_scale * uu * dlam;
            }
        } else
        if (a.do_kick) {
#pragma unroll
            for (int k = 0; k < kPP; k++) {
                int i, j; double fx, fy;
                const bool in = locate(a.kg, x[k], y[k], i, j, fx, fy);
                double2 e00, e10, e01, e11;
                const int li = i - a.kg.wi0, lj = j - a.kg.wj0;
                if (EW && in && (unsigned)li < (unsigned)(a.kg.wnx - 1) && (unsigned)lj < (unsigned)(a.kg.wny - 1)) {
                    SC_ASSERT(a.counters, lj * ewnx + li + ewnx + 1 < ewcells);
                    const double2* sp = s_E + lj * ewnx + li;
                    e00 = sp[0]; e10 = sp[1]; e01 = sp[ewnx]; e11 = sp[ewnx + 1];
                } else {
                    SC_ASSERT(a.counters, !in || (i >= 0 && j >= 0 && (j + 1) * a.kg.nx + i + 1 < a.kg.nx * a.kg.ny));
                    const double2* ep = a.kg.E + (in ? j * a.kg.nx + i : 0);
                    // the four node fields are in flight while lambda is interpolated
                    e00 = __ldg(ep); e10 = __ldg(ep + 1); e01 = __ldg(ep + a.kg.nx); e11 = __ldg(ep + a.kg.nx + 1);
                }
                double lam = a.lam_const, dlam = 0.0;
                if (use_lam) {
                    const double tt = __dmul_rn(__dsub_rn(sg[k], a.kg.smin), a.kg.inv_ds);
                    // pair table: entry m holds (lambda_{m-1}, lambda_m); u = t + 0.5 puts the bin centres on the integers
                    const double u = tt + 0.5;
                    const int ib = __double2int_rz(u);
                    const bool inb = tt >= 0.0 && tt < a.kg.dnbins;
                    const double f = u - (double)ib;
                    SC_ASSERT(a.counters, !inb || (ib >= 0 && ib <= a.kg.nbins));
                    const double2 l = EW ? s_lam[inb ? ib : 0] : __ldg(a.kg.lam + (inb ? ib : 0));
                    lam = inb ? (1.0 - f) * l.x + f * l.y : 0.0;
                    dlam = inb ? (l.y - l.x) * a.kg.inv_ds : 0.0;     // slope of the piecewise-linear lambda (eq. 13)
                }
                const double gx = 1.0 - fx, gy = 1.0 - fy;
                const double w00 = gx * gy, w10 = fx * gy, w01 = gx * fy, w11 = fx * fy;
                const double ex = w00 * e00.x + w10 * e10.x + w01 * e01.x + w11 * e11.x;
                const double ey = w00 * e00.y + w10 * e10.y + w01 * e01.y + w11 * e11.y;
                const double kk = a.kick_scale * lam;
                if (in) { px[k] += kk * ex; py[k] += kk * ey; }
                if (SIXD && a.kg.long_kick) {
                    // eq. 13: psigma -= kappa L u~(x,y) lambda'(sigma), u~ bilinear with the same weights; both kicks are
                    // taken at the pre-kick (x, y, sigma)
                    const double* up = a.kg.phi + (in ? j * a.kg.nx + i : 0);
                    const double u00 = __ldg(up), u10 = __ldg(up + 1), u01 = __ldg(up + a.kg.nx), u11 = __ldg(up + a.kg.nx + 1);
                    const double uu = w00 * u00 + w10 * u10 + w01 * u01 + w11 * u11;
                    if (in) ps[k] -= a.kick_scale * uu * dlam;
                }
            }
        }

        // ---- single-particle maps of this segment, in table order (pre-decoded slots, constant bank)
        double dd[kPP], pg[kPP];                            // change only at an RF row
#pragma unroll
        for (int k = 0; k < kPP; k++) { dd[k] = 1.0 - ps[k]; pg[k] = ps[k] * a.inv_gamma2; }
#define SC_EACH _Pragma("unroll") for (int k = 0; k < kPP; k++)
#define SC_DRIFT_BODY(L)                                                              \
        SC_EACH {                                                                     \
            const double tl_ = (L) * dd[k];                                           \
            if (SIXD) sg[k] += (L) * (pg[k] - 0.5 * (px[k] * px[k] + py[k] * py[k])); \
            x[k] += tl_ * px[k];                                                      \
            y[k] += tl_ * py[k];                                                      \
        }
#define SC_M1_BODY(K) SC_EACH { px[k] -= (K) * x[k]; py[k] += (K) * y[k]; }
#define SC_M2_BODY(K) SC_EACH { px[k] -= (K) * (0.5 * (x[k] * x[k] - y[k] * y[k])); py[k] += (K) * (x[k] * y[k]); }
#define SC_M3_BODY(K)                                                                 \
        SC_EACH {                                                                     \
            const double xx_ = x[k] * x[k], yy_ = y[k] * y[k];                        \
            px[k] -= (K) * (x[k] * (xx_ - 3.0 * yy_) * (1.0 / 6.0));                  \
            py[k] += (K) * (y[k] * (3.0 * xx_ - yy_) * (1.0 / 6.0));                  \
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
                else SC_EACH { px[k] -= kq.x; py[k] += kq.y; }
            } else if (op == OP_DRIFT) {
                pc += 1;
                SC_DRIFT_BODY(v)
            } else if (op <= OP_M3) {
                if (op == OP_M2) { pc += 1; SC_M2_BODY(v) }
                else if (op == OP_M3) { pc += 1; SC_M3_BODY(v) }
                else if (op == OP_M1) { pc += 1; SC_M1_BODY(v) }
                else { const double k0s = a.prog[pc + 1].x; pc += 2; SC_EACH { px[k] -= v; py[k] += k0s; } }
            } else if (op == OP_LINMAP) {
                const double2 m0 = a.prog[pc + 1], m1 = a.prog[pc + 2], m2 = a.prog[pc + 3], m3 = a.prog[pc + 4];
                pc += 5;
                SC_EACH {
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
                pc += 2;
                SC_EACH {
                    double zr = x[k], zi = y[k];           // n >= 1
                    for (int m = 2; m <= n; m++) {
                        const double inv = 1.0 / (double)m;
                        const double nr = (zr * x[k] - zi * y[k]) * inv;
                        zi = (zr * y[k] + zi * x[k]) * inv;
                        zr = nr;
                    }
                    px[k] -= v * zr - ks * zi;
                    py[k] += v * zi + ks * zr;
                }
            } else if (CQ && op == OP_CQUAD) {
                // eq. 6 as printed, per particle: strength k1 (1 - psigma); v = k1
                const double L = a.prog[pc + 1].x;
                pc += 2;
                const double ak = fabs(v);
                const bool fx_ = v > 0.0;                  // k1 > 0 focuses x
                SC_EACH {
                    const double w = sqrt(ak * dd[k]);
                    double s_, c_;
                    sincos(w * L, &s_, &c_);
                    const double ep = exp(w * L), em = 1.0 / ep;
                    const double ch = 0.5 * (ep + em), sh = 0.5 * (ep - em);
                    const double ca = sqrt(dd[k] / ak), cb = sqrt(ak / dd[k]);
                    const double f0 = fx_ ? x[k] : y[k], pf0 = fx_ ? px[k] : py[k];
                    const double g0 = fx_ ? y[k] : x[k], pg0 = fx_ ? py[k] : px[k];
                    const double f1 = f0 * c_ + ca * pf0 * s_, pf1 = pf0 * c_ - cb * f0 * s_;
                    const double g1 = g0 * ch + ca * pg0 * sh, pg1 = pg0 * ch + cb * g0 * sh;
                    if (SIXD) {
                        const double rf = f0 * ak / w, rg = g0 * ak / w;
                        const double If = 0.5 * L * (pf0 * pf0 + rf * rf) + (pf0 * pf0 - rf * rf) * s_ * c_ / (2.0 * w) - pf0 * rf * s_ * s_ / w;
                        const double Ig = 0.5 * L * (pg0 * pg0 - rg * rg) + (pg0 * pg0 + rg * rg) * sh * ch / (2.0 * w) + pg0 * rg * sh * sh / w;
                        sg[k] += L * pg[k] - 0.5 * (If + Ig);
                    }
                    x[k] = fx_ ? f1 : g1; px[k] = fx_ ? pf1 : pg1;
                    y[k] = fx_ ? g1 : f1; py[k] = fx_ ? pg1 : pf1;
                }
            } else if (CQ && op == OP_XDRIFT) {
                // exact drift: straight line with eq. 3's longitudinal momentum (PAPER.md:53-95 at B = 0); v = L
                pc += 1;
                SC_EACH {
                    const double pz = sqrt(1.0 + 2.0 * ps[k] + a.beta0_2 * ps[k] * ps[k] - px[k] * px[k] - py[k] * py[k]);
                    const double lz = v / pz;
                    x[k] += lz * px[k];
                    y[k] += lz * py[k];
                    if (SIXD) sg[k] += v - lz * (1.0 + a.beta0_2 * ps[k]);
                }
            } else if (CQ && op == OP_SBEND) {
                // exact sector bend: the particle's circle cut by the exit plane; v = L, lengths in rho
                const double hh = a.prog[pc + 1].x;
                const double2 sc_ = a.prog[pc + 2];        // sin(L h), cos(L h)
                pc += 3;
                const double rho = 1.0 / hh, th = v * hh;
                SC_EACH {
                    const double pz = sqrt(1.0 + 2.0 * ps[k] + a.beta0_2 * ps[k] * ps[k] - px[k] * px[k] - py[k] * py[k]);
                    const double R = sqrt(px[k] * px[k] + pz * pz);
                    const double cx = 1.0 + hh * x[k] - pz, cz = px[k];
                    const double D = cx * sc_.x - cz * sc_.y;
                    const double phi = th + asin(D / R) + atan2(px[k], pz);
                    x[k] = rho * (cx * sc_.y + cz * sc_.x + sqrt(R * R - D * D) - 1.0);
                    px[k] = -D;
                    y[k] += py[k] * rho * phi;
                    if (SIXD) sg[k] += v - rho * phi * (1.0 + a.beta0_2 * ps[k]);
                }
            } else if (op == OP_RF) {
                const double2 kp = a.prog[pc + 1];         // 2 pi h/C, phi0;  v = q V/(beta0^2 E0)
                pc += 2;
                if (SIXD) {
                    SC_EACH {
                        ps[k] -= v * sin(kp.x * sg[k] + kp.y);
                        dd[k] = 1.0 - ps[k];
                        pg[k] = ps[k] * a.inv_gamma2;
                    }
                }
            } else {
                break;                                     // OP_END
            }
        }
#undef SC_DRIFT_BODY
#undef SC_M1_BODY
#undef SC_M2_BODY
#undef SC_M3_BODY

        // ---- results straight to HBM: 16 bytes per lane and coordinate, coalesced (512 B per warp store); psigma only when a
        //      row of this launch can change it (an RF row, the longitudinal kick): 88 instead of 96 bytes per particle otherwise
        {
#pragma unroll
            for (int hh = 0; hh < kPP / 2; hh++) {
                const int i0 = hh * 64 + 2 * lane;
                if (i0 + 1 < cnt) {
#define SC_ST2(q_, v) reinterpret_cast<double2*>(a.q[q_] + base)[hh * 32 + lane] = make_double2(v[2 * hh], v[2 * hh + 1]);
                    SC_ST2(0, x) SC_ST2(1, px) SC_ST2(2, y) SC_ST2(3, py)
                    if (SIXD) { SC_ST2(4, sg) if (a.ps_changes) { SC_ST2(5, ps) } }
#undef SC_ST2
                } else if (i0 < cnt) {
                    a.q[0][base + i0] = x[2 * hh]; a.q[1][base + i0] = px[2 * hh];
                    a.q[2][base + i0] = y[2 * hh]; a.q[3][base + i0] = py[2 * hh];
                    if (SIXD) { a.q[4][base + i0] = sg[2 * hh]; if (a.ps_changes) a.q[5][base + i0] = ps[2 * hh]; }
                }
            }
        }
        if (STAGE) {
            // every coordinate register has been consumed by the stores above, so the warp's shared-memory reads of the
            // buffer have completed: refill it with the next piece while this one is deposited
            nxt = grab();
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            prefetch(nxt);
        }
        // ---- deposit at the SC node that ends this segment (eq. 14) + lambda histogram
        if (DEP == 2 || (DEP == 1 && SC_F64_INT)) {
            // integer accumulation (fixed point; and the fp64 mode's private grid, see the file header).  Branch-free over the
            // lane's particles so that the shared atomics of all of them are in flight together: first every low-word add
            // (returning), then every high-word add with its carry.
            int cw[kPP];                                   // swizzled word index of the home cell's low word (lo_word)
            unsigned long long w[kPP][4];
            const unsigned int S = 1u << a.dg.bits;
            const int wnx = a.dg.wnx;
            unsigned int* const words = reinterpret_cast<unsigned int*>(s_grid);
#pragma unroll
            for (int k = 0; k < kPP; k++) {
                const bool valid = (k >> 1) * 64 + 2 * lane + (k & 1) < cnt;
                int i, j; double fx, fy;
                const bool in = locate(a.dg, x[k], y[k], i, j, fx, fy) && valid;
                const int li = i - a.dg.wi0, lj = j - a.dg.wj0;
                const bool inw = (unsigned)li < (unsigned)(a.dg.wnx - 1) && (unsigned)lj < (unsigned)(a.dg.wny - 1);
                // ax, ay in [0, 2^s], s <= 20: 32 x 32 -> 64-bit products
                const unsigned int ax = (unsigned int)__double2int_rn(__dmul_rn(fx, a.dg.fixed_scale));
                const unsigned int ay = (unsigned int)__double2int_rn(__dmul_rn(fy, a.dg.fixed_scale));
                const unsigned int bx = S - ax, by = S - ay;
                const bool sm = in && inw;
                double d00 = 0.0, d10 = 0.0, d01 = 0.0, d11 = 0.0;
                if (DEP == 1) {                            // eq. 14's weights as doubles, then as integers of 2^-e
                    const double gx = __dsub_rn(1.0, fx), gy = __dsub_rn(1.0, fy);
                    d00 = __dmul_rn(gx, gy); d10 = __dmul_rn(fx, gy); d01 = __dmul_rn(gx, fy); d11 = __dmul_rn(fx, fy);
                    w[k][0] = sm ? (unsigned long long)__double2ll_rn(d00 * a.dep_scale) : 0ull;
                    w[k][1] = sm ? (unsigned long long)__double2ll_rn(d10 * a.dep_scale) : 0ull;
                    w[k][2] = sm ? (unsigned long long)__double2ll_rn(d01 * a.dep_scale) : 0ull;
                    w[k][3] = sm ? (unsigned long long)__double2ll_rn(d11 * a.dep_scale) : 0ull;
                } else {
                    w[k][0] = sm ? (unsigned long long)bx * by : 0ull;
                    w[k][1] = sm ? (unsigned long long)ax * by : 0ull;
                    w[k][2] = sm ? (unsigned long long)bx * ay : 0ull;
                    w[k][3] = sm ? (unsigned long long)ax * ay : 0ull;
                }
                cw[k] = sm ? lj * wnx + li : 0;            // weight 0 lands on cell 0
                SC_ASSERT(a.counters, cw[k] >= 0 && cw[k] + wnx + 1 < wcells && (DEP == 1 || !sm || (ax <= S && ay <= S)));
                SC_ASSERT(a.counters, !(in && !inw) || (i >= 0 && j >= 0 && (j + 1) * a.dg.nx + i + 1 < a.dg.nx * a.dg.ny));
                if (DEP == 1 && in && !inw) {              // outside the shared-memory window: L2 atomics on the double accumulators
                    double* cg = reinterpret_cast<double*>(a.dg.rho) + (size_t)j * a.dg.nx + i;
                    atomicAdd(cg, d00); atomicAdd(cg + 1, d10);
                    atomicAdd(cg + a.dg.nx, d01); atomicAdd(cg + a.dg.nx + 1, d11);
                }
                if (DEP == 2 && in && !inw) {              // outside the shared-memory window: L2 atomics
                    unsigned long long* cg = a.dg.rho + (size_t)j * a.dg.nx + i;
                    atomicAdd(cg, (unsigned long long)bx * by);
                    atomicAdd(cg + 1, (unsigned long long)ax * by);
                    atomicAdd(cg + a.dg.nx, (unsigned long long)bx * ay);
                    atomicAdd(cg + a.dg.nx + 1, (unsigned long long)ax * ay);
                }
                if (valid && !in) n_out++;
                if (SIXD && nh > 0 && valid) {
                    const double tt = __dmul_rn(__dsub_rn(sg[k], a.dg.smin), a.dg.inv_ds);
                    SC_ASSERT(a.counters, !(tt >= 0.0 && tt < a.dg.dnbins) || __double2int_rz(tt) < nh);
                    if (tt >= 0.0 && tt < a.dg.dnbins) atomicAdd(&s_hist[__double2int_rz(tt)], 1u);
                }
            }
            unsigned int old[kPP][4];
#pragma unroll
            for (int k = 0; k < kPP; k++) {
                old[k][0] = atomicAdd(words + lo_word(cw[k]), (unsigned int)w[k][0]);
                old[k][1] = atomicAdd(words + lo_word(cw[k] + 1), (unsigned int)w[k][1]);
                old[k][2] = atomicAdd(words + lo_word(cw[k] + wnx), (unsigned int)w[k][2]);
                old[k][3] = atomicAdd(words + lo_word(cw[k] + wnx + 1), (unsigned int)w[k][3]);
            }
#pragma unroll
            for (int k = 0; k < kPP; k++) {
                // carry out of the low word is seen by exactly one adder; weights are ~2^(2s-2), the high word is never idle
#define SC_HI(c_, off_) { const unsigned int lo_ = (unsigned int)w[k][c_];                                                   \
                          atomicAdd(words + (lo_word(cw[k] + (off_)) ^ 1), (unsigned int)(w[k][c_] >> 32) + ((old[k][c_] + lo_ < lo_) ? 1u : 0u)); }
                SC_HI(0, 0) SC_HI(1, 1) SC_HI(2, wnx) SC_HI(3, wnx + 1)
#undef SC_HI
            }
        } else if (DEP == 1) {
#pragma unroll
            for (int k = 0; k < kPP; k++) {
                if ((k >> 1) * 64 + 2 * lane + (k & 1) >= cnt) continue;
                int i, j; double fx, fy;
                if (locate(a.dg, x[k], y[k], i, j, fx, fy)) {
                    const int li = i - a.dg.wi0, lj = j - a.dg.wj0;
                    const bool inw = (unsigned)li < (unsigned)(a.dg.wnx - 1) && (unsigned)lj < (unsigned)(a.dg.wny - 1);
                    const double gx = __dsub_rn(1.0, fx), gy = __dsub_rn(1.0, fy);
                    const double w00 = __dmul_rn(gx, gy), w10 = __dmul_rn(fx, gy), w01 = __dmul_rn(gx, fy), w11 = __dmul_rn(fx, fy);
                    SC_ASSERT(a.counters, inw ? lj * a.dg.wnx + li + a.dg.wnx + 1 < wcells : (j + 1) * a.dg.nx + i + 1 < a.dg.nx * a.dg.ny);
                    if (inw) {
                        double* cs = reinterpret_cast<double*>(s_grid) + lj * a.dg.wnx + li;
                        atomicAdd(cs, w00); atomicAdd(cs + 1, w10);
                        atomicAdd(cs + a.dg.wnx, w01); atomicAdd(cs + a.dg.wnx + 1, w11);
                    } else {
                        double* cg = reinterpret_cast<double*>(a.dg.rho) + (size_t)j * a.dg.nx + i;
                        atomicAdd(cg, w00); atomicAdd(cg + 1, w10);
                        atomicAdd(cg + a.dg.nx, w01); atomicAdd(cg + a.dg.nx + 1, w11);
                    }
                } else {
                    n_out++;
                }
                if (SIXD && nh > 0) {
                    const double tt = __dmul_rn(__dsub_rn(sg[k], a.dg.smin), a.dg.inv_ds);
                    if (tt >= 0.0 && tt < a.dg.dnbins) atomicAdd(&s_hist[__double2int_rz(tt)], 1u);
                }
            }
        }
    }
#undef SC_EACH
#undef SC_WBAR

    // ---- flush the CTA-private grid and histogram into the global accumulators: one RED per non-zero cell of the rows
    //      that hold charge (~3500 per CTA at cfg3).  SC_BULK_FLUSH = 1 sends those rows as TMA bulk reductions instead
    //      (cp.reduce.async.bulk .add.u64 / .add.f64, SASS UBLKRED, the adds done by the L2): parity-green, measured slower.
    if (DEP) {
        int* const s_rows = reinterpret_cast<int*>(smem_push + 4 * nh) + 1;        // [0] first, [1] last non-zero window row
        SC_STAMPP(3);
        __syncthreads();                                                            // every warp's deposits are in
        SC_STAMPP(4);
        if (len > 0 && !SC_BULK_FLUSH) {
            // ONE pass over the private grid, a warp per row, 16 bytes (two cells) per lane: un-swizzle in registers (cells with
            // bit 4 set hold (high, low); a 16-byte pair of cells shares that bit) and one RED per non-zero cell.  (A first pass
            // that un-swizzled in place and found the rows holding charge, then a barrier, then the RED pass over those rows,
            // took 3.5 us of the launch at cfg3 by the global-timer stamps -- the two block barriers and the proxy fence between
            // the passes, not the work; this takes ~1.)
            const int wnx = a.dg.wnx;
            for (int lj = warp; lj < a.dg.wny; lj += NW) {
                const ulonglong2* row = reinterpret_cast<const ulonglong2*>(s_grid + (size_t)lj * wnx);
                unsigned long long* grow = a.dg.rho + (size_t)(a.dg.wj0 + lj) * a.dg.nx + a.dg.wi0;
                for (int q = lane; q < (wnx >> 1); q += 32) {
                    ulonglong2 v = row[q];
                    if (SC_SWIZZLE && (DEP == 2 || SC_F64_INT) && ((lj * wnx + 2 * q) & 16)) { v.x = (v.x >> 32) | (v.x << 32); v.y = (v.y >> 32) | (v.y << 32); }
                    if (DEP == 2) {
                        if (v.x) atomicAdd(grow + 2 * q, v.x);
                        if (v.y) atomicAdd(grow + 2 * q + 1, v.y);
                    } else {
                        if (v.x) atomicAdd(reinterpret_cast<double*>(grow + 2 * q), SC_F64_INT ? __ll2double_rn((long long)v.x) * a.dep_inv : __longlong_as_double((long long)v.x));
                        if (v.y) atomicAdd(reinterpret_cast<double*>(grow + 2 * q + 1), SC_F64_INT ? __ll2double_rn((long long)v.y) * a.dep_inv : __longlong_as_double((long long)v.y));
                    }
                }
            }
        }
        if (len > 0 && SC_BULK_FLUSH) {
            const int wnx = a.dg.wnx;
            // first pass: find the rows that hold charge and (fixed point) un-swizzle in place
            for (int lj = warp; lj < a.dg.wny; lj += NW) {
                ulonglong2* row = reinterpret_cast<ulonglong2*>(s_grid + (size_t)lj * wnx);
                bool nz = false;
                for (int q = lane; q < (wnx >> 1); q += 32) {
                    ulonglong2 v = row[q];
                    nz = nz || (v.x | v.y) != 0ull;
                    if (SC_SWIZZLE && DEP == 2 && ((lj * wnx + 2 * q) & 16)) {
                        v.x = (v.x >> 32) | (v.x << 32); v.y = (v.y >> 32) | (v.y << 32);
                        row[q] = v;
                    }
                }
                if (__any_sync(0xffffffffu, nz) && lane == 0) { atomicMin(&s_rows[0], lj); atomicMax(&s_rows[1], lj); }
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");          // generic-proxy writes -> visible to the bulk engine
            __syncthreads();
            const int r_lo = s_rows[0], r_hi = s_rows[1];
            if (r_hi >= r_lo) {
                const bool whole = a.dg.wnx == a.dg.nx && a.dg.wny == a.dg.ny;
                // blocks of rows: contiguous in shared AND global memory when the window is the whole grid, else one row each
                const int rows_per_op = whole ? 8 : 1;
                const int n_ops = (r_hi - r_lo + rows_per_op) / rows_per_op;
                for (int op = tid; op < n_ops; op += NT) {
                    const int r0 = r_lo + op * rows_per_op;
                    const int r1 = r0 + rows_per_op - 1 < r_hi ? r0 + rows_per_op - 1 : r_hi;
                    const uint32_t src = (uint32_t)__cvta_generic_to_shared(s_grid + (size_t)r0 * wnx);
                    unsigned long long* dst = a.dg.rho + (size_t)(a.dg.wj0 + r0) * a.dg.nx + a.dg.wi0;
                    const uint32_t bytes = (uint32_t)((r1 - r0 + 1) * wnx * 8);
                    if (DEP == 2) asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.u64 [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes) : "memory");
                    else asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f64 [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes) : "memory");
                }
                if (tid < n_ops) asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            }
        }
        if (len > 0) {
            for (int b = tid; b < nh; b += NT) {
                const unsigned int v = s_hist[b];
                if (v) atomicAdd(a.dg.hist + b, v);
            }
            if (SC_BULK_FLUSH) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");   // reductions complete (not only read) before the CTA exits
        }
        SC_STAMPP(6);
        n_out = __reduce_add_sync(0xffffffffu, n_out);
        if (lane == 0 && n_out) atomicAdd(a.counters, (unsigned long long)n_out);
    }
}

}  // namespace sc
