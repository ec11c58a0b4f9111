// sc_device.cuh -- structures shared by the host side of libsc_track and its kernels.
// (Product code; shares nothing with oracle/.)
#pragma once
#include <stdint.h>
#include <cuda_runtime.h>
#include "../../include/sc_track.h"

namespace sc {

constexpr int kMaxProgSlots = 160;       // 16-byte program slots per push launch (they travel as kernel parameters)
#ifndef SC_PP
#define SC_PP 2
#endif
#ifndef SC_PUSH_WARPS
#define SC_PUSH_WARPS 32
#endif
#ifndef SC_FUSED_GROUPS
#define SC_FUSED_GROUPS 4
#endif
constexpr int kPP = SC_PP;               // particles per lane and iteration, in registers (one 16-byte pair per coordinate
                                         // and 2 particles): halves the row dispatch and constant-bank traffic per
                                         // particle and gives every lane two independent fp64 dependency chains
constexpr int kChunk = 32 * kPP;         // particles per warp-iteration: lane l holds the pairs (64h + 2l, 64h + 2l + 1)
constexpr int kPushWarps = SC_PUSH_WARPS;           // warps per CTA, one CTA per SM: 32 x 64 registers fill the register
                                                    // file; the kernel is latency-bound, warps are what hides it
constexpr int kPushThreads = 32 * kPushWarps;
#ifndef SC_PUSH_THREADS_CQ
#define SC_PUSH_THREADS_CQ 512
#endif
constexpr int kPushThreadsCQ = SC_PUSH_THREADS_CQ;      // the heavy instantiation (chromatic / exact rows, bicubic kick): 16 warps x up to 128 registers
constexpr int kMaxBins = 4096;
constexpr int kSmemBudget = 227 * 1024;  // opt-in dynamic shared memory per CTA on sm_100a

// Checked builds (-DSC_CHECK, `python -m paper_2010_11540_b200.build --check` -> libsc_track_check.so): every index the kernels
// form from particle data or table parameters is tested before use; a failed test is counted in counters[6] and reported by
// sc_moments as an error.  compute-sanitizer is closed on the GPU pool this was developed on: this build is what
// `python -m paper_2010_11540_b200.selfcheck --check` runs instead (profiles/r02_sanitizer.md).
#ifdef SC_CHECK
#define SC_ASSERT(cnt_, cond_) do { if (!(cond_)) atomicAdd((cnt_) + 6, 1ull); } while (0)
#else
#define SC_ASSERT(cnt_, cond_) do { } while (0)
#endif

// Pre-decoded table rows ("program"): 16-byte slots {header, value}; header = opcode (low int) and
// an integer parameter (high int); extra slots hold further parameters.  Built per launch by
// sc_track.cu:encode_piece and passed in the kernel parameters (constant bank).  A DRIFT row followed
// by a thin normal multipole of order <= 3 is fused into one DMn slot pair (one dispatch, two rows).
enum {
    OP_DM0 = 0,     // {hdr, L} {k0L, k0sL}    drift, then order-0 kick: px -= k0L, py += k0sL
    OP_DM1 = 1,     // {hdr, L} {k1L, 0}       drift, then normal thin quadrupole kick
    OP_DM2 = 2,     // {hdr, L} {k2L, 0}       drift, then normal thin sextupole kick
    OP_DM3 = 3,     // {hdr, L} {k3L, 0}       drift, then normal thin octupole kick
    OP_DRIFT = 4,   // {hdr, L}
    OP_M0 = 5,      // {hdr, k0L} {k0sL, 0}
    OP_M1 = 6,      // {hdr, k1L}
    OP_M2 = 7,      // {hdr, k2L}
    OP_M3 = 8,      // {hdr, k3L}
    OP_LINMAP = 9,  // {hdr, L} {m11,m12} {m21,m22} {n11,n12} {n21,n22}
    OP_MULTG = 10,  // {hdr(n), knL} {ksL, 0}  any order n >= 1, normal + skew
    OP_RF = 11,     // {hdr, qV/(beta0^2 E0)} {2 pi h/C, phi0}
    OP_CQUAD = 12,  // {hdr, k1} {L, 0}        chromatic thick quadrupole (eq. 6 per particle)
    OP_XDRIFT = 13, // {hdr, L}                exact drift (sqrt + division per particle)
    OP_SBEND = 14,  // {hdr, L} {h, 0} {sin(L h), cos(L h)}   exact sector bend
    OP_END = 15     // terminator (always present)
};

// Everything a kernel needs to know about one transverse grid.  Passed BY VALUE in kernel params.
struct GridDev {
    int nx, ny;
    double xmin, ymin, inv_dx, inv_dy, dx, dy;
    double nxm1, nym1;                   // (double)(nx-1), (double)(ny-1): inside test bounds
    int nbins;
    double smin, ds, inv_ds, dnbins;
    int mode, bits;                      // SC_DEPOSIT_*, fixed_bits
    int long_kick;                       // the kick also changes psigma (eq. 13)
    int interp;                          // SC_INTERP_*: bilinear gather of E (0) or bicubic surface of the potential, eqs. 28-29 (1)
    int boundary;                        // SC_BOUNDARY_*: zero padding (open) or odd extension (pipe) in the FFT kernels
    double fixed_scale;                  // 2^s
    double fixed_inv;                    // 2^(-2s)
    // shared-memory window of the deposit grid (nodes); the whole grid when it fits
    int wi0, wj0, wnx, wny;
    // device buffers
    unsigned long long* rho;             // nx*ny accumulators: double bits (mode 0) or int64 (mode 1)
    unsigned int* hist;                  // nbins
    double* rho_last;                    // nx*ny  Q of the last node (double)
    long long* rhoi_last;                // nx*ny  raw int64 of the last node (mode 1)
    long long* hist_last;                // nbins
    double2* lam;                        // nbins+1  pairs (lambda_{m-1}, lambda_m) [1/m], lambda_{-1} = lambda_nbins = 0:
                                         //          one 16-byte load gives both neighbours of an interpolation point
    double2* A;                          // (nx+1)*ny   row-transformed density, [kx][j]
    double2* BU;                         // (nx+1)*ny   potential, x-spectral / y-real, [kx][j]
    double2* BV;                         // (nx+1)*ny   -d/dy of it; BV == BU + (nx+1)*ny: the fused kernel uses both as one
                                         //             [j][kx][2] array (U, V)
    double* phi;                         // nx*ny
    double2* E;                          // nx*ny  (Ex, Ey) interleaved
    const double* Ghat;                  // (nx+1)*(2ny) real multiplier of the spectrum, [kx][ky]: transform of the Green's
                                         //   function (open) or 1/(dx dy) over the symbol of eq. 25 (pipe)
    const double2* twx;                  // nx   entries exp(-2 pi i k/(2nx))
    const double2* twy;                  // ny   entries exp(-2 pi i k/(2ny))
};

struct PushArgs {
    double* q[6];                        // x px y py sigma psigma (SoA)
    long long n;
    int nslots;                          // program slots used, including the OP_END terminator
    long long per_cta;                   // particles per CTA (even)
    int do_kick;                         // apply the pending space-charge kick first
    double kick_scale;                   // kappa * L_sc
    double lam_const;                    // coasting: line density; bunched: unused
    double lam_scale;                    // bunched: n_real / (N ds)
    int do_dep;                          // deposit at the end
    double dep_scale, dep_inv;           // fp64 deposit mode: 2^e and 2^-e of the CTA-private integer accumulation (k_push.cuh)
    int ps_changes;                      // some row of this launch (RF, longitudinal kick) changes psigma: it must be stored
    double inv_gamma2;
    double beta0_2;                      // beta0^2 (exact drift)
    int noop;                            // measurement: wait for the predecessor and return (launch floor of the graph)
    unsigned long long* counters;        // [0] n_outside of the last deposit
    GridDev kg;                          // grid of the pending kick
    GridDev dg;                          // grid of the deposit
    double2 prog[kMaxProgSlots + 1];     // pre-decoded rows of this launch (constant bank); +1: prefetch slack
};
static_assert(sizeof(PushArgs) <= 4096, "kernel parameters must stay within 4 KB");

// Programmatic dependent launch (sm_90+): every kernel of the turn lets its successor be scheduled at once and
// blocks, after whatever set-up does not touch the predecessor's results, until the predecessor grid has
// completed and flushed.  All four kernels of a node execute pdl_wait(), so completion is transitive.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

struct PoissonArgs {
    GridDev g;
    double scale;                        // 1 / (Lx Ly N)
    double lam_scale;                    // n_real / (N ds)
    int noop;                            // measurement: wait for the predecessor and return (launch floor of the graph)
};

}  // namespace sc
