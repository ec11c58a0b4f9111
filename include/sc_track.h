/*
 * sc_track.h -- C ABI of libsc_track: the per-turn hot path of the 2D particle-in-cell
 * space-charge tracker of arXiv 2010.11540 (Kurimoto), hand-written CUDA for sm_100a (B200).
 *
 * Per turn, every macroparticle is carried through the ring's table rows in order (PAPER.md:22,
 * 314): symplectic single-particle maps (section III) and, at every SCNODE row,
 * the four space-charge steps of section IV: cloud-in-cell deposit (eq. 14),
 * Poisson solve (here: open boundary, FFT convolution with the cell-integrated 2D Green's function
 * on the doubled Hockney grid, ref [1] of the paper), field gather (bilinear) and the kick of
 * eq. 12 weighted by the longitudinal line density lambda(sigma).
 * DESIGN.md lists every reading taken where the paper is silent or garbled.
 *
 * Conventions
 *  - Every call returns SC_OK (0) or a negative code; no C++ exception crosses the ABI;
 *    sc_last_error() gives a message for the last failing call on that context.
 *  - Pointers are HOST pointers unless a parameter says "device".  Inputs are copied: the caller
 *    keeps ownership of every array it passes.  A context is not thread-safe.
 *  - All device work is issued on the CUDA stream given to sc_create (0 = default stream); calls
 *    that return data to the host synchronise that stream; sc_track/sc_step are asynchronous.
 *  - Device memory: the caller hands sc_create ONE device workspace (e.g. a torch uint8 tensor's
 *    data_ptr) of at least sc_workspace_bytes(); the library allocates no device memory itself
 *    unless workspace == NULL, in which case it cudaMallocs (and frees in sc_destroy) its own.
 *  - There is no CPU fallback: without a CUDA device every compute call returns SC_ECUDA.
 *  - Coordinates: x, px, y, py, sigma = s - beta0 c t, psigma; SoA fp64.
 *    Passing sigma == psigma == NULL to sc_load_particles selects the 4D coasting-beam variant
 *    (psigma = 0, no RF rows, grids must have nbins == 0).
 */
#ifndef SC_TRACK_H
#define SC_TRACK_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SC_OK            0
#define SC_EINVAL       -1   /* bad argument / malformed table                                   */
#define SC_ENOMEM       -2   /* workspace too small / allocation failed                          */
#define SC_ECUDA        -3   /* CUDA runtime error (message in sc_last_error)                    */
#define SC_FLAG_NO_PDL  1ull /* sc_create flag, see there                                           */
#define SC_FLAG_FUSED_POISSON 2ull /* sc_create flag, see there                                    */
#define SC_FLAG_NO_FIELD_WINDOW 4ull /* sc_create flag, see there                                    */
#define SC_FLAG_BLOCK_FFT_POISSON 8ull /* sc_create flag, see there                                  */
#define SC_FLAG_WARP_FFT_POISSON 16ull /* sc_create flag, see there                                  */
#define SC_ESTATE       -4   /* call out of order (e.g. sc_track before sc_load_particles)       */
#define SC_EUNSUPPORTED -5   /* valid request this build does not implement (e.g. nx not 2^k)    */

typedef struct sc_ctx sc_ctx;          /* opaque */

/* One lattice table row: 88-byte POD. */
typedef struct { int32_t kind, ipar; double p[10]; } sc_elem;
enum {
    SC_DRIFT  = 0, /* p0 = L [m].  Flow of H0, eq. 7:
                      x += L (1-psigma) px, y likewise, sigma += L (psigma/gamma0^2 - (px^2+py^2)/2) */
    SC_LINMAP = 1, /* p0..3 = Mx (m11 m12 m21 m22), p4..7 = My, p8 = L.  Uncoupled linear map;
                      sigma += L psigma/gamma0^2 (eq. 6 at psigma = 0)           */
    SC_MULT   = 2, /* ipar = n >= 0, p0 = knL, p1 = ksL [m^-n].  Thin kick:
                      px - i py += -(knL + i ksL) (x + i y)^n / n!                                 */
    SC_RF     = 3, /* p0 = V [volt], p1 = h, p2 = phi0 [rad]:
                      psigma -= q V/(beta0^2 E0) sin(2 pi h sigma/C + phi0)                        */
    SC_SCNODE = 4, /* ipar = grid id, p0 = L_sc [m] = distance since the previous node (eq. 12,
                      PAPER.md:163-167): deposit, solve, gather, kick                             */
    SC_QUAD   = 5, /* p0 = k1 [m^-2], p1 = L: thick quadrupole, converted by sc_create to the
                      LINMAP of eq. 6 at psigma = 0 (k1 > 0 focuses x)                            */
    SC_CQUAD  = 6, /* p0 = k1 [m^-2], p1 = L: thick quadrupole, eq. 6 AS PRINTED, per particle
                      (PAPER.md:97-125): strength k1 (1 - psigma), sin/cos and sinh/cosh of
                      sqrt(|k1| (1-psigma)) L per particle, and
                      sigma += L psigma/gamma0^2 - 1/2 int (px^2 + py^2) ds in closed form;
                      k1 = 0 is a DRIFT                                                            */
    SC_SEXT   = 7, /* p0 = k2 [m^-3], p1 = L: thick sextupole, eqs. 7-8:
                      H0 drift aL, kick k2 bL, drift cL, kick k2 bL, drift aL with
                      a = (1 - 1/sqrt 3)/2, b = 1/2, c = 1/sqrt 3                                  */
    SC_XDRIFT = 8, /* p0 = L: EXACT drift, the B = 0 case of section III.A: with
                      pz = sqrt(1 + 2 psigma + beta0^2 psigma^2 - px^2 - py^2) (eq. 3)
                      x += L px/pz, y += L py/pz, sigma += L (1 - (1 + beta0^2 psigma)/pz)         */
    SC_SBEND  = 9  /* p0 = L, p1 = h = 1/rho [1/m]: EXACT sector bend, section III.A (eqs. 2-5):
                      uniform field that bends the reference particle on the reference orbit; the particle's
                      circle is intersected with the exit plane at angle L h (closed form in DESIGN.md / the
                      oracle); h = 0 is SC_XDRIFT                                                  */
};

/* Transverse grid of nx x ny NODES ("grids" are the representative points) and the
 * lambda(sigma) histogram.  dx = (xmax-xmin)/(nx-1); a particle is inside iff
 * 0 <= (x-xmin)/dx < nx-1 on both axes; outside particles deposit nothing and get no kick.      */
typedef struct {
    int32_t nx, ny;                 /* powers of two, 8..512                                      */
    double xmin, xmax, ymin, ymax;  /* coordinates of the first / last node                       */
    int32_t nbins;                  /* 0: coasting beam (lambda = beam.line_density); else <= 4096 */
    double smin, smax;              /* histogram range [smin, smax), e.g. one RF bucket           */
    int32_t deposit_mode;           /* 0: fp64 atomic accumulation; 1: deterministic int64 fixed point */
    int32_t fixed_bits;             /* mode 1: per-axis fraction bits s, 1..20 (weights sum to 2^(2s));
                                       max_particles * 2^(2s) must stay below 2^63 (SC_EINVAL otherwise)  */
    int32_t boundary;               /* SC_BOUNDARY_OPEN: free space (Hockney convolution with the cell-integrated
                                       Green's function on the doubled grid).  SC_BOUNDARY_PIPE: the paper's solver
                                       (eqs. 15-27): conducting rectangular pipe, u = 0 on the
                                       wall = node 0 and the virtual node nx (ny) one spacing beyond the last node;
                                       five-point Laplacian, odd extension to 2nx x 2ny, eq. 25; charge deposited
                                       on the wall node 0 is dropped                                            */
    int32_t long_kick;              /* 1: the kick of a node on this grid also changes psigma (eq. 13):
                                       psigma -= kappa L_sc u~(x,y) dlambda/dsigma, u~ gathered bilinearly, the slope
                                       that of the piecewise-linear lambda(sigma); needs nbins > 0.  The potential's
                                       zero is the pipe wall: physically meaningful with SC_BOUNDARY_PIPE            */
    int32_t interp;                 /* SC_INTERP_BILINEAR: bilinear gather of the node field with the deposit's weights (north_star's
                                       hot path).  SC_INTERP_BICUBIC: the paper's interpolation (eqs. 28-29):
                                       bicubic Bezier surface of the POTENTIAL on the 4x4 stencil around the particle's cell and
                                       its analytic gradient; control net = B-spline-to-Bezier conversion of the stencil (the
                                       uniform cubic B-spline, C^2; reading A9 in DESIGN.md); stencil nodes beyond the grid edge
                                       are linear extrapolations; the longitudinal kick then uses the same surface.  Note: no prefilter,
                                       so the surface smooths the solved potential, u(x_i) = (U_{i-1} + 4 U_i + U_{i+1})/6 per axis: an
                                       O(h^2) low-pass bias of the field, about (h/sigma)^2/3 per axis for a Gaussian beam (A9)  */
} sc_grid;
#define SC_DEPOSIT_F64   0
#define SC_DEPOSIT_FIXED 1
#define SC_BOUNDARY_OPEN 0
#define SC_BOUNDARY_PIPE 1
#define SC_INTERP_BILINEAR 0
#define SC_INTERP_BICUBIC  1

typedef struct {
    double kinetic_eV, mass_eV;     /* reference particle                                          */
    int32_t charge;                 /* in units of e                                               */
    double line_density;            /* coasting beams: particles per metre                         */
    double n_real;                  /* bunched beams: real particles per bunch                     */
    double circumference;           /* [m]; 0 => sum of the DRIFT/LINMAP/QUAD lengths              */
} sc_beam;

/* Bytes of device workspace sc_create needs for this table, these grids and max_particles. */
int sc_workspace_bytes(const sc_elem* lat, int64_t n_elem, const sc_grid* grids, int32_t n_grids,
                       int64_t max_particles, int64_t* bytes_out);

/* Build a context: validates and copies the table, converts QUAD rows, precomputes per grid the
 * real transform of the Green's function and the FFT twiddles, uploads everything.
 *   workspace: DEVICE pointer, 256-byte aligned, workspace_bytes >= sc_workspace_bytes(); or NULL.
 *   stream: a cudaStream_t (as void*), 0 for the default stream.  Pass a stream you created: whole turns are then captured
 *   once into a CUDA graph and replayed (one graph launch per turn).  The legacy default stream (0) cannot be captured, so
 *   with stream = 0 every turn is issued as its individual kernel launches (433 per turn at cfg3): same results, slower,
 *   and sc_profile_replay returns SC_ESTATE.
 *   flags: 0, or SC_FLAG_NO_PDL to launch the kernels of a turn strictly one after the other
 *   (default: programmatic dependent launch, each kernel's set-up overlaps its predecessor's tail;
 *   results are identical, the flag exists for A/B timing); SC_FLAG_FUSED_POISSON to solve 64- and 128-node
 *   grids with ONE launch (register transforms, two grid-wide barriers) instead of the three-launch
 *   shared-memory FFT path (same mathematics; measured slower on B200, kept for A/B timing and cross-checking);
 *   SC_FLAG_NO_FIELD_WINDOW to gather every particle's node fields through the L1 cache instead of from the
 *   shared-memory copy of the grid's central window (A/B timing; results agree to rounding);
 *   Field solve: 128 x 128 grids take ONE launch of one 16-CTA thread-block cluster by default (16-lane register transforms,
 *   the stages handing over through distributed shared memory, k_poisson_cluster.cuh; if the device cannot place such a
 *   cluster the library falls back to the next path by itself); other grids with 64- or 128-node axes take three launches of
 *   warp-per-transform kernels (hand-over through L2), all other sizes three launches of block-per-transform shared-memory FFT
 *   kernels.  SC_FLAG_WARP_FFT_POISSON selects the warp-per-transform path for 128 x 128 as well, SC_FLAG_BLOCK_FFT_POISSON
 *   the block-per-transform path for every size (same mathematics, results agree to rounding; A/B timing and cross-checking). */
int sc_create(sc_ctx** out, const sc_elem* lat, int64_t n_elem, const sc_grid* grids, int32_t n_grids,
              const sc_beam* beam, int64_t max_particles, void* workspace, int64_t workspace_bytes,
              void* stream, uint64_t flags);

/* Copy n <= max_particles particles into the SoA store and rewind to row 0 of turn 0.
 * on_device != 0: the six pointers are DEVICE pointers.  sigma = psigma = NULL: 4D beam.  Synchronises the
 * context's stream before returning (host or device sources may be freed or overwritten at once); device sources
 * written on another stream must be complete before the call.                                   */
int sc_load_particles(sc_ctx* c, const double* x, const double* px, const double* y, const double* py,
                      const double* sigma, const double* psigma, int64_t n, int32_t on_device);

/* Advance n_turns whole turns (all rows, in order).  Asynchronous on the context's stream. */
int sc_track(sc_ctx* c, int64_t n_turns);

/* Test hook: advance exactly n_rows table rows (wrapping over turns).  If the last row is an SCNODE
 * the call stops after its deposit and field solve, BEFORE its kick (the kick is applied first thing
 * by the next sc_step/sc_track), so that particles and grids can be compared mid-node.          */
int sc_step(sc_ctx* c, int64_t n_rows);

/* Copy the particles back (synchronises).  on_device as in sc_load_particles; NULL pointers are skipped. */
int sc_get_particles(sc_ctx* c, double* x, double* px, double* y, double* py, double* sigma, double* psigma,
                     int32_t on_device);

/* Grids of the LAST executed SC node on grid `grid_id`, row-major [ny][nx] (x fastest):          */
enum { SC_GRID_RHO_F64 = 0, /* deposited charge Q (eq. 14), double; in fixed mode = int * 2^(-2s) */
       SC_GRID_RHO_I64 = 1, /* fixed mode only: the raw int64 accumulators                        */
       SC_GRID_PHI     = 2, /* u~ = (1/N) sum G Q, double                                         */
       SC_GRID_EX      = 3, /* -du~/dx, double                                                    */
       SC_GRID_EY      = 4, /* -du~/dy, double                                                    */
       SC_GRID_LAMBDA  = 5  /* int64 histogram counts, nbins entries                              */ };
int sc_get_grid(sc_ctx* c, int32_t grid_id, int32_t which, void* out, int64_t bytes);

/* out[0]=N, out[1..6]=means (x,px,y,py,sigma,psigma), out[7..27]=upper-triangular central second
 * moments (row-major), out[28..30]=rms emittances eps_x, eps_y, eps_sigma
 * (sqrt(<u^2><pu^2>-<u pu>^2)), out[31]=particles outside the grid at the last SC node,
 * out[32]=particles with a non-finite coordinate.  n_out must be >= 33.  Synchronises.          */
#define SC_N_MOMENTS 33
int sc_moments(sc_ctx* c, double* out, int32_t n_out);

/* The moments of sc_moments() for callers that cannot allocate device memory: no context, no workspace, no cudaMalloc.
 *
 * Who needs it: sc_moments() works on a context, and a context lives in a device workspace that somebody has to
 * allocate.  A diagnostics hook inside a process whose allocator already owns the GPU's memory (a torch job whose
 * caching pool has grown to the card, a batch job with a fixed device budget) cannot get one: a raw cudaMalloc there
 * fails or starves the pool, and the hook has no access to the pool.  A beam monitor that runs while tracking streams
 * are busy should not try: cudaMalloc / cudaFree hold up every stream of the device while they run.  This call takes
 * the particle arrays where they already are and needs no memory of the caller's beyond the 33 results.
 *
 *   x, px, y, py, sigma, psigma: DEVICE pointers to n doubles each, read only (sigma = psigma = NULL: 4D beam, the two
 *       coordinates count as zero).  out: DEVICE pointer to SC_N_MOMENTS doubles, laid out as sc_moments() writes them,
 *       except out[31] = 0 (there is no context, so no space-charge node to count outside particles at).
 *   stream: a cudaStream_t (as void*) of the CURRENT device, 0 for the default stream.  The call is asynchronous: it
 *       queues one 64-byte memset and two kernels on `stream` and returns; `out` is valid once that work is complete.
 *       The pointers and the stream must belong to the device that is current in the calling thread.
 *
 * Where the scratch comes from: the per-CTA partial sums go into an array that is built into the library's device code,
 * 688,256 bytes (0.66 MiB), which every GPU that loads the library holds until the process exits.  It holds one
 * partial per 4096 particles, hence the limit: n > SC_MOMENTS_STATIC_MAX_PARTICLES (2^24) is refused with SC_EINVAL and
 * a message naming the limit (use sc_moments() on a context for larger beams).  The call makes no cudaMalloc, cudaFree
 * or other allocating call, and creates no stream, event or handle.
 *
 * First call on a device: it looks up the array's device address (cudaGetSymbolAddress, which also makes the CUDA
 * runtime load this library's device code on that GPU) and keeps it; later calls on that device skip this.  Make that
 * first call at set-up time, on each device you will use, with that device current, and before any stream capture.
 *
 * Sharing: all calls on a device use the same array, and it keeps what the last call left in it.  Each call overwrites
 * every partial it later reads and zeroes its two completion counters first, so calls that run one after the other
 * (same stream, or ordered by events) are independent of each other.  Two calls that can overlap on the GPU (different
 * streams or threads without ordering) write the same partials and counters and give wrong results: order them.
 *
 * Results: same two-pass scheme as sc_moments() (means, then centred second moments) but its own summation order, so
 * the two agree to rounding (about 1e-15 relative to the rms sizes), not bit for bit; two calls on the same data agree
 * bit for bit with each other, on any B200.  Errors: SC_EINVAL (null pointers, only one of sigma / psigma, n < 1, n beyond
 * the limit), SC_ECUDA (no device, failed look-up or launch), SC_EUNSUPPORTED (device ordinal above 63); the message is
 * returned by sc_last_error(NULL) on the calling thread.                                                            */
#define SC_MOMENTS_STATIC_MAX_PARTICLES 16777216
int sc_moments_static(const double* x, const double* px, const double* y, const double* py,
                      const double* sigma, const double* psigma, int64_t n, double* out, void* stream);

/* Measurement hook: advance ONE whole turn with plain (non-graph) launches and a CUDA-event pair
 * around every launch group, on the context's stream.  Must start at a turn boundary.  Synchronises.
 * out[0] = summed duration of the k_push launches [ms], out[1] = their number,
 * out[2] = summed duration of the field-solve launch groups (1 or 3 kernels each) [ms], out[3] = their number,
 * out[4] = duration of the whole turn [ms].  n_out >= 5.                                         */
int sc_profile_turn(sc_ctx* c, double* out, int32_t n_out);

/* Measurement hook: ONE turn's launches are captured into a CUDA graph in one of four modes and replayed `reps` times
 * back to back between one CUDA-event pair on the context's stream (one warm-up replay first): kernel durations as
 * they are inside a turn's graph, free of the launch latency an event pair around a single plain launch includes.
 *   SC_REPLAY_TURN     every launch of the turn (what sc_track replays)
 *   SC_REPLAY_PUSH     only the k_push launches (kick + segment maps + deposit + flush each, same arguments and
 *                      particle count; the fields the kicks read are those of the last solved node)
 *   SC_REPLAY_POISSON  only the field-solve launches (the k_push launches wait for their predecessor and return)
 *   SC_REPLAY_EMPTY    every kernel of the turn launched, each waits for its predecessor and returns: the launch
 *                      floor of the graph
 * Particles, accumulators and the pending kick are saved before and restored after: `scratch` is a DEVICE buffer of
 * at least 8 x (6 or 4) x n bytes supplied by the caller (the library allocates nothing).  Must start at a turn
 * boundary; synchronises.  NOT restored: what sc_get_grid returns (charge, potential, fields, line density of the last
 * node per grid) -- after the hook these are the replay's (PUSH, TURN: of the replayed turn's last node; POISSON, EMPTY:
 * solved on zero density, i.e. zeros), not those of the last node sc_track / sc_step executed.  Tracking itself is
 * unaffected: every node recomputes them before its kick.
 * out[0] = ms per replayed turn, out[1] = kernels per turn in this mode, out[2] = SC nodes per turn,
 * out[3] = particles outside the grid per deposit (PUSH: mean over the replay; TURN: at the last node; else 0),
 * out[4] = reps, out[5] = n.  n_out >= 6.  With n_out >= 7 also out[6] = how many of the turn's k_push launches store
 * psigma (6D beams: a launch writes psigma back only if one of its rows is an RF row or its kick is a longitudinal one;
 * every other launch reads six coordinates and writes five, 88 instead of 96 bytes per particle; 4D beams: 0).       */
enum { SC_REPLAY_TURN = 0, SC_REPLAY_PUSH = 1, SC_REPLAY_POISSON = 2, SC_REPLAY_EMPTY = 3 };
int sc_profile_replay(sc_ctx* c, int32_t mode, int32_t reps, void* scratch, int64_t scratch_bytes, double* out, int32_t n_out);

/* Measurement hook: a plain copy kernel over the particle store's arrays (6 or 4 x n doubles read, as many written to
 * `scratch`, a 16-byte aligned DEVICE buffer of 8 x coordinates x (n rounded up to even) bytes), `reps` times between
 * one event pair after one warm-up: the attainable ceiling for k_push's algorithmic traffic at this n.
 * out[0] = ms per copy, out[1] = bytes read + written per copy.  n_out >= 2.  Synchronises.                          */
int sc_profile_copy(sc_ctx* c, int32_t reps, void* scratch, int64_t scratch_bytes, double* out, int32_t n_out);

/* Derived reference-particle constants: out[0]=gamma0, [1]=beta0, [2]=E0_eV, [3]=r_c [m],
 * [4]=kappa = 4 pi r_c/(beta0^2 gamma0^3), [5]=circumference used.                               */
int sc_get_constants(const sc_ctx* c, double* out, int32_t n_out);

/* Number of kernels launched by this context so far (graph-replayed kernels included). */
int64_t sc_kernel_launches(const sc_ctx* c);

/* sizeof(sc_elem), sizeof(sc_grid), sizeof(sc_beam) of THIS build, so that a binding can check its own struct
 * layouts before the first call.  n_out >= 3.                                                        */
int sc_abi_sizes(int32_t* out, int32_t n_out);

const char* sc_last_error(const sc_ctx* c);   /* never NULL; c may be NULL (global create error)   */
void sc_destroy(sc_ctx* c);                    /* NULL is a no-op                                   */

#ifdef __cplusplus
}
#endif
#endif
