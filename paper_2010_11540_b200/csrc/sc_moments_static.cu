// sc_moments_static.cu -- sc_moments_static(): the beam moments of sc_moments() for callers that may not allocate
// device memory (declared and documented in include/sc_track.h).
//
// Who that is.  sc_moments() needs a context, and a context needs a device workspace: either the caller cuts one out
// of memory it already owns, or sc_create() calls cudaMalloc.  Two kinds of caller have neither option.  (1) A
// diagnostics hook that runs beside a job whose allocator has already taken the GPU's memory for its own pool (a torch
// process with the caching allocator grown to the card, a batch job with a fixed device budget): a raw cudaMalloc there
// fails, or succeeds only by pushing the pool into an out-of-memory error later, and the hook has no handle on the pool.
// (2) A monitor that looks at the beam while tracking streams are busy: cudaMalloc and cudaFree stall every stream of
// the device until the allocation is done, which would show up as a gap in every turn it coincides with.
//
// What this file does instead.  The per-CTA partial sums -- the only memory the moment kernels need beyond the
// particle arrays and the 33 results -- live in g_scratch below, a file-scope __device__ array that is part of the
// library's device image: the CUDA runtime places it when the library's module is loaded on a device, and every device
// that loads the module keeps those kStaticBytes (about 0.66 MiB) until the process exits.  Nothing else is needed, so
// the call makes no cudaMalloc / cudaFree / cudaMallocAsync and creates no stream, event, graph or library handle.
//
// g_scratch in HOST code is only the runtime's handle for the symbol, not an address a kernel can use: the kernels get
// the pointer cudaGetSymbolAddress() returns for the current device (scratch_for_current_device below), looked up once
// per device and kept.
//
// The kernels are this file's own (same two-pass scheme as k_moments.cuh, which stays as it is): a CTA owns a fixed,
// contiguous run of kChunk particles, so the number of partials grows with n -- hence the size limit -- and the result
// does not depend on the number of SMs; the last CTA to finish a pass (a ticket counter in the scratch) adds the
// partials up in a fixed order, so two calls on the same data give the same bits.
#include <cstdint>
#include <mutex>
#include <string>

#include <cuda_runtime.h>

#include "../../include/sc_track.h"
#include "sc_host.h"

namespace {

constexpr int kThreads = 256;                      // threads per CTA
constexpr int kPerThread = 16;                     // particles per thread
constexpr int kChunk = kThreads * kPerThread;      // 4096 particles per CTA
constexpr int kMaxBlocks = SC_MOMENTS_STATIC_MAX_PARTICLES / kChunk;   // 4096 CTAs
constexpr int kStride = 21;                        // doubles per CTA partial (pass 1 uses 7 of them, pass 2 all 21)
constexpr int kNumSums = 8;                        // pass-1 totals: 6 coordinate sums, non-finite count, spare
// layout of the scratch, in bytes: [partials: kMaxBlocks x kStride doubles][sums: 8 doubles][tickets: 2 x u32, padded]
constexpr size_t kOffSums = (size_t)kMaxBlocks * kStride * sizeof(double);
constexpr size_t kOffTickets = kOffSums + kNumSums * sizeof(double);
constexpr size_t kTicketBytes = 64;
constexpr size_t kStaticBytes = kOffTickets + kTicketBytes;            // 688,256 bytes
static_assert(SC_MOMENTS_STATIC_MAX_PARTICLES % kChunk == 0, "the particle limit is a whole number of CTA chunks");
static_assert(kOffTickets % 8 == 0, "tickets are 4-byte words behind 8-byte doubles");

// The scratch itself.  Shared by every call on a device, never cleared as a whole: a call overwrites every partial and
// total it later reads, and zeroes the two ticket words (the one thing that must start at zero) before its first kernel.
static __device__ __align__(256) unsigned char g_scratch[kStaticBytes];

struct Scratch {
    double* partial;
    double* sums;
    unsigned int* tickets;
};

__device__ __forceinline__ Scratch carve(unsigned char* base) {
    Scratch s;
    s.partial = reinterpret_cast<double*>(base);
    s.sums = reinterpret_cast<double*>(base + kOffSums);
    s.tickets = reinterpret_cast<unsigned int*>(base + kOffTickets);
    return s;
}

// CTA-wide sum of NV per-thread values into partial[blockIdx.x][0..NV); returns true (to every thread) in the CTA
// that finished last, after the partials of all CTAs have become visible to it.
template <int NV>
__device__ __forceinline__ bool reduce_store_and_take_ticket(double (&v)[NV], double* partial, unsigned int* ticket) {
    __shared__ double s_part[kThreads / 32][NV];
    __shared__ bool s_last;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < NV; k++) {
        double t = v[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        if (lane == 0) s_part[warp][k] = t;
    }
    __syncthreads();
    if (threadIdx.x < NV) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < kThreads / 32; w++) t += s_part[w][threadIdx.x];
        partial[(size_t)blockIdx.x * kStride + threadIdx.x] = t;
        __threadfence();                                       // the partial is visible device-wide before the ticket is
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned int t = atomicAdd(ticket, 1u);
        s_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    const bool last = s_last;
    if (last) __threadfence();
    return last;
}

// Sum of column k over the first nblocks partials, by one warp, in an order that depends on nblocks only:
// lane l adds blocks l, l+32, ... in turn, then the 32 lane totals are folded by xor-shuffles.
__device__ __forceinline__ double warp_column_total(const double* partial, int nblocks, int k) {
    const int lane = threadIdx.x & 31;
    double t = 0.0;
    for (int b = lane; b < nblocks; b += 32) t += __ldcg(&partial[(size_t)b * kStride + k]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    return t;
}

struct Coords { const double* q[6]; };

// pass 1: sums of the coordinates and the count of particles with a non-finite coordinate -> scratch sums[0..6]
__global__ void __launch_bounds__(kThreads) k_static_sum(const Coords c, int ncoord, long long n, unsigned char* scratch) {
    const Scratch s = carve(scratch);
    double v[7] = { 0, 0, 0, 0, 0, 0, 0 };
    const long long base = (long long)blockIdx.x * kChunk + threadIdx.x;
#pragma unroll 4
    for (int j = 0; j < kPerThread; j++) {
        const long long p = base + (long long)j * kThreads;
        if (p < n) {
            bool bad = false;
#pragma unroll
            for (int k = 0; k < 6; k++)
                if (k < ncoord) { const double t = c.q[k][p]; v[k] += t; bad |= !isfinite(t); }
            v[6] += bad ? 1.0 : 0.0;
        }
    }
    if (!reduce_store_and_take_ticket<7>(v, s.partial, s.tickets + 0)) return;
    const int warp = threadIdx.x >> 5;
    if (warp < 7) {
        const double t = warp_column_total(s.partial, (int)gridDim.x, warp);
        if ((threadIdx.x & 31) == 0) s.sums[warp] = t;
    }
}

// pass 2: the 21 centred second moments about the means of pass 1; the last CTA writes the 33 results
__global__ void __launch_bounds__(kThreads) k_static_cov(const Coords c, int ncoord, long long n, unsigned char* scratch, double* out) {
    const Scratch s = carve(scratch);
    double mean[6];
#pragma unroll
    for (int k = 0; k < 6; k++) mean[k] = s.sums[k] / (double)n;
    double v[21];
#pragma unroll
    for (int k = 0; k < 21; k++) v[k] = 0.0;
    const long long base = (long long)blockIdx.x * kChunk + threadIdx.x;
#pragma unroll 2
    for (int j = 0; j < kPerThread; j++) {
        const long long p = base + (long long)j * kThreads;
        if (p < n) {
            double d[6];
#pragma unroll
            for (int k = 0; k < 6; k++) d[k] = k < ncoord ? c.q[k][p] - mean[k] : 0.0;
            int m = 0;
#pragma unroll
            for (int r = 0; r < 6; r++)
#pragma unroll
                for (int cc = r; cc < 6; cc++) v[m++] += d[r] * d[cc];
        }
    }
    if (!reduce_store_and_take_ticket<21>(v, s.partial, s.tickets + 1)) return;
    __shared__ double s_cov[21];
    const int warp = threadIdx.x >> 5;
    for (int k = warp; k < 21; k += kThreads / 32) {
        const double t = warp_column_total(s.partial, (int)gridDim.x, k);
        if ((threadIdx.x & 31) == 0) s_cov[k] = t;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const double dn = (double)n;
        out[0] = dn;
        for (int k = 0; k < 6; k++) out[1 + k] = mean[k];
        for (int k = 0; k < 21; k++) out[7 + k] = s_cov[k] / dn;
        // rms emittances of the three planes; products and difference rounded one by one (no fused multiply-add), as the
        // host arithmetic of sc_moments() does
        for (int pl = 0; pl < 3; pl++) {
            const int r = 2 * pl;
            const int i_aa = 7 + r * 6 - r * (r - 1) / 2;             // (r, r) of the row-major upper triangle
            const int i_ab = i_aa + 1;                                // (r, r+1)
            const int i_bb = 7 + (r + 1) * 6 - (r + 1) * r / 2;       // (r+1, r+1)
            const double det = __dsub_rn(__dmul_rn(out[i_aa], out[i_bb]), __dmul_rn(out[i_ab], out[i_ab]));
            out[28 + pl] = det > 0.0 ? sqrt(det) : 0.0;
        }
        out[31] = 0.0;                                                // no context, hence no space-charge node to count at
        out[32] = s.sums[6];
    }
}

// ---- host side ---------------------------------------------------------------------------------------------------

constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
unsigned char* g_scratch_on_device[kMaxDevices] = {};   // device address of g_scratch, per device ordinal; null = not looked up yet

int fail(int code, const std::string& msg) {
    sc::set_global_error(msg);
    return code;
}

// Set-up, once per device, with that device current: ask the runtime where g_scratch lives on the current device.
// (This is also what makes the runtime load the library's module there, which is when the array's memory is taken.)
int scratch_for_current_device(unsigned char** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess)
        return fail(SC_ECUDA, std::string("sc_moments_static: cudaGetDevice: ") + cudaGetErrorString(e) + " (no CPU fallback: a CUDA device is required)");
    if (dev < 0 || dev >= kMaxDevices) return fail(SC_EUNSUPPORTED, "sc_moments_static: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_on_device[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_scratch);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return fail(SC_ECUDA, std::string("sc_moments_static: cudaGetSymbolAddress(g_scratch): ") + cudaGetErrorString(e));
        }
        g_scratch_on_device[dev] = static_cast<unsigned char*>(p);
    }
    *out = g_scratch_on_device[dev];
    return SC_OK;
}

}  // namespace

extern "C" int sc_moments_static(const double* x, const double* px, const double* y, const double* py,
                                 const double* sigma, const double* psigma, int64_t n, double* out, void* stream) {
    if (!x || !px || !y || !py || !out) return fail(SC_EINVAL, "sc_moments_static: x, px, y, py and out must be device pointers");
    if ((sigma == nullptr) != (psigma == nullptr)) return fail(SC_EINVAL, "sc_moments_static: pass both sigma and psigma, or neither (4D beam)");
    if (n < 1) return fail(SC_EINVAL, "sc_moments_static: n must be at least 1");
    if (n > (int64_t)SC_MOMENTS_STATIC_MAX_PARTICLES)
        return fail(SC_EINVAL, "sc_moments_static: n = " + std::to_string(n) + " exceeds SC_MOMENTS_STATIC_MAX_PARTICLES = " +
                               std::to_string((long long)SC_MOMENTS_STATIC_MAX_PARTICLES) +
                               " (the built-in scratch holds one partial per 4096 particles; use sc_moments() on a context for larger beams)");
    unsigned char* scratch = nullptr;
    const int rc = scratch_for_current_device(&scratch);
    if (rc != SC_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int ncoord = sigma ? 6 : 4;
    const int blocks = (int)((n + kChunk - 1) / kChunk);
    Coords c;
    c.q[0] = x; c.q[1] = px; c.q[2] = y; c.q[3] = py; c.q[4] = sigma; c.q[5] = psigma;
    cudaError_t e = cudaMemsetAsync(scratch + kOffTickets, 0, kTicketBytes, st);   // the ticket counters start every call at zero
    if (e != cudaSuccess) return fail(SC_ECUDA, std::string("sc_moments_static: cudaMemsetAsync: ") + cudaGetErrorString(e));
    k_static_sum<<<blocks, kThreads, 0, st>>>(c, ncoord, (long long)n, scratch);
    k_static_cov<<<blocks, kThreads, 0, st>>>(c, ncoord, (long long)n, scratch, out);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(SC_ECUDA, std::string("sc_moments_static: kernel launch: ") + cudaGetErrorString(e));
    return SC_OK;
}
