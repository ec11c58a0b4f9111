// k_moments.cuh -- rms moments by warp-shuffle reductions (beta(s) from the rms of
// the tracked particles).  Two passes (means, then centred second moments) so that the variances do
// not cancel against the squared means; per-CTA partial sums are combined in a fixed order by a
// second tiny kernel, so the result is deterministic.
#pragma once
#include "sc_device.cuh"

namespace sc {

constexpr int kMomThreads = 256;

template <int NV>
__device__ __forceinline__ void block_reduce_store(double (&v)[NV], double* out_partial) {
    __shared__ double s_part[kMomThreads / 32][NV];
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
        for (int w = 0; w < kMomThreads / 32; w++) t += s_part[w][threadIdx.x];
        out_partial[(size_t)blockIdx.x * NV + threadIdx.x] = t;
    }
}

// pass 1: sums of the 6 coordinates (+ count of non-finite particles in slot 6)
__global__ void __launch_bounds__(kMomThreads) k_mom_sum(int ncoord, long long n, double* partial,
                                                         double* q0, double* q1, double* q2, double* q3, double* q4, double* q5) {
    const double* q[6] = { q0, q1, q2, q3, q4, q5 };
    double v[7] = { 0, 0, 0, 0, 0, 0, 0 };
    for (long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += (long long)gridDim.x * blockDim.x) {
        bool bad = false;
#pragma unroll
        for (int k = 0; k < 6; k++) {
            if (k < ncoord) { const double t = q[k][p]; v[k] += t; bad |= !isfinite(t); }
        }
        v[6] += bad ? 1.0 : 0.0;
    }
    block_reduce_store<7>(v, partial);
}

// combine per-CTA partials in CTA order: out[k] = sum_b partial[b][k] (one CTA)
__global__ void k_mom_combine(const double* partial, int nblocks, int nv, double* out) {
    const int k = threadIdx.x;
    if (k < nv) {
        double t = 0.0;
        for (int b = 0; b < nblocks; b++) t += partial[(size_t)b * nv + k];
        out[k] = t;
    }
}

// pass 2: 21 centred second moments; mean[k] = sums[k]/n read from device memory
__global__ void __launch_bounds__(kMomThreads) k_mom_cov(int ncoord, long long n, const double* sums, double* partial,
                                                         double* q0, double* q1, double* q2, double* q3, double* q4, double* q5) {
    const double* q[6] = { q0, q1, q2, q3, q4, q5 };
    double mean[6];
#pragma unroll
    for (int k = 0; k < 6; k++) mean[k] = sums[k] / (double)n;
    double v[21];
#pragma unroll
    for (int k = 0; k < 21; k++) v[k] = 0.0;
    for (long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += (long long)gridDim.x * blockDim.x) {
        double d[6];
#pragma unroll
        for (int k = 0; k < 6; k++) d[k] = k < ncoord ? q[k][p] - mean[k] : 0.0;
        int m = 0;
#pragma unroll
        for (int r = 0; r < 6; r++)
#pragma unroll
            for (int c = r; c < 6; c++) v[m++] += d[r] * d[c];
    }
    block_reduce_store<21>(v, partial);
}

// measurement only (sc_profile_copy): a plain copy of the particle store's arrays, 16 bytes per thread and step --
// the attainable ceiling for a kernel that reads and writes every coordinate once (k_push's algorithmic traffic)
struct CopyArgs { const double* src[6]; double* dst[6]; int nco; long long n2; };
__global__ void __launch_bounds__(512) k_copy_soa(const CopyArgs a) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < a.n2; i += (long long)gridDim.x * blockDim.x) {
#pragma unroll
        for (int k = 0; k < 6; k++)
            if (k < a.nco) reinterpret_cast<double2*>(a.dst[k])[i] = reinterpret_cast<const double2*>(a.src[k])[i];
    }
}

}  // namespace sc
