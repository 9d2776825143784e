// anm_alias.cuh -- A0 set-up on the device: the alias table over the active voxels (
// PAPER.md:L65 "probability density ... linear conversion of the PET value").
//
// Walker / Vose alias tables are usually built by a sequential sweep: light items (scaled weight w <= 1) are taken in
// order, each bucket topped up by the current heavy item (w > 1), whose residual shrinks until it is light itself and
// the next heavy item tops it up.  After i light and j heavy items are finished (k = i + j buckets), the residual of
// heavy item j is  r = L[i] + H[j+1] - k  (L, H = exclusive prefix sums of the light / heavy weights), so the state of
// the sweep at step k is a function of k alone:  i_k = min{ i : L[i] + H[k-i] - k < 0 }  (monotone in i, found by
// bisection), and step k finishes light item i (if r >= 1) or heavy item j = k - i (else).  Every bucket is therefore
// computed independently by one thread -- no sequential pass and no host copy of the activity volume.
//
// entry k = {threshold = floor(P(own) 2^32), own voxel, alias voxel, 0}; the SOURCE event draws a bucket uniformly
// (64 random bits) and takes `own` iff a 32-bit uniform is below the threshold.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace anm {

constexpr int kAliasThreads = 256;

// pass 1: validation, number of active voxels and total activity; one partial per block (summed in block order on
// the host: deterministic).  flags bit 0 = a negative / non-finite value was seen.
__global__ void __launch_bounds__(kAliasThreads)
activity_stats_kernel(const float* __restrict__ act, size_t V, double* __restrict__ block_sum,
                      unsigned long long* __restrict__ block_cnt, unsigned* __restrict__ flags) {
    __shared__ double s_sum[kAliasThreads / 32];
    __shared__ unsigned long long s_cnt[kAliasThreads / 32];
    double sum = 0.0;
    unsigned long long cnt = 0ull;
    unsigned bad = 0u;
    for (size_t i = (size_t)blockIdx.x * kAliasThreads + threadIdx.x; i < V; i += (size_t)gridDim.x * kAliasThreads) {
        const float a = act[i];
        if (!(a >= 0.0f) || !(a <= 3.402823466e38f)) bad = 1u;
        else if (a > 0.0f) { sum += (double)a; ++cnt; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        sum += __shfl_xor_sync(0xffffffffu, sum, o);
        cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    }
    if ((threadIdx.x & 31) == 0) { s_sum[threadIdx.x >> 5] = sum; s_cnt[threadIdx.x >> 5] = cnt; }
    if (bad) atomicOr(flags, 1u);
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        unsigned long long n = 0ull;
        for (int w = 0; w < kAliasThreads / 32; ++w) { t += s_sum[w]; n += s_cnt[w]; }
        block_sum[blockIdx.x] = t;
        block_cnt[blockIdx.x] = n;
    }
}

// selection predicates over voxel indices and the weight of a selected voxel (scaled so that the mean is 1)
struct AliasIsLight {
    const float* act; double scale;
    __host__ __device__ bool operator()(const uint32_t v) const { const float a = act[v]; return a > 0.0f && (double)a * scale <= 1.0; }
};
struct AliasIsHeavy {
    const float* act; double scale;
    __host__ __device__ bool operator()(const uint32_t v) const { const float a = act[v]; return a > 0.0f && (double)a * scale > 1.0; }
};
struct AliasWeight {
    const float* act; const uint32_t* idx; double scale;
    __host__ __device__ double operator()(const uint32_t i) const { return (double)act[idx[i]] * scale; }
};

__device__ __forceinline__ unsigned alias_threshold(double prob) {
    const double t = floor(fmin(fmax(prob, 0.0), 1.0) * 4294967296.0);
    return t >= 4294967295.0 ? 0xffffffffu : (unsigned)t;
}

// pass 3: bucket k of the sweep (see the header comment).  L[0..nl], H[0..nh]: exclusive prefix sums with the total
// in the last element.
__global__ void __launch_bounds__(kAliasThreads)
alias_build_kernel(const float* __restrict__ act, double scale, const uint32_t* __restrict__ lidx,
                   const uint32_t* __restrict__ hidx, const double* __restrict__ L, const double* __restrict__ H,
                   unsigned nl, unsigned nh, uint4* __restrict__ tab) {
    const unsigned M = nl + nh;
    const unsigned k = blockIdx.x * kAliasThreads + threadIdx.x;
    if (k >= M) return;
    if (nh == 0u) {                         // every weight is exactly the mean: P(own) = 1
        const uint32_t v = lidx[k];
        tab[k] = make_uint4(0xffffffffu, v, v, 0u);
        return;
    }
    unsigned lo = k >= nh ? k - (nh - 1u) : 0u, hi = min(k, nl);
    const double kd = (double)k;
    while (lo < hi) {
        const unsigned mid = (lo + hi) >> 1;
        if (L[mid] + H[k - mid] - kd < 0.0) hi = mid; else lo = mid + 1u;
    }
    const unsigned i = lo, j = k - lo;
    const double r = L[i] + H[j + 1u] - kd;                     // residual of heavy item j at step k
    if (i < nl && r >= 1.0) {                                   // light item i, topped up by heavy item j
        const uint32_t v = lidx[i];
        tab[k] = make_uint4(alias_threshold((double)act[v] * scale), v, hidx[j], 0u);
    } else {                                                    // heavy item j has become light: next heavy tops it up
        const uint32_t v = hidx[j];
        tab[k] = make_uint4(alias_threshold(r), v, j + 1u < nh ? hidx[j + 1u] : v, 0u);
    }
}

}  // namespace anm
