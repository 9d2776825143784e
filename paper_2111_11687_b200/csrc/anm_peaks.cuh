// anm_peaks.cuh -- roofline microbenchmarks (BASELINE.json metric "% of L2/atomic
// roofline"): what THIS device sustains for the three things the transport kernel does, measured by hand-written
// kernels with the same access shapes, so that the bench line's fractions have measured denominators:
//   issue_kernel   a dependency-free stream of FFMA (fma pipes) and LOP3 (alu pipe)         -> thread-instructions / s
//   philox_kernel  back-to-back Philox4x32-10 blocks (the generator of the kernels)        -> blocks / s
//   gather_kernel  random 4-byte ld.global.nc over an array (the texel fetch)              -> loads / s
//   red_kernel     random fp32 RED.ADD over an array (the tally)                          -> atomics / s
//   mix_kernel     both at once, 5 loads : 2 REDs over two arrays (the transport's mix)    -> accesses / s
// each at two array sizes: one that fits the 126 MB L2 (cfg3's 105 MB volumes) and one that does not (cfg4's 630 MB).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace anm {

constexpr int kPeakThreads = 1024;

// cheap per-thread index stream: a 32-bit xorshift, mapped to [0, n) by a multiply-high (n < 2^32)
__device__ __forceinline__ unsigned peak_next(unsigned& s) {
    s ^= s << 13; s ^= s >> 17; s ^= s << 5;
    return s;
}

// kIssuePerIter counted instructions per unrolled step: 8 FFMA (fma pipes) + 8 LOP3 (alu pipe) on 16 independent
// registers, pinned with inline PTX so that the count is exact (the loop's own add / compare / branch, 3 per
// kIssueUnroll steps, are NOT counted: the figure is a lower bound of the issue rate, within 2 %)
constexpr int kIssuePerIter = 16;
constexpr int kIssueUnroll = 8;
__device__ __forceinline__ void issue_ffma(float& f, float a, float b) { asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f) : "f"(a), "f"(b)); }
__device__ __forceinline__ void issue_lop3(unsigned& i, unsigned j, unsigned k) { asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(i) : "r"(j), "r"(k)); }
__global__ void __launch_bounds__(kPeakThreads)
issue_kernel(float* __restrict__ out, long long* __restrict__ cycles, int iters, float a, float b, unsigned k) {
    const long long c0 = clock64();
    float f0 = threadIdx.x, f1 = f0 + 1, f2 = f0 + 2, f3 = f0 + 3, f4 = f0 + 4, f5 = f0 + 5, f6 = f0 + 6, f7 = f0 + 7;
    unsigned i0 = threadIdx.x, i1 = i0 + 1, i2 = i0 + 2, i3 = i0 + 3, i4 = blockIdx.x, i5 = i4 + 1, i6 = i4 + 2, i7 = i4 + 3;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < kIssueUnroll; ++u) {
            issue_ffma(f0, a, b); issue_lop3(i0, i4, k); issue_ffma(f1, a, b); issue_lop3(i1, i5, k);
            issue_ffma(f2, a, b); issue_lop3(i2, i6, k); issue_ffma(f3, a, b); issue_lop3(i3, i7, k);
            issue_ffma(f4, a, b); issue_lop3(i4, i0, k); issue_ffma(f5, a, b); issue_lop3(i5, i1, k);
            issue_ffma(f6, a, b); issue_lop3(i6, i2, k); issue_ffma(f7, a, b); issue_lop3(i7, i3, k);
        }
    }
    const float r = f0 + f1 + f2 + f3 + f4 + f5 + f6 + f7 + (float)(i0 ^ i1 ^ i2 ^ i3 ^ i4 ^ i5 ^ i6 ^ i7);
    if (r == 123.456f) out[0] = r;      // never true for the launch's arguments; keeps the chains alive
    if (blockIdx.x == 0 && threadIdx.x == 0) cycles[0] = clock64() - c0;    // SM cycles of one warp's whole loop -> the clock held
}

__global__ void __launch_bounds__(kPeakThreads)
philox_chain_kernel(const __grid_constant__ TransportParams p, unsigned* __restrict__ out, int blocks_per_thread) {
    uint4 c = make_uint4(threadIdx.x, blockIdx.x, 0u, 1u);
    for (int i = 0; i < blocks_per_thread; ++i) c = philox4x32_10(c, p);
    if ((c.x ^ c.y ^ c.z ^ c.w) == 0x12345678u) out[0] = c.x;
}

// IF independent random accesses per thread per trip.  The host sweeps IF over {4, 8, 16, 32} at full occupancy
// (64 resident warps per SM) and keeps the best rate: the denominators are then what the memory system gives when it
// is saturated, not what one arbitrary depth happens to reach.
template <int IF>
__global__ void __launch_bounds__(kPeakThreads)
gather_kernel(const uint32_t* __restrict__ a, unsigned n, int trips, unsigned* __restrict__ out) {
    unsigned s = (blockIdx.x * kPeakThreads + threadIdx.x) * 2654435761u + 0x9E3779B9u;
    unsigned acc = 0;
    for (int t = 0; t < trips; ++t) {
        unsigned v[IF];
#pragma unroll
        for (int k = 0; k < IF; ++k) v[k] = __ldg(a + __umulhi(peak_next(s), n));
#pragma unroll
        for (int k = 0; k < IF; ++k) acc += v[k];
    }
    if (acc == 0x12345678u) out[0] = acc;
}

template <int IF>
__global__ void __launch_bounds__(kPeakThreads)
red_kernel(float* __restrict__ a, unsigned n, int trips) {
    unsigned s = (blockIdx.x * kPeakThreads + threadIdx.x) * 2654435761u + 0x9E3779B9u;
    for (int t = 0; t < trips; ++t) {
#pragma unroll
        for (int k = 0; k < IF; ++k) atomicAdd(a + __umulhi(peak_next(s), n), 1.0f);
    }
}

// The transport kernel's mix: per trip kMixGathers random 4-byte loads from one array (texels) and kMixReds fp32 REDs
// into ANOTHER array of the same size (the tally) -- 5 : 2, cfg3's 15.6 sub-steps : 6.2 deposits per decay.  Both
// streams compete for the same L2 / HBM, so the sum of the separate gather and RED fractions overstates the headroom;
// this is the rate (loads + REDs per second) with both in flight.
constexpr int kMixGathers = 10, kMixReds = 4;
__global__ void __launch_bounds__(kPeakThreads)
mix_kernel(const uint32_t* __restrict__ a, float* __restrict__ b, unsigned n, int trips, unsigned* __restrict__ out) {
    unsigned s = (blockIdx.x * kPeakThreads + threadIdx.x) * 2654435761u + 0x9E3779B9u;
    unsigned acc = 0;
    for (int t = 0; t < trips; ++t) {
        unsigned v[kMixGathers];
#pragma unroll
        for (int k = 0; k < kMixGathers; ++k) v[k] = __ldg(a + __umulhi(peak_next(s), n));
#pragma unroll
        for (int k = 0; k < kMixReds; ++k) atomicAdd(b + __umulhi(peak_next(s), n), 1.0f);
#pragma unroll
        for (int k = 0; k < kMixGathers; ++k) acc += v[k];
    }
    if (acc == 0x12345678u) out[0] = acc;
}

}  // namespace anm
