// anm_static.cu -- anm_organ_summary_static (include/anm.h): the per-organ pass of A11 for callers that cannot let
// the library allocate device memory.
//
// Who that is: a process that has handed the whole HBM to an allocator of its own (a PyTorch job whose caching
// allocator already holds the card, a planning server working out of one fixed arena) -- there a cudaMalloc made
// behind its back fails or fragments the arena; and a host thread on a deadline, for which cudaMalloc / cudaFree are
// off limits because they take driver locks and can wait for the whole device.  Every other entry point of libanm.so
// lives on an anm_ctx, and creating one allocates.
//
// finalize_kernel (anm_kernels.cuh) adds its per-organ accumulators into a ctx-owned device buffer.  The variant here
// does the same arithmetic, but its accumulators live in the file-scope __device__ array below: fixed size, part of
// the loaded module on every GPU that uses the library, held until the process exits.  This file calls no cudaMalloc,
// cudaFree, memory-pool or library routine that allocates; it shares no state with the anm_ctx code paths.
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <mutex>

#include "../../include/anm.h"

namespace {

constexpr int kStaticThreads = 256;
constexpr int kStaticRow = 3;                                              // {sum of rel^2, voxels with energy, energy} per label
constexpr int kStaticDoubles = kStaticRow * (ANM_STATIC_MAX_ORGANS + 1);   // 768 doubles = 6144 bytes
constexpr int kStaticMaxDevices = 64;

// The scratch.  In HOST code this name is only a stand-in the runtime uses to look the array up: it is not a device
// address and must never be handed to a kernel or to cudaMemsetAsync.  Host code uses the pointer static_setup() gets
// from cudaGetSymbolAddress for the current device.
static __device__ __align__(256) double g_static_scratch[kStaticDoubles];

struct StaticDevice { double* scratch = nullptr; int num_sms = 0; };
StaticDevice g_static_dev[kStaticMaxDevices];
std::mutex g_static_mutex;

int static_fail(char* errbuf, size_t errbuf_len, int code, const char* fmt, ...) {
    if (errbuf && errbuf_len) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(errbuf, errbuf_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

// Once per device, with that device current: where this device keeps its copy of g_static_scratch, and its SM count.
cudaError_t static_setup(int device, StaticDevice* out) {
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticDevice& d = g_static_dev[device];
    if (!d.scratch) {
        double* p = nullptr;
        int sms = 0;
        cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_static_scratch);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
        if (e != cudaSuccess) return e;
        if (!p || sms <= 0) return cudaErrorUnknown;
        d.num_sms = sms;
        d.scratch = p;
    }
    *out = d;
    return cudaSuccess;
}

// the voxel's relative sigma, as rel_sigma() of anm_kernels.cuh: sqrt((B Q / S^2 - 1) / (B - 1))
__device__ __forceinline__ float static_rel_sigma(float S, float Q, double B) {
    if (!(S > 0.0f)) return 0.0f;
    const double r2 = (B * (double)Q / ((double)S * (double)S) - 1.0) / (B - 1.0);
    return r2 > 0.0 ? (float)sqrt(r2) : 0.0f;
}

// One pass over the volume; `scratch` is this device's g_static_scratch, zeroed on the same stream just before.
// scratch[3 l + 0] += rel^2, [3 l + 1] += 1, [3 l + 2] += S over the voxels of label l in 1..n_organs with S != 0;
// scratch[2] (label 0's energy word) += S over every voxel.
__global__ void __launch_bounds__(kStaticThreads)
organ_summary_static_kernel(const float* __restrict__ sum, const float* __restrict__ sumsq, const uint8_t* __restrict__ labels,
                            size_t V, int n_organs, double B, double* __restrict__ scratch) {
    __shared__ double s_rel2[256], s_nz[256], s_en[256];
    __shared__ double s_tot;
    s_rel2[threadIdx.x] = 0.0; s_nz[threadIdx.x] = 0.0; s_en[threadIdx.x] = 0.0;
    if (threadIdx.x == 0) s_tot = 0.0;
    __syncthreads();
    double tot = 0.0;
    for (size_t i = (size_t)blockIdx.x * kStaticThreads + threadIdx.x; i < V; i += (size_t)gridDim.x * kStaticThreads) {
        const float S = sum[i];
        if (S == 0.0f) continue;
        tot += (double)S;
        if (labels) {
            const unsigned l = labels[i];
            if (l) {
                const float r = static_rel_sigma(S, sumsq[i], B);
                atomicAdd(&s_rel2[l], (double)r * (double)r);
                atomicAdd(&s_nz[l], 1.0);
                atomicAdd(&s_en[l], (double)S);
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
    if ((threadIdx.x & 31) == 0 && tot != 0.0) atomicAdd(&s_tot, tot);
    __syncthreads();
    if (threadIdx.x == 0 && s_tot != 0.0) atomicAdd(scratch + 2, s_tot);
    if (labels && threadIdx.x > 0 && (int)threadIdx.x <= n_organs && s_nz[threadIdx.x] != 0.0) {
        atomicAdd(scratch + kStaticRow * threadIdx.x + 0, s_rel2[threadIdx.x]);
        atomicAdd(scratch + kStaticRow * threadIdx.x + 1, s_nz[threadIdx.x]);
        atomicAdd(scratch + kStaticRow * threadIdx.x + 2, s_en[threadIdx.x]);
    }
}

// scratch -> the caller's rows: Eq. 3 (RMS of the voxels' relative sigma), the voxel count, the energy.
__global__ void __launch_bounds__(kStaticThreads)
organ_summary_emit_kernel(const double* __restrict__ scratch, double* __restrict__ out, int n_organs) {
    const int o = (int)threadIdx.x;
    if (o > n_organs) return;
    const double rel2 = scratch[kStaticRow * o], nz = scratch[kStaticRow * o + 1], en = scratch[kStaticRow * o + 2];
    out[kStaticRow * o + 0] = (o > 0 && nz > 0.0) ? sqrt(rel2 / nz) : 0.0;
    out[kStaticRow * o + 1] = o > 0 ? nz : 0.0;
    out[kStaticRow * o + 2] = en;
}

}  // namespace

extern "C" int anm_organ_summary_static(const float* d_sum, const float* d_sumsq, const uint8_t* d_labels, size_t n_voxels,
                                        int n_organs, double n_samples, double* d_out, void* cuda_stream,
                                        char* errbuf, size_t errbuf_len) {
    if (errbuf && errbuf_len) errbuf[0] = '\0';
    if (n_organs < 0 || n_organs > ANM_STATIC_MAX_ORGANS)
        return static_fail(errbuf, errbuf_len, ANM_E_ARG,
                           "organ summary (static scratch): n_organs = %d, but the built-in scratch array holds at most %d organs (%d bytes, fixed when the library was built)",
                           n_organs, ANM_STATIC_MAX_ORGANS, (int)(kStaticDoubles * sizeof(double)));
    if (!d_sum || !d_sumsq || !d_out) return static_fail(errbuf, errbuf_len, ANM_E_ARG, "organ summary (static scratch): d_sum, d_sumsq and d_out must not be NULL");
    if (n_organs > 0 && !d_labels) return static_fail(errbuf, errbuf_len, ANM_E_ARG, "organ summary (static scratch): n_organs = %d needs d_labels", n_organs);
    if (n_voxels == 0) return static_fail(errbuf, errbuf_len, ANM_E_ARG, "organ summary (static scratch): n_voxels = 0");
    if (!(n_samples >= 2.0)) return static_fail(errbuf, errbuf_len, ANM_E_ARG, "organ summary (static scratch): n_samples must be >= 2 (batches, or histories for history-by-history sums)");

    int device = -1;
    cudaError_t e = cudaGetDevice(&device);
    if (e != cudaSuccess) { cudaGetLastError(); return static_fail(errbuf, errbuf_len, ANM_E_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e)); }
    if (device < 0 || device >= kStaticMaxDevices) return static_fail(errbuf, errbuf_len, ANM_E_UNSUPPORTED, "organ summary (static scratch): device ordinal %d is beyond the %d this build keeps a scratch address for", device, kStaticMaxDevices);
    StaticDevice dev;
    e = static_setup(device, &dev);
    if (e != cudaSuccess) { cudaGetLastError(); return static_fail(errbuf, errbuf_len, ANM_E_CUDA, "cudaGetSymbolAddress(scratch) on device %d: %s", device, cudaGetErrorString(e)); }

    cudaStream_t st = (cudaStream_t)cuda_stream;
    // the array still holds the previous call's sums: everything the kernel adds into starts at zero again
    e = cudaMemsetAsync(dev.scratch, 0, kStaticDoubles * sizeof(double), st);
    if (e != cudaSuccess) { cudaGetLastError(); return static_fail(errbuf, errbuf_len, ANM_E_CUDA, "clearing the scratch: %s", cudaGetErrorString(e)); }
    const size_t want = (n_voxels + kStaticThreads - 1) / kStaticThreads, cap = (size_t)dev.num_sms * 8;
    const int blocks = (int)(want < cap ? want : cap);
    organ_summary_static_kernel<<<blocks, kStaticThreads, 0, st>>>(d_sum, d_sumsq, n_organs > 0 ? d_labels : nullptr, n_voxels, n_organs, n_samples, dev.scratch);
    e = cudaGetLastError();
    if (e != cudaSuccess) return static_fail(errbuf, errbuf_len, ANM_E_CUDA, "organ_summary_static_kernel: %s", cudaGetErrorString(e));
    organ_summary_emit_kernel<<<1, kStaticThreads, 0, st>>>(dev.scratch, d_out, n_organs);
    e = cudaGetLastError();
    if (e != cudaSuccess) return static_fail(errbuf, errbuf_len, ANM_E_CUDA, "organ_summary_emit_kernel: %s", cudaGetErrorString(e));
    return ANM_OK;
}
