// anm_frontend.cuh -- image front end of libanm.so: CT (HU) and PET
// (Bq/mL) images on their own grids -> the simulation grid's texels and activity volume.  Hand-written CUDA for
// sm_100a; no oracle code is shared.
//
//   resample_kernel<int16_t, CT>   "The CT images are resampled to obtain the same size as the PET images"
//                                  (PAPER.md:L81): volume-weighted mean of the piecewise-constant HU image over
//                                  every simulation voxel, then "converted into mass density and material composition
//                                  using the HU-to-density conversion curve": continuous piecewise-
//                                  linear density ramp, one material per HU interval -> packed texel.  One pass,
//                                  nothing but the texels is written.
//   resample_kernel<float, PET>    the same mean of the Bq/mL image, x voxel volume in mL = Bq per voxel ("linear
//                                  conversion of the PET value"); the block-reduced fp64 sum is the
//                                  whole-body activity A(t_s) of Eq. 1.
//
// Streaming and HBM-bound: every source voxel is read by the one or two destination voxels that overlap it (adjacent
// threads read adjacent source columns, the re-reads hit L1/L2), every destination voxel is written once.  The
// overlap weights and the accumulation are fp64 so that the HU -> material decision is taken on the same number the
// definition gives (the paper fixes no precision; a destination voxel sums at most a few dozen terms).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace anm {

constexpr int kMaxRampNodes = 16;
constexpr int kResampleThreads = 256;

struct RampParams {
    int n_nodes;
    double hu[kMaxRampNodes], rho[kMaxRampNodes];
    int material[kMaxRampNodes];
    double hu_outside;
};

struct ResampleParams {
    int nx, ny, nz;          // destination (simulation) grid
    double dx, dy, dz;       // mm
    int snx, sny, snz;       // source image
    double sdx, sdy, sdz;    // mm
    double ox, oy, oz;       // position of the source image's corner in the destination frame, mm
    double fill;             // value of the field outside the source image
    double scale;            // PET: voxel volume in mL
};

// One axis of a destination voxel [a, b): the source indices j0..j1 that overlap it (may be empty: j1 < j0) and their
// weights = overlap length / (b - a).  Only the first and the last source voxel can be cut by the destination voxel's
// faces; every one in between lies wholly inside it and weighs sd / (b - a).  `inside` = the fraction of [a, b) that
// lies inside the image.
struct AxisOverlap {
    int j0, j1;
    double w_first, w_mid, w_last, inside;
    __device__ __forceinline__ double w(int j) const { return j == j0 ? w_first : (j == j1 ? w_last : w_mid); }
};

__device__ __forceinline__ AxisOverlap axis_overlap(int i, double d, int sn, double sd, double off) {
    AxisOverlap o;
    const double a = (double)i * d, b = (double)(i + 1) * d, inv_d = 1.0 / d;
    o.j0 = max(0, (int)floor((a - off) / sd));
    o.j1 = min(sn - 1, (int)ceil((b - off) / sd) - 1);
    const double lo0 = off + (double)o.j0 * sd, hi0 = off + (double)(o.j0 + 1) * sd;
    const double lo1 = off + (double)o.j1 * sd, hi1 = off + (double)(o.j1 + 1) * sd;
    o.w_first = fmax(0.0, fmin(b, hi0) - fmax(a, lo0)) * inv_d;
    o.w_last = fmax(0.0, fmin(b, hi1) - fmax(a, lo1)) * inv_d;
    o.w_mid = sd * inv_d;
    o.inside = fmax(0.0, fmin(b, off + (double)sn * sd) - fmax(a, off)) * inv_d;
    return o;
}

enum : int { RS_CT = 0, RS_PET = 1 };

// MODE RS_CT : out_texels[V] = material<<24 | round(rho 2^20);  max_mat = largest material id written
// MODE RS_PET: out_act[V] = mean Bq/mL x scale (fp32), also copied to out_copy if not null; total += sum (fp64);
//              flags bit 0 set if a source value under a destination voxel is negative or not finite
template <typename T, int MODE>
__global__ void __launch_bounds__(kResampleThreads)
resample_kernel(const T* __restrict__ src, const __grid_constant__ ResampleParams p, const __grid_constant__ RampParams ramp,
                uint32_t* __restrict__ out_texels, float* __restrict__ out_act, float* __restrict__ out_copy,
                double* __restrict__ total, unsigned* __restrict__ flags, unsigned* __restrict__ max_mat) {
    const size_t V = (size_t)p.nx * p.ny * p.nz;
    double local_total = 0.0;
    unsigned bad = 0, mm = 0;
    for (size_t idx = (size_t)blockIdx.x * kResampleThreads + threadIdx.x; idx < V; idx += (size_t)gridDim.x * kResampleThreads) {
        const int ix = (int)(idx % (size_t)p.nx), iy = (int)((idx / (size_t)p.nx) % (size_t)p.ny), iz = (int)(idx / ((size_t)p.nx * p.ny));
        const AxisOverlap X = axis_overlap(ix, p.dx, p.snx, p.sdx, p.ox);
        const AxisOverlap Y = axis_overlap(iy, p.dy, p.sny, p.sdy, p.oy);
        const AxisOverlap Z = axis_overlap(iz, p.dz, p.snz, p.sdz, p.oz);
        double acc = 0.0;
        for (int c = Z.j0; c <= Z.j1; ++c) {
            const double wz = Z.w(c);
            for (int b = Y.j0; b <= Y.j1; ++b) {
                const double wzy = wz * Y.w(b);
                const T* row = src + ((size_t)c * p.sny + b) * (size_t)p.snx;
                double racc = 0.0;
                for (int a = X.j0; a <= X.j1; ++a) {
                    const double v = (double)__ldg(row + a);
                    if (MODE == RS_PET && !(v >= 0.0 && v < 1e300)) bad = 1;
                    racc = fma(X.w(a), v, racc);
                }
                acc = fma(wzy, racc, acc);
            }
        }
        const double mean = acc + (1.0 - Z.inside * Y.inside * X.inside) * p.fill;
        if (MODE == RS_CT) {
            // HU -> (material, density): interval k with hu[k] <= mean < hu[k+1], clamped at both ends
            int k = 0;
#pragma unroll 1
            for (int n = 1; n < ramp.n_nodes - 1; ++n) if (mean >= ramp.hu[n]) k = n;
            const double hc = fmin(fmax(mean, ramp.hu[0]), ramp.hu[ramp.n_nodes - 1]);
            const double f = (hc - ramp.hu[k]) / (ramp.hu[k + 1] - ramp.hu[k]);
            const double rho = ramp.rho[k] + f * (ramp.rho[k + 1] - ramp.rho[k]);
            const unsigned m = (unsigned)ramp.material[k];
            const double counts = fmin(rint(rho * 1048576.0), 16777215.0);
            out_texels[idx] = (m << 24) | (unsigned)counts;
            mm = max(mm, m);
        } else {
            const float a = (float)(mean * p.scale);
            out_act[idx] = a;
            if (out_copy) out_copy[idx] = a;
            local_total += mean * p.scale;
        }
    }
    if (MODE == RS_CT) {
        atomicMax(max_mat, mm);
    } else {
        __shared__ double s_tot[kResampleThreads / 32];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) local_total += __shfl_xor_sync(0xffffffffu, local_total, o);
        if ((threadIdx.x & 31) == 0) s_tot[threadIdx.x >> 5] = local_total;
        __syncthreads();
        if (threadIdx.x == 0) {
            double t = 0.0;
            for (int w = 0; w < kResampleThreads / 32; ++w) t += s_tot[w];
            if (t != 0.0) atomicAdd(total, t);
        }
        if (bad) atomicOr(flags, 1u);
    }
}

// inspection: texels -> material u8 + density f32
__global__ void __launch_bounds__(kResampleThreads)
unpack_texels_kernel(const uint32_t* __restrict__ texels, uint8_t* __restrict__ material, float* __restrict__ density, size_t V) {
    for (size_t i = (size_t)blockIdx.x * kResampleThreads + threadIdx.x; i < V; i += (size_t)gridDim.x * kResampleThreads) {
        const unsigned t = texels[i];
        material[i] = (uint8_t)(t >> 24);
        density[i] = (float)(t & 0xffffffu) * (1.0f / 1048576.0f);
    }
}

}  // namespace anm
