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
    double inv_dhu[kMaxRampNodes];      // 1 / (hu[k+1] - hu[k])
    int material[kMaxRampNodes];
    double hu_outside;
    // density grid (readings C18, C30): texel counts = min(rint(rho * q_scale), q_cap) * q_mult
    // 2^-20 grid: 1048576, 16777215, 1;  2^-12 grid: 4096, 65535, 256 (the same word with its low 8 bits zero)
    double q_scale, q_cap, q_mult;
};

struct ResampleParams {
    int nx, ny, nz;          // destination (simulation) grid
    double dx, dy, dz;       // mm
    double inv_dx, inv_dy, inv_dz;
    int snx, sny, snz;       // source image
    double sdx, sdy, sdz;    // mm
    double inv_sdx, inv_sdy, inv_sdz;
    double ox, oy, oz;       // position of the source image's corner in the destination frame, mm
    double fill;             // value of the field outside the source image
    double scale;            // PET: voxel volume in mL
};

// One axis of a destination voxel [a, b): the source indices j0..j1 that overlap it (may be empty: j1 < j0) and their
// weights = overlap length / (b - a).  Only the first and the last source voxel can be cut by the destination voxel's
// faces; every one in between lies wholly inside it and weighs w_mid = sd / (b - a) (one number per axis).  `inside` =
// the fraction of [a, b) that lies inside the image.  The weights are separable, so the three tables (nx + ny + nz
// entries, filled on the host in fp64 by axis_overlap_table in anm_api.cu) are all the geometry the kernel needs:
// per voxel it loads three entries and streams the source voxels under it.
struct AxisOverlap {
    int j0, j1;
    double w_first, w_last, inside;
};

__device__ __forceinline__ double axis_w(const AxisOverlap& o, double w_mid, int j) {
    return j == o.j0 ? o.w_first : (j == o.j1 ? o.w_last : w_mid);
}

enum : int { RS_CT = 0, RS_PET = 1 };

// MODE RS_CT : out_texels[V] = material<<24 | round(rho 2^20);  max_mat = largest material id written
// MODE RS_PET: out_act[V] = mean Bq/mL x scale (fp32), also copied to out_copy if not null; total += sum (fp64);
//              flags bit 0 set if a source value under a destination voxel is negative or not finite
template <typename T, int MODE>
__global__ void __launch_bounds__(kResampleThreads)
resample_kernel(const T* __restrict__ src, const AxisOverlap* __restrict__ tab, const __grid_constant__ ResampleParams p, const __grid_constant__ RampParams ramp,
                uint32_t* __restrict__ out_texels, float* __restrict__ out_act, float* __restrict__ out_copy,
                double* __restrict__ total, unsigned* __restrict__ flags, unsigned* __restrict__ max_mat) {
    const double wmx = p.sdx * p.inv_dx, wmy = p.sdy * p.inv_dy, wmz = p.sdz * p.inv_dz;
    double local_total = 0.0;
    unsigned bad = 0, mm = 0;
    // a thread keeps its x column(s) and walks down the destination rows (iy, iz) its block owns: the X entry is loaded
    // once per column, the Y and Z entries of a row are block-uniform (broadcast loads, no index division)
    const unsigned rows = (unsigned)p.ny * (unsigned)p.nz;
    for (unsigned ux = threadIdx.x; ux < (unsigned)p.nx; ux += kResampleThreads) {
      const AxisOverlap X = tab[ux];
      for (unsigned row_id = blockIdx.x; row_id < rows; row_id += gridDim.x) {
        const unsigned uz = row_id / (unsigned)p.ny, uy = row_id - uz * (unsigned)p.ny;
        const AxisOverlap Y = tab[(unsigned)p.nx + uy];
        const AxisOverlap Z = tab[(unsigned)p.nx + (unsigned)p.ny + uz];
        const double inside_yz = Z.inside * Y.inside;
        const size_t idx = (size_t)row_id * (unsigned)p.nx + ux;
        double acc = 0.0;
        for (int c = Z.j0; c <= Z.j1; ++c) {
            const double wz = axis_w(Z, wmz, c);
            for (int b = Y.j0; b <= Y.j1; ++b) {
                const double wzy = wz * axis_w(Y, wmy, b);
                const T* row = src + ((size_t)c * p.sny + b) * (size_t)p.snx;
                double racc = 0.0;
                for (int a = X.j0; a <= X.j1; ++a) {
                    const double v = (double)__ldg(row + a);
                    if (MODE == RS_PET && !(v >= 0.0 && v < 1e300)) bad = 1;
                    racc = fma(axis_w(X, wmx, a), v, racc);
                }
                acc = fma(wzy, racc, acc);
            }
        }
        const double mean = acc + (1.0 - inside_yz * X.inside) * p.fill;
        if (MODE == RS_CT) {
            // HU -> (material, density): interval k with hu[k] <= mean < hu[k+1], clamped at both ends
            int k = 0;
#pragma unroll 1
            for (int n = 1; n < ramp.n_nodes - 1; ++n) if (mean >= ramp.hu[n]) k = n;
            const double hc = fmin(fmax(mean, ramp.hu[0]), ramp.hu[ramp.n_nodes - 1]);
            const double f = (hc - ramp.hu[k]) * ramp.inv_dhu[k];
            const double rho = ramp.rho[k] + f * (ramp.rho[k + 1] - ramp.rho[k]);
            const unsigned m = (unsigned)ramp.material[k];
            const double counts = fmin(rint(rho * ramp.q_scale), ramp.q_cap) * ramp.q_mult;
            out_texels[idx] = (m << 24) | (unsigned)counts;
            mm = max(mm, m);
        } else {
            const float a = (float)(mean * p.scale);
            out_act[idx] = a;
            if (out_copy) out_copy[idx] = a;
            local_total += mean * p.scale;
        }
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

// The same resample for the common geometry -- a destination voxel overlaps at most KX source voxels along x (KX = 2, 3
// or 4: image spacing >= half / a third of the grid's) and the image has < 2^31 voxels.  A thread owns one x column for
// the whole launch, so its x weights are computed ONCE and sit in registers (zero where the column overlaps fewer than
// KX voxels): the inner loop is KX loads and KX fp64 FMAs, branch-free; the y and z loops have block-uniform trip counts
// and weights; all indices are 32-bit.  Same arithmetic in the same order as resample_kernel (fp64 weights from the same
// host tables, fp64 accumulation x -> y -> z), so the two kernels agree bit for bit wherever both apply.
// Measured (CT 512 x 512 x 400 -> 256 x 256 x 400): 0.26 ms against 0.36 ms, 238 against 280 instructions per voxel; both
// are issue-bound by the fp64 weight selection, the per-row index arithmetic and the fp64 ramp.
template <typename T, int MODE, int KX>
__global__ void __launch_bounds__(kResampleThreads)
resample_fast_kernel(const T* __restrict__ src, const AxisOverlap* __restrict__ tab, const __grid_constant__ ResampleParams p,
                     const __grid_constant__ RampParams ramp, uint32_t* __restrict__ out_texels, float* __restrict__ out_act,
                     float* __restrict__ out_copy, double* __restrict__ total, unsigned* __restrict__ flags, unsigned* __restrict__ max_mat) {
    const double wmx = p.sdx * p.inv_dx, wmy = p.sdy * p.inv_dy, wmz = p.sdz * p.inv_dz;
    double local_total = 0.0;
    unsigned bad = 0, mm = 0;
    const unsigned rows = (unsigned)p.ny * (unsigned)p.nz;
    const unsigned snx = (unsigned)p.snx, sny = (unsigned)p.sny;
    for (unsigned ux = threadIdx.x; ux < (unsigned)p.nx; ux += kResampleThreads) {
        const AxisOverlap X = tab[ux];
        double wx[KX];
        unsigned off[KX];
#pragma unroll
        for (int k = 0; k < KX; ++k) {
            const int a = X.j0 + k;
            wx[k] = a <= X.j1 ? axis_w(X, wmx, a) : 0.0;
            off[k] = (unsigned)max(0, min(a, X.j1));             // a valid index even where the weight is zero
        }
        const bool none_x = X.j1 < X.j0;                         // the column lies outside the image
        for (unsigned row_id = blockIdx.x; row_id < rows; row_id += gridDim.x) {
            const unsigned uz = row_id / (unsigned)p.ny, uy = row_id - uz * (unsigned)p.ny;
            const AxisOverlap Y = tab[(unsigned)p.nx + uy];
            const AxisOverlap Z = tab[(unsigned)p.nx + (unsigned)p.ny + uz];
            const unsigned idx = row_id * (unsigned)p.nx + ux;
            double acc = 0.0;
            if (!none_x) {
                for (int c = Z.j0; c <= Z.j1; ++c) {
                    const double wz = axis_w(Z, wmz, c);
                    for (int b = Y.j0; b <= Y.j1; ++b) {
                        const double wzy = wz * axis_w(Y, wmy, b);
                        const T* row = src + ((unsigned)c * sny + (unsigned)b) * snx;
                        double racc = 0.0;
#pragma unroll
                        for (int k = 0; k < KX; ++k) {
                            const double v = (double)__ldg(row + off[k]);
                            if (MODE == RS_PET && wx[k] != 0.0 && !(v >= 0.0 && v < 1e300)) bad = 1;
                            racc = fma(wx[k], v, racc);
                        }
                        acc = fma(wzy, racc, acc);
                    }
                }
            }
            const double mean = acc + (1.0 - Z.inside * Y.inside * X.inside) * p.fill;
            if (MODE == RS_CT) {
                int k = 0;
#pragma unroll 1
                for (int n = 1; n < ramp.n_nodes - 1; ++n) if (mean >= ramp.hu[n]) k = n;
                const double hc = fmin(fmax(mean, ramp.hu[0]), ramp.hu[ramp.n_nodes - 1]);
                const double f = (hc - ramp.hu[k]) * ramp.inv_dhu[k];
                const double rho = ramp.rho[k] + f * (ramp.rho[k + 1] - ramp.rho[k]);
                const unsigned m = (unsigned)ramp.material[k];
                const double counts = fmin(rint(rho * ramp.q_scale), ramp.q_cap) * ramp.q_mult;
                out_texels[idx] = (m << 24) | (unsigned)counts;
                mm = max(mm, m);
            } else {
                const float a = (float)(mean * p.scale);
                out_act[idx] = a;
                if (out_copy) out_copy[idx] = a;
                local_total += mean * p.scale;
            }
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

// PET image already on the simulation grid (the paper's case: the CT is resampled to the PET grid, so the
// PET grid IS the simulation grid): the mean over a voxel is the voxel's own value, so the front end is one streaming
// pass  activity = Bq/mL x mL  with the fp64 block-reduced total and the same validation.  n4 = ceil(V / 4) float4s
// (the buffers are padded to a multiple of 4 by anm_set_grid; the padding of src is not read: tail handled by V).
__global__ void __launch_bounds__(kResampleThreads)
pet_same_grid_kernel(const float* __restrict__ src, double scale, float* __restrict__ out_act, float* __restrict__ out_copy,
                     size_t V, double* __restrict__ total, unsigned* __restrict__ flags) {
    double local_total = 0.0;
    unsigned bad = 0;
    const size_t n4 = V / 4;
    const bool aligned = ((reinterpret_cast<size_t>(src) | reinterpret_cast<size_t>(out_copy)) & 15u) == 0;
    const size_t stride = (size_t)gridDim.x * kResampleThreads, tid = (size_t)blockIdx.x * kResampleThreads + threadIdx.x;
    auto one = [&](float v) -> float {
        if (!(v >= 0.0f && v < 3.0e38f)) bad = 1;
        const double a = (double)v * scale;
        local_total += a;
        return (float)a;
    };
    size_t done = 0;
    if (aligned) {
        for (size_t i = tid; i < n4; i += stride) {
            const float4 v = __ldcs(reinterpret_cast<const float4*>(src) + i);
            const float4 a = make_float4(one(v.x), one(v.y), one(v.z), one(v.w));
            reinterpret_cast<float4*>(out_act)[i] = a;
            if (out_copy) reinterpret_cast<float4*>(out_copy)[i] = a;
        }
        done = n4 * 4;
    }
    for (size_t i = done + tid; i < V; i += stride) {
        const float a = one(src[i]);
        out_act[i] = a;
        if (out_copy) out_copy[i] = a;
    }
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
