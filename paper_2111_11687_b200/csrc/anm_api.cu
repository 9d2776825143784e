// anm_api.cu -- host side of libanm.so: the C ABI of include/anm.h, device memory, set-up (texel packing,
// alias table, majorant) and the batch loop.  All arithmetic of the method runs in anm_kernels.cuh.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/anm.h"
#include "anm_kernels.cuh"
#include "anm_alias.cuh"
#include "anm_frontend.cuh"
#include "anm_peaks.cuh"

#include <cub/device/device_scan.cuh>
#include <cub/device/device_select.cuh>
#include <thrust/iterator/counting_iterator.h>
#include <thrust/iterator/transform_iterator.h>

using namespace anm;

namespace {

constexpr double kGyPerMeVPerGram = 1.602176634e-10;
constexpr uint64_t kBatchBudget = 4ull << 30;   // bytes of per-batch tallies in flight (anm_options.batches_per_launch = 0)
constexpr uint64_t kLaunchHistCap = 0xF0000000ull;   // histories one transport launch may cover (anm_options.batches_per_launch)
constexpr int kAutoSchedule = 2;   // anm_options.schedule = 0: the warp event pool (1.4x schedule 1 on cfg3, profiles/)

// Device buffers come from the device's default stream-ordered memory pool (its release threshold is raised in
// anm_create, so freed blocks stay cached in the process): creating and destroying contexts then costs microseconds
// instead of driver allocations of hundreds of MB.  alloc / release keep cudaMalloc / cudaFree semantics: the pointer
// is usable on any stream on return, and a release waits for the device like cudaFree does.
template <typename T>
struct DevBuf {
    T* p = nullptr;
    size_t n = 0;
    cudaError_t alloc(size_t count) {
        if (count == n && p) return cudaSuccess;
        release();
        if (count == 0) return cudaSuccess;
        cudaError_t e = cudaMallocAsync(reinterpret_cast<void**>(&p), count * sizeof(T), (cudaStream_t)0);
        if (e == cudaSuccess) e = cudaStreamSynchronize((cudaStream_t)0);
        if (e == cudaSuccess) n = count; else p = nullptr;
        return e;
    }
    void release(bool synced = false) {      // synced: the caller has just synchronised the device (anm_destroy frees ~30 buffers)
        if (p) { if (!synced) cudaDeviceSynchronize(); cudaFreeAsync(p, (cudaStream_t)0); }
        p = nullptr; n = 0;
    }
    // a local buffer is given back on every return path, the early error returns included
    DevBuf() = default;
    DevBuf(const DevBuf&) = delete;
    DevBuf& operator=(const DevBuf&) = delete;
    ~DevBuf() { release(); }
};

// cudaEvent_t locals that are destroyed on every return path
template <int N>
struct Events {
    cudaEvent_t e[N] = {};
    Events() = default;
    Events(const Events&) = delete;
    Events& operator=(const Events&) = delete;
    cudaError_t create() {
        for (auto& x : e) {
            const cudaError_t r = cudaEventCreate(&x);
            if (r != cudaSuccess) { x = nullptr; return r; }
        }
        return cudaSuccess;
    }
    ~Events() { for (auto x : e) if (x) cudaEventDestroy(x); }
};

}  // namespace

struct anm_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    std::string err;
    int num_sms = 0;

    // grid
    bool have_grid = false;
    int nx = 0, ny = 0, nz = 0;
    double dx = 0, dy = 0, dz = 0;        // cm
    double dx_mm = 0, dy_mm = 0, dz_mm = 0;   // as given to anm_set_grid
    size_t V = 0, Vpad = 0;

    // inputs
    bool have_phantom = false, have_source = false, have_tables = false, have_organs = false;
    bool point_source = false;
    double px = 0, py = 0, pz = 0;        // cm
    unsigned max_material = 0;
    unsigned rho_max_counts[ANM_MAX_MATERIALS] = {0};   // per material, in texel counts
    // hull box: voxel index range [lo, hi) enclosing every voxel denser than 5 % of the densest one, and the
    // per-material maximum density outside it; hull_ok = the box exists and is worth using (anm_options.hull_majorant)
    bool hull_ok = false;
    unsigned hull_lo[3] = {0, 0, 0}, hull_hi[3] = {0, 0, 0};
    unsigned rho_max_out_counts[ANM_MAX_MATERIALS] = {0};
    int n_organs = 0;
    anm_options opt;
    // tables (host copies)
    int nm = 0, ne = 0, n_x2 = 0;
    double lnE_min = 0, dlnE = 0;
    std::vector<float> mu_pe, mu_co, mu_ra, ray_x2, ray_cum;
    bool dev_tables_dirty = true;
    // electron tables (host copy + device)
    bool have_etables = false;
    int e_nm = 0, e_nt = 0;
    double e_tmin = 0, e_dt = 0;
    std::vector<float> e_range;

    // device memory
    DevBuf<uint32_t> texels;
    DevBuf<uint16_t> texels16;            // the same volume in 16 bits, valid iff tex16_ok (every voxel exactly representable)
    bool tex16_ok = false;
    DevBuf<float> batch, sum, sumsq, scratch;   // batch: [pipeline depth][batches per launch][Vpad] per-batch tallies
    bool batch_clean = false;             // `batch` holds zeros (the folds of a completed run leave it so)
    uint64_t batch_budget = kBatchBudget; // bytes of per-batch tallies a ctx may hold in flight (anm_set_tally_budget)
    size_t auto_group = 1;                // batches per launch that anm_set_grid found room for (<= the budget's figure)
    cudaEvent_t batch_zero_ev = nullptr;  // the memset of anm_set_grid (internal stream) has completed
    cudaStream_t pipe[3] = {nullptr, nullptr, nullptr};   // internal streams of the pipeline, created on first use
    DevBuf<float> e_ring;                 // waiting electrons of the event pool (electron_transport)
    DevBuf<float> hbh_sq;                 // [Vpad] sum over histories of X_h^2 (anm_options.uncertainty = 1)
    DevBuf<uint2> hbh_list;               // [(kHbhCap + 1) * hbh_nslots] per-slot deposit lists
    // tile-binned tally (anm_options.tally): per launch in flight the tiles' counters and deposit records; one table of
    // {offset, capacity} per tile; the device counter of deposits that overflowed their segment
    DevBuf<unsigned> bin_cnt;
    DevBuf<uint2> bin_seg, bin_seg0, bin_rec;
    DevBuf<unsigned long long> bin_ovf;
    bool run_hbh = false;                 // the last run scored history by history
    DevBuf<uint8_t> labels;
    DevBuf<uint4> alias;
    DevBuf<unsigned> counters;
    DevBuf<DeviceStats> dstats;
    DevBuf<double> organ_batch;           // [B][256]
    DevBuf<OrganAccum> organ_acc;         // [256]
    DevBuf<double> organ_mass;            // [256]
    DevBuf<unsigned long long> organ_count;   // [256]
    DevBuf<double> total_energy;          // [1] total energy, [1..4] run-level sigma accumulators, [5] maximum of S / rho (bits)
    DevBuf<float> d_tot, d_maj, d_majo, d_x2, d_cum, d_erange;
    DevBuf<float2> d_pec;
    DevBuf<unsigned> d_flags;             // [2 + ANM_MAX_MATERIALS] + [6 + ANM_MAX_MATERIALS] for the hull pass
    unsigned n_alias = 0;

    // results of the last run
    bool have_results = false;
    uint64_t run_decays = 0;
    int run_batches = 0;
    std::vector<anm_organ> organs;
    anm_stats stats;
    double run_sigma[5] = {0, 0, 0, 0, 0};   // rms > 10 %, n > 10 %, rms > 50 %, n > 50 %, max S / rho (last finalize)
    double ms_setup = 0, ms_load_ct = 0, ms_load_pet = 0;

    anm_ctx() { std::memset(&stats, 0, sizeof stats); anm_default_options(&opt); }
};

namespace {

int fail(anm_ctx* c, int code, const char* fmt, ...) {
    if (c) {
        char buf[512];
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(buf, sizeof buf, fmt, ap);
        va_end(ap);
        c->err = buf;
    }
    return code;
}

#define ANM_CUDA(c, call)                                                                         \
    do {                                                                                          \
        cudaError_t e_ = (call);                                                                  \
        if (e_ != cudaSuccess) {                                                                  \
            cudaGetLastError();                                                                   \
            return fail((c), e_ == cudaErrorMemoryAllocation ? ANM_E_NOMEM : ANM_E_CUDA,          \
                        "%s: %s", #call, cudaGetErrorString(e_));                                 \
        }                                                                                         \
    } while (0)

int grid_blocks(const anm_ctx* c, size_t items, int per_block) {
    const size_t want = (items + per_block - 1) / per_block;
    const size_t cap = (size_t)c->num_sms * 8;
    return (int)std::max<size_t>(1, std::min(want, cap));
}

// Alias table over the active voxels, built on the device (anm_alias.cuh): statistics pass, stable selection of the
// light / heavy voxel indices and prefix sums of their weights (CUB device primitives), one thread per bucket.
// d_act: activity[V] on the device.
int build_alias(anm_ctx* c, const float* d_act) {
    const size_t V = c->V;
    cudaStream_t st = c->stream;
    const int blocks = grid_blocks(c, V, kAliasThreads);
    DevBuf<double> bsum, L, H;
    DevBuf<unsigned long long> bcnt;
    DevBuf<uint32_t> lidx, hidx;
    DevBuf<unsigned char> temp;
    DevBuf<unsigned> nsel;
    struct Cleanup { DevBuf<double>&a, &b, &d; DevBuf<unsigned long long>& e; DevBuf<uint32_t>&f, &g; DevBuf<unsigned char>& h; DevBuf<unsigned>& i;
                     ~Cleanup() { a.release(); b.release(); d.release(); e.release(); f.release(); g.release(); h.release(); i.release(); } }
        cleanup{bsum, L, H, bcnt, lidx, hidx, temp, nsel};
    ANM_CUDA(c, bsum.alloc((size_t)blocks));
    ANM_CUDA(c, bcnt.alloc((size_t)blocks));
    ANM_CUDA(c, nsel.alloc(2));
    ANM_CUDA(c, cudaMemsetAsync(c->d_flags.p, 0, 4, st));
    activity_stats_kernel<<<blocks, kAliasThreads, 0, st>>>(d_act, V, bsum.p, bcnt.p, c->d_flags.p);
    ANM_CUDA(c, cudaGetLastError());
    std::vector<double> hs((size_t)blocks);
    std::vector<unsigned long long> hc((size_t)blocks);
    unsigned flags = 0;
    ANM_CUDA(c, cudaMemcpyAsync(hs.data(), bsum.p, (size_t)blocks * 8, cudaMemcpyDeviceToHost, st));
    ANM_CUDA(c, cudaMemcpyAsync(hc.data(), bcnt.p, (size_t)blocks * 8, cudaMemcpyDeviceToHost, st));
    ANM_CUDA(c, cudaMemcpyAsync(&flags, c->d_flags.p, 4, cudaMemcpyDeviceToHost, st));
    ANM_CUDA(c, cudaStreamSynchronize(st));
    if (flags & 1u) return fail(c, ANM_E_ARG, "activity holds a negative or non-finite value");
    double total = 0.0;
    unsigned long long M = 0;
    for (int b = 0; b < blocks; ++b) { total += hs[(size_t)b]; M += hc[(size_t)b]; }
    if (M == 0) return fail(c, ANM_E_ARG, "activity is zero everywhere");
    if (M > 0xfffffff0ull) return fail(c, ANM_E_ARG, "too many active voxels");
    const double scale = (double)M / total;

    // stable selection of the light (w <= 1) and heavy (w > 1) voxel indices
    ANM_CUDA(c, lidx.alloc((size_t)M));
    ANM_CUDA(c, hidx.alloc((size_t)M));
    thrust::counting_iterator<uint32_t> vox(0u);
    const AliasIsLight is_light{d_act, scale};
    const AliasIsHeavy is_heavy{d_act, scale};
    size_t tb1 = 0, tb2 = 0, tb3 = 0;
    const long long nV = (long long)V;
    ANM_CUDA(c, cub::DeviceSelect::If(nullptr, tb1, vox, lidx.p, nsel.p, nV, is_light, st));
    ANM_CUDA(c, cub::DeviceSelect::If(nullptr, tb2, vox, hidx.p, nsel.p + 1, nV, is_heavy, st));
    {   // scan scratch size: bounded by the larger of the two item counts (<= M)
        auto w = thrust::make_transform_iterator(thrust::counting_iterator<uint32_t>(0u), AliasWeight{d_act, lidx.p, scale});
        ANM_CUDA(c, cub::DeviceScan::InclusiveSum(nullptr, tb3, w, (double*)nullptr, (long long)M, st));
    }
    ANM_CUDA(c, temp.alloc(std::max(tb1, std::max(tb2, tb3))));
    size_t tb = temp.n;
    ANM_CUDA(c, cub::DeviceSelect::If(temp.p, tb, vox, lidx.p, nsel.p, nV, is_light, st));
    tb = temp.n;
    ANM_CUDA(c, cub::DeviceSelect::If(temp.p, tb, vox, hidx.p, nsel.p + 1, nV, is_heavy, st));
    unsigned n_lh[2] = {0, 0};
    ANM_CUDA(c, cudaMemcpyAsync(n_lh, nsel.p, 8, cudaMemcpyDeviceToHost, st));
    ANM_CUDA(c, cudaStreamSynchronize(st));
    const unsigned nl = n_lh[0], nh = n_lh[1];
    if ((unsigned long long)nl + nh != M) return fail(c, ANM_E_CUDA, "alias: selection counted %u + %u voxels, expected %llu", nl, nh, M);

    // exclusive prefix sums with the total in the last element: L[0..nl], H[0..nh]
    ANM_CUDA(c, L.alloc((size_t)nl + 1));
    ANM_CUDA(c, H.alloc((size_t)nh + 1));
    ANM_CUDA(c, cudaMemsetAsync(L.p, 0, 8, st));
    ANM_CUDA(c, cudaMemsetAsync(H.p, 0, 8, st));
    if (nl) {
        auto w = thrust::make_transform_iterator(thrust::counting_iterator<uint32_t>(0u), AliasWeight{d_act, lidx.p, scale});
        tb = temp.n;
        ANM_CUDA(c, cub::DeviceScan::InclusiveSum(temp.p, tb, w, L.p + 1, (long long)nl, st));
    }
    if (nh) {
        auto w = thrust::make_transform_iterator(thrust::counting_iterator<uint32_t>(0u), AliasWeight{d_act, hidx.p, scale});
        tb = temp.n;
        ANM_CUDA(c, cub::DeviceScan::InclusiveSum(temp.p, tb, w, H.p + 1, (long long)nh, st));
    }
    ANM_CUDA(c, c->alias.alloc((size_t)M));
    alias_build_kernel<<<(unsigned)((M + kAliasThreads - 1) / kAliasThreads), kAliasThreads, 0, st>>>(
        d_act, scale, lidx.p, hidx.p, L.p, H.p, nl, nh, c->alias.p);
    ANM_CUDA(c, cudaGetLastError());
    ANM_CUDA(c, cudaStreamSynchronize(st));
    c->n_alias = (unsigned)M;
    return ANM_OK;
}

// tot / {pe, pe+co} / majorant tables on the device, for the current options and phantom
int upload_tables(anm_ctx* c) {
    const int nm = c->nm, ne = c->ne;
    std::vector<float> tot((size_t)nm * ne), maj(ne), majo(ne);
    std::vector<float2> pec((size_t)nm * ne);
    for (int m = 0; m < nm; ++m)
        for (int k = 0; k < ne; ++k) {
            const size_t i = (size_t)m * ne + k;
            pec[i] = make_float2(c->mu_pe[i], c->mu_pe[i] + c->mu_co[i]);
            tot[i] = pec[i].y + (c->opt.rayleigh_on ? c->mu_ra[i] : 0.0f);
        }
    // majorant at the grid nodes: max over materials of rho_max,m * tot_m; linear interpolation of the node
    // maxima bounds every material's interpolated value, so it is a majorant at every energy
    for (int k = 0; k < ne; ++k) {
        float mx = 0.0f;
        for (int m = 0; m < nm; ++m) {
            const float rho = (float)c->rho_max_counts[m] * kDensityStep;
            mx = std::max(mx, rho * tot[(size_t)m * ne + k]);
        }
        maj[k] = mx * 1.000001f + 1e-30f;    // head-room for fp32 rounding of rho * lerp
        float mo = 0.0f;                     // the same bound over the voxels outside the hull box
        for (int m = 0; m < nm; ++m)
            mo = std::max(mo, (float)c->rho_max_out_counts[m] * kDensityStep * tot[(size_t)m * ne + k]);
        majo[k] = c->hull_ok ? mo * 1.000001f + 1e-30f : maj[k];
    }
    ANM_CUDA(c, c->d_tot.alloc(tot.size()));
    ANM_CUDA(c, c->d_pec.alloc(pec.size()));
    ANM_CUDA(c, c->d_maj.alloc(maj.size()));
    ANM_CUDA(c, c->d_majo.alloc(majo.size()));
    ANM_CUDA(c, c->d_x2.alloc(c->ray_x2.size()));
    ANM_CUDA(c, c->d_cum.alloc(c->ray_cum.size()));
    ANM_CUDA(c, cudaMemcpyAsync(c->d_tot.p, tot.data(), tot.size() * 4, cudaMemcpyHostToDevice, c->stream));
    ANM_CUDA(c, cudaMemcpyAsync(c->d_pec.p, pec.data(), pec.size() * 8, cudaMemcpyHostToDevice, c->stream));
    ANM_CUDA(c, cudaMemcpyAsync(c->d_maj.p, maj.data(), maj.size() * 4, cudaMemcpyHostToDevice, c->stream));
    ANM_CUDA(c, cudaMemcpyAsync(c->d_majo.p, majo.data(), majo.size() * 4, cudaMemcpyHostToDevice, c->stream));
    ANM_CUDA(c, cudaMemcpyAsync(c->d_x2.p, c->ray_x2.data(), c->ray_x2.size() * 4, cudaMemcpyHostToDevice, c->stream));
    ANM_CUDA(c, cudaMemcpyAsync(c->d_cum.p, c->ray_cum.data(), c->ray_cum.size() * 4, cudaMemcpyHostToDevice, c->stream));
    ANM_CUDA(c, cudaStreamSynchronize(c->stream));
    c->dev_tables_dirty = false;
    return ANM_OK;
}

void fill_run_sigma(const anm_ctx* c, anm_stats& s) {
    s.rms_rel_sigma_gt10 = c->run_sigma[0]; s.n_voxels_gt10 = (uint64_t)(c->run_sigma[1] + 0.5);
    s.rms_rel_sigma_gt50 = c->run_sigma[2]; s.n_voxels_gt50 = (uint64_t)(c->run_sigma[3] + 0.5);
    s.max_dose_Gy_per_decay = c->run_sigma[4];
}

using TransportFn = void (*)(const TransportParams);

// schedule 1 (history-based lanes) or 2 (warp-scope event pool), with / without counters; tally = TALLY_RED / _WAGG / _BINNED
TransportFn pick_transport(int schedule, bool stats, int tally, bool elec, bool hbh, bool t16) {
    if (schedule == 2) {
        if (t16 && !elec && !hbh && tally != TALLY_BINNED) {
            if (tally == TALLY_WAGG) return stats ? transport_pool_kernel<true, false, false, TALLY_WAGG, true> : transport_pool_kernel<false, false, false, TALLY_WAGG, true>;
            return stats ? transport_pool_kernel<true, false, false, TALLY_RED, true> : transport_pool_kernel<false, false, false, TALLY_RED, true>;
        }
        if (hbh) return elec ? (stats ? transport_pool_kernel<true, true, true> : transport_pool_kernel<false, true, true>)
                             : (stats ? transport_pool_kernel<true, false, true> : transport_pool_kernel<false, false, true>);
        if (elec) return stats ? transport_pool_kernel<true, true, false> : transport_pool_kernel<false, true, false>;
        if (tally == TALLY_WAGG) return stats ? transport_pool_kernel<true, false, false, TALLY_WAGG> : transport_pool_kernel<false, false, false, TALLY_WAGG>;
        if (tally == TALLY_BINNED) return stats ? transport_pool_kernel<true, false, false, TALLY_BINNED> : transport_pool_kernel<false, false, false, TALLY_BINNED>;
        return stats ? transport_pool_kernel<true, false, false> : transport_pool_kernel<false, false, false>;
    }
    return stats ? (tally == TALLY_WAGG ? transport_kernel<true, TALLY_WAGG> : transport_kernel<true, TALLY_RED>)
                 : (tally == TALLY_WAGG ? transport_kernel<false, TALLY_WAGG> : transport_kernel<false, TALLY_RED>);
}

// A11 on the current sum / sumsq volumes: finalize_kernel, then the organ arithmetic of SURVEY.md §8(c) step 7 on the
// host over the B x 256 fp64 organ rows (rows_host, or the ctx's own device rows when null):
// d_{o,b} = row[b][o] k / (n_b N_o); mean and batch sigma over b.  Fills c->organs and c->stats.deposited_MeV.
int finalize_and_collect(anm_ctx* c, int B, uint64_t nb, uint64_t n_decays, const double* rows_host) {
    cudaStream_t st = c->stream;
    ANM_CUDA(c, cudaMemsetAsync(c->organ_acc.p, 0, 256 * sizeof(OrganAccum), st));
    ANM_CUDA(c, cudaMemsetAsync(c->total_energy.p, 0, 6 * 8, st));
    finalize_kernel<<<grid_blocks(c, c->V, kFoldThreads), kFoldThreads, 0, st>>>(
        c->sum.p, c->run_hbh ? c->hbh_sq.p : c->sumsq.p, c->have_organs ? c->labels.p : nullptr, c->organ_acc.p,
        c->total_energy.p, c->n_organs, c->V, c->run_hbh ? (double)n_decays : (double)B);
    ANM_CUDA(c, cudaGetLastError());
    // run-level figure (reading C17): RMS relative sigma over the non-air voxels above 10 % / 50 % of the maximum dose
    dose_max_kernel<<<grid_blocks(c, c->V, kFoldThreads), kFoldThreads, 0, st>>>(
        c->sum.p, c->texels.p, c->V, reinterpret_cast<unsigned*>(c->total_energy.p + 5));
    ANM_CUDA(c, cudaGetLastError());
    run_sigma_kernel<<<grid_blocks(c, c->V, kFoldThreads), kFoldThreads, 0, st>>>(
        c->sum.p, c->run_hbh ? c->hbh_sq.p : c->sumsq.p, c->texels.p, c->V, c->run_hbh ? (double)n_decays : (double)B,
        reinterpret_cast<const unsigned*>(c->total_energy.p + 5), c->total_energy.p + 1);
    ANM_CUDA(c, cudaGetLastError());
    std::vector<double> ob;
    OrganAccum acc[256];
    double mass[256];
    unsigned long long cnt[256];
    double tot6[6] = {0, 0, 0, 0, 0, 0};
    ANM_CUDA(c, cudaMemcpyAsync(tot6, c->total_energy.p, sizeof tot6, cudaMemcpyDeviceToHost, st));
    if (c->have_organs) {
        if (!rows_host) {
            ob.resize((size_t)B * 256);
            ANM_CUDA(c, cudaMemcpyAsync(ob.data(), c->organ_batch.p, ob.size() * 8, cudaMemcpyDeviceToHost, st));
            rows_host = ob.data();
        }
        ANM_CUDA(c, cudaMemcpyAsync(acc, c->organ_acc.p, sizeof acc, cudaMemcpyDeviceToHost, st));
        ANM_CUDA(c, cudaMemcpyAsync(mass, c->organ_mass.p, sizeof mass, cudaMemcpyDeviceToHost, st));
        ANM_CUDA(c, cudaMemcpyAsync(cnt, c->organ_count.p, sizeof cnt, cudaMemcpyDeviceToHost, st));
    }
    ANM_CUDA(c, cudaStreamSynchronize(st));
    c->organs.assign((size_t)c->n_organs, anm_organ{});
    if (c->have_organs) {
        for (int o = 1; o <= c->n_organs; ++o) {
            anm_organ& r = c->organs[(size_t)o - 1];
            r.n_voxels = cnt[o];
            r.mass_g = mass[o];
            r.n_voxels_nonzero = (uint64_t)(acc[o].n_nonzero + 0.5);
            if (cnt[o] == 0) continue;
            double s1 = 0, s2 = 0;
            for (int b = 0; b < B; ++b) {
                const double d = rows_host[(size_t)b * 256 + o] * kGyPerMeVPerGram / ((double)nb * (double)cnt[o]);
                s1 += d; s2 += d * d;
            }
            const double mean = s1 / B;
            r.mean_Gy_per_decay = mean;
            r.sigma_mean = std::sqrt(std::max(0.0, (s2 / B - mean * mean) / (B - 1)));
            r.rms_voxel_rel_sigma = acc[o].n_nonzero > 0 ? std::sqrt(acc[o].rel2 / acc[o].n_nonzero) : 0.0;
            r.mass_weighted_Gy_per_decay = mass[o] > 0 ? acc[o].energy * kGyPerMeVPerGram / ((double)n_decays * mass[o]) : 0.0;
        }
    }
    c->stats.deposited_MeV = tot6[0];
    {
        unsigned bits; std::memcpy(&bits, &tot6[5], 4);
        float smax; std::memcpy(&smax, &bits, 4);
        c->run_sigma[0] = tot6[2] > 0 ? std::sqrt(tot6[1] / tot6[2]) : 0.0; c->run_sigma[1] = tot6[2];
        c->run_sigma[2] = tot6[4] > 0 ? std::sqrt(tot6[3] / tot6[4]) : 0.0; c->run_sigma[3] = tot6[4];
        c->run_sigma[4] = (double)smax * kGyPerMeVPerGram / ((double)n_decays * c->dx * c->dy * c->dz);
    }
    return ANM_OK;
}

}  // namespace

// =================================================================================================
extern "C" {

int anm_default_options(anm_options* o) {
    if (!o) return ANM_E_ARG;
    std::memset(o, 0, sizeof *o);
    o->n_batches = 100;
    o->photons_per_decay = 2;
    o->rayleigh_on = 1;
    o->photon_cutoff_MeV = 0.010;
    o->positron_ke_MeV = 0.0;
    o->schedule = 0;
    return ANM_OK;
}

int anm_create(anm_ctx** out, int cuda_device) {
    if (!out) return ANM_E_ARG;
    *out = nullptr;
    int count = 0;
    cudaError_t e = cudaGetDeviceCount(&count);
    if (e != cudaSuccess || cuda_device < 0 || cuda_device >= count) { cudaGetLastError(); return ANM_E_CUDA; }
    if (cudaSetDevice(cuda_device) != cudaSuccess) { cudaGetLastError(); return ANM_E_CUDA; }
    anm_ctx* c = new (std::nothrow) anm_ctx();
    if (!c) return ANM_E_NOMEM;
    c->device = cuda_device;
    // (one attribute query: cudaGetDeviceProperties fills the whole property struct and costs ~1 ms per context)
    if (cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, cuda_device) != cudaSuccess) { delete c; return ANM_E_CUDA; }
    {   // keep freed device memory cached in the default pool (see DevBuf)
        cudaMemPool_t pool;
        if (cudaDeviceGetDefaultMemPool(&pool, cuda_device) == cudaSuccess) {
            unsigned long long keep = ~0ull;
            cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        }
        cudaGetLastError();
    }
    *out = c;
    return ANM_OK;
}

int anm_destroy(anm_ctx* c) {
    if (!c) return ANM_OK;
    cudaSetDevice(c->device);
    cudaDeviceSynchronize();
    c->texels.release(true); c->texels16.release(true); c->batch.release(true); c->sum.release(true); c->sumsq.release(true); c->scratch.release(true);
    c->labels.release(true); c->alias.release(true); c->counters.release(true); c->dstats.release(true);
    c->organ_batch.release(true); c->organ_acc.release(true); c->organ_mass.release(true); c->organ_count.release(true);
    c->total_energy.release(true); c->d_tot.release(true); c->d_maj.release(true); c->d_majo.release(true); c->d_x2.release(true); c->d_cum.release(true);
    c->d_pec.release(true); c->d_flags.release(true); c->d_erange.release(true); c->e_ring.release(true); c->hbh_sq.release(true); c->hbh_list.release(true);
    c->bin_cnt.release(true); c->bin_seg.release(true); c->bin_seg0.release(true); c->bin_rec.release(true); c->bin_ovf.release(true);
    for (auto& ps : c->pipe) if (ps) { cudaStreamDestroy(ps); ps = nullptr; }
    if (c->batch_zero_ev) cudaEventDestroy(c->batch_zero_ev);
    delete c;
    return ANM_OK;
}

const char* anm_last_error(const anm_ctx* c) { return c ? c->err.c_str() : "null context"; }

int anm_set_stream(anm_ctx* c, void* cuda_stream) {
    if (!c) return ANM_E_ARG;
    c->stream = (cudaStream_t)cuda_stream;
    return ANM_OK;
}

int anm_set_tally_budget(anm_ctx* c, uint64_t bytes) {
    if (!c) return ANM_E_ARG;
    c->batch_budget = bytes == 0 ? kBatchBudget : bytes;
    return ANM_OK;
}

int anm_set_grid(anm_ctx* c, int nx, int ny, int nz, double dx_mm, double dy_mm, double dz_mm) {
    if (!c) return ANM_E_ARG;
    if (nx < 1 || ny < 1 || nz < 1 || !(dx_mm > 0) || !(dy_mm > 0) || !(dz_mm > 0) ||
        !std::isfinite(dx_mm) || !std::isfinite(dy_mm) || !std::isfinite(dz_mm))
        return fail(c, ANM_E_ARG, "grid: sizes must be >= 1 and spacings > 0");
    const unsigned long long V = (unsigned long long)nx * ny * nz;
    if (V > 0xfffffff0ull) return fail(c, ANM_E_ARG, "grid: more than 2^32 voxels");
    ANM_CUDA(c, cudaSetDevice(c->device));
    c->nx = nx; c->ny = ny; c->nz = nz;
    c->dx = dx_mm / 10.0; c->dy = dy_mm / 10.0; c->dz = dz_mm / 10.0;
    c->dx_mm = dx_mm; c->dy_mm = dy_mm; c->dz_mm = dz_mm;
    c->V = (size_t)V;
    c->Vpad = (c->V + 3) / 4 * 4;
    c->have_grid = true;
    c->have_phantom = c->have_organs = c->have_results = false;
    // a point source set for the previous grid stays only if it lies inside the new extents (else the decay voxel
    // would index past the volumes); an activity map never survives a grid change
    c->have_source = c->point_source && c->have_source && c->px >= 0 && c->px < nx * c->dx && c->py >= 0 &&
                     c->py < ny * c->dy && c->pz >= 0 && c->pz < nz * c->dz;
    if (!c->have_source) c->point_source = false;
    ANM_CUDA(c, c->texels.alloc(c->Vpad));
    ANM_CUDA(c, c->sum.alloc(c->Vpad));
    ANM_CUDA(c, c->sumsq.alloc(c->Vpad));
    ANM_CUDA(c, cudaMemsetAsync(c->texels.p, 0, c->Vpad * 4, c->stream));
    {   // per-batch tallies of the launches in flight (anm_options.batches_per_launch): the auto size -- 2 sets of as many
        // volumes as fit kBatchBudget -- is allocated here and zeroed on an internal stream, so that the memset overlaps
        // the uploads that follow; anm_run re-sizes it only when the options ask for more
        // If the device cannot give that much, the group is halved down to one volume per set before the call gives up
        // (ANM_E_NOMEM): a smaller group only costs launch tails, the results are the same.
        size_t g_auto = std::max<size_t>(1, std::min<size_t>(kMaxGroup, c->batch_budget / (c->Vpad * 4 * 2)));
        for (;;) {
            const cudaError_t e = c->batch.alloc(2 * g_auto * c->Vpad);
            if (e == cudaSuccess) break;
            cudaGetLastError();
            if (e != cudaErrorMemoryAllocation || g_auto == 1)
                return fail(c, e == cudaErrorMemoryAllocation ? ANM_E_NOMEM : ANM_E_CUDA, "grid: per-batch tallies (2 x %zu volumes of %zu bytes): %s",
                            g_auto, c->Vpad * 4, cudaGetErrorString(e));
            g_auto = (g_auto + 1) / 2;
        }
        c->auto_group = g_auto;
        if (!c->pipe[0]) ANM_CUDA(c, cudaStreamCreateWithFlags(&c->pipe[0], cudaStreamNonBlocking));
        if (!c->batch_zero_ev) ANM_CUDA(c, cudaEventCreateWithFlags(&c->batch_zero_ev, cudaEventDisableTiming));
        ANM_CUDA(c, cudaMemsetAsync(c->batch.p, 0, c->batch.n * 4, c->pipe[0]));
        ANM_CUDA(c, cudaEventRecord(c->batch_zero_ev, c->pipe[0]));
        c->batch_clean = true;
    }
    ANM_CUDA(c, c->d_flags.alloc(2 + ANM_MAX_MATERIALS + 6 + ANM_MAX_MATERIALS));
    ANM_CUDA(c, c->dstats.alloc(1));
    ANM_CUDA(c, c->total_energy.alloc(6));
    ANM_CUDA(c, c->organ_acc.alloc(256));
    ANM_CUDA(c, c->organ_mass.alloc(256));
    ANM_CUDA(c, c->organ_count.alloc(256));
    return ANM_OK;
}

static int phantom_setup(anm_ctx* c);

int anm_load_phantom(anm_ctx* c, const uint8_t* material, const float* density, int on_device) {
    if (!c) return ANM_E_ARG;
    if (!material || !density) return fail(c, ANM_E_ARG, "phantom: null pointer");
    if (!c->have_grid) return fail(c, ANM_E_STATE, "phantom: set the grid first");
    ANM_CUDA(c, cudaSetDevice(c->device));
    Events<2> evs;
    ANM_CUDA(c, evs.create());
    const cudaEvent_t e0 = evs.e[0], e1 = evs.e[1];
    ANM_CUDA(c, cudaEventRecord(e0, c->stream));
    const uint8_t* d_mat = material;
    const float* d_rho = density;
    DevBuf<uint8_t> stage_m;
    if (!on_device) {
        ANM_CUDA(c, stage_m.alloc(c->V));
        ANM_CUDA(c, c->scratch.alloc(c->Vpad));
        ANM_CUDA(c, cudaMemcpyAsync(stage_m.p, material, c->V, cudaMemcpyHostToDevice, c->stream));
        ANM_CUDA(c, cudaMemcpyAsync(c->scratch.p, density, c->V * 4, cudaMemcpyHostToDevice, c->stream));
        d_mat = stage_m.p; d_rho = c->scratch.p;
    }
    ANM_CUDA(c, cudaMemsetAsync(c->d_flags.p, 0, (2 + ANM_MAX_MATERIALS + 6 + ANM_MAX_MATERIALS) * 4, c->stream));
    pack_texels_kernel<<<grid_blocks(c, c->V, kFoldThreads), kFoldThreads, 0, c->stream>>>(
        d_mat, d_rho, c->texels.p, c->V, c->d_flags.p, c->d_flags.p + 1);
    ANM_CUDA(c, cudaGetLastError());
    unsigned flags[2] = {0, 0};
    ANM_CUDA(c, cudaMemcpyAsync(flags, c->d_flags.p, 8, cudaMemcpyDeviceToHost, c->stream));
    ANM_CUDA(c, cudaEventRecord(e1, c->stream));
    ANM_CUDA(c, cudaStreamSynchronize(c->stream));
    stage_m.release();
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    c->ms_setup += ms;
    c->have_phantom = false;
    if (flags[0] & 1u) return fail(c, ANM_E_ARG, "phantom: density must be finite and in [0, 16) g/cm^3");
    if (flags[1] >= ANM_MAX_MATERIALS) return fail(c, ANM_E_ARG, "phantom: material id %u >= %d", flags[1], ANM_MAX_MATERIALS);
    c->max_material = flags[1];
    return phantom_setup(c);
}

// after the texels are written and c->max_material is set: per-material maximum density, hull box (shared by
// anm_load_phantom and anm_load_ct)
static int phantom_setup(anm_ctx* c) {
    // per-material maximum density (texel counts): a second tiny pass on the host copy of the texels would cost a
    // D2H of the volume; instead reduce on the device with one atomicMax per (block, material)
    {
        rho_max_kernel<<<grid_blocks(c, c->V, kFoldThreads), kFoldThreads, 0, c->stream>>>(c->texels.p, c->V, c->d_flags.p + 2);
        ANM_CUDA(c, cudaGetLastError());
        // the 16-bit copy of the texels for the transport kernels' random reads (used when it is exact)
        unsigned not_exact = 1;
        ANM_CUDA(c, c->texels16.alloc(c->Vpad));
        ANM_CUDA(c, cudaMemsetAsync(c->d_flags.p, 0, 4, c->stream));
        pack_texels16_kernel<<<grid_blocks(c, c->V, kFoldThreads), kFoldThreads, 0, c->stream>>>(c->texels.p, c->texels16.p, c->V, c->d_flags.p);
        ANM_CUDA(c, cudaGetLastError());
        ANM_CUDA(c, cudaMemcpyAsync(c->rho_max_counts, c->d_flags.p + 2, ANM_MAX_MATERIALS * 4, cudaMemcpyDeviceToHost, c->stream));
        ANM_CUDA(c, cudaMemcpyAsync(&not_exact, c->d_flags.p, 4, cudaMemcpyDeviceToHost, c->stream));
        ANM_CUDA(c, cudaStreamSynchronize(c->stream));
        c->tex16_ok = (not_exact == 0);
        if (!c->tex16_ok) c->texels16.release();
    }
    {   // hull box: bounding box of the voxels denser than 5 % of the densest voxel; outside it the majorant is
        // that of the low-density margin (air around a patient).  Used only when the box is a proper part of the grid.
        unsigned rmax = 0;
        for (int m = 0; m < ANM_MAX_MATERIALS; ++m) rmax = std::max(rmax, c->rho_max_counts[m]);
        unsigned* d_box = c->d_flags.p + 2 + ANM_MAX_MATERIALS;
        const unsigned init[6] = {0xffffffffu, 0xffffffffu, 0xffffffffu, 0u, 0u, 0u};
        ANM_CUDA(c, cudaMemcpyAsync(d_box, init, sizeof init, cudaMemcpyHostToDevice, c->stream));
        hull_box_kernel<<<grid_blocks(c, (size_t)c->ny * c->nz, kFoldThreads / 32), kFoldThreads, 0, c->stream>>>(
            c->texels.p, c->nx, c->ny, c->nz, rmax / 20u, d_box);
        ANM_CUDA(c, cudaGetLastError());
        unsigned box[6];
        ANM_CUDA(c, cudaMemcpyAsync(box, d_box, sizeof box, cudaMemcpyDeviceToHost, c->stream));
        ANM_CUDA(c, cudaStreamSynchronize(c->stream));
        c->hull_ok = false;
        std::memset(c->rho_max_out_counts, 0, sizeof c->rho_max_out_counts);
        if (box[3] > box[0] && box[4] > box[1] && box[5] > box[2]) {
            const double vol = (double)(box[3] - box[0]) * (box[4] - box[1]) * (box[5] - box[2]);
            if (vol <= 0.9 * (double)c->V) {
                rho_max_outside_kernel<<<grid_blocks(c, c->V, kFoldThreads), kFoldThreads, 0, c->stream>>>(
                    c->texels.p, c->nx, c->ny, c->nz, box[0], box[1], box[2], box[3], box[4], box[5], d_box + 6);
                ANM_CUDA(c, cudaGetLastError());
                ANM_CUDA(c, cudaMemcpyAsync(c->rho_max_out_counts, d_box + 6, ANM_MAX_MATERIALS * 4, cudaMemcpyDeviceToHost, c->stream));
                ANM_CUDA(c, cudaStreamSynchronize(c->stream));
                for (int k = 0; k < 3; ++k) { c->hull_lo[k] = box[k]; c->hull_hi[k] = box[3 + k]; }
                c->hull_ok = true;
            }
        }
    }
    c->have_phantom = true;
    c->have_results = false;
    c->dev_tables_dirty = true;
    if (c->have_organs) c->have_organs = false;   // masses depend on the phantom: reload the labels
    return ANM_OK;
}

int anm_load_activity(anm_ctx* c, const float* activity, int on_device) {
    if (!c) return ANM_E_ARG;
    if (!activity) return fail(c, ANM_E_ARG, "activity: null pointer");
    if (!c->have_grid) return fail(c, ANM_E_STATE, "activity: set the grid first");
    ANM_CUDA(c, cudaSetDevice(c->device));
    const float* d_act = activity;
    if (!on_device) {
        ANM_CUDA(c, c->scratch.alloc(c->Vpad));
        ANM_CUDA(c, cudaMemcpyAsync(c->scratch.p, activity, c->V * 4, cudaMemcpyHostToDevice, c->stream));
        d_act = c->scratch.p;
    }
    c->have_source = false;
    Events<2> evs;
    ANM_CUDA(c, evs.create());
    const cudaEvent_t e0 = evs.e[0], e1 = evs.e[1];
    cudaEventRecord(e0, c->stream);
    int rc;
    try {
        rc = build_alias(c, d_act);
    } catch (const std::bad_alloc&) {
        rc = fail(c, ANM_E_NOMEM, "activity: host allocation failed");
    }
    cudaEventRecord(e1, c->stream);
    cudaEventSynchronize(e1);
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    c->ms_setup += ms;
    if (rc != ANM_OK) return rc;
    c->point_source = false;
    c->have_source = true;
    c->have_results = false;
    return ANM_OK;
}


// ---- image front end (anm_frontend.cuh) -----------------------------------------------

int anm_default_hu_ramp(anm_hu_ramp* r) {
    if (!r) return ANM_E_ARG;
    std::memset(r, 0, sizeof *r);
    // air / lung / soft tissue as water / compact bone; node values of the usual four-segment CT
    // ramp, restated from memory and therefore approximate (reading C27)
    const double hu[5] = {-1024.0, -974.0, -724.0, 101.0, 1976.0};
    const double rho[5] = {0.001, 0.044, 0.302, 1.101, 2.088};
    const int mat[4] = {0, 1, 2, 3};
    r->n_nodes = 5;
    for (int k = 0; k < 5; ++k) { r->hu[k] = hu[k]; r->rho[k] = rho[k]; }
    for (int k = 0; k < 4; ++k) r->material[k] = mat[k];
    r->hu_outside = -1024.0;
    return ANM_OK;
}

static int check_image_grid(anm_ctx* c, const char* what, int n0, int n1, int n2, double d0, double d1, double d2,
                            double o0, double o1, double o2) {
    if (n0 < 1 || n1 < 1 || n2 < 1 || !(d0 > 0) || !(d1 > 0) || !(d2 > 0) || !std::isfinite(d0) || !std::isfinite(d1) ||
        !std::isfinite(d2) || !std::isfinite(o0) || !std::isfinite(o1) || !std::isfinite(o2))
        return fail(c, ANM_E_ARG, "%s: image sizes must be >= 1, spacings > 0, offsets finite", what);
    if ((unsigned long long)n0 * n1 * n2 > 0x7fffffff0ull) return fail(c, ANM_E_ARG, "%s: image too large", what);
    return ANM_OK;
}

static ResampleParams resample_params(const anm_ctx* c, int n0, int n1, int n2, double d0, double d1, double d2,
                                      double o0, double o1, double o2, double fill, double scale) {
    ResampleParams p;
    p.nx = c->nx; p.ny = c->ny; p.nz = c->nz;
    p.dx = c->dx_mm; p.dy = c->dy_mm; p.dz = c->dz_mm;
    p.snx = n0; p.sny = n1; p.snz = n2; p.sdx = d0; p.sdy = d1; p.sdz = d2;
    p.inv_dx = 1.0 / p.dx; p.inv_dy = 1.0 / p.dy; p.inv_dz = 1.0 / p.dz;
    p.inv_sdx = 1.0 / d0; p.inv_sdy = 1.0 / d1; p.inv_sdz = 1.0 / d2;
    p.ox = o0; p.oy = o1; p.oz = o2; p.fill = fill; p.scale = scale;
    return p;
}

// The overlap geometry of one axis (anm_frontend.cuh): destination voxel i = [i d, (i+1) d) against the source voxels
// [off + j sd, off + (j+1) sd), j = 0..sn-1.  fp64 on the host; nx + ny + nz entries per image.
static void axis_overlap_table(AxisOverlap* out, int n, double d, int sn, double sd, double off) {
    for (int i = 0; i < n; ++i) {
        AxisOverlap o;
        const double a = (double)i * d, b = (double)(i + 1) * d;
        const double f0 = std::floor((a - off) / sd), f1 = std::ceil((b - off) / sd) - 1.0;
        o.j0 = (int)std::max(0.0, std::min(f0, (double)sn));          // may end up > j1: empty
        o.j1 = (int)std::min((double)(sn - 1), std::max(f1, -1.0));
        const double lo0 = off + (double)o.j0 * sd, hi0 = off + (double)(o.j0 + 1) * sd;
        const double lo1 = off + (double)o.j1 * sd, hi1 = off + (double)(o.j1 + 1) * sd;
        o.w_first = std::max(0.0, std::min(b, hi0) - std::max(a, lo0)) / d;
        o.w_last = std::max(0.0, std::min(b, hi1) - std::max(a, lo1)) / d;
        o.inside = std::max(0.0, std::min(b, off + (double)sn * sd) - std::max(a, off)) / d;
        out[i] = o;
    }
}

// one destination row (iy, iz) per block and trip; a few resident waves
static int resample_blocks(const anm_ctx* c) {
    return (int)std::max<size_t>(1, std::min<size_t>((size_t)c->ny * c->nz, (size_t)c->num_sms * 16));
}

// kx_max (if not null) = the largest number of source voxels a destination voxel overlaps along x
static int upload_overlap_tables(anm_ctx* c, const ResampleParams& p, DevBuf<AxisOverlap>& tab, int* kx_max = nullptr) {
    std::vector<AxisOverlap> h((size_t)p.nx + p.ny + p.nz);
    axis_overlap_table(h.data(), p.nx, p.dx, p.snx, p.sdx, p.ox);
    if (kx_max) { *kx_max = 0; for (int i = 0; i < p.nx; ++i) *kx_max = std::max(*kx_max, h[(size_t)i].j1 - h[(size_t)i].j0 + 1); }
    axis_overlap_table(h.data() + p.nx, p.ny, p.dy, p.sny, p.sdy, p.oy);
    axis_overlap_table(h.data() + p.nx + p.ny, p.nz, p.dz, p.snz, p.sdz, p.oz);
    ANM_CUDA(c, tab.alloc(h.size()));
    ANM_CUDA(c, cudaMemcpyAsync(tab.p, h.data(), h.size() * sizeof(AxisOverlap), cudaMemcpyHostToDevice, c->stream));
    ANM_CUDA(c, cudaStreamSynchronize(c->stream));     // h goes out of scope
    return ANM_OK;
}

int anm_load_ct(anm_ctx* c, const int16_t* hu, int cnx, int cny, int cnz, double cdx_mm, double cdy_mm, double cdz_mm,
                double ox_mm, double oy_mm, double oz_mm, const anm_hu_ramp* ramp, int on_device) {
    if (!c) return ANM_E_ARG;
    if (!hu) return fail(c, ANM_E_ARG, "ct: null pointer");
    if (!c->have_grid) return fail(c, ANM_E_STATE, "ct: set the grid first");
    { const int rc = check_image_grid(c, "ct", cnx, cny, cnz, cdx_mm, cdy_mm, cdz_mm, ox_mm, oy_mm, oz_mm); if (rc != ANM_OK) return rc; }
    anm_hu_ramp def;
    if (!ramp) { anm_default_hu_ramp(&def); ramp = &def; }
    if (ramp->n_nodes < 2 || ramp->n_nodes > ANM_MAX_RAMP_NODES) return fail(c, ANM_E_ARG, "ct: ramp needs 2..%d nodes", ANM_MAX_RAMP_NODES);
    RampParams rp;
    std::memset(&rp, 0, sizeof rp);
    rp.n_nodes = ramp->n_nodes;
    for (int k = 0; k < ramp->n_nodes; ++k) {
        if (!std::isfinite(ramp->hu[k]) || (k > 0 && !(ramp->hu[k] > ramp->hu[k - 1]))) return fail(c, ANM_E_ARG, "ct: ramp HU nodes must be finite and increase");
        if (!(ramp->rho[k] >= 0.0) || !(ramp->rho[k] < 16.0)) return fail(c, ANM_E_ARG, "ct: ramp densities must be in [0, 16) g/cm^3");
        if (k < ramp->n_nodes - 1 && (ramp->material[k] < 0 || ramp->material[k] >= ANM_MAX_MATERIALS)) return fail(c, ANM_E_ARG, "ct: ramp material id out of range");
        rp.hu[k] = ramp->hu[k]; rp.rho[k] = ramp->rho[k]; rp.material[k] = ramp->material[k];
    }
    if (!std::isfinite(ramp->hu_outside)) return fail(c, ANM_E_ARG, "ct: hu_outside must be finite");
    if (ramp->density_bits != 0 && ramp->density_bits != 12 && ramp->density_bits != 20) return fail(c, ANM_E_ARG, "ct: ramp density_bits must be 0 (= 20), 12 or 20");
    if (ramp->density_bits == 12) { rp.q_scale = 4096.0; rp.q_cap = 65535.0; rp.q_mult = 256.0; }
    else { rp.q_scale = 1048576.0; rp.q_cap = 16777215.0; rp.q_mult = 1.0; }
    rp.hu_outside = ramp->hu_outside;
    for (int k = 0; k + 1 < ramp->n_nodes; ++k) rp.inv_dhu[k] = 1.0 / (ramp->hu[k + 1] - ramp->hu[k]);
    ANM_CUDA(c, cudaSetDevice(c->device));
    const size_t n_src = (size_t)cnx * cny * cnz;
    DevBuf<int16_t> stage;
    const int16_t* d_src = hu;
    if (!on_device) {
        ANM_CUDA(c, stage.alloc(n_src));
        ANM_CUDA(c, cudaMemcpyAsync(stage.p, hu, n_src * 2, cudaMemcpyHostToDevice, c->stream));
        d_src = stage.p;
    }
    c->have_phantom = false;
    Events<2> evs;
    ANM_CUDA(c, evs.create());
    const cudaEvent_t e0 = evs.e[0], e1 = evs.e[1];
    ANM_CUDA(c, cudaMemsetAsync(c->d_flags.p, 0, (2 + ANM_MAX_MATERIALS + 6 + ANM_MAX_MATERIALS) * 4, c->stream));
    const ResampleParams p = resample_params(c, cnx, cny, cnz, cdx_mm, cdy_mm, cdz_mm, ox_mm, oy_mm, oz_mm, ramp->hu_outside, 1.0);
    DevBuf<AxisOverlap> tab;
    int kx = 0;
    { const int rc = upload_overlap_tables(c, p, tab, &kx); if (rc != ANM_OK) { stage.release(); tab.release(); return rc; } }
    ANM_CUDA(c, cudaEventRecord(e0, c->stream));
    // resample_fast_kernel where a destination voxel overlaps <= 4 source voxels along x and the image indexes in 32 bits
    const bool fast = n_src < 0x7fffffffull && kx <= 4;
#define ANM_RS_ARGS d_src, tab.p, p, rp, c->texels.p, nullptr, nullptr, nullptr, c->d_flags.p, c->d_flags.p + 1
    if (fast && kx <= 2) resample_fast_kernel<int16_t, RS_CT, 2><<<resample_blocks(c), kResampleThreads, 0, c->stream>>>(ANM_RS_ARGS);
    else if (fast && kx == 3) resample_fast_kernel<int16_t, RS_CT, 3><<<resample_blocks(c), kResampleThreads, 0, c->stream>>>(ANM_RS_ARGS);
    else if (fast) resample_fast_kernel<int16_t, RS_CT, 4><<<resample_blocks(c), kResampleThreads, 0, c->stream>>>(ANM_RS_ARGS);
    else resample_kernel<int16_t, RS_CT><<<resample_blocks(c), kResampleThreads, 0, c->stream>>>(ANM_RS_ARGS);
#undef ANM_RS_ARGS
    ANM_CUDA(c, cudaGetLastError());
    ANM_CUDA(c, cudaEventRecord(e1, c->stream));
    unsigned flags[2] = {0, 0};
    ANM_CUDA(c, cudaMemcpyAsync(flags, c->d_flags.p, 8, cudaMemcpyDeviceToHost, c->stream));
    ANM_CUDA(c, cudaStreamSynchronize(c->stream));
    stage.release(); tab.release();
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    c->ms_setup += ms; c->ms_load_ct = ms;
    c->max_material = flags[1];
    return phantom_setup(c);
}

int anm_get_phantom(anm_ctx* c, uint8_t* material, float* density, size_t n, int on_device) {
    if (!c) return ANM_E_ARG;
    if (!material || !density) return fail(c, ANM_E_ARG, "get_phantom: null pointer");
    if (!c->have_phantom) return fail(c, ANM_E_STATE, "get_phantom: no phantom loaded");
    if (n != c->V) return fail(c, ANM_E_ARG, "get_phantom: n = %zu but the grid has %zu voxels", n, c->V);
    ANM_CUDA(c, cudaSetDevice(c->device));
    DevBuf<uint8_t> dm;
    DevBuf<float> dr;
    uint8_t* pm = material; float* pr = density;
    if (!on_device) { ANM_CUDA(c, dm.alloc(c->V)); ANM_CUDA(c, dr.alloc(c->V)); pm = dm.p; pr = dr.p; }
    unpack_texels_kernel<<<grid_blocks(c, c->V, kResampleThreads), kResampleThreads, 0, c->stream>>>(c->texels.p, pm, pr, c->V);
    ANM_CUDA(c, cudaGetLastError());
    if (!on_device) {
        ANM_CUDA(c, cudaMemcpyAsync(material, pm, c->V, cudaMemcpyDeviceToHost, c->stream));
        ANM_CUDA(c, cudaMemcpyAsync(density, pr, c->V * 4, cudaMemcpyDeviceToHost, c->stream));
    }
    ANM_CUDA(c, cudaStreamSynchronize(c->stream));
    dm.release(); dr.release();
    return ANM_OK;
}

int anm_load_pet(anm_ctx* c, const float* bq_per_ml, int pnx, int pny, int pnz, double pdx_mm, double pdy_mm, double pdz_mm,
                 double ox_mm, double oy_mm, double oz_mm, int on_device, double* total_activity_Bq,
                 float* out_activity_Bq, size_t n) {
    if (!c) return ANM_E_ARG;
    if (!bq_per_ml) return fail(c, ANM_E_ARG, "pet: null pointer");
    if (!c->have_grid) return fail(c, ANM_E_STATE, "pet: set the grid first");
    if (out_activity_Bq && n != c->V) return fail(c, ANM_E_ARG, "pet: n = %zu but the grid has %zu voxels", n, c->V);
    { const int rc = check_image_grid(c, "pet", pnx, pny, pnz, pdx_mm, pdy_mm, pdz_mm, ox_mm, oy_mm, oz_mm); if (rc != ANM_OK) return rc; }
    ANM_CUDA(c, cudaSetDevice(c->device));
    const size_t n_src = (size_t)pnx * pny * pnz;
    DevBuf<float> stage;
    DevBuf<double> d_total;
    const float* d_src = bq_per_ml;
    if (!on_device) {
        ANM_CUDA(c, stage.alloc(n_src));
        ANM_CUDA(c, cudaMemcpyAsync(stage.p, bq_per_ml, n_src * 4, cudaMemcpyHostToDevice, c->stream));
        d_src = stage.p;
    }
    ANM_CUDA(c, c->scratch.alloc(c->Vpad));
    ANM_CUDA(c, d_total.alloc(1));
    ANM_CUDA(c, cudaMemsetAsync(d_total.p, 0, 8, c->stream));
    ANM_CUDA(c, cudaMemsetAsync(c->d_flags.p, 0, 8, c->stream));
    c->have_source = false;
    Events<3> evs;
    ANM_CUDA(c, evs.create());
    const cudaEvent_t e0 = evs.e[0], e1 = evs.e[1], e2 = evs.e[2];
    const double vox_ml = c->dx * c->dy * c->dz;     // cm^3 = mL
    const ResampleParams p = resample_params(c, pnx, pny, pnz, pdx_mm, pdy_mm, pdz_mm, ox_mm, oy_mm, oz_mm, 0.0, vox_ml);
    RampParams rp;
    std::memset(&rp, 0, sizeof rp);
    float* d_copy = (out_activity_Bq && on_device) ? out_activity_Bq : nullptr;
    DevBuf<AxisOverlap> tab;
    const bool same_grid = pnx == c->nx && pny == c->ny && pnz == c->nz && ox_mm == 0.0 && oy_mm == 0.0 && oz_mm == 0.0 &&
                           pdx_mm == p.dx && pdy_mm == p.dy && pdz_mm == p.dz;
    if (same_grid) {     // the PET grid is the simulation grid -> one streaming pass
        cudaEventRecord(e0, c->stream);
        pet_same_grid_kernel<<<grid_blocks(c, c->V / 4 + 1, kResampleThreads), kResampleThreads, 0, c->stream>>>(
            d_src, vox_ml, c->scratch.p, d_copy, c->V, d_total.p, c->d_flags.p);
    } else {
        int kx = 0;
        { const int rc = upload_overlap_tables(c, p, tab, &kx); if (rc != ANM_OK) { stage.release(); tab.release(); d_total.release(); return rc; } }
        cudaEventRecord(e0, c->stream);
        const bool fast = (unsigned long long)pnx * pny * pnz < 0x7fffffffull && kx <= 4;
#define ANM_RS_ARGS d_src, tab.p, p, rp, nullptr, c->scratch.p, d_copy, d_total.p, c->d_flags.p, c->d_flags.p + 1
        if (fast && kx <= 2) resample_fast_kernel<float, RS_PET, 2><<<resample_blocks(c), kResampleThreads, 0, c->stream>>>(ANM_RS_ARGS);
        else if (fast && kx == 3) resample_fast_kernel<float, RS_PET, 3><<<resample_blocks(c), kResampleThreads, 0, c->stream>>>(ANM_RS_ARGS);
        else if (fast) resample_fast_kernel<float, RS_PET, 4><<<resample_blocks(c), kResampleThreads, 0, c->stream>>>(ANM_RS_ARGS);
        else resample_kernel<float, RS_PET><<<resample_blocks(c), kResampleThreads, 0, c->stream>>>(ANM_RS_ARGS);
#undef ANM_RS_ARGS
    }
    ANM_CUDA(c, cudaGetLastError());
    cudaEventRecord(e1, c->stream);
    unsigned flags = 0;
    double total = 0.0;
    ANM_CUDA(c, cudaMemcpyAsync(&flags, c->d_flags.p, 4, cudaMemcpyDeviceToHost, c->stream));
    ANM_CUDA(c, cudaMemcpyAsync(&total, d_total.p, 8, cudaMemcpyDeviceToHost, c->stream));
    if (out_activity_Bq && !on_device)
        ANM_CUDA(c, cudaMemcpyAsync(out_activity_Bq, c->scratch.p, c->V * 4, cudaMemcpyDeviceToHost, c->stream));
    ANM_CUDA(c, cudaStreamSynchronize(c->stream));
    stage.release(); d_total.release(); tab.release();
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    c->ms_load_pet = ms;
    if (flags & 1u) return fail(c, ANM_E_ARG, "pet: values must be finite and >= 0");
    int rc;
    try {
        rc = build_alias(c, c->scratch.p);
    } catch (const std::bad_alloc&) {
        rc = fail(c, ANM_E_NOMEM, "pet: host allocation failed");
    }
    cudaEventRecord(e2, c->stream);
    cudaEventSynchronize(e2);
    cudaEventElapsedTime(&ms, e0, e2);
    c->ms_setup += ms;
    if (rc != ANM_OK) return rc;
    if (total_activity_Bq) *total_activity_Bq = total;
    c->point_source = false;
    c->have_source = true;
    c->have_results = false;
    return ANM_OK;
}

int anm_set_point_source(anm_ctx* c, double x_mm, double y_mm, double z_mm) {
    if (!c) return ANM_E_ARG;
    if (!c->have_grid) return fail(c, ANM_E_STATE, "point source: set the grid first");
    const double x = x_mm / 10.0, y = y_mm / 10.0, z = z_mm / 10.0;
    if (!(x >= 0 && x < c->nx * c->dx && y >= 0 && y < c->ny * c->dy && z >= 0 && z < c->nz * c->dz))
        return fail(c, ANM_E_ARG, "point source outside the grid");
    c->px = x; c->py = y; c->pz = z;
    c->point_source = true;
    c->have_source = true;
    c->have_results = false;
    return ANM_OK;
}

int anm_load_organs(anm_ctx* c, const uint8_t* labels, int n_organs, int on_device) {
    if (!c) return ANM_E_ARG;
    if (!labels) return fail(c, ANM_E_ARG, "organs: null pointer");
    if (n_organs < 1 || n_organs > ANM_MAX_ORGANS) return fail(c, ANM_E_ARG, "organs: n_organs must be 1..%d", ANM_MAX_ORGANS);
    if (!c->have_phantom) return fail(c, ANM_E_STATE, "organs: load the phantom first (organ masses need it)");
    ANM_CUDA(c, cudaSetDevice(c->device));
    ANM_CUDA(c, c->labels.alloc(c->Vpad));
    ANM_CUDA(c, cudaMemsetAsync(c->labels.p, 0, c->Vpad, c->stream));
    ANM_CUDA(c, cudaMemcpyAsync(c->labels.p, labels, c->V, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, c->stream));
    ANM_CUDA(c, cudaMemsetAsync(c->organ_mass.p, 0, 256 * 8, c->stream));
    ANM_CUDA(c, cudaMemsetAsync(c->organ_count.p, 0, 256 * 8, c->stream));
    organ_mass_kernel<<<grid_blocks(c, c->V, kFoldThreads), kFoldThreads, 0, c->stream>>>(
        c->labels.p, c->texels.p, c->organ_mass.p, c->organ_count.p, c->V, (float)(c->dx * c->dy * c->dz));
    ANM_CUDA(c, cudaGetLastError());
    unsigned long long cnt[256];
    ANM_CUDA(c, cudaMemcpyAsync(cnt, c->organ_count.p, sizeof cnt, cudaMemcpyDeviceToHost, c->stream));
    ANM_CUDA(c, cudaStreamSynchronize(c->stream));
    c->have_organs = false;
    for (int l = n_organs + 1; l < 256; ++l)
        if (cnt[l]) return fail(c, ANM_E_ARG, "organs: label %d > n_organs = %d", l, n_organs);
    c->n_organs = n_organs;
    c->have_organs = true;
    c->have_results = false;
    return ANM_OK;
}

int anm_set_physics_tables(anm_ctx* c, const anm_tables* t) {
    if (!c) return ANM_E_ARG;
    if (!t || !t->mu_pe || !t->mu_compton || !t->mu_rayleigh || !t->ray_x2 || !t->ray_cum)
        return fail(c, ANM_E_ARG, "tables: null pointer");
    if (t->n_materials < 1 || t->n_materials > ANM_MAX_MATERIALS || t->n_energy < 2 || t->n_energy > 1024 ||
        t->n_x2 < 2 || t->n_x2 > 1024 || !(t->dlnE > 0) || !std::isfinite(t->lnE_min))
        return fail(c, ANM_E_ARG, "tables: sizes out of range");
    const size_t n = (size_t)t->n_materials * t->n_energy;
    for (size_t i = 0; i < n; ++i)
        if (!(t->mu_pe[i] > 0) || !(t->mu_compton[i] > 0) || !(t->mu_rayleigh[i] > 0) ||
            !std::isfinite(t->mu_pe[i]) || !std::isfinite(t->mu_compton[i]) || !std::isfinite(t->mu_rayleigh[i]))
            return fail(c, ANM_E_ARG, "tables: coefficients must be finite and > 0");
    if (t->ray_x2[0] != 0.0f) return fail(c, ANM_E_ARG, "tables: ray_x2[0] must be 0");
    for (int i = 1; i < t->n_x2; ++i)
        if (!(t->ray_x2[i] > t->ray_x2[i - 1])) return fail(c, ANM_E_ARG, "tables: ray_x2 must increase");
    for (int m = 0; m < t->n_materials; ++m)
        for (int i = 1; i < t->n_x2; ++i)
            if (!(t->ray_cum[(size_t)m * t->n_x2 + i] >= t->ray_cum[(size_t)m * t->n_x2 + i - 1]))
                return fail(c, ANM_E_ARG, "tables: ray_cum must be non-decreasing");
    const double e_hi = std::exp(t->lnE_min + t->dlnE * (t->n_energy - 1));
    if (e_hi < 0.51099895) return fail(c, ANM_E_ARG, "tables: energy grid must reach 0.51099895 MeV");
    const double xm = 0.51099895 * 1000.0 / 12.398419843;
    if (t->ray_x2[t->n_x2 - 1] < xm * xm) return fail(c, ANM_E_ARG, "tables: ray_x2 must reach (E0/hc)^2");
    try {
        c->nm = t->n_materials; c->ne = t->n_energy; c->n_x2 = t->n_x2;
        c->lnE_min = t->lnE_min; c->dlnE = t->dlnE;
        c->mu_pe.assign(t->mu_pe, t->mu_pe + n);
        c->mu_co.assign(t->mu_compton, t->mu_compton + n);
        c->mu_ra.assign(t->mu_rayleigh, t->mu_rayleigh + n);
        c->ray_x2.assign(t->ray_x2, t->ray_x2 + t->n_x2);
        c->ray_cum.assign(t->ray_cum, t->ray_cum + (size_t)t->n_materials * t->n_x2);
    } catch (const std::bad_alloc&) {
        return fail(c, ANM_E_NOMEM, "tables: host allocation failed");
    }
    c->have_tables = true;
    c->dev_tables_dirty = true;
    c->have_results = false;
    return ANM_OK;
}

// electron part of the kernel parameters (zeros when no tables are set)
static void fill_electron_params(const anm_ctx* c, TransportParams& p) {
    p.e_range = c->have_etables ? c->d_erange.p : nullptr;
    p.n_t = c->e_nt; p.e_nm = c->e_nm;
    p.t_min = (float)c->e_tmin; p.e_dt = (float)c->e_dt; p.e_inv_dt = c->e_dt > 0 ? (float)(1.0 / c->e_dt) : 0.0f;
}

int anm_set_electron_tables(anm_ctx* c, const anm_electron_tables* t) {
    if (!c) return ANM_E_ARG;
    if (!t || !t->range) return fail(c, ANM_E_ARG, "electron tables: null pointer");
    if (t->n_materials < 1 || t->n_materials > ANM_MAX_MATERIALS || t->n_t < 2 || t->n_t > 1024 || !(t->dt > 0) ||
        !(t->t_min > 0) || !std::isfinite(t->t_min) || !std::isfinite(t->dt))
        return fail(c, ANM_E_ARG, "electron tables: sizes out of range");
    // photo-electrons take the whole photon energy (reading C28), so the grid must cover E0, not only the Compton edge
    if (t->t_min + t->dt * (t->n_t - 1) < 0.51099895) return fail(c, ANM_E_ARG, "electron tables: the grid must reach the photon energy 0.51099895 MeV (photo-electrons)");
    for (int m = 0; m < t->n_materials; ++m) {
        const float* R = t->range + (size_t)m * t->n_t;
        if (R[0] != 0.0f) return fail(c, ANM_E_ARG, "electron tables: range[m][0] must be 0 (t_min is the cutoff)");
        for (int k = 1; k < t->n_t; ++k)
            if (!(R[k] > R[k - 1]) || !std::isfinite(R[k])) return fail(c, ANM_E_ARG, "electron tables: range must increase strictly");
    }
    ANM_CUDA(c, cudaSetDevice(c->device));
    try { c->e_range.assign(t->range, t->range + (size_t)t->n_materials * t->n_t); }
    catch (const std::bad_alloc&) { return fail(c, ANM_E_NOMEM, "electron tables: host allocation failed"); }
    c->e_nm = t->n_materials; c->e_nt = t->n_t; c->e_tmin = t->t_min; c->e_dt = t->dt;
    ANM_CUDA(c, c->d_erange.alloc(c->e_range.size()));
    ANM_CUDA(c, cudaMemcpyAsync(c->d_erange.p, c->e_range.data(), c->e_range.size() * 4, cudaMemcpyHostToDevice, c->stream));
    ANM_CUDA(c, cudaStreamSynchronize(c->stream));
    c->have_etables = true;
    c->have_results = false;
    return ANM_OK;
}

int anm_philox_blocks(anm_ctx* c, uint64_t seed, const uint32_t* counters, size_t n, uint32_t* out) {
    if (!c) return ANM_E_ARG;
    if (!counters || !out || n == 0 || n > (1u << 24)) return fail(c, ANM_E_ARG, "philox: null pointer or bad count");
    ANM_CUDA(c, cudaSetDevice(c->device));
    DevBuf<uint4> d_in, d_out;
    struct Rel { DevBuf<uint4>&a, &b; ~Rel() { a.release(); b.release(); } } rel{d_in, d_out};
    ANM_CUDA(c, d_in.alloc(n));
    ANM_CUDA(c, d_out.alloc(n));
    ANM_CUDA(c, cudaMemcpyAsync(d_in.p, counters, n * 16, cudaMemcpyHostToDevice, c->stream));
    TransportParams p;
    std::memset(&p, 0, sizeof p);
    for (int r = 0; r < 10; ++r) {      // the same round keys anm_run sets
        p.rk[2 * r] = (unsigned)seed + (unsigned)r * 0x9E3779B9u;
        p.rk[2 * r + 1] = (unsigned)(seed >> 32) + (unsigned)r * 0xBB67AE85u;
    }
    philox_probe_kernel<<<(unsigned)((n + 127) / 128), 128, 0, c->stream>>>(p, d_in.p, d_out.p, (unsigned)n);
    ANM_CUDA(c, cudaGetLastError());
    ANM_CUDA(c, cudaMemcpyAsync(out, d_out.p, n * 16, cudaMemcpyDeviceToHost, c->stream));
    ANM_CUDA(c, cudaStreamSynchronize(c->stream));
    return ANM_OK;
}

int anm_trace_electrons(anm_ctx* c, const float* electrons, size_t n, float* out_MeV, size_t n_voxels, double* escaped_MeV) {
    if (!c) return ANM_E_ARG;
    if (!electrons || !out_MeV || !escaped_MeV || n == 0 || n > 0x7fffffffu) return fail(c, ANM_E_ARG, "trace: null pointer or bad count");
    if (!c->have_grid || !c->have_phantom || !c->have_etables) return fail(c, ANM_E_STATE, "trace: need grid, phantom and electron tables");
    if (n_voxels != c->V) return fail(c, ANM_E_ARG, "trace: n_voxels = %zu but the grid has %zu voxels", n_voxels, c->V);
    if ((int)c->max_material >= c->e_nm) return fail(c, ANM_E_ARG, "trace: phantom uses material %u but the electron tables hold %d", c->max_material, c->e_nm);
    std::vector<float> in(electrons, electrons + 7 * n);
    for (size_t i = 0; i < n; ++i) {
        float* e = in.data() + 7 * i;
        e[0] *= 0.1f; e[1] *= 0.1f; e[2] *= 0.1f;       // mm -> cm
        if (!(e[0] >= 0 && e[0] < c->nx * c->dx && e[1] >= 0 && e[1] < c->ny * c->dy && e[2] >= 0 && e[2] < c->nz * c->dz))
            return fail(c, ANM_E_ARG, "trace: electron %zu starts outside the grid", i);
        if (!(e[6] > c->e_tmin) || !(e[6] <= c->e_tmin + c->e_dt * (c->e_nt - 1))) return fail(c, ANM_E_ARG, "trace: electron %zu energy outside the table", i);
        const double n2 = (double)e[3] * e[3] + (double)e[4] * e[4] + (double)e[5] * e[5];
        if (!(std::fabs(n2 - 1.0) < 1e-3)) return fail(c, ANM_E_ARG, "trace: electron %zu direction is not a unit vector", i);
    }
    ANM_CUDA(c, cudaSetDevice(c->device));
    DevBuf<float> d_in, d_vol;
    DevBuf<double> d_esc;
    struct Rel { DevBuf<float>&a, &b; DevBuf<double>& d; ~Rel() { a.release(); b.release(); d.release(); } } rel{d_in, d_vol, d_esc};
    ANM_CUDA(c, d_in.alloc(in.size()));
    ANM_CUDA(c, d_vol.alloc(c->Vpad));
    ANM_CUDA(c, d_esc.alloc(1));
    ANM_CUDA(c, cudaMemcpyAsync(d_in.p, in.data(), in.size() * 4, cudaMemcpyHostToDevice, c->stream));
    ANM_CUDA(c, cudaMemsetAsync(d_vol.p, 0, c->Vpad * 4, c->stream));
    ANM_CUDA(c, cudaMemsetAsync(d_esc.p, 0, 8, c->stream));
    TransportParams p;
    std::memset(&p, 0, sizeof p);
    p.texels = c->texels.p; p.batch = d_vol.p;
    p.nx = c->nx; p.ny = c->ny; p.nz = c->nz; p.n_vox = (unsigned)c->V; p.stats = c->dstats.p;
    p.dx = (float)c->dx; p.dy = (float)c->dy; p.dz = (float)c->dz;
    p.inv_dx = (float)(1.0 / c->dx); p.inv_dy = (float)(1.0 / c->dy); p.inv_dz = (float)(1.0 / c->dz);
    fill_electron_params(c, p);
    electron_trace_kernel<<<(unsigned)((n + 127) / 128), 128, 0, c->stream>>>(p, d_in.p, (unsigned)n, d_esc.p);
    ANM_CUDA(c, cudaGetLastError());
    ANM_CUDA(c, cudaMemcpyAsync(out_MeV, d_vol.p, c->V * 4, cudaMemcpyDeviceToHost, c->stream));
    ANM_CUDA(c, cudaMemcpyAsync(escaped_MeV, d_esc.p, 8, cudaMemcpyDeviceToHost, c->stream));
    ANM_CUDA(c, cudaStreamSynchronize(c->stream));
    return ANM_OK;
}

int anm_set_options(anm_ctx* c, const anm_options* o) {
    if (!c) return ANM_E_ARG;
    if (!o) return fail(c, ANM_E_ARG, "options: null pointer");
    if (o->n_batches < 2) return fail(c, ANM_E_ARG, "options: n_batches must be >= 2");
    if (o->n_batches > 65536) return fail(c, ANM_E_ARG, "options: n_batches must be <= 65536");
    if (o->photons_per_decay != 1 && o->photons_per_decay != 2) return fail(c, ANM_E_ARG, "options: photons_per_decay must be 1 or 2");
    if (!(o->photon_cutoff_MeV > 0) || !(o->photon_cutoff_MeV < 0.51099895)) return fail(c, ANM_E_ARG, "options: photon cutoff out of range");
    if (!(o->positron_ke_MeV >= 0) || !std::isfinite(o->positron_ke_MeV)) return fail(c, ANM_E_ARG, "options: positron energy must be >= 0");
    if (o->schedule < 0 || o->schedule > 2) return fail(c, ANM_E_ARG, "options: schedule must be 0, 1 or 2");
    if (o->hull_majorant < 0 || o->hull_majorant > 2) return fail(c, ANM_E_ARG, "options: hull_majorant must be 0, 1 or 2");
    if (o->warp_aggregate < 0 || o->warp_aggregate > 2) return fail(c, ANM_E_ARG, "options: warp_aggregate must be 0 (auto), 1 (on) or 2 (off)");
    if (o->warp_aggregate == 1 && (o->electron_transport || o->uncertainty == 1))
        return fail(c, ANM_E_UNSUPPORTED, "options: warp_aggregate merges direct tally atomics; electron_transport / history-by-history scoring do not use them");
    if (o->electron_transport != 0 && o->electron_transport != 1) return fail(c, ANM_E_ARG, "options: electron_transport must be 0 or 1");
    if (o->batch_pipeline < 0 || o->batch_pipeline > 3) return fail(c, ANM_E_ARG, "options: batch_pipeline must be 0 (auto), 1, 2 or 3");
    if (o->uncertainty != 0 && o->uncertainty != 1) return fail(c, ANM_E_ARG, "options: uncertainty must be 0 (batch) or 1 (history by history)");
    if (o->batches_per_launch < 0 || o->batches_per_launch > 256) return fail(c, ANM_E_ARG, "options: batches_per_launch must be 0 (auto) or 1..256");
    if (o->texel_bits != 0 && o->texel_bits != 16 && o->texel_bits != 32) return fail(c, ANM_E_ARG, "options: texel_bits must be 0 (auto), 16 or 32");
    if (o->tally < 0 || o->tally > 2) return fail(c, ANM_E_ARG, "options: tally must be 0 (auto), 1 (direct atomics) or 2 (tile-binned)");
    if (o->tally == 2 && (o->schedule == 1 || o->electron_transport || o->uncertainty == 1 || o->warp_aggregate == 1))
        return fail(c, ANM_E_UNSUPPORTED, "options: the tile-binned tally runs in the event-pool schedule with the batch estimator, local electrons and no warp aggregation");
    if (o->uncertainty == 1 && o->schedule == 1) return fail(c, ANM_E_UNSUPPORTED, "options: history-by-history scoring runs in the event-pool schedule (0 or 2)");
    if (o->electron_transport && o->schedule == 1) return fail(c, ANM_E_UNSUPPORTED, "options: electron transport runs in the event-pool schedule (0 or 2)");
    c->opt = *o;
    c->dev_tables_dirty = true;
    c->have_results = false;
    return ANM_OK;
}

int anm_run(anm_ctx* c, uint64_t n_decays, uint64_t seed) {
    if (!c) return ANM_E_ARG;
    if (!c->have_grid || !c->have_phantom || !c->have_tables || !c->have_source)
        return fail(c, ANM_E_STATE, "run: need grid, phantom, physics tables and a source (missing:%s%s%s%s)",
                    c->have_grid ? "" : " grid", c->have_phantom ? "" : " phantom", c->have_tables ? "" : " tables",
                    c->have_source ? "" : " source");
    const int B = c->opt.n_batches;
    if (n_decays == 0 || n_decays % (uint64_t)B) return fail(c, ANM_E_ARG, "run: n_decays must be a positive multiple of n_batches = %d", B);
    const uint64_t nb = n_decays / (uint64_t)B;
    if (nb > 0x7fffffffull) return fail(c, ANM_E_ARG, "run: more than 2^31 decays per batch");
    if ((int)c->max_material >= c->nm) return fail(c, ANM_E_ARG, "run: phantom uses material %u but the tables hold %d", c->max_material, c->nm);
    if (std::exp(c->lnE_min) > c->opt.photon_cutoff_MeV * (1 + 1e-9)) return fail(c, ANM_E_ARG, "run: energy grid starts above the photon cutoff");
    if (c->opt.electron_transport) {
        if (!c->have_etables) return fail(c, ANM_E_STATE, "run: electron_transport needs anm_set_electron_tables");
        if ((int)c->max_material >= c->e_nm) return fail(c, ANM_E_ARG, "run: phantom uses material %u but the electron tables hold %d", c->max_material, c->e_nm);
    }
    ANM_CUDA(c, cudaSetDevice(c->device));
    c->have_results = false;
    if (c->dev_tables_dirty) { const int rc = upload_tables(c); if (rc != ANM_OK) return rc; }

    ANM_CUDA(c, c->organ_batch.alloc((size_t)B * 256));
    cudaStream_t st = c->stream;
    ANM_CUDA(c, cudaMemsetAsync(c->sum.p, 0, c->Vpad * 4, st));
    ANM_CUDA(c, cudaMemsetAsync(c->sumsq.p, 0, c->Vpad * 4, st));
    ANM_CUDA(c, cudaMemsetAsync(c->organ_batch.p, 0, (size_t)B * 256 * 8, st));
    ANM_CUDA(c, cudaMemsetAsync(c->organ_acc.p, 0, 256 * sizeof(OrganAccum), st));
    ANM_CUDA(c, cudaMemsetAsync(c->dstats.p, 0, sizeof(DeviceStats), st));
    ANM_CUDA(c, cudaMemsetAsync(c->total_energy.p, 0, 8, st));

    TransportParams p;
    std::memset(&p, 0, sizeof p);
    p.texels = c->texels.p; p.batch = c->batch.p; p.alias = c->alias.p; p.stats = c->dstats.p;
    p.tab_tot = c->d_tot.p; p.tab_pec = c->d_pec.p; p.tab_maj = c->d_maj.p; p.ray_x2 = c->d_x2.p; p.ray_cum = c->d_cum.p;
    p.n_hist = (unsigned)nb; p.n_alias = c->n_alias; p.n_vox = (unsigned)c->V;
    for (int r = 0; r < 10; ++r) {      // Philox4x32-10 round keys
        p.rk[2 * r] = (unsigned)seed + (unsigned)r * 0x9E3779B9u;
        p.rk[2 * r + 1] = (unsigned)(seed >> 32) + (unsigned)r * 0xBB67AE85u;
    }
    p.nx = c->nx; p.ny = c->ny; p.nz = c->nz; p.nm = c->nm; p.ne = c->ne; p.n_x2 = c->n_x2;
    p.dx = (float)c->dx; p.dy = (float)c->dy; p.dz = (float)c->dz;
    p.inv_dx = (float)(1.0 / c->dx); p.inv_dy = (float)(1.0 / c->dy); p.inv_dz = (float)(1.0 / c->dz);
    p.lnE_min = (float)c->lnE_min; p.inv_dlnE = (float)(1.0 / c->dlnE);
    p.cutoff = (float)c->opt.photon_cutoff_MeV; p.positron_ke = (float)c->opt.positron_ke_MeV;
    p.px = (float)c->px; p.py = (float)c->py; p.pz = (float)c->pz;
    p.point_source = c->point_source ? 1 : 0;
    p.photons_per_decay = c->opt.photons_per_decay; p.rayleigh_on = c->opt.rayleigh_on;
    p.tab_maj_out = c->d_majo.p;
    fill_electron_params(c, p);
    p.hull = (c->hull_ok && c->opt.hull_majorant != 2) ? 1 : 0;
    if (p.hull) {
        p.hx0 = (int)c->hull_lo[0]; p.hy0 = (int)c->hull_lo[1]; p.hz0 = (int)c->hull_lo[2];
        p.hnx = (int)(c->hull_hi[0] - c->hull_lo[0]); p.hny = (int)(c->hull_hi[1] - c->hull_lo[1]);
        p.hnz = (int)(c->hull_hi[2] - c->hull_lo[2]);
    }
    {   // ln-E grid coordinate of E0, in fp32 like the device's
        const float t = (logf(kE0) - p.lnE_min) * p.inv_dlnE;
        const int i = std::max(0, std::min((int)t, c->ne - 2));
        p.ie0 = i; p.fe0 = t - (float)i;
    }

    const int schedule = c->opt.schedule == 0 ? kAutoSchedule : c->opt.schedule;
    const size_t smem_tables = (size_t)c->nm * c->ne * 12 + (size_t)c->ne * 8 + (size_t)c->n_x2 * 4 + (size_t)c->nm * c->n_x2 * 4;
    const int threads = schedule == 2 ? kPoolThreads : kThreads;
    const size_t smem_el = (c->opt.electron_transport && schedule == 2) ? (size_t)c->e_nm * c->e_nt * 4 : 0;   // range tables
    const size_t smem = smem_tables + smem_el + (schedule == 2 ? (size_t)kPoolWarps * kPoolWarpBytes : (size_t)6 * kThreads * 4);
    const bool EL = c->opt.electron_transport != 0;
    const bool HB = c->opt.uncertainty == 1;
    // warp-aggregated tally atomics: on request, or (auto) where every decay's positron energy lands in one or a few
    // voxels -- a point source or a handful of active voxels -- and 32 same-address atomics per SOURCE trip would
    // serialise at the L2 (measured: 160 ms -> 18 ms per 1e8 histories on cfg1 with positron energy)
    const bool hot_source = c->opt.positron_ke_MeV > 0 && (c->point_source || c->n_alias < 1024u);
    // (an explicit tally = 2 is a request too: it keeps the automatic aggregation off; tally = 2 with warp_aggregate = 1 is refused in anm_set_options)
    const bool S = c->opt.collect_stats != 0, W = c->opt.warp_aggregate == 1 || (c->opt.warp_aggregate == 0 && hot_source && !EL && !HB && c->opt.tally != 2);
    // tile-binned tally: on request only -- measured +3 % on cfg4 (630 MB volumes) and 0.43x on cfg3, the
    // tile counters' same-address atomics bound it; needs the event pool, the batch estimator and local electrons
    const bool can_bin = schedule == 2 && !EL && !HB && !W;
    const bool BIN = can_bin && c->opt.tally == 2;
    // 16-bit texels (anm_options.texel_bits): the default kernel of the event pool reads the exact 16-bit copy when there is one
    const bool T16 = c->tex16_ok && c->opt.texel_bits != 32 && schedule == 2 && !EL && !HB && !BIN;
    p.texels16 = T16 ? c->texels16.p : nullptr;
    const TransportFn kern = pick_transport(schedule, S, BIN ? TALLY_BINNED : (W ? TALLY_WAGG : TALLY_RED), EL, HB, T16);
    {   // the event pool needs 152 KiB of slots plus the staged tables: large tables (the header admits n_energy = 1024
        // with 8 materials) do not fit the 227 KiB a CTA may opt into -- say so instead of failing in the attribute call
        int optin = 0;
        ANM_CUDA(c, cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, c->device));
        if (smem > (size_t)optin)
            return fail(c, ANM_E_UNSUPPORTED, "run: tables too large for shared memory (%zu bytes needed, %d available%s)", smem, optin,
                        schedule == 2 ? "; schedule = 1 needs 146 KiB less" : "");
    }
    ANM_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 0;
    ANM_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, smem));
    if (per_sm < 1) return fail(c, ANM_E_UNSUPPORTED, "run: tables too large for shared memory (%zu bytes)", smem);
    const int fold_blocks = grid_blocks(c, c->Vpad / 4, kFoldThreads);
    const float inv_vox = (float)(1.0 / (c->dx * c->dy * c->dz));
    c->run_hbh = HB;
    if (HB && nb > (uint64_t)kHbhHistMask) return fail(c, ANM_E_UNSUPPORTED, "run: history-by-history scoring holds at most 2^26 decays per batch");
    // Batch groups (anm_options.batches_per_launch): one transport launch covers G consecutive batches, each with its own
    // tally volume (batch-tagged deposits: the decay's batch within the group sits in its slot's meta word), and the G
    // folds follow the launch.  A launch is one resident wave of persistent CTAs whose tail (the last decays draining,
    // queues below 32 entries in every warp at the same time) costs ~0.25 ms whatever its size; with G batches per launch
    // that cost is paid B / G times instead of B times.  Same histories, same per-batch tallies.
    // G = 1 for the history-based schedule and the tile-binned tally (its per-launch lists are per batch); else the largest group that keeps depth * G tally volumes within the memory budget, at most 256
    // (8 bits of the meta word), G * nb <= 0xF0000000 histories per launch (2^26 with history-by-history scoring).
    int G = 1;
    if (schedule == 2 && !BIN) {
        // The launch's history counter is a 32-bit atomicAdd, and every warp adds to it a little past n_hist (its last
        // request plus the one it has asked for ahead: <= 2 kChunk per warp, a few million over the whole grid).  The cap
        // leaves 2^28 of headroom so that the counter can never wrap and hand out history 0 a second time.
        const uint64_t hist_cap = HB ? (uint64_t)kHbhHistMask : kLaunchHistCap;
        uint64_t gmax = std::min<uint64_t>({(uint64_t)B, (uint64_t)kMaxGroup, std::max<uint64_t>(1, hist_cap / nb)});
        if (c->opt.batches_per_launch > 0) gmax = std::min<uint64_t>(gmax, (uint64_t)c->opt.batches_per_launch);
        else {
            gmax = std::min<uint64_t>(gmax, (uint64_t)c->auto_group);      // auto: what anm_set_grid sized the tallies for
        }
        const int n_groups0 = (int)(((uint64_t)B + gmax - 1) / gmax);
        G = (B + n_groups0 - 1) / n_groups0;                           // even groups
    }
    const int n_groups = (B + G - 1) / G;
    if (HB && nb * (uint64_t)G > (uint64_t)kHbhHistMask) return fail(c, ANM_E_UNSUPPORTED, "run: history-by-history scoring holds at most 2^26 decays per launch");
    // Launch pipeline (anm_options.batch_pipeline): with `depth` sets of G batch tallies the launches of consecutive
    // groups go to `depth` internal streams: the CTAs of group g+1 take over each SM as the CTAs of group g exit, the folds
    // of group g run in the gaps.  The folds are serialised among themselves (they all update sum / sumsq); group g+depth
    // reuses the tallies of group g after their folds (same stream).
    const int depth = std::max(1, std::min(c->opt.batch_pipeline == 0 ? (G > 1 ? 2 : 3) : c->opt.batch_pipeline, n_groups));
    const size_t set_floats = (size_t)G * c->Vpad;
    if (c->batch.n < (size_t)depth * set_floats) {                     // more than anm_set_grid's auto size
        c->batch_clean = false;
        ANM_CUDA(c, c->batch.alloc((size_t)depth * set_floats));
    }
    if (c->batch_zero_ev) ANM_CUDA(c, cudaStreamWaitEvent(st, c->batch_zero_ev, 0));
    if (!c->batch_clean) ANM_CUDA(c, cudaMemsetAsync(c->batch.p, 0, (size_t)depth * set_floats * 4, st));   // the folds leave them zero
    c->batch_clean = false;                                            // until this run's folds have completed
    ANM_CUDA(c, c->counters.alloc((size_t)n_groups));
    ANM_CUDA(c, cudaMemsetAsync(c->counters.p, 0, (size_t)n_groups * 4, st));
    if (depth > 1)
        for (int k = 0; k < depth; ++k)
            if (!c->pipe[k]) ANM_CUDA(c, cudaStreamCreateWithFlags(&c->pipe[k], cudaStreamNonBlocking));
    const uint64_t per_block = schedule == 2 ? (uint64_t)kPoolWarps * kSlots : (uint64_t)kThreads;
    const int blocks = (int)std::max<uint64_t>(1, std::min<uint64_t>((uint64_t)c->num_sms * per_sm, (nb * (uint64_t)G + per_block - 1) / per_block));
    if (EL) {   // per-warp arrays of electrons waiting for their walk, one per launch in flight
        ANM_CUDA(c, c->e_ring.alloc((size_t)depth * blocks * kPoolWarps * kEFields * kPend));
        p.e_ring = c->e_ring.p;
    }
    if (HB) {   // history-by-history scoring: sum of X_h^2 over the whole run + one deposit list per decay slot
        const size_t nslots = (size_t)blocks * kPoolWarps * kSlots;
        ANM_CUDA(c, c->hbh_sq.alloc(c->Vpad));
        ANM_CUDA(c, c->hbh_list.alloc((size_t)depth * kHbhCap * nslots));      // one set of lists per launch in flight
        ANM_CUDA(c, cudaMemsetAsync(c->hbh_sq.p, 0, c->Vpad * 4, st));
        p.hbh_list = c->hbh_list.p; p.hbh_sq = c->hbh_sq.p; p.hbh_nslots = (unsigned)nslots;
    }
    p.n_per_batch = (unsigned)nb; p.batch_stride = c->Vpad;

    // events: [0] start, [1 + g] after the folds of group g, [n_groups + 1] pipeline join, [n_groups + 2] end;
    // serial mode (depth 1) also [n_groups + 3 + g] between launch g and its folds, for per-phase times
    std::vector<cudaEvent_t> ev((size_t)2 * n_groups + 3, nullptr);
    auto free_events = [&]() { for (auto e : ev) if (e) cudaEventDestroy(e); };
    for (auto& e : ev) if (cudaEventCreate(&e) != cudaSuccess) { free_events(); return fail(c, ANM_E_CUDA, "cudaEventCreate failed"); }
#define ANM_CUDA_EV(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { cudaGetLastError(); free_events(); \
        return fail(c, ANM_E_CUDA, "%s: %s", #call, cudaGetErrorString(e_)); } } while (0)

    // tile-binned tally: counters per launch in flight, one {offset, capacity} table; the capacities come from batch 0,
    // which runs with empty segments (every deposit takes the direct-RED path and is counted per tile)
    const unsigned n_tiles = (unsigned)((c->Vpad + kTileVoxels - 1) >> kTileShift);
    const unsigned n_lists = n_tiles * kTileSub;
    size_t bin_total = 0;                 // records per launch in flight
    if (BIN) {
        ANM_CUDA_EV(c->bin_cnt.alloc((size_t)depth * n_lists));
        ANM_CUDA_EV(c->bin_seg.alloc(n_lists));
        ANM_CUDA_EV(c->bin_seg0.alloc(n_lists));
        ANM_CUDA_EV(cudaMemsetAsync(c->bin_seg0.p, 0, (size_t)n_lists * 8, st));
        ANM_CUDA_EV(c->bin_ovf.alloc(2));      // [0] the run's overflow count, [1] the counting batch's (discarded)
        ANM_CUDA_EV(cudaMemsetAsync(c->bin_cnt.p, 0, (size_t)depth * n_lists * 4, st));
        ANM_CUDA_EV(cudaMemsetAsync(c->bin_seg.p, 0, (size_t)n_lists * 8, st));
        ANM_CUDA_EV(cudaMemsetAsync(c->bin_ovf.p, 0, 16, st));
        ANM_CUDA_EV(cudaFuncSetAttribute(bin_fold_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kTileVoxels * 4)));
        p.bin_seg = c->bin_seg.p;
    }
    uint64_t n_fold_launches = 0;
    ANM_CUDA_EV(cudaEventRecord(ev[0], st));
    if (depth > 1) for (int k = 0; k < depth; ++k) ANM_CUDA_EV(cudaStreamWaitEvent(c->pipe[k], ev[0], 0));
    for (int g = 0; g < n_groups; ++g) {
        const int b0 = g * G, nbg = std::min(G, B - b0);          // batches b0 .. b0 + nbg - 1
        const int set = g % depth;
        cudaStream_t sb = depth > 1 ? c->pipe[set] : st;
        p.batch = c->batch.p + (size_t)set * set_floats;
        p.n_group = (unsigned)nbg;
        p.n_hist = (unsigned)(nb * (uint64_t)nbg);
        if (BIN) {
            p.bin_cnt = c->bin_cnt.p + (size_t)set * n_lists;
            p.bin_rec = c->bin_rec.p ? c->bin_rec.p + (size_t)set * bin_total : nullptr;
        }
        if (EL) p.e_ring = c->e_ring.p + (size_t)set * blocks * kPoolWarps * kEFields * kPend;
        if (HB) p.hbh_list = c->hbh_list.p + (size_t)set * kHbhCap * p.hbh_nslots;
        p.counter = c->counters.p + g;
        p.hist_base = c->opt.history_offset + (unsigned long long)b0 * nb;
        kern<<<blocks, threads, smem, sb>>>(p);
        ANM_CUDA_EV(cudaGetLastError());
        if (BIN && g == 0) {
            // the counting batch has run: size every tile's segment for the batches to come -- its count plus six
            // standard deviations of a Poisson count plus 32 (a tile that still overflows loses nothing: the surplus
            // takes the direct-RED path into the batch volume, bin_fold_kernel adds both)
            std::vector<unsigned> cnt(n_lists);
            ANM_CUDA_EV(cudaMemcpyAsync(cnt.data(), p.bin_cnt, (size_t)n_lists * 4, cudaMemcpyDeviceToHost, sb));
            ANM_CUDA_EV(cudaStreamSynchronize(sb));
            std::vector<uint2> seg(n_lists);
            const char* cap_env = std::getenv("ANM_TALLY_CAPACITY");      // test hook (anm.h): a fixed capacity per tile
            const long cap_test = cap_env ? std::atol(cap_env) : 0;
            for (unsigned t = 0; t < n_lists; ++t) {
                const double want = (double)cnt[t] + 6.0 * std::sqrt((double)cnt[t]) + 32.0;
                const unsigned cap = cap_test > 0 ? (unsigned)cap_test : (unsigned)std::min(want, 4.0e9 - 1.0);
                if (bin_total + cap > 0xfffffff0ull) { free_events(); return fail(c, ANM_E_UNSUPPORTED, "run: more than 2^32 deposit records per batch; use more batches or tally = 1"); }
                seg[t] = make_uint2((unsigned)bin_total, cap);
                bin_total += cap;
            }
            ANM_CUDA_EV(c->bin_rec.alloc((size_t)depth * bin_total));
            ANM_CUDA_EV(cudaMemcpyAsync(c->bin_seg.p, seg.data(), (size_t)n_lists * 8, cudaMemcpyHostToDevice, sb));
            ANM_CUDA_EV(cudaStreamSynchronize(sb));     // seg is a host temporary; every later launch (any stream) sees the table
        }
        if (depth > 1 && g > 0) ANM_CUDA_EV(cudaStreamWaitEvent(sb, ev[1 + (g - 1)], 0));    // after the previous group's folds
        if (depth == 1) ANM_CUDA_EV(cudaEventRecord(ev[n_groups + 3 + g], sb));
        // the folds of the group: one fused pass over its tallies (fold_group_kernel), in sub-groups whose per-batch
        // organ bins fit 48 KB of shared memory; the tile-binned tally and single-batch launches fold batch by batch
        const int fuse = (!BIN && nbg > 1) ? std::max(1, std::min(nbg, (int)(49152 / ((size_t)(c->n_organs + 1) * 8)))) : 1;
        for (int j = 0; fuse > 1 && j < nbg; j += fuse) {
            const int gj = std::min(fuse, nbg - j);
            fold_group_kernel<<<fold_blocks, kFoldThreads, (size_t)gj * (c->n_organs + 1) * 8, sb>>>(
                (float4*)(p.batch + (size_t)j * c->Vpad), c->Vpad / 4, gj, (float4*)c->sum.p, (float4*)c->sumsq.p,
                c->have_organs ? (const uint32_t*)c->labels.p : nullptr, (const uint4*)c->texels.p,
                c->organ_batch.p + (size_t)(b0 + j) * 256, c->n_organs, c->Vpad / 4, inv_vox);
            ANM_CUDA_EV(cudaGetLastError());
            n_fold_launches += 1;
        }
        for (int j = 0; fuse == 1 && j < nbg; ++j) {
            const int b = b0 + j;
            float* tally = p.batch + (size_t)j * c->Vpad;
            n_fold_launches += 1;
            if (BIN) {
                // batch 0 counted against empty segments; its fold must see them empty too (the table is already final)
                bin_fold_kernel<<<std::min<unsigned>(n_tiles, (unsigned)c->num_sms * 3u), kBinFoldThreads, kTileVoxels * 4, sb>>>(
                    p.bin_cnt, b == 0 ? c->bin_seg0.p : c->bin_seg.p, p.bin_rec, (float4*)tally, (float4*)c->sum.p, (float4*)c->sumsq.p,
                    c->have_organs ? (const uint32_t*)c->labels.p : nullptr, (const uint4*)c->texels.p,
                    c->organ_batch.p + (size_t)b * 256, c->n_organs, c->Vpad / 4, n_tiles, inv_vox, c->bin_ovf.p + (b == 0 ? 1 : 0));
            } else {
                fold_kernel<<<fold_blocks, kFoldThreads, 0, sb>>>(
                    (float4*)tally, (float4*)c->sum.p, (float4*)c->sumsq.p,
                    c->have_organs ? (const uint32_t*)c->labels.p : nullptr, (const uint4*)c->texels.p,
                    c->organ_batch.p + (size_t)b * 256, c->n_organs, c->Vpad / 4, inv_vox);
            }
            ANM_CUDA_EV(cudaGetLastError());
        }
        ANM_CUDA_EV(cudaEventRecord(ev[1 + g], sb));
    }
    if (depth > 1) {    // join: the caller's stream continues after the last folds (which follow every other launch)
        ANM_CUDA_EV(cudaStreamWaitEvent(st, ev[1 + (n_groups - 1)], 0));
        for (int g = std::max(0, n_groups - depth); g < n_groups - 1; ++g) ANM_CUDA_EV(cudaStreamWaitEvent(st, ev[1 + g], 0));
    }
    ANM_CUDA_EV(cudaEventRecord(ev[n_groups + 1], st));
    {
        const int rc = finalize_and_collect(c, B, nb, n_decays, nullptr);
        if (rc != ANM_OK) { free_events(); return rc; }
    }
    ANM_CUDA_EV(cudaEventRecord(ev[n_groups + 2], st));
    DeviceStats ds;
    unsigned long long bin_overflow = 0;
    if (BIN) ANM_CUDA_EV(cudaMemcpyAsync(&bin_overflow, c->bin_ovf.p, 8, cudaMemcpyDeviceToHost, st));
    ANM_CUDA_EV(cudaMemcpyAsync(&ds, c->dstats.p, sizeof ds, cudaMemcpyDeviceToHost, st));
    ANM_CUDA_EV(cudaStreamSynchronize(st));
    c->batch_clean = true;      // every fold has run: the tallies are zero again

    double ms_t = 0, ms_f = 0, ms_fin = 0;
    if (depth > 1) {
        // overlapped launches have no separate durations: the whole pipeline (transport with the folds inside it) is
        // reported as transport time, conservatively; ms_fold = 0
        float a = 0;
        cudaEventElapsedTime(&a, ev[0], ev[n_groups + 1]);
        ms_t = a;
    } else for (int g = 0; g < n_groups; ++g) {
        float a = 0, f = 0;
        cudaEventElapsedTime(&a, ev[g == 0 ? 0 : g], ev[n_groups + 3 + g]);       // [g] = after the folds of group g - 1
        cudaEventElapsedTime(&f, ev[n_groups + 3 + g], ev[1 + g]);
        ms_t += a; ms_f += f;
    }
    { float f = 0; cudaEventElapsedTime(&f, ev[n_groups + 1], ev[n_groups + 2]); ms_fin = f; }
    free_events();
#undef ANM_CUDA_EV

    const double tot_e = c->stats.deposited_MeV;
    anm_stats& s = c->stats;
    std::memset(&s, 0, sizeof s);
    s.n_decays = n_decays;
    s.emitted_MeV = (double)n_decays * ((double)kE0 * c->opt.photons_per_decay + c->opt.positron_ke_MeV);
    s.deposited_MeV = tot_e;
    s.escaped_MeV = ds.escaped_MeV;
    s.n_steps = ds.n_steps; s.n_real = ds.n_real; s.n_pe = ds.n_pe; s.n_compton = ds.n_compton;
    s.n_rayleigh = ds.n_rayleigh; s.n_escaped = ds.n_escaped; s.n_cutoff = ds.n_cutoff; s.n_electrons = ds.n_electrons;
    s.n_hbh_overflow = ds.n_hbh_overflow;
    s.n_fly_trips = ds.n_fly_trips; s.n_compton_tries = ds.n_compton_tries; s.n_rayleigh_tries = ds.n_rayleigh_tries;
    s.n_check_violations = 0;
    for (int k = 0; k < 12; ++k) {
        s.n_check_violations += ds.n_violations[k];
        if (ds.n_violations[k] && std::getenv("ANM_CHECK_VERBOSE")) fprintf(stderr, "anm bounds check %d: %llu violations\n", k, ds.n_violations[k]);
    }
    s.ms_transport = ms_t; s.ms_fold = ms_f; s.ms_finalize = ms_fin; s.ms_setup = c->ms_setup;
    s.ms_load_ct = c->ms_load_ct; s.ms_load_pet = c->ms_load_pet;
    s.n_launches = (uint64_t)n_groups + n_fold_launches + 1;
    s.batches_per_launch = (uint64_t)G;
    s.texel_bits = T16 ? 16 : 32;
    s.tally_binned = BIN ? 1 : 0;
    s.n_tally_overflow = bin_overflow;
    s.n_launches += 2;     // dose_max + run_sigma of the finalize
    fill_run_sigma(c, s);
    c->run_decays = n_decays;
    c->run_batches = B;
    c->have_results = true;
    return ANM_OK;
}

static int readout(anm_ctx* c, float* out, size_t n, int on_device, int mode, double scale) {
    if (!c) return ANM_E_ARG;
    if (!out) return fail(c, ANM_E_ARG, "get: null pointer");
    if (!c->have_results) return fail(c, ANM_E_STATE, "get: no completed run");
    if (n != c->V) return fail(c, ANM_E_ARG, "get: n = %zu but the grid has %zu voxels", n, c->V);
    ANM_CUDA(c, cudaSetDevice(c->device));
    float* dst = out;
    if (!on_device) { ANM_CUDA(c, c->scratch.alloc(c->Vpad)); dst = c->scratch.p; }
    const double factor = kGyPerMeVPerGram * scale / ((double)c->run_decays * c->dx * c->dy * c->dz);
    readout_kernel<<<grid_blocks(c, c->V, kFoldThreads), kFoldThreads, 0, c->stream>>>(
        c->sum.p, c->run_hbh ? c->hbh_sq.p : c->sumsq.p, c->texels.p, dst, c->V, mode, factor,
        c->run_hbh ? (double)c->run_decays : (double)c->run_batches, c->opt.zero_air_dose);
    ANM_CUDA(c, cudaGetLastError());
    if (!on_device) ANM_CUDA(c, cudaMemcpyAsync(out, dst, c->V * 4, cudaMemcpyDeviceToHost, c->stream));
    ANM_CUDA(c, cudaStreamSynchronize(c->stream));
    return ANM_OK;
}

int anm_get_energy(anm_ctx* c, float* out, size_t n, int on_device) { return readout(c, out, n, on_device, 0, 1.0); }
int anm_get_dose(anm_ctx* c, float* out, size_t n, int on_device) { return readout(c, out, n, on_device, 1, 1.0); }
int anm_get_dose_rate(anm_ctx* c, double total_activity_Bq, float* out, size_t n, int on_device) {
    if (c && !(total_activity_Bq >= 0 && std::isfinite(total_activity_Bq))) return fail(c, ANM_E_ARG, "dose rate: activity must be >= 0");
    return readout(c, out, n, on_device, 1, total_activity_Bq);
}
int anm_get_uncertainty(anm_ctx* c, float* out, size_t n, int on_device) { return readout(c, out, n, on_device, 2, 1.0); }

int anm_get_organ_doses(anm_ctx* c, anm_organ* out, int n_organs) {
    if (!c) return ANM_E_ARG;
    if (!out) return fail(c, ANM_E_ARG, "organ doses: null pointer");
    if (!c->have_results || !c->have_organs) return fail(c, ANM_E_STATE, "organ doses: no completed run with organ labels");
    if (n_organs != c->n_organs) return fail(c, ANM_E_ARG, "organ doses: n_organs = %d but %d were loaded", n_organs, c->n_organs);
    std::memcpy(out, c->organs.data(), sizeof(anm_organ) * (size_t)n_organs);
    return ANM_OK;
}

int anm_get_alias_table(anm_ctx* c, uint32_t* out, size_t capacity_entries, size_t* n_entries) {
    if (!c) return ANM_E_ARG;
    if (!n_entries) return fail(c, ANM_E_ARG, "alias table: null pointer");
    if (!c->have_source || c->point_source) return fail(c, ANM_E_STATE, "alias table: no activity map is loaded");
    *n_entries = c->n_alias;
    if (!out) return ANM_OK;
    if (capacity_entries < c->n_alias) return fail(c, ANM_E_ARG, "alias table: %zu entries needed, room for %zu", (size_t)c->n_alias, capacity_entries);
    ANM_CUDA(c, cudaSetDevice(c->device));
    ANM_CUDA(c, cudaMemcpyAsync(out, c->alias.p, (size_t)c->n_alias * sizeof(uint4), cudaMemcpyDeviceToHost, c->stream));
    ANM_CUDA(c, cudaStreamSynchronize(c->stream));
    return ANM_OK;
}

// ---- multi-GPU merge ----------------------------------------------------------------
int anm_get_tally_buffers(anm_ctx* c, float** d_sum, float** d_sumsq, size_t* n_floats, double** d_organ_rows, int* n_rows) {
    if (!c) return ANM_E_ARG;
    if (!d_sum || !d_sumsq || !n_floats || !d_organ_rows || !n_rows) return fail(c, ANM_E_ARG, "tally buffers: null pointer");
    if (!c->have_results) return fail(c, ANM_E_STATE, "tally buffers: no completed run");
    // the sum-of-squares volume of the run's estimator: over batches, or over histories (uncertainty = 1) -- both add up
    // across shards
    *d_sum = c->sum.p; *d_sumsq = c->run_hbh ? c->hbh_sq.p : c->sumsq.p; *n_floats = c->Vpad;
    *d_organ_rows = c->organ_batch.p; *n_rows = c->run_batches;
    return ANM_OK;
}

int anm_merge(anm_ctx* c, uint64_t total_decays, int total_batches, const double* organ_rows_all, const anm_stats* summed) {
    if (!c) return ANM_E_ARG;
    if (!c->have_results) return fail(c, ANM_E_STATE, "merge: no completed run");
    if (total_batches < c->run_batches || total_batches < 2 || total_decays == 0 || total_decays % (uint64_t)total_batches)
        return fail(c, ANM_E_ARG, "merge: total_decays must be a positive multiple of total_batches >= this run's batches");
    const uint64_t nb = c->run_decays / (uint64_t)c->run_batches;
    if (total_decays / (uint64_t)total_batches != nb)
        return fail(c, ANM_E_ARG, "merge: every shard must use the same decays per batch (%llu here)", (unsigned long long)nb);
    if (c->have_organs && !organ_rows_all) return fail(c, ANM_E_ARG, "merge: organ rows of all batches are required");
    ANM_CUDA(c, cudaSetDevice(c->device));
    const anm_stats mine = c->stats;
    const int rc = finalize_and_collect(c, total_batches, nb, total_decays, organ_rows_all);
    if (rc != ANM_OK) { c->have_results = false; return rc; }
    anm_stats& s = c->stats;
    const double dep = s.deposited_MeV;
    if (summed) s = *summed; else { s = mine; s.escaped_MeV = 0; s.n_steps = s.n_real = s.n_pe = s.n_compton = s.n_rayleigh = s.n_escaped = s.n_cutoff = s.n_electrons = s.n_hbh_overflow = 0; }
    s.n_launches += 3;     // the finalize launches of the merge
    fill_run_sigma(c, s);
    s.n_decays = total_decays;
    s.emitted_MeV = (double)total_decays * ((double)kE0 * c->opt.photons_per_decay + c->opt.positron_ke_MeV);
    s.deposited_MeV = dep;
    c->run_decays = total_decays;
    c->run_batches = total_batches;
    return ANM_OK;
}

// ---- roofline microbenchmarks (anm_peaks.cuh) -------------------------------------------------------------------
int anm_measure_peaks(anm_ctx* c, uint64_t small_bytes, uint64_t large_bytes, anm_peaks* out) {
    if (!c) return ANM_E_ARG;
    if (!out) return fail(c, ANM_E_ARG, "peaks: null pointer");
    const uint64_t sizes[2] = {small_bytes / 4 * 4, large_bytes / 4 * 4};
    for (uint64_t b : sizes)
        if (b < 4096 || b >= (16ull << 30)) return fail(c, ANM_E_ARG, "peaks: array sizes must be in [4096, 16 GiB)");
    ANM_CUDA(c, cudaSetDevice(c->device));
    std::memset(out, 0, sizeof *out);
    cudaStream_t st = c->stream;
    Events<2> evs;
    ANM_CUDA(c, evs.create());
    const cudaEvent_t e0 = evs.e[0], e1 = evs.e[1];
    DevBuf<float> arr, sink;
    ANM_CUDA(c, sink.alloc(4));
    const int blocks = c->num_sms * 2;            // 64 resident warps per SM
    const double threads = (double)blocks * kPeakThreads;
    // best of 3 timed launches after one warm-up; returns seconds
    auto timed = [&](auto&& launch, double* sec) -> int {
        double best = 1e30;
        for (int rep = 0; rep < 4; ++rep) {
            ANM_CUDA(c, cudaEventRecord(e0, st));
            launch();
            ANM_CUDA(c, cudaGetLastError());
            ANM_CUDA(c, cudaEventRecord(e1, st));
            ANM_CUDA(c, cudaEventSynchronize(e1));
            float ms = 0;
            ANM_CUDA(c, cudaEventElapsedTime(&ms, e0, e1));
            if (rep > 0) best = std::min(best, (double)ms * 1e-3);
        }
        *sec = best;
        return ANM_OK;
    };
    double sec = 0;
    int rc;
    {
        const int iters = 4096;
        DevBuf<long long> cyc;
        ANM_CUDA(c, cyc.alloc(1));
        rc = timed([&] { issue_kernel<<<blocks, kPeakThreads, 0, st>>>(sink.p, cyc.p, iters, 1.0000001f, 1e-9f, 0x5bd1e995u); }, &sec);
        long long cycles = 0;
        if (rc == ANM_OK && cudaMemcpy(&cycles, cyc.p, 8, cudaMemcpyDeviceToHost) != cudaSuccess) rc = fail(c, ANM_E_CUDA, "peaks: copy failed");
        cyc.release();
        if (rc != ANM_OK) return rc;
        out->issue_gtis = threads * iters * kIssueUnroll * kIssuePerIter / sec * 1e-9;
        // two CTAs share an SM and run the whole launch side by side, so the first warp's loop spans the launch
        out->issue_sm_mhz = (double)cycles / sec * 1e-6;
    }
    {
        TransportParams p;
        std::memset(&p, 0, sizeof p);
        for (int r = 0; r < 10; ++r) { p.rk[2 * r] = 42u + (unsigned)r * 0x9E3779B9u; p.rk[2 * r + 1] = (unsigned)r * 0xBB67AE85u; }
        const int nb = 2048;
        rc = timed([&] { philox_chain_kernel<<<blocks, kPeakThreads, 0, st>>>(p, (unsigned*)sink.p, nb); }, &sec);
        if (rc != ANM_OK) return rc;
        out->philox_gblocks = threads * nb / sec * 1e-9;
    }
    DevBuf<float> arr2;
    for (int k = 0; k < 2; ++k) {
        const size_t n = (size_t)(sizes[k] / 4);
        out->bytes[k] = sizes[k];
        ANM_CUDA(c, arr.alloc(n));
        ANM_CUDA(c, cudaMemsetAsync(arr.p, 0, n * 4, st));
        const unsigned n32 = (unsigned)std::min<size_t>(n, 0xffffffffu);
        const int accesses = 2048;                 // per thread and launch, whatever the depth
        // sweep of the accesses in flight per thread (full occupancy throughout): the best rate is the denominator
        const int depths[4] = {4, 8, 16, 32};
        for (int d = 0; d < 4; ++d) {
            const int trips = accesses / depths[d];
            rc = timed([&] {
                const uint32_t* a = (const uint32_t*)arr.p; unsigned* o = (unsigned*)sink.p;
                switch (depths[d]) {
                    case 4: gather_kernel<4><<<blocks, kPeakThreads, 0, st>>>(a, n32, trips, o); break;
                    case 8: gather_kernel<8><<<blocks, kPeakThreads, 0, st>>>(a, n32, trips, o); break;
                    case 16: gather_kernel<16><<<blocks, kPeakThreads, 0, st>>>(a, n32, trips, o); break;
                    default: gather_kernel<32><<<blocks, kPeakThreads, 0, st>>>(a, n32, trips, o); break;
                } }, &sec);
            if (rc != ANM_OK) return rc;
            const double g = threads * trips * depths[d] / sec * 1e-9;
            if (g > out->gather_gps[k]) { out->gather_gps[k] = g; out->gather_in_flight[k] = depths[d]; }
        }
        for (int d = 0; d < 4; ++d) {
            const int trips = accesses / 4 / depths[d];
            rc = timed([&] {
                switch (depths[d]) {
                    case 4: red_kernel<4><<<blocks, kPeakThreads, 0, st>>>(arr.p, n32, trips); break;
                    case 8: red_kernel<8><<<blocks, kPeakThreads, 0, st>>>(arr.p, n32, trips); break;
                    case 16: red_kernel<16><<<blocks, kPeakThreads, 0, st>>>(arr.p, n32, trips); break;
                    default: red_kernel<32><<<blocks, kPeakThreads, 0, st>>>(arr.p, n32, trips); break;
                } }, &sec);
            if (rc != ANM_OK) return rc;
            const double r = threads * trips * depths[d] / sec * 1e-9;
            if (r > out->red_gps[k]) { out->red_gps[k] = r; out->red_in_flight[k] = depths[d]; }
        }
        // both at once over two arrays of this size (loads from one, REDs into the other)
        ANM_CUDA(c, arr2.alloc(n));
        ANM_CUDA(c, cudaMemsetAsync(arr2.p, 0, n * 4, st));
        const int mtrips = 64;
        rc = timed([&] { mix_kernel<<<blocks, kPeakThreads, 0, st>>>((const uint32_t*)arr.p, arr2.p, n32, mtrips, (unsigned*)sink.p); }, &sec);
        if (rc != ANM_OK) return rc;
        out->mix_gps[k] = threads * mtrips * (kMixGathers + kMixReds) / sec * 1e-9;
    }
    return ANM_OK;
}

int anm_get_stats(anm_ctx* c, anm_stats* out) {
    if (!c) return ANM_E_ARG;
    if (!out) return fail(c, ANM_E_ARG, "stats: null pointer");
    if (c->have_results) *out = c->stats;
    else std::memset(out, 0, sizeof *out);     // before a run: only the set-up timings are meaningful
    out->ms_setup = c->ms_setup; out->ms_load_ct = c->ms_load_ct; out->ms_load_pet = c->ms_load_pet;
    return ANM_OK;
}

}  // extern "C"
