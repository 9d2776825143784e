// anm_kernels.cuh -- device code of libanm.so (sm_100a).  Hand-written CUDA; no oracle code is shared.
//
// Kernels
//   transport_pool_kernel / transport_kernel : source sampling + Woodcock photon transport + fp32 RED tally
//                      (the two schedules below)
//   fold_group_kernel : the G per-batch tallies of one launch folded in one pass: sum += x, sumsq += x^2, x = 0,
//                      organ partial sums per batch (A10);  fold_kernel: the same for a single batch tally;
//                      bin_fold_kernel: the same from the tile-binned deposit lists (anm_options.tally = 2)
//   finalize_kernel  : organ Eq. 3 accumulators, organ energy / mass / counts, total energy (A11)
//   readout_kernel   : dose / dose rate / relative sigma read-out                           (A11)
//   dose_max_kernel, run_sigma_kernel : run-level RMS relative sigma above 10 % / 50 % of the maximum dose (A11)
//   pack_texels / pack_texels16 (the exact 16-bit texel copy, anm_options.texel_bits) / rho_max / rho_max_outside /
//   hull_box / organ_mass kernels : set-up (A0); the alias table is in anm_alias.cuh,
//                      the image front end in anm_frontend.cuh
//   electron_walk (device function) + electron_trace_kernel : secondary electrons
//   hbh_push / hbh_flush (device functions)                 : history-by-history scoring (NEXT-4)
//   philox_probe_kernel                                     : parity hook of the generator (anm_philox_blocks)
//
// Two schedules of the same per-event code (anm_options.schedule):
//   1  transport_kernel       history-based: every lane owns one photon and runs a per-lane state machine;
//   2  transport_pool_kernel  event-based at warp scope: each warp owns kSlotsPerWarp photon slots in shared
//                             memory, every trip votes for ONE event type, compacts up to 32 slots waiting for
//                             it and runs that event with (nearly) all lanes active; finished slots regenerate
//                             a new history in place (no global queues, no extra HBM traffic).
// Scheduling (1): history-based persistent lanes run as a per-lane state machine.  Each trip of the warp's
// loop draws ONE Philox4x32-10 block per live lane (common code), then every lane spends it on its own
// event: SOURCE (new decay), FLY (two Woodcock sub-steps), COMPTON (one Klein-Nishina try + azimuth) or
// RAYLEIGH (one form-factor try + azimuth).  A lane whose photon ends starts the partner photon from a
// shared-memory stash, or takes a new history index from a warp-level pool refilled by one atomic per
// kChunk histories.  Results depend only on (seed, history index): counter = (h_lo, h_hi, block, stream),
// stream 0 = source, 1 = photon A, 2 = photon B.
#pragma once
#include <cstdint>
#include <cstdio>
#include <cuda_runtime.h>

namespace anm {

#ifdef ANM_TRACE
#define ANM_TR(...) printf(__VA_ARGS__)
#else
#define ANM_TR(...) do {} while (0)
#endif

constexpr int kThreads = 256;
constexpr int kMinBlocksPerSM = 4;
#ifndef ANM_CHUNK
#define ANM_CHUNK 128
#endif
constexpr unsigned kChunk = ANM_CHUNK;      // histories a warp takes per atomic
#ifndef ANM_CHUNK_TAIL
#define ANM_CHUNK_TAIL 32
#endif
constexpr unsigned kChunkTail = ANM_CHUNK_TAIL;   // ... near the end of a launch (event pool: guided chunk sizes)
constexpr float kE0 = 0.51099895f;          // MeV, "0.511 MeV"
constexpr float kInvE0 = 1.0f / 0.51099895f;
constexpr float kTwoPi = 6.283185307179586f;
constexpr float kKeVAngstromInv = 1000.0f / 12.398419843f;   // x_max (1/Angstrom) = E[MeV] * this
constexpr float kDensityStep = 1.0f / 1048576.0f;            // 2^-20 g/cm^3 per texel count

enum : int { ST_NEED = 0, ST_SOURCE = 1, ST_FLY = 2, ST_COMPTON = 3, ST_RAYLEIGH = 4, ST_DONE = 5 };

struct DeviceStats {   // accumulated with atomics at kernel exit (collect_stats only)
    double escaped_MeV;
    unsigned long long n_steps, n_real, n_pe, n_compton, n_rayleigh, n_escaped, n_cutoff, n_electrons, n_hbh_overflow;
    unsigned long long n_fly_trips, n_compton_tries, n_rayleigh_tries;   // event trips (event pool): FLY events, Klein-Nishina / form-factor tries
    unsigned long long n_violations[12];   // ANM_BOUNDS_CHECK builds: indices found out of range, per check (counted, never trapped)
};

// Bounds-check build (-DANM_BOUNDS_CHECK; profiles/r2_sanitizer.md): every index the transport kernels form -- voxel,
// material, energy-grid cell, alias bucket, pool slot, ring fill, deposit-list and electron-array position -- is tested
// against its range and a violation is COUNTED in DeviceStats::n_violations (anm_stats.n_check_violations) instead of
// trapping, so a bad build cannot wedge the GPU.  Compiled out otherwise.
#ifdef ANM_BOUNDS_CHECK
#define ANM_CHK(p, id, cond) do { if (!(cond)) atomicAdd(&(p).stats->n_violations[id], 1ull); } while (0)
#else
#define ANM_CHK(p, id, cond) do {} while (0)
#endif

struct TransportParams {
    const uint32_t* texels;      // [V] material<<24 | density/2^-20
    const uint16_t* texels16;    // [V] material<<13 | density/2^-12: the same volume in 16 bits when every voxel is exactly
                                 // representable (anm_options.texel_bits; reading C18), else null
    float* batch;                // [V] energy of the current batch (MeV)
    const uint4* alias;          // [n_alias] {threshold, own voxel, alias voxel, 0}
    unsigned int* counter;       // history counter of this launch (starts at 0)
    DeviceStats* stats;
    const float* tab_tot;        // [nm][ne]  total mu/rho (Rayleigh included iff rayleigh_on)
    const float2* tab_pec;       // [nm][ne]  {pe, pe + compton}
    const float* tab_maj;        // [ne]      majorant (1/cm)
    const float* ray_x2;         // [n_x2]
    const float* ray_cum;        // [nm][n_x2]
    unsigned long long hist_base;   // global index of this launch's first history
    unsigned int n_hist;         // histories in this launch
    unsigned int n_alias;
    unsigned int n_vox;          // nx * ny * nz
    // batch group (event pool): one launch covers n_group consecutive batches of n_per_batch histories each; history hl of
    // the launch belongs to local batch hl / n_per_batch, whose tally is batch + local batch * batch_stride
    unsigned int n_per_batch, n_group;
    size_t batch_stride;         // floats between the tallies of consecutive batches of the group
    unsigned int rk[20];         // Philox round keys: rk[2r] = seed_lo + r*0x9E3779B9, rk[2r+1] = seed_hi + r*0xBB67AE85
    int nx, ny, nz;
    int nm, ne, n_x2;
    float dx, dy, dz;            // cm
    float inv_dx, inv_dy, inv_dz;
    float lnE_min, inv_dlnE;
    float cutoff, positron_ke;
    float px, py, pz;            // point source (cm)
    int point_source, photons_per_decay, rayleigh_on;
    // ln-E grid coordinate of E0 (every photon starts there): ie0 + fe0
    int ie0; float fe0;
    // hull majorant (anm_options.hull_majorant): an axis-aligned box of voxels encloses every voxel denser than the
    // hull threshold.  A photon that has left the box on a straight line flies against tab_maj_out (the bound of the
    // voxels outside the box); every other photon against tab_maj (fly_substep).
    int hull;
    int hx0, hy0, hz0, hnx, hny, hnz;         // the box in voxel indices: [hx0, hx0 + hnx) x ...
    const float* tab_maj_out;    // [ne]
    // secondary-electron transport (anm_options.electron_transport; reading C28): residual CSDA range above
    // the electron cutoff, [nm][n_t] g/cm^2 on the kinetic-energy grid t_min + k dt; t_min = the cutoff
    const float* e_range;
    int n_t, e_nm;               // e_nm materials in the electron tables
    float* e_ring;               // [warps of the launch][kEFields][kPend] electrons waiting for their walk (event pool)
    float t_min, e_dt, e_inv_dt;
    // history-by-history scoring (anm_options.uncertainty = 1, Walters et al. 2002): per decay slot a
    // list of the decay's deposits {voxel, energy} in global scratch, hbh_list[i * hbh_nslots + slot] (its length in the
    // slot's shared-memory history word); merged per voxel when the slot is re-used: batch[v] += X, hbh_sq[v] += X^2
    uint2* hbh_list;
    float* hbh_sq;               // [V] sum over histories of X_h^2 (MeV^2), whole run
    unsigned hbh_nslots;
    // tile-binned tally (anm_options.tally): when the tally volume does not fit the L2, a deposit is not a
    // random RED into HBM but a record {voxel, energy} appended to the list of the voxel's tile (kTileVoxels consecutive
    // voxels): bin_cnt[tile] hands out positions, bin_seg[tile] = {offset, capacity} of the tile's segment of bin_rec;
    // a deposit beyond the capacity goes to the batch volume as before.  bin_fold_kernel sums the lists in shared memory.
    unsigned* bin_cnt;
    const uint2* bin_seg;
    uint2* bin_rec;
};

// ------------------------------------------------------------------------------------------------
// Philox4x32-10 (north_star (d)); rk[2r], rk[2r+1] = the key of round r (key + r * Weyl constants, computed on the
// host: they sit in the constant bank and cost no instruction).
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, const TransportParams& p) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long p0 = (unsigned long long)0xD2511F53u * c.x;
        const unsigned long long p1 = (unsigned long long)0xCD9E8D57u * c.z;
        c = make_uint4((unsigned)(p1 >> 32) ^ c.y ^ p.rk[2 * r], (unsigned)p1,
                       (unsigned)(p0 >> 32) ^ c.w ^ p.rk[2 * r + 1], (unsigned)p0);
    }
    return c;
}

// inspection / parity hook (anm_philox_blocks): the generator exactly as the transport kernels call it
__global__ void philox_probe_kernel(const __grid_constant__ TransportParams p, const uint4* __restrict__ ctr, uint4* __restrict__ out, unsigned n) {
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = philox4x32_10(ctr[i], p);
}

// uniform on (0,1): ((r >> 8) + 0.5) 2^-24
__device__ __forceinline__ float u01(unsigned r) {
    return fmaf(__uint2float_rn(r >> 8), 5.9604644775390625e-08f, 2.98023223876953125e-08f);
}

// The library is compiled with -fmad=false: every fused multiply-add below is written out, so the two schedules
// (which inline these functions in different contexts) round identically and run bit-identical histories.
__device__ __forceinline__ void rotate(float& u, float& v, float& w, float cos_t, float phi) {
    const float sin_t = sqrtf(fmaxf(0.0f, fmaf(-cos_t, cos_t, 1.0f)));
    float sp, cp;
    __sincosf(phi, &sp, &cp);
    float a, b, c;
    if (fabsf(w) < 0.99999f) {
        const float s = sqrtf(fmaf(-w, w, 1.0f));
        const float k = __fdividef(sin_t, s);
        a = fmaf(k, fmaf(u * w, cp, -(v * sp)), u * cos_t);
        b = fmaf(k, fmaf(v * w, cp, u * sp), v * cos_t);
        c = fmaf(-(sin_t * s), cp, w * cos_t);
    } else {
        a = sin_t * cp; b = sin_t * sp; c = copysignf(cos_t, w);
    }
    const float n = rsqrtf(fmaf(a, a, fmaf(b, b, c * c)));
    u = a * n; v = b * n; w = c * n;
}

// How a deposit reaches the tally (template parameter of the transport kernels)
enum : int { TALLY_RED = 0, TALLY_WAGG = 1, TALLY_BINNED = 2 };
constexpr int kTileShift = 14;                       // tile = 2^14 consecutive voxels = 64 KB of fp32 in shared memory
constexpr unsigned kTileVoxels = 1u << kTileShift;
#ifndef ANM_TILE_SUBLISTS
#define ANM_TILE_SUBLISTS 1
#endif
constexpr unsigned kTileSub = ANM_TILE_SUBLISTS;     // lists per tile (a CTA appends to list blockIdx % kTileSub).  Same-address atomics serialise at the L2:
                                                     // 8 lists per tile took cfg3 from 559 to 348 ms per 1e9 decays, but cfg4 from 505 to 534 ms (more open
                                                     // write streams); neither beats direct atomics on cfg3 (238 ms), cfg4 gains 3 % at 1

template <int TALLY>
__device__ __forceinline__ void deposit(const TransportParams& p, float* __restrict__ tally, unsigned vox, float e) {
    ANM_CHK(p, 0, vox < p.n_vox && e >= 0.0f);
    if (TALLY == TALLY_WAGG) {
        // merge the deposits of lanes that hit the same voxel OF THE SAME BATCH in this trip: one RED per distinct word
        const unsigned act = __activemask();
        const unsigned peers = __match_any_sync(act, reinterpret_cast<unsigned long long>(tally + vox));
        float total = 0.0f;
        for (unsigned rem = peers; rem; rem &= rem - 1) total += __shfl_sync(peers, e, __ffs(rem) - 1);
        if ((threadIdx.x & 31) == (unsigned)(__ffs(peers) - 1)) atomicAdd(tally + vox, total);
    } else if (TALLY == TALLY_BINNED) {
        // append {voxel, energy} to the tile's list; the lanes of this trip that hit the same tile share one atomic
        const unsigned tile = (vox >> kTileShift) * kTileSub + (blockIdx.x & (kTileSub - 1u));
        const unsigned act = __activemask();
        const unsigned peers = __match_any_sync(act, tile);
        const int leader = __ffs(peers) - 1;
        unsigned base = 0;
        if ((int)(threadIdx.x & 31) == leader) base = atomicAdd(p.bin_cnt + tile, (unsigned)__popc(peers));
        base = __shfl_sync(peers, base, leader);
        const unsigned pos = base + __popc(peers & ((1u << (threadIdx.x & 31)) - 1u));
        const uint2 seg = __ldg(p.bin_seg + tile);
        if (pos < seg.y) __stcs(p.bin_rec + (size_t)seg.x + pos, make_uint2(vox, __float_as_uint(e)));
        else atomicAdd(tally + vox, e);              // the segment is full (or this is the counting batch): direct RED
    } else {
        atomicAdd(tally + vox, e);
    }
}

// Woodcock flight: two sub-steps from one Philox block (words x,y then z,w), stopping at the
// first real collision or escape.  A sub-step: exponential flight against the majorant, voxel lookup, real / virtual
// decision from one more uniform, which also picks the channel.
//
// The second sub-step is evaluated speculatively, as if the first were a virtual collision: its landing point, voxel
// index and majorant need no memory, so both texel loads are in flight together (one exposed L2 round trip per event
// instead of two) and the event is branch-free.  The arithmetic of each sub-step is exactly the sequential one.
//
// Hull majorant (reading C24), branch-free.  hull_bits: bit 0 = IN, the photon's last landing point (or its
// start) was inside the hull box; bit 1 = AWAY, the photon is outside the box and has flown straight since a point
// inside it.  A straight ray that has left a convex box never re-enters it, so an AWAY photon flies against the
// majorant of the voxels outside the box; every other photon against the global majorant, which is valid everywhere.
// A scatter clears AWAY (the caller does), a landing inside the box sets IN.
enum : int { FLY_GO = 0, FLY_ESCAPED = 1, FLY_PE = 2, FLY_COMPTON = 3, FLY_RAYLEIGH = 4 };

struct FlyCounters { unsigned steps, real; };

struct SubStep {        // one landing point
    float x, y, z, m_here;
    unsigned vox, hull_bits;
    bool inside;        // inside the grid (else the photon has escaped)
};

__device__ __forceinline__ SubStep fly_land(const TransportParams& p, const float x, const float y, const float z,
                                            const float u, const float v, const float w, const float maj,
                                            const float inv_maj, const float maj_out, const float inv_maj_out,
                                            const unsigned r_s, const unsigned hull_bits) {
    SubStep o;
    const float nl = -__logf(u01(r_s));
    const bool away = (hull_bits & 2u) != 0u;
    o.m_here = away ? maj_out : maj;
    const float s = nl * (away ? inv_maj_out : inv_maj);
    o.x = fmaf(s, u, x); o.y = fmaf(s, v, y); o.z = fmaf(s, w, z);
    const int ix = __float2int_rd(o.x * p.inv_dx), iy = __float2int_rd(o.y * p.inv_dy), iz = __float2int_rd(o.z * p.inv_dz);
    o.inside = (unsigned)ix < (unsigned)p.nx && (unsigned)iy < (unsigned)p.ny && (unsigned)iz < (unsigned)p.nz;
    o.hull_bits = hull_bits;
    if (p.hull) {
        const bool in = (unsigned)(ix - p.hx0) < (unsigned)p.hnx && (unsigned)(iy - p.hy0) < (unsigned)p.hny &&
                        (unsigned)(iz - p.hz0) < (unsigned)p.hnz;
        o.hull_bits = in ? 1u : ((hull_bits + 1u) & 2u);     // IN or AWAY -> AWAY; neither -> neither
    }
    o.vox = (unsigned)ix + (unsigned)p.nx * ((unsigned)iy + (unsigned)p.ny * (unsigned)iz);
    return o;
}

// A texel read of the Woodcock flight.  T16: from the 16-bit copy, expanded to the 32-bit format (13-bit density counts
// of 2^-12 g/cm^3 = that count << 8 in units of 2^-20): the SAME material and density values, half the bytes per
// random read and half the footprint in the L2 -- what matters once the volume no longer fits it (cfg4).
constexpr unsigned kT16DensityBits = 13, kT16Shift = 8;        // 2^-12 g/cm^3 steps, below 2 g/cm^3; material ids 0..7
template <bool T16>
__device__ __forceinline__ unsigned load_texel(const TransportParams& p, unsigned vox) {
    if (T16) {
        const unsigned t = __ldg(p.texels16 + vox);
        return ((t >> kT16DensityBits) << 24) | ((t & ((1u << kT16DensityBits) - 1u)) << kT16Shift);
    }
    return __ldg(p.texels + vox);
}

template <bool STATS, bool T16 = false>
__device__ __forceinline__ int fly_two(const TransportParams& p, const float* __restrict__ s_tot,
                                       const float2* __restrict__ s_pec, float& x, float& y, float& z,
                                       const float u, const float v, const float w, const int ie, const float fe,
                                       const float maj, const float inv_maj, const float maj_out, const float inv_maj_out,
                                       const uint4 r, unsigned& hull_bits, unsigned& vox, int& mat, FlyCounters& cnt) {
    const SubStep a = fly_land(p, x, y, z, u, v, w, maj, inv_maj, maj_out, inv_maj_out, r.x, hull_bits);
    const unsigned ta = a.inside ? load_texel<T16>(p, a.vox) : 0u;
    const SubStep b = fly_land(p, a.x, a.y, a.z, u, v, w, maj, inv_maj, maj_out, inv_maj_out, r.z, a.hull_bits);
    const bool b_inside = a.inside && b.inside;
    const unsigned tb = b_inside ? load_texel<T16>(p, b.vox) : 0u;
    // real / virtual: u' * majorant < rho * (mu/rho)_tot(E)
    const int mat_a = (int)(ta >> 24), mat_b = (int)(tb >> 24);
    ANM_CHK(p, 1, mat_a < p.nm && mat_b < p.nm && ie >= 0 && ie <= p.ne - 2 && (!a.inside || a.vox < p.n_vox) && (!b_inside || b.vox < p.n_vox));
    const float rho_a = (float)(ta & 0xffffffu) * kDensityStep, rho_b = (float)(tb & 0xffffffu) * kDensityStep;
    const float* row_a = s_tot + mat_a * p.ne + ie;
    const float* row_b = s_tot + mat_b * p.ne + ie;
    const float rr_a = u01(r.y) * a.m_here, rr_b = u01(r.w) * b.m_here;
    const bool real_a = a.inside && rr_a < rho_a * fmaf(fe, row_a[1] - row_a[0], row_a[0]);
    const bool real_b = b_inside && rr_b < rho_b * fmaf(fe, row_b[1] - row_b[0], row_b[0]);
    const bool first = real_a || !a.inside;            // the event ends at the first sub-step
    if (STATS) { cnt.steps += first ? 1u : 2u; cnt.real += (real_a || (!first && real_b)) ? 1u : 0u; }
    x = first ? a.x : b.x; y = first ? a.y : b.y; z = first ? a.z : b.z;
    hull_bits = first ? a.hull_bits : b.hull_bits;
    vox = first ? a.vox : b.vox;
    mat = first ? mat_a : mat_b;
    const float rho = first ? rho_a : rho_b, rr = first ? rr_a : rr_b;
    const bool escaped = !a.inside || (!real_a && !b.inside);
    const bool real = real_a || real_b;                // real_b implies a.inside; if real_a the first one counts
    // A5: the draw that accepted the collision also picks the channel: rr < mu_pe -> photoelectric,
    // < mu_pe + mu_compton -> Compton, else Rayleigh
    const float2 c0 = s_pec[mat * p.ne + ie], c1 = s_pec[mat * p.ne + ie + 1];
    const bool pe = rr < rho * fmaf(fe, c1.x - c0.x, c0.x);
    const bool co = rr < rho * fmaf(fe, c1.y - c0.y, c0.y) || !p.rayleigh_on;
    const int ch = pe ? FLY_PE : (co ? FLY_COMPTON : FLY_RAYLEIGH);
    return escaped ? FLY_ESCAPED : (real ? ch : FLY_GO);
}

// One Klein-Nishina try by composition-rejection on f(eps) = (1/eps + eps) g(eps).
// Returns true when accepted; then eps = E'/E and t = 1 - cos(theta).
__device__ __forceinline__ bool compton_try(const float E, const uint4 r, float& eps, float& t) {
    const float alpha = E * kInvE0;
    const float eps0 = __fdividef(1.0f, fmaf(2.0f, alpha, 1.0f));
    const float eps0sq = eps0 * eps0;
    const float a1 = -__logf(eps0);
    const float a2 = fmaf(0.5f, 1.0f - eps0sq, a1);
    const float u2 = u01(r.y);
    float epssq;
    if (a1 > a2 * u01(r.x)) { eps = __expf(-a1 * u2); epssq = eps * eps; }
    else { epssq = fmaf(1.0f - eps0sq, u2, eps0sq); eps = sqrtf(epssq); }
    t = __fdividef(1.0f - eps, alpha * eps);
    const float sint2 = fmaxf(0.0f, t * (2.0f - t));
    const float g = 1.0f - __fdividef(eps * sint2, 1.0f + epssq);
    return g >= u01(r.z);
}

// One Rayleigh try: x^2 from the material's cumulative form factor restricted to
// [0, (E/hc)^2], accepted with probability (1 + cos^2)/2.  Returns true when accepted; c = cos(theta).
__device__ __forceinline__ bool rayleigh_try(const float E, const uint4 r, const float* __restrict__ s_x2,
                                             const float* __restrict__ cum, const int n_x2, float& c) {
    const float xm = E * kKeVAngstromInv;
    const float T = xm * xm;
    int lo = 0, hi = n_x2 - 1;                       // A(T) on the piecewise-linear cumulative
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (s_x2[mid] <= T) lo = mid; else hi = mid; }
    const float A_T = fmaf(__fdividef(T - s_x2[lo], s_x2[hi] - s_x2[lo]), cum[hi] - cum[lo], cum[lo]);
    const float target = u01(r.x) * A_T;
    lo = 0; hi = n_x2 - 1;
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (cum[mid] <= target) lo = mid; else hi = mid; }
    float x2 = s_x2[lo];
    const float dc = cum[hi] - cum[lo];
    if (dc > 0.0f) x2 = fmaf(__fdividef(target - cum[lo], dc), s_x2[hi] - s_x2[lo], x2);
    x2 = fminf(x2, T);
    c = fmaf(-2.0f, __fdividef(x2, T), 1.0f);
    return 2.0f * u01(r.y) <= fmaf(c, c, 1.0f);
}

__device__ __forceinline__ bool hull_in(const TransportParams& p, int ix, int iy, int iz) {
    return p.hull && (unsigned)(ix - p.hx0) < (unsigned)p.hnx && (unsigned)(iy - p.hy0) < (unsigned)p.hny &&
           (unsigned)(iz - p.hz0) < (unsigned)p.hnz;
}

// A2 + A3: the decay of history h: voxel pick (alias table, 64 random bits for the bin), uniform point in the voxel,
// isotropic direction.  Philox stream 0, blocks 0 and 1.  Returns the decay voxel; in_box = hull_in(decay voxel).
__device__ __forceinline__ unsigned sample_source(const TransportParams& p, const unsigned long long h, float& x, float& y,
                                                  float& z, float& u, float& v, float& w, bool& in_box) {
    const uint4 r = philox4x32_10(make_uint4((unsigned)h, (unsigned)(h >> 32), 0u, 0u), p);
    const uint4 r2 = philox4x32_10(make_uint4((unsigned)h, (unsigned)(h >> 32), 1u, 0u), p);
    unsigned voxel, ix, iy, iz;
    if (p.point_source) {
        x = p.px; y = p.py; z = p.pz;
        ix = (unsigned)__float2int_rd(x * p.inv_dx); iy = (unsigned)__float2int_rd(y * p.inv_dy);
        iz = (unsigned)__float2int_rd(z * p.inv_dz);
        voxel = ix + (unsigned)p.nx * (iy + (unsigned)p.ny * iz);
    } else {
        const unsigned long long r64 = ((unsigned long long)r.x << 32) | r.y;
        const unsigned j = (unsigned)__umul64hi(r64, (unsigned long long)p.n_alias);
        ANM_CHK(p, 2, j < p.n_alias);
        const uint4 a = __ldcs(p.alias + j);      // one use per decay, 16 B out of ~100 MB: evict-first, keep L2 for texels + tally
        voxel = (r.z < a.x) ? a.y : a.z;
        ANM_CHK(p, 3, voxel < p.n_vox);
        const unsigned nxy = (unsigned)p.nx * (unsigned)p.ny;
        iz = voxel / nxy;
        const unsigned rem = voxel - iz * nxy;
        iy = rem / (unsigned)p.nx; ix = rem - iy * (unsigned)p.nx;
        x = ((float)ix + u01(r.w)) * p.dx;       // uniform inside the voxel
        y = ((float)iy + u01(r2.x)) * p.dy;
        z = ((float)iz + u01(r2.y)) * p.dz;
    }
    in_box = hull_in(p, (int)ix, (int)iy, (int)iz);
    const float ct = fmaf(2.0f, u01(r2.z), -1.0f);    // isotropic direction
    const float st = sqrtf(fmaxf(0.0f, fmaf(-ct, ct, 1.0f)));
    float sp, cp;
    __sincosf(kTwoPi * u01(r2.w), &sp, &cp);
    u = st * cp; v = st * sp; w = ct;
    return voxel;
}

// ------------------------------------------------------------------------------------------------
// Secondary electrons (electrons are followed down to a 200 keV cutoff, the rest is deposited locally;
// DESIGN.md reading C28): continuous slowing down along a straight line.  r = R_m(T) is the residual mass range above
// the cutoff (piecewise linear in T); a chord l through a voxel of density rho leaves r' = r - rho l and
// T' = R_m^{-1}(r'); T - T' goes into the voxel; r' <= 0: the electron reaches the cutoff here and all of T is local.
// Starts in voxel `vox` (the photon's collision voxel) at (x, y, z) with unit direction (ex, ey, ez).  Returns the
// energy carried out of the grid.  No random numbers: photon histories are the same with and without it.
__device__ __forceinline__ float e_range_of(const TransportParams& p, const float* __restrict__ R, float T, int& k) {
    const float xq = fmaxf((T - p.t_min) * p.e_inv_dt, 0.0f);
    k = min((int)xq, p.n_t - 2);
    const float r0 = R[k], r1 = R[k + 1];
    return fmaf(xq - (float)k, r1 - r0, r0);
}

// `er` = the range tables [nm][n_t] (the transport kernel's shared-memory copy, or p.e_range).
// dep(voxel, energy) receives the deposits: a RED into the batch tally, or an append to the decay's list (HBH).
template <class Dep>
__device__ __forceinline__ float electron_walk_to(const TransportParams& p, const float* __restrict__ er, float x, float y, float z,
                                               float ex, float ey, float ez, unsigned vox, float T, Dep dep) {
    const unsigned nxy = (unsigned)p.nx * (unsigned)p.ny;
    int iz = (int)(vox / nxy);
    const unsigned rem = vox - (unsigned)iz * nxy;
    int iy = (int)(rem / (unsigned)p.nx), ix = (int)(rem - (unsigned)iy * (unsigned)p.nx);
    const float inf = __int_as_float(0x7f800000);
    // distance along the ray to the next face on each axis, and between faces
    float tx = ex > 0.0f ? __fdividef((float)(ix + 1) * p.dx - x, ex) : (ex < 0.0f ? __fdividef((float)ix * p.dx - x, ex) : inf);
    float ty = ey > 0.0f ? __fdividef((float)(iy + 1) * p.dy - y, ey) : (ey < 0.0f ? __fdividef((float)iy * p.dy - y, ey) : inf);
    float tz = ez > 0.0f ? __fdividef((float)(iz + 1) * p.dz - z, ez) : (ez < 0.0f ? __fdividef((float)iz * p.dz - z, ez) : inf);
    tx = fmaxf(tx, 0.0f); ty = fmaxf(ty, 0.0f); tz = fmaxf(tz, 0.0f);
    const float dtx = ex != 0.0f ? fabsf(__fdividef(p.dx, ex)) : inf, dty = ey != 0.0f ? fabsf(__fdividef(p.dy, ey)) : inf,
                dtz = ez != 0.0f ? fabsf(__fdividef(p.dz, ez)) : inf;
    float t = 0.0f;
    for (;;) {
        ANM_CHK(p, 4, vox < p.n_vox);
        const unsigned texel = __ldg(p.texels + vox);
        const float rho = (float)(texel & 0xffffffu) * kDensityStep;
        const float* R = er + (texel >> 24) * (unsigned)p.n_t;
        const float t_next = fminf(tx, fminf(ty, tz));
        int k;
        const float r = e_range_of(p, R, T, k);
        const float r_new = r - rho * (t_next - t);
        if (!(r_new > 0.0f)) { dep(vox, T); return 0.0f; }
        while (k > 0 && R[k] > r_new) --k;                         // segment with R[k] <= r_new < R[k+1]
        const float r0 = R[k], r1 = R[k + 1];
        const float T_new = fmaf((float)k + __fdividef(r_new - r0, r1 - r0), p.e_dt, p.t_min);
        if (T > T_new) dep(vox, T - T_new);
        T = fminf(T, T_new);
        t = t_next;
        if (tx <= ty && tx <= tz) { ix += ex > 0.0f ? 1 : -1; tx += dtx; if ((unsigned)ix >= (unsigned)p.nx) return T; }
        else if (ty <= tz) { iy += ey > 0.0f ? 1 : -1; ty += dty; if ((unsigned)iy >= (unsigned)p.ny) return T; }
        else { iz += ez > 0.0f ? 1 : -1; tz += dtz; if ((unsigned)iz >= (unsigned)p.nz) return T; }
        vox = (unsigned)ix + (unsigned)p.nx * ((unsigned)iy + (unsigned)p.ny * (unsigned)iz);
    }
}

// `tally`: the energy volume of the batch the electron's decay belongs to
__device__ __forceinline__ float electron_walk(const TransportParams& p, float* __restrict__ tally, const float* __restrict__ er, float x, float y,
                                            float z, float ex, float ey, float ez, unsigned vox, float T) {
    return electron_walk_to(p, er, x, y, z, ex, ey, ez, vox, T, [&](unsigned v, float e) { atomicAdd(tally + v, e); });
}

// inspection / parity hook (anm_trace_electrons): one given electron per thread, in = {x, y, z (cm), ex, ey, ez, T}
__global__ void electron_trace_kernel(const __grid_constant__ TransportParams p, const float* __restrict__ in, unsigned n,
                                      double* __restrict__ escaped) {
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float* e = in + 7 * (size_t)i;
    const float x = e[0], y = e[1], z = e[2];
    const int ix = __float2int_rd(x * p.inv_dx), iy = __float2int_rd(y * p.inv_dy), iz = __float2int_rd(z * p.inv_dz);
    const unsigned vox = (unsigned)ix + (unsigned)p.nx * ((unsigned)iy + (unsigned)p.ny * (unsigned)iz);
    const float out = electron_walk(p, p.batch, p.e_range, x, y, z, e[3], e[4], e[5], vox, e[6]);
    if (out > 0.0f) atomicAdd(escaped, (double)out);
}

template <bool STATS, int TALLY>
__global__ void __launch_bounds__(kThreads, kMinBlocksPerSM)
transport_kernel(const __grid_constant__ TransportParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* s_pec = reinterpret_cast<float2*>(smem_raw);            // [nm*ne]
    float* s_tot = reinterpret_cast<float*>(s_pec + p.nm * p.ne);   // [nm*ne]
    float* s_maj = s_tot + p.nm * p.ne;                             // [ne]
    float* s_majo = s_maj + p.ne;                                   // [ne]  majorant outside the hull box
    float* s_x2 = s_majo + p.ne;                                    // [n_x2]
    float* s_cum = s_x2 + p.n_x2;                                   // [nm*n_x2]
    float* s_stash = s_cum + p.nm * p.n_x2;                         // [6][kThreads]
    for (int i = threadIdx.x; i < p.nm * p.ne; i += kThreads) { s_pec[i] = p.tab_pec[i]; s_tot[i] = p.tab_tot[i]; }
    for (int i = threadIdx.x; i < p.ne; i += kThreads) { s_maj[i] = p.tab_maj[i]; s_majo[i] = p.tab_maj_out[i]; }
    for (int i = threadIdx.x; i < p.n_x2; i += kThreads) s_x2[i] = p.ray_x2[i];
    for (int i = threadIdx.x; i < p.nm * p.n_x2; i += kThreads) s_cum[i] = p.ray_cum[i];
    __syncthreads();

    const unsigned lane = threadIdx.x & 31u;
    const unsigned lanemask_lt = (1u << lane) - 1u;
    float* stash = s_stash + threadIdx.x;

    int state = ST_NEED, photon = 0, mat = 0, ie = 0;
    unsigned hl = 0, blk = 0, vox = 0, hb = 0, hb_src = 0;
    float x = 0, y = 0, z = 0, u = 0, v = 0, w = 1, E = 0, fe = 0, maj = 1, inv_maj = 1, majo = 1, inv_majo = 1;
    unsigned pool_next = 0, pool_end = 0;   // warp-uniform
    bool exhausted = false;                 // warp-uniform

    float esc = 0.0f;
    unsigned c_pe = 0, c_co = 0, c_ra = 0, c_esc = 0, c_cut = 0;
    FlyCounters fc = {0u, 0u};

    const float t0 = (float)p.ie0 + p.fe0;  // ln-E grid coordinate of E0
    const float t_max = (float)(p.ne - 1) - 1.0f / 1024.0f;
    // energy-dependent quantities from the ln-E grid coordinate t (the same arithmetic as schedule 2)
    auto set_t = [&](float t) {
        ie = (int)t; fe = t - (float)ie;
        maj = fmaf(fe, s_maj[ie + 1] - s_maj[ie], s_maj[ie]);
        inv_maj = __fdividef(1.0f, maj);
        majo = fmaf(fe, s_majo[ie + 1] - s_majo[ie], s_majo[ie]);
        inv_majo = __fdividef(1.0f, majo);
    };
    auto set_energy = [&](float e) { set_t(fminf(fmaxf((__logf(e) - p.lnE_min) * p.inv_dlnE, 0.0f), t_max)); };

    for (;;) {
        // ---- hand out history indices --------------------------------------------------------
        const unsigned need = __ballot_sync(0xffffffffu, state == ST_NEED);
        if (need) {
            if (pool_next == pool_end && !exhausted) {
                unsigned base = 0;
                if (lane == 0) base = atomicAdd(p.counter, kChunk);
                base = __shfl_sync(0xffffffffu, base, 0);
                pool_next = min(base, p.n_hist);
                pool_end = min(base + kChunk, p.n_hist);
                exhausted = (pool_next == pool_end);
            }
            const unsigned avail = pool_end - pool_next;
            const unsigned rank = __popc(need & lanemask_lt);
            if (state == ST_NEED) {
                if (rank < avail) { hl = pool_next + rank; blk = 0; state = ST_SOURCE; }
                else if (exhausted) state = ST_DONE;
            }
            pool_next += min((unsigned)__popc(need), avail);
        }
        if (__all_sync(0xffffffffu, state == ST_DONE)) break;
        if (state == ST_NEED || state == ST_DONE) continue;

        const unsigned long long h = p.hist_base + hl;
        bool dead = false;
        if (state == ST_SOURCE) {
            bool in_box;
            const unsigned voxel = sample_source(p, h, x, y, z, u, v, w, in_box);
            stash[0 * kThreads] = x; stash[1 * kThreads] = y; stash[2 * kThreads] = z;
            stash[3 * kThreads] = u; stash[4 * kThreads] = v; stash[5 * kThreads] = w;
            if (p.positron_ke > 0.0f) deposit<TALLY>(p, p.batch, voxel, p.positron_ke);
            E = kE0; set_t(t0);
            hb_src = in_box ? 1u : 0u; hb = hb_src;
            photon = 0; blk = 0; state = ST_FLY;
            continue;
        }

        // ---- one Philox block per live photon --------------------------------------------------
        const uint4 r = philox4x32_10(make_uint4((unsigned)h, (unsigned)(h >> 32), blk, 1u + (unsigned)photon), p);
        ++blk;
        if (state == ST_FLY) {
            const int code = fly_two<STATS>(p, s_tot, s_pec, x, y, z, u, v, w, ie, fe, maj, inv_maj, majo, inv_majo, r, hb, vox, mat, fc);
            ANM_TR("S1 h=%llu ph=%d blk=%u FLY code=%d E=%.9g t=%d+%.9g pos=%.9g %.9g %.9g vox=%u hb=%u\n", h, photon, blk - 1, code, E, ie, fe, x, y, z, vox, hb);
            if (code == FLY_ESCAPED) { if (STATS) { esc += E; ++c_esc; } dead = true; }
            else if (code == FLY_PE) { if (STATS) ++c_pe; deposit<TALLY>(p, p.batch, vox, E); dead = true; }   // all energy local
            else if (code == FLY_COMPTON) state = ST_COMPTON;
            else if (code == FLY_RAYLEIGH) state = ST_RAYLEIGH;
        } else if (state == ST_COMPTON) {
            float eps, t;
            if (compton_try(E, r, eps, t)) {
                if (STATS) ++c_co;
                float dep = E * (1.0f - eps);     // recoil electron deposited locally
                E *= eps;
                if (E < p.cutoff) { dep += E; dead = true; if (STATS) ++c_cut; }
                else { rotate(u, v, w, 1.0f - t, kTwoPi * u01(r.w)); set_energy(E); hb &= 1u; state = ST_FLY; }
                deposit<TALLY>(p, p.batch, vox, dep);
            }
        } else {   // ST_RAYLEIGH
            float c;
            if (rayleigh_try(E, r, s_x2, s_cum + mat * p.n_x2, p.n_x2, c)) {
                if (STATS) ++c_ra;
                rotate(u, v, w, c, kTwoPi * u01(r.z));
                set_energy(E);      // E is unchanged; recomputed like schedule 2, whose slot held the voxel in its place
                hb &= 1u;
                state = ST_FLY;
            }
        }

        if (dead) {
            if (photon == 0 && p.photons_per_decay == 2) {   // the partner photon: same point, opposite direction
                photon = 1; blk = 0; state = ST_FLY; hb = hb_src;
                x = stash[0 * kThreads]; y = stash[1 * kThreads]; z = stash[2 * kThreads];
                u = -stash[3 * kThreads]; v = -stash[4 * kThreads]; w = -stash[5 * kThreads];
                E = kE0; set_t(t0);
            } else {
                state = ST_NEED;
            }
        }
    }

    if (STATS) {
        unsigned c_steps = fc.steps, c_real = fc.real;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            esc += __shfl_xor_sync(0xffffffffu, esc, o);
            c_steps += __shfl_xor_sync(0xffffffffu, c_steps, o);
            c_real += __shfl_xor_sync(0xffffffffu, c_real, o);
            c_pe += __shfl_xor_sync(0xffffffffu, c_pe, o);
            c_co += __shfl_xor_sync(0xffffffffu, c_co, o);
            c_ra += __shfl_xor_sync(0xffffffffu, c_ra, o);
            c_esc += __shfl_xor_sync(0xffffffffu, c_esc, o);
            c_cut += __shfl_xor_sync(0xffffffffu, c_cut, o);
        }
        if (lane == 0) {
            atomicAdd(&p.stats->escaped_MeV, (double)esc);
            atomicAdd(&p.stats->n_steps, (unsigned long long)c_steps);
            atomicAdd(&p.stats->n_real, (unsigned long long)c_real);
            atomicAdd(&p.stats->n_pe, (unsigned long long)c_pe);
            atomicAdd(&p.stats->n_compton, (unsigned long long)c_co);
            atomicAdd(&p.stats->n_rayleigh, (unsigned long long)c_ra);
            atomicAdd(&p.stats->n_escaped, (unsigned long long)c_esc);
            atomicAdd(&p.stats->n_cutoff, (unsigned long long)c_cut);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// History-by-history scoring.  X_h = the energy ONE decay (positron energy,
// both photons) leaves in a voxel; the estimator needs sum_h X_h^2, so the deposits of a decay cannot go to the tally
// one by one.  They are appended to the decay slot's list; the list is merged per voxel -- each distinct voxel gets one
// RED into the batch tally (X) and one into hbh_sq (X^2) -- when the freed slot is handed its next history (the SOURCE
// event, up to 32 slots at once) or, for the last decays of a launch, in a sweep at the end.  A decay with more than
// kHbhCap deposits is merged early (its X is then split in two; counted in n_hbh_overflow, expected 0).
constexpr unsigned kHbhCap = 63;
constexpr unsigned kHbhShift = 26;          // the list length lives in bits 26-31 of the slot's history word (shared memory)
constexpr unsigned kHbhHistMask = (1u << kHbhShift) - 1u;   // so a launch may hold at most 2^26 histories in this mode

// hl = the slot's history word in shared memory: history index of the launch | list length << 26
// The first kHbhReg entries of the list are fetched by independent loads (one exposed latency instead of a chain of
// dependent ones) and merged per voxel in registers; a longer list (rare: a decay leaves ~7 deposits) folds its tail
// into them where the voxel matches and handles what is left entry by entry.
constexpr int kHbhReg = 12;
__device__ __forceinline__ void hbh_flush(const TransportParams& p, float* __restrict__ tally, unsigned gslot, unsigned& hl) {
    const uint2* L = p.hbh_list + gslot;
    const unsigned n = hl >> kHbhShift;
    hl &= kHbhHistMask;
    if (n == 0u) return;
    constexpr unsigned kNone = 0xffffffffu;
    unsigned vx[kHbhReg];
    float ex[kHbhReg];
#pragma unroll
    for (int k = 0; k < kHbhReg; ++k) {
        const uint2 a = (unsigned)k < n ? L[(size_t)k * p.hbh_nslots] : make_uint2(kNone, 0u);
        vx[k] = a.x; ex[k] = __uint_as_float(a.y);
    }
    // tail (n > kHbhReg): add an entry to the register entry of the same voxel, else merge it with the later tail entries
    // of its voxel here (an earlier tail entry of the same voxel has already taken it: skip)
    for (unsigned j = kHbhReg; j < n; ++j) {
        const uint2 b = L[(size_t)j * p.hbh_nslots];
        bool taken = false;
#pragma unroll
        for (int k = 0; k < kHbhReg; ++k)
            if (!taken && vx[k] == b.x) { ex[k] += __uint_as_float(b.y); taken = true; }
        for (unsigned i = kHbhReg; i < j && !taken; ++i) taken = (L[(size_t)i * p.hbh_nslots].x == b.x);
        if (taken) continue;
        float X = __uint_as_float(b.y);
        for (unsigned i = j + 1; i < n; ++i) {
            const uint2 c = L[(size_t)i * p.hbh_nslots];
            if (c.x == b.x) X += __uint_as_float(c.y);
        }
        atomicAdd(tally + b.x, X);
        atomicAdd(p.hbh_sq + b.x, X * X);
    }
    // register entries: every later entry of the same voxel is added to the first one and retired
#pragma unroll
    for (int k = 0; k < kHbhReg; ++k) {
        if (vx[k] == kNone) continue;
        float X = ex[k];
#pragma unroll
        for (int m = k + 1; m < kHbhReg; ++m)
            if (vx[m] == vx[k]) { X += ex[m]; vx[m] = kNone; }
        atomicAdd(tally + vx[k], X);
        atomicAdd(p.hbh_sq + vx[k], X * X);
    }
}

__device__ __forceinline__ void hbh_push(const TransportParams& p, float* __restrict__ tally, unsigned gslot, unsigned& hl, unsigned vox, float e, unsigned& overflow) {
    if ((hl >> kHbhShift) == kHbhCap) { hbh_flush(p, tally, gslot, hl); ++overflow; }
    ANM_CHK(p, 5, (hl >> kHbhShift) < kHbhCap && gslot < p.hbh_nslots && vox < p.n_vox);
    p.hbh_list[gslot + (size_t)(hl >> kHbhShift) * p.hbh_nslots] = make_uint2(vox, __float_as_uint(e));
    hl += 1u << kHbhShift;
}

// ------------------------------------------------------------------------------------------------
// Schedule 2: event-based at warp scope.  Each warp owns kSlots decay slots in shared memory (SoA, one word per
// field per slot; two banks of photon state, bank 0 = photon A, bank 1 = photon B, both written at the decay) and
// four ring queues of slot numbers, one per event type (FLY, COMPTON, SOURCE = free, RAYLEIGH).  A trip: pick the
// event type with the longest queue, pop up to 32 slots, run that ONE event with (nearly) all lanes active, push every
// slot onto the queue of its next event (ballot + prefix popcount).  A slot whose decay is complete is free and waits
// for SOURCE, which hands it the next history index of the launch: regenerate in place, compact by event type, no
// global queues and no extra HBM traffic.  Same Philox counters and per-event arithmetic as schedule 1: the two
// schedules produce the same histories; only the order of the fp32 atomics differs.
#ifndef ANM_POOL_THREADS
#define ANM_POOL_THREADS 1024
#endif

#ifndef ANM_POOL_MIN_BLOCKS
#define ANM_POOL_MIN_BLOCKS 1
#endif
constexpr int kPoolThreads = ANM_POOL_THREADS;
constexpr int kPoolWarps = kPoolThreads / 32;
constexpr int kPoolMinBlocksPerSM = ANM_POOL_MIN_BLOCKS;
constexpr int kSlots = 64;                  // per warp (a power of two: the queues are rings)
constexpr unsigned kPend = 64;              // capacity of a warp's array of waiting electrons (ELEC)
constexpr unsigned kEFields = 9;            // x, y, z, ex, ey, ez, T, voxel, local batch of the decay
#ifndef ANM_RAYBATCH
#define ANM_RAYBATCH 8
#endif
constexpr int kRayleighBatch = ANM_RAYBATCH;           // run the (rare) Rayleigh event once this many slots wait for it
// photon bank fields (bank b at word offset b * kBankFields * kSlots)
enum : int { F_X = 0, F_Y, F_Z, F_U, F_V, F_W, F_E, F_TV /* FLY: ln-E grid coordinate; COMPTON/RAYLEIGH: voxel */,
             kBankFields, F_HL = 2 * kBankFields, F_META, kSlotFields };
// meta = photon (bit 0) | hull bits IN, AWAY (bits 1-2) | decay voxel inside the hull box (bit 3) | material (bits 4-6)
//        | local batch of the decay within the launch's batch group (bits 8-15) | Philox block counter (bits 16-31)
constexpr unsigned kBlkInc = 1u << 16;      // one more Philox block
constexpr unsigned kMaxGroup = 256;         // batches per launch (8 bits of the meta word)
enum : int { Q_F = 0, Q_C = 1, Q_S = 2, Q_R = 3, Q_NONE = 4 };
constexpr size_t kPoolWarpBytes = (size_t)kSlotFields * kSlots * 4 + 4 * kSlots;   // slots + the four queues (bytes)

template <bool STATS, bool ELEC, bool HBH, int TALLY = TALLY_RED, bool T16 = false>
__global__ void __launch_bounds__(kPoolThreads, kPoolMinBlocksPerSM)
transport_pool_kernel(const __grid_constant__ TransportParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* s_pec = reinterpret_cast<float2*>(smem_raw);            // [nm*ne]
    float* s_tot = reinterpret_cast<float*>(s_pec + p.nm * p.ne);   // [nm*ne]
    float* s_maj = s_tot + p.nm * p.ne;                             // [ne]
    float* s_majo = s_maj + p.ne;                                   // [ne]
    float* s_x2 = s_majo + p.ne;                                    // [n_x2]
    float* s_cum = s_x2 + p.n_x2;                                   // [nm*n_x2]
    float* s_er = s_cum + p.nm * p.n_x2;                            // [nm*n_t] electron range tables (ELEC only)
    unsigned char* s_pool = reinterpret_cast<unsigned char*>(s_er + (ELEC ? p.e_nm * p.n_t : 0));
    if (ELEC) for (int i = threadIdx.x; i < p.e_nm * p.n_t; i += kPoolThreads) s_er[i] = p.e_range[i];
    for (int i = threadIdx.x; i < p.nm * p.ne; i += kPoolThreads) { s_pec[i] = p.tab_pec[i]; s_tot[i] = p.tab_tot[i]; }
    for (int i = threadIdx.x; i < p.ne; i += kPoolThreads) { s_maj[i] = p.tab_maj[i]; s_majo[i] = p.tab_maj_out[i]; }
    for (int i = threadIdx.x; i < p.n_x2; i += kPoolThreads) s_x2[i] = p.ray_x2[i];
    for (int i = threadIdx.x; i < p.nm * p.n_x2; i += kPoolThreads) s_cum[i] = p.ray_cum[i];

    const unsigned lane = threadIdx.x & 31u;
    const unsigned lanemask_lt = (1u << lane) - 1u;
    float* slots = reinterpret_cast<float*>(s_pool + (size_t)(threadIdx.x >> 5) * kPoolWarpBytes);
    unsigned* slots_u = reinterpret_cast<unsigned*>(slots);
    unsigned char* q = reinterpret_cast<unsigned char*>(slots + kSlotFields * kSlots);   // [4][kSlots]
#pragma unroll
    for (int k = 0; k < kSlots / 32; ++k) q[Q_S * kSlots + lane + 32 * k] = (unsigned char)(lane + 32 * k);   // all free
    if (HBH) for (int k = 0; k < kSlots / 32; ++k) slots_u[F_HL * kSlots + lane + 32 * k] = 0u;                  // empty deposit lists
    __syncthreads();

    // ring heads and lengths, one byte per event type (byte Q_F .. Q_R), warp-uniform; all slots start free (Q_S)
    unsigned heads = 0u, cnts = (unsigned)kSlots << (8 * Q_S);
    unsigned pool_next = 0, pool_end = 0;   // warp-uniform
    bool exhausted = false;                 // warp-uniform
    // History indices are taken from the launch's counter in chunks, one atomic per chunk, asked for before the warp runs
    // out (the reply is read a few trips later, so its latency never shows).  Guided sizes: kChunk while much of the
    // launch is left, kChunkTail once fewer than two full chunks per warp of the grid remain -- the warps then finish
    // within a few decays of each other instead of up to kChunk decays apart (the drain at the end of a launch).
    unsigned pend_base = 0, pend_take = 0;  // pend_base: lane 0
    bool pend_valid = false;                // warp-uniform
    const unsigned tail_zone = gridDim.x * (unsigned)kPoolWarps * kChunk * 2u;
    auto chunk_size = [&](const unsigned seen) { return (p.n_hist - min(seen, p.n_hist) > tail_zone) ? kChunk : kChunkTail; };
    const float t0 = (float)p.ie0 + p.fe0;  // ln-E grid coordinate of E0
    const float t_max = (float)(p.ne - 1) - 1.0f / 1024.0f;

    float esc = 0.0f;
    unsigned c_pe = 0, c_co = 0, c_ra = 0, c_esc = 0, c_cut = 0, c_el = 0, c_ovf = 0, c_fly = 0, c_ctry = 0, c_rtry = 0;
    FlyCounters fc = {0u, 0u};
    const unsigned gslot0 = (blockIdx.x * (unsigned)kPoolWarps + (threadIdx.x >> 5)) * (unsigned)kSlots;   // HBH: this warp's lists

    // the tally of the batch a slot's decay belongs to (meta bits 8-15 = its local batch within the launch's group)
    auto tally_of = [&](const unsigned meta) { return p.batch + (size_t)((meta >> 8) & 0xffu) * p.batch_stride; };

    // Push every processed slot onto the ring of its next event (all 32 lanes call it; idle lanes pass Q_NONE):
    // one match groups the lanes by destination, the rank inside the group is the ring offset, one packed warp
    // reduction counts the four groups (head + length per byte stays below 128: no carry between the bytes).
    auto push_all = [&](const int next, const unsigned slot) {
        const unsigned same = __match_any_sync(0xffffffffu, next);
        const unsigned rank = __popc(same & lanemask_lt);
        const unsigned sh = 8u * (unsigned)(next & 3);
        if (next != Q_NONE)
            q[next * kSlots + ((((heads + cnts) >> sh) + rank) & (kSlots - 1))] = (unsigned char)slot;
        cnts += __reduce_add_sync(0xffffffffu, next != Q_NONE ? 1u << sh : 0u);
    };

    // ELEC: electrons set free by this warp's photons wait in a per-warp array (global scratch, [field][kPend]) and are
    // walked 32 at a time by all lanes -- inside the COMPTON event only the quarter of the lanes whose recoil electron
    // exceeds the cutoff would walk while the others wait.  pend < 32 between trips, so an event adds at most 32 more.
    unsigned pend = 0;                      // warp-uniform
    float* ering = ELEC ? p.e_ring + (size_t)(gslot0 / (unsigned)kSlots) * (kEFields * kPend) : nullptr;
    bool e_want = false;
    float e_x = 0, e_y = 0, e_z = 0, e_ex = 0, e_ey = 0, e_ez = 1, e_T = 0;
    unsigned e_vox = 0, e_bl = 0;
    auto e_append = [&]() {                 // all 32 lanes call it
        const unsigned b = __ballot_sync(0xffffffffu, e_want);
        if (b) {
            if (e_want) {
                ANM_CHK(p, 6, pend + __popc(b & lanemask_lt) < kPend);
                float* E = ering + pend + __popc(b & lanemask_lt);
                E[0 * kPend] = e_x; E[1 * kPend] = e_y; E[2 * kPend] = e_z;
                E[3 * kPend] = e_ex; E[4 * kPend] = e_ey; E[5 * kPend] = e_ez;
                E[6 * kPend] = e_T; E[7 * kPend] = __uint_as_float(e_vox); E[8 * kPend] = __uint_as_float(e_bl);
            }
            pend += __popc(b);
            e_want = false;
        }
    };
    auto e_drain = [&](const unsigned min_fill) {
        while (pend >= min_fill && pend > 0u) {
            __syncwarp();
            const unsigned n = min(pend, 32u);
            pend -= n;
            if (lane < n) {
                const float* E = ering + pend + lane;
                const float out = electron_walk(p, p.batch + (size_t)__float_as_uint(E[8 * kPend]) * p.batch_stride, s_er, E[0 * kPend],
                                                E[1 * kPend], E[2 * kPend], E[3 * kPend], E[4 * kPend], E[5 * kPend],
                                                __float_as_uint(E[7 * kPend]), E[6 * kPend]);
                if (STATS) { esc += out; ++c_el; }
            }
            __syncwarp();
        }
    };

    for (;;) {
        __syncwarp();
        // ---- pick the event type with the longest queue ------------------------------------------------
        const unsigned nF = cnts & 255u, nC = (cnts >> 8) & 255u, nS = (cnts >> 16) & 255u, nR = cnts >> 24;
        ANM_CHK(p, 7, nF + nC + nS + nR == (unsigned)kSlots);      // every slot waits in exactly one ring between trips
        int X = Q_F;
        unsigned best = nF;
        if (nC > best) { X = Q_C; best = nC; }
        if (!exhausted && nS > best) { X = Q_S; best = nS; }
        if (nR > best || nR >= (unsigned)kRayleighBatch) { X = Q_R; best = nR; }
        if (best == 0u) break;              // every slot is free and the launch has no history left
        unsigned n = min(best, 32u);
        unsigned hl_new = 0;
        if (X == Q_S) {                     // hand out history indices (warp-uniform bookkeeping)
            if (pool_next == pool_end) {
                // the chunk asked for at the end of an earlier SOURCE trip (its atomic has been in flight since), else now
                if (!pend_valid) { pend_take = chunk_size(pool_end); if (lane == 0) pend_base = atomicAdd(p.counter, pend_take); }
                const unsigned base = __shfl_sync(0xffffffffu, pend_base, 0);
                pend_valid = false;
                pool_next = min(base, p.n_hist);
                pool_end = min(base + pend_take, p.n_hist);
                if (pool_next == pool_end) { exhausted = true; continue; }
            }
            n = min(n, pool_end - pool_next);
            hl_new = pool_next + lane;
            pool_next += n;
            if (pool_end - pool_next < 32u && !pend_valid) {      // ask for the next chunk now, use it a few trips later
                pend_take = chunk_size(pool_end);
                if (lane == 0) pend_base = atomicAdd(p.counter, pend_take);
                pend_valid = true;
            }
        }
        const unsigned shX = 8u * (unsigned)X;
        const unsigned head = heads >> shX;
        heads = (heads + (n << shX)) & (0x01010101u * (unsigned)(kSlots - 1));     // pop n slots
        cnts -= n << shX;
        const unsigned slot = q[X * kSlots + ((head + lane) & (kSlots - 1))];
        const bool active = lane < n;
        ANM_CHK(p, 8, !active || slot < (unsigned)kSlots);
        float* S = slots + slot;
        unsigned* SU = slots_u + slot;
        int next = Q_NONE;

        // a finished photon: start the partner (bank 1, written at the decay) or free the slot
        auto photon_ends = [&](unsigned meta) {
            if (!(meta & 1u) && p.photons_per_decay == 2) {
                SU[F_META * kSlots] = 1u | (meta & 0xff08u) | ((meta & 8u) >> 2);   // photon B, block 0, IN = decay voxel's, same batch
                next = Q_F;
            } else {
                next = Q_S;
            }
        };

        if (X == Q_F) {
            if (active) {
                const unsigned meta = SU[F_META * kSlots];
                const unsigned ph = meta & 1u;
                const unsigned long long h = p.hist_base + (HBH ? SU[F_HL * kSlots] & kHbhHistMask : SU[F_HL * kSlots]);
                const uint4 r = philox4x32_10(make_uint4((unsigned)h, (unsigned)(h >> 32), meta >> 16, 1u + ph), p);
                float* Bk = S + ph * (kBankFields * kSlots);
                float x = Bk[F_X * kSlots], y = Bk[F_Y * kSlots], z = Bk[F_Z * kSlots];
                const float u = Bk[F_U * kSlots], v = Bk[F_V * kSlots], w = Bk[F_W * kSlots];
                const float t = Bk[F_TV * kSlots];
                const int ie = (int)t;
                const float fe = t - (float)ie;
                const float maj = fmaf(fe, s_maj[ie + 1] - s_maj[ie], s_maj[ie]);
                const float inv_maj = __fdividef(1.0f, maj);
                const float majo = fmaf(fe, s_majo[ie + 1] - s_majo[ie], s_majo[ie]);
                const float inv_majo = __fdividef(1.0f, majo);
                unsigned vox = 0, hb = (meta >> 1) & 3u;
                int mat = 0;
                const int code = fly_two<STATS, T16>(p, s_tot, s_pec, x, y, z, u, v, w, ie, fe, maj, inv_maj, majo, inv_majo, r, hb, vox, mat, fc);
                if (STATS) ++c_fly;
                ANM_TR("S2 h=%llu ph=%u blk=%u FLY code=%d t=%d+%.9g pos=%.9g %.9g %.9g vox=%u hb=%u\n", h, ph, meta >> 16, code, ie, fe, x, y, z, vox, hb);
                Bk[F_X * kSlots] = x; Bk[F_Y * kSlots] = y; Bk[F_Z * kSlots] = z;
                // next event and slot header, branch-free: GO -> FLY; COMPTON / RAYLEIGH -> their queues, the voxel in
                // place of the energy coordinate; PE / ESCAPED end the photon: start the partner (bank 1, written at
                // the decay) or free the slot
                const bool coll = code == FLY_COMPTON || code == FLY_RAYLEIGH;
                const bool ended = code == FLY_PE || code == FLY_ESCAPED;
                const bool partner = !ph && p.photons_per_decay == 2;
                const unsigned meta_go = (((meta & ~0x76u) | (hb << 1)) + kBlkInc) | (code == FLY_RAYLEIGH ? (unsigned)mat << 4 : 0u);
                const unsigned meta_end = 1u | (meta & 0xff08u) | ((meta & 8u) >> 2);   // photon B, block 0, IN = decay voxel's, same batch
                SU[F_META * kSlots] = ended ? meta_end : meta_go;
                if (coll) reinterpret_cast<unsigned*>(Bk)[F_TV * kSlots] = vox;
                next = code == FLY_COMPTON ? Q_C : (code == FLY_RAYLEIGH ? Q_R : ((ended && !partner) ? Q_S : Q_F));
                if (code == FLY_PE) {               // all energy to one electron: local, or transported along the photon's direction
                    if (STATS) ++c_pe;
                    const float Epe = Bk[F_E * kSlots];
                    if (ELEC && Epe > p.t_min) {          // rare (0.002 per decay): walked on the spot, not queued
                        const float out = HBH ? electron_walk_to(p, s_er, x, y, z, u, v, w, vox, Epe, [&](unsigned vv, float ee) {
                                                    hbh_push(p, tally_of(meta), gslot0 + slot, SU[F_HL * kSlots], vv, ee, c_ovf); })
                                              : electron_walk(p, tally_of(meta), s_er, x, y, z, u, v, w, vox, Epe);
                        if (STATS) { esc += out; ++c_el; }
                    } else if (HBH) hbh_push(p, tally_of(meta), gslot0 + slot, SU[F_HL * kSlots], vox, Epe, c_ovf);
                    else deposit<TALLY>(p, tally_of(meta), vox, Epe);
                }
                if (STATS && code == FLY_ESCAPED) { esc += Bk[F_E * kSlots]; ++c_esc; }
            }
            push_all(next, slot);
        } else if (X == Q_C) {
            if (active) {
                const unsigned meta = SU[F_META * kSlots];
                const unsigned ph = meta & 1u;
                const unsigned long long h = p.hist_base + (HBH ? SU[F_HL * kSlots] & kHbhHistMask : SU[F_HL * kSlots]);
                const uint4 r = philox4x32_10(make_uint4((unsigned)h, (unsigned)(h >> 32), meta >> 16, 1u + ph), p);
                float* Bk = S + ph * (kBankFields * kSlots);
                float E = Bk[F_E * kSlots];
                float eps, t;
                if (STATS) ++c_ctry;
                if (compton_try(E, r, eps, t)) {
                    if (STATS) ++c_co;
                    const unsigned vox = reinterpret_cast<unsigned*>(Bk)[F_TV * kSlots];
                    float dep = E * (1.0f - eps);     // recoil electron: deposited locally, or transported (ELEC)
                    const bool walk = ELEC && dep > p.t_min;
                    float u = 0.0f, v = 0.0f, w = 1.0f;
                    E *= eps;
                    const bool ends = E < p.cutoff;
                    if (!ends || walk) {
                        u = Bk[F_U * kSlots]; v = Bk[F_V * kSlots]; w = Bk[F_W * kSlots];
                        const float u0 = u, v0 = v, w0 = w;
                        rotate(u, v, w, 1.0f - t, kTwoPi * u01(r.w));
                        if (walk) {                   // along the electron's momentum d - eps d' (photon momentum = E / c)
                            float ex = fmaf(-eps, u, u0), ey = fmaf(-eps, v, v0), ez = fmaf(-eps, w, w0);
                            const float n2 = fmaf(ex, ex, fmaf(ey, ey, ez * ez));
                            if (n2 > 0.0f) { const float inv = rsqrtf(n2); ex *= inv; ey *= inv; ez *= inv; } else { ex = u0; ey = v0; ez = w0; }
                            if (HBH) {            // the deposits belong to this decay's list: walked on the spot
                                const float out = electron_walk_to(p, s_er, Bk[F_X * kSlots], Bk[F_Y * kSlots], Bk[F_Z * kSlots], ex, ey, ez,
                                                                   vox, dep, [&](unsigned vv, float ee) {
                                                                       hbh_push(p, tally_of(meta), gslot0 + slot, SU[F_HL * kSlots], vv, ee, c_ovf); });
                                if (STATS) { esc += out; ++c_el; }
                            } else {
                                e_want = true; e_x = Bk[F_X * kSlots]; e_y = Bk[F_Y * kSlots]; e_z = Bk[F_Z * kSlots];
                                e_ex = ex; e_ey = ey; e_ez = ez; e_T = dep; e_vox = vox; e_bl = (meta >> 8) & 0xffu;
                            }
                            dep = 0.0f;
                        }
                    }
                    if (ends) {                       // the rest is deposited locally
                        dep += E;
                        if (STATS) ++c_cut;
                        photon_ends(meta);
                    } else {
                        Bk[F_U * kSlots] = u; Bk[F_V * kSlots] = v; Bk[F_W * kSlots] = w;
                        Bk[F_E * kSlots] = E;
                        Bk[F_TV * kSlots] = fminf(fmaxf((__logf(E) - p.lnE_min) * p.inv_dlnE, 0.0f), t_max);
                        SU[F_META * kSlots] = (meta & ~0x74u) + kBlkInc;     // a scatter clears AWAY
                        next = Q_F;
                    }
                    if (dep > 0.0f) { if (HBH) hbh_push(p, tally_of(meta), gslot0 + slot, SU[F_HL * kSlots], vox, dep, c_ovf); else deposit<TALLY>(p, tally_of(meta), vox, dep); }
                } else {
                    SU[F_META * kSlots] = meta + kBlkInc;
                    next = Q_C;
                }
            }
            if (ELEC && !HBH) { e_append(); e_drain(32u); }
            push_all(next, slot);
        } else if (X == Q_S) {
            if (active) {
                // HBH: the slot's previous decay is complete; its deposits are merged per voxel HERE, where up to 32 freed
                // slots are handled by 32 lanes at once, not at the photon's end, where one or two lanes of a trip would do it
                if (HBH) hbh_flush(p, tally_of(SU[F_META * kSlots]), gslot0 + slot, SU[F_HL * kSlots]);
                const unsigned long long h = p.hist_base + hl_new;
                const unsigned bl = p.n_group > 1u ? hl_new / p.n_per_batch : 0u;      // the decay's batch within the group
                ANM_CHK(p, 9, bl < p.n_group);
                float x, y, z, u, v, w;
                bool in_box;
                const unsigned voxel = sample_source(p, h, x, y, z, u, v, w, in_box);
                S[F_X * kSlots] = x; S[F_Y * kSlots] = y; S[F_Z * kSlots] = z;
                S[F_U * kSlots] = u; S[F_V * kSlots] = v; S[F_W * kSlots] = w;
                S[F_E * kSlots] = kE0; S[F_TV * kSlots] = t0;
                float* B1 = S + kBankFields * kSlots;
                B1[F_X * kSlots] = x; B1[F_Y * kSlots] = y; B1[F_Z * kSlots] = z;
                B1[F_U * kSlots] = -u; B1[F_V * kSlots] = -v; B1[F_W * kSlots] = -w;
                B1[F_E * kSlots] = kE0; B1[F_TV * kSlots] = t0;
                SU[F_HL * kSlots] = hl_new;
                SU[F_META * kSlots] = (in_box ? (2u | 8u) : 0u) | (bl << 8);
                if (p.positron_ke > 0.0f) { if (HBH) hbh_push(p, p.batch + (size_t)bl * p.batch_stride, gslot0 + slot, SU[F_HL * kSlots], voxel, p.positron_ke, c_ovf); else deposit<TALLY>(p, p.batch + (size_t)bl * p.batch_stride, voxel, p.positron_ke); }
                q[Q_F * kSlots + ((heads + cnts + lane) & (kSlots - 1))] = (unsigned char)slot;
            }
            cnts += n;
        } else {   // Q_R
            if (active) {
                const unsigned meta = SU[F_META * kSlots];
                const unsigned ph = meta & 1u;
                const unsigned long long h = p.hist_base + (HBH ? SU[F_HL * kSlots] & kHbhHistMask : SU[F_HL * kSlots]);
                const uint4 r = philox4x32_10(make_uint4((unsigned)h, (unsigned)(h >> 32), meta >> 16, 1u + ph), p);
                float* Bk = S + ph * (kBankFields * kSlots);
                const float E = Bk[F_E * kSlots];
                float c;
                if (STATS) ++c_rtry;
                if (rayleigh_try(E, r, s_x2, s_cum + ((meta >> 4) & 7u) * p.n_x2, p.n_x2, c)) {
                    if (STATS) ++c_ra;
                    float u = Bk[F_U * kSlots], v = Bk[F_V * kSlots], w = Bk[F_W * kSlots];
                    rotate(u, v, w, c, kTwoPi * u01(r.z));
                    Bk[F_U * kSlots] = u; Bk[F_V * kSlots] = v; Bk[F_W * kSlots] = w;
                    Bk[F_TV * kSlots] = fminf(fmaxf((__logf(E) - p.lnE_min) * p.inv_dlnE, 0.0f), t_max);
                    SU[F_META * kSlots] = (meta & ~0x74u) + kBlkInc;         // a scatter clears AWAY
                    next = Q_F;
                } else {
                    SU[F_META * kSlots] = meta + kBlkInc;
                    next = Q_R;
                }
            }
            push_all(next, slot);
        }
    }

    if (ELEC && !HBH) e_drain(1u);          // the electrons still waiting
    if (HBH) {      // the decays that completed after the last SOURCE trip
        __syncwarp();
#pragma unroll 1
        for (int k = 0; k < kSlots / 32; ++k)
            hbh_flush(p, tally_of(slots_u[F_META * kSlots + lane + 32 * k]), gslot0 + lane + 32u * (unsigned)k, slots_u[F_HL * kSlots + lane + 32 * k]);
    }
    if (STATS) {
        unsigned c_steps = fc.steps, c_real = fc.real;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            esc += __shfl_xor_sync(0xffffffffu, esc, o);
            c_steps += __shfl_xor_sync(0xffffffffu, c_steps, o);
            c_real += __shfl_xor_sync(0xffffffffu, c_real, o);
            c_pe += __shfl_xor_sync(0xffffffffu, c_pe, o);
            c_co += __shfl_xor_sync(0xffffffffu, c_co, o);
            c_ra += __shfl_xor_sync(0xffffffffu, c_ra, o);
            c_esc += __shfl_xor_sync(0xffffffffu, c_esc, o);
            c_cut += __shfl_xor_sync(0xffffffffu, c_cut, o);
            c_el += __shfl_xor_sync(0xffffffffu, c_el, o);
            c_ovf += __shfl_xor_sync(0xffffffffu, c_ovf, o);
            c_fly += __shfl_xor_sync(0xffffffffu, c_fly, o);
            c_ctry += __shfl_xor_sync(0xffffffffu, c_ctry, o);
            c_rtry += __shfl_xor_sync(0xffffffffu, c_rtry, o);
        }
        if (lane == 0) {
            atomicAdd(&p.stats->escaped_MeV, (double)esc);
            atomicAdd(&p.stats->n_steps, (unsigned long long)c_steps);
            atomicAdd(&p.stats->n_real, (unsigned long long)c_real);
            atomicAdd(&p.stats->n_pe, (unsigned long long)c_pe);
            atomicAdd(&p.stats->n_compton, (unsigned long long)c_co);
            atomicAdd(&p.stats->n_rayleigh, (unsigned long long)c_ra);
            atomicAdd(&p.stats->n_escaped, (unsigned long long)c_esc);
            atomicAdd(&p.stats->n_cutoff, (unsigned long long)c_cut);
            atomicAdd(&p.stats->n_electrons, (unsigned long long)c_el);
            atomicAdd(&p.stats->n_hbh_overflow, (unsigned long long)c_ovf);
            atomicAdd(&p.stats->n_fly_trips, (unsigned long long)c_fly);
            atomicAdd(&p.stats->n_compton_tries, (unsigned long long)c_ctry);
            atomicAdd(&p.stats->n_rayleigh_tries, (unsigned long long)c_rtry);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// A10: fold one batch.  x = batch[i]; sum += x; sumsq += x*x; batch = 0; organ_row[label] += x / (rho V).
// Streaming; most voxels of a patient volume are untouched air (x == 0) and cost one 16-byte read per 4.
constexpr int kFoldThreads = 256;

// one group of four voxels: sum += x, sumsq += x^2, organ bins += x / (rho V)
__device__ __forceinline__ void fold_group(const float4 xv, const size_t i, float4* __restrict__ sum, float4* __restrict__ sumsq,
                                           const uint32_t* __restrict__ labels4, const uint4* __restrict__ texels4,
                                           double* s_org, const float inv_vox_cm3) {
    float4 s = sum[i], q = sumsq[i];
    s.x += xv.x; s.y += xv.y; s.z += xv.z; s.w += xv.w;
    q.x = fmaf(xv.x, xv.x, q.x); q.y = fmaf(xv.y, xv.y, q.y); q.z = fmaf(xv.z, xv.z, q.z); q.w = fmaf(xv.w, xv.w, q.w);
    sum[i] = s; sumsq[i] = q;
    if (labels4 != nullptr) {
        const uint32_t l4 = labels4[i];
        if (l4) {
            const uint4 t = texels4[i];
            const float xs[4] = {xv.x, xv.y, xv.z, xv.w};
            const unsigned ts[4] = {t.x, t.y, t.z, t.w};
            // x / (rho V) in fp32 (1e-7 relative), accumulated in fp64.  The four voxels of a thread usually carry one
            // label: one shared-memory atomic per thread instead of four (neighbouring lanes hit the same organ bin).
            const unsigned l0 = l4 & 0xffu;
            if (l4 == l0 * 0x01010101u) {
                double acc = 0.0;
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    if (xs[k] != 0.0f) acc += (double)__fdividef(xs[k] * inv_vox_cm3, (float)(ts[k] & 0xffffffu) * kDensityStep);
                if (acc != 0.0) atomicAdd(&s_org[l0], acc);
            } else {
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const unsigned l = (l4 >> (8 * k)) & 0xffu;
                    if (l && xs[k] != 0.0f)
                        atomicAdd(&s_org[l], (double)__fdividef(xs[k] * inv_vox_cm3, (float)(ts[k] & 0xffffffu) * kDensityStep));
                }
            }
        }
    }
}

__global__ void __launch_bounds__(kFoldThreads)
fold_kernel(float4* __restrict__ batch, float4* __restrict__ sum, float4* __restrict__ sumsq,
            const uint32_t* __restrict__ labels4, const uint4* __restrict__ texels4, double* __restrict__ organ_row,
            int n_organs, size_t n4, float inv_vox_cm3) {
    __shared__ double s_org[256];
    const bool organs = (labels4 != nullptr);
    if (organs) { s_org[threadIdx.x] = 0.0; __syncthreads(); }
    for (size_t i = (size_t)blockIdx.x * kFoldThreads + threadIdx.x; i < n4; i += (size_t)gridDim.x * kFoldThreads) {
        const float4 xv = batch[i];
        if (xv.x == 0.0f && xv.y == 0.0f && xv.z == 0.0f && xv.w == 0.0f) continue;
        batch[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        fold_group(xv, i, sum, sumsq, labels4, texels4, s_org, inv_vox_cm3);
    }
    if (organs) {
        __syncthreads();
        if ((int)threadIdx.x <= n_organs && threadIdx.x > 0 && s_org[threadIdx.x] != 0.0)
            atomicAdd(organ_row + threadIdx.x, s_org[threadIdx.x]);
    }
}

// A10 for a batch group (anm_options.batches_per_launch): the G per-batch tallies of one launch folded in ONE pass.
// A thread takes a group of four voxels and reads it from all G tallies (independent loads, kFoldMlp at a time), adds
// what it finds to register accumulators, zeroes the touched words, and updates sum / sumsq once -- per touched voxel the
// run sums are read and written once per GROUP instead of once per batch, and the untouched (air) part of the volume is
// streamed with G loads in flight per thread.  Organ partials stay per batch: s_org[j][label], rows row0 + j.
// The same arithmetic per batch as fold_kernel (x, x^2 in fp32; x / (rho V) in fp32, summed in fp64); the G values of a
// voxel are summed before they are added to the run sum (fp32, <= 256 terms of the same sign).
constexpr int kFoldMlp = 4;                 // measured: 4 loads in flight at 4 CTAs per SM (64 registers) beat 8 at 3 CTAs (79 registers) by 24 %
__global__ void __launch_bounds__(kFoldThreads, 4)
fold_group_kernel(float4* __restrict__ batch, size_t stride4, int G, float4* __restrict__ sum, float4* __restrict__ sumsq,
                  const uint32_t* __restrict__ labels4, const uint4* __restrict__ texels4, double* __restrict__ organ_rows,
                  int n_organs, size_t n4, float inv_vox_cm3) {
    extern __shared__ double s_orgs[];                 // [G][n_organs + 1]
    const bool organs = (labels4 != nullptr);
    const int n1 = n_organs + 1;
    if (organs) { for (int k = threadIdx.x; k < G * n1; k += kFoldThreads) s_orgs[k] = 0.0; __syncthreads(); }
    for (size_t i = (size_t)blockIdx.x * kFoldThreads + threadIdx.x; i < n4; i += (size_t)gridDim.x * kFoldThreads) {
        float4 s = make_float4(0.f, 0.f, 0.f, 0.f), q = s;
        bool any = false;
        uint32_t l4 = 0;
        float w[4] = {1.f, 1.f, 1.f, 1.f};             // densities of the four voxels, loaded when first needed
        for (int j0 = 0; j0 < G; j0 += kFoldMlp) {
            float4 xv[kFoldMlp];
#pragma unroll
            for (int k = 0; k < kFoldMlp; ++k) xv[k] = j0 + k < G ? batch[(size_t)(j0 + k) * stride4 + i] : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
            for (int k = 0; k < kFoldMlp; ++k) {
                const float4 x = xv[k];
                if (x.x == 0.0f && x.y == 0.0f && x.z == 0.0f && x.w == 0.0f) continue;
                batch[(size_t)(j0 + k) * stride4 + i] = make_float4(0.f, 0.f, 0.f, 0.f);
                s.x += x.x; s.y += x.y; s.z += x.z; s.w += x.w;
                q.x = fmaf(x.x, x.x, q.x); q.y = fmaf(x.y, x.y, q.y); q.z = fmaf(x.z, x.z, q.z); q.w = fmaf(x.w, x.w, q.w);
                if (organs) {
                    if (!any) {
                        l4 = labels4[i];
                        if (l4) {
                            const uint4 t = texels4[i];
                            const unsigned ts[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
                            for (int v = 0; v < 4; ++v) w[v] = (float)(ts[v] & 0xffffffu) * kDensityStep;
                        }
                    }
                    if (l4) {
                        double* so = s_orgs + (size_t)(j0 + k) * n1;
                        const float xs[4] = {x.x, x.y, x.z, x.w};
                        const unsigned l0 = l4 & 0xffu;
                        if (l4 == l0 * 0x01010101u) {
                            double acc = 0.0;
#pragma unroll
                            for (int v = 0; v < 4; ++v) if (xs[v] != 0.0f) acc += (double)__fdividef(xs[v] * inv_vox_cm3, w[v]);
                            if (acc != 0.0) atomicAdd(&so[l0], acc);
                        } else {
#pragma unroll
                            for (int v = 0; v < 4; ++v) {
                                const unsigned l = (l4 >> (8 * v)) & 0xffu;
                                if (l && xs[v] != 0.0f) atomicAdd(&so[l], (double)__fdividef(xs[v] * inv_vox_cm3, w[v]));
                            }
                        }
                    }
                }
                any = true;
            }
        }
        if (any) {
            float4 S = sum[i], Q = sumsq[i];
            S.x += s.x; S.y += s.y; S.z += s.z; S.w += s.w;
            Q.x += q.x; Q.y += q.y; Q.z += q.z; Q.w += q.w;
            sum[i] = S; sumsq[i] = Q;
        }
    }
    if (organs) {
        __syncthreads();
        for (int k = threadIdx.x; k < G * n1; k += kFoldThreads) {
            const int j = k / n1, l = k - j * n1;
            if (l > 0 && s_orgs[k] != 0.0) atomicAdd(organ_rows + (size_t)j * 256 + l, s_orgs[k]);
        }
    }
}

// A10 for the tile-binned tally: a CTA takes one tile at a time, sums the tile's deposit list into a
// 64 KB shared-memory image of the tile (fp32 shared-memory atomics), adds what overflowed into the batch volume (only
// if the tile's counter exceeded its capacity), folds the image like fold_kernel and resets the counter.  Tiles that
// received nothing cost one 4-byte read.  overflow[0] += deposits that did not fit their segment (diagnostic).
constexpr int kBinFoldThreads = 512;
__global__ void __launch_bounds__(kBinFoldThreads)
bin_fold_kernel(unsigned* __restrict__ bin_cnt, const uint2* __restrict__ bin_seg, const uint2* __restrict__ bin_rec,
                float4* __restrict__ batch, float4* __restrict__ sum, float4* __restrict__ sumsq,
                const uint32_t* __restrict__ labels4, const uint4* __restrict__ texels4, double* __restrict__ organ_row,
                int n_organs, size_t n4, unsigned n_tiles, float inv_vox_cm3, unsigned long long* __restrict__ overflow) {
    extern __shared__ __align__(16) float s_tile[];        // [kTileVoxels]
    __shared__ double s_org[256];
    const bool organs = (labels4 != nullptr);
    if (threadIdx.x < 256) s_org[threadIdx.x] = 0.0;
    for (unsigned tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        unsigned cnt[kTileSub], any = 0u;
#pragma unroll
        for (unsigned k = 0; k < kTileSub; ++k) { cnt[k] = bin_cnt[tile * kTileSub + k]; any |= cnt[k]; }
        if (any == 0u) continue;                           // block-uniform
        bool ovf = false;
        __syncthreads();                                   // everyone has read the counters; the previous tile's image is done with
        for (unsigned j = threadIdx.x; j < kTileVoxels / 4; j += kBinFoldThreads) reinterpret_cast<float4*>(s_tile)[j] = make_float4(0.f, 0.f, 0.f, 0.f);
        __syncthreads();
#pragma unroll 1
        for (unsigned k = 0; k < kTileSub; ++k) {
            if (cnt[k] == 0u) continue;
            const uint2 seg = bin_seg[tile * kTileSub + k];
            const unsigned n = min(cnt[k], seg.y);
            if (cnt[k] > seg.y) { ovf = true; if (threadIdx.x == 0) atomicAdd(overflow, (unsigned long long)(cnt[k] - seg.y)); }
            if (threadIdx.x == 0) bin_cnt[tile * kTileSub + k] = 0u;
            const uint2* rec = bin_rec + (size_t)seg.x;
            for (unsigned i = threadIdx.x; i < n; i += kBinFoldThreads) {
                const uint2 r = __ldcs(rec + i);
                atomicAdd(&s_tile[r.x & (kTileVoxels - 1u)], __uint_as_float(r.y));
            }
        }
        __syncthreads();
        const size_t g0 = (size_t)tile * (kTileVoxels / 4);
        for (unsigned j = threadIdx.x; j < kTileVoxels / 4 && g0 + j < n4; j += kBinFoldThreads) {
            float4 xv = reinterpret_cast<const float4*>(s_tile)[j];
            if (ovf) {
                const float4 o = batch[g0 + j];
                if (o.x != 0.0f || o.y != 0.0f || o.z != 0.0f || o.w != 0.0f) {
                    xv.x += o.x; xv.y += o.y; xv.z += o.z; xv.w += o.w;
                    batch[g0 + j] = make_float4(0.f, 0.f, 0.f, 0.f);
                }
            }
            if (xv.x == 0.0f && xv.y == 0.0f && xv.z == 0.0f && xv.w == 0.0f) continue;
            fold_group(xv, g0 + j, sum, sumsq, labels4, texels4, s_org, inv_vox_cm3);
        }
    }
    if (organs) {
        __syncthreads();
        if ((int)threadIdx.x <= n_organs && threadIdx.x > 0 && threadIdx.x < 256 && s_org[threadIdx.x] != 0.0)
            atomicAdd(organ_row + threadIdx.x, s_org[threadIdx.x]);
    }
}

// ------------------------------------------------------------------------------------------------
// A11: one pass over the run's sums: per organ  sum of rel^2 over voxels with dose > 0, their count, organ
// energy;  total deposited energy.  rel^2 = (B Q / S^2 - 1) / (B - 1)  (batch standard error of the mean / mean).
struct OrganAccum { double rel2, n_nonzero, energy; };

// (B, Q) = (batches, sum of squared batch sums), or for history-by-history scoring (histories, sum of X_h^2): the same
// formula, PAPER.md:L67 / Walters et al. 2002.
__device__ __forceinline__ float rel_sigma(float S, float Q, double B) {
    if (!(S > 0.0f)) return 0.0f;
    const double r2 = (B * (double)Q / ((double)S * (double)S) - 1.0) / (B - 1.0);
    return r2 > 0.0 ? (float)sqrt(r2) : 0.0f;
}

__global__ void __launch_bounds__(kFoldThreads)
finalize_kernel(const float* __restrict__ sum, const float* __restrict__ sumsq, const uint8_t* __restrict__ labels,
                OrganAccum* __restrict__ organ, double* __restrict__ total_energy, int n_organs, size_t V, double B) {
    __shared__ double s_rel2[256], s_nz[256], s_en[256];
    __shared__ double s_tot;
    s_rel2[threadIdx.x] = 0.0; s_nz[threadIdx.x] = 0.0; s_en[threadIdx.x] = 0.0;
    if (threadIdx.x == 0) s_tot = 0.0;
    __syncthreads();
    double tot = 0.0;
    for (size_t i = (size_t)blockIdx.x * kFoldThreads + threadIdx.x; i < V; i += (size_t)gridDim.x * kFoldThreads) {
        const float S = sum[i];
        if (S == 0.0f) continue;
        tot += (double)S;
        if (labels) {
            const unsigned l = labels[i];
            if (l) {
                const float r = rel_sigma(S, sumsq[i], B);
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
    if (threadIdx.x == 0 && s_tot != 0.0) atomicAdd(total_energy, s_tot);
    if (labels && threadIdx.x > 0 && (int)threadIdx.x <= n_organs && s_nz[threadIdx.x] != 0.0) {
        atomicAdd(&organ[threadIdx.x].rel2, s_rel2[threadIdx.x]);
        atomicAdd(&organ[threadIdx.x].n_nonzero, s_nz[threadIdx.x]);
        atomicAdd(&organ[threadIdx.x].energy, s_en[threadIdx.x]);
    }
}

// A11, the run-level "statistical uncertainty" figure ("0.47 %", L117 "1.19 %"; reading C17): the
// RMS of the voxels' relative sigma over the non-air voxels whose dose exceeds 10 % / 50 % of the maximum dose.  Dose is
// proportional to S / rho (voxel volume and decay count are constants), so both passes work on that ratio.
// Pass 1: maximum of S / rho over the non-air voxels (material id != 0), as the bits of a positive float.
__global__ void __launch_bounds__(kFoldThreads)
dose_max_kernel(const float* __restrict__ sum, const uint32_t* __restrict__ texels, size_t V, unsigned* __restrict__ max_bits) {
    float m = 0.0f;
    for (size_t i = (size_t)blockIdx.x * kFoldThreads + threadIdx.x; i < V; i += (size_t)gridDim.x * kFoldThreads) {
        const float S = sum[i];
        if (!(S > 0.0f)) continue;
        const unsigned t = texels[i];
        const float rho = (float)(t & 0xffffffu) * kDensityStep;
        if ((t >> 24) != 0u && rho > 0.0f) m = fmaxf(m, S / rho);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0 && m > 0.0f) atomicMax(max_bits, __float_as_uint(m));
}

// Pass 2: acc[0] += rel^2, acc[1] += 1 over the voxels above 10 % of the maximum; acc[2], acc[3] the same above 50 %.
__global__ void __launch_bounds__(kFoldThreads)
run_sigma_kernel(const float* __restrict__ sum, const float* __restrict__ sumsq, const uint32_t* __restrict__ texels, size_t V,
                 double B, const unsigned* __restrict__ max_bits, double* __restrict__ acc) {
    const float dmax = __uint_as_float(*max_bits);
    double a[4] = {0.0, 0.0, 0.0, 0.0};
    for (size_t i = (size_t)blockIdx.x * kFoldThreads + threadIdx.x; i < V; i += (size_t)gridDim.x * kFoldThreads) {
        const float S = sum[i];
        if (!(S > 0.0f)) continue;
        const unsigned t = texels[i];
        const float rho = (float)(t & 0xffffffu) * kDensityStep;
        if ((t >> 24) == 0u || !(rho > 0.0f)) continue;
        const float d = S / rho;
        if (d > 0.1f * dmax) {
            const double r = (double)rel_sigma(S, sumsq[i], B);
            a[0] += r * r; a[1] += 1.0;
            if (d > 0.5f * dmax) { a[2] += r * r; a[3] += 1.0; }
        }
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) a[k] += __shfl_xor_sync(0xffffffffu, a[k], o);
    }
    if ((threadIdx.x & 31) == 0 && a[1] != 0.0) {
#pragma unroll
        for (int k = 0; k < 4; ++k) atomicAdd(acc + k, a[k]);
    }
}

// organ mass and voxel counts (once per load of labels / phantom)
__global__ void __launch_bounds__(kFoldThreads)
organ_mass_kernel(const uint8_t* __restrict__ labels, const uint32_t* __restrict__ texels, double* __restrict__ mass,
                  unsigned long long* __restrict__ count, size_t V, float vox_cm3) {
    __shared__ double s_m[256];
    __shared__ unsigned long long s_c[256];
    s_m[threadIdx.x] = 0.0; s_c[threadIdx.x] = 0ull;
    __syncthreads();
    for (size_t i = (size_t)blockIdx.x * kFoldThreads + threadIdx.x; i < V; i += (size_t)gridDim.x * kFoldThreads) {
        const unsigned l = labels[i];
        if (l) {
            atomicAdd(&s_m[l], (double)(texels[i] & 0xffffffu) * (double)kDensityStep * (double)vox_cm3);
            atomicAdd(&s_c[l], 1ull);
        }
    }
    __syncthreads();
    if (s_c[threadIdx.x]) { atomicAdd(mass + threadIdx.x, s_m[threadIdx.x]); atomicAdd(count + threadIdx.x, s_c[threadIdx.x]); }
}

// read-out: mode 0 energy (MeV), 1 dose = S k / (N rho V) * scale (scale = 1 or A(t_s), Eq. 1), 2 relative sigma
__global__ void __launch_bounds__(kFoldThreads)
readout_kernel(const float* __restrict__ sum, const float* __restrict__ sumsq, const uint32_t* __restrict__ texels,
               float* __restrict__ out, size_t V, int mode, double dose_factor /* k*scale/(N V_vox) */, double B, int zero_air) {
    for (size_t i = (size_t)blockIdx.x * kFoldThreads + threadIdx.x; i < V; i += (size_t)gridDim.x * kFoldThreads) {
        const float S = sum[i];
        float o;
        if (mode == 0) o = S;
        else if (mode == 1) {
            const unsigned t = texels[i];
            const double rho = (double)(t & 0xffffffu) * (double)kDensityStep;
            o = (S > 0.0f && rho > 0.0 && !(zero_air && (t >> 24) == 0u)) ? (float)((double)S * dose_factor / rho) : 0.0f;
        } else o = rel_sigma(S, sumsq[i], B);
        out[i] = o;
    }
}

// phantom packing + validation on the device: texel = material<<24 | round(rho * 2^20); flags bit0 = bad density,
// max_mat = largest material id seen
__global__ void __launch_bounds__(kFoldThreads)
pack_texels_kernel(const uint8_t* __restrict__ material, const float* __restrict__ density, uint32_t* __restrict__ texels,
                   size_t V, unsigned* __restrict__ flags, unsigned* __restrict__ max_mat) {
    unsigned bad = 0, mm = 0;
    for (size_t i = (size_t)blockIdx.x * kFoldThreads + threadIdx.x; i < V; i += (size_t)gridDim.x * kFoldThreads) {
        const float r = density[i];
        const unsigned m = material[i];
        if (!(r >= 0.0f) || !(r < 16.0f)) { bad = 1; texels[i] = m << 24; }
        else texels[i] = (m << 24) | min(0xffffffu, (unsigned)__float2uint_rn(r * 1048576.0f));
        mm = max(mm, m);
    }
    if (bad) atomicOr(flags, 1u);
    atomicMax(max_mat, mm);
}

// 16-bit copy of the texels (anm_options.texel_bits): material<<13 | density / 2^-12.  not_exact is set when a voxel is
// not exactly representable (density off the 2^-12 grid or >= 2 g/cm^3; material ids always fit, < 8): the copy is then
// not used.
__global__ void __launch_bounds__(kFoldThreads)
pack_texels16_kernel(const uint32_t* __restrict__ texels, uint16_t* __restrict__ texels16, size_t V, unsigned* __restrict__ not_exact) {
    unsigned bad = 0;
    for (size_t i = (size_t)blockIdx.x * kFoldThreads + threadIdx.x; i < V; i += (size_t)gridDim.x * kFoldThreads) {
        const unsigned t = texels[i], m = t >> 24, r = t & 0xffffffu;
        if ((r & ((1u << kT16Shift) - 1u)) != 0u || (r >> kT16Shift) >= (1u << kT16DensityBits) || m >= 8u) bad = 1;
        texels16[i] = (uint16_t)((m << kT16DensityBits) | ((r >> kT16Shift) & ((1u << kT16DensityBits) - 1u)));
    }
    if (bad) atomicOr(not_exact, 1u);
}

// per-material maximum density (texel counts) -> majorant
constexpr int kMaxMaterials = 8;
__global__ void __launch_bounds__(kFoldThreads)
rho_max_kernel(const uint32_t* __restrict__ t, size_t V, unsigned* __restrict__ out) {
    __shared__ unsigned s[kMaxMaterials];
    if (threadIdx.x < kMaxMaterials) s[threadIdx.x] = 0;
    __syncthreads();
    unsigned loc[kMaxMaterials];
#pragma unroll
    for (int m = 0; m < kMaxMaterials; ++m) loc[m] = 0;
    for (size_t i = (size_t)blockIdx.x * kFoldThreads + threadIdx.x; i < V; i += (size_t)gridDim.x * kFoldThreads) {
        const unsigned v = t[i], m = v >> 24, r = v & 0xffffffu;
#pragma unroll
        for (int k = 0; k < kMaxMaterials; ++k) if (m == (unsigned)k) loc[k] = max(loc[k], r);
    }
#pragma unroll
    for (int m = 0; m < kMaxMaterials; ++m) if (loc[m]) atomicMax(&s[m], loc[m]);
    __syncthreads();
    if (threadIdx.x < kMaxMaterials && s[threadIdx.x]) atomicMax(out + threadIdx.x, s[threadIdx.x]);
}

// hull box (anm_options.hull_majorant): bounding box of the voxels denser than `thr` texel counts.
// box = {x0, y0, z0 (atomicMin, start at 0xffffffff), x1, y1, z1 (atomicMax of index + 1, start at 0)}
__global__ void __launch_bounds__(kFoldThreads)
hull_box_kernel(const uint32_t* __restrict__ t, int nx, int ny, int nz, unsigned thr, unsigned* __restrict__ box) {
    __shared__ unsigned s[6];
    if (threadIdx.x < 6) s[threadIdx.x] = threadIdx.x < 3 ? 0xffffffffu : 0u;
    __syncthreads();
    unsigned lo[3] = {0xffffffffu, 0xffffffffu, 0xffffffffu}, hi[3] = {0u, 0u, 0u};
    const size_t rows = (size_t)ny * nz;
    for (size_t row = (size_t)blockIdx.x * (kFoldThreads / 32) + (threadIdx.x >> 5); row < rows;
         row += (size_t)gridDim.x * (kFoldThreads / 32)) {
        const unsigned iy = (unsigned)(row % (size_t)ny), iz = (unsigned)(row / (size_t)ny);
        const uint32_t* r = t + row * (size_t)nx;
        for (unsigned ix = threadIdx.x & 31u; ix < (unsigned)nx; ix += 32u) {
            if ((r[ix] & 0xffffffu) > thr) {
                lo[0] = min(lo[0], ix); hi[0] = max(hi[0], ix + 1u);
                lo[1] = min(lo[1], iy); hi[1] = max(hi[1], iy + 1u);
                lo[2] = min(lo[2], iz); hi[2] = max(hi[2], iz + 1u);
            }
        }
    }
    if (hi[0]) {
#pragma unroll
        for (int k = 0; k < 3; ++k) { atomicMin(&s[k], lo[k]); atomicMax(&s[3 + k], hi[k]); }
    }
    __syncthreads();
    if (threadIdx.x < 3 && s[3] != 0u) atomicMin(box + threadIdx.x, s[threadIdx.x]);
    else if (threadIdx.x >= 3 && threadIdx.x < 6 && s[3] != 0u) atomicMax(box + threadIdx.x, s[threadIdx.x]);
}

// per-material maximum density (texel counts) over the voxels OUTSIDE the box [x0,x1) x [y0,y1) x [z0,z1)
__global__ void __launch_bounds__(kFoldThreads)
rho_max_outside_kernel(const uint32_t* __restrict__ t, int nx, int ny, int nz, unsigned x0, unsigned y0, unsigned z0,
                       unsigned x1, unsigned y1, unsigned z1, unsigned* __restrict__ out) {
    __shared__ unsigned s[kMaxMaterials];
    if (threadIdx.x < kMaxMaterials) s[threadIdx.x] = 0;
    __syncthreads();
    unsigned loc[kMaxMaterials];
#pragma unroll
    for (int m = 0; m < kMaxMaterials; ++m) loc[m] = 0;
    const size_t V = (size_t)nx * ny * nz;
    for (size_t i = (size_t)blockIdx.x * kFoldThreads + threadIdx.x; i < V; i += (size_t)gridDim.x * kFoldThreads) {
        const unsigned ix = (unsigned)(i % (size_t)nx), iy = (unsigned)((i / (size_t)nx) % (size_t)ny),
                       iz = (unsigned)(i / ((size_t)nx * ny));
        if (ix >= x0 && ix < x1 && iy >= y0 && iy < y1 && iz >= z0 && iz < z1) continue;
        const unsigned v = t[i], m = v >> 24, r = v & 0xffffffu;
#pragma unroll
        for (int k = 0; k < kMaxMaterials; ++k) if (m == (unsigned)k) loc[k] = max(loc[k], r);
    }
#pragma unroll
    for (int m = 0; m < kMaxMaterials; ++m) if (loc[m]) atomicMax(&s[m], loc[m]);
    __syncthreads();
    if (threadIdx.x < kMaxMaterials && s[threadIdx.x]) atomicMax(out + threadIdx.x, s[threadIdx.x]);
}

}  // namespace anm
