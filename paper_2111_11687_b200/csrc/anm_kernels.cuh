// anm_kernels.cuh -- device code of libanm.so (sm_100a).  Hand-written CUDA; no oracle code is shared.
//
// Kernels
//   transport_kernel : source sampling + Woodcock photon transport + fp32 RED tally
//   fold_kernel      : per-batch fold  sum += x, sumsq += x^2, x = 0, organ partial sums   (A10)
//   finalize_kernel  : organ Eq. 3 accumulators, organ energy / mass / counts, total energy (A11)
//   get_*_kernel     : dose / dose rate / relative sigma read-out                           (A11)
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
#include <cuda_runtime.h>

namespace anm {

constexpr int kThreads = 256;
constexpr int kMinBlocksPerSM = 4;
constexpr unsigned kChunk = 128;            // histories a warp takes per atomic
constexpr float kE0 = 0.51099895f;          // MeV, "0.511 MeV"
constexpr float kInvE0 = 1.0f / 0.51099895f;
constexpr float kTwoPi = 6.283185307179586f;
constexpr float kKeVAngstromInv = 1000.0f / 12.398419843f;   // x_max (1/Angstrom) = E[MeV] * this
constexpr float kDensityStep = 1.0f / 1048576.0f;            // 2^-20 g/cm^3 per texel count

enum : int { ST_NEED = 0, ST_SOURCE = 1, ST_FLY = 2, ST_COMPTON = 3, ST_RAYLEIGH = 4, ST_DONE = 5 };

struct DeviceStats {   // accumulated with atomics at kernel exit (collect_stats only)
    double escaped_MeV;
    unsigned long long n_steps, n_real, n_pe, n_compton, n_rayleigh, n_escaped, n_cutoff;
};

struct TransportParams {
    const uint32_t* texels;      // [V] material<<24 | density/2^-20
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
    unsigned int key0, key1;     // Philox key = seed
    int nx, ny, nz;
    int nm, ne, n_x2;
    float dx, dy, dz;            // cm
    float inv_dx, inv_dy, inv_dz;
    float lnE_min, inv_dlnE;
    float cutoff, positron_ke;
    float px, py, pz;            // point source (cm)
    int point_source, photons_per_decay, rayleigh_on;
    // energy-dependent quantities at E0 (every photon starts there)
    int ie0; float fe0, maj0, inv_maj0;
    // hull majorant (anm_options.hull_majorant): the axis-aligned box (b?0, b?1) cm encloses every voxel denser than
    // the hull threshold (faces pushed outwards by a rounding margin).  A photon beyond a face and moving away from
    // it flies against tab_maj_out (the bound of the voxels outside the box); every other photon against tab_maj.
    int hull;
    float bx0, bx1, by0, by1, bz0, bz1;      // faces (cm)
    float majo0, inv_majo0;                   // tab_maj_out at E0
    const float* tab_maj_out;    // [ne]
};

// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, unsigned k0, unsigned k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        const unsigned hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
        c = make_uint4(hi1 ^ c.y ^ k0, lo1, hi0 ^ c.w ^ k1, lo0);
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return c;
}

// uniform on (0,1): ((r >> 8) + 0.5) 2^-24
__device__ __forceinline__ float u01(unsigned r) {
    return fmaf(__uint2float_rn(r >> 8), 5.9604644775390625e-08f, 2.98023223876953125e-08f);
}

__device__ __forceinline__ void rotate(float& u, float& v, float& w, float cos_t, float phi) {
    const float sin_t = sqrtf(fmaxf(0.0f, 1.0f - cos_t * cos_t));
    float sp, cp;
    __sincosf(phi, &sp, &cp);
    float a, b, c;
    if (fabsf(w) < 0.99999f) {
        const float s = sqrtf(1.0f - w * w);
        const float k = __fdividef(sin_t, s);
        a = u * cos_t + k * (u * w * cp - v * sp);
        b = v * cos_t + k * (v * w * cp + u * sp);
        c = w * cos_t - sin_t * s * cp;
    } else {
        a = sin_t * cp; b = sin_t * sp; c = copysignf(cos_t, w);
    }
    const float n = rsqrtf(a * a + b * b + c * c);
    u = a * n; v = b * n; w = c * n;
}

template <bool WAGG>
__device__ __forceinline__ void deposit(float* __restrict__ batch, unsigned vox, float e) {
    if (WAGG) {
        // merge the deposits of lanes that hit the same voxel in this trip: one RED per distinct voxel
        const unsigned act = __activemask();
        const unsigned peers = __match_any_sync(act, vox);
        float total = 0.0f;
        for (unsigned rem = peers; rem; rem &= rem - 1) total += __shfl_sync(peers, e, __ffs(rem) - 1);
        if ((threadIdx.x & 31) == (unsigned)(__ffs(peers) - 1)) atomicAdd(batch + vox, total);
    } else {
        atomicAdd(batch + vox, e);
    }
}

// One Woodcock sub-step: exponential flight against the majorant of the region the photon
// is in, then the real / virtual decision and the channel choice from one more uniform.
enum : int { FLY_GO = 0, FLY_ESCAPED = 1, FLY_PE = 2, FLY_COMPTON = 3, FLY_RAYLEIGH = 4 };

struct FlyCounters { unsigned steps, real; };

template <bool STATS>
__device__ __forceinline__ int fly_substep(const TransportParams& p, const float* __restrict__ s_tot,
                                           const float2* __restrict__ s_pec,
                                           float& x, float& y, float& z, const float u, const float v, const float w,
                                           const int ie, const float fe, const float maj, const float inv_maj,
                                           const float maj_out, const float inv_maj_out,
                                           const unsigned r_s, const unsigned r_a, unsigned& vox, int& mat,
                                           FlyCounters& cnt) {
    const float nl = -__logf(u01(r_s));
    if (STATS) ++cnt.steps;
    // Hull majorant (reading C24), branch-free: a photon that is beyond a face of the hull box and moving
    // away from it stays outside the (convex) box along its whole ray, so the majorant of the voxels outside the box
    // bounds mu on every point it can reach; any other photon uses the global majorant, which is valid everywhere.
    bool away = false;
    if (p.hull)
        away = (x >= p.bx1 && u >= 0.0f) || (x < p.bx0 && u <= 0.0f) || (y >= p.by1 && v >= 0.0f) ||
               (y < p.by0 && v <= 0.0f) || (z >= p.bz1 && w >= 0.0f) || (z < p.bz0 && w <= 0.0f);
    const float m_here = away ? maj_out : maj;
    const float s = nl * (away ? inv_maj_out : inv_maj);
    x = fmaf(s, u, x); y = fmaf(s, v, y); z = fmaf(s, w, z);
    const int ix = __float2int_rd(x * p.inv_dx), iy = __float2int_rd(y * p.inv_dy), iz = __float2int_rd(z * p.inv_dz);
    if ((unsigned)ix >= (unsigned)p.nx || (unsigned)iy >= (unsigned)p.ny || (unsigned)iz >= (unsigned)p.nz)
        return FLY_ESCAPED;
    vox = (unsigned)ix + (unsigned)p.nx * ((unsigned)iy + (unsigned)p.ny * (unsigned)iz);
    const unsigned t = __ldg(p.texels + vox);
    const int m = (int)(t >> 24);
    const float rho = (float)(t & 0xffffffu) * kDensityStep;
    const float* row = s_tot + m * p.ne + ie;
    const float mu = rho * fmaf(fe, row[1] - row[0], row[0]);
    const float rr = u01(r_a) * m_here;
    if (rr >= mu) return FLY_GO;                     // virtual collision
    if (STATS) ++cnt.real;
    const float2 a = s_pec[m * p.ne + ie], b = s_pec[m * p.ne + ie + 1];
    if (rr < rho * fmaf(fe, b.x - a.x, a.x)) return FLY_PE;              // the same draw picks the channel
    if (rr < rho * fmaf(fe, b.y - a.y, a.y) || !p.rayleigh_on) return FLY_COMPTON;
    mat = m;
    return FLY_RAYLEIGH;
}

// One Klein-Nishina try by composition-rejection on f(eps) = (1/eps + eps) g(eps).
// Returns true when accepted; then eps = E'/E and t = 1 - cos(theta).
__device__ __forceinline__ bool compton_try(const float E, const uint4 r, float& eps, float& t) {
    const float alpha = E * kInvE0;
    const float eps0 = __fdividef(1.0f, 1.0f + 2.0f * alpha);
    const float eps0sq = eps0 * eps0;
    const float a1 = -__logf(eps0);
    const float a2 = a1 + 0.5f * (1.0f - eps0sq);
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
    c = 1.0f - 2.0f * __fdividef(x2, T);
    return 2.0f * u01(r.y) <= 1.0f + c * c;
}

template <bool STATS, bool WAGG>
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
    unsigned hl = 0, blk = 0, vox = 0;
    float x = 0, y = 0, z = 0, u = 0, v = 0, w = 1, E = 0, fe = 0, maj = 1, inv_maj = 1, majo = 1, inv_majo = 1;
    unsigned pool_next = 0, pool_end = 0;   // warp-uniform
    bool exhausted = false;                 // warp-uniform

    float esc = 0.0f;
    unsigned c_steps = 0, c_real = 0, c_pe = 0, c_co = 0, c_ra = 0, c_esc = 0, c_cut = 0;

    auto set_energy = [&](float e) {
        const float t = (__logf(e) - p.lnE_min) * p.inv_dlnE;
        int i = (int)t;
        i = max(0, min(i, p.ne - 2));
        ie = i; fe = t - (float)i;
        maj = fmaf(fe, s_maj[i + 1] - s_maj[i], s_maj[i]);
        inv_maj = __fdividef(1.0f, maj);
        majo = fmaf(fe, s_majo[i + 1] - s_majo[i], s_majo[i]);
        inv_majo = __fdividef(1.0f, majo);
    };

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

        // ---- one Philox block per live lane ---------------------------------------------------
        const unsigned long long h = p.hist_base + hl;
        const unsigned stream = (state == ST_SOURCE) ? 0u : 1u + (unsigned)photon;
        const uint4 r = philox4x32_10(make_uint4((unsigned)h, (unsigned)(h >> 32), blk, stream), p.key0, p.key1);
        ++blk;

        bool dead = false;
        if (state == ST_FLY) {
            FlyCounters fc = {0u, 0u};
            int code = fly_substep<STATS>(p, s_tot, s_pec, x, y, z, u, v, w, ie, fe, maj, inv_maj, majo, inv_majo, r.x, r.y, vox, mat, fc);
            if (code == FLY_GO)
                code = fly_substep<STATS>(p, s_tot, s_pec, x, y, z, u, v, w, ie, fe, maj, inv_maj, majo, inv_majo, r.z, r.w, vox, mat, fc);
            if (STATS) { c_steps += fc.steps; c_real += fc.real; }
            if (code == FLY_ESCAPED) { if (STATS) { esc += E; ++c_esc; } dead = true; }
            else if (code == FLY_PE) { if (STATS) ++c_pe; deposit<WAGG>(p.batch, vox, E); dead = true; }   // all energy local
            else if (code == FLY_COMPTON) state = ST_COMPTON;
            else if (code == FLY_RAYLEIGH) state = ST_RAYLEIGH;
        } else if (state == ST_COMPTON) {
            float eps, t;
            if (compton_try(E, r, eps, t)) {
                if (STATS) ++c_co;
                float dep = E * (1.0f - eps);     // recoil electron deposited locally
                E *= eps;
                rotate(u, v, w, 1.0f - t, kTwoPi * u01(r.w));
                if (E < p.cutoff) { dep += E; dead = true; if (STATS) ++c_cut; }
                else { set_energy(E); state = ST_FLY; }
                deposit<WAGG>(p.batch, vox, dep);
            }
        } else if (state == ST_RAYLEIGH) {
            float c;
            if (rayleigh_try(E, r, s_x2, s_cum + mat * p.n_x2, p.n_x2, c)) {
                if (STATS) ++c_ra;
                rotate(u, v, w, c, kTwoPi * u01(r.z));
                state = ST_FLY;
            }
        } else {   // ST_SOURCE
            const uint4 r2 = philox4x32_10(make_uint4((unsigned)h, (unsigned)(h >> 32), 1u, 0u), p.key0, p.key1);
            unsigned voxel;
            if (p.point_source) {
                x = p.px; y = p.py; z = p.pz;
                voxel = 0;
                if (p.positron_ke > 0.0f) {
                    const int ix = __float2int_rd(x * p.inv_dx), iy = __float2int_rd(y * p.inv_dy),
                              iz = __float2int_rd(z * p.inv_dz);
                    voxel = (unsigned)ix + (unsigned)p.nx * ((unsigned)iy + (unsigned)p.ny * (unsigned)iz);
                }
            } else {
                // alias table over the active voxels; 64 random bits pick the bin (n_alias can exceed 2^24)
                const unsigned long long r64 = ((unsigned long long)r.x << 32) | r.y;
                const unsigned j = (unsigned)__umul64hi(r64, (unsigned long long)p.n_alias);
                const uint4 a = __ldg(p.alias + j);
                voxel = (r.z < a.x) ? a.y : a.z;
                const unsigned nxy = (unsigned)p.nx * (unsigned)p.ny;
                const unsigned iz = voxel / nxy, rem = voxel - iz * nxy;
                const unsigned iy = rem / (unsigned)p.nx, ix = rem - iy * (unsigned)p.nx;
                x = ((float)ix + u01(r.w)) * p.dx;       // uniform inside the voxel
                y = ((float)iy + u01(r2.x)) * p.dy;
                z = ((float)iz + u01(r2.y)) * p.dz;
            }
            const float ct = 2.0f * u01(r2.z) - 1.0f;    // isotropic direction
            const float st = sqrtf(fmaxf(0.0f, 1.0f - ct * ct));
            float sp, cp;
            __sincosf(kTwoPi * u01(r2.w), &sp, &cp);
            u = st * cp; v = st * sp; w = ct;
            stash[0 * kThreads] = x; stash[1 * kThreads] = y; stash[2 * kThreads] = z;
            stash[3 * kThreads] = u; stash[4 * kThreads] = v; stash[5 * kThreads] = w;
            if (p.positron_ke > 0.0f) deposit<WAGG>(p.batch, voxel, p.positron_ke);
            E = kE0; ie = p.ie0; fe = p.fe0; maj = p.maj0; inv_maj = p.inv_maj0; majo = p.majo0; inv_majo = p.inv_majo0;
            photon = 0; blk = 0; state = ST_FLY;
        }

        if (dead) {
            if (photon == 0 && p.photons_per_decay == 2) {   // the partner photon: same point, opposite direction
                photon = 1; blk = 0; state = ST_FLY;
                x = stash[0 * kThreads]; y = stash[1 * kThreads]; z = stash[2 * kThreads];
                u = -stash[3 * kThreads]; v = -stash[4 * kThreads]; w = -stash[5 * kThreads];
                E = kE0; ie = p.ie0; fe = p.fe0; maj = p.maj0; inv_maj = p.inv_maj0; majo = p.majo0; inv_majo = p.inv_majo0;
            } else {
                state = ST_NEED;
            }
        }
    }

    if (STATS) {
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
// Schedule 2: event-based at warp scope.  Each warp owns kSlots photon slots in shared memory (SoA, one word per
// field per slot).  A trip: count the slots waiting for each event type (one redux), pick the type with the most
// waiting slots, compact up to 32 of them (ballot + prefix), run that ONE event type with those lanes, write the
// slots back.  A slot whose decay is complete waits for SOURCE, which hands it the next history index of the launch.
// Same Philox counters and the same per-event arithmetic as schedule 1: the two schedules produce the same
// histories; only the order of the fp32 atomics differs.
#ifndef ANM_POOL_THREADS
#define ANM_POOL_THREADS 1024
#endif
#ifndef ANM_POOL_MIN_BLOCKS
#define ANM_POOL_MIN_BLOCKS 1
#endif
constexpr int kPoolThreads = ANM_POOL_THREADS;
constexpr int kPoolWarps = kPoolThreads / 32;
constexpr int kPoolMinBlocksPerSM = ANM_POOL_MIN_BLOCKS;
constexpr int kSlots = 64;                  // per warp
constexpr int kRayleighBatch = 8;           // run the (rare) Rayleigh event once this many slots wait for it
enum : int { F_X = 0, F_Y, F_Z, F_U, F_V, F_W, F_E, F_TV /* FLY: ln-E grid coordinate; COMPTON/RAYLEIGH: voxel */,
             F_HL, F_META, F_SX, F_SY, F_SZ, F_SU, F_SV, F_SW, kSlotFields };
// meta = state (bits 0-2) | photon (bit 3) | material (bits 4-6) | Philox block counter (bits 7-31)
constexpr size_t kPoolWarpBytes = (size_t)kSlotFields * kSlots * 4 + 32;   // + the compaction list (one byte per lane)

template <bool STATS>
__global__ void __launch_bounds__(kPoolThreads, kPoolMinBlocksPerSM)
transport_pool_kernel(const __grid_constant__ TransportParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* s_pec = reinterpret_cast<float2*>(smem_raw);            // [nm*ne]
    float* s_tot = reinterpret_cast<float*>(s_pec + p.nm * p.ne);   // [nm*ne]
    float* s_maj = s_tot + p.nm * p.ne;                             // [ne]
    float* s_majo = s_maj + p.ne;                                   // [ne]
    float* s_x2 = s_majo + p.ne;                                    // [n_x2]
    float* s_cum = s_x2 + p.n_x2;                                   // [nm*n_x2]
    unsigned char* s_pool = reinterpret_cast<unsigned char*>(s_cum + p.nm * p.n_x2);
    for (int i = threadIdx.x; i < p.nm * p.ne; i += kPoolThreads) { s_pec[i] = p.tab_pec[i]; s_tot[i] = p.tab_tot[i]; }
    for (int i = threadIdx.x; i < p.ne; i += kPoolThreads) { s_maj[i] = p.tab_maj[i]; s_majo[i] = p.tab_maj_out[i]; }
    for (int i = threadIdx.x; i < p.n_x2; i += kPoolThreads) s_x2[i] = p.ray_x2[i];
    for (int i = threadIdx.x; i < p.nm * p.n_x2; i += kPoolThreads) s_cum[i] = p.ray_cum[i];

    const unsigned lane = threadIdx.x & 31u;
    const unsigned lanemask_lt = (1u << lane) - 1u;
    float* slots = reinterpret_cast<float*>(s_pool + (size_t)(threadIdx.x >> 5) * kPoolWarpBytes);
    unsigned* slots_u = reinterpret_cast<unsigned*>(slots);
    unsigned char* list = reinterpret_cast<unsigned char*>(slots + kSlotFields * kSlots);
#pragma unroll
    for (int k = 0; k < kSlots / 32; ++k) slots_u[F_META * kSlots + lane + 32 * k] = ST_SOURCE;
    __syncthreads();

    unsigned pool_next = 0, pool_end = 0;   // warp-uniform
    bool exhausted = false;                 // warp-uniform
    unsigned trip = 0;
    const float t0 = (float)p.ie0 + p.fe0;  // ln-E grid coordinate of E0
    const float t_max = (float)(p.ne - 1) - 1.0f / 1024.0f;

    float esc = 0.0f;
    unsigned c_pe = 0, c_co = 0, c_ra = 0, c_esc = 0, c_cut = 0;
    FlyCounters fc = {0u, 0u};

    for (;; ++trip) {
        __syncwarp();
        // ---- vote: how many slots wait for each event type --------------------------------------------
        const unsigned m0 = slots_u[F_META * kSlots + lane], m1 = slots_u[F_META * kSlots + lane + 32];
        const int st0 = (int)(m0 & 7u), st1 = (int)(m1 & 7u);
        // byte 0 FLY, byte 1 COMPTON, byte 2 SOURCE (and NEED), byte 3 RAYLEIGH; DONE counts nowhere
        constexpr unsigned kShift = 16u | (16u << 5) | (0u << 10) | (8u << 15) | (24u << 20);
        const unsigned inc0 = (st0 == ST_DONE) ? 0u : 1u << ((kShift >> (5 * st0)) & 31u);
        const unsigned inc1 = (st1 == ST_DONE) ? 0u : 1u << ((kShift >> (5 * st1)) & 31u);
        const unsigned tot = __reduce_add_sync(0xffffffffu, inc0 + inc1);
        if (tot == 0u) break;
        const unsigned nF = tot & 255u, nC = (tot >> 8) & 255u, nS = (tot >> 16) & 255u, nR = tot >> 24;
        int X = ST_FLY;
        unsigned best = nF;
        if (nC > best) { X = ST_COMPTON; best = nC; }
        if (nS > best) { X = ST_SOURCE; best = nS; }
        if (nR > best || nR >= (unsigned)kRayleighBatch) X = ST_RAYLEIGH;
        // ---- compact the waiting slots; the half of the pool that goes first alternates ------------------
        const bool h0 = (X == ST_SOURCE) ? (st0 <= ST_SOURCE) : (st0 == X);
        const bool h1 = (X == ST_SOURCE) ? (st1 <= ST_SOURCE) : (st1 == X);
        const unsigned b0 = __ballot_sync(0xffffffffu, h0), b1 = __ballot_sync(0xffffffffu, h1);
        const bool flip = (trip & 1u) != 0u;
        const unsigned r0 = __popc(b0 & lanemask_lt) + (flip ? __popc(b1) : 0u);
        const unsigned r1 = __popc(b1 & lanemask_lt) + (flip ? 0u : __popc(b0));
        if (h0 && r0 < 32u) list[r0] = (unsigned char)lane;
        if (h1 && r1 < 32u) list[r1] = (unsigned char)(lane + 32u);
        __syncwarp();
        unsigned n = min((unsigned)(__popc(b0) + __popc(b1)), 32u);
        unsigned hl_new = 0;
        if (X == ST_SOURCE) {                 // hand out history indices (warp-uniform bookkeeping)
            if (pool_next == pool_end && !exhausted) {
                unsigned base = 0;
                if (lane == 0) base = atomicAdd(p.counter, kChunk);
                base = __shfl_sync(0xffffffffu, base, 0);
                pool_next = min(base, p.n_hist);
                pool_end = min(base + kChunk, p.n_hist);
                exhausted = (pool_next == pool_end);
            }
            const unsigned avail = pool_end - pool_next;
            if (exhausted) {                  // nothing left in this launch: the waiting slots are finished
                if (lane < n) slots_u[F_META * kSlots + list[lane]] = ST_DONE;
                continue;
            }
            n = min(n, avail);
            hl_new = pool_next + lane;
            pool_next += n;
        }
        if (lane >= n) continue;
        const unsigned slot = list[lane];
        float* S = slots + slot;
        unsigned* SU = slots_u + slot;

        // a finished photon: start the partner (same point, opposite direction) or wait for a new history
        auto photon_ends = [&](unsigned meta) {
            if (!(meta & 8u) && p.photons_per_decay == 2) {
                S[F_X * kSlots] = S[F_SX * kSlots]; S[F_Y * kSlots] = S[F_SY * kSlots]; S[F_Z * kSlots] = S[F_SZ * kSlots];
                S[F_U * kSlots] = -S[F_SU * kSlots]; S[F_V * kSlots] = -S[F_SV * kSlots]; S[F_W * kSlots] = -S[F_SW * kSlots];
                S[F_E * kSlots] = kE0; S[F_TV * kSlots] = t0;
                SU[F_META * kSlots] = (unsigned)ST_FLY | 8u;
            } else {
                SU[F_META * kSlots] = ST_SOURCE;
            }
        };

        if (X == ST_SOURCE) {
            const unsigned long long h = p.hist_base + hl_new;
            const uint4 r = philox4x32_10(make_uint4((unsigned)h, (unsigned)(h >> 32), 0u, 0u), p.key0, p.key1);
            const uint4 r2 = philox4x32_10(make_uint4((unsigned)h, (unsigned)(h >> 32), 1u, 0u), p.key0, p.key1);
            float x, y, z;
            unsigned voxel;
            if (p.point_source) {
                x = p.px; y = p.py; z = p.pz;
                voxel = 0;
                if (p.positron_ke > 0.0f) {
                    const int ix = __float2int_rd(x * p.inv_dx), iy = __float2int_rd(y * p.inv_dy), iz = __float2int_rd(z * p.inv_dz);
                    voxel = (unsigned)ix + (unsigned)p.nx * ((unsigned)iy + (unsigned)p.ny * (unsigned)iz);
                }
            } else {
                const unsigned long long r64 = ((unsigned long long)r.x << 32) | r.y;
                const unsigned j = (unsigned)__umul64hi(r64, (unsigned long long)p.n_alias);
                const uint4 a = __ldg(p.alias + j);
                voxel = (r.z < a.x) ? a.y : a.z;
                const unsigned nxy = (unsigned)p.nx * (unsigned)p.ny;
                const unsigned iz = voxel / nxy, rem = voxel - iz * nxy;
                const unsigned iy = rem / (unsigned)p.nx, ix = rem - iy * (unsigned)p.nx;
                x = ((float)ix + u01(r.w)) * p.dx;
                y = ((float)iy + u01(r2.x)) * p.dy;
                z = ((float)iz + u01(r2.y)) * p.dz;
            }
            const float ct = 2.0f * u01(r2.z) - 1.0f;
            const float st = sqrtf(fmaxf(0.0f, 1.0f - ct * ct));
            float sp, cp;
            __sincosf(kTwoPi * u01(r2.w), &sp, &cp);
            const float u = st * cp, v = st * sp, w = ct;
            S[F_X * kSlots] = x; S[F_Y * kSlots] = y; S[F_Z * kSlots] = z;
            S[F_U * kSlots] = u; S[F_V * kSlots] = v; S[F_W * kSlots] = w;
            S[F_SX * kSlots] = x; S[F_SY * kSlots] = y; S[F_SZ * kSlots] = z;
            S[F_SU * kSlots] = u; S[F_SV * kSlots] = v; S[F_SW * kSlots] = w;
            S[F_E * kSlots] = kE0; S[F_TV * kSlots] = t0;
            SU[F_HL * kSlots] = hl_new;
            SU[F_META * kSlots] = ST_FLY;
            if (p.positron_ke > 0.0f) atomicAdd(p.batch + voxel, p.positron_ke);
            continue;
        }

        const unsigned meta = SU[F_META * kSlots];
        const unsigned long long h = p.hist_base + SU[F_HL * kSlots];
        const uint4 r = philox4x32_10(make_uint4((unsigned)h, (unsigned)(h >> 32), meta >> 7, 1u + ((meta >> 3) & 1u)), p.key0, p.key1);
        const unsigned meta_next = meta + 128u;    // block counter + 1

        if (X == ST_FLY) {
            float x = S[F_X * kSlots], y = S[F_Y * kSlots], z = S[F_Z * kSlots];
            const float u = S[F_U * kSlots], v = S[F_V * kSlots], w = S[F_W * kSlots];
            const float t = S[F_TV * kSlots];
            const int ie = (int)t;
            const float fe = t - (float)ie;
            const float maj = fmaf(fe, s_maj[ie + 1] - s_maj[ie], s_maj[ie]);
            const float inv_maj = __fdividef(1.0f, maj);
            const float majo = fmaf(fe, s_majo[ie + 1] - s_majo[ie], s_majo[ie]);
            const float inv_majo = __fdividef(1.0f, majo);
            unsigned vox = 0;
            int mat = 0;
            int code = fly_substep<STATS>(p, s_tot, s_pec, x, y, z, u, v, w, ie, fe, maj, inv_maj, majo, inv_majo, r.x, r.y, vox, mat, fc);
            if (code == FLY_GO)
                code = fly_substep<STATS>(p, s_tot, s_pec, x, y, z, u, v, w, ie, fe, maj, inv_maj, majo, inv_majo, r.z, r.w, vox, mat, fc);
            if (code == FLY_GO) {
                S[F_X * kSlots] = x; S[F_Y * kSlots] = y; S[F_Z * kSlots] = z;
                SU[F_META * kSlots] = meta_next;
            } else if (code == FLY_COMPTON || code == FLY_RAYLEIGH) {
                S[F_X * kSlots] = x; S[F_Y * kSlots] = y; S[F_Z * kSlots] = z;
                SU[F_TV * kSlots] = vox;
                SU[F_META * kSlots] = (meta_next & ~0x77u) | (code == FLY_COMPTON ? (unsigned)ST_COMPTON : (unsigned)ST_RAYLEIGH | ((unsigned)mat << 4));
            } else {
                const float E = S[F_E * kSlots];
                if (code == FLY_PE) { if (STATS) ++c_pe; atomicAdd(p.batch + vox, E); }      // all energy local
                else if (STATS) { esc += E; ++c_esc; }
                photon_ends(meta);
            }
        } else if (X == ST_COMPTON) {
            float E = S[F_E * kSlots];
            float eps, t;
            if (compton_try(E, r, eps, t)) {
                if (STATS) ++c_co;
                float u = S[F_U * kSlots], v = S[F_V * kSlots], w = S[F_W * kSlots];
                const unsigned vox = SU[F_TV * kSlots];
                float dep = E * (1.0f - eps);     // recoil electron deposited locally
                E *= eps;
                if (E < p.cutoff) {               // the rest is deposited locally
                    dep += E;
                    if (STATS) ++c_cut;
                    photon_ends(meta);
                } else {
                    rotate(u, v, w, 1.0f - t, kTwoPi * u01(r.w));
                    S[F_U * kSlots] = u; S[F_V * kSlots] = v; S[F_W * kSlots] = w;
                    S[F_E * kSlots] = E;
                    S[F_TV * kSlots] = fminf(fmaxf((__logf(E) - p.lnE_min) * p.inv_dlnE, 0.0f), t_max);
                    SU[F_META * kSlots] = (meta_next & ~0x77u) | (unsigned)ST_FLY;
                }
                atomicAdd(p.batch + vox, dep);
            } else {
                SU[F_META * kSlots] = meta_next;
            }
        } else {   // ST_RAYLEIGH
            const float E = S[F_E * kSlots];
            float c;
            if (rayleigh_try(E, r, s_x2, s_cum + ((meta >> 4) & 7u) * p.n_x2, p.n_x2, c)) {
                if (STATS) ++c_ra;
                float u = S[F_U * kSlots], v = S[F_V * kSlots], w = S[F_W * kSlots];
                rotate(u, v, w, c, kTwoPi * u01(r.z));
                S[F_U * kSlots] = u; S[F_V * kSlots] = v; S[F_W * kSlots] = w;
                S[F_TV * kSlots] = fminf(fmaxf((__logf(E) - p.lnE_min) * p.inv_dlnE, 0.0f), t_max);
                SU[F_META * kSlots] = (meta_next & ~0x77u) | (unsigned)ST_FLY;
            } else {
                SU[F_META * kSlots] = meta_next;
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
// A10: fold one batch.  x = batch[i]; sum += x; sumsq += x*x; batch = 0; organ_row[label] += x / (rho V).
// Streaming; most voxels of a patient volume are untouched air (x == 0) and cost one 16-byte read per 4.
constexpr int kFoldThreads = 256;

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
        float4 s = sum[i], q = sumsq[i];
        s.x += xv.x; s.y += xv.y; s.z += xv.z; s.w += xv.w;
        q.x = fmaf(xv.x, xv.x, q.x); q.y = fmaf(xv.y, xv.y, q.y); q.z = fmaf(xv.z, xv.z, q.z); q.w = fmaf(xv.w, xv.w, q.w);
        sum[i] = s; sumsq[i] = q;
        batch[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (organs) {
            const uint32_t l4 = labels4[i];
            if (l4) {
                const uint4 t = texels4[i];
                const float xs[4] = {xv.x, xv.y, xv.z, xv.w};
                const unsigned ts[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const unsigned l = (l4 >> (8 * k)) & 0xffu;
                    if (l && xs[k] != 0.0f)
                        atomicAdd(&s_org[l], (double)xs[k] * (double)inv_vox_cm3 /
                                                 ((double)(ts[k] & 0xffffffu) * (double)kDensityStep));
                }
            }
        }
    }
    if (organs) {
        __syncthreads();
        if ((int)threadIdx.x <= n_organs && threadIdx.x > 0 && s_org[threadIdx.x] != 0.0)
            atomicAdd(organ_row + threadIdx.x, s_org[threadIdx.x]);
    }
}

// ------------------------------------------------------------------------------------------------
// A11: one pass over the run's sums: per organ  sum of rel^2 over voxels with dose > 0, their count, organ
// energy;  total deposited energy.  rel^2 = (B Q / S^2 - 1) / (B - 1)  (batch standard error of the mean / mean).
struct OrganAccum { double rel2, n_nonzero, energy; };

__device__ __forceinline__ float rel_sigma(float S, float Q, int B) {
    if (!(S > 0.0f)) return 0.0f;
    const double r2 = ((double)B * (double)Q / ((double)S * (double)S) - 1.0) / (double)(B - 1);
    return r2 > 0.0 ? (float)sqrt(r2) : 0.0f;
}

__global__ void __launch_bounds__(kFoldThreads)
finalize_kernel(const float* __restrict__ sum, const float* __restrict__ sumsq, const uint8_t* __restrict__ labels,
                OrganAccum* __restrict__ organ, double* __restrict__ total_energy, int n_organs, size_t V, int B) {
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
               float* __restrict__ out, size_t V, int mode, double dose_factor /* k*scale/(N V_vox) */, int B, int zero_air) {
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
