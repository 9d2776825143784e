// anm_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, single-threaded fp64 CPU transport of 0.511 MeV annihilation photons through a
// voxel phantom, written step by step from the paper (arxiv 2111.11687, "PAPER.md") in the
// reading DESIGN.md lists.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may call it.  It shares no code with paper_2111_11687_b200/ (the CUDA
// path): only input arrays produced by anm_inputs/ are common to both.
//
// Deliberate algorithmic differences from the CUDA path (same distributions, different routes,
// so that the two check each other):
//   decay voxel   : inverse CDF, binary search on the fp64 cumulative activity   (CUDA: alias table)
//   direction     : Marsaglia (1972), the paper's choice, PAPER.md:L65          (CUDA: cos/phi)
//   tracking      : exact voxel-boundary stepping (3-D DDA)                      (CUDA: Woodcock)
//   Klein-Nishina : plain rejection from the uniform envelope on epsilon         (CUDA: Kahn-style)
//   arithmetic    : fp64 throughout, fp64 tallies                                (CUDA: fp32)
//
// A second, LOCKSTEP mode (tracking = 2 / 3, namespace lockstep below) restates the CUDA path's documented algorithm
// and draw schedule in fp64 so that the two can be compared history by history; it is pinned against
// the exact transport above (tests/test_oracle_lockstep.py).
//
// Parity pins (tests/test_oracle_*.py, -m "not gpu"): P1 Philox known answers; P3 KN sampler vs
// closed-form CDF and mean energy transfer; P4 flight vs brute-force line integrals of mu and
// exp(-mu x); P5 energy conservation; P6 infinite medium; P7 first-collision kerma; P8 source
// chi^2 / isotropy; P9 Rayleigh -> Thomson limit; P10 batch sigma calibration; P11 symmetry;
// P12 unit conversion.  No function here is "parity unpinned".
//
// Units: cm, MeV, g/cm^3.  Linear voxel index = ix + nx*(iy + ny*iz).

#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <vector>

namespace {

const double kElectronMassMeV = 0.51099895;   // "0.511 MeV", PAPER.md:L65 (reading C9)
const double kHcKeVAngstrom = 12.398419843;
const double kTwoPi = 6.283185307179586476925;

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al. 2011): the counter-based generator north_star (d) names.
// key = (seed lo, seed hi); counter = (history lo, history hi, block number, 0).
// ---------------------------------------------------------------------------------------------
inline void philox_round(uint32_t c[4], const uint32_t k[2]) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c[0];
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * c[2];
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    const uint32_t n0 = hi1 ^ c[1] ^ k[0];
    const uint32_t n1 = lo1;
    const uint32_t n2 = hi0 ^ c[3] ^ k[1];
    const uint32_t n3 = lo0;
    c[0] = n0; c[1] = n1; c[2] = n2; c[3] = n3;
}

void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c[4] = {ctr[0], ctr[1], ctr[2], ctr[3]};
    uint32_t k[2] = {key[0], key[1]};
    for (int r = 0; r < 10; ++r) {
        philox_round(c, k);
        k[0] += 0x9E3779B9u;
        k[1] += 0xBB67AE85u;
    }
    for (int i = 0; i < 4; ++i) out[i] = c[i];
}

struct Rng {
    uint32_t key[2];
    uint32_t ctr[4];
    uint32_t buf[4];
    int have;
    void start(uint64_t seed, uint64_t history) {
        key[0] = (uint32_t)seed; key[1] = (uint32_t)(seed >> 32);
        ctr[0] = (uint32_t)history; ctr[1] = (uint32_t)(history >> 32); ctr[2] = 0; ctr[3] = 0;
        have = 0;
    }
    uint32_t u32() {
        if (have == 0) { philox4x32_10(ctr, key, buf); ctr[2] += 1; have = 4; }
        return buf[4 - have--];
    }
    // uniform on (0,1): (r + 0.5) 2^-32 (reading C14)
    double uniform() { return ((double)u32() + 0.5) * (1.0 / 4294967296.0); }
    // 64 random bits -> uniform on [0,1) with 53-bit resolution (voxel pick needs > 32 bits)
    double uniform64() {
        const uint64_t hi = u32(), lo = u32();
        return (double)(((hi << 32) | lo) >> 11) * (1.0 / 9007199254740992.0);
    }
};

}  // namespace

extern "C" {

struct OrcTables {
    int32_t n_materials, n_energy;
    double lnE_min, dlnE;
    const float *mu_pe, *mu_compton, *mu_rayleigh;   // [n_materials][n_energy] cm^2/g
    int32_t n_x2, pad_;
    const float *ray_x2;                              // [n_x2]
    const float *ray_cum;                             // [n_materials][n_x2]
};

struct OrcProblem {
    int32_t nx, ny, nz, pad0_;
    double dx, dy, dz;                     // cm
    const uint8_t* material;               // [V]
    const float* density;                  // [V] g/cm^3
    const double* cdf;                     // [V] cumulative activity (orc_build_cdf) or null
    int32_t use_point_source, pad1_;
    double px, py, pz;                     // cm
    const uint8_t* labels;                 // [V] or null
    int32_t n_organs;
    int32_t photons_per_decay;             // 1 | 2
    int32_t rayleigh_on;
    int32_t tracking;                      // 0 exact DDA (the oracle); 1 Woodcock (cross-check only);
                                           // 2 | 3 lockstep with the CUDA path's documented schedule (global | hull majorant)
    double photon_cutoff;                  // MeV, 0.010
    double positron_ke;                    // MeV, 0 or 0.2498
    uint64_t n_total;                      // N decays of the whole run
    int32_t n_batches, pad2_;
    uint64_t seed;
    OrcTables t;
    // secondary-electron transport (PAPER.md:L67 electron cutoff 200 keV; reading C28)
    int32_t electron_on, n_t;              // n_t points of the kinetic-energy grid T_k = t_min + k dt
    double electron_cutoff;                // MeV; must equal t_min (the range table is "range above the cutoff")
    double t_min, dt;
    const float* e_range;                  // [n_materials][n_t] residual CSDA range above the cutoff, g/cm^2
    const float* activity;                 // [V] the activity map itself (lockstep mode rebuilds the alias table from it)
};

struct OrcStats {
    double emitted, deposited, escaped, max_history_residual;
    uint64_t n_histories, n_photons, n_crossings, n_collisions, n_pe, n_compton, n_rayleigh,
        n_escaped, n_cutoff, n_virtual, n_electrons, n_electron_crossings,
        n_substeps;   // lockstep mode (tracking 2 | 3): every Woodcock sub-step, real or virtual (the CUDA path's n_steps)
};

// ------------------------------------------------------------------ P1
void orc_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
    philox4x32_10(ctr, key, out);
}

// Table reader (reading C19): linear interpolation in ln E on a uniform ln E grid.
double orc_interp(const float* row, int n, double lnE_min, double dlnE, double E) {
    const double t = (std::log(E) - lnE_min) / dlnE;
    int i = (int)std::floor(t);
    if (i < 0) i = 0;
    if (i > n - 2) i = n - 2;
    const double f = t - (double)i;
    return (1.0 - f) * (double)row[i] + f * (double)row[i + 1];
}

// PAPER.md:L65 "The probability density distribution of the decay events ... is constructed through
// a linear conversion of the PET value": p_v = a_v / sum(a).  cdf[v] = a_0 + ... + a_v.
void orc_build_cdf(const float* activity, uint64_t n_voxels, double* cdf) {
    double run = 0.0;
    for (uint64_t v = 0; v < n_voxels; ++v) { run += (double)activity[v]; cdf[v] = run; }
}

// Inverse CDF: the first voxel v with cdf[v] > u * total  (u in [0,1)); zero-activity voxels have
// zero-width intervals and are never returned.
uint64_t orc_pick_voxel(const double* cdf, uint64_t n_voxels, double u) {
    const double target = u * cdf[n_voxels - 1];
    uint64_t lo = 0, hi = n_voxels - 1;
    while (lo < hi) {
        const uint64_t mid = lo + (hi - lo) / 2;
        if (cdf[mid] > target) hi = mid; else lo = mid + 1;
    }
    return lo;
}

}  // extern "C"

namespace {

// Marsaglia (1972): x1,x2 ~ U(-1,1) until s = x1^2+x2^2 < 1;
// d = (2 x1 sqrt(1-s), 2 x2 sqrt(1-s), 1-2s).
void isotropic_marsaglia(Rng& g, double d[3]) {
    for (;;) {
        const double x1 = 2.0 * g.uniform() - 1.0, x2 = 2.0 * g.uniform() - 1.0;
        const double s = x1 * x1 + x2 * x2;
        if (s >= 1.0) continue;
        const double r = std::sqrt(1.0 - s);
        d[0] = 2.0 * x1 * r; d[1] = 2.0 * x2 * r; d[2] = 1.0 - 2.0 * s;
        return;
    }
}

// Klein-Nishina ("Compton scattering ... explicitly considered"; reading C3: free
// electron).  eps = E'/E in [1/(1+2a), 1], a = E/mc^2, density f(eps) ~ eps + 1/eps - sin^2(theta),
// cos(theta) = 1 + 1/a - 1/(a eps).  Plain rejection: eps uniform, accept with f / (eps_min + 1/eps_min)
// (f <= eps + 1/eps, which decreases on (0,1]).
double kn_sample_eps(Rng& g, double E) {
    const double a = E / kElectronMassMeV;
    const double eps_min = 1.0 / (1.0 + 2.0 * a);
    const double bound = eps_min + 1.0 / eps_min;
    for (;;) {
        const double eps = eps_min + (1.0 - eps_min) * g.uniform();
        const double c = 1.0 + 1.0 / a - 1.0 / (a * eps);
        const double f = eps + 1.0 / eps - (1.0 - c * c);
        if (g.uniform() * bound <= f) return eps;
    }
}

double interp_grid(const float* x, const float* y, int n, double xq) {
    // piecewise-linear y(x) on an increasing grid; xq clamped to the grid
    if (xq <= (double)x[0]) return (double)y[0];
    if (xq >= (double)x[n - 1]) return (double)y[n - 1];
    int lo = 0, hi = n - 1;
    while (hi - lo > 1) { const int mid = (lo + hi) / 2; if ((double)x[mid] <= xq) lo = mid; else hi = mid; }
    const double f = (xq - (double)x[lo]) / ((double)x[hi] - (double)x[lo]);
    return (1.0 - f) * (double)y[lo] + f * (double)y[hi];
}

// Rayleigh (north_star "optional Rayleigh"; reading C4): form-factor sampling.  T = x_max^2 = (E/hc)^2.
// Draw x^2 from the tabulated piecewise-linear cumulative A(x^2) restricted to [0, T]; cos = 1 - 2 x^2/T;
// accept with probability (1 + cos^2)/2.
double rayleigh_sample_cos(Rng& g, const OrcTables& t, int m, double E) {
    const double xm = E * 1000.0 / kHcKeVAngstrom;
    const double T = xm * xm;
    const float* cum = t.ray_cum + (size_t)m * t.n_x2;
    const double A_T = interp_grid(t.ray_x2, cum, t.n_x2, T);
    for (;;) {
        const double target = g.uniform() * A_T;
        // invert the piecewise-linear cumulative
        int lo = 0, hi = t.n_x2 - 1;
        while (hi - lo > 1) { const int mid = (lo + hi) / 2; if ((double)cum[mid] <= target) lo = mid; else hi = mid; }
        const double c0 = cum[lo], c1 = cum[hi];
        double x2 = (double)t.ray_x2[lo];
        if (c1 > c0) x2 += (target - c0) / (c1 - c0) * ((double)t.ray_x2[hi] - (double)t.ray_x2[lo]);
        if (x2 > T) x2 = T;
        const double c = 1.0 - 2.0 * x2 / T;
        if (g.uniform() * 2.0 <= 1.0 + c * c) return c;
    }
}

// Rotate unit vector d by polar angle (cos_t) and azimuth phi about itself.
void rotate(const double d[3], double cos_t, double phi, double out[3]) {
    const double sin_t = std::sqrt(std::fmax(0.0, 1.0 - cos_t * cos_t));
    const double cp = std::cos(phi), sp = std::sin(phi);
    const double u = d[0], v = d[1], w = d[2];
    double o[3];
    if (std::fabs(w) < 0.99999) {
        const double s = std::sqrt(1.0 - w * w);
        o[0] = u * cos_t + sin_t * (u * w * cp - v * sp) / s;
        o[1] = v * cos_t + sin_t * (v * w * cp + u * sp) / s;
        o[2] = w * cos_t - sin_t * s * cp;
    } else {
        const double sg = w > 0 ? 1.0 : -1.0;
        o[0] = sin_t * cp; o[1] = sin_t * sp; o[2] = sg * cos_t;
    }
    const double n = std::sqrt(o[0] * o[0] + o[1] * o[1] + o[2] * o[2]);
    out[0] = o[0] / n; out[1] = o[1] / n; out[2] = o[2] / n;
}

struct Xs { double pe[8], co[8], ra[8], tot[8]; };   // per material, at the current energy

void load_xs(const OrcProblem& p, double E, Xs& xs) {
    const OrcTables& t = p.t;
    for (int m = 0; m < t.n_materials; ++m) {
        xs.pe[m] = orc_interp(t.mu_pe + (size_t)m * t.n_energy, t.n_energy, t.lnE_min, t.dlnE, E);
        xs.co[m] = orc_interp(t.mu_compton + (size_t)m * t.n_energy, t.n_energy, t.lnE_min, t.dlnE, E);
        xs.ra[m] = p.rayleigh_on
            ? orc_interp(t.mu_rayleigh + (size_t)m * t.n_energy, t.n_energy, t.lnE_min, t.dlnE, E) : 0.0;
        xs.tot[m] = xs.pe[m] + xs.co[m] + xs.ra[m];
    }
}

inline int64_t vox_index(const OrcProblem& p, const int i[3]) {
    return (int64_t)i[0] + (int64_t)p.nx * ((int64_t)i[1] + (int64_t)p.ny * (int64_t)i[2]);
}

// Exact flight: spend optical depth tau walking voxel to voxel along d.
// pos/vox are updated to the interaction point.  Returns 1 = collision, 0 = left the grid
// (reading C13: outside iff coordinate < 0 or >= L).
int flight_dda(const OrcProblem& p, const Xs& xs, double pos[3], const double d[3], int vox[3],
               double tau, double* dist_out, uint64_t* crossings) {
    const double h[3] = {p.dx, p.dy, p.dz};
    const int n[3] = {p.nx, p.ny, p.nz};
    double tmax[3], tdelta[3];
    int step[3];
    for (int a = 0; a < 3; ++a) {
        if (d[a] > 0.0) {
            step[a] = 1; tdelta[a] = h[a] / d[a];
            tmax[a] = ((double)(vox[a] + 1) * h[a] - pos[a]) / d[a];
        } else if (d[a] < 0.0) {
            step[a] = -1; tdelta[a] = -h[a] / d[a];
            tmax[a] = ((double)vox[a] * h[a] - pos[a]) / d[a];
        } else {
            step[a] = 0; tdelta[a] = std::numeric_limits<double>::infinity();
            tmax[a] = std::numeric_limits<double>::infinity();
        }
        if (tmax[a] < 0.0) tmax[a] = 0.0;
    }
    double t = 0.0;
    for (;;) {
        int a = 0;
        if (tmax[1] < tmax[a]) a = 1;
        if (tmax[2] < tmax[a]) a = 2;
        const int64_t v = vox_index(p, vox);
        const double mu = (double)p.density[v] * xs.tot[p.material[v]];
        const double seg = tmax[a] - t;
        if (tau <= mu * seg) {
            t += tau / mu;
            for (int k = 0; k < 3; ++k) pos[k] += t * d[k];
            *dist_out = t;
            return 1;
        }
        tau -= mu * seg;
        t = tmax[a];
        vox[a] += step[a];
        if (crossings) ++*crossings;
        if (vox[a] < 0 || vox[a] >= n[a]) {
            for (int k = 0; k < 3; ++k) pos[k] += t * d[k];
            *dist_out = t;
            return 0;
        }
        tmax[a] += tdelta[a];
    }
}

// Woodcock delta tracking against a global majorant -- NOT the oracle's tracking; kept only as a
// statistical cross-check of flight_dda (tests) and selected with OrcProblem.tracking = 1.
int flight_woodcock(const OrcProblem& p, const Xs& xs, double majorant, Rng& g, double pos[3],
                    const double d[3], int vox[3], double* dist_out, uint64_t* n_virtual) {
    const double h[3] = {p.dx, p.dy, p.dz};
    const int n[3] = {p.nx, p.ny, p.nz};
    double t = 0.0;
    for (;;) {
        const double s = -std::log(g.uniform()) / majorant;
        t += s;
        for (int k = 0; k < 3; ++k) {
            pos[k] += s * d[k];
            vox[k] = (int)std::floor(pos[k] / h[k]);
        }
        for (int k = 0; k < 3; ++k)
            if (vox[k] < 0 || vox[k] >= n[k]) { *dist_out = t; return 0; }
        const int64_t v = vox_index(p, vox);
        const double mu = (double)p.density[v] * xs.tot[p.material[v]];
        if (g.uniform() * majorant < mu) { *dist_out = t; return 1; }
        if (n_virtual) ++*n_virtual;
    }
}

struct Tally {
    double* batch;           // [V] energy of the current batch (MeV)
    double deposited;        // this history
    // history-by-history scoring ("the corresponding uncertainty is evaluated using the history-by-
    // history method (Walters et al., 2002)"), all null / unused unless requested:
    double* hbh_sumsq;       // [V] sum over finished histories of X_h^2, X_h = energy history h left in the voxel
    double* hbh_temp;        // [V] energy the voxel has received from the history last seen there
    int64_t* hbh_last;       // [V] index of that history (-1: none yet)
    int64_t history;         // the current history
};

// Walters' bookkeeping: a voxel's per-history energy is accumulated in hbh_temp while the same history keeps hitting
// it; the first hit by a NEW history closes the previous one: its square goes to hbh_sumsq.  (The sum of X_h itself
// is the batch tally's sum.)  A final sweep closes what is still open (hbh_close).
inline void deposit(Tally& ty, int64_t v, double e) {
    ty.batch[v] += e;
    ty.deposited += e;
    if (ty.hbh_sumsq) {
        if (ty.hbh_last[v] == ty.history) ty.hbh_temp[v] += e;
        else {
            ty.hbh_sumsq[v] += ty.hbh_temp[v] * ty.hbh_temp[v];
            ty.hbh_temp[v] = e;
            ty.hbh_last[v] = ty.history;
        }
    }
}

inline void hbh_close(Tally& ty, uint64_t V) {
    for (uint64_t v = 0; v < V; ++v) { ty.hbh_sumsq[v] += ty.hbh_temp[v] * ty.hbh_temp[v]; ty.hbh_temp[v] = 0.0; }
}

struct Workspace {
    std::vector<double> rho_max;   // per material, for the Woodcock cross-check
};

// ---------------------------------------------------------------------------------------------
// Secondary electrons ("A photon or an electron is transported ... until its energy falls below
// cutoff energy ... its remaining energy is deposited locally.  The cutoff energies for photons and electrons are
// set to 10 keV and 200 keV").  The paper does not describe its electron physics; reading C28: continuous
// slowing down along a STRAIGHT line in the electron's initial direction, no angular deflection, no secondaries.
//   residual range above the cutoff in material m:  r = R_m(T)  [g/cm^2], R_m piecewise linear on the T grid;
//   after a chord of length l in a voxel of density rho:  r' = r - rho l,  T' = R_m^{-1}(r')  (the exact inverse of
//   that piecewise-linear function);  T - T' is deposited in the voxel;
//   r' <= 0: the electron reaches the cutoff inside this voxel: all of T is deposited here (the slowing down to the
//   cutoff plus the cutoff energy itself, "deposited locally").
// An electron that leaves the grid carries its remaining energy out (counted as escaped).
// ---------------------------------------------------------------------------------------------
double e_range_of(const OrcProblem& p, int m, double T) {          // R_m(T)
    const float* R = p.e_range + (size_t)m * p.n_t;
    double x = (T - p.t_min) / p.dt;
    if (x <= 0.0) return 0.0;
    int k = (int)std::floor(x);
    if (k > p.n_t - 2) k = p.n_t - 2;                              // (orc_run requires the grid to reach E0, the largest electron)
    return (double)R[k] + (x - (double)k) * ((double)R[k + 1] - (double)R[k]);
}

double e_energy_of(const OrcProblem& p, int m, double r) {         // R_m^{-1}(r)
    const float* R = p.e_range + (size_t)m * p.n_t;
    if (r <= 0.0) return p.t_min;
    int k = 0;
    while (k < p.n_t - 2 && (double)R[k + 1] <= r) ++k;            // segment with R[k] <= r < R[k+1]
    const double f = (r - (double)R[k]) / ((double)R[k + 1] - (double)R[k]);
    return p.t_min + ((double)k + f) * p.dt;
}

// Walk one electron from pos (inside voxel vox) along unit vector e with kinetic energy T > cutoff.
// dep(v, energy) is called once per voxel that receives energy.  Returns the energy carried out of the grid (0 if
// the electron stopped inside).
template <class Dep>
double electron_walk(const OrcProblem& p, const double pos[3], const double e[3], const int vox0[3], double T,
                     Dep dep, uint64_t* crossings) {
    const double h[3] = {p.dx, p.dy, p.dz};
    const int n[3] = {p.nx, p.ny, p.nz};
    int vox[3] = {vox0[0], vox0[1], vox0[2]};
    double tmax[3], tdelta[3];
    int step[3];
    for (int a = 0; a < 3; ++a) {                                  // the same voxel-boundary stepping as flight_dda
        if (e[a] > 0.0) { step[a] = 1; tdelta[a] = h[a] / e[a]; tmax[a] = ((double)(vox[a] + 1) * h[a] - pos[a]) / e[a]; }
        else if (e[a] < 0.0) { step[a] = -1; tdelta[a] = -h[a] / e[a]; tmax[a] = ((double)vox[a] * h[a] - pos[a]) / e[a]; }
        else { step[a] = 0; tdelta[a] = tmax[a] = std::numeric_limits<double>::infinity(); }
        if (tmax[a] < 0.0) tmax[a] = 0.0;
    }
    double t = 0.0;
    for (;;) {
        int a = 0;
        if (tmax[1] < tmax[a]) a = 1;
        if (tmax[2] < tmax[a]) a = 2;
        const int64_t v = vox_index(p, vox);
        const int m = p.material[v];
        const double rho = (double)p.density[v];
        const double chord = tmax[a] - t;
        const double r = e_range_of(p, m, T);
        if (rho * chord >= r) { dep(v, T); return 0.0; }           // reaches the cutoff here: everything local
        const double T_new = e_energy_of(p, m, r - rho * chord);
        if (T > T_new) dep(v, T - T_new);
        T = T_new;
        t = tmax[a];
        vox[a] += step[a];
        if (crossings) ++*crossings;
        if (vox[a] < 0 || vox[a] >= n[a]) return T;
        tmax[a] += tdelta[a];
    }
}

// Direction of the Compton recoil electron: momentum conservation, p_e = k - k' with photon momenta k = E d / c,
// k' = eps E d' / c.  (Textbook check: cot(phi_e) = (1 + alpha) tan(theta / 2).)
void compton_electron_direction(double E, double eps, const double d[3], const double d_new[3], double out[3]) {
    double pe[3] = {E * d[0] - E * eps * d_new[0], E * d[1] - E * eps * d_new[1], E * d[2] - E * eps * d_new[2]};
    const double nrm = std::sqrt(pe[0] * pe[0] + pe[1] * pe[1] + pe[2] * pe[2]);
    for (int a = 0; a < 3; ++a) out[a] = nrm > 0.0 ? pe[a] / nrm : d[a];
}

// Energy T set free as an electron at pos in voxel vox with direction e: transported if the option is on and T is
// above the electron cutoff, else deposited on the spot (north_star's reading C2).
void release_electron(const OrcProblem& p, const double pos[3], const double e[3], const int vox[3], double T,
                      Tally& ty, OrcStats& st, double* escaped) {
    if (!(T > 0.0)) return;
    if (!p.electron_on || T <= p.electron_cutoff) { deposit(ty, vox_index(p, vox), T); return; }
    ++st.n_electrons;
    *escaped += electron_walk(p, pos, e, vox, T, [&](int64_t v, double x) { deposit(ty, v, x); }, &st.n_electron_crossings);
}

// One photon from (pos, d, E) until absorbed, below cutoff, or out of the grid.
// fc_* : first-collision record (P7), may be null.
void transport_photon(const OrcProblem& p, const Workspace& ws, Rng& g, double pos[3], double d[3],
                      int vox[3], double E, Tally& ty, OrcStats& st, double* escaped,
                      double* fc_dist, double* fc_dep) {
    Xs xs;
    load_xs(p, E, xs);
    bool first = true;
    ++st.n_photons;
    for (;;) {
        double dist = 0.0;
        int hit;
        if (p.tracking == 0) {
            const double tau = -std::log(g.uniform());
            hit = flight_dda(p, xs, pos, d, vox, tau, &dist, &st.n_crossings);
        } else {
            double maj = 0.0;
            for (int m = 0; m < p.t.n_materials; ++m) maj = std::fmax(maj, ws.rho_max[m] * xs.tot[m]);
            hit = flight_woodcock(p, xs, maj, g, pos, d, vox, &dist, &st.n_virtual);
        }
        if (!hit) {   // "photons are killed at the phantom boundary" (BASELINE.json cfg0)
            *escaped += E;
            ++st.n_escaped;
            if (first && fc_dist) { *fc_dist = -1.0; *fc_dep = 0.0; }
            return;
        }
        ++st.n_collisions;
        const int64_t v = vox_index(p, vox);
        const int m = p.material[v];
        // interaction type proportional to the partial coefficients
        const double u = g.uniform() * xs.tot[m];
        double dep_here = 0.0, dep_first = 0.0;   // dep_here: photon energy left on the spot; dep_first: energy transferred
        bool alive = true;
        if (u < xs.pe[m]) {
            // photoelectric: all energy to one electron moving in the photon's direction (reading C5: no
            // fluorescence, binding energy neglected; C28); deposited locally unless electron transport is on
            ++st.n_pe;
            release_electron(p, pos, d, vox, E, ty, st, escaped);
            dep_first = E;
            alive = false;
        } else if (u < xs.pe[m] + xs.co[m]) {
            ++st.n_compton;
            const double a = E / kElectronMassMeV;
            const double eps = kn_sample_eps(g, E);
            const double cos_t = 1.0 + 1.0 / a - 1.0 / (a * eps);
            const double phi = kTwoPi * g.uniform();
            const double T = E * (1.0 - eps);   // recoil electron: deposited locally (north_star; reading C2) ...
            double nd[3];
            rotate(d, cos_t, phi, nd);
            {   // ... or transported (C28) along its momentum
                double pe[3];
                compton_electron_direction(E, eps, d, nd, pe);
                release_electron(p, pos, pe, vox, T, ty, st, escaped);
            }
            dep_first = T;
            E *= eps;
            d[0] = nd[0]; d[1] = nd[1]; d[2] = nd[2];
            if (E < p.photon_cutoff) {       // below cutoff, remaining energy deposited locally
                dep_here += E;
                dep_first += E;
                ++st.n_cutoff;
                alive = false;
            } else {
                load_xs(p, E, xs);
            }
        } else {
            ++st.n_rayleigh;
            const double cos_t = rayleigh_sample_cos(g, p.t, m, E);
            const double phi = kTwoPi * g.uniform();
            double nd[3];
            rotate(d, cos_t, phi, nd);
            d[0] = nd[0]; d[1] = nd[1]; d[2] = nd[2];
        }
        if (dep_here > 0.0) deposit(ty, v, dep_here);
        if (first && fc_dist) { *fc_dist = dist; *fc_dep = dep_first; }
        first = false;
        if (!alive) return;
    }
}

void sample_source(const OrcProblem& p, Rng& g, double pos[3], double d[3], int vox[3]) {
    const double h[3] = {p.dx, p.dy, p.dz};
    if (p.use_point_source) {
        pos[0] = p.px; pos[1] = p.py; pos[2] = p.pz;
        for (int a = 0; a < 3; ++a) vox[a] = (int)std::floor(pos[a] / h[a]);   // reading C13
    } else {
        const uint64_t V = (uint64_t)p.nx * p.ny * p.nz;
        const uint64_t v = orc_pick_voxel(p.cdf, V, g.uniform64());
        vox[0] = (int)(v % (uint64_t)p.nx);
        vox[1] = (int)((v / (uint64_t)p.nx) % (uint64_t)p.ny);
        vox[2] = (int)(v / ((uint64_t)p.nx * (uint64_t)p.ny));
        for (int a = 0; a < 3; ++a) pos[a] = ((double)vox[a] + g.uniform()) * h[a];   // uniform in the voxel (C11)
    }
    isotropic_marsaglia(g, d);
}

}  // namespace

extern "C" {

// ----------------------------------------------------------------- exposed pieces (pins)
void orc_isotropic_many(uint64_t seed, uint64_t n, double* dirs /*[n][3]*/) {
    for (uint64_t i = 0; i < n; ++i) { Rng g; g.start(seed, i); isotropic_marsaglia(g, dirs + 3 * i); }
}

void orc_kn_sample_many(double E, uint64_t seed, uint64_t n, double* eps) {
    for (uint64_t i = 0; i < n; ++i) { Rng g; g.start(seed, i); eps[i] = kn_sample_eps(g, E); }
}

void orc_rayleigh_sample_many(const OrcTables* t, int material, double E, uint64_t seed, uint64_t n,
                              double* cos_out) {
    for (uint64_t i = 0; i < n; ++i) { Rng g; g.start(seed, i); cos_out[i] = rayleigh_sample_cos(g, *t, material, E); }
}

void orc_rotate(const double* d, double cos_t, double phi, double* out) { rotate(d, cos_t, phi, out); }

void orc_sample_source_many(const OrcProblem* p, uint64_t h0, uint64_t n, double* pos /*[n][3]*/,
                            double* dirs /*[n][3]*/, int64_t* voxel /*[n]*/) {
    for (uint64_t i = 0; i < n; ++i) {
        Rng g; g.start(p->seed, h0 + i);
        int vox[3];
        sample_source(*p, g, pos + 3 * i, dirs + 3 * i, vox);
        voxel[i] = vox_index(*p, vox);
    }
}

// One exact flight with a GIVEN optical depth tau from pos along d at energy E.  Returns 1 and the
// interaction point/voxel/distance, or 0 (escaped; out_pos = exit point).
int orc_flight(const OrcProblem* p, const double* pos, const double* d, double E, double tau,
               double* out_pos, int64_t* out_voxel, double* out_dist) {
    Xs xs;
    load_xs(*p, E, xs);
    const double h[3] = {p->dx, p->dy, p->dz};
    double q[3] = {pos[0], pos[1], pos[2]};
    int vox[3];
    for (int a = 0; a < 3; ++a) vox[a] = (int)std::floor(q[a] / h[a]);
    const int hit = flight_dda(*p, xs, q, d, vox, tau, out_dist, nullptr);
    out_pos[0] = q[0]; out_pos[1] = q[1]; out_pos[2] = q[2];
    *out_voxel = hit ? vox_index(*p, vox) : -1;
    return hit;
}

// Electron pins: R_m(T), its inverse, and one walk.  out_voxel/out_dep receive up to cap (voxel, energy) pairs in
// path order; returns the number of pairs, *escaped = energy carried out of the grid.
void orc_compton_electron_direction(double E, double eps, const double* d, const double* d_new, double* out) {
    compton_electron_direction(E, eps, d, d_new, out);
}
double orc_e_range(const OrcProblem* p, int m, double T) { return e_range_of(*p, m, T); }
double orc_e_energy(const OrcProblem* p, int m, double r) { return e_energy_of(*p, m, r); }
int orc_electron_walk(const OrcProblem* p, const double* pos, const double* e, double T, int64_t* out_voxel,
                      double* out_dep, int cap, double* escaped) {
    const double h[3] = {p->dx, p->dy, p->dz};
    int vox[3];
    for (int a = 0; a < 3; ++a) vox[a] = (int)std::floor(pos[a] / h[a]);
    int n = 0;
    *escaped = electron_walk(*p, pos, e, vox, T, [&](int64_t v, double x) { if (n < cap) { out_voxel[n] = v; out_dep[n] = x; } ++n; }, nullptr);
    return n;
}

// ---------------------------------------------------------------------------------------------
// LOCKSTEP mode (OrcProblem.tracking = 2; "a --lockstep mode re-implements Woodcock with the GPU's draw
// schedule for per-history debugging").  NOT the oracle's own route: it restates, in fp64 and from DESIGN.md alone
// (readings C13, C14, C19, C23 and §5.1), the algorithm the CUDA path documents -- Woodcock delta tracking against the
// global majorant (hull majorant off), Kahn-style Klein-Nishina composition-rejection, the form-factor Rayleigh try,
// and the draw schedule: counter = (history lo, hi, block, stream), stream 0 = source, 1 + k = photon k, one block per
// event trip (FLY: two sub-steps {path, accept / channel} x 2; COMPTON: {branch, eps, accept, phi}; RAYLEIGH:
// {x^2, accept, phi}), uniforms u = ((r >> 8) + 0.5) 2^-24.  With the same seed it follows the SAME histories as the
// CUDA path up to fp32 rounding, so the two can be compared history by history (tests/test_gpu_lockstep.py).
// Decay sites: the given point, or from the activity map through an alias table rebuilt here by the ordered Walker /
// Vose sweep the CUDA set-up is defined by (build_alias below).
// ---------------------------------------------------------------------------------------------
namespace lockstep {

inline double u24(uint32_t r) { return ((double)(r >> 8) + 0.5) * (1.0 / 16777216.0); }

struct Tables {
    std::vector<float> maj_f;       // [ne] majorant at the grid nodes, 1/cm (fp32 like the cross-section tables)
    double t_max, t0;
    // hull majorant (reading C24; tracking = 3): the box of voxel indices [lo, hi) that encloses every voxel
    // denser than 1/20 of the densest one, and the majorant of the voxels OUTSIDE it
    bool hull = false;
    int lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0};
    std::vector<float> majo_f;
    // decay-voxel sampler of the CUDA path (DESIGN.md §5.1a SOURCE; anm.h anm_get_alias_table): alias table over the
    // active voxels, built by the ordered sweep described in build_alias below
    std::vector<uint32_t> a_thr, a_own, a_alias;
    bool in_box(const int v[3]) const { return v[0] >= lo[0] && v[0] < hi[0] && v[1] >= lo[1] && v[1] < hi[1] && v[2] >= lo[2] && v[2] < hi[2]; }
};

inline void block(const OrcProblem& p, uint64_t h, uint32_t blk, uint32_t stream, uint32_t out[4]) {
    const uint32_t key[2] = {(uint32_t)p.seed, (uint32_t)(p.seed >> 32)};
    const uint32_t ctr[4] = {(uint32_t)h, (uint32_t)(h >> 32), blk, stream};
    philox4x32_10(ctr, key, out);
}

// value of a [n_energy] float table at grid coordinate t (linear in the coordinate = linear in ln E, reading C19)
inline double lerp_t(const float* row, double t) {
    const int i = (int)t;
    const double f = t - (double)i;
    return (double)row[i] + f * ((double)row[i + 1] - (double)row[i]);
}

inline double energy_coordinate(const OrcProblem& p, const Tables& T, double E) {
    const double t = (std::log(E) - p.t.lnE_min) / p.t.dlnE;
    return std::fmin(std::fmax(t, 0.0), T.t_max);
}

// Walker / Vose alias table by the ORDERED sweep (DESIGN.md §2 "alias"): the M active voxels, weights w = a M / sum(a)
// (mean 1), are split in index order into light (w <= 1) and heavy (w > 1) ones.  Buckets are filled one by one: the
// current light voxel owns a bucket with probability w and the current heavy voxel tops it up; the heavy voxel's
// residual r shrinks by 1 - w each time, and once r < 1 the heavy voxel itself owns the next bucket with probability r,
// topped up by the next heavy voxel (whose residual absorbs the difference).  With L, H the exclusive prefix sums of the
// light / heavy weights, after i light and j heavy voxels are done the residual of heavy voxel j is
// r = L[i] + H[j+1] - (i + j).  threshold = floor(P(own) 2^32), saturated.
void build_alias(const OrcProblem& p, Tables& T) {
    const uint64_t V = (uint64_t)p.nx * p.ny * p.nz;
    double total = 0.0;
    uint64_t M = 0;
    for (uint64_t v = 0; v < V; ++v) if (p.activity[v] > 0.0f) { total += (double)p.activity[v]; ++M; }
    const double scale = (double)M / total;
    std::vector<uint32_t> light, heavy;
    for (uint64_t v = 0; v < V; ++v) {
        const float a = p.activity[v];
        if (a > 0.0f) ((double)a * scale <= 1.0 ? light : heavy).push_back((uint32_t)v);
    }
    const size_t nl = light.size(), nh = heavy.size();
    std::vector<double> L(nl + 1, 0.0), H(nh + 1, 0.0);
    for (size_t i = 0; i < nl; ++i) L[i + 1] = L[i] + (double)p.activity[light[i]] * scale;
    for (size_t j = 0; j < nh; ++j) H[j + 1] = H[j] + (double)p.activity[heavy[j]] * scale;
    auto thr = [](double prob) -> uint32_t {
        const double t = std::floor(std::fmin(std::fmax(prob, 0.0), 1.0) * 4294967296.0);
        return t >= 4294967295.0 ? 0xffffffffu : (uint32_t)t;
    };
    T.a_thr.resize(M); T.a_own.resize(M); T.a_alias.resize(M);
    size_t i = 0, j = 0;
    for (uint64_t k = 0; k < M; ++k) {
        if (nh == 0) { T.a_thr[k] = 0xffffffffu; T.a_own[k] = T.a_alias[k] = light[k]; continue; }
        const double r = L[i] + (j + 1 <= nh ? H[j + 1] : H[nh]) - (double)k;       // residual of heavy voxel j
        if (i < nl && (r >= 1.0 || j >= nh)) {
            const uint32_t v = light[i];
            T.a_thr[k] = thr((double)p.activity[v] * scale); T.a_own[k] = v; T.a_alias[k] = heavy[std::min(j, nh - 1)];
            ++i;
        } else {
            const uint32_t v = heavy[j];
            T.a_thr[k] = thr(r); T.a_own[k] = v; T.a_alias[k] = j + 1 < nh ? heavy[j + 1] : v;
            ++j;
        }
    }
}

Tables make_tables(const OrcProblem& p) {
    Tables T;
    const int ne = p.t.n_energy, nm = p.t.n_materials;
    const uint64_t V = (uint64_t)p.nx * p.ny * p.nz;
    std::vector<double> rho_max(nm, 0.0);
    for (uint64_t v = 0; v < V; ++v) rho_max[p.material[v]] = std::fmax(rho_max[p.material[v]], (double)p.density[v]);
    T.maj_f.assign(ne, 0.0f);
    for (int k = 0; k < ne; ++k) {
        double mx = 0.0;
        for (int m = 0; m < nm; ++m) {
            const size_t i = (size_t)m * ne + k;
            const double tot = (double)p.t.mu_pe[i] + (double)p.t.mu_compton[i] + (p.rayleigh_on ? (double)p.t.mu_rayleigh[i] : 0.0);
            mx = std::fmax(mx, rho_max[m] * tot);
        }
        T.maj_f[k] = (float)(mx * 1.000001 + 1e-30);   // DESIGN.md C19: x (1 + 1e-6), stored in fp32
    }
    T.t_max = (double)(ne - 1) - 1.0 / 1024.0;
    T.t0 = energy_coordinate(p, T, kElectronMassMeV);
    T.majo_f = T.maj_f;
    if (!p.use_point_source) build_alias(p, T);
    if (p.tracking == 3) {
        // densities sit on the 2^-20 g/cm^3 grid (C18): compare in counts, threshold = floor(max count / 20)
        uint64_t cmax = 0;
        for (uint64_t v = 0; v < V; ++v) cmax = std::max<uint64_t>(cmax, (uint64_t)std::llround((double)p.density[v] * 1048576.0));
        const uint64_t thr = cmax / 20;
        int lo[3] = {p.nx, p.ny, p.nz}, hi[3] = {0, 0, 0};
        for (int iz = 0; iz < p.nz; ++iz) for (int iy = 0; iy < p.ny; ++iy) for (int ix = 0; ix < p.nx; ++ix) {
            const int64_t v = (int64_t)ix + (int64_t)p.nx * ((int64_t)iy + (int64_t)p.ny * iz);
            if ((uint64_t)std::llround((double)p.density[v] * 1048576.0) > thr) {
                const int q[3] = {ix, iy, iz};
                for (int a = 0; a < 3; ++a) { lo[a] = std::min(lo[a], q[a]); hi[a] = std::max(hi[a], q[a] + 1); }
            }
        }
        const bool ok = hi[0] > lo[0] && hi[1] > lo[1] && hi[2] > lo[2] &&
                        (double)(hi[0] - lo[0]) * (hi[1] - lo[1]) * (hi[2] - lo[2]) <= 0.9 * (double)V;
        if (ok) {
            T.hull = true;
            for (int a = 0; a < 3; ++a) { T.lo[a] = lo[a]; T.hi[a] = hi[a]; }
            std::vector<double> rho_out(nm, 0.0);
            for (int iz = 0; iz < p.nz; ++iz) for (int iy = 0; iy < p.ny; ++iy) for (int ix = 0; ix < p.nx; ++ix) {
                const int q[3] = {ix, iy, iz};
                if (T.in_box(q)) continue;
                const int64_t v = (int64_t)ix + (int64_t)p.nx * ((int64_t)iy + (int64_t)p.ny * iz);
                rho_out[p.material[v]] = std::fmax(rho_out[p.material[v]], (double)p.density[v]);
            }
            for (int k = 0; k < ne; ++k) {
                double mo = 0.0;
                for (int m = 0; m < nm; ++m) {
                    const size_t i = (size_t)m * ne + k;
                    const double tot = (double)p.t.mu_pe[i] + (double)p.t.mu_compton[i] + (p.rayleigh_on ? (double)p.t.mu_rayleigh[i] : 0.0);
                    mo = std::fmax(mo, rho_out[m] * tot);
                }
                T.majo_f[k] = (float)(mo * 1.000001 + 1e-30);
            }
        }
    }
    return T;
}

// rotate d by polar angle (cos_t) and azimuth phi, in the CUDA path's convention (DESIGN.md §5.1 "rotate")
inline void rotate_ls(double d[3], double cos_t, double phi) {
    const double sin_t = std::sqrt(std::fmax(0.0, 1.0 - cos_t * cos_t));
    const double sp = std::sin(phi), cp = std::cos(phi);
    const double u = d[0], v = d[1], w = d[2];
    double a, b, c;
    if (std::fabs(w) < 0.99999) {
        const double s = std::sqrt(1.0 - w * w);
        const double k = sin_t / s;
        a = k * (u * w * cp - v * sp) + u * cos_t;
        b = k * (v * w * cp + u * sp) + v * cos_t;
        c = -(sin_t * s) * cp + w * cos_t;
    } else {
        a = sin_t * cp; b = sin_t * sp; c = std::copysign(cos_t, w);
    }
    const double n = 1.0 / std::sqrt(a * a + b * b + c * c);
    d[0] = a * n; d[1] = b * n; d[2] = c * n;
}

// One photon, stream = 1 + k, from (pos, d) at E0.  Returns nothing; tallies into ty, escaped energy into *escaped.
// Hull state of a photon (C24): IN = its last landing point (or its start) was inside the box; AWAY = it is outside the
// box and has flown straight since a point inside it -- a straight ray that has left a convex box never re-enters it,
// so an AWAY photon flies against the majorant of the voxels outside the box.  A scatter clears AWAY.
void photon(const OrcProblem& p, const Tables& T, uint64_t h, uint32_t stream, double pos[3], double d[3], Tally& ty,
            OrcStats& st, double* escaped, bool start_in_box) {
    bool hull_in = start_in_box, hull_away = false;
    const double hvox[3] = {p.dx, p.dy, p.dz};
    const int n[3] = {p.nx, p.ny, p.nz};
    const int ne = p.t.n_energy;
    double E = kElectronMassMeV, t = T.t0;
    uint32_t blk = 0;
    ++st.n_photons;
    for (;;) {
        // ---- FLY: sub-steps until a real collision or escape, two per block
        int channel = -1;          // 0 photoelectric, 1 Compton, 2 Rayleigh
        int64_t v = -1;
        int m = 0;
        int cvox[3] = {0, 0, 0};   // the collision voxel
        while (channel < 0) {
            uint32_t r[4];
            block(p, h, blk++, stream, r);
            for (int sub = 0; sub < 2 && channel < 0; ++sub) {
                const double maj = lerp_t(hull_away ? T.majo_f.data() : T.maj_f.data(), t);
                const double s = -std::log(u24(r[2 * sub])) / maj;
                int vox[3];
                bool inside = true;
                for (int a = 0; a < 3; ++a) {
                    pos[a] += s * d[a];
                    vox[a] = (int)std::floor(pos[a] / hvox[a]);
                    inside = inside && vox[a] >= 0 && vox[a] < n[a];
                }
                ++st.n_substeps;
                if (!inside) { *escaped += E; ++st.n_escaped; return; }
                if (T.hull) {
                    if (T.in_box(vox)) { hull_in = true; hull_away = false; }
                    else { hull_away = hull_in || hull_away; hull_in = false; }
                }
                v = vox_index(p, vox);
                cvox[0] = vox[0]; cvox[1] = vox[1]; cvox[2] = vox[2];
                m = p.material[v];
                const double rho = (double)p.density[v];
                const size_t row = (size_t)m * ne;
                const double pe = lerp_t(p.t.mu_pe + row, t), co = lerp_t(p.t.mu_compton + row, t);
                const double ra = p.rayleigh_on ? lerp_t(p.t.mu_rayleigh + row, t) : 0.0;
                const double rr = u24(r[2 * sub + 1]) * maj;
                if (rr < rho * (pe + co + ra)) {                  // real; the same draw picks the channel
                    ++st.n_collisions;
                    channel = rr < rho * pe ? 0 : ((rr < rho * (pe + co) || !p.rayleigh_on) ? 1 : 2);
                }
            }
        }
        if (channel == 0) { ++st.n_pe; release_electron(p, pos, d, cvox, E, ty, st, escaped); return; }   // electron along the photon
        if (channel == 1) {
            // ---- COMPTON: one Kahn-style composition-rejection try per block
            for (;;) {
                uint32_t r[4];
                block(p, h, blk++, stream, r);
                const double alpha = E / kElectronMassMeV;
                const double eps0 = 1.0 / (1.0 + 2.0 * alpha), eps0sq = eps0 * eps0;
                const double a1 = -std::log(eps0), a2 = a1 + 0.5 * (1.0 - eps0sq);
                const double u2 = u24(r[1]);
                double eps, epssq;
                if (a1 > a2 * u24(r[0])) { eps = std::exp(-a1 * u2); epssq = eps * eps; }
                else { epssq = eps0sq + (1.0 - eps0sq) * u2; eps = std::sqrt(epssq); }
                const double tt = (1.0 - eps) / (alpha * eps);                 // 1 - cos(theta)
                const double sint2 = std::fmax(0.0, tt * (2.0 - tt));
                const double g = 1.0 - eps * sint2 / (1.0 + epssq);
                if (!(g >= u24(r[2]))) continue;
                ++st.n_compton;
                const double Te = E * (1.0 - eps);                      // recoil electron
                const double E_old = E;
                E *= eps;
                const bool ends = E < p.photon_cutoff;
                const bool walk = p.electron_on && Te > p.electron_cutoff;
                const double d_old[3] = {d[0], d[1], d[2]};
                if (!ends || walk) rotate_ls(d, 1.0 - tt, kTwoPi * u24(r[3]));
                if (walk) {
                    double pe[3];
                    compton_electron_direction(E_old, eps, d_old, d, pe);
                    release_electron(p, pos, pe, cvox, Te, ty, st, escaped);
                } else {
                    deposit(ty, v, Te);
                }
                if (ends) { ++st.n_cutoff; deposit(ty, v, E); return; }
                hull_away = false;
                t = energy_coordinate(p, T, E);
                break;
            }
        } else {
            // ---- RAYLEIGH: one form-factor try per block
            for (;;) {
                uint32_t r[4];
                block(p, h, blk++, stream, r);
                const float* x2 = p.t.ray_x2;
                const float* cum = p.t.ray_cum + (size_t)m * p.t.n_x2;
                const double xm = E * (1000.0 / 12.398419843), TT = xm * xm;
                const double A_T = interp_grid(x2, cum, p.t.n_x2, TT);
                const double target = u24(r[0]) * A_T;
                int lo = 0, hi = p.t.n_x2 - 1;
                while (hi - lo > 1) { const int mid = (lo + hi) / 2; if ((double)cum[mid] <= target) lo = mid; else hi = mid; }
                double xx = (double)x2[lo];
                const double dc = (double)cum[hi] - (double)cum[lo];
                if (dc > 0.0) xx += (target - (double)cum[lo]) / dc * ((double)x2[hi] - (double)x2[lo]);
                xx = std::fmin(xx, TT);
                const double c = 1.0 - 2.0 * xx / TT;
                if (!(2.0 * u24(r[1]) <= 1.0 + c * c)) continue;
                ++st.n_rayleigh;
                rotate_ls(d, c, kTwoPi * u24(r[2]));
                hull_away = false;
                break;
            }
        }
    }
}

// One decay in point-source mode: stream 0 block 1 words 2, 3 give cos(theta) and phi of photon A; photon B = -A.
void history(const OrcProblem& p, const Tables& T, uint64_t h, Tally& ty, OrcStats& st, double* escaped, double* emitted) {
    const double hvox[3] = {p.dx, p.dy, p.dz};
    uint32_t r1[4], r2[4];
    block(p, h, 0, 0, r1);
    block(p, h, 1, 0, r2);
    const double ct = 2.0 * u24(r2[2]) - 1.0, sn = std::sqrt(std::fmax(0.0, 1.0 - ct * ct)), phi = kTwoPi * u24(r2[3]);
    const double d0[3] = {sn * std::cos(phi), sn * std::sin(phi), ct};
    int vox[3];
    double src[3] = {p.px, p.py, p.pz};
    if (p.use_point_source) {
        for (int a = 0; a < 3; ++a) vox[a] = (int)std::floor(src[a] / hvox[a]);
    } else {
        // bucket = floor(r64 M / 2^64) from 64 random bits; own voxel iff w2 < threshold, else the alias voxel;
        // uniform point inside the voxel from w3 and the first two words of block 1
        const unsigned __int128 r64 = ((unsigned __int128)r1[0] << 32) | r1[1];
        const uint64_t k = (uint64_t)((r64 * (unsigned __int128)T.a_thr.size()) >> 64);
        const uint32_t v = r1[2] < T.a_thr[k] ? T.a_own[k] : T.a_alias[k];
        vox[0] = (int)(v % (uint32_t)p.nx); vox[1] = (int)((v / (uint32_t)p.nx) % (uint32_t)p.ny); vox[2] = (int)(v / ((uint32_t)p.nx * (uint32_t)p.ny));
        const double off[3] = {u24(r1[3]), u24(r2[0]), u24(r2[1])};
        for (int a = 0; a < 3; ++a) src[a] = ((double)vox[a] + off[a]) * hvox[a];
    }
    if (p.positron_ke > 0.0) { *emitted += p.positron_ke; deposit(ty, vox_index(p, vox), p.positron_ke); }
    for (int k = 0; k < p.photons_per_decay; ++k) {
        double pos[3] = {src[0], src[1], src[2]};
        double d[3] = {k == 0 ? d0[0] : -d0[0], k == 0 ? d0[1] : -d0[1], k == 0 ? d0[2] : -d0[2]};
        *emitted += kElectronMassMeV;
        photon(p, T, h, 1u + (uint32_t)k, pos, d, ty, st, escaped, T.hull && T.in_box(vox));
    }
}

}  // namespace lockstep

// ----------------------------------------------------------------- the run
// Histories [h0, h1) of a run of n_total decays in n_batches batches; h0 and h1 must be batch
// boundaries (batch b = h / (n_total / n_batches); reading C15: n_total % n_batches == 0).
//   sum[V], sumsq[V]       += per-batch voxel energies x_{b,i} and x_{b,i}^2 (MeV, MeV^2)
//   organ_batch[B][n_organs+1] = sum over the organ's voxels of x_{b,i} / (rho_i V_vox)  (MeV/g); column 0 = unlabelled
//   fc_dist/fc_dep[h1-h0]  first-collision distance (cm; -1 = escaped uncollided) and deposit of photon A (may be null)
// Returns 0, or -1 on bad arguments.
//   hbh_sumsq[V]           += sum over the histories of this call of X_{h,i}^2 (MeV^2), history-by-history (may be null)
int orc_run(const OrcProblem* pp, uint64_t h0, uint64_t h1, double* sum, double* sumsq,
            double* organ_batch, OrcStats* stats, double* fc_dist, double* fc_dep, double* hbh_sumsq) {
    const OrcProblem& p = *pp;
    if (p.n_batches < 1 || p.n_total == 0 || p.n_total % (uint64_t)p.n_batches) return -1;
    const uint64_t nb = p.n_total / (uint64_t)p.n_batches;
    if (h0 % nb || h1 % nb || h1 < h0 || h1 > p.n_total) return -1;
    if (!p.use_point_source && !p.cdf) return -1;
    if (p.photons_per_decay != 1 && p.photons_per_decay != 2) return -1;
    if (p.electron_on && (!p.e_range || p.n_t < 2 || !(p.dt > 0.0) || p.electron_cutoff != p.t_min ||
                          p.t_min + p.dt * (p.n_t - 1) < kElectronMassMeV)) return -1;   // photo-electrons carry the whole photon energy (<= E0)
    const uint64_t V = (uint64_t)p.nx * p.ny * p.nz;
    const double vox_cm3 = p.dx * p.dy * p.dz;

    Workspace ws;
    ws.rho_max.assign(8, 0.0);
    if (p.tracking == 1)
        for (uint64_t v = 0; v < V; ++v)
            ws.rho_max[p.material[v]] = std::fmax(ws.rho_max[p.material[v]], (double)p.density[v]);

    if (p.tracking >= 2 && !p.use_point_source && !p.activity) return -1;
    lockstep::Tables ls_tables;
    if (p.tracking >= 2) ls_tables = lockstep::make_tables(p);
    std::vector<double> batch(V, 0.0);
    std::vector<double> hbh_acc, hbh_temp;
    std::vector<int64_t> hbh_last;
    if (hbh_sumsq) { hbh_acc.assign(V, 0.0); hbh_temp.assign(V, 0.0); hbh_last.assign(V, -1); }
    Tally ty{batch.data(), 0.0, hbh_sumsq ? hbh_acc.data() : nullptr, hbh_temp.data(), hbh_last.data(), -1};
    OrcStats st;
    std::memset(&st, 0, sizeof st);

    for (uint64_t b = h0 / nb; b < h1 / nb; ++b) {
        for (uint64_t h = b * nb; h < (b + 1) * nb; ++h) {
            if (p.tracking >= 2) {              // lockstep with the CUDA path's draw schedule (point source only)
                double emitted = 0.0, escaped = 0.0;
                ty.deposited = 0.0;
                ty.history = (int64_t)h;
                lockstep::history(p, ls_tables, h, ty, st, &escaped, &emitted);
                st.emitted += emitted; st.deposited += ty.deposited; st.escaped += escaped;
                const double res = std::fabs(ty.deposited + escaped - emitted);
                if (res > st.max_history_residual) st.max_history_residual = res;
                ++st.n_histories;
                continue;
            }
            Rng g;
            g.start(p.seed, h);
            double pos[3], d[3];
            int vox[3];
            sample_source(p, g, pos, d, vox);
            double emitted = 0.0, escaped = 0.0;
            ty.deposited = 0.0;
            ty.history = (int64_t)h;           // one decay (positron energy + both photons + their electrons) = one history
            if (p.positron_ke > 0.0) {   // constant positron kinetic energy deposited in the decay voxel (C10)
                emitted += p.positron_ke;
                deposit(ty, vox_index(p, vox), p.positron_ke);
            }
            // two photons of equal energy (0.511 MeV) in opposite directions
            for (int k = 0; k < p.photons_per_decay; ++k) {
                double q[3] = {pos[0], pos[1], pos[2]};
                double dd[3] = {k == 0 ? d[0] : -d[0], k == 0 ? d[1] : -d[1], k == 0 ? d[2] : -d[2]};
                int vv[3] = {vox[0], vox[1], vox[2]};
                emitted += kElectronMassMeV;
                const bool rec = (k == 0 && fc_dist != nullptr);
                transport_photon(p, ws, g, q, dd, vv, kElectronMassMeV, ty, st, &escaped,
                                 rec ? fc_dist + (h - h0) : nullptr, rec ? fc_dep + (h - h0) : nullptr);
            }
            st.emitted += emitted; st.deposited += ty.deposited; st.escaped += escaped;
            const double res = std::fabs(ty.deposited + escaped - emitted);
            if (res > st.max_history_residual) st.max_history_residual = res;
            ++st.n_histories;
        }
        // fold the batch
        double* ob = organ_batch ? organ_batch + (size_t)b * (size_t)(p.n_organs + 1) : nullptr;
        for (uint64_t v = 0; v < V; ++v) {
            const double x = batch[v];
            if (x != 0.0) {
                sum[v] += x;
                sumsq[v] += x * x;
                if (ob) ob[p.labels ? p.labels[v] : 0] += x / ((double)p.density[v] * vox_cm3);
                batch[v] = 0.0;
            }
        }
    }
    if (hbh_sumsq) {
        hbh_close(ty, V);
        for (uint64_t v = 0; v < V; ++v) hbh_sumsq[v] += hbh_acc[v];
    }
    if (stats) *stats = st;
    return 0;
}

}  // extern "C"
