/* anm.h -- C ABI of libanm.so: voxel Monte Carlo dose from annihilation photons on one B200.
 *
 * What it computes (arxiv 2111.11687 "ARCHER-NM", cited as PAPER.md:L<line>):
 *   PAPER.md:L65  a voxel phantom of (material, density) from CT; a decay pdf that is a linear
 *                 conversion of the PET voxel value; each decay -> two 0.511 MeV photons in opposite,
 *                 isotropically distributed directions.
 *   PAPER.md:L67  photoelectric absorption and Compton scattering (pair production impossible below
 *                 1.02 MeV); a photon is followed until its energy falls below the 10 keV cutoff, the
 *                 remaining energy is deposited locally; dose and its statistical uncertainty are
 *                 scored per voxel, maps have the size of the phantom.
 *   PAPER.md:L71-75 (Eq. 1)  dose rate = D / N_evts x A(t_s).
 *   PAPER.md:L91-96 (Eq. 2,3) organ mean dose = unweighted mean over the organ's voxels; organ
 *                 uncertainty = RMS of the voxel uncertainties.
 * Readings where the paper is silent or BASELINE.json's north_star binds: secondary
 * electrons are deposited locally; uncertainty by the batch method; Woodcock delta tracking; optional
 * Rayleigh scattering; optional constant positron kinetic energy deposited in the decay voxel;
 * Philox4x32-10 keyed by (seed, history index).
 *
 * Conventions
 *   - Every function returns an anm_status (0 = ok, negative = error); nothing throws or exits.
 *     anm_last_error(ctx) returns a ctx-owned, NUL-terminated message valid until the next call on ctx.
 *   - Volumes are dense arrays of nx*ny*nz elements, linear index = ix + nx*(iy + ny*iz); voxel (ix,iy,iz)
 *     spans [ix*dx,(ix+1)*dx) x ... in mm from the grid corner (0,0,0).  A point exactly on a face belongs
 *     to the upper voxel; a photon is outside (killed, energy counted as escaped) iff a coordinate is < 0
 *     or >= the grid length.
 *   - `on_device` = 0: the pointer is host memory (borrowed for the duration of the call, copied);
 *     `on_device` = 1: it is a CUDA device pointer on the ctx's device (e.g. torch.Tensor.data_ptr()),
 *     read / written on the ctx stream.  The caller owns every buffer it passes in or receives into.
 *   - The ctx owns all device memory it allocates and frees it in anm_destroy (the blocks come from the device's
 *     default stream-ordered memory pool, whose release threshold anm_create raises so that they stay cached in the
 *     process -- the one process-wide setting the library touches).  A ctx is not thread-safe;
 *     separate ctxs are independent.  There is no global state, no CPU fallback and no other backend:
 *     every call that needs the GPU fails with ANM_E_CUDA when there is none.
 *   - Units: mm at this interface for lengths, MeV for energies, g/cm^3, cm^2/g, Gy, Bq.
 */
#ifndef ANM_H_
#define ANM_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct anm_ctx anm_ctx;

typedef enum {
    ANM_OK = 0,
    ANM_E_ARG = -1,          /* invalid argument (range, NaN, size mismatch, N % n_batches != 0, ...) */
    ANM_E_STATE = -2,        /* call order: something required has not been set yet                   */
    ANM_E_CUDA = -3,         /* a CUDA call failed; the CUDA error string is in anm_last_error        */
    ANM_E_NOMEM = -4,        /* host or device allocation failed                                      */
    ANM_E_UNSUPPORTED = -5   /* valid request this build does not implement                           */
} anm_status;

#define ANM_MAX_MATERIALS 8
#define ANM_MAX_ORGANS 255

/* Photon interaction data (set once; copied).  All tables are sampled on a grid uniform in ln(E/MeV):
 * lnE_k = lnE_min + k*dlnE, k = 0..n_energy-1, and are read by linear interpolation in ln E.  The grid
 * must cover [photon_cutoff_MeV, 0.51099895 MeV].
 *   mu_pe, mu_compton, mu_rayleigh : [n_materials][n_energy] mass attenuation coefficients, cm^2/g (> 0)
 *   ray_x2  : [n_x2]  increasing momentum-transfer grid x^2 (Angstrom^-2), ray_x2[0] = 0, last >= (E_max/hc)^2
 *   ray_cum : [n_materials][n_x2]  integral_0^{x^2} F_m^2 dt (any positive scale), non-decreasing;
 *             the Rayleigh angle is sampled from this piecewise-linear cumulative restricted to
 *             [0, (E/hc)^2], cos(theta) = 1 - 2 x^2 / (E/hc)^2, accepted with probability (1+cos^2)/2. */
typedef struct {
    int32_t n_materials;      /* 1..ANM_MAX_MATERIALS */
    int32_t n_energy;         /* 2..1024 */
    double lnE_min, dlnE;
    const float* mu_pe;
    const float* mu_compton;
    const float* mu_rayleigh;
    int32_t n_x2;             /* 2..1024 */
    int32_t reserved0;
    const float* ray_x2;
    const float* ray_cum;
} anm_tables;

typedef struct {
    int32_t n_batches;          /* >= 2; n_decays must be a multiple (batch-method uncertainty)        */
    int32_t photons_per_decay;  /* 2 = annihilation pair; 1 = single photon per history  */
    int32_t rayleigh_on;        /* 0 | 1                                                                */
    int32_t zero_air_dose;      /* 1: dose getters return 0 in voxels of material 0     */
    double photon_cutoff_MeV;   /* 0.010                                                  */
    double positron_ke_MeV;     /* 0, or e.g. 0.2498: deposited in the decay voxel                      */
    int32_t schedule;           /* 0 auto, 1 history-based persistent lanes, 2 event-based warp pool
                                   (regenerate in place, compact by event type); same histories either way */
    int32_t collect_stats;      /* 1: fill the counters and escaped energy of anm_stats (slower)         */
    int32_t warp_aggregate;     /* deposits of the lanes of a warp that hit the same voxel in one trip are merged
                                   (__match_any_sync) into one atomic.  Pays only where deposits pile onto few voxels
                                   (DESIGN.md §5.1 has the measurement): 0 auto = on iff positron energy is deposited and
                                   the source is a point or fewer than 1024 active voxels, and tally is not 2 (the tile-binned
                                   tally was asked for: it wins over the automatic choice); 1 on; 2 off.  Same tallies up
                                   to fp32 atomic order.  1 with electron_transport or uncertainty = 1: ANM_E_UNSUPPORTED */
    int32_t hull_majorant;      /* 0 auto / 1 on: a photon that has left the bounding box of the dense voxels on a
                                   straight line (it cannot re-enter a convex box) flies against the majorant of
                                   the low-density margin outside the box until it scatters; 2 off            */
    uint64_t history_offset;    /* index of the first history: anm_run simulates offset .. offset+n_decays-1
                                   (multi-GPU sharding of one logical run by whole batches); default 0      */
    int32_t electron_transport; /* 0: secondary electrons deposited where they are set free (north_star);
                                   1: Compton / photo-electrons above the electron cutoff are transported
                                   (needs anm_set_electron_tables; schedule 0 or 2 only)      */
    int32_t uncertainty;        /* 0: batch method (north_star; reading C1);
                                   1: history by history, the paper's estimator (Walters et al. 2002):
                                      one decay = one history, X_h = the energy it leaves in a voxel,
                                      s^2 of the mean = (sum X_h^2 / N - (sum X_h / N)^2) / (N - 1).  anm_get_uncertainty
                                      and the organs' Eq. 3 value then use it; the organ sigma_mean stays the batch
                                      one.  Schedule 0 or 2.  With electron_transport the
                                      electrons are walked inside the events (their deposits belong to the decay).
                                      Limits of this mode: at most 2^26 decays per launch (ANM_E_UNSUPPORTED beyond); a
                                      decay with more than 63 deposits is merged early (anm_stats.n_hbh_overflow); the sum
                                      of X_h^2 is ONE fp32 volume accumulated over the whole run, so a voxel that receives
                                      more than ~1e7 similar contributions (a point source with positron energy at 1e8
                                      decays; not a patient activity map) stops resolving further ones and reports
                                      sigma = 0 there -- use the batch method for such sources.                       */
    int32_t batch_pipeline;     /* launch pipeline over batch groups: 0 auto (2 sets of tallies when a launch covers more
                                   than one batch, see batches_per_launch; 3 when it covers one), 1 serial (one launch at
                                   a time on the ctx stream; per-launch ms_transport / ms_fold), 2 | 3: that many sets of
                                   batch tallies and internal streams, so that the CTAs of launch g+1 take over the SMs as
                                   those of launch g drain; never more than there are launches; the same histories and
                                   tallies; then ms_transport covers the whole pipeline (folds inside it) and ms_fold is 0. */
    int32_t tally;              /* how deposits reach the per-batch tally: 1 = one fp32 atomic (RED) per
                                   deposit into the batch volume; 2 = tile-binned: a deposit is appended as an 8-byte record
                                   {voxel, energy} to the list of the voxel's tile (2^14 consecutive voxels; position from
                                   one atomic on the tile's counter, shared by the lanes of a warp that hit the same
                                   tile) and the per-batch fold sums each tile's list in shared memory -- streaming HBM
                                   traffic instead of random read-modify-writes once the volume no longer fits the L2.
                                   The first batch of a run counts the deposits per tile (it runs with direct atomics)
                                   and sizes the lists; a deposit that finds its list full takes the direct path
                                   (anm_stats.n_tally_overflow), so the result never depends on the sizing.  0 auto = 1:
                                   measured on one B200 the binned path gains 3 % on BASELINE.json cfg4 (630 MB volumes)
                                   and loses on cfg3 (the tile counters' same-address atomics bound it).
                                   2 needs the event-pool schedule, the batch estimator, local electrons and no warp
                                   aggregation (else ANM_E_UNSUPPORTED).  Same tallies up to fp32 summation order.
                                   Test hook: the environment variable ANM_TALLY_CAPACITY=<n> fixes every list at n
                                   records (forces the overflow path).                                              */
    int32_t batches_per_launch; /* batch groups: one transport launch covers this many consecutive batches, each with its own
                                   tally volume (deposits are batch-tagged), followed by their folds -- the fixed cost of a
                                   launch (its last decays draining, ~0.25 ms) is paid n_batches / G times instead of
                                   n_batches times.  0 auto: as many as keep the tallies in flight within 4 GiB (at most
                                   256, and at most 0xF0000000 histories per launch, which keeps the launch's 32-bit history counter
                                   from wrapping); 1..256: at most that many.  Always 1 with
                                   schedule 1 or tally = 2.  Same histories, same per-batch tallies.
                                   The ctx then owns pipeline depth x G tally volumes (anm_stats.batches_per_launch = G). */
    int32_t texel_bits;         /* width of the (material, density) texel the Woodcock flight reads at random: 32 =
                                   material<<24 | density / 2^-20 g/cm^3 (every phantom); 16 = material<<13 | density / 2^-12,
                                   used only when it holds EXACTLY the same values -- every density of the loaded phantom on
                                   the 2^-12 grid and below 2 g/cm^3 (checked at load) -- so the histories are the same and
                                   the random-access footprint halves (reading C18; what matters when the volume
                                   exceeds the L2, BASELINE.json cfg4).  0 auto / 16: 16-bit when exact and the run uses the
                                   default event-pool kernel (no electron_transport, uncertainty = 1, tally = 2), else
                                   32-bit; 32: always 32-bit.  anm_stats.texel_bits tells which the last run read.        */
} anm_options;

/* Electron data for anm_options.electron_transport ("The cutoff energies for
 * photons and electrons are set to 10 keV and 200 keV"; reading C28): continuous slowing down along a
 * straight line in the electron's initial direction (Compton: its momentum k - k'; photoelectric: the photon's
 * direction), no deflection, no secondaries.  range[m][k] = residual CSDA mass range ABOVE THE CUTOFF (g/cm^2) at the
 * kinetic energy t_min + k*dt (MeV): t_min IS the electron cutoff, range[m][0] = 0, strictly increasing in k, read
 * by linear interpolation and inverted as that piecewise-linear function; the grid must reach 0.51099895 MeV
 * (a photo-electron takes the whole photon energy; Compton electrons stop at the edge 2/3 * 0.511 MeV; else ANM_E_ARG).  Crossing a voxel of density rho along a chord l takes rho*l off the
 * residual range; the energy difference is deposited in the voxel; when the range runs out inside a voxel the whole
 * remaining energy (cutoff energy included, "deposited locally") goes there; an electron that leaves the grid carries
 * its energy out (counted in escaped_MeV). */
typedef struct {
    int32_t n_materials;      /* must cover the phantom's material ids */
    int32_t n_t;              /* 2..1024 */
    double t_min, dt;         /* MeV */
    const float* range;       /* [n_materials][n_t] */
} anm_electron_tables;

typedef struct {
    double mean_Gy_per_decay;          /* Eq. 2: (1/N_o) sum of voxel doses             */
    double sigma_mean;                 /* batch standard error of that mean (absolute, Gy per decay)    */
    double rms_voxel_rel_sigma;        /* Eq. 3 over the organ's voxels with dose > 0    */
    double mass_weighted_Gy_per_decay; /* organ energy / organ mass                                     */
    double mass_g;
    uint64_t n_voxels, n_voxels_nonzero;
} anm_organ;

typedef struct {
    double emitted_MeV, deposited_MeV, escaped_MeV;   /* escaped and the counters need collect_stats   */
    uint64_t n_decays, n_steps, n_real, n_pe, n_compton, n_rayleigh, n_escaped, n_cutoff;
    uint64_t n_electrons;                                  /* electrons transported (collect_stats)         */
    uint64_t n_hbh_overflow;                               /* decays whose deposit list was merged early (uncertainty = 1, collect_stats; expected 0) */
    double ms_transport, ms_fold, ms_finalize, ms_setup;   /* device time of the last anm_run / last setup */
    uint64_t n_launches;                                   /* kernels launched by the last anm_run         */
    double ms_load_ct, ms_load_pet;                        /* device time of the last anm_load_ct / anm_load_pet
                                                              resample kernels (also counted in ms_setup)   */
    uint64_t tally_binned;                                 /* 1: the last run used the tile-binned tally (anm_options.tally) */
    uint64_t n_tally_overflow;                             /* deposits that found their tile's list full and took the
                                                              direct path; the counting batch is not included        */
    /* Run-level "statistical uncertainty" ("0.47 %", L117 "1.19 %": quoted per run, definition not given;
     * DESIGN.md reading C17): RMS of the voxels' relative sigma over the NON-AIR voxels (material id != 0; PAPER.md:L119
     * sets the dose in air to zero) whose dose exceeds 10 % / 50 % of the largest non-air voxel dose, and how many voxels
     * that is.  Uses the run's estimator (batch, or history by history with uncertainty = 1); after anm_merge: of the
     * merged run. */
    double rms_rel_sigma_gt10, rms_rel_sigma_gt50;
    uint64_t n_voxels_gt10, n_voxels_gt50;
    double max_dose_Gy_per_decay;                          /* the largest non-air voxel dose                          */
    uint64_t batches_per_launch;                           /* G of the last run (anm_options.batches_per_launch)      */
    uint64_t n_fly_trips, n_compton_tries, n_rayleigh_tries; /* event trips of the event pool (collect_stats; 0 with schedule 1):
                                                              FLY events (each evaluates up to two Woodcock sub-steps from one
                                                              Philox block), Klein-Nishina tries and form-factor tries (one
                                                              block each; n_compton / n_rayleigh count the accepted ones)   */
    uint64_t texel_bits;                                   /* 16 | 32: the texels the last run read (anm_options.texel_bits) */
    uint64_t n_check_violations;                           /* library built with -DANM_BOUNDS_CHECK: indices the transport
                                                              kernels found out of range (counted, not trapped); 0 in a
                                                              normal build, and expected 0 in a checking one               */
} anm_stats;

/* HU -> (material, density) conversion curve ("Hounsfield unit (HU)-to-density conversion curve";
 * four materials "each having a density specified by the HU").  A continuous piecewise-linear density over
 * n_nodes HU nodes, one material per HU interval:
 *   density(h)  = linear interpolation of (hu[k], rho[k]); rho[0] below hu[0], rho[n_nodes-1] above the last node
 *   material(h) = material[k] for hu[k] <= h < hu[k+1]; material[0] below hu[0]; material[n_nodes-2] at and above
 *                 the last node (material[n_nodes-1] is ignored)
 * hu must increase strictly, rho in [0, 16) g/cm^3, material < ANM_MAX_MATERIALS.  hu_outside is the HU assumed
 * where the simulation grid reaches beyond the CT image (air). */
#define ANM_MAX_RAMP_NODES 16
typedef struct {
    int32_t n_nodes;          /* 2..ANM_MAX_RAMP_NODES */
    int32_t density_bits;     /* the grid the densities are rounded to (to nearest): 0 or 20 = 2^-20 g/cm^3, the 32-bit
                                 texel's (every phantom); 12 = 2^-12 g/cm^3, on which the exact 16-bit texel copy exists
                                 (anm_options.texel_bits) as long as every density is below 2 g/cm^3 -- HU < 1809 on the
                                 default ramp; otherwise the run uses the 32-bit texels as before.  The rounding error,
                                 <= 1.2e-4 g/cm^3, is a quarter of what one HU step resolves (reading C30).
                                 anm_default_hu_ramp sets 0.  Other values: ANM_E_ARG */
    double hu[ANM_MAX_RAMP_NODES];
    double rho[ANM_MAX_RAMP_NODES];
    int32_t material[ANM_MAX_RAMP_NODES];
    double hu_outside;
} anm_hu_ramp;

/* --- lifetime ---------------------------------------------------------------------------------- */
int anm_create(anm_ctx** out, int cuda_device);    /* ANM_E_CUDA if the device cannot be used          */
int anm_destroy(anm_ctx* c);                       /* frees everything the ctx allocated; NULL is ok   */
const char* anm_last_error(const anm_ctx* c);
int anm_set_stream(anm_ctx* c, void* cuda_stream); /* cudaStream_t; NULL = the default stream          */
/* How many bytes of per-batch energy tallies this ctx may keep in flight (default, and bytes = 0: 4 GiB).  Call it BEFORE
 * anm_set_grid, which allocates them: several ctxs on one device (one per rank sharing a GPU, one per worker thread)
 * each pay this amount.  A smaller budget means fewer batches per launch (anm_options.batches_per_launch = 0 follows it;
 * an explicit batches_per_launch may still ask anm_run for more), never different results; the floor is two volumes of
 * nx*ny*nz floats.  Takes effect at the next anm_set_grid.  ANM_E_ARG for a NULL ctx. */
int anm_set_tally_budget(anm_ctx* c, uint64_t bytes);

/* --- inputs (any order; set_grid first) -------------------------------------------------------- */
/* Sets the voxel grid (origin = grid corner, linear index = ix + nx*(iy + ny*iz)) and allocates the ctx's volumes: texels,
 * the run sums, and the per-batch energy tallies of the launches in flight -- two sets of as many volumes of nx*ny*nz
 * floats as fit the tally budget (4 GiB unless anm_set_tally_budget said otherwise; at least one per set, at most 256;
 * anm_options.batches_per_launch), zeroed on an internal stream while the caller goes on loading inputs.  If the device
 * cannot give that much the number of volumes per set is halved, down to one, before the call fails with ANM_E_NOMEM.  Drops the phantom, the activity map and the organ labels of a previous
 * grid; a point source is kept only if it still lies inside the new extents.  ANM_E_ARG, ANM_E_NOMEM. */
int anm_set_grid(anm_ctx* c, int nx, int ny, int nz, double dx_mm, double dy_mm, double dz_mm);
/* material[V] < n_materials (checked at run), density[V] in [0, 16) g/cm^3, stored on a 2^-20 grid. */
int anm_load_phantom(anm_ctx* c, const uint8_t* material, const float* density_g_cm3, int on_device);
/* --- image front end: the scanner's images instead of ready-made volumes ---------------
 * anm_load_ct replaces anm_load_phantom: a CT image of int16 HU on ITS OWN grid (cnx*cny*cnz voxels of
 * cdx x cdy x cdz mm, x fastest, its corner at (ox, oy, oz) mm in the simulation grid's frame) is resampled to the
 * simulation grid ("The CT images are resampled to obtain the same size as the PET images") -- the
 * value of a simulation voxel is the volume-weighted MEAN of the piecewise-constant HU image over that voxel, with
 * ramp->hu_outside wherever the voxel reaches beyond the image -- and converted to (material, density) by `ramp`
 * (NULL = anm_default_hu_ramp), densities rounded to the 2^-20 g/cm^3 texel grid, or to the 2^-12 grid on request
 * (anm_hu_ramp.density_bits = 12: the phantom can then use the 16-bit texels).  One fused kernel; fp64 weights
 * and accumulation.  ANM_E_ARG for a bad ramp or sizes; ANM_E_STATE before anm_set_grid.
 * anm_get_phantom returns the (material, density) volumes the ctx holds (after anm_load_ct or anm_load_phantom). */
int anm_default_hu_ramp(anm_hu_ramp* r);   /* air / lung / water / compact bone; numbers approximate */
int anm_load_ct(anm_ctx* c, const int16_t* hu, int cnx, int cny, int cnz, double cdx_mm, double cdy_mm, double cdz_mm,
                double ox_mm, double oy_mm, double oz_mm, const anm_hu_ramp* ramp, int on_device);
int anm_get_phantom(anm_ctx* c, uint8_t* material, float* density_g_cm3, size_t n, int on_device);
/* anm_load_pet replaces anm_load_activity: a PET image of float32 Bq/mL on its own grid (same conventions; 0 outside
 * the image) is resampled by the same volume-weighted mean and converted linearly ("linear conversion
 * of the PET value"): activity of a simulation voxel [Bq] = mean concentration x voxel volume [mL].  The decay pdf is
 * built from it as in anm_load_activity.  *total_activity_Bq (may be NULL) receives the sum = the whole-body activity
 * A(t_s) of Eq. 1 for anm_get_dose_rate; out_activity_Bq (may be NULL; n = nx*ny*nz floats, host
 * or device like the input) receives the activity volume.  ANM_E_ARG for negative / non-finite values or an image
 * that leaves the grid without activity. */
int anm_load_pet(anm_ctx* c, const float* bq_per_ml, int pnx, int pny, int pnz, double pdx_mm, double pdy_mm, double pdz_mm,
                 double ox_mm, double oy_mm, double oz_mm, int on_device, double* total_activity_Bq,
                 float* out_activity_Bq, size_t n);

/* activity[V] >= 0, finite, arbitrary units, not all zero: decay pdf = activity / sum;
 * the decay point is uniform inside the chosen voxel. */
int anm_load_activity(anm_ctx* c, const float* activity, int on_device);
/* Replaces the activity map: every decay happens at this point (BASELINE.json cfg0). */
int anm_set_point_source(anm_ctx* c, double x_mm, double y_mm, double z_mm);
/* labels[V]: 0 = none, 1..n_organs (n_organs <= ANM_MAX_ORGANS).  Optional. */
int anm_load_organs(anm_ctx* c, const uint8_t* labels, int n_organs, int on_device);
int anm_set_physics_tables(anm_ctx* c, const anm_tables* t);
int anm_set_electron_tables(anm_ctx* c, const anm_electron_tables* t);   /* host struct, copied */
int anm_set_options(anm_ctx* c, const anm_options* o);
int anm_default_options(anm_options* o);   /* 100 batches, pairs, Rayleigh on, cutoff 0.010, no positron KE */

/* --- run --------------------------------------------------------------------------------------- */
/* Simulates histories 0..n_decays-1 with Philox4x32-10 key `seed`, counter (history, block, stream), in
 * n_batches consecutive batches; replaces the previous run's tallies.  Synchronous: results are complete
 * on return.  ANM_E_STATE unless grid, phantom, tables and a source are set.  ANM_E_UNSUPPORTED when the staged
 * tables do not fit the shared memory a CTA may opt into (227 KiB on sm_100a): the event pool (schedule 0 | 2) keeps
 * 152 KiB of photon slots beside n_materials * n_energy * 12 + n_energy * 8 + (n_materials + 1) * n_x2 * 4 bytes of
 * tables (+ the electron range tables) -- e.g. 8 materials x 1024 energies do not fit; schedule 1 needs 6 KiB + tables.
 * Every call leaves cuda_device current (cudaSetDevice) on the calling thread. */
int anm_run(anm_ctx* c, uint64_t n_decays, uint64_t seed);

/* --- results of the last run (n must equal nx*ny*nz) -------------------------------------------- */
int anm_get_energy(anm_ctx* c, float* out_MeV, size_t n, int on_device);          /* sum over batches   */
int anm_get_dose(anm_ctx* c, float* out_Gy_per_decay, size_t n, int on_device);
int anm_get_dose_rate(anm_ctx* c, double total_activity_Bq, float* out_Gy_per_s, size_t n, int on_device); /* Eq. 1 */
int anm_get_uncertainty(anm_ctx* c, float* out_rel_sigma, size_t n, int on_device); /* batch sigma of the mean / mean; 0 where the mean is 0 */
int anm_get_organ_doses(anm_ctx* c, anm_organ* out, int n_organs);                  /* host array, out[k] = label k+1 */
int anm_get_stats(anm_ctx* c, anm_stats* out);    /* before a completed run: zeros except the ms_setup / ms_load_* timings */

/* --- inspection ---------------------------------------------------------------------------------
 * The decay-voxel sampler of the loaded activity map: n_entries buckets of four uint32
 * {threshold, own voxel, alias voxel, 0}; a decay picks a bucket uniformly and takes `own` iff a 32-bit uniform is
 * below `threshold`, else `alias`, so P(voxel v) = [sum over buckets owning v of threshold/2^32 + sum over buckets
 * aliasing v of (1 - threshold/2^32)] / n_entries = activity[v] / sum(activity).  out == NULL only returns the
 * count; otherwise out is a HOST array with room for capacity_entries * 4 uint32.  ANM_E_STATE without an
 * activity map (point-source mode has no table). */
int anm_get_alias_table(anm_ctx* c, uint32_t* out, size_t capacity_entries, size_t* n_entries);

/* Parity hook of the random number generator (north_star (d): Philox4x32 keyed by history index; 10 rounds, DESIGN.md
 * reading C23): out[i] = Philox4x32-10(counter = counters[4i .. 4i+3], key = (seed low 32 bits, seed high 32 bits)),
 * computed on the device by the very function the transport kernels call (round keys in the kernel parameters).
 * counters and out are HOST arrays of 4 n uint32.  Needs only a ctx. */
int anm_philox_blocks(anm_ctx* c, uint64_t seed, const uint32_t* counters, size_t n, uint32_t* out);

/* Parity hook of the electron walk: the n given electrons {x, y, z (mm), ex, ey, ez (unit vector), T (MeV)} (HOST
 * array of 7 n floats, T above the cutoff, start points inside the grid) are walked by the same device function the
 * transport kernel calls; out_MeV (HOST, nx*ny*nz floats) receives the energy each voxel got, *escaped_MeV the
 * energy carried out of the grid.  Needs grid, phantom and electron tables; leaves the run state untouched. */
int anm_trace_electrons(anm_ctx* c, const float* electrons, size_t n, float* out_MeV, size_t n_voxels, double* escaped_MeV);

/* --- roofline microbenchmarks (BASELINE.json metric "% of L2/atomic roofline") ----------
 * What this device sustains for the three things the transport kernel does, measured with hand-written kernels of the
 * same access shape (csrc/anm_peaks.cuh), best of 3 timed launches after a warm-up, CUDA events on the ctx stream:
 *   issue_gtis      1e9 thread-instructions/s of a dependency-free FFMA + LOP3 stream at full occupancy (the
 *                   denominator of the ALU / issue roofline; the loop's own overhead is not counted: a lower bound)
 *   philox_gblocks  1e9 Philox4x32-10 blocks/s, back to back (the generator the kernels call)
 *   gather_gps[k]   1e9 random 4-byte ld.global.nc per second over an array of bytes[k] (the texel fetch)
 *   red_gps[k]      1e9 random fp32 RED.ADD per second over an array of bytes[k] (the tally)
 *   mix_gps[k]      1e9 accesses per second of both together, 5 loads : 2 REDs (cfg3's sub-steps : deposits) over TWO arrays
 *                   of bytes[k], uniformly random: the two streams share the L2 and the HBM, so the separate gather and
 *                   RED fractions must not be added up.  A reference point rather than a ceiling: the transport kernel's
 *                   accesses are concentrated on the body, which fits the L2 where two whole volumes do not, and it
 *                   exceeds this rate (measured 1.36x on cfg3, 1.5x on cfg4)
 * gather_gps and red_gps are the best of a sweep over 4, 8, 16 and 32 independent accesses in flight per thread at full
 * occupancy (64 warps per SM); gather_in_flight / red_in_flight say where the best was.
 * k = 0: small_bytes (choose a size that fits the L2, e.g. cfg3's 105 MB volume), k = 1: large_bytes (one that does not,
 * e.g. cfg4's 630 MB).  Sizes are rounded down to a multiple of 4, must be >= 4096 and < 16 GiB.  Scratch memory (two
 * arrays of the size under test) is allocated for the call and released.  Needs only a ctx.  ANM_E_ARG for bad sizes, ANM_E_NOMEM / ANM_E_CUDA. */
typedef struct {
    double issue_gtis;
    double issue_sm_mhz;      /* SM clock held during the issue stream (clock64 over the launch / its duration): a pure
                                 FFMA + LOP3 stream on every SM is power-limited, so the clock drops below clocks.max.sm;
                                 issue_gtis / (SMs x 128 lanes x issue_sm_mhz) = the fraction of issue slots filled */
    double philox_gblocks;
    double gather_gps[2];
    double red_gps[2];
    uint64_t bytes[2];
    double mix_gps[2];        /* loads + REDs per second (1e9) with both in flight */
    int32_t gather_in_flight[2], red_in_flight[2];   /* the depth per thread at which the best rate was seen */
} anm_peaks;
int anm_measure_peaks(anm_ctx* c, uint64_t small_bytes, uint64_t large_bytes, anm_peaks* out);

/* --- one logical run over several GPUs ---------------------------------------
 * Histories are independent and keyed by index (Philox counter = history index), so a run of N decays in B batches
 * shards by whole batches: rank r sets anm_options.history_offset = (first batch of r) * N/B and n_batches = its own
 * batch count, and calls anm_run on its N/B * n_batches decays.  The one exchange step is the merge of the tallies:
 *
 *   anm_get_tally_buffers  returns the ctx-owned DEVICE pointers of the last run's per-voxel sum and sum of squares
 *                          over batches (over histories when uncertainty = 1: sum of X_h^2, additive as well) (n_floats = nx*ny*nz rounded up to a multiple of 4, fp32, MeV and MeV^2)
 *                          and of its organ rows (n_rows = this run's n_batches rows of 256 fp64: row[b][label] =
 *                          sum over the organ's voxels of x / (rho V_vox) in batch b).  The caller sum-all-reduces
 *                          d_sum and d_sumsq IN PLACE across ranks (NCCL over NVLink) and gathers the organ rows of
 *                          all ranks in batch order; the pointers stay valid until the next anm_run / anm_set_grid.
 *   anm_merge              recomputes A11 (finalize) on the reduced volumes for the whole run: total_decays and
 *                          total_batches are the logical run's; organ_rows_all is a HOST array [total_batches][256]
 *                          (required when organ labels are loaded, else may be NULL); summed, if not NULL, is the
 *                          caller's element-wise sum of every rank's anm_stats (counters and escaped energy).
 *                          Afterwards every anm_get_* call on this ctx returns the merged result.
 * ANM_E_STATE without a completed run; ANM_E_ARG if total_decays / total_batches differs from this run's decays per
 * batch. */
int anm_get_tally_buffers(anm_ctx* c, float** d_sum, float** d_sumsq, size_t* n_floats, double** d_organ_rows, int* n_rows);
int anm_merge(anm_ctx* c, uint64_t total_decays, int total_batches, const double* organ_rows_all, const anm_stats* summed);

/* --- per-organ summary without any allocation by the library (csrc/anm_static.cu) ----------------------------------
 * For callers that cannot let this library allocate device memory: a process whose own allocator already owns the
 * whole HBM (a PyTorch job whose caching allocator holds the card, a server working out of one fixed arena), where a
 * cudaMalloc behind its back fails or eats into the arena; and a host thread on a deadline, which must stay away
 * from cudaMalloc / cudaFree because they take driver locks and can wait for the device.  Every other call of this
 * header needs an anm_ctx, and a ctx allocates.  This one needs none: it takes tally volumes the caller already holds
 * on the device (its own, or the ones anm_get_tally_buffers returns) and computes, per organ label, what A11's
 * finalize pass computes (Eq. 3), with the same arithmetic:
 *
 *   d_out[3 o + 0]  RMS over the organ's voxels with energy of the voxel's relative sigma
 *                   sqrt((n_samples Q / S^2 - 1) / (n_samples - 1)),  S = d_sum[v], Q = d_sumsq[v]     (o = 1..n_organs)
 *   d_out[3 o + 1]  how many of the organ's voxels hold energy (S != 0), as a double
 *   d_out[3 o + 2]  the organ's energy, sum of S (MeV)
 *   d_out[0], d_out[1] = 0;  d_out[2] = sum of S over ALL n_voxels voxels (the total deposited energy)
 *
 * d_sum, d_sumsq: DEVICE, n_voxels fp32 each.  d_labels: DEVICE, n_voxels uint8, 0 = no organ, labels above
 * n_organs are ignored; may be NULL when n_organs = 0 (then only d_out[2] is of interest).  d_out: DEVICE, caller-
 * owned, 3 (n_organs + 1) fp64, overwritten.  n_samples: the batches behind the sums (or the histories, for history-
 * by-history sums), >= 2.  All pointers belong to the CURRENT device (cudaSetDevice is the caller's business); the
 * work is queued on cuda_stream (a cudaStream_t, NULL = default stream) and the call returns without waiting.
 *
 * Where the accumulators live: in an array that is part of the library image, 3 (ANM_STATIC_MAX_ORGANS + 1) fp64
 * = 6144 bytes, present on every GPU that loads libanm.so until the process ends.  n_organs above
 * ANM_STATIC_MAX_ORGANS is refused with ANM_E_ARG and a message saying so.  The call makes no cudaMalloc / cudaFree
 * and uses no routine that allocates.  The first call on a device looks up where that device keeps the array
 * (cudaGetSymbolAddress; the driver may load the module at that point): make that first call during start-up, not
 * on the deadline path, and before any stream capture begins.  Later calls only queue a memset and two kernels.
 * There is ONE such array per device and every call uses it: it is cleared at the start of each call, so results
 * never carry over, but two calls whose GPU work can overlap (different streams without an ordering between them,
 * or two host threads on the same device) race on it and both results are garbage.  Keep calls on one stream, or
 * order them with events.
 *
 * errbuf (may be NULL) receives the message of a failed call, at most errbuf_len bytes with the terminator -- there
 * is no ctx to keep it.  ANM_E_ARG: NULL pointer, n_voxels = 0, n_samples < 2, n_organs out of range;
 * ANM_E_UNSUPPORTED: device ordinal >= 64;  ANM_E_CUDA: the runtime refused a step. */
#define ANM_STATIC_MAX_ORGANS 255
int anm_organ_summary_static(const float* d_sum, const float* d_sumsq, const uint8_t* d_labels, size_t n_voxels,
                             int n_organs, double n_samples, double* d_out, void* cuda_stream,
                             char* errbuf, size_t errbuf_len);

#ifdef __cplusplus
}
#endif
#endif /* ANM_H_ */
