/*
 * fdc.h -- C-ABI boundary of the B200-native track-repeating proton dose engine.
 *
 * The hot path of Yepes, Mirkovic & Taddei, "A GPU implementation of a track-repeating algorithm
 * for proton radiotherapy dose calculations", as named by BASELINE.json:north_star:
 *   fdc_create(CT HU grid, voxel spacing, HU -> density / stopping-power / scattering-power table)
 *   fdc_load_tracks(SoA track database binned by incident energy)
 *   fdc_run(beam fields, proton count, seed) -> dose grid
 * plus the final conversion fdc_to_gy as its own call, the paper's uncertainty estimates, phase-space source,
 * gamma index and profile comparators, and -- in a section of their own at the end -- two
 * diagnostics that are not part of the method (what the last call did; a trace of where its reductions went).
 * What each call computes is defined rule by rule in DESIGN.md §3 (R1-R15); citations below are
 * PAPER.md line numbers.  Every stage runs in CUDA kernels compiled for sm_100a; there is no CPU
 * fallback (FDC_EARCH on any other device).
 *
 * Conventions: mm, MeV, g/cm^3.  The grid occupies [0,nx*sx] x [0,ny*sy] x [0,nz*sz]; voxel
 * (ix,iy,iz) has linear index ix + nx*(iy + ny*iz) (x fastest) in every array crossing this ABI.
 * All calls are asynchronous on the context's stream except where they return host data, in which
 * case they synchronise that stream before returning.  Functions return 0 or a negative FDC_E*
 * code; they never abort or throw, and leave no partial state behind on failure.
 */
#ifndef FDC_H
#define FDC_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fdc_ctx fdc_ctx;                 /* opaque; one per device */

/* Knot of the piecewise-linear HU -> material table ("scaling parameters of the step
 * length and scattering angle for all the materials"; L98 density from HU).  mass_spr / mass_scpr:
 * mass stopping-power / mass scattering-power ratio to water (R1). */
typedef struct { float hu, density_g_cc, mass_spr, mass_scpr; } fdc_knot;

/* Database of pre-computed water tracks (per step "the direction, length and energy
 * loss is stored"), SoA, binned by incident energy.  Step k: displacement (dx,dy,dz) mm, energy
 * loss dE MeV, E[k] = kinetic energy at the start of the step.  Track j owns steps
 * [track_off[j], track_off[j+1]); bin b owns tracks [bin_first[b], bin_first[b+1]) and has nominal
 * energy e_min_mev + b*e_bin_mev; bin_first[n_bins] <= n_tracks (tracks past the last bin: see
 * fdc_set_secondaries).  Requirements (else FDC_EINVAL): offsets non-decreasing and
 * consistent with n_steps / n_tracks; within a track E non-increasing; 0 <= dE < 256; step length
 * either 0 or within [1e-12, 1e6] mm; all values finite. */
typedef struct {
    const float *dx, *dy, *dz, *dE, *E;         /* n_steps each */
    uint64_t n_steps;
    const uint64_t *track_off;                  /* n_tracks + 1 */
    uint32_t n_tracks;
    const uint32_t *bin_first;                  /* n_bins + 1 */
    uint32_t n_bins;
    float e_min_mev, e_bin_mev;
} fdc_trackdb;

/* One (field, energy layer, spot) of a beam plan -- the paper's phase-space generator with fixed
 * energy and direction and a transverse position spread.  (e1, e2, dir) must be
 * orthonormal within 1e-5 with e1 x e2 = dir.  Protons start at
 * origin + (spot_u + N(0,sigma)) e1 + (spot_v + N(0,sigma)) e2 and travel along dir. */
typedef struct {
    float origin[3], e1[3], e2[3], dir[3];
    float energy_mev, spot_u_mm, spot_v_mm, sigma_mm;
    uint64_t n_protons;
} fdc_beamlet;

/* One proton of a phase-space array: where it is, where it goes, its kinetic energy. */
typedef struct {
    float pos[3];            /* mm, phantom coordinates (may lie outside the grid: R6 moves it to the entry point) */
    float dir[3];            /* unit vector within 1e-5 */
    float energy_mev;        /* > 0; must map to a loaded, non-empty energy bin (R4) */
    float reserved;          /* ignored */
} fdc_particle;

typedef struct {
    uint64_t protons;        /* protons executed */
    uint64_t proton_steps;   /* database steps begun */
    uint64_t deposits;       /* non-zero (step, voxel) shares added to the grid (R8); the kernel merges the shares
                                one proton leaves in one voxel into one atomic, so it issues fewer atomics */
    uint64_t missed;         /* never entered the grid */
    uint64_t escaped;        /* left the grid before the track ended */
    uint64_t stopped;        /* track ended inside the grid */
    uint64_t grid_sum;       /* sum of the fixed-point grid (computed by fdc_get_stats) */
    uint64_t q_replayed;     /* sum of Q over all steps from each proton's start step on */
    uint64_t q_escaped;      /* part of q_replayed not tallied because the proton escaped;
                                grid_sum + q_escaped == q_replayed exactly (R8) */
} fdc_stats;

enum {
    FDC_OK        =  0,
    FDC_EINVAL    = -1,   /* null pointer, bad size / spacing / table / frame / proton range, stride 0 */
    FDC_ENOTRACKS = -2,   /* fdc_run before fdc_load_tracks */
    FDC_ERANGE    = -3,   /* beamlet energy above the top bin, or its bin is empty */
    FDC_ENOMEM    = -4,
    FDC_ECUDA     = -5,   /* CUDA error; text via fdc_last_error */
    FDC_EARCH     = -6,   /* device is not compute capability 10.x (no fallback by design) */
    /* positive codes are warnings: the call did its work and every output is valid; fdc_last_error says what to know */
    FDC_WSEGMENTED = 1    /* fdc_uncertainty_history: the squares grid holds FDC_SQUARES_BY_HISTORY runs in which some histories
                             visited more voxels than the per-history table holds and were squared in segments, so for them
                             eq. (2)'s D_i^2 is a sum of squares of partial sums (between the per-stay and the exact tally) */
};

enum {
    FDC_RANDOM_AZIMUTH = 1u,   /* rotate each re-used track by a random azimuth about the beam (R5) */
    FDC_DOSE_TO_HOST   = 2u,   /* dose_gy is a host pointer (else device) */
    FDC_NO_SORT        = 4u,   /* debug: do not group protons by track (same result, slower) */
    FDC_NO_AGGREGATE   = 8u,   /* debug: one atomic per share, no per-voxel merging (same result) */
    FDC_TALLY_SQUARES  = 16u,  /* also tally the sum of squares (second grid; R10) */
    FDC_REALIGN_START  = 32u,  /* rotate a sub-track that starts at a step k0 > first so that step k0 points along
                                  the beam (R14); off: the track keeps the deflection it had */
    FDC_SORT_SPATIAL   = 128u, /* scheduling only (same result): group protons by where they start on the source plane
                                  instead of by the track they replay; beam plans only */
    FDC_PRIVATE_TALLY  = 512u, /* scheduling only (same result): route the reductions through a per-CTA table in shared memory
                                  that is emptied into the grid every few rounds (north_star (4)); meant to be
                                  used with FDC_SORT_SPATIAL; ignored with FDC_TALLY_SQUARES / FDC_NO_AGGREGATE */
    FDC_NO_LAT         = 256u, /* debug: run a small plan (at most one wave of thread blocks) through the same instantiation as a
                                  large one; by default it runs with the CTA-private tally of FDC_PRIVATE_TALLY in blocks sized at launch so
                                  that its warps spread evenly over the SMs (same result) */
    FDC_MAT_TILED      = 2048u,/* scheduling only (same result): the transport kernel reads the material of the voxel ahead from the
                                  library's tiled copy of the material grid (4 x 4 x 1 voxels per 32-byte sector) ... */
    FDC_MAT_LINEAR     = 4096u,/* ... or from the x-fastest one.  Default, per launch: tiled for an oblique field (second direction
                                  component >= 0.3), or if the material and energy grids together (10 bytes per voxel) exceed the
                                  device's L2 cache */
    FDC_SQUARES_BY_HISTORY = 8192u, /* implies FDC_TALLY_SQUARES; the squares tally follows eq. (2)'s definition: for
                                  every history, everything it -- its primary and its secondaries -- left in a voxel is summed before
                                  it is squared, whereas FDC_TALLY_SQUARES alone squares every uninterrupted stay in a voxel
                                  (R10).  Each thread keeps the voxels its history has visited (up to 2048) in local
                                  memory; slower */
    FDC_WARP_AGGREGATE = 1024u,/* scheduling only (same result): a small plan runs the latency-oriented instantiation that sums the
                                  shares of the lanes leaving the same voxel over the warp and sends one reduction per distinct
                                  voxel (north_star (4)), instead of the CTA-private tally; ignored for larger plans */
    FDC_DIAG_REDS      = 64u   /* diagnostics: run the instrumented instantiation of the transport kernel, which counts
                                  the 64-bit reductions it sends and records their voxel indices (fdc_trace_reds);
                                  same tallies, slower; not combinable with FDC_TALLY_SQUARES / FDC_NO_AGGREGATE */
};

/*
 * Create a context on `device` using `cuda_stream` (a cudaStream_t; NULL = default stream).
 * hu: nx*ny*nz int16 Hounsfield units, x fastest ("three dimensional array with a
 * material index for each voxel"); values are clamped to [-1024, 3071].  The array (host, or device if
 * hu_is_device_ptr) is read during this call only: the library derives its own material-index grid
 * from it before returning.  table: n_knots >= 1 knots, strictly increasing in hu, all of
 * density, mass_spr, mass_scpr > 0 (host pointer, copied).  Builds the material LUT (R1) and a
 * zeroed u64 energy grid (quantum 2^-24 MeV).
 */
int fdc_create(fdc_ctx **out, int device, void *cuda_stream,
               const int16_t *hu, int nx, int ny, int nz, float sx, float sy, float sz,
               const fdc_knot *table, int n_knots, int hu_is_device_ptr);

/* Load (replace) the track database.  The five step arrays are host or device pointers per
 * arrays_are_device_ptrs; track_off and bin_first are always host pointers.  Nothing is borrowed:
 * the library derives its own device-resident step store (unit direction, length, fixed-point
 * energy, suffix sums) before returning, so the caller may free its arrays afterwards. */
int fdc_load_tracks(fdc_ctx *ctx, const fdc_trackdb *db, int arrays_are_device_ptrs);

/*
 * Histories with several trajectories (a history holds the primary "and all secondary"
 * trajectories; L71 "selecting the trajectory"; R15).  Tracks past the last
 * energy bin (ids >= bin_first[n_bins]; fdc_load_tracks accepts them) are never drawn by R4: they can only
 * be secondaries.  For parent track j, sec_track[sec_first[j] .. sec_first[j+1]) are its secondaries and
 * sec_step[] the parent's step (counted from the parent's first step, ascending within a parent) at
 * whose END each one starts, from the parent's position and frame there, replaying all its own steps
 * under R7/R8.  A proton that joins the parent at a later step skips the earlier branches; a parent
 * that escapes before a branch step never starts that secondary.  Counters: escaped / stopped count
 * primaries; steps, deposits, q_replayed, q_escaped include the secondaries.  At most 6 secondaries
 * per parent; secondaries have none of their own.  Host arrays, copied.  n_sec = 0 removes the table;
 * fdc_load_tracks removes it too.  FDC_EINVAL on an inconsistent table, FDC_ENOTRACKS before a load.
 */
int fdc_set_secondaries(fdc_ctx *ctx, const uint32_t *sec_first /* n_tracks + 1 */, const uint32_t *sec_track,
                        const uint32_t *sec_step, uint32_t n_sec);

/*
 * Transport protons and ADD their energy deposits to the context's grid.
 * b[0..n_beamlets) (host) defines the global proton index space [0, sum n_protons); the call
 * executes indices first_proton + m*proton_stride for m in [0, n_protons), all of which must lie
 * in that space.  Proton i draws the same random numbers whatever the call that executes it
 * (Philox4x32-10 keyed by seed, counter i; R3), so run(0..N) == run(0..a) + run(a..N) bit for bit.
 * If dose_gy is not NULL it receives nx*ny*nz floats: the grid as it stands after this call
 * converted to Gy (R9) -- device memory, or host memory with FDC_DOSE_TO_HOST.
 */
int fdc_run(fdc_ctx *ctx, const fdc_beamlet *b, uint32_t n_beamlets,
            uint64_t first_proton, uint64_t n_protons, uint64_t proton_stride,
            uint64_t seed, uint32_t flags, float *dose_gy);

/*
 * The same transport started from a phase-space array instead of a beam plan ("the
 * phase space ... position, direction and energy of the incident protons"; DESIGN.md
 * R12).  Particle m (ps[m], host or device per ps_is_device_ptr; a host array is copied) is the
 * proton with random-number identity first_id + m: it draws its track (R4) and azimuth (R5) from
 * Philox(seed, first_id + m), has no lateral offset, starts at pos along dir with energy_mev, and
 * its transverse frame is fixed by dir (a = axis of the smallest |dir_a|, lowest index on ties;
 * e1 = (unit_a - dir_a dir) normalised; e2 = dir x e1).  It then behaves exactly like a one-proton
 * beamlet with that frame: ADDS to the grid, same flags, same dose_gy convention as fdc_run.
 * Energies may differ from particle to particle (each starts at the first step with E <= energy).
 * Errors: FDC_EINVAL (non-finite field, energy <= 0, |dir| != 1), FDC_ERANGE (energy bin outside the
 * database or empty); the array is validated on the device before anything is tallied.
 */
int fdc_run_phase_space(fdc_ctx *ctx, const fdc_particle *ps, uint64_t n, int ps_is_device_ptr,
                        uint64_t first_id, uint64_t seed, uint32_t flags, float *dose_gy);

/*
 * Stage 5 on its own ("At the end of the run the energy deposited in each voxel was converted to
 * absorbed dose by dividing by the mass of the voxel"; R9): the grid as it stands -> nx*ny*nz floats in
 * Gy, device memory or (is_device_ptr = 0; synchronises) host memory.  fdc_run's dose_gy argument is this call
 * appended to the transport; a multi-GPU run calls it once after the grids have been summed.
 */
int fdc_to_gy(fdc_ctx *ctx, float *dose_gy, int is_device_ptr);

/* Copy out the raw fixed-point grid (nx*ny*nz u64, quanta of 2^-24 MeV). */
int fdc_get_edep_fixed(fdc_ctx *ctx, uint64_t *grid_out, int is_device_ptr);

/* Overwrite the raw fixed-point grid, e.g. with the sum over GPUs after an integer all-reduce (the
 * paper's "absorbed dose from both threads was combined"); counters are unchanged. */
int fdc_set_edep_fixed(fdc_ctx *ctx, const uint64_t *grid_in, int is_device_ptr);

/* The context's own device arrays, BORROWED (valid until fdc_destroy; owned by the library): the u64 energy grid
 * and, if one exists (else NULL), the sum-of-squares grid -- so that the integer all-reduce over GPUs
 * can run in place on the caller's stream instead of through get / set copies.  The caller must
 * order its work against the context's stream. */
int fdc_edep_device_ptr(fdc_ctx *ctx, uint64_t **edep, uint64_t **squares /* may be NULL */);

/*
 * Sum-of-squares tally ("a second tallying array ... the sum of the squares of the
 * deposited energy", needed by eq. (2)).  fdc_run with FDC_TALLY_SQUARES adds, for every stay of
 * a proton in a voxel (from entering it to crossing out of it, or to the end of the track), the
 * square of e' = min((energy left there) >> 8, 2^32 - 1) to a second nx*ny*nz u64 grid (quanta of
 * 2^-32 MeV^2; R10).  The grid is created zeroed by the first such run and zeroed by
 * fdc_reset.  Not combinable with FDC_NO_AGGREGATE (FDC_EINVAL).  get: FDC_EINVAL before the first
 * such run; set (multi-GPU all-reduce) creates the grid if needed.
 */
int fdc_get_sq_fixed(fdc_ctx *ctx, uint64_t *grid_out, int is_device_ptr);
int fdc_set_sq_fixed(fdc_ctx *ctx, const uint64_t *grid_in, int is_device_ptr);

/*
 * History-by-history statistical uncertainty, eq. (2) (L86; sums over all N primaries),
 * from the energy grid S1 and the squares grid S2 as they stand, per voxel in f64:
 *   m = S1*2^-24/N,  m2 = S2*2^-32/N,  sigma = sqrt(max(0, (m2 - m*m)/(N - 1))),  rel = sigma/m (0 if m = 0).
 * rel_sigma (may be NULL): nx*ny*nz floats, host or device per rel_is_device_ptr.  *mean_rel: the
 * paper's "mean dose uncertainty" (L92): the average of rel over the voxels whose dose m/rho
 * exceeds half the maximum dose; *n_voxels_averaged: how many.  Synchronises.  FDC_EINVAL if
 * n_histories < 2 or no squares grid exists.  Returns FDC_WSEGMENTED (> 0, outputs valid) instead of FDC_OK when
 * FDC_SQUARES_BY_HISTORY runs since the last fdc_reset emptied a history's table early (fdc_call_info.sq_history_flushes > 0).
 */
int fdc_uncertainty_history(fdc_ctx *ctx, uint64_t n_histories, float *rel_sigma, int rel_is_device_ptr,
                            double *mean_rel, uint64_t *n_voxels_averaged);

/*
 * Batch-method uncertainty, eq. (1) (L82): batch_grids is a HOST array of n_batches
 * DEVICE pointers to u64 energy grids (nx*ny*nz, as returned by fdc_get_edep_fixed with a device
 * pointer), each from an independent run of histories_per_batch histories.  Per voxel in f64:
 *   mean = (sum_b D_b)/n,  sigma = sqrt(sum_b (D_b - mean)^2 / (n (n - 1))),  rel = sigma/mean,
 * D_b = grid_b*2^-24 MeV, the sums taken in batch order.  Outputs as fdc_uncertainty_history (the dose for the
 * half-maximum selection is mean/rho).  2 <= n_batches <= 64.
 */
int fdc_uncertainty_batch(fdc_ctx *ctx, const uint64_t *const *batch_grids, int n_batches, uint64_t histories_per_batch,
                          float *rel_sigma, int rel_is_device_ptr, double *mean_rel, uint64_t *n_voxels_averaged);

/*
 * Gamma index (Gamma(3 %, 3 mm), Low et al. 1998) of dose_eval against dose_ref,
 * both DEVICE arrays of nx*ny*nz floats (>= 0) on the context's grid.  Per reference voxel r:
 *   Gamma(r) = min over whole-voxel offsets o with |o| <= search_mm and r + o inside the grid of
 *              sqrt(|o|^2 / dist_tol_mm^2 + (D_eval(r + o) - D_ref(r))^2 / dD^2),  dD = dose_tol_frac * max(D_ref)
 * (global dose criterion, no interpolation; f64, R13).  gamma_out: DEVICE array of nx*ny*nz
 * floats or NULL.  *pass_fraction: share of the voxels with D_ref > cutoff_frac * max(D_ref) whose
 * Gamma <= 1; *n_evaluated: their number.  search_mm may cover at most 5 voxels per axis
 * (FDC_EINVAL otherwise).  Synchronises.
 */
int fdc_gamma_index(fdc_ctx *ctx, const float *dose_ref, const float *dose_eval, float dose_tol_frac, float dist_tol_mm,
                    float search_mm, float cutoff_frac, float *gamma_out, double *pass_fraction, uint64_t *n_evaluated);

/* Counters accumulated since creation / the last fdc_reset (host struct; synchronises). */
int fdc_get_stats(fdc_ctx *ctx, fdc_stats *out);

/* Zero the grid and the counters. */
int fdc_reset(fdc_ctx *ctx);

void fdc_destroy(fdc_ctx *ctx);

const char *fdc_strerror(int code);
const char *fdc_last_error(const fdc_ctx *ctx);      /* text of the last FDC_ECUDA / FDC_EINVAL */

/*
 * Profile comparators (Fig. 2-3; R16, R17).
 *
 * fdc_profile: the paper's depth and cross-field profiles, "calculated along a five voxel thick line" (L104).
 * values: DEVICE array of nx*ny*nz floats (a dose grid), or NULL for the context's own energy grid in MeV (Fig. 2
 * plots deposited energy).  The line runs along `axis` (0 = x, 1 = y, 2 = z) through the voxel whose indices on
 * the other two axes (a = the lower-numbered one, b = the other) are (fixed_a, fixed_b); it is thickened to the
 * bundle of columns |a - fixed_a| <= half_width_a, |b - fixed_b| <= half_width_b clipped to the grid (2, 2 = five
 * voxels thick; 2, 0 = a five-voxel slab), and out[k], k < n_axis, is the mean over the bundle (f64; summed b
 * outer, a inner, then divided by the number of columns).  out: n_axis doubles, host (synchronises) or device.
 * FDC_EINVAL if the line lies outside the grid.
 *
 * fdc_rms_diff: "the difference between the ... doses for each voxel ... divided by the maximum [reference] voxel
 * dose has a RMS value of 0.5 %" (L108): *rms_over_max = sqrt(mean over ALL voxels of ((eval - ref) * (1 / max
 * ref))^2), f64 per voxel, summed exactly in 128-bit fixed point (quantum 2^-64: independent of the order of the
 * additions).  Both arrays DEVICE, nx*ny*nz floats.  *max_ref (may be NULL) receives the maximum.  Synchronises.
 */
int fdc_profile(fdc_ctx *ctx, const float *values, int axis, int fixed_a, int fixed_b, int half_width_a, int half_width_b,
                double *out, int out_is_device_ptr);
int fdc_rms_diff(fdc_ctx *ctx, const float *dose_ref, const float *dose_eval, double *rms_over_max, double *max_ref);

/* ------------------------------------------------------------------------------------------------------------
 * Eq. (1) without any device allocation.
 *
 * Who this is for.  The paper's way of using the batch estimate is a loop: run a batch, evaluate eq. (1), stop
 * once the mean dose uncertainty is below the target.  A planning service that runs this
 * loop in steady state has often given every byte of device memory to its own arena at start-up (or lives inside
 * a host framework whose caching allocator has), so a cudaMalloc made on its behalf either fails or takes memory
 * the arena believes it owns; and cudaFree waits for all work on the device (cudaMalloc may too), which a loop
 * that overlaps the next batch's transport with this evaluation cannot afford.  fdc_uncertainty_batch
 * allocates its scratch lazily (a pointer table, four accumulator words, and a whole float grid when rel_sigma is a
 * host array), so such callers cannot know when it will allocate.  This call never does: it makes no cudaMalloc,
 * cudaFree or allocating library call, on any path.
 *
 * How.  Its scratch is a fixed FDC_NOALLOC_SCRATCH_BYTES (512) array that is part of the library image: every GPU
 * on which libfdc.so gets loaded holds those bytes until the process exits, whether or not this call is used.
 * Words 0-2 are the reduction accumulators (maximum dose, fixed-point sum, voxel count), the second half is the
 * table of batch-grid pointers.  Hence the limit: 2 <= n_batches <= FDC_NOALLOC_MAX_BATCHES (32; the paper uses
 * 6); more is refused with FDC_EINVAL and a message naming the limit (fdc_uncertainty_batch takes up to 64).
 *
 * Arguments and results are those of fdc_uncertainty_batch (same kernel, same arithmetic, bit-identical
 * *mean_rel, *n_voxels_averaged and rel_sigma), except that rel_sigma_dev is a DEVICE array of nx*ny*nz floats
 * or NULL: the caller owns every input and output, the library only borrows them for the call.  batch_grids is
 * a HOST array of DEVICE pointers.  Synchronises the context's stream before it returns.
 *
 * First call on a device.  The address of the array on the context's device is looked up once per device, by the
 * first call made with a context on that device (cudaGetSymbolAddress, with that device current); that call may
 * initialise the CUDA module, so make it once during set-up, before any stream capture is begun.
 *
 * Sharing.  There is ONE array per device, shared by every context and every call in the process.  A call
 * clears the accumulators it needs and overwrites the pointers it uses; it keeps nothing from call to call.
 * Two calls whose device work overlaps in time (different contexts / streams / host threads on one device)
 * race on it and both results are garbage: serialise them.  Calls on different devices do not interact.
 * ------------------------------------------------------------------------------------------------------------ */
#define FDC_NOALLOC_MAX_BATCHES 32
#define FDC_NOALLOC_SCRATCH_BYTES 512
int fdc_uncertainty_batch_noalloc(fdc_ctx *ctx, const uint64_t *const *batch_grids, int n_batches, uint64_t histories_per_batch,
                                  float *rel_sigma_dev, double *mean_rel, uint64_t *n_voxels_averaged);

/* ------------------------------------------------------------------------------------------------------------
 * Diagnostics.  NOT part of the method and not among the calls SURVEY §8(b) lists: they report what the library
 * did, for bench.py's timing split, its end-to-end byte counts and its contention-limited roofline ceiling.  The
 * roofline microbenchmarks themselves live in a separate library (csrc/bench_peaks.cu -> libfdcpeaks.so).
 * ------------------------------------------------------------------------------------------------------------ */

/* What the most recent fdc_run / fdc_run_phase_space did, together with any fdc_to_gy calls made since (their
 * kernel and copy are added to launches, ms_gy, d2h_bytes; ms_total then spans from the start of the run to the
 * end of the last conversion).  Times are device times from CUDA events on the context's stream.  Synchronises. */
typedef struct {
    float ms_total;          /* whole call on the device */
    float ms_transport;      /* transport + deposit kernels */
    float ms_sort;           /* sampling-key + grouping kernels */
    float ms_gy;             /* Gy kernel (and the device-to-host copy of the dose grid, if any) */
    uint32_t launches;       /* kernels launched by the call */
    uint32_t sq_history_flushes; /* FDC_SQUARES_BY_HISTORY runs since the last fdc_reset: histories whose table of visited voxels
                                    filled up and was emptied early (such a history is squared in segments; 0 = eq. (2) exact) */
    uint64_t h2d_bytes;      /* bytes the call copied from host memory to the device (0 when the plan was cached) */
    uint64_t d2h_bytes;      /* bytes it copied back */
    uint64_t reds_sent;      /* FDC_DIAG_REDS runs since the last fdc_reset: 64-bit reductions actually sent */
    uint64_t reds_traced;    /* of those of the last call, how many are in the trace buffer */
} fdc_call_info;
int fdc_last_call_info(fdc_ctx *ctx, fdc_call_info *out);

/* Set (or, with NULL / 0, remove) a DEVICE buffer of `capacity` uint32 that FDC_DIAG_REDS runs fill with the voxel
 * index of every reduction they send, in the order the hardware serialises the appends; each such run starts
 * again at entry 0.  Borrowed until replaced. */
int fdc_trace_reds(fdc_ctx *ctx, uint32_t *trace_dev, uint64_t capacity);

#ifdef __cplusplus
}
#endif
#endif /* FDC_H */
