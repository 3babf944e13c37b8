/* include/pmc.h — C-ABI boundary of libpmc: B200-native condensed-history proton Monte Carlo.
 *
 * Hot path of arxiv 1409.8336 (Wan Chan Tseung, Ma, Beltran): proton transport through a CT voxel grid
 * with continuous energy loss + straggling, multiple Coulomb scattering, nuclear elastic scattering and
 * non-elastic collisions (intranuclear cascade + evaporation), dose tallied with batch statistical errors.
 * Citations are "PAPER.md:Lnn (§section)"; "Reading Rk" refers to DESIGN.md.
 *
 * Conventions
 *   - plain C types only; every pointer argument says whether it is HOST or DEVICE memory;
 *   - all calls return 0 (PMC_OK) or a negative pmc_status; the message is available from pmc_last_error();
 *   - the context owns its internal device scratch (particle queues, batch tallies, tables);
 *   - caller-owned device arrays (HU grid, dose, sigma, secondaries) are never freed by the library;
 *   - every call is synchronous on return (the context's stream is synchronised), so CUDA errors and queue
 *     overflows surface as the return code; nothing is ever silently dropped;
 *   - there is NO CPU fallback: without a CUDA device pmc_create() fails with PMC_E_CUDA.
 *   - call order: pmc_create -> pmc_load_physics_tables -> pmc_set_hu_materials -> pmc_load_ct -> pmc_simulate;
 *     pmc_nonelastic needs only the physics tables.
 */
#ifndef PMC_H
#define PMC_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define PMC_MAX_ELEM 8

typedef enum {
  PMC_OK = 0,
  PMC_E_INVALID_ARG = -1,
  PMC_E_STATE = -2,        /* call order violated */
  PMC_E_CAPACITY = -3,     /* an output or internal queue is too small; nothing was truncated silently */
  PMC_E_CUDA = -4,
  PMC_E_UNSUPPORTED = -5
} pmc_status;

/* Physics input tables (HOST pointers, copied at call time).  The paper reads these from Geant4.9.6p2:
 * dE/dx and CSDA range tables for water, air and titanium with pre-computed cubic-spline second derivatives
 * (§II.A.2), non-elastic (L75 §II.A.4) and elastic (L83 §II.A.5) cross-section tables, and the
 * evaporation model's parameters (L79 ref [21]).  Layout: all 2-D arrays are row-major [row][column].
 * The kinetic-energy grid is log-uniform: E_i = e_min * (e_max/e_min)^(i/(n_e-1)). */
typedef struct pmc_tables {
  int32_t n_e; double e_min, e_max;            /* MeV */
  int32_t n_sr;                                 /* stopping/range media: 0 water, 1 air, 2 titanium */
  const double *stop_mass;                      /* [n_sr][n_e] MeV cm2/g (informational; the path uses ranges) */
  const double *ln_range, *ln_range_d2;         /* [n_sr][n_e] ln R(g/cm2) at the knots ln E_i, and spline y'' */
  int32_t n_r;
  const double *ln_r_lo, *ln_r_hi;              /* [n_sr] abscissa range of the inverse table, ln(g/cm2) */
  const double *ln_energy, *ln_energy_d2;       /* [n_sr][n_r] ln E on a uniform ln R grid, and spline y'' */
  int32_t n_elem; const int32_t *elem_z, *elem_a;   /* one isotope per element (Reading R5) */
  const double *sigma_ne_mb, *sigma_el_mb;      /* [n_elem][n_e] millibarn, linear in ln E between knots */
  int32_t mass_zdim, mass_adim;
  const double *nuclear_mass;                   /* [zdim][adim] ground-state nuclear masses, MeV; 0 = no such nuclide */
  const double *evap_k, *evap_c;                /* [6][zdim] Dostrovsky k_j, c_j vs daughter Z; j = n,p,d,t,3He,alpha */
  double e_cut;                                 /* 0.1 MeV */
  double highland_factor;                       /* 1.07 */
  double kappa_gauss;                           /* Reading R4: Vavilov kappa above which straggling is Gaussian */
  double s_max_wet_cm;                          /* Reading R3.2: step cap in g/cm2 of the table medium; <=0: none */
  int32_t n_batches;                            /* 10 */
  /* Full Moliere option (Reading R12; may be 0/NULL if "mcs_model" stays 0): cumulative Moliere
   * functions C_k[m] = int_0^{m mol_dtheta} x f^(k)(x) dx, k = 0, 1, 2, on a uniform grid of the reduced angle x */
  int32_t mol_n; double mol_dtheta;
  const double *mol_c0, *mol_c1, *mol_c2;       /* [mol_n] */
} pmc_tables;

/* One HU bin of the HU -> material conversion (§II.A.1; Eq.1/Eq.2; L59). */
typedef struct pmc_hu_bin {
  int32_t hu_lo, hu_hi;          /* HU in [hu_lo, hu_hi); bins sorted and contiguous; HU outside is clamped */
  double rho_lo, rho_hi;         /* g/cm3 at hu_lo / hu_hi, linear in between */
  double w[PMC_MAX_ELEM];        /* mass fractions over the element list of pmc_tables (sum 1 within 1e-6) */
  double f_m;                    /* Eq.1/Eq.2 water-scaling factor (used when table_id == 0) */
  double x0_gcm2;                /* radiation length */
  int32_t table_id;              /* 0: water table scaled by Eq.1/Eq.2; k>0: own stopping/range table k, unscaled */
} pmc_hu_bin;

/* One scanned-beam spot (§II.A.6 restated as a parametric Gaussian spot, Reading R2).
 * 13 doubles.  The transverse axes are e_x = unit(a x dir), e_y = dir x e_x with a = (0,1,0) if |dir_z| >= 0.9
 * else (0,0,1). */
typedef struct pmc_spot {
  double pos_cm[3];              /* spot centre on the source plane, same frame as the CT origin */
  double dir[3];                 /* central axis (normalised by the library) */
  double e_mev, sigma_e_mev;
  double sigma_x_cm, sigma_y_cm;
  double div_x_rad, div_y_rad;
  double weight;                 /* relative number of histories */
} pmc_spot;

/* One product of a non-elastic collision, 24 bytes. */
typedef struct pmc_secondary {
  int16_t Z, A;                  /* n=(0,1) p=(1,1) d=(1,2) t=(1,3) 3He=(2,3) alpha=(2,4); residual=(Z_r,A_r) */
  uint8_t origin;                /* 0 intranuclear cascade, 1 evaporation, 2 final residual nucleus */
  uint8_t pad[3];
  float ke_mev;
  float dir[3];                  /* unit vector; the incident proton travels along +z */
} pmc_secondary;

typedef struct pmc_counters {    /* totals of the last pmc_simulate / pmc_nonelastic call */
  uint64_t n_steps, n_elastic, n_nonelastic, n_secondary_protons, n_missed, n_inc_tries, n_generations;
  /* energy ledger, MeV: e_source = all the sinks below, up to fp32 rounding */
  double e_source, e_deposit, e_escape, e_neutron, e_gamma, e_q, e_air;
  uint64_t n_zab_violations;     /* events whose charge or baryon number failed to balance (must be 0) */
  /* Reading R6.8 bookkeeping of the cascade: attempts abandoned by the 1024-step guard, attempts abandoned because the
   * fixed capacities were reached (16 waiting or 16 outgoing nucleons), and the deepest stack / most outgoing nucleons seen */
  uint64_t n_inc_guard_trips, n_inc_cap_trips, inc_max_stack, inc_max_out;
  uint64_t n_host_waits;         /* times the scheduler waited for the device to learn a queue size (one per sub-group if <= 6 generations) */
} pmc_counters;

typedef struct pmc_timing {      /* CUDA-event time (ms) per kernel class over the last pmc_simulate call */
  float total_ms, sampler_ms, transport_ms, elastic_ms, inc_ms, evaporation_ms, statistics_ms;
  uint32_t launches_total, launches_transport;
} pmc_timing;

typedef struct pmc_ctx pmc_ctx;

/* Create a context on CUDA device `device`.  `cuda_stream` is a cudaStream_t owned by the caller (NULL = the
 * legacy default stream); all kernels of this context are launched on it. */
int  pmc_create(pmc_ctx **out, int device, void *cuda_stream);
/* The same with the caller's device allocator ("so PyTorch's allocator owns the memory"): every device
 * buffer of the context - tables, particle queues (6 x 48 B x 1.25 x sub-group), per-batch tallies (4 B x n_batches x
 * voxels), scratch - is obtained from alloc_fn(bytes, user) (a DEVICE pointer on `device`, 256-byte aligned, or NULL on
 * failure -> PMC_E_CUDA from the call that needed it) and returned with free_fn(ptr, user); both are called from the
 * thread that calls into the library, never from a CUDA callback.  Both NULL = cudaMalloc / cudaFree (pmc_create). */
typedef void *(*pmc_alloc_fn)(size_t bytes, void *user);
typedef void (*pmc_free_fn)(void *ptr, void *user);
int  pmc_create_with_allocator(pmc_ctx **out, int device, void *cuda_stream, pmc_alloc_fn alloc_fn, pmc_free_fn free_fn,
                               void *user);
void pmc_destroy(pmc_ctx *ctx);

/* load the physics tables (HOST, copied).  Builds the device tables and the
 * 15-shell nucleus models (L77) for every element with A > 1.
 * Errors: null pointers, sizes out of range, non-monotone range table, element missing from the mass table, non-zero
 * sigma_ne_mb for an element with A < 2 (hydrogen has no non-elastic channel below 250 MeV). */
int  pmc_load_physics_tables(pmc_ctx *ctx, const pmc_tables *tables_host);

/* HU -> density + composition (HOST array, copied).  Needs the physics tables. */
int  pmc_set_hu_materials(pmc_ctx *ctx, const pmc_hu_bin *bins_host, int nbins);

/* PAPER.md:L144 "CT geometry in global memory".  hu_dev: DEVICE pointer to nx*ny*nz int16 HU values, x fastest,
 * then y, then z; BORROWED until the next pmc_load_ct / pmc_load_ct_host / pmc_destroy.  Voxel sizes in cm; origin_cm (HOST, 3 doubles,
 * may be NULL = 0) is the position of the grid's lower corner in the frame of pmc_spot.pos_cm.
 * Errors: null pointer, non-positive sizes, nx*ny*nz >= 2^31. */
int  pmc_load_ct(pmc_ctx *ctx, const int16_t *hu_dev, int nx, int ny, int nz,
                 double dx_cm, double dy_cm, double dz_cm, const double *origin_cm);
/* Same with a HOST HU array: copied to a device buffer owned by the context (end-to-end path). */
int  pmc_load_ct_host(pmc_ctx *ctx, const int16_t *hu_host, int nx, int ny, int nz,
                      double dx_cm, double dy_cm, double dz_cm, const double *origin_cm);

/* Options: "straggling" "mcs" "elastic" "nonelastic" (0/1), "mcs_model" (0 = Highland x 1.07, the paper's choice;
 * 1 = full Moliere theory, needs the mol_* tables), "s_max_wet_cm", "n_batches",
 * "chunk_histories" (histories per sub-group), "history_offset" (first history id, for sharding
 * a run over several GPUs), "dose_aggregate" (0/1, default 0: merge the lanes of a warp that score into the same voxel before the atomic), "score_letd" (0/1, see pmc_get_letd),
 * "dose_scoring" (0/1, default 1; 0 is for measurement only: the step kernel skips its dose atomics, which bounds what any
 * other scoring scheme could gain - profiles/r02_c1_atomics.md),
 * "profile" (0/1, default 1: a CUDA-event pair is recorded on the context's stream around every kernel launch and
 * resolved into pmc_timing at the end of the call; no extra synchronisation). */
int  pmc_set_option(pmc_ctx *ctx, const char *key, double value);

/* PAPER.md:L134-138 (Fig 2): simulate n_histories primaries drawn from the spot list (HOST, nspots entries),
 * in n_batches groups; history h uses the Philox4x32-10 stream keyed (seed, h).  dose_dev / sigma_dev: DEVICE
 * arrays of nx*ny*nz float, overwritten: mean dose in Gy per primary history and its standard error from the
 * batch-to-batch scatter (Reading R8).  n_batches <= n_histories < 2^32 per call (a batch needs a history, L134): a
 * run of fewer histories than the default 10 batches is refused with PMC_E_INVALID_ARG; lower option "n_batches" (>= 2)
 * first.
 * Errors: PMC_E_STATE (tables/materials/CT missing), PMC_E_CUDA, PMC_E_CAPACITY (particle queue overflow).  Overflow is
 * not looked for generation by generation: a kernel that cannot append to a full queue sets a flag on the device and
 * drops the particle, the scheduler keeps enqueuing, and the flag is read with the counters once the call's work has
 * drained.  A call that returns PMC_E_CAPACITY has therefore done all its work, and its dose, sigma, LET_d and dose
 * influence are NOT valid (particles are missing): lower "chunk_histories" and call again. */
int  pmc_simulate(pmc_ctx *ctx, const pmc_spot *spots_host, int nspots, uint64_t n_histories, uint64_t seed,
                  float *dose_dev, float *sigma_dev);
/* Same with HOST output arrays (device -> host copies included; end-to-end path). */
int  pmc_simulate_host(pmc_ctx *ctx, const pmc_spot *spots_host, int nspots, uint64_t n_histories, uint64_t seed,
                       float *dose_host, float *sigma_host);

/* PAPER.md:L75-79, Table I: n standalone non-elastic collisions of a proton of kinetic energy e_mev (along +z)
 * with nucleus (Z,A): intranuclear cascade then evaporation.  out_dev: DEVICE array of `capacity` records,
 * grouped by event; event_offsets_dev: DEVICE array of n+1 uint32 (CSR); *n_out_host (HOST) = records needed.
 * The last record of each event is the final residual nucleus (origin 2).  Event i uses the Philox stream
 * (seed, i).  Errors: PMC_E_CAPACITY if capacity < *n_out_host (nothing valid is written beyond capacity),
 * PMC_E_UNSUPPORTED if (Z,A) or its neighbours are not in the mass table. */
int  pmc_nonelastic(pmc_ctx *ctx, int Z, int A, double e_mev, uint64_t n, uint64_t seed,
                    pmc_secondary *out_dev, uint64_t capacity, uint32_t *event_offsets_dev, uint64_t *n_out_host);

/* PAPER.md:L270 ("MC-based IMPT optimisation" needs the dose of every spot separately; Reading R11):
 * per-spot dose influence on a list of region-of-interest voxels.  roi_voxels_host: HOST array of n_roi distinct linear
 * voxel indices (x fastest) of the loaded CT, copied; dij_dev: DEVICE array of dij_capacity floats, caller-owned and
 * borrowed until the next pmc_set_dose_influence / pmc_load_ct / pmc_destroy.  Every following pmc_simulate call also
 * overwrites dij_dev[spot * n_roi + k] with the dose (Gy per primary history of the call) that the histories of that
 * spot, with all their secondaries and local deposits, give to voxel roi_voxels[k]; the rows add up to the dose in
 * that voxel (exactly so when n_batches divides n_histories).  n_roi = 0 switches it off.
 * Errors: PMC_E_STATE (no CT), PMC_E_INVALID_ARG (index out of range or repeated, null pointers); pmc_simulate returns
 * PMC_E_CAPACITY if nspots * n_roi exceeds dij_capacity. */
int  pmc_set_dose_influence(pmc_ctx *ctx, const int32_t *roi_voxels_host, int n_roi, float *dij_dev, uint64_t dij_capacity);

/* PAPER.md:L282 (Fig 9; Reading R9): dose-averaged LET scored "simultaneously" with the dose.  With option
 * "score_letd" = 1, pmc_simulate also tallies, for every step of every proton (primaries and secondaries; heavy
 * recoils and fragments do not enter, L282), e x LET and e per voxel, where e is the energy the step deposits and LET
 * the range table's mean energy loss over the step divided by the step length.  pmc_get_letd writes
 * sum(e x LET) / sum(e) in keV/um (0 where no proton step deposited energy) into letd_dev: DEVICE array of nx*ny*nz
 * float, caller-owned.  Errors: PMC_E_STATE if the last pmc_simulate did not score LET_d. */
int  pmc_get_letd(pmc_ctx *ctx, float *letd_dev);

/* PAPER.md:L166 ("3D gamma index ... 2 %/2 mm ... also computed on the GPU", ref [34]; Reading R10): gamma index of
 * the evaluated dose grid against the reference grid, both DEVICE arrays of nx*ny*nz float (x fastest), voxel sizes
 * in cm.  For every reference voxel r with D_ref(r) >= low_dose_frac * max(D_ref):
 *   gamma(r) = min over evaluated voxel centres r' with |r' - r| <= search_cm of
 *              sqrt(|r' - r|^2 / dta_cm^2 + (D_eval(r') - D_ref(r))^2 / (dd_frac * max(D_ref))^2)
 * (global dose criterion, no sub-voxel interpolation); other voxels get -1.  search_cm <= 0 selects 2 * dta_cm.
 * gamma_dev: DEVICE, nx*ny*nz float, caller-owned, overwritten.  pass_rate_host (HOST, may be NULL): fraction of the
 * evaluated voxels with gamma <= 1 (1 if none is evaluated).  Needs no tables, materials or CT.
 * Errors: PMC_E_INVALID_ARG (null pointers, non-positive sizes or criteria), PMC_E_UNSUPPORTED (nz > 65535, search
 * sphere of more than 4e6 voxels or reaching more than 32767 voxels along an axis). */
int  pmc_gamma_index(pmc_ctx *ctx, const float *ref_dev, const float *eval_dev, int nx, int ny, int nz,
                     double dx_cm, double dy_cm, double dz_cm, double dd_frac, double dta_cm, double low_dose_frac,
                     double search_cm, float *gamma_dev, double *pass_rate_host);

/* The same gamma index for callers that must not allocate device memory.  pmc_gamma_index obtains its working memory
 * (the offsets of the search sphere, two voxel counts, the maximum of the reference grid) from cudaMalloc or from the
 * context's allocator, on first use and again whenever the search sphere grows.  That rules it out for a dose-comparison
 * loop that shares the GPU with a framework whose pool already owns all of the device memory (the allocation fails), for
 * one with a latency budget (cudaMalloc and cudaFree may wait for everything else running on the device), and for
 * services that allow no allocation once they are up.  pmc_gamma_index_static takes the same arguments, gives the same
 * gamma_dev and *pass_rate_host, and calls no cudaMalloc, no cudaFree, no context allocator and no other allocating
 * routine: its working memory is one fixed array of PMC_GAMMA_STATIC_SCRATCH_BYTES inside the library image, which every
 * GPU that loads libpmc holds until the process exits, used or not.  Inputs and outputs stay the caller's.
 *   Limit: the search sphere may hold at most PMC_GAMMA_STATIC_MAX_OFFSETS voxel centres, i.e. about
 * (4 pi / 3) search_cm^3 / (dx dy dz) <= 8192 (2 mm DTA with the default 4 mm search radius on 1 mm voxels needs 257,
 * on 0.5 mm voxels 2109).  Beyond it the call returns PMC_E_CAPACITY with a message that names the limit and writes nothing.
 *   First call on a device: it looks up the device address of the array (once per device, with that device current)
 *   before it launches anything, so make that first call outside any stream capture.
 *   Sharing: there is one array per GPU and every call uses it, so it still holds the previous call's offsets and
 * counts when the next one starts; each call clears the counts and the maximum on the stream before its first kernel
 * and overwrites as much of the offset list as it reads.  Two calls in flight on one GPU at the same time would
 * corrupt each other's list and counts.  Within a process the entry point rules that out itself: it holds a lock from
 * its first enqueue until its stream has drained, which serialises calls from all threads and contexts (so it is
 * synchronous on return, like every call here).  Do not let anything else write the array.
 * Errors: as pmc_gamma_index, plus PMC_E_CAPACITY (above) and PMC_E_UNSUPPORTED for a device ordinal above 63. */
#define PMC_GAMMA_STATIC_MAX_OFFSETS 8192
#define PMC_GAMMA_STATIC_SCRATCH_BYTES (256 + 12 * PMC_GAMMA_STATIC_MAX_OFFSETS)
int  pmc_gamma_index_static(pmc_ctx *ctx, const float *ref_dev, const float *eval_dev, int nx, int ny, int nz,
                            double dx_cm, double dy_cm, double dz_cm, double dd_frac, double dta_cm, double low_dose_frac,
                            double search_cm, float *gamma_dev, double *pass_rate_host);

int  pmc_get_counters(pmc_ctx *ctx, pmc_counters *out_host);
int  pmc_get_timing(pmc_ctx *ctx, pmc_timing *out_host);
const char *pmc_last_error(pmc_ctx *ctx);     /* owned by ctx, valid until the next call on ctx */

/* ---- sub-step entry points (device implementations of single steps of the path, used by the parity tests) ---- */
/* Philox4x32-10 (north_star): in_dev [n][6] = ctr0..3,key0,key1 ; out_dev [n][4]. */
int  pmc_philox4x32_10(pmc_ctx *ctx, const uint32_t *in_dev, uint64_t n, uint32_t *out_dev);
/* CSDA range R(E) (g/cm2) of table `table` and its inverse; e_dev/r_dev DEVICE float[n]. */
int  pmc_range_of_energy(pmc_ctx *ctx, int table, const float *e_dev, uint64_t n, float *r_dev);
int  pmc_energy_of_range(pmc_ctx *ctx, int table, const float *r_dev, uint64_t n, float *e_dev);
/* The same two functions through the step kernel's own look-up: tables staged in shared memory,
 * knot index from log2(E), interleaved spline knots, for HU bin `hu_bin` (index into the array given to
 * pmc_set_hu_materials; its table_id selects the table).  Needs the materials.  Ranges are g/cm2 of the table medium,
 * i.e. before the f_m scaling of Eq.1/Eq.2.  Errors: PMC_E_STATE (no tables or materials), PMC_E_INVALID_ARG (bin). */
int  pmc_step_range_of_energy(pmc_ctx *ctx, int hu_bin, const float *e_dev, uint64_t n, float *r_dev);
int  pmc_step_energy_of_range(pmc_ctx *ctx, int hu_bin, const float *r_dev, uint64_t n, float *e_dev);
/* n straggled losses for a step with mean loss mean_loss, mass thickness rhoL (g/cm2), <Z/A>. */
int  pmc_straggle(pmc_ctx *ctx, double e_mev, double mean_loss, double rhoL_gcm2, double z_over_a,
                  uint64_t n, uint64_t seed, float *out_dev);
/* n p-A (p-p if A==1) elastic events: out_dev [n][4] = |t| (GeV/c)^2, T_out, T_recoil,
 * opening angle (rad). */
int  pmc_elastic(pmc_ctx *ctx, int Z, int A, double t_mev, uint64_t n, uint64_t seed, float *out_dev);
/* follow n primaries of spot[0] for at most max_steps condensed steps (no secondaries);
 * out_dev [n][8] = x,y,z (cm, grid frame), u,v,w, E, path length.  A debug path: the dose of these steps goes to an
 * internal tally that is not returned, LET_d and dose influence are not scored even if switched on, the counters hold
 * n_generations = 1 and the sums of that one generation, and a queue overflow cannot occur (nothing is appended). */
int  pmc_first_steps(pmc_ctx *ctx, const pmc_spot *spot_host, uint64_t n, uint64_t seed, int max_steps,
                     float *out_dev);
#ifdef __cplusplus
}
#endif
#endif
