/* oracle/opmc.h — C interface of the fp64 CPU ORACLE.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing in the product path (paper_1409_8336_b200/,
 * include/, csrc/) includes, links or calls this.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may use it.
 *
 * The oracle follows arxiv 1409.8336 step by step in fp64, one history at a
 * time; every place where the paper is silent is resolved by the reading listed in
 * DESIGN.md ("Readings").  It shares no code with the CUDA path: this header is NOT
 * include/pmc.h, although the five calls mirror it (host pointers everywhere).
 *
 * Parity pins (tests/test_oracle_*.py): Philox known answers; CSDA range vs direct
 * integration; Eq.1/Eq.2 identity; Highland 1.07*theta0; Fermi-Eyges hinge moments;
 * straggling cumulants; per-history energy ledger; exact Z/A conservation; Ranft
 * t-distribution; INC collision-probability closed form; evaporation spectra; Cugnon joint
 * and interior values; NN angular law vs its analytic CDF (alone and inside the cascade);
 * shell-boundary refraction/reflection vs the classical scattering angle; Pauli blocking and
 * the trapping rule; event rate 1 - exp(-Sigma L) and n_i sigma_i branching; spot
 * frequencies and divergence; cascade step-guard trip rate (tests/test_oracle_pins_nuclear.py).
 * Parity UNPINNED (comparison material missing from the container): agreement with
 * Chibani's Vavilov sampler (ref [18]), with the INC of ref [13], with Furihata's GEM
 * (ref [21]) and with any Geant4-derived table.
 */
#ifndef OPMC_H
#define OPMC_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define OPMC_MAX_ELEM 8

typedef struct {                 /* all input data */
  int32_t n_e; double e_min, e_max;            /* log-uniform kinetic-energy grid, MeV */
  int32_t n_sr;                                 /* stopping/range tables: 0 water, 1 air, 2 Ti */
  const double *stop_mass;                      /* [n_sr][n_e] MeV cm2/g */
  const double *ln_range, *ln_range_d2;         /* [n_sr][n_e] ln R(g/cm2) vs ln E knots + spline y'' */
  int32_t n_r;
  const double *ln_r_lo, *ln_r_hi;              /* [n_sr] inverse-table abscissa range (ln g/cm2) */
  const double *ln_energy, *ln_energy_d2;       /* [n_sr][n_r] ln E vs uniform ln R + spline y'' */
  int32_t n_elem; const int32_t *elem_z, *elem_a;
  const double *sigma_ne_mb, *sigma_el_mb;      /* [n_elem][n_e] */
  int32_t mass_zdim, mass_adim;
  const double *nuclear_mass;                   /* [zdim][adim] MeV, 0 = not a nuclide */
  const double *evap_k, *evap_c;                /* [6][zdim] Dostrovsky k_j, c_j vs daughter Z */
  double e_cut, highland_factor, kappa_gauss, s_max_wet_cm;
  int32_t n_batches;
  /* Moliere option (Reading R12): cumulative functions C_k[m] = int_0^{m dtheta} theta f^(k) dtheta, k = 0,1,2 */
  int32_t mol_n; double mol_dtheta; const double *mol_c0, *mol_c1, *mol_c2;
} opmc_tables;

typedef struct {                 /* PAPER.md:L49, Eq.1, Eq.2 */
  int32_t hu_lo, hu_hi;          /* HU in [hu_lo, hu_hi) */
  double rho_lo, rho_hi;         /* g/cm3 at hu_lo / hu_hi, linear in between */
  double w[OPMC_MAX_ELEM];       /* mass fractions over the tables' element list */
  double f_m;                    /* Eq.1/Eq.2 scaling factor (table_id 0 only) */
  double x0_gcm2;                /* radiation length */
  int32_t table_id;              /* 0: water table scaled by Eq.1/2; k>0: own table k, unscaled */
} opmc_hu_bin;

typedef struct {                 /* PAPER.md:L102-106 restated as a Gaussian spot */
  double pos_cm[3], dir[3];
  double e_mev, sigma_e_mev, sigma_x_cm, sigma_y_cm, div_x_rad, div_y_rad, weight;
} opmc_spot;

typedef struct {
  int16_t Z, A;                  /* n=(0,1) p=(1,1) d t 3He alpha, residual=(Zr,Ar) */
  uint8_t origin;                /* 0 INC, 1 evaporation, 2 final residual */
  uint8_t pad[3];
  float ke_mev; float dir[3];
} opmc_secondary;

typedef struct {
  uint64_t n_steps, n_draws, n_elastic, n_nonelastic, n_secondary_protons, n_missed, n_inc_tries;
  double e_source, e_deposit, e_escape, e_neutron, e_gamma, e_q, e_air;
  double max_ledger_residual;    /* max over histories of |E0 - sum of all sinks| (MeV) */
  double max_event_residual;     /* max |4-momentum imbalance| over INC/evaporation/elastic events */
  uint64_t n_zab_violations;     /* events where charge or baryon number failed to balance (must be 0) */
  /* Reading R6.8 bookkeeping: cascade attempts ended by the step guard / by the 200-nucleon stack limit, and the
     deepest stack of waiting nucleons and the largest number of outgoing nucleons seen in one attempt */
  uint64_t n_inc_guard_trips, n_inc_stack_trips, inc_max_stack, inc_max_out;
} opmc_counters;

typedef struct opmc_ctx opmc_ctx;

int  opmc_create(opmc_ctx **out);
void opmc_destroy(opmc_ctx *);
int  opmc_load_physics_tables(opmc_ctx *, const opmc_tables *);
int  opmc_set_hu_materials(opmc_ctx *, const opmc_hu_bin *bins, int nbins);
int  opmc_load_ct(opmc_ctx *, const int16_t *hu, int nx, int ny, int nz,
                  double dx, double dy, double dz, const double origin[3]);
/* keys: "straggling" "mcs" "elastic" "nonelastic" (0/1), "s_max_wet_cm", "n_batches", "threads", "score_letd", "mcs_model",
 * "inc_step_guard" (tracking steps per cascade attempt, Reading R6.8; default 1024 - changed only by the pin test of the guard) */
int  opmc_set_option(opmc_ctx *, const char *key, double value);
int  opmc_simulate(opmc_ctx *, const opmc_spot *spots, int nspots, uint64_t n_histories, uint64_t seed,
                   double *dose, double *sigma);
int  opmc_nonelastic(opmc_ctx *, int Z, int A, double e_mev, uint64_t n, uint64_t seed,
                     opmc_secondary *out, uint64_t capacity, uint32_t *event_offsets, uint64_t *n_out);
int  opmc_get_counters(opmc_ctx *, opmc_counters *);
/* PAPER.md:L270 (Reading R11): per-spot dose influence on a list of ROI voxels; see opmc.cpp. out: nspots*n_roi doubles. */
int  opmc_set_dose_influence(opmc_ctx *, const int32_t *roi_voxels, int n_roi);
int  opmc_get_dose_influence(opmc_ctx *, double *out);
/* PAPER.md:L282 (Reading R9): dose-averaged LET of the last opmc_simulate call made with option "score_letd" = 1;
 * out: nx*ny*nz doubles, keV/um, 0 where no proton step deposited energy. */
int  opmc_get_letd(opmc_ctx *, double *out);
const char *opmc_last_error(opmc_ctx *);

/* ---- hooks used only by the pin tests ---- */
void   opmc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
double opmc_test_range_gcm2(opmc_ctx *, int table, double e_mev);
double opmc_test_energy_of_range(opmc_ctx *, int table, double r_gcm2);
/* n straggled losses for a step of wet-path rho*L (g/cm2) in a medium of given <Z/A> */
int    opmc_test_straggle(opmc_ctx *, double e_mev, double mean_loss, double rhoL_gcm2, double z_over_a,
                          uint64_t n, uint64_t seed, double *out);
/* follow n primaries of spot[0] for at most max_steps condensed steps; out[n][8]=x,y,z,u,v,w,E,pathlen */
int    opmc_test_first_steps(opmc_ctx *, const opmc_spot *spot, uint64_t n, uint64_t seed, int max_steps,
                             double *out);
/* n p-A (or p-p when A==1) elastic events at kinetic energy t: out[n][4] = |t| (GeV/c)^2, T_out, T_recoil,
   opening angle between the two outgoing lab directions (rad) */
int    opmc_test_elastic(opmc_ctx *, int Z, int A, double t_mev, uint64_t n, uint64_t seed, double *out);
/* single uniform shell of radius R (fm), nucleon density rho (fm^-3, all neutrons), constant sigma (mb),
   potentials zero, Pauli off: returns fraction of entries with >= 1 collision */
double opmc_test_inc_uniform_sphere(double radius_fm, double rho_fm3, double sigma_mb, double t_mev,
                                    uint64_t n, uint64_t seed);
/* shells of nucleus (Z,A): out[15][6] = r_out, rho_p, rho_n, pF_p, EF_p, V_p ; returns r_max */
double opmc_test_nucleus(opmc_ctx *, int Z, int A, double *out);
double opmc_test_nucleus_neutron(opmc_ctx *, int Z, int A, double *out);   /* out[15][3] = pF_n, EF_n, V_n; returns B_C */
/* mean of p^2 over n sampled Fermi partners in the central shell divided by pF^2 (-> 3/5) */
double opmc_test_fermi_p2(opmc_ctx *, int Z, int A, uint64_t n, uint64_t seed);
/* evaporation of (Z,A,E*) at rest: widths[6] by quadrature; first emission of n samples restricted to
   channel_mask (bit j): out_channel[n], out_eps[n]; spectrum[6*64] = the discretised P_j(eps) bins */
int    opmc_test_evap_first(opmc_ctx *, int Z, int A, double estar, uint32_t channel_mask, uint64_t n,
                            uint64_t seed, double *widths, int32_t *out_channel, double *out_eps,
                            double *out_cos);
/* n samples of cos(theta_cm) of the NN elastic angular law (PAPER.md:L77 ref [20]; Reading R6.6) */
int    opmc_test_nn_cos(int same_type, double p_lab_gev, double pcm_mev, uint64_t n, uint64_t seed, double *out);
/* cascade attempts on a hand-made shell nucleus (see opmc.cpp): closed-form pins of refraction/reflection, Pauli
   blocking and of the NN angular law as the cascade uses it */
int    opmc_test_inc_custom(int nshell, const double *rout, const double *rho, const double *pF, const double *V,
                            double coulomb, int pauli, double const_sigma_mb, double t_in, uint64_t n, uint64_t seed,
                            int32_t *out_n, double *out_rec);
/* n primaries of a plan from the beam-spot sampler: out[n][8] = spot, x, y, z, u, v, w, E */
int    opmc_test_sample_primaries(opmc_ctx *, const opmc_spot *spots, int nspots, uint64_t n, uint64_t seed, double *out);
/* events of the last opmc_simulate per class and element: out[16] = elastic[8], non-elastic[8] */
int    opmc_test_event_counts(opmc_ctx *, uint64_t *out);
double opmc_test_cugnon(int which /*0 sigma_pp,1 sigma_np,2 B_pp,3 B_np,4 a_np*/, double p_gev);
#ifdef __cplusplus
}
#endif
#endif
