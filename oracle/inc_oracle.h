/* inc_oracle.h — CPU fp64 ORACLE of the INC + evaporation model of arXiv:1309.7963.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this.  The CUDA
 * product (paper_1309_7963_b200/) shares no code with it and never routes through it.
 *
 * Plain, slow, single-threaded, one event at a time, explicit LIFO stack of tracks.
 * Every step cites PAPER.md (P:NN) and, where the paper is silent, the reading
 * frozen in DESIGN.md ("R-x" tags).  All host pointers.
 *
 * Parity pins: see the header of inc_oracle.c and DESIGN.md section "Oracle pins".
 * Physics fidelity to the authors' unpublished code / figures: PARITY UNPINNED
 * (the paper prints no physics numbers; figures are absent).
 */
#ifndef INC_ORACLE_H
#define INC_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ORC_MAX_SHELLS 32
#define ORC_MAX_SEC 64          /* R-C5: per-event cap on secondaries               */
#define ORC_MAX_SEG 1024        /* R-C2: per-track cap on segments                  */
#define ORC_MAX_ATTEMPT 256     /* R-C6: attempts 0..255                            */
#define ORC_MAX_TRIAL 64        /* R-E4: rejection-sampler trial cap                */

/* status word (same bit meaning as the product's, restated independently) */
#define ORC_ST_ATTEMPT_MASK 0xFFu
#define ORC_ST_FAILED (1u << 8)
#define ORC_ST_SEC_TRUNC (1u << 9)
#define ORC_ST_DEPTH_CAP (1u << 10)
#define ORC_ST_SEG_CAP (1u << 11)
#define ORC_ST_TRIAL_CAP (1u << 12)

/* flags */
#define ORC_F_CASCADE_ONLY 1u      /* stop after the cascade epilogue (no evaporation)           */
#define ORC_F_KEEP_TRANSPARENT 2u  /* debug: accept n_real == 0 attempts instead of retrying     */
#define ORC_F_FIFO 4u              /* debug: process pending tracks first-in-first-out (R-R4 pin)*/

typedef struct orc_tables { /* caller-supplied model inputs ("precalculated ... tables") */
  int32_t version;          /* 1: the fields up to evap_a_div; 2: also the level-density block at the end */
  int32_t n_xs;             /* NN grid points; plab_k = k*plab_max/(n_xs-1) GeV/c */
  double plab_max;
  const double *sig_pp, *sig_np;     /* mb */
  const double *B_pp, *B_np, *a_np;  /* (GeV/c)^-2, -, np backward weight */
  int32_t n_evz;
  const double *ev_Z, *ev_kp, *ev_cp, *ev_ka, *ev_ca; /* Dostrovsky k,c vs Z_d */
  double ws_c0, ws_delta, ws_rpad;   /* 1.07, 0.545, 2.5 */
  int32_t n_shells;                  /* 15 */
  double semf[5];                    /* a_v a_s a_c a_a a_p */
  double evap_r0, evap_rj, evap_a_div;
  /* ---- version 2: evaporation level density ("generalized evaporation model (GEM) [18]") */
  int32_t level_density;    /* 0: rho ~ exp(2 sqrt(a U)), a = A_d / evap_a_div (R-Q19); 1: GEM level density (R-G1..G6) */
  int32_t n_ldZ, n_ldN;     /* lengths of the arrays below, indexed by Z_d resp. N_d (beyond the end: 0) */
  const double *pair_Z, *pair_N;     /* pairing energies, MeV: delta = pair_Z[Z_d] + pair_N[N_d] (R-G3) */
  const double *shell_Z, *shell_N;   /* shell corrections S, MeV: a = A_d (gc_a0 + gc_a1 (S_Z + S_N)) (R-G2) */
  double gc_a0, gc_a1;      /* 1/8 and 0.00917 MeV^-1 */
} orc_tables;

typedef struct orc_ld {     /* level-density constants of one daughter nucleus (R-G2..G4) */
  double a, delta;          /* level-density parameter MeV^-1, pairing energy MeV */
  double Ux, Ex;            /* matching energy U_x = 150/A_d + 2.5 and E_x = U_x + delta */
  double T, E0;             /* constant-temperature branch: rho = exp((U - E0)/T)/T below E_x */
} orc_ld;

typedef struct orc_nucleus {
  int32_t A, Z, n_shells;
  double c, R, delta_r;
  double r[ORC_MAX_SHELLS + 1];         /* r[i] = i*delta_r                     */
  double rho[ORC_MAX_SHELLS];           /* total density fm^-3 (R-N2)           */
  double rho_p[ORC_MAX_SHELLS], rho_n[ORC_MAX_SHELLS];
  double pF_p[ORC_MAX_SHELLS], pF_n[ORC_MAX_SHELLS]; /* MeV/c (R-N3)            */
  double EF_p[ORC_MAX_SHELLS], EF_n[ORC_MAX_SHELLS]; /* MeV                     */
  double V_p[ORC_MAX_SHELLS + 1], V_n[ORC_MAX_SHELLS + 1]; /* P:45; [n_shells]=0 outside */
  double EB_p, EB_n, EC, M;             /* R-N4, R-N6, nuclear mass             */
} orc_nucleus;

typedef struct orc_stats { /* algorithmic-work counters */
  uint64_t events, failed, attempts, retry_transparent, retry_invalid, retry_estar;
  uint64_t segments, boundaries, reflections, escapes;
  uint64_t collisions, blocked, allowed, absorbed;
  uint64_t evap_steps, evap_trials, evap_emitted;
  uint64_t cap_seg, cap_depth, cap_sec, cap_trial;
  uint64_t philox_blocks;
} orc_stats;

/* ---- whole-path entry points ------------------------------------------------ */

/* N-steps: nuclear setup for (A,Z).  Returns 0, or <0 on bad arguments. */
int orc_setup_nucleus(int A, int Z, const orc_tables *t, orc_nucleus *out);

/* Simulate events e = e0 .. e0+n-1 (global event indices key the RNG).
 * E_in[i], target[i] (index into nuc[]) are the inputs of event e0+i.
 * Secondaries are appended event after event into sec_* (capacity cap); counts[i]
 * is the per-event count; res_* and status are per event.  casc_* (nullable) receive
 * the post-cascade residual (A,Z,E*,P) and the number of cascade secondaries.
 * Returns total secondaries (>=0) or <0 on error (-3: capacity). */
int64_t orc_simulate(const orc_tables *t, const orc_nucleus *nuc, int n_nuc,
                     int64_t e0, int64_t n, const double *E_in, const int32_t *target,
                     uint64_t seed, uint32_t flags,
                     uint8_t *sec_species, double *sec_T, double *sec_ux, double *sec_uy,
                     double *sec_uz, int64_t cap, int32_t *counts,
                     int32_t *res_A, int32_t *res_Z, double *res_Estar, double *res_px,
                     double *res_py, double *res_pz, uint32_t *status,
                     int32_t *casc_A, int32_t *casc_Z, double *casc_Estar, double *casc_P,
                     int32_t *casc_count, orc_stats *stats,
                     const uint8_t *projectile /* [n] 0 = neutron, 1 = proton; NULL = all protons (NEXT-3) */);

/* ---- one cascade attempt with its collision log (for the pins of the C2/C3 decision logic) ---- */
typedef struct orc_coll_rec {     /* one collision (C3), allowed or blocked */
  uint32_t pi, k;                 /* path code of the projectile track, Philox block of the collision */
  int32_t shell, type1, type2;    /* collision shell; species of the projectile and of the partner (1 = p) */
  int32_t blocked, keep1, keep2;  /* Pauli-blocked; scattered projectile / recoil survived the cutoff */
  double T_in;                    /* kinetic energy of the projectile before the collision */
  double plab, B, a_back;         /* GeV/c; slope and np backward weight read from the tables */
  double Sp, Sigma;               /* rho_p sigma_p and the total macroscopic cross section, fm^-1 */
  double T1, T2, costheta;        /* kinetic energies after the collision; cos(theta_cm) */
} orc_coll_rec;
/* Runs attempt `attempt` of global event `event` (R-R2 counters) and returns n_real (allowed collisions), or
 * -1 on bad arguments.  coll[0..min(*n_coll, cap_coll)) are the collisions in processing order (*n_coll counts
 * all of them); esc_* (each nullable, capacity ORC_MAX_SEC; esc_p is [3 * ORC_MAX_SEC]) the escaped particles in
 * ascending path code. */
int orc_cascade_trace(const orc_tables *t, const orc_nucleus *nu, uint64_t seed, uint64_t event, uint32_t attempt,
                      double E_in, int proj, uint32_t flags,
                      int cap_coll, orc_coll_rec *coll, int *n_coll,
                      uint32_t *esc_pi, int32_t *esc_type, double *esc_T, double *esc_p, int *n_esc,
                      uint32_t *status);

/* ---- single steps, exported so the pins can test each in isolation ----------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
double orc_u01(uint32_t x);                                   /* R-R3 */
int orc_valid_nucleus(int A, int Z);
double orc_binding(int A, int Z, const orc_tables *t);        /* MeV; NaN if invalid */
double orc_mass(int A, int Z, const orc_tables *t);
double orc_lerp_table(const double *y, int n, double plab_max, double plab);
/* R-T: Dostrovsky k, c versus daughter charge: linear in Z_d, clamped outside the grid */
double orc_lerp_z(const double *zz, const double *y, int n, double z);
/* R-C2 partner: p2 = pF * cbrt(u_mag) * n(u_cos,u_phi) */
void orc_partner(double pF, double u_mag, double u_cos, double u_phi, double p2[3]);
/* R-C2: partner-rest-frame momentum (GeV/c) of particle 1 */
double orc_plab(const double p1[3], double m1, const double p2[3], double m2);
/* R-C2 geometry: distances to the outer / inner sphere (inf if none) */
void orc_shell_distances(const double x[3], const double d[3], double r_in, double r_out,
                         int has_inner, double *d_in, double *d_out);
/* R-C3: two-body elastic scatter.  same_species selects pp/nn (no backward term). */
void orc_collide(const double p1[3], double m1, const double p2[3], double m2,
                 double B, double a_back, int same_species,
                 double u_t, double u_back, double u_phi,
                 double p1_out[3], double p2_out[3], double *costheta_cm);
/* R-C4: potential step at |x|; returns 0 refract (shell changes), 1 reflect. */
int orc_boundary(const double x[3], double p[3], double m, double V_from, double V_to,
                 double *T_new);
/* R-E1/E2: emission widths of the six channels; returns sum.  X[j]<=0 => closed. */
double orc_evap_widths(int A, int Z, double Estar, const orc_tables *t,
                       double W[6], double X[6], double Q[6], double V[6],
                       double beta[6], double a_d[6]);
/* R-G2..G4: level-density constants of the daughter (A_d, Z_d); returns 0, or -1 if a <= 0 */
int orc_gem_ld(int A_d, int Z_d, const orc_tables *t, orc_ld *out);
/* R-G5: ln rho(U) of the GEM level density (common factor pi/12 dropped), U >= 0 */
double orc_gem_lnrho(const orc_ld *ld, double U);
/* R-G5: int_0^X (x + beta) rho(X - x) dx by composite 16-point Gauss-Legendre (the definition, written out) */
double orc_gem_integral(const orc_ld *ld, double X, double beta);
/* R-G6: like orc_evap_sample_x, for the pdf (x + beta) rho(X - x) */
double orc_evap_sample_x_gem(const orc_ld *ld, double X, double beta, const uint32_t key[2],
                             uint32_t c1, uint32_t c2, uint32_t c3, uint32_t *k, int *trials);
/* R-E3: channel chosen by the cumulative sum of W in the E1 order against u_ch * Wsum; -1 if no W > 0 */
int orc_evap_choose(const double W[6], double Wsum, double u_ch);
/* R-E4: sample x in [0,X] from (x+beta)exp(2 sqrt(a (X-x))) using Philox stream
 * (key, ctr base c1,c2,c3) starting at block *k; returns x, advances *k, *trials. */
double orc_evap_sample_x(double a, double X, double beta, const uint32_t key[2],
                         uint32_t c1, uint32_t c2, uint32_t c3, uint32_t *k, int *trials);
/* R-E5: one emission: parent (A,Z,E*,P) emits channel j with channel energy
 * eps = V_j + x in direction from (u_cos,u_phi).  Outputs lab ejectile (T, p[3]) and
 * daughter (E*, P[3]). */
void orc_evap_emit(int A, int Z, double Estar, const double P[3], int j, double eps_tot,
                   double Estar_d, double u_cos, double u_phi, const orc_tables *t,
                   double *T_ej, double p_ej[3], double P_d[3]);

#ifdef __cplusplus
}
#endif
#endif
