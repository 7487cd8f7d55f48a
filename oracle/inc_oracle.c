/* inc_oracle.c — CPU fp64 ORACLE of the INC + evaporation model of arXiv:1309.7963.
 *
 * TEST INFRASTRUCTURE ONLY (see inc_oracle.h).  Build: gcc -O2 -ffp-contract=off.
 *
 * The method is a stochastic simulation, so the oracle is the algorithm written out
 * step by step in the paper's order, one event at a time, with an explicit
 * LIFO stack, every random draw addressed by a counter (R-R1..R5).  Where PAPER.md is
 * silent the reading is the one frozen in DESIGN.md section 3; tags "R-xx" below refer
 * to that list.  No blocking, fusion or reordering.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`):
 *   Philox          vs cuRAND's host Philox4_32_10 generator (library, independent)
 *   nuclear setup   closed forms of P:45, sum rho_i V_i = A, scipy.quad of Eq. (1)
 *   partner         analytic Fermi-gas CDF x^3, <p^2> = 3/5 pF^2
 *   collision       4-momentum to 1e-12, analytic exp(Bt) CDF, isotropy at B = 0
 *   Pauli           blocked fraction vs brute-force quadrature (independent kinematics)
 *   boundary        p_t conserved, energy step, |p| on reflection, L conserved through
 *                   a whole transparent traversal
 *   widths          closed form vs scipy.quad of the Weisskopf-Ewing integrand
 *   sampler         chi^2 vs the normalised pdf; Maxwellian limit
 *   events          exact A,Z conservation; 4-momentum 1e-6; LIFO == FIFO
 *   decision logic  (tests/test_oracle_decisions.py) zeroed / flat sigma tables with closed forms for the
 *                   transparent fraction and the partner share, uniform entry disc, blocked fraction of first
 *                   collisions vs quadrature, cutoff thresholds in the escape spectra, track tree, B / a wiring,
 *                   retry counters recounted from traces, channel frequencies vs W_j / Sum W, Dostrovsky rows vs
 *                   numpy.interp; tests/test_pins_bite.py breaks this file 27 ways and each pin must turn red
 *   GEM             (tests/test_oracle_gem.py) constants and matching, widths vs scipy.quad (2e-10), sampler chi^2
 *                   and envelope inequality, mode 0 == the Weisskopf-Ewing model
 * PARITY UNPINNED: agreement of the resulting spectra with the paper's Figs. 1-3
 * (figures absent, no numbers printed; cited sub-models [10,12,17,18] not in PAPER.md).
 */
#include "inc_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

/* ---- constants (R-K: standard values, fp64 literals) ------------------------ */
static const double HBARC = 197.3269804;   /* MeV fm */
static const double E2 = 1.43996448;       /* MeV fm */
static const double M_P = 938.27208816;    /* MeV */
static const double M_N = 939.56542052;    /* MeV */
static const double B_D = 2.224566, B_T = 8.481798, B_H3 = 7.718043, B_H4 = 28.29566;
static const double PI = 3.14159265358979323846;

static const int EV_A[6] = {1, 1, 2, 3, 3, 4};
static const int EV_Z[6] = {0, 1, 1, 1, 2, 2};
static const double EV_G[6] = {2, 2, 3, 2, 2, 1}; /* 2S+1 (R-E1) */

static double nucleon_mass(int type) { return type ? M_P : M_N; }

/* ---- R-R1: Philox4x32-10 ----------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t prod0 = (uint64_t)0xD2511F53u * c0;
    uint64_t prod1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t hi0 = (uint32_t)(prod0 >> 32), lo0 = (uint32_t)prod0;
    uint32_t hi1 = (uint32_t)(prod1 >> 32), lo1 = (uint32_t)prod1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* R-R3: u in (0,1), exact in fp64 */
double orc_u01(uint32_t x) { return ((double)x + 0.5) * (1.0 / 4294967296.0); }

typedef struct {
  uint32_t key[2];
  uint32_t c2, c3; /* event index lo, hi */
  orc_stats *st;
} rng_ctx;

/* R-R2: block k of stream (attempt, pi) of this event -> 4 uniforms */
static void draw4(const rng_ctx *g, uint32_t attempt, uint32_t pi, uint32_t k, double u[4]) {
  uint32_t ctr[4] = {k, (attempt << 24) | pi, g->c2, g->c3};
  uint32_t out[4];
  orc_philox4x32_10(ctr, g->key, out);
  for (int i = 0; i < 4; ++i) u[i] = orc_u01(out[i]);
  if (g->st) g->st->philox_blocks++;
}

/* ---- masses (R-K) ------------------------------------------------------------ */
int orc_valid_nucleus(int A, int Z) {
  if (A < 1 || Z < 0 || Z > A) return 0;
  if (A >= 5) return 1;
  if (A == 1) return 1;                 /* n, p */
  if (A == 2) return Z == 1;            /* d */
  if (A == 3) return Z == 1 || Z == 2;  /* t, 3He */
  return Z == 2;                        /* 4He */
}

double orc_binding(int A, int Z, const orc_tables *t) {
  if (!orc_valid_nucleus(A, Z)) return NAN;
  if (A == 1) return 0.0;
  if (A == 2) return B_D;
  if (A == 3) return Z == 1 ? B_T : B_H3;
  if (A == 4) return B_H4;
  /* semi-empirical mass formula (coefficients R-Q4) */
  double a = (double)A, z = (double)Z;
  double A13 = cbrt(a);
  double B = t->semf[0] * a - t->semf[1] * A13 * A13 - t->semf[2] * z * (z - 1.0) / A13 -
             t->semf[3] * (a - 2.0 * z) * (a - 2.0 * z) / a;
  int N = A - Z;
  if ((Z % 2 == 0) && (N % 2 == 0)) B += t->semf[4] / sqrt(a);
  else if ((Z % 2 == 1) && (N % 2 == 1)) B -= t->semf[4] / sqrt(a);
  return B;
}

double orc_mass(int A, int Z, const orc_tables *t) {
  return Z * M_P + (A - Z) * M_N - orc_binding(A, Z, t);
}

/* ---- R-N7: linear table lookup, clamped ---------------------------------------- */
double orc_lerp_table(const double *y, int n, double plab_max, double plab) {
  double dp = plab_max / (double)(n - 1);
  double x = plab / dp;
  if (x < 0.0) x = 0.0;
  if (x > (double)(n - 1)) x = (double)(n - 1);
  int k = (int)floor(x);
  if (k > n - 2) k = n - 2;
  double f = x - (double)k;
  return y[k] + f * (y[k + 1] - y[k]);
}

double orc_lerp_z(const double *zz, const double *y, int n, double z) {
  /* Dostrovsky parameters vs Z_d: linear, clamped outside the grid (R-T) */
  if (z <= zz[0]) return y[0];
  if (z >= zz[n - 1]) return y[n - 1];
  int k = 0;
  while (k < n - 2 && z > zz[k + 1]) ++k;
  double f = (z - zz[k]) / (zz[k + 1] - zz[k]);
  return y[k] + f * (y[k + 1] - y[k]);
}

/* ---- N: nuclear setup -------------------------------------------------- */
static double ws_shape(double r, double c, double d) { return 1.0 / (1.0 + exp((r - c) / d)); } /* Eq.(1) */

int orc_setup_nucleus(int A, int Z, const orc_tables *t, orc_nucleus *nu) {
  if (!t || !nu || (t->version != 1 && t->version != 2)) return -2;
  if (t->n_shells < 1 || t->n_shells > ORC_MAX_SHELLS) return -2;
  if (A < 2 || Z < 1 || Z >= A) return -1;
  memset(nu, 0, sizeof(*nu));
  int ns = t->n_shells;
  nu->A = A; nu->Z = Z; nu->n_shells = ns;
  nu->c = t->ws_c0 * cbrt((double)A);          /* N1: c = 1.07 A^(1/3)            */
  nu->R = nu->c + t->ws_rpad;                  /* N1: R = c + 2.5 fm              */
  nu->delta_r = nu->R / (double)ns;            /* N1: equal thickness             */
  for (int i = 0; i <= ns; ++i) nu->r[i] = (double)i * nu->delta_r;
  /* N2: w_i = int_shell rho(r) 4 pi r^2 dr, composite Simpson, 2000 panels */
  double w[ORC_MAX_SHELLS], wsum = 0.0;
  const int NP = 2000;
  for (int i = 0; i < ns; ++i) {
    double a = nu->r[i], b = nu->r[i + 1], h = (b - a) / (double)NP;
    double s = 0.0;
    for (int k = 0; k <= NP; ++k) {
      double r = a + h * (double)k;
      double f = ws_shape(r, nu->c, t->ws_delta) * 4.0 * PI * r * r;
      double wt = (k == 0 || k == NP) ? 1.0 : ((k & 1) ? 4.0 : 2.0);
      s += wt * f;
    }
    w[i] = s * h / 3.0;
    wsum += w[i];
  }
  double N = (double)(A - Z);
  for (int i = 0; i < ns; ++i) {
    double vol = 4.0 * PI / 3.0 * (nu->r[i + 1] * nu->r[i + 1] * nu->r[i + 1] - nu->r[i] * nu->r[i] * nu->r[i]);
    nu->rho[i] = (double)A * w[i] / (vol * wsum);          /* N2: sum rho_i V_i = A */
    nu->rho_p[i] = nu->rho[i] * (double)Z / (double)A;     /* N2 (R-Q2)             */
    nu->rho_n[i] = nu->rho[i] * N / (double)A;
    /* N3: Fermi momentum and relativistic Fermi energy */
    nu->pF_p[i] = HBARC * cbrt(3.0 * PI * PI * nu->rho_p[i]);
    nu->pF_n[i] = HBARC * cbrt(3.0 * PI * PI * nu->rho_n[i]);
    nu->EF_p[i] = sqrt(nu->pF_p[i] * nu->pF_p[i] + M_P * M_P) - M_P;
    nu->EF_n[i] = sqrt(nu->pF_n[i] * nu->pF_n[i] + M_N * M_N) - M_N;
  }
  /* N4: separation energies from the SEMF ("binding energy E_B ... SEMF") */
  double BA = orc_binding(A, Z, t);
  nu->EB_p = BA - orc_binding(A - 1, Z - 1, t);
  nu->EB_n = BA - orc_binding(A - 1, Z, t);
  /* N5: V = E_F + E_B; outside V = 0 */
  for (int i = 0; i < ns; ++i) {
    nu->V_p[i] = nu->EF_p[i] + nu->EB_p;
    nu->V_n[i] = nu->EF_n[i] + nu->EB_n;
  }
  nu->V_p[ns] = 0.0; nu->V_n[ns] = 0.0;
  nu->EC = E2 * (double)Z / nu->R;             /* N6 (R-Q6) */
  nu->M = orc_mass(A, Z, t);
  return 0;
}

/* ---- small vector helpers ------------------------------------------------------ */
static double dot3(const double a[3], const double b[3]) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

static void unit_from_u(double u_cos, double u_phi, double n[3]) {
  double c = 2.0 * u_cos - 1.0;
  double phi = 2.0 * PI * u_phi;
  double s = sqrt(1.0 - c * c);
  n[0] = s * cos(phi); n[1] = s * sin(phi); n[2] = c;
}

/* ---- C2: partner from the Fermi sea ("quadratic distribution") -------------- */
void orc_partner(double pF, double u_mag, double u_cos, double u_phi, double p2[3]) {
  double n[3];
  unit_from_u(u_cos, u_phi, n);
  double f = cbrt(u_mag);     /* pdf of |p| proportional to p^2 on [0,pF] */
  for (int i = 0; i < 3; ++i) p2[i] = pF * f * n[i];
}

/* C2: momentum of 1 in the rest frame of 2, GeV/c */
double orc_plab(const double p1[3], double m1, const double p2[3], double m2) {
  double E1 = sqrt(dot3(p1, p1) + m1 * m1), E2_ = sqrt(dot3(p2, p2) + m2 * m2);
  double P[3] = {p1[0] + p2[0], p1[1] + p2[1], p1[2] + p2[2]};
  double s = (E1 + E2_) * (E1 + E2_) - dot3(P, P);
  double Elab = (s - m1 * m1 - m2 * m2) / (2.0 * m2);
  double q = Elab * Elab - m1 * m1;
  if (q < 0.0) q = 0.0;       /* rounding guard (R-RG1) */
  return sqrt(q) / 1000.0;
}

/* C2 geometry */
void orc_shell_distances(const double x[3], const double d[3], double r_in, double r_out,
                         int has_inner, double *d_in, double *d_out) {
  double beta = dot3(x, d), r2 = dot3(x, x);
  double disc_out = beta * beta - r2 + r_out * r_out;
  if (disc_out < 0.0) disc_out = 0.0;   /* rounding guard (R-RG2): x sits on/inside r_out */
  *d_out = -beta + sqrt(disc_out);
  *d_in = INFINITY;
  if (has_inner && beta < 0.0) {
    double D = beta * beta - r2 + r_in * r_in;
    if (D > 0.0) *d_in = -beta - sqrt(D);
  }
}

/* ---- C3: relativistic two-body elastic scatter --------------------------- */
static void boost(const double p[3], double E, const double bv[3], double gamma, double sign,
                  double out[3]) {
  /* sign = -1: lab -> frame moving with bv; +1: back.  identity if |bv|^2 < 1e-30 */
  double b2 = dot3(bv, bv);
  if (b2 < 1e-30) { out[0] = p[0]; out[1] = p[1]; out[2] = p[2]; return; }
  double pb = dot3(p, bv);
  double f = (gamma - 1.0) * pb / b2 + sign * gamma * E;
  for (int i = 0; i < 3; ++i) out[i] = p[i] + f * bv[i];
}

void orc_collide(const double p1[3], double m1, const double p2[3], double m2,
                 double B, double a_back, int same_species,
                 double u_t, double u_back, double u_phi,
                 double p1_out[3], double p2_out[3], double *costheta_cm) {
  double E1 = sqrt(dot3(p1, p1) + m1 * m1), E2_ = sqrt(dot3(p2, p2) + m2 * m2);
  double P[3] = {p1[0] + p2[0], p1[1] + p2[1], p1[2] + p2[2]};
  double E = E1 + E2_;
  double s = E * E - dot3(P, P);
  double bv[3] = {P[0] / E, P[1] / E, P[2] / E};
  double gamma = E / sqrt(s);
  double q[3];
  boost(p1, E1, bv, gamma, -1.0, q);            /* p1* in the CM frame */
  double pcm2 = dot3(q, q), pcm = sqrt(pcm2);
  /* angle: dsigma/dt ~ exp(B t), t in (GeV/c)^2 (R-Q10) */
  double pg2 = pcm2 * 1e-6;
  double tmin = -4.0 * pg2;
  double t;
  if (B * (-tmin) < 1e-9) t = u_t * tmin;
  else t = log1p(-u_t * (-expm1(B * tmin))) / B;
  double ct = 1.0 + t / (2.0 * pg2);
  if (ct < -1.0) ct = -1.0;                      /* rounding guard (R-RG3) */
  if (ct > 1.0) ct = 1.0;
  if (!same_species && u_back * (1.0 + a_back) < a_back) ct = -ct;
  double st = sqrt(1.0 - ct * ct);
  double phi = 2.0 * PI * u_phi;
  /* rotation: frame (e1,e2,n) around n = unit vector of p1 in the CM frame */
  double n[3] = {q[0] / pcm, q[1] / pcm, q[2] / pcm};
  double q2 = n[0] * n[0] + n[1] * n[1];
  double e1[3], e2[3];
  if (q2 > 1e-24) {
    double qq = sqrt(q2);
    e1[0] = n[0] * n[2] / qq; e1[1] = n[1] * n[2] / qq; e1[2] = -q2 / qq;
    e2[0] = -n[1] / qq; e2[1] = n[0] / qq; e2[2] = 0.0;
  } else {
    double sg = n[2] >= 0.0 ? 1.0 : -1.0;
    e1[0] = 1.0; e1[1] = 0.0; e1[2] = 0.0;
    e2[0] = 0.0; e2[1] = sg; e2[2] = 0.0;
  }
  double cp = cos(phi), sp = sin(phi);
  double q1[3], q2v[3];
  for (int i = 0; i < 3; ++i) {
    q1[i] = pcm * (st * cp * e1[i] + st * sp * e2[i] + ct * n[i]);
    q2v[i] = -q1[i];
  }
  double E1cm = sqrt(pcm2 + m1 * m1), E2cm = sqrt(pcm2 + m2 * m2);
  boost(q1, E1cm, bv, gamma, +1.0, p1_out);
  boost(q2v, E2cm, bv, gamma, +1.0, p2_out);
  if (costheta_cm) *costheta_cm = ct;
}

/* ---- C4: potential step at a shell boundary ("refraction and reflection") --- */
int orc_boundary(const double x[3], double p[3], double m, double V_from, double V_to,
                 double *T_new) {
  double r = sqrt(dot3(x, x));
  double n[3] = {x[0] / r, x[1] / r, x[2] / r};
  double pr = dot3(p, n);
  double pt[3] = {p[0] - pr * n[0], p[1] - pr * n[1], p[2] - pr * n[2]};
  double Ti = sqrt(dot3(p, p) + m * m) - m;
  double Tj = Ti + V_to - V_from;
  int reflect = 0;
  double prj2 = 0.0;
  if (Tj <= 0.0) reflect = 1;
  else {
    double pj2 = Tj * (Tj + 2.0 * m);
    prj2 = pj2 - dot3(pt, pt);
    if (prj2 <= 0.0) reflect = 1;
  }
  if (reflect) {
    for (int i = 0; i < 3; ++i) p[i] = p[i] - 2.0 * pr * n[i];
    if (T_new) *T_new = Ti;
    return 1;
  }
  double sg = pr >= 0.0 ? 1.0 : -1.0;
  double prj = sg * sqrt(prj2);
  for (int i = 0; i < 3; ++i) p[i] = pt[i] + prj * n[i];
  if (T_new) *T_new = Tj;
  return 0;
}

/* ---- E: evaporation --------------------------------------------------------------- */
/* G_n(s) = int_0^s t^n e^t dt, n = 1, 3 */
static double G_series(int n, double s) {
  double sum = 0.0, term = pow(s, n + 1); /* k = 0: s^(n+1)/(0! (n+1)) */
  double kfact = 1.0;
  for (int k = 0; k < 40; ++k) {
    if (k > 0) { term *= s; kfact *= (double)k; }
    sum += term / (kfact * (double)(n + 1 + k));
  }
  return sum;
}
static double G1(double s) { return s < 0.5 ? G_series(1, s) : (s - 1.0) * exp(s) + 1.0; }
static double G3(double s) {
  return s < 0.5 ? G_series(3, s) : (s * s * s - 3.0 * s * s + 6.0 * s - 6.0) * exp(s) + 6.0;
}

double orc_evap_widths(int A, int Z, double Estar, const orc_tables *t,
                       double W[6], double X[6], double Q[6], double V[6],
                       double beta[6], double a_d[6]) {
  double sum = 0.0;
  double Mi = orc_mass(A, Z, t);
  for (int j = 0; j < 6; ++j) {
    W[j] = 0.0; X[j] = -1.0; Q[j] = 0.0; V[j] = 0.0; beta[j] = 0.0; a_d[j] = 0.0;
    int Ad = A - EV_A[j], Zd = Z - EV_Z[j];
    if (Ad < 1 || !orc_valid_nucleus(Ad, Zd)) continue;     /* E1: closed */
    double Mj = orc_mass(EV_A[j], EV_Z[j], t);
    Q[j] = orc_mass(Ad, Zd, t) + Mj - Mi;
    double ad13 = cbrt((double)Ad);
    double alpha;
    if (j == 0) {                                           /* neutron (Dostrovsky) */
      alpha = 0.76 + 2.2 / ad13;
      beta[j] = (2.12 / (ad13 * ad13) - 0.05) / alpha;
      V[j] = 0.0;
    } else {
      double zd = (double)Zd;
      double kp = orc_lerp_z(t->ev_Z, t->ev_kp, t->n_evz, zd);
      double cp = orc_lerp_z(t->ev_Z, t->ev_cp, t->n_evz, zd);
      double ka = orc_lerp_z(t->ev_Z, t->ev_ka, t->n_evz, zd);
      double ca = orc_lerp_z(t->ev_Z, t->ev_ca, t->n_evz, zd);
      double k, c, rj;
      switch (j) {
        case 1: k = kp; c = cp; rj = 0.0; break;
        case 2: k = kp + 0.06; c = cp / 2.0; rj = t->evap_rj; break;
        case 3: k = kp + 0.12; c = cp / 3.0; rj = t->evap_rj; break;
        case 4: k = ka - 0.06; c = 4.0 * ca / 3.0; rj = t->evap_rj; break;
        default: k = ka; c = ca; rj = t->evap_rj; break;
      }
      alpha = 1.0 + c;
      beta[j] = 0.0;
      V[j] = k * E2 * (double)EV_Z[j] * zd / (t->evap_r0 * ad13 + rj);
    }
    X[j] = Estar - Q[j] - V[j];
    if (!(X[j] > 0.0)) { X[j] = -1.0; continue; }           /* E1: closed */
    if (t->version >= 2 && t->level_density == 1) {         /* NEXT-2: GEM level density (R-G1..G5) */
      orc_ld ld;
      if (orc_gem_ld(Ad, Zd, t, &ld) != 0) { X[j] = -1.0; continue; }
      a_d[j] = ld.a;
      W[j] = EV_G[j] * Mj * ad13 * ad13 * alpha * orc_gem_integral(&ld, X[j], beta[j]);
      if (W[j] < 0.0) W[j] = 0.0;
      sum += W[j];
      continue;
    }
    double a = (double)Ad / t->evap_a_div;
    a_d[j] = a;
    double s = 2.0 * sqrt(a * X[j]);
    double I0 = G1(s) / (2.0 * a);
    double I1 = X[j] * I0 - G3(s) / (8.0 * a * a);
    W[j] = EV_G[j] * Mj * ad13 * ad13 * alpha * (I1 + beta[j] * I0);   /* E2 */
    if (W[j] < 0.0) W[j] = 0.0;
    sum += W[j];
  }
  return sum;
}

/* ---- NEXT-2: GEM level density ("we adopt the generalized evaporation model (GEM) [18]"; DESIGN R-G1..G6) ---- */
static double ld_table(const double *y, int n, int i) { return (y && i >= 0 && i < n) ? y[i] : 0.0; }

int orc_gem_ld(int A_d, int Z_d, const orc_tables *t, orc_ld *ld) {
  int N_d = A_d - Z_d;
  double S = ld_table(t->shell_Z, t->n_ldZ, Z_d) + ld_table(t->shell_N, t->n_ldN, N_d);
  ld->a = (double)A_d * (t->gc_a0 + t->gc_a1 * S);                                   /* R-G2 */
  ld->delta = ld_table(t->pair_Z, t->n_ldZ, Z_d) + ld_table(t->pair_N, t->n_ldN, N_d);   /* R-G3 */
  ld->Ux = 150.0 / (double)A_d + 2.5;                                                /* R-G4 */
  ld->Ex = ld->Ux + ld->delta;
  if (!(ld->a > 0.0)) return -1;
  double invT = sqrt(ld->a / ld->Ux) - 1.5 / ld->Ux;
  if (!(invT > 0.0)) return -1;                    /* R-G7: no constant-temperature branch exists: channel closed */
  ld->T = 1.0 / invT;
  ld->E0 = ld->Ex - ld->T * (log(ld->T) - 0.25 * log(ld->a) - 1.25 * log(ld->Ux) + 2.0 * sqrt(ld->a * ld->Ux));
  return 0;
}

double orc_gem_lnrho(const orc_ld *ld, double U) {
  if (U >= ld->Ex) {                               /* Fermi gas with the pre-exponential factor */
    double u = U - ld->delta;
    return 2.0 * sqrt(ld->a * u) - 0.25 * log(ld->a) - 1.25 * log(u);
  }
  return (U - ld->E0) / ld->T - log(ld->T);        /* constant temperature */
}

/* 16-point Gauss-Legendre nodes and weights on [-1, 1], found by Newton iteration on P_16 */
static void gl16(double x[16], double w[16]) {
  for (int i = 0; i < 16; ++i) {
    double z = cos(PI * ((double)i + 0.75) / 16.5), dp = 1.0;
    for (int it = 0; it < 100; ++it) {
      double p0 = 1.0, p1 = z;
      for (int k = 2; k <= 16; ++k) { double p2 = ((2.0 * k - 1.0) * z * p1 - (k - 1.0) * p0) / k; p0 = p1; p1 = p2; }
      dp = 16.0 * (z * p1 - p0) / (z * z - 1.0);
      double dz = p1 / dp;
      z -= dz;
      if (fabs(dz) < 1e-16) break;
    }
    x[i] = z; w[i] = 2.0 / ((1.0 - z * z) * dp * dp);
  }
}

static double gem_range(const orc_ld *ld, double X, double beta, double x0, double x1, const double gx[16], const double gw[16]) {
  /* int_x0^x1 (x + beta) rho(X - x) dx, panels of at most 8 MeV */
  if (!(x1 > x0)) return 0.0;
  int np = (int)ceil((x1 - x0) / 8.0);
  if (np < 1) np = 1;
  double h = (x1 - x0) / (double)np, sum = 0.0;
  for (int p = 0; p < np; ++p) {
    double a = x0 + h * (double)p;
    for (int q = 0; q < 16; ++q) {
      double x = a + 0.5 * h * (gx[q] + 1.0);
      double U = X - x;
      if (U < 0.0) U = 0.0;
      sum += 0.5 * h * gw[q] * (x + beta) * exp(orc_gem_lnrho(ld, U));
    }
  }
  return sum;
}

double orc_gem_integral(const orc_ld *ld, double X, double beta) {
  double gx[16], gw[16];
  gl16(gx, gw);
  double xs = X - ld->Ex;                          /* x below xs: daughter above E_x (Fermi gas) */
  if (xs <= 0.0 || xs >= X) return gem_range(ld, X, beta, 0.0, X, gx, gw);   /* one branch on all of [0, X] (R-G7: E_x <= 0) */
  return gem_range(ld, X, beta, 0.0, xs, gx, gw) + gem_range(ld, X, beta, xs, X, gx, gw);
}

double orc_evap_sample_x_gem(const orc_ld *ld, double X, double beta, const uint32_t key[2],
                             uint32_t c1, uint32_t c2, uint32_t c3, uint32_t *k, int *trials) {
  /* R-G6: rejection from the two envelopes of R-E4 with ln rho in place of 2 sqrt(a U).  ln rho(U) rises with a
   * slope that is 1/T on the constant-temperature branch and falls from there on the Fermi-gas branch, so
   * ln rho(X - x) <= ln rho(X) - x m with m the smallest slope on [0, X]: envelope (A) is (x + beta) e^(-x m). */
  double m = 1.0 / ld->T;
  if (X > ld->Ex) {
    double u = X - ld->delta;
    double sfg = sqrt(ld->a / u) - 1.25 / u;
    if (sfg < m) m = sfg;
  }
  double T = 1.0 / m;
  double l0 = orc_gem_lnrho(ld, X);
  double areaA = T * (T + beta), areaB = 0.5 * X * X + beta * X;
  for (int n = 0; n < ORC_MAX_TRIAL; ++n) {
    uint32_t ctr[4] = {*k, c1, c2, c3}, out[4];
    orc_philox4x32_10(ctr, key, out);
    (*k)++;
    if (trials) (*trials)++;
    double u_mix = orc_u01(out[0]), u1 = orc_u01(out[1]), u2 = orc_u01(out[2]), u_acc = orc_u01(out[3]);
    double x;
    if (areaB < areaA) {
      x = -beta + sqrt(beta * beta + u1 * (X * X + 2.0 * beta * X));
      double rem = X - x;
      if (rem < 0.0) rem = 0.0;
      if (log(u_acc) < orc_gem_lnrho(ld, rem) - l0) return x < X ? x : X;
    } else {
      if (u_mix * (T + beta) < T) x = -T * log(u1 * u2);
      else x = -T * log(u1);
      if (x < X && log(u_acc) < orc_gem_lnrho(ld, X - x) - l0 + x / T) return x;
    }
  }
  return -1.0;
}

/* E3: channel by cumulative sum over j in the E1 order against u_ch * Sum W (R-E3) */
int orc_evap_choose(const double W[6], double Wsum, double u_ch) {
  int j = -1;
  double cum = 0.0, thr = u_ch * Wsum;
  for (int q = 0; q < 6; ++q) {
    if (W[q] > 0.0) { cum += W[q]; j = q; if (thr < cum) break; }
  }
  return j;
}

double orc_evap_sample_x(double a, double X, double beta, const uint32_t key[2],
                         uint32_t c1, uint32_t c2, uint32_t c3, uint32_t *k, int *trials) {
  /* E4: exact rejection sampling of f(x) ~ (x+beta) exp(2 sqrt(a (X-x))) on [0,X].
   * Two envelopes, both >= f/e^s:  (A) g(x) = (x+beta) e^(-x/T), T = sqrt(X/a), valid
   * because 2 sqrt(a(X-x)) <= s - x/T (concavity); (B) g(x) = (x+beta) on [0,X], valid
   * because 2 sqrt(a(X-x)) <= s.  The one with the smaller area is used (R-E4); this
   * keeps the acceptance above ~0.36 for every (a, X, beta). */
  double s = 2.0 * sqrt(a * X);
  double T = sqrt(X / a);
  double areaA = T * (T + beta), areaB = 0.5 * X * X + beta * X;
  for (int n = 0; n < ORC_MAX_TRIAL; ++n) {
    uint32_t ctr[4] = {*k, c1, c2, c3}, out[4];
    orc_philox4x32_10(ctr, key, out);
    (*k)++;
    if (trials) (*trials)++;
    double u_mix = orc_u01(out[0]), u1 = orc_u01(out[1]), u2 = orc_u01(out[2]), u_acc = orc_u01(out[3]);
    double x;
    if (areaB < areaA) {
      /* (B) inverse CDF of (x+beta) on [0,X] */
      x = -beta + sqrt(beta * beta + u1 * (X * X + 2.0 * beta * X));
      double rem = X - x;
      if (rem < 0.0) rem = 0.0;
      if (log(u_acc) < 2.0 * sqrt(a * rem) - s) return x < X ? x : X;
    } else {
      /* (A) mixture: Gamma(2,T) with weight T/(T+beta), else Exp(T) */
      if (u_mix * (T + beta) < T) x = -T * log(u1 * u2);
      else x = -T * log(u1);
      if (x < X && log(u_acc) < 2.0 * sqrt(a * (X - x)) - s + x / T) return x;
    }
  }
  return -1.0; /* cap reached */
}

void orc_evap_emit(int A, int Z, double Estar, const double P[3], int j, double eps_tot,
                   double Estar_d, double u_cos, double u_phi, const orc_tables *t,
                   double *T_ej, double p_ej[3], double P_d[3]) {
  /* E5: exact two-body decay M_par -> M_j + (M_d + E*_d) in the parent rest frame,
   * isotropic, then boost to the lab with the parent velocity. */
  (void)eps_tot;
  double Mpar = orc_mass(A, Z, t) + Estar;
  double Mj = orc_mass(EV_A[j], EV_Z[j], t);
  double Mds = orc_mass(A - EV_A[j], Z - EV_Z[j], t) + Estar_d;
  double lam = (Mpar * Mpar - (Mj + Mds) * (Mj + Mds)) * (Mpar * Mpar - (Mj - Mds) * (Mj - Mds));
  if (lam < 0.0) lam = 0.0;
  double pmag = sqrt(lam) / (2.0 * Mpar);
  double Ej = sqrt(pmag * pmag + Mj * Mj);
  double n[3];
  unit_from_u(u_cos, u_phi, n);
  double q[3] = {pmag * n[0], pmag * n[1], pmag * n[2]};
  double Epar = sqrt(Mpar * Mpar + dot3(P, P));
  double bv[3] = {P[0] / Epar, P[1] / Epar, P[2] / Epar};
  double gamma = Epar / Mpar;
  boost(q, Ej, bv, gamma, +1.0, p_ej);
  *T_ej = sqrt(dot3(p_ej, p_ej) + Mj * Mj) - Mj;
  for (int i = 0; i < 3; ++i) P_d[i] = P[i] - p_ej[i];
}

/* ---- the event loop ---------------------------------------------------------------- */
typedef struct {
  double x[3], p[3];
  int type, shell;
  uint32_t pi, k;
  int nseg;
} track;

typedef struct {
  uint32_t pi; int type; double T; double p[3];
} esc_rec;

static int cmp_esc(const void *a, const void *b) {
  uint32_t x = ((const esc_rec *)a)->pi, y = ((const esc_rec *)b)->pi;
  return x < y ? -1 : (x > y ? 1 : 0);
}

#define STACK_MAX 256

/* One cascade attempt (C0-C5).  Returns n_real; fills esc[0..*n_esc). */
/* trace: optional log of every collision of the attempt (decision inputs and outcomes), filled only for
 * orc_cascade_trace -- the window through which the pins check the C2/C3 wiring (which table, which species'
 * E_F, which cutoff, which child codes).  Recording changes nothing of the attempt. */
typedef struct { orc_coll_rec *rec; int cap, n; } coll_trace;

static int cascade_attempt(const orc_tables *t, const orc_nucleus *nu, const rng_ctx *g,
                           uint32_t attempt, double E_in, int proj, uint32_t flags,
                           esc_rec *esc, int *n_esc, uint32_t *status, orc_stats *st, coll_trace *trc) {
  int ns = nu->n_shells;
  int n_real = 0;
  *n_esc = 0;
  track stack[STACK_MAX];
  int sp = 0, head = 0; /* head used for FIFO debug order */

  /* C0: entry — uniform disc, beam +z (R-Q15) */
  double u[4];
  draw4(g, attempt, 1u, 0u, u);
  double b = nu->R * sqrt(u[0]);
  double phib = 2.0 * PI * u[1];
  track tr;
  tr.x[0] = b * cos(phib); tr.x[1] = b * sin(phib);
  { double zz = nu->R * nu->R - b * b; if (zz < 0.0) zz = 0.0; tr.x[2] = -sqrt(zz); }
  /* NEXT-3 ("nucleon-nucleus interaction"): the incident nucleon is a proton (proj = 1) or a neutron
     (proj = 0); it enters with its own mass and feels its own species' potential */
  const double m0 = nucleon_mass(proj);
  tr.p[0] = 0.0; tr.p[1] = 0.0; tr.p[2] = sqrt(E_in * (E_in + 2.0 * m0));
  tr.type = proj; tr.pi = 1u; tr.k = 1u; tr.nseg = 0;
  {
    int refl = orc_boundary(tr.x, tr.p, m0, 0.0, proj ? nu->V_p[ns - 1] : nu->V_n[ns - 1], NULL);
    (void)refl; /* cannot reflect: V rises inward */
    tr.shell = ns - 1;
  }
  stack[sp++] = tr;

  while (sp > head) {
    /* C1: next pending track (order immaterial, R-R4) */
    if (flags & ORC_F_FIFO) tr = stack[head++];
    else tr = stack[--sp];
    if (head > 0 && head == sp) { head = 0; sp = 0; }
    int alive = 1;
    while (alive) {
      if (tr.nseg >= ORC_MAX_SEG) { *status |= ORC_ST_SEG_CAP; if (st) { st->cap_seg++; st->absorbed++; } break; }
      tr.nseg++;
      if (st) st->segments++;
      int i = tr.shell;
      double m1 = nucleon_mass(tr.type);
      /* C2: segment — partner first, then the exponential path (R-Q8) */
      draw4(g, attempt, tr.pi, tr.k++, u);
      double p2p[3], p2n[3];
      orc_partner(nu->pF_p[i], u[0], u[1], u[2], p2p);
      orc_partner(nu->pF_n[i], u[0], u[1], u[2], p2n);
      double plab_p = orc_plab(tr.p, m1, p2p, M_P);
      double plab_n = orc_plab(tr.p, m1, p2n, M_N);
      double sig_p = orc_lerp_table(tr.type == 1 ? t->sig_pp : t->sig_np, t->n_xs, t->plab_max, plab_p) * 0.1;
      double sig_n = orc_lerp_table(tr.type == 0 ? t->sig_pp : t->sig_np, t->n_xs, t->plab_max, plab_n) * 0.1;
      double Sp = nu->rho_p[i] * sig_p, Sn = nu->rho_n[i] * sig_n;
      double Sigma = Sp + Sn;
      double d_coll = Sigma > 0.0 ? -log(u[3]) / Sigma : INFINITY;
      double pm = sqrt(dot3(tr.p, tr.p));
      double dir[3] = {tr.p[0] / pm, tr.p[1] / pm, tr.p[2] / pm};
      double d_in, d_out;
      orc_shell_distances(tr.x, dir, nu->r[i], nu->r[i + 1], i > 0, &d_in, &d_out);
      double d_min = d_in < d_out ? d_in : d_out;
      if (d_coll < d_min) {
        /* C3: collision at x + d_coll dir */
        for (int q = 0; q < 3; ++q) tr.x[q] += d_coll * dir[q];
        if (st) st->collisions++;
        draw4(g, attempt, tr.pi, tr.k++, u);
        int t2 = (u[0] * Sigma < Sp) ? 1 : 0;
        double m2 = nucleon_mass(t2);
        const double *p2 = t2 ? p2p : p2n;
        double plab = t2 ? plab_p : plab_n;
        int same = (t2 == tr.type);
        double B = orc_lerp_table(same ? t->B_pp : t->B_np, t->n_xs, t->plab_max, plab);
        double ab = same ? 0.0 : orc_lerp_table(t->a_np, t->n_xs, t->plab_max, plab);
        double q1[3], q2[3];
        double ct_cm;
        orc_collide(tr.p, m1, p2, m2, B, ab, same, u[1], u[2], u[3], q1, q2, &ct_cm);
        double T1 = sqrt(dot3(q1, q1) + m1 * m1) - m1;
        double T2 = sqrt(dot3(q2, q2) + m2 * m2) - m2;
        double EF1 = tr.type ? nu->EF_p[i] : nu->EF_n[i];
        double EF2 = t2 ? nu->EF_p[i] : nu->EF_n[i];
        orc_coll_rec *lg = NULL;
        if (trc && trc->n < trc->cap) {
          lg = &trc->rec[trc->n];
          lg->pi = tr.pi; lg->k = tr.k - 1u; lg->shell = i; lg->type1 = tr.type; lg->type2 = t2;
          lg->blocked = 0; lg->keep1 = 0; lg->keep2 = 0;
          lg->T_in = sqrt(dot3(tr.p, tr.p) + m1 * m1) - m1;
          lg->plab = plab; lg->B = B; lg->a_back = ab; lg->Sp = Sp; lg->Sigma = Sigma;
          lg->T1 = T1; lg->T2 = T2; lg->costheta = ct_cm;
        }
        if (trc) trc->n++;
        if (!(T1 > EF1 && T2 > EF2)) {           /* Pauli, strict > (R-Q12) */
          if (st) st->blocked++;
          if (lg) lg->blocked = 1;
          continue;                              /* projectile continues unchanged (R-Q13) */
        }
        n_real++;
        if (st) st->allowed++;
        alive = 0;
        if (2u * tr.pi + 1u >= (1u << 24)) {     /* depth cap (R-C3) */
          *status |= ORC_ST_DEPTH_CAP;
          if (st) { st->cap_depth++; st->absorbed += 2; }
          break;
        }
        /* children + cutoff: eps = T' - V; absorbed if eps <= 0 (n) / <= E_C (p) */
        track ch[2];
        for (int c = 0; c < 2; ++c) {
          ch[c].type = c == 0 ? tr.type : t2;
          ch[c].pi = 2u * tr.pi + (uint32_t)c;
          ch[c].k = 0u; ch[c].nseg = 0; ch[c].shell = i;
          for (int q = 0; q < 3; ++q) { ch[c].x[q] = tr.x[q]; ch[c].p[q] = c == 0 ? q1[q] : q2[q]; }
        }
        for (int c = 1; c >= 0; --c) {           /* push recoil first, scattered on top */
          double Tc = c == 0 ? T1 : T2;
          double Vc = ch[c].type ? nu->V_p[i] : nu->V_n[i];
          double eps = Tc - Vc;
          double cut = ch[c].type ? nu->EC : 0.0;
          if (eps <= cut) { if (st) st->absorbed++; continue; }
          if (lg) { if (c == 0) lg->keep1 = 1; else lg->keep2 = 1; }
          if (sp < STACK_MAX) stack[sp++] = ch[c];
        }
      } else {
        /* C4: boundary */
        if (st) st->boundaries++;
        int j = (d_in < d_out) ? i - 1 : i + 1;
        double rb = (d_in < d_out) ? nu->r[i] : nu->r[i + 1];
        for (int q = 0; q < 3; ++q) tr.x[q] += d_min * dir[q];
        double rr = sqrt(dot3(tr.x, tr.x));
        for (int q = 0; q < 3; ++q) tr.x[q] *= rb / rr;   /* renormalise onto the sphere */
        const double *V = tr.type ? nu->V_p : nu->V_n;
        double Tn;
        int refl = orc_boundary(tr.x, tr.p, m1, V[i], V[j], &Tn);
        if (refl) { if (st) st->reflections++; continue; }
        tr.shell = j;
        if (j == ns) {                           /* escape */
          alive = 0;
          if (st) st->escapes++;
          if (*n_esc < ORC_MAX_SEC) {
            esc_rec *r = &esc[(*n_esc)++];
            r->pi = tr.pi; r->type = tr.type; r->T = Tn;
            r->p[0] = tr.p[0]; r->p[1] = tr.p[1]; r->p[2] = tr.p[2];
          } else { *status |= ORC_ST_SEC_TRUNC; if (st) st->cap_sec++; }
        }
      }
    }
  }
  return n_real;
}

/* One cascade attempt (C0-C5) of one event with its collision log and its escaped list in ascending path
 * code.  For the pins of the decision logic; orc_simulate runs the very same cascade_attempt. */
int orc_cascade_trace(const orc_tables *t, const orc_nucleus *nu, uint64_t seed, uint64_t event, uint32_t attempt,
                      double E_in, int proj, uint32_t flags,
                      int cap_coll, orc_coll_rec *coll, int *n_coll,
                      uint32_t *esc_pi, int32_t *esc_type, double *esc_T, double *esc_p, int *n_esc_out,
                      uint32_t *status) {
  if (!t || !nu || !n_coll || !n_esc_out || (proj != 0 && proj != 1)) return -1;
  rng_ctx g;
  g.key[0] = (uint32_t)seed; g.key[1] = (uint32_t)(seed >> 32);
  g.c2 = (uint32_t)event; g.c3 = (uint32_t)(event >> 32);
  g.st = NULL;
  esc_rec esc[ORC_MAX_SEC];
  int n_esc = 0;
  uint32_t st_try = 0;
  coll_trace trc = {coll, coll ? cap_coll : 0, 0};
  int n_real = cascade_attempt(t, nu, &g, attempt, E_in, proj, flags, esc, &n_esc, &st_try, NULL, &trc);
  qsort(esc, (size_t)n_esc, sizeof(esc_rec), cmp_esc);
  for (int k = 0; k < n_esc; ++k) {
    if (esc_pi) esc_pi[k] = esc[k].pi;
    if (esc_type) esc_type[k] = esc[k].type;
    if (esc_T) esc_T[k] = esc[k].T;
    if (esc_p) { esc_p[3 * k] = esc[k].p[0]; esc_p[3 * k + 1] = esc[k].p[1]; esc_p[3 * k + 2] = esc[k].p[2]; }
  }
  *n_coll = trc.n;
  *n_esc_out = n_esc;
  if (status) *status = st_try;
  return n_real;
}

int64_t orc_simulate(const orc_tables *t, const orc_nucleus *nuc, int n_nuc,
                     int64_t e0, int64_t n, const double *E_in, const int32_t *target,
                     uint64_t seed, uint32_t flags,
                     uint8_t *sec_species, double *sec_T, double *sec_ux, double *sec_uy,
                     double *sec_uz, int64_t cap, int32_t *counts,
                     int32_t *res_A, int32_t *res_Z, double *res_Estar, double *res_px,
                     double *res_py, double *res_pz, uint32_t *status,
                     int32_t *casc_A, int32_t *casc_Z, double *casc_Estar, double *casc_P,
                     int32_t *casc_count, orc_stats *stats, const uint8_t *projectile) {
  if (!t || !nuc || n < 0 || !E_in || !target || !counts) return -1;
  int64_t total = 0;
  if (stats) memset(stats, 0, sizeof(*stats));
  for (int64_t idx = 0; idx < n; ++idx) {
    uint64_t e = (uint64_t)(e0 + idx);
    int tg = target[idx];
    if (tg < 0 || tg >= n_nuc) return -1;
    const orc_nucleus *nu = &nuc[tg];
    double Ein = E_in[idx];
    rng_ctx g;
    g.key[0] = (uint32_t)seed; g.key[1] = (uint32_t)(seed >> 32);
    g.c2 = (uint32_t)e; g.c3 = (uint32_t)(e >> 32);
    g.st = stats;
    if (stats) stats->events++;

    esc_rec esc[ORC_MAX_SEC];
    int n_esc = 0;
    uint32_t st_bits = 0;
    int ok = 0;
    int A_res = nu->A, Z_res = nu->Z;
    double Estar = 0.0, Pres[3] = {0, 0, 0};
    uint32_t attempt = 0;
    const int proj = projectile ? (int)projectile[idx] : 1;      /* NULL: protons (the paper's case, P:9) */
    if (proj != 0 && proj != 1) return -1;
    const double m_in = nucleon_mass(proj);
    double p_in = sqrt(Ein * (Ein + 2.0 * m_in));
    for (attempt = 0; attempt < ORC_MAX_ATTEMPT; ++attempt) {
      if (stats) stats->attempts++;
      uint32_t st_try = 0;
      int n_real = cascade_attempt(t, nu, &g, attempt, Ein, proj, flags, esc, &n_esc, &st_try, stats, NULL);
      /* C6: epilogue — sums in ascending path-code order */
      qsort(esc, (size_t)n_esc, sizeof(esc_rec), cmp_esc);
      int n_p = 0;
      double sumE = 0.0, sumP[3] = {0, 0, 0};
      for (int k = 0; k < n_esc; ++k) {
        n_p += esc[k].type;
        sumE += esc[k].T + nucleon_mass(esc[k].type);
        for (int q = 0; q < 3; ++q) sumP[q] += esc[k].p[q];
      }
      A_res = nu->A + 1 - n_esc;
      Z_res = nu->Z + proj - n_p;
      double Eres = Ein + m_in + nu->M - sumE;
      Pres[0] = -sumP[0]; Pres[1] = -sumP[1]; Pres[2] = p_in - sumP[2];
      int transparent = (n_real == 0);
      if (transparent && !(flags & ORC_F_KEEP_TRANSPARENT)) { if (stats) stats->retry_transparent++; continue; }
      if (!orc_valid_nucleus(A_res, Z_res)) { if (stats) stats->retry_invalid++; continue; }
      double M2 = Eres * Eres - dot3(Pres, Pres);
      double Mstar = M2 > 0.0 ? sqrt(M2) : 0.0;
      Estar = Mstar - orc_mass(A_res, Z_res, t);
      if (Estar < 0.0 && !(transparent && (flags & ORC_F_KEEP_TRANSPARENT))) { if (stats) stats->retry_estar++; continue; }
      st_bits = st_try;
      ok = 1;
      break;
    }
    int count = 0;
    uint8_t sp_loc[ORC_MAX_SEC];
    double T_loc[ORC_MAX_SEC], ux[ORC_MAX_SEC], uy[ORC_MAX_SEC], uz[ORC_MAX_SEC];
    if (!ok) {
      /* FAILED: count 0, residual = target at rest */
      st_bits = ORC_ST_FAILED | 0xFFu;
      if (stats) stats->failed++;
      A_res = nu->A; Z_res = nu->Z; Estar = 0.0; Pres[0] = Pres[1] = Pres[2] = 0.0;
      if (casc_A) { casc_A[idx] = A_res; casc_Z[idx] = Z_res; casc_Estar[idx] = 0.0;
                    casc_P[3 * idx] = casc_P[3 * idx + 1] = casc_P[3 * idx + 2] = 0.0; casc_count[idx] = 0; }
    } else {
      st_bits |= (attempt + 1u > 255u ? 255u : attempt + 1u);   /* attempts used */
      for (int k = 0; k < n_esc; ++k) {
        double pm = sqrt(dot3(esc[k].p, esc[k].p));
        sp_loc[count] = (uint8_t)esc[k].type;
        T_loc[count] = esc[k].T;
        ux[count] = esc[k].p[0] / pm; uy[count] = esc[k].p[1] / pm; uz[count] = esc[k].p[2] / pm;
        count++;
      }
      if (casc_A) { casc_A[idx] = A_res; casc_Z[idx] = Z_res; casc_Estar[idx] = Estar;
                    casc_P[3 * idx] = Pres[0]; casc_P[3 * idx + 1] = Pres[1]; casc_P[3 * idx + 2] = Pres[2];
                    casc_count[idx] = n_esc; }
      /* E: evaporation until the residual cannot emit */
      if (!(flags & ORC_F_CASCADE_ONLY) && Estar > 0.0) {
        uint32_t k = 0;
        uint32_t c1 = (attempt << 24) | 0u;
        for (;;) {
          double W[6], X[6], Q[6], V[6], beta[6], a_d[6];
          double Wsum = orc_evap_widths(A_res, Z_res, Estar, t, W, X, Q, V, beta, a_d);
          if (!(Wsum > 0.0)) break;
          if (count >= ORC_MAX_SEC) { st_bits |= ORC_ST_SEC_TRUNC; if (stats) stats->cap_sec++; break; }
          if (stats) stats->evap_steps++;
          double u[4];
          draw4(&g, attempt, 0u, k++, u);        /* E3: (u_ch, u_cos, u_phi, -) */
          int j = orc_evap_choose(W, Wsum, u[0]);
          int trials = 0;
          double x;
          if (t->version >= 2 && t->level_density == 1) {
            orc_ld ld;
            orc_gem_ld(A_res - EV_A[j], Z_res - EV_Z[j], t, &ld);
            x = orc_evap_sample_x_gem(&ld, X[j], beta[j], g.key, c1, g.c2, g.c3, &k, &trials);
          } else {
            x = orc_evap_sample_x(a_d[j], X[j], beta[j], g.key, c1, g.c2, g.c3, &k, &trials);
          }
          if (stats) { stats->evap_trials += (uint64_t)trials; stats->philox_blocks += (uint64_t)trials; }
          if (x < 0.0) { st_bits |= ORC_ST_TRIAL_CAP; if (stats) stats->cap_trial++; break; }
          double Tej, pej[3], Pd[3];
          orc_evap_emit(A_res, Z_res, Estar, Pres, j, V[j] + x, X[j] - x, u[1], u[2], t, &Tej, pej, Pd);
          double pm = sqrt(dot3(pej, pej));
          sp_loc[count] = (uint8_t)(0x80 | j);
          T_loc[count] = Tej;
          ux[count] = pej[0] / pm; uy[count] = pej[1] / pm; uz[count] = pej[2] / pm;
          count++;
          if (stats) stats->evap_emitted++;
          A_res -= EV_A[j]; Z_res -= EV_Z[j];
          Estar = X[j] - x;
          Pres[0] = Pd[0]; Pres[1] = Pd[1]; Pres[2] = Pd[2];
        }
      }
    }
    /* output */
    if (total + count > cap) return -3;
    for (int k = 0; k < count; ++k) {
      sec_species[total + k] = sp_loc[k];
      sec_T[total + k] = T_loc[k];
      sec_ux[total + k] = ux[k]; sec_uy[total + k] = uy[k]; sec_uz[total + k] = uz[k];
    }
    total += count;
    counts[idx] = count;
    if (res_A) { res_A[idx] = A_res; res_Z[idx] = Z_res; res_Estar[idx] = Estar;
                 res_px[idx] = Pres[0]; res_py[idx] = Pres[1]; res_pz[idx] = Pres[2]; }
    if (status) status[idx] = st_bits;
  }
  return total;
}
