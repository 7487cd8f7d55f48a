// inc_lib.cu — host side of the C ABI declared in include/inc.h.
//
// Built twice: -DINC_REAL_IS_DOUBLE (parity build, -fmad=false) and default (float, production).
// Host work: nuclear setup in fp64, model tables, workspace, kernel launches on the
// caller's stream.  No CPU compute path exists: every compute entry point needs a CUDA device.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <functional>
#include <string>
#include <vector>

#include "inc_device.cuh"

using namespace inc;
typedef INC_REAL real;

namespace {

// ---- constants used by the host setup (standard values, R-K) ----------------------------------
const double kHbarc = 197.3269804, kE2 = 1.43996448;
const double kMp = 938.27208816, kMn = 939.56542052;
const double kPi = 3.14159265358979323846;
const int kEvA[6] = {1, 1, 2, 3, 3, 4};
const int kEvZ[6] = {0, 1, 1, 1, 2, 2};
const double kEvG[6] = {2, 2, 3, 2, 2, 1};

struct HostNucleus {
  bool live = false;
  int A = 0, Z = 0, ns = 0;
  double R = 0, dr = 0, EC = 0, EB_p = 0, EB_n = 0, Bt = 0;
  std::vector<double> r, rho_p, rho_n, pF_p, pF_n, EF_p, EF_n, V_p, V_n;
};

struct TablesHost {
  bool captured = false;
  int n_xs = 0, n_evz = 0, n_shells = 0;
  double plab_max = 0, ws_c0 = 0, ws_delta = 0, ws_rpad = 0, semf[5] = {0, 0, 0, 0, 0};
  double evap_r0 = 0, evap_rj = 0, evap_a_div = 0;
  std::vector<double> sig_pp, sig_np, B_pp, B_np, a_np, ev_Z, ev_kp, ev_cp, ev_ka, ev_ca;
  // version 2 block: level density of the evaporation stage (NEXT-2)
  int level_density = 0;
  double gc_a0 = 0.125, gc_a1 = 0.00917;
  std::vector<double> pair_Z, pair_N, shell_Z, shell_N;
};

struct State {
  cudaStream_t stream = nullptr;
  uint32_t flags = 0;
  TablesHost tab;
  HostNucleus nuc[INC_MAX_TARGETS];
  // device model
  real *d_tabS = nullptr, *d_tabC = nullptr, *d_bind = nullptr;
  EvChan<real> *d_evch = nullptr;
  LdDev<real> *d_ld = nullptr;
  int32_t *d_ldrow = nullptr;       // GEM width tables (level_density = 1)
  GemNode<real> *d_gtab = nullptr;
  NucDev<real> *d_nuc = nullptr;
  DevCounters *d_ctr = nullptr;
  uint32_t *d_wtrace = nullptr; int wtrace_warps = 0;   // inc_get_warp_trace (INC_F_TIMING)
  // workspace.  A lane is what launch_chunk enqueues on: a stream with its workspace, counters and scan buffers.  There
  // is one (the members below on the caller's stream).  A second lane for inc_simulate_host, alternating chunks so that
  // one chunk's cascade kernel would start on the SMs the previous chunk's cascade CTAs have left, was measured and
  // dropped: the evaporation CTAs of the older chunk take those SMs first, and config 2's e2e fell from 2.8e8 to 2.3e8.
  struct Lane {
    cudaStream_t stream = nullptr;
    Workspace<real> ws{};
    DevCounters *ctr = nullptr;
    long long *tiles = nullptr;
    long long *offsets = nullptr;
  };
  Lane *cur = nullptr;              // the lane launch_chunk enqueues on
  size_t ws_chunk = 0;
  Workspace<real> ws{};
  long long *d_offsets = nullptr; size_t offsets_cap = 0;
  long long *d_tiles = nullptr; size_t tiles_cap = 0;
  // host-buffer path (inc_simulate_host): a ring of kRing chunk-sized sets of device buffers, so that device memory
  // is O(chunk) whatever the call's n
  struct HostSlot {
    real *E = nullptr; int32_t *tid = nullptr, *counts = nullptr, *A = nullptr, *Z = nullptr;
    real *Es = nullptr, *px = nullptr, *py = nullptr, *pz = nullptr; uint32_t *status = nullptr;
    uint8_t *sp = nullptr; real *T = nullptr, *ux = nullptr, *uy = nullptr, *uz = nullptr;
    cudaEvent_t computed = nullptr, copied = nullptr;
  };
  static constexpr int kRing = 3;
  struct HostPath {
    size_t chunk_cap = 0;                     // events per slot; a slot holds kMaxSec secondaries per event
    HostSlot slot[kRing];
    cudaStream_t copy_stream = nullptr;
    unsigned long long *h_tot = nullptr;      // pinned, [kRing]: secondaries of the chunk in the slot
    unsigned int *h_err = nullptr;            // pinned: the call's device error word
  } hp;
  size_t host_chunk_events = (size_t)1 << 19;
  // last call
  long long last_n = -1;
  int last_chunks = 0;              // chunks of the last inc_simulate (the cascade stage survives single-chunk calls only)
  bool last_offsets_valid = false;  // inc_get_offsets: the last call left the offsets of the whole call on the device
  long long reruns = 0;             // calls run again: lane kernel after a queue overflow of the wavefront kernel, or a larger pool
  bool ovf_all = false;             // a call has exhausted the staging overflow pool: from then on a row for every event
  long long ovf_rows_user = 0;      // inc_set_stage_overflow_rows (0 = automatic)
  long long last_total = 0;
  long long event_offset = 0;
  // stage timing (INC_F_TIMING)
  cudaEvent_t tev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
  float stage_ms[4] = {0, 0, 0, 0};
  int stage_launches[4] = {0, 0, 0, 0};
  std::vector<cudaEvent_t> pending_events;   // 5 per chunk, resolved after the stream sync
  int vote_coll = 8, vote_epi = 8;
  int long_seg = kLongSegDefault;
  int taper_min = -1;               // inc_set_event_taper (-1 = automatic, 0 = off)
  int seg_per_pass = 0;             // 0 = chosen from the targets
  size_t chunk_events = (size_t)1 << 22;
  const uint8_t *projectile = nullptr;   // DEVICE, caller-owned; nullptr = protons
  int sm_count = 0, smem_max = 0;
  std::string err;
};

State g;

void free_host_ring();

int fail(int code, const std::string &msg) { g.err = msg; return code; }

#define CU_TRY(expr)                                                                           \
  do {                                                                                         \
    cudaError_t _e = (expr);                                                                   \
    if (_e != cudaSuccess)                                                                     \
      return fail(INC_E_CUDA, std::string(#expr) + ": " + cudaGetErrorString(_e));            \
  } while (0)

// ---- mass model ("semi-empirical mass formula"; R-Q4) -------------------------------------
bool valid_nucleus(int A, int Z) {
  if (A < 1 || Z < 0 || Z > A) return false;
  if (A >= 5 || A == 1) return true;
  if (A == 2) return Z == 1;
  if (A == 3) return Z == 1 || Z == 2;
  return Z == 2;
}

double binding(int A, int Z, const TablesHost &t) {
  static const double light[5][3] = {{0, 0, 0}, {0, 0, 0}, {0, 2.224566, 0}, {0, 8.481798, 7.718043}, {0, 0, 28.29566}};
  if (A <= 4) return (A >= 0 && Z >= 0 && Z <= 2) ? light[A][Z] : 0.0;
  const double a = A, z = Z, a13 = std::cbrt(a);
  double B = t.semf[0] * a - t.semf[1] * a13 * a13 - t.semf[2] * z * (z - 1.0) / a13 -
             t.semf[3] * (a - 2.0 * z) * (a - 2.0 * z) / a;
  const bool ze = (Z % 2) == 0, ne = ((A - Z) % 2) == 0;
  if (ze && ne) B += t.semf[4] / std::sqrt(a);
  else if (!ze && !ne) B -= t.semf[4] / std::sqrt(a);
  return B;
}

// Gauss-Legendre nodes on [-1,1] by Newton iteration (for the shell integrals of Eq. (1))
void gauss_legendre(int n, std::vector<double> &x, std::vector<double> &w) {
  x.resize(n); w.resize(n);
  for (int i = 0; i < n; ++i) {
    double z = std::cos(kPi * (i + 0.75) / (n + 0.5)), pp = 1;
    for (int it = 0; it < 100; ++it) {
      double p1 = 1, p2 = 0;
      for (int j = 0; j < n; ++j) { double p3 = p2; p2 = p1; p1 = ((2.0 * j + 1.0) * z * p2 - j * p3) / (j + 1.0); }
      pp = n * (z * p1 - p2) / (z * z - 1.0);
      const double dz = p1 / pp;
      z -= dz;
      if (std::fabs(dz) < 1e-16) break;
    }
    x[i] = z; w[i] = 2.0 / ((1.0 - z * z) * pp * pp);
  }
}

double lerp_z(const std::vector<double> &zz, const std::vector<double> &y, double z) {
  const int n = (int)zz.size();
  if (z <= zz[0]) return y[0];
  if (z >= zz[n - 1]) return y[n - 1];
  int k = 0;
  while (k < n - 2 && z > zz[k + 1]) ++k;
  return y[k] + (z - zz[k]) / (zz[k + 1] - zz[k]) * (y[k + 1] - y[k]);
}

int setup_nucleus(int A, int Z, const TablesHost &t, HostNucleus &nu) {
  const int ns = t.n_shells;
  nu.A = A; nu.Z = Z; nu.ns = ns;
  const double c = t.ws_c0 * std::cbrt((double)A);
  nu.R = c + t.ws_rpad;
  nu.dr = nu.R / ns;
  nu.r.resize(ns + 1);
  for (int i = 0; i <= ns; ++i) nu.r[i] = i * nu.dr;
  // shell weights w_i = int rho(r) r^2 dr by 8 panels of 16-point Gauss-Legendre (R-N2: volume average)
  std::vector<double> gx, gw, w(ns);
  gauss_legendre(16, gx, gw);
  double wsum = 0;
  for (int i = 0; i < ns; ++i) {
    double acc = 0;
    const int NP = 8;
    const double h = (nu.r[i + 1] - nu.r[i]) / NP;
    for (int p = 0; p < NP; ++p) {
      const double a = nu.r[i] + p * h;
      for (int q = 0; q < 16; ++q) {
        const double r = a + 0.5 * h * (gx[q] + 1.0);
        acc += 0.5 * h * gw[q] * r * r / (1.0 + std::exp((r - c) / t.ws_delta));   // Eq. (1)
      }
    }
    w[i] = acc; wsum += acc;
  }
  const double N = A - Z;
  auto vec = [&](std::vector<double> &v, int n) { v.assign(n, 0.0); };
  vec(nu.rho_p, ns); vec(nu.rho_n, ns); vec(nu.pF_p, ns); vec(nu.pF_n, ns);
  vec(nu.EF_p, ns); vec(nu.EF_n, ns); vec(nu.V_p, ns + 1); vec(nu.V_n, ns + 1);
  nu.Bt = binding(A, Z, t);
  nu.EB_p = nu.Bt - binding(A - 1, Z - 1, t);             // R-N4 separation energies
  nu.EB_n = nu.Bt - binding(A - 1, Z, t);
  for (int i = 0; i < ns; ++i) {
    const double vol = (nu.r[i + 1] * nu.r[i + 1] * nu.r[i + 1] - nu.r[i] * nu.r[i] * nu.r[i]) / 3.0;  // /4pi
    const double rho = A * w[i] / (vol * wsum) / (4.0 * kPi);
    nu.rho_p[i] = rho * Z / A; nu.rho_n[i] = rho * N / A;
    nu.pF_p[i] = kHbarc * std::cbrt(3.0 * kPi * kPi * nu.rho_p[i]);   // R-N3
    nu.pF_n[i] = kHbarc * std::cbrt(3.0 * kPi * kPi * nu.rho_n[i]);
    nu.EF_p[i] = std::sqrt(nu.pF_p[i] * nu.pF_p[i] + kMp * kMp) - kMp;
    nu.EF_n[i] = std::sqrt(nu.pF_n[i] * nu.pF_n[i] + kMn * kMn) - kMn;
    nu.V_p[i] = nu.EF_p[i] + nu.EB_p;                      // P:45  V = E_F + E_B
    nu.V_n[i] = nu.EF_n[i] + nu.EB_n;
  }
  nu.EC = kE2 * Z / nu.R;                                  // R-N6
  nu.live = true;
  return 0;
}

void fill_nucdev(const HostNucleus &h, NucDev<real> &d) {
  std::memset(&d, 0, sizeof(d));
  d.A = h.A; d.Z = h.Z; d.ns = h.ns; d.live = 1;
  d.Rn = (real)h.R; d.dr = (real)h.dr; d.Bt = (real)h.Bt; d.iRn = (real)(1.0 / h.R);
  for (int i = 0; i <= h.ns; ++i) {
    ShellDev<real> &s = d.sh[i];
    if (i < h.ns) {
      s.r_in = (real)h.r[i]; s.r_out = (real)h.r[i + 1];
      s.ir_in = i > 0 ? (real)(1.0 / h.r[i]) : (real)0; s.ir_out = (real)(1.0 / h.r[i + 1]);
      s.rho_p = (real)h.rho_p[i]; s.rho_n = (real)h.rho_n[i];
      s.pF_p = (real)h.pF_p[i]; s.pF_n = (real)h.pF_n[i];
      s.pF2_p = (real)(h.pF_p[i] * h.pF_p[i]); s.pF2_n = (real)(h.pF_n[i] * h.pF_n[i]);
      const double tp = h.V_p[i] + h.EC, tn = h.V_n[i];    // cutoff kinetic energies
      s.pc2_p = (real)(tp * (tp + 2.0 * kMp)); s.pc2_n = (real)(tn * (tn + 2.0 * kMn));
      s.V_p = (real)h.V_p[i]; s.V_n = (real)h.V_n[i];
    }
  }
}

int check_tables(const inc_tables *t) {
  if (!t) return fail(INC_E_BADARG, "tables is NULL");
  if (t->version != 1 && t->version != 2) return fail(INC_E_TABLES, "tables.version must be 1 or 2");
  if (t->version >= 2) {
    if (t->level_density != 0 && t->level_density != 1) return fail(INC_E_TABLES, "level_density must be 0 or 1");
    if (t->n_ldZ < 0 || t->n_ldN < 0 || t->n_ldZ > 4096 || t->n_ldN > 4096) return fail(INC_E_TABLES, "bad level-density array length");
    if ((t->n_ldZ > 0 && (!t->pair_Z || !t->shell_Z)) || (t->n_ldN > 0 && (!t->pair_N || !t->shell_N)))
      return fail(INC_E_TABLES, "NULL level-density array");
    for (int i = 0; i < t->n_ldZ; ++i) if (!std::isfinite(t->pair_Z[i]) || !std::isfinite(t->shell_Z[i])) return fail(INC_E_TABLES, "NaN in pair_Z / shell_Z");
    for (int i = 0; i < t->n_ldN; ++i) if (!std::isfinite(t->pair_N[i]) || !std::isfinite(t->shell_N[i])) return fail(INC_E_TABLES, "NaN in pair_N / shell_N");
    if (t->level_density == 1 && !(t->gc_a0 > 0)) return fail(INC_E_TABLES, "gc_a0 must be positive");
  }
  if (t->n_xs < 2 || t->n_xs > 4096 || !(t->plab_max > 0)) return fail(INC_E_TABLES, "bad NN grid");
  if (!t->sig_pp || !t->sig_np || !t->B_pp || !t->B_np || !t->a_np) return fail(INC_E_TABLES, "NULL NN table");
  if (t->n_evz < 1 || t->n_evz > 16 || !t->ev_Z || !t->ev_kp || !t->ev_cp || !t->ev_ka || !t->ev_ca)
    return fail(INC_E_TABLES, "bad evaporation table");
  for (int i = 1; i < t->n_evz; ++i)
    if (!(t->ev_Z[i] > t->ev_Z[i - 1])) return fail(INC_E_TABLES, "ev_Z grid not increasing");
  if (t->n_shells < 1 || t->n_shells > kMaxShells) return fail(INC_E_TABLES, "n_shells outside 1..32");
  if (!(t->ws_delta > 0) || !(t->ws_c0 > 0) || !(t->ws_rpad >= 0) || !(t->evap_a_div > 0) || !(t->evap_r0 > 0))
    return fail(INC_E_TABLES, "bad scalar model constant");
  for (int i = 0; i < t->n_xs; ++i)
    if (!(t->sig_pp[i] >= 0) || !(t->sig_np[i] >= 0) || !(t->B_pp[i] >= 0) || !(t->B_np[i] >= 0) || !(t->a_np[i] >= 0))
      return fail(INC_E_TABLES, "negative or NaN NN table entry");
  return 0;
}

void copy_tables(const inc_tables *t, TablesHost &h) {
  h.n_xs = t->n_xs; h.n_evz = t->n_evz; h.n_shells = t->n_shells; h.plab_max = t->plab_max;
  h.ws_c0 = t->ws_c0; h.ws_delta = t->ws_delta; h.ws_rpad = t->ws_rpad;
  for (int i = 0; i < 5; ++i) h.semf[i] = t->semf[i];
  h.evap_r0 = t->evap_r0; h.evap_rj = t->evap_rj; h.evap_a_div = t->evap_a_div;
  auto cp = [](std::vector<double> &v, const double *p, int n) { v.assign(p, p + n); };
  cp(h.sig_pp, t->sig_pp, t->n_xs); cp(h.sig_np, t->sig_np, t->n_xs); cp(h.B_pp, t->B_pp, t->n_xs);
  cp(h.B_np, t->B_np, t->n_xs); cp(h.a_np, t->a_np, t->n_xs);
  cp(h.ev_Z, t->ev_Z, t->n_evz); cp(h.ev_kp, t->ev_kp, t->n_evz); cp(h.ev_cp, t->ev_cp, t->n_evz);
  cp(h.ev_ka, t->ev_ka, t->n_evz); cp(h.ev_ca, t->ev_ca, t->n_evz);
  h.level_density = 0; h.gc_a0 = 0.125; h.gc_a1 = 0.00917;
  h.pair_Z.clear(); h.pair_N.clear(); h.shell_Z.clear(); h.shell_N.clear();
  if (t->version >= 2) {
    h.level_density = t->level_density; h.gc_a0 = t->gc_a0; h.gc_a1 = t->gc_a1;
    cp(h.pair_Z, t->pair_Z, t->n_ldZ); cp(h.shell_Z, t->shell_Z, t->n_ldZ);
    cp(h.pair_N, t->pair_N, t->n_ldN); cp(h.shell_N, t->shell_N, t->n_ldN);
  }
  h.captured = true;
}

bool same_tables(const inc_tables *t, const TablesHost &h) {
  if (t->n_xs != h.n_xs || t->n_evz != h.n_evz || t->n_shells != h.n_shells || t->plab_max != h.plab_max) return false;
  if (t->ws_c0 != h.ws_c0 || t->ws_delta != h.ws_delta || t->ws_rpad != h.ws_rpad) return false;
  if (t->evap_r0 != h.evap_r0 || t->evap_rj != h.evap_rj || t->evap_a_div != h.evap_a_div) return false;
  for (int i = 0; i < 5; ++i) if (t->semf[i] != h.semf[i]) return false;
  auto eq = [](const std::vector<double> &v, const double *p) { return v.empty() || std::memcmp(v.data(), p, v.size() * sizeof(double)) == 0; };
  {
    // version 2 block (a version 1 struct means: level_density 0, no arrays)
    const int ld = t->version >= 2 ? t->level_density : 0;
    if (ld != h.level_density) return false;
    if (t->version >= 2) {
      if (t->gc_a0 != h.gc_a0 || t->gc_a1 != h.gc_a1) return false;
      if ((size_t)t->n_ldZ != h.pair_Z.size() || (size_t)t->n_ldN != h.pair_N.size()) return false;
      if (!eq(h.pair_Z, t->pair_Z) || !eq(h.shell_Z, t->shell_Z) || !eq(h.pair_N, t->pair_N) || !eq(h.shell_N, t->shell_N)) return false;
    } else if (!h.pair_Z.empty() || !h.pair_N.empty()) return false;
  }
  return eq(h.sig_pp, t->sig_pp) && eq(h.sig_np, t->sig_np) && eq(h.B_pp, t->B_pp) && eq(h.B_np, t->B_np) &&
         eq(h.a_np, t->a_np) && eq(h.ev_Z, t->ev_Z) && eq(h.ev_kp, t->ev_kp) && eq(h.ev_cp, t->ev_cp) &&
         eq(h.ev_ka, t->ev_ka) && eq(h.ev_ca, t->ev_ca);
}

int upload_model() {
  const TablesHost &t = g.tab;
  const int n = t.n_xs;
  std::vector<real> S(4 * (size_t)n), Cc(8 * (size_t)n);
  for (int k = 0; k < n; ++k) {
    const int k1 = k + 1 < n ? k + 1 : k;
    // mb -> fm^2 folded in; slopes stored so that a lookup is y + f * dy (R-N7)
    S[4 * k + 0] = (real)(t.sig_pp[k] * 0.1); S[4 * k + 1] = (real)(t.sig_pp[k1] * 0.1) - (real)(t.sig_pp[k] * 0.1);
    S[4 * k + 2] = (real)(t.sig_np[k] * 0.1); S[4 * k + 3] = (real)(t.sig_np[k1] * 0.1) - (real)(t.sig_np[k] * 0.1);
    Cc[8 * k + 0] = (real)t.B_pp[k]; Cc[8 * k + 1] = (real)t.B_pp[k1] - (real)t.B_pp[k];
    Cc[8 * k + 2] = (real)t.B_np[k]; Cc[8 * k + 3] = (real)t.B_np[k1] - (real)t.B_np[k];
    Cc[8 * k + 4] = (real)t.a_np[k]; Cc[8 * k + 5] = (real)t.a_np[k1] - (real)t.a_np[k];
    Cc[8 * k + 6] = 0; Cc[8 * k + 7] = 0;
  }
  std::vector<real> bind((size_t)kAmax * kZmax, (real)-1e30);
  std::vector<EvChan<real>> ev((size_t)kAmax * kZmax * 6);
  std::memset(ev.data(), 0, ev.size() * sizeof(EvChan<real>));
  for (int A = 1; A < kAmax; ++A)
    for (int Z = 0; Z < kZmax && Z <= A; ++Z)
      if (valid_nucleus(A, Z)) bind[(size_t)A * kZmax + Z] = (real)binding(A, Z, t);
  for (int Ad = 1; Ad < kAmax; ++Ad)
    for (int Zd = 0; Zd < kZmax && Zd <= Ad; ++Zd) {
      if (!valid_nucleus(Ad, Zd)) continue;
      const double Bd = binding(Ad, Zd, t), ad13 = std::cbrt((double)Ad);
      for (int j = 0; j < 6; ++j) {
        const double Bj = binding(kEvA[j], kEvZ[j], t);
        const double Mj = kEvZ[j] * kMp + (kEvA[j] - kEvZ[j]) * kMn - Bj;
        double alpha, beta = 0, V = 0;
        if (j == 0) {                                          // Dostrovsky neutron (R-E1)
          alpha = 0.76 + 2.2 / ad13;
          beta = (2.12 / (ad13 * ad13) - 0.05) / alpha;
        } else {
          const double kp = lerp_z(t.ev_Z, t.ev_kp, Zd), cp = lerp_z(t.ev_Z, t.ev_cp, Zd);
          const double ka = lerp_z(t.ev_Z, t.ev_ka, Zd), ca = lerp_z(t.ev_Z, t.ev_ca, Zd);
          double k, c, rj = t.evap_rj;
          if (j == 1) { k = kp; c = cp; rj = 0; }
          else if (j == 2) { k = kp + 0.06; c = cp / 2; }
          else if (j == 3) { k = kp + 0.12; c = cp / 3; }
          else if (j == 4) { k = ka - 0.06; c = 4 * ca / 3; }
          else { k = ka; c = ca; }
          alpha = 1 + c;
          V = k * kE2 * kEvZ[j] * Zd / (t.evap_r0 * ad13 + rj);
        }
        EvChan<real> &e = ev[((size_t)Ad * kZmax + Zd) * 6 + j];
        e.V = (real)V; e.pref = (real)(kEvG[j] * Mj * ad13 * ad13 * alpha); e.beta = (real)beta; e.BdBj = (real)(Bd + Bj);
      }
    }
  // NEXT-2: level-density constants per daughter nucleus (R-G2..G4) and the 16 Gauss-Legendre nodes of the width integral
  std::vector<LdDev<real>> ldv((size_t)kAmax * kZmax);
  std::memset(ldv.data(), 0, ldv.size() * sizeof(LdDev<real>));
  if (t.level_density == 1) {
    auto tab = [](const std::vector<double> &y, int i) { return (i >= 0 && i < (int)y.size()) ? y[i] : 0.0; };
    for (int Ad = 1; Ad < kAmax; ++Ad)
      for (int Zd = 0; Zd < kZmax && Zd <= Ad; ++Zd) {
        if (!valid_nucleus(Ad, Zd)) continue;
        const int Nd = Ad - Zd;
        const double S = tab(t.shell_Z, Zd) + tab(t.shell_N, Nd);
        const double a = (double)Ad * (t.gc_a0 + t.gc_a1 * S);                      // R-G2
        const double delta = tab(t.pair_Z, Zd) + tab(t.pair_N, Nd);                 // R-G3
        const double Ux = 150.0 / (double)Ad + 2.5;                                 // R-G4
        LdDev<real> &d = ldv[(size_t)Ad * kZmax + Zd];
        if (!(a > 0.0)) continue;                                                   // a = 0 in the table: channel closed
        const double Ex = Ux + delta;
        const double invT = std::sqrt(a / Ux) - 1.5 / Ux;
        if (!(invT > 0.0)) continue;                                                // R-G7: no constant-temperature branch: closed as well
        const double T = 1.0 / invT;
        const double E0 = Ex - T * (std::log(T) - 0.25 * std::log(a) - 1.25 * std::log(Ux) + 2.0 * std::sqrt(a * Ux));
        d.a = (real)a; d.delta = (real)delta; d.Ux = (real)Ux; d.Ex = (real)Ex; d.T = (real)T; d.E0 = (real)E0;
        d.lnT = (real)std::log(T); d.lna4 = (real)(0.25 * std::log(a));
      }
    std::vector<double> gx, gw;
    gauss_legendre(16, gx, gw);
    // R-G5 tables: J0(X) = int_0^X rho, J1(X) = int_0^X (X - U) rho(U) dU per daughter nucleus, X = E_x + k h.  Below E_x the
    // density is the constant-temperature form and both are elementary (the kernel evaluates them directly); from E_x on
    // they are accumulated interval by interval with the 16-point rule on the Fermi-gas density:
    //   J0(X + h) = J0(X) + int_X^{X+h} rho,   J1(X + h) = J1(X) + h J0(X) + int_X^{X+h} (X + h - U) rho(U) dU.
    // The kernel interpolates ln J0 and ln J1 (cubic Hermite with the exact derivatives rho / J0 and J0 / J1).
    {
      std::vector<int32_t> ldrow((size_t)kAmax * kZmax, -1);
      int rows = 0;
      for (size_t i = 0; i < ldv.size(); ++i) if (ldv[i].a > (real)0) ldrow[i] = rows++;
      std::vector<GemNode<real>> gt((size_t)(rows > 0 ? rows : 1) * kGemPoints);
      const double h = INC_GEM_STEP;
      auto tab = [](const std::vector<double> &y, int i) { return (i >= 0 && i < (int)y.size()) ? y[i] : 0.0; };
      for (int Ad = 1; Ad < kAmax; ++Ad)
        for (int Zd = 0; Zd < kZmax && Zd <= Ad; ++Zd) {
          const int r = ldrow[(size_t)Ad * kZmax + Zd];
          if (r < 0) continue;
          // (the constants again in double: the table must not inherit the f32 rounding of LdDev)
          const double S = tab(t.shell_Z, Zd) + tab(t.shell_N, Ad - Zd);
          const double a = (double)Ad * (t.gc_a0 + t.gc_a1 * S), delta = tab(t.pair_Z, Zd) + tab(t.pair_N, Ad - Zd);
          const double Ux = 150.0 / (double)Ad + 2.5, Ex = Ux + delta;
          const double T = 1.0 / (std::sqrt(a / Ux) - 1.5 / Ux);
          const double E0 = Ex - T * (std::log(T) - 0.25 * std::log(a) - 1.25 * std::log(Ux) + 2.0 * std::sqrt(a * Ux));
          auto lnrho_fg = [&](double U) { const double u = U - delta; return 2.0 * std::sqrt(a * u) - 0.25 * std::log(a) - 1.25 * std::log(u); };
          // at E_x from the constant-temperature forms (E_x <= 0 can happen with negative pairing inputs: start from 0)
          double X = Ex, J0, J1;
          if (Ex > 0.0) {
            const double z = Ex / T, c = std::exp(-E0 / T);
            J0 = c * std::expm1(z);
            J1 = c * T * (std::expm1(z) - z);
          } else { X = 0.0; J0 = 0.0; J1 = 0.0; }
          // scaled by e^{-ref} to stay in range whatever the inputs: ref follows the running maximum of ln rho
          GemNode<real> *row = &gt[(size_t)r * kGemPoints];
          double ref = 0.0;                       // J0, J1 hold the true values times e^{-ref}
          for (int k = 0; k < kGemPoints; ++k) {
            const double Xk = X + k * h;
            if (k > 0) {
              const double Xa = Xk - h;
              double A0 = 0, A1 = 0;
              const double lr = lnrho_fg(Xk > delta + 1e-9 ? Xk : delta + 1e-9);
              const double nref = lr > ref ? lr : ref;
              const double sc = std::exp(ref - nref);
              J0 *= sc; J1 *= sc; ref = nref;
              for (int q = 0; q < 16; ++q) {
                const double U = Xa + 0.5 * h * (gx[q] + 1.0);
                const double u = U - delta;
                const double rho = u > 0.0 ? std::exp(lnrho_fg(U) - ref) : 0.0;
                A0 += 0.5 * h * gw[q] * rho;
                A1 += 0.5 * h * gw[q] * (Xk - U) * rho;
              }
              J1 += h * J0 + A1;
              J0 += A0;
            }
            const double rhoX = Xk >= Ex ? ((Xk - delta) > 0.0 ? std::exp(lnrho_fg(Xk) - ref) : 0.0) : std::exp((Xk - E0) / T - std::log(T) - ref);
            const bool ok = J0 > 0.0 && J1 > 0.0;
            row[k].l0 = (real)(ok ? std::log(J0) + ref : -1e30);
            row[k].l1 = (real)(ok ? std::log(J1) + ref : -1e30);
            row[k].d0 = (real)(ok ? rhoX / J0 : 0.0);
            row[k].d1 = (real)(ok ? J0 / J1 : 0.0);
          }
        }
      auto up2 = [&](void **dst, const void *src, size_t bytes) -> cudaError_t {
        if (*dst) cudaFree(*dst);
        cudaError_t e = cudaMalloc(dst, bytes);
        if (e != cudaSuccess) return e;
        return cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice);
      };
      CU_TRY(up2((void **)&g.d_ldrow, ldrow.data(), ldrow.size() * sizeof(int32_t)));
      CU_TRY(up2((void **)&g.d_gtab, gt.data(), gt.size() * sizeof(GemNode<real>)));
    }
    // (nodes in the order of the Newton start values cos(pi (i + 3/4) / 16.5), i = 0..15, so that a panel sum runs in one fixed order)
    GaussNodes<real> gn;
    for (int i = 0; i < 16; ++i) { gn.x[i] = (real)gx[i]; gn.w[i] = (real)gw[i]; }
    CU_TRY(cudaMemcpyToSymbol(c_gl, &gn, sizeof(gn)));
  }
  auto up = [&](void **dst, const void *src, size_t bytes) -> cudaError_t {
    if (*dst) cudaFree(*dst);
    cudaError_t e = cudaMalloc(dst, bytes);
    if (e != cudaSuccess) return e;
    return cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice);
  };
  CU_TRY(up((void **)&g.d_tabS, S.data(), S.size() * sizeof(real)));
  CU_TRY(up((void **)&g.d_tabC, Cc.data(), Cc.size() * sizeof(real)));
  CU_TRY(up((void **)&g.d_bind, bind.data(), bind.size() * sizeof(real)));
  // the channel constants re-indexed by parent nucleus, eight entries (128 bytes in f32) per parent
  std::vector<EvChan<real>> evp((size_t)kAmax * kZmax * 8);
  std::memset(evp.data(), 0, evp.size() * sizeof(EvChan<real>));
  for (int A = 1; A < kAmax; ++A)
    for (int Z = 0; Z < kZmax && Z <= A; ++Z) {
      EvChan<real> *row = &evp[((size_t)A * kZmax + Z) * 8];
      for (int j = 0; j < 6; ++j) {
        const int Ad = A - kEvA[j], Zd = Z - kEvZ[j];
        if (Ad >= 1 && Zd >= 0 && Zd <= Ad && Zd < kZmax) row[j] = ev[((size_t)Ad * kZmax + Zd) * 6 + j];
      }
      row[6].V = bind[(size_t)A * kZmax + Z];
    }
  CU_TRY(up((void **)&g.d_evch, evp.data(), evp.size() * sizeof(EvChan<real>)));
  CU_TRY(up((void **)&g.d_ld, ldv.data(), ldv.size() * sizeof(LdDev<real>)));
  if (!g.d_nuc) {
    CU_TRY(cudaMalloc((void **)&g.d_nuc, sizeof(NucDev<real>) * INC_MAX_TARGETS));
    CU_TRY(cudaMemset(g.d_nuc, 0, sizeof(NucDev<real>) * INC_MAX_TARGETS));
  }
  if (!g.d_ctr) CU_TRY(cudaMalloc((void **)&g.d_ctr, sizeof(DevCounters)));
  int dev = 0;
  CU_TRY(cudaGetDevice(&dev));
  CU_TRY(cudaDeviceGetAttribute(&g.sm_count, cudaDevAttrMultiProcessorCount, dev));
  CU_TRY(cudaDeviceGetAttribute(&g.smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
  return 0;
}

ModelDev<real> model_dev() {
  ModelDev<real> m;
  m.tabS = g.d_tabS; m.tabC = g.d_tabC; m.bind = g.d_bind; m.evp = g.d_evch; m.nuc = g.d_nuc; m.ld = g.d_ld; m.ldrow = g.d_ldrow; m.gtab = g.d_gtab;
  m.n_xs = g.tab.n_xs;
  m.inv_dp = (real)(1.0 / (g.tab.plab_max / (g.tab.n_xs - 1) * 1000.0));
  m.a_div = (real)g.tab.evap_a_div;
  return m;
}

void free_ws() {
  void **p[] = {(void **)&g.ws.st, (void **)&g.ws.ovf, (void **)&g.ws.ovf_id, (void **)&g.ws.crec, (void **)&g.ws.frec, (void **)&g.ws.done_list};
  g.ws.ovf_rows = 0;
  for (auto q : p) { if (*q) cudaFree(*q); *q = nullptr; }
  g.ws_chunk = 0;
}

int ensure_ws(size_t chunk, size_t n_total) {
  // overflow pool of the staging rows: a row for one event in 64 (at least 4096 rows; none of 6e4 250 MeV p-48Ti events
  // has more than 16 secondaries); for every event once a call has
  // exhausted the pool (g.ovf_all), or what the caller says (inc_set_stage_overflow_rows)
  auto rows_for = [&](size_t c) -> size_t {
    size_t r = g.ovf_rows_user > 0 ? (size_t)g.ovf_rows_user : (g.ovf_all ? c : (c / 64 > 4096 ? c / 64 : 4096));
    if (r > c) r = c;
    return r < 1 ? 1 : r;
  };
  const size_t ws_c = chunk > g.ws_chunk ? chunk : g.ws_chunk;
  const bool rows_bad = g.ovf_rows_user > 0 ? (size_t)g.ws.ovf_rows != rows_for(ws_c) : (size_t)g.ws.ovf_rows < rows_for(chunk);
  if (chunk > g.ws_chunk || rows_bad) {
    free_ws();
    chunk = ws_c;
    const size_t want_rows = rows_for(chunk);
    const size_t ns = chunk * kStageMain;
    CU_TRY(cudaMalloc((void **)&g.ws.st, ns * sizeof(StageRec<real>)));
    CU_TRY(cudaMalloc((void **)&g.ws.ovf, want_rows * kStageOvf * sizeof(StageRec<real>)));
    CU_TRY(cudaMalloc((void **)&g.ws.ovf_id, chunk * sizeof(int32_t)));
    g.ws.ovf_rows = (int32_t)want_rows;
    CU_TRY(cudaMalloc((void **)&g.ws.crec, chunk * sizeof(NucRec<real>)));
    CU_TRY(cudaMalloc((void **)&g.ws.frec, chunk * sizeof(NucRec<real>)));
    CU_TRY(cudaMalloc((void **)&g.ws.done_list, chunk * sizeof(uint32_t)));
    g.ws_chunk = chunk;
  }
  if (n_total + 1 > g.offsets_cap) {
    if (g.d_offsets) cudaFree(g.d_offsets);
    g.d_offsets = nullptr;
    CU_TRY(cudaMalloc((void **)&g.d_offsets, (n_total + 1) * sizeof(long long)));
    g.offsets_cap = n_total + 1;
  }
  const size_t tiles = (chunk + kScanTile - 1) / kScanTile + 1;
  if (tiles > g.tiles_cap) {
    if (g.d_tiles) cudaFree(g.d_tiles);
    g.d_tiles = nullptr;
    CU_TRY(cudaMalloc((void **)&g.d_tiles, tiles * sizeof(long long)));
    g.tiles_cap = tiles;
  }
  return 0;
}

// lane 0 = the library's main workspace on the caller's stream
State::Lane lane0() {
  State::Lane l;
  l.stream = g.stream; l.ws = g.ws; l.ctr = g.d_ctr; l.tiles = g.d_tiles; l.offsets = g.d_offsets;
  return l;
}

// Launch shapes are queried once per (kernel, block size, dynamic shared memory): the attribute and occupancy calls cost
// microseconds each, and they sit between two steps of a caller's loop, when the GPU has nothing to do.
struct LaunchShape { const void *kern; int threads; size_t smem; int occ; };
std::vector<LaunchShape> g_shapes;

int launch_shape(const void *kern, int threads, size_t smem, int *occ) {
  for (const auto &sh : g_shapes)
    if (sh.kern == kern && sh.threads == threads && sh.smem == smem) { *occ = sh.occ; return 0; }
  // the dynamic shared-memory limit is per kernel: it only ever grows (a launch needs limit >= its size)
  size_t limit = 0;
  for (const auto &sh : g_shapes) if (sh.kern == kern && sh.smem > limit) limit = sh.smem;
  if (smem > limit) CU_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int o = 0;
  CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, kern, threads, smem));
  g_shapes.push_back(LaunchShape{kern, threads, smem, o});
  *occ = o;
  return 0;
}

int mark(bool timing) {
  if (!timing) return 0;
  cudaEvent_t e;
  CU_TRY(cudaEventCreate(&e));
  CU_TRY(cudaEventRecord(e, g.cur->stream));
  g.pending_events.push_back(e);
  return 0;
}

// R-R1: the ten round keys of the call's seed, to constant memory (ordered on the stream like everything else)
int set_round_keys(uint64_t seed) {
  RoundKeys rk;
  uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
  for (int r = 0; r < 10; ++r) { rk.k0[r] = k0; rk.k1[r] = k1; k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
  CU_TRY(cudaMemcpyToSymbolAsync(c_rk, &rk, sizeof(rk), 0, cudaMemcpyHostToDevice, g.stream));
  return 0;
}

template <bool STATS>
int launch_chunk(long long e_base, int n_chunk, const real *E_in, const int32_t *tid, const uint8_t *proj, uint64_t seed,
                 inc_secondaries *sec, int32_t *counts, inc_residual *res, long long *offsets) {
  const ModelDev<real> model = model_dev();
  State::Lane &L = *g.cur;
  // --- cascade ---
  CascadeParams<real> cp;
  cp.model = model; cp.ws = L.ws; cp.ctr = L.ctr; cp.E_in = E_in; cp.target_id = tid; cp.projectile = proj;
  cp.e_base = e_base + g.event_offset; cp.n_chunk = n_chunk; cp.seed_lo = (uint32_t)seed; cp.seed_hi = (uint32_t)(seed >> 32);
  cp.flags = g.flags;
  const bool naive = (g.flags & INC_F_LANE_PER_EVENT) != 0;
  cp.vote_coll = naive ? 1 : g.vote_coll; cp.vote_epi = naive ? 1 : g.vote_epi;
  cp.long_seg = g.long_seg;
  // event taper: automatic = 8 events per warp for a chunk smaller than the grid's slot count, where it spreads the batch
  // over all SMs (config 1, 1e4 events: 0.51 -> 0.44 ms); off for large chunks, where it was measured to change nothing
  // (the tail of a large chunk is the chain of attempts of its last events, not events queueing in a few warps)
  const int taper = g.taper_min >= 0 ? g.taper_min : (n_chunk < 100000 ? 8 : 0);
  cp.taper_min = taper;
  {
    // segment steps per pass of the wavefront kernel: three pay while collisions are rare (light targets), two otherwise
    int a_max = 0;
    for (int i = 0; i < INC_MAX_TARGETS; ++i) if (g.nuc[i].live && g.nuc[i].A > a_max) a_max = g.nuc[i].A;
    cp.seg_per_pass = g.seg_per_pass > 0 ? g.seg_per_pass : (a_max <= 20 ? 3 : 2);
  }
  cp.wtrace = nullptr;
  int n_stage = 0;
  for (int i = 0; i < INC_MAX_TARGETS; ++i) if (g.nuc[i].live) n_stage = i + 1;
  cp.n_stage = n_stage;
  // staged nucleus records: 15 shells (+ the outside) when the tables have at most 15, as the paper's have; else all 32
  const bool wide = g.tab.n_shells > 15;
  cp.nuc_stride = nuc_stride_bytes<real>(wide ? kMaxShells : 15);
  const bool timing = (g.flags & INC_F_TIMING) != 0;
  const int need = (n_chunk + 255) / 256;
  const int smem_max = g.smem_max;
  const size_t wsmem = wave_smem_bytes<real>(model.n_xs, n_stage, wide ? kMaxShells : 15);
  const bool lane_kernel = naive || (g.flags & INC_F_LANE_STATE_MACHINE) != 0 || wsmem > (size_t)smem_max;
  CU_TRY(cudaMemsetAsync(&L.ctr->next_event_casc, 0, 4 * sizeof(unsigned long long), L.stream));   // + next_event_evap, n_done, ovf_next
  CU_TRY(cudaMemsetAsync(L.ws.ovf_id, 0xFF, (size_t)n_chunk * sizeof(int32_t), L.stream));         // -1: no overflow row
  CU_TRY(cudaMemsetAsync(L.ws.done_list, 0xFF, (size_t)n_chunk * sizeof(uint32_t), L.stream));      // kNotDone
  // the evaporation kernel writes the count of every event it finishes; if the cascade kernel gives up (queue overflow,
  // watchdog, failed index check) the events it abandoned are never finished, and the scan and the compaction, which are
  // enqueued all the same, must find zeros there rather than whatever the caller's buffer held
  CU_TRY(cudaMemsetAsync(counts, 0, (size_t)n_chunk * sizeof(int32_t), L.stream));
  if (mark(timing)) return INC_E_CUDA;
  if (lane_kernel) {
    const size_t smem = model_smem_bytes<real>(model.n_xs, n_stage, wide ? kMaxShells : 15);
    auto kern = cascade_lane_kernel<real, STATS>;
    int occ = 0;
    if (int lr = launch_shape((const void *)kern, 256, smem, &occ)) return lr;
    if (occ < 1) return fail(INC_E_CUDA, "cascade kernel does not fit on an SM");
    int blocks = occ * g.sm_count;
    if (blocks > need) blocks = need;
    kern<<<blocks, 256, smem, L.stream>>>(cp);
  } else {
    // one persistent CTA per SM; each warp keeps WaveCfg::NS events in flight in its shared-memory queues
    auto kern = wide ? cascade_wavefront_kernel<real, STATS, kMaxShells> : cascade_wavefront_kernel<real, STATS, 15>;
    const int threads = WaveCfg<real>::WARPS * 32;
    int occ = 0;
    if (int lr = launch_shape((const void *)kern, threads, wsmem, &occ)) return lr;
    if (occ < 1) return fail(INC_E_CUDA, "wavefront cascade kernel does not fit on an SM");
    int blocks = occ * g.sm_count;
    // a small batch: 32 events per warp -- or, with the taper, its minimum per warp, so that the batch is spread over
    // more SMs (the kernel is latency-bound per warp: fewer events per warp finish sooner)
    const int per_cta = WaveCfg<real>::WARPS * (taper > 0 ? taper : 32);
    const int wneed = (n_chunk + per_cta - 1) / per_cta;
    if (blocks > wneed) blocks = wneed;
    cp.wtrace = nullptr;
    if (timing) {
      const int nw = blocks * WaveCfg<real>::WARPS;
      if (!g.d_wtrace) CU_TRY(cudaMalloc((void **)&g.d_wtrace, sizeof(uint32_t) * kWTrace * 8192));
      if (nw <= 8192) { CU_TRY(cudaMemsetAsync(g.d_wtrace, 0, sizeof(uint32_t) * kWTrace * nw, L.stream)); cp.wtrace = g.d_wtrace; g.wtrace_warps = nw; }
    }
    kern<<<blocks, threads, wsmem, L.stream>>>(cp);
  }
  CU_TRY(cudaGetLastError());
  if (mark(timing)) return INC_E_CUDA;
  // --- evaporation ---
  EvapParams<real> ep;
  ep.model = model; ep.ws = L.ws; ep.ctr = L.ctr; ep.e_base = e_base + g.event_offset; ep.n_chunk = n_chunk;
  ep.seed_lo = cp.seed_lo; ep.seed_hi = cp.seed_hi; ep.flags = g.flags;
  ep.out_counts = counts;
  auto ekern = g.tab.level_density == 1 ? evap_kernel<real, STATS, true> : evap_kernel<real, STATS, false>;
  int eocc = 0;
  if (int lr = launch_shape((const void *)ekern, 256, 0, &eocc)) return lr;
  if (eocc < 1) return fail(INC_E_CUDA, "evaporation kernel does not fit on an SM");
  int eblocks = eocc * g.sm_count;
  if (eblocks > need) eblocks = need;
  {
    // Programmatic dependent launch: the evaporation CTAs may be scheduled while the cascade kernel's last CTAs are
    // still draining; they consume the completion list, so they never run ahead of the data.  With INC_F_TIMING the
    // stages are separated by events and run one after the other, so that each has a duration of its own.
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)eblocks); cfg.blockDim = dim3(256); cfg.dynamicSmemBytes = 0; cfg.stream = L.stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = (timing || (g.flags & INC_F_NO_OVERLAP)) ? 0 : 1;
    cudaError_t le = cudaLaunchKernelEx(&cfg, ekern, ep);
    if (le != cudaSuccess && cfg.numAttrs) {      // (a driver without programmatic dependent launch: plain stream order)
      (void)cudaGetLastError();
      cfg.numAttrs = 0;
      le = cudaLaunchKernelEx(&cfg, ekern, ep);
    }
    CU_TRY(le);
  }
  CU_TRY(cudaGetLastError());
  if (mark(timing)) return INC_E_CUDA;
  // --- prefix sum of counts (running base carried across chunks in ctr->total_sec) ---
  const int tiles = (n_chunk + kScanTile - 1) / kScanTile;
  scan_tile_sums<<<tiles, kScanBlock, 0, L.stream>>>(counts, n_chunk, L.tiles);
  scan_tiles<<<1, kScanBlock, 0, L.stream>>>(L.tiles, tiles, &L.ctr->total_sec);
  scan_write_offsets<<<tiles, kScanBlock, 0, L.stream>>>(counts, n_chunk, L.tiles, offsets);
  CU_TRY(cudaGetLastError());
  if (mark(timing)) return INC_E_CUDA;
  // --- compaction into the caller's SoA ---
  CompactParams<real> kp;
  kp.ws = L.ws; kp.offsets = offsets; kp.counts = counts; kp.n_chunk = n_chunk;
  kp.species = sec->species; kp.T = sec->T; kp.ux = sec->ux; kp.uy = sec->uy; kp.uz = sec->uz;
  kp.capacity = sec->capacity;
  kp.rA = res->A; kp.rZ = res->Z; kp.rE = res->Estar; kp.rPx = res->px; kp.rPy = res->py; kp.rPz = res->pz; kp.rstatus = res->status;
  const int cwarps = (n_chunk + 31) / 32;
  const int cblocks = (cwarps + 7) / 8;
  compact_kernel<real><<<cblocks, 256, 0, L.stream>>>(kp);
  CU_TRY(cudaGetLastError());
  if (mark(timing)) return INC_E_CUDA;
  return 0;
}

}  // namespace

// =================================================================================================
extern "C" {

const char *inc_last_error(void) { return g.err.c_str(); }

const char *inc_build_info(void) {
#ifdef INC_REAL_IS_DOUBLE
  return "inc-b200 f64 parity build (-fmad=false) sm_100a";
#else
  return "inc-b200 f32 production build (fast intrinsics) sm_100a";
#endif
}

int inc_set_stream(void *s) { g.stream = (cudaStream_t)s; return 0; }
int inc_set_flags(uint32_t f) { g.flags = f; return 0; }
int inc_set_event_offset(int64_t e0) {
  if (e0 < 0) return fail(INC_E_BADARG, "negative event offset");
  g.event_offset = e0;
  return 0;
}

int inc_init(int A, int Z, const inc_tables *t) {
  int rc = check_tables(t);
  if (rc) return rc;
  if (A < 6 || A > 64 || Z < 2 || Z > A - 2) return fail(INC_E_BADARG, "unsupported (A,Z): need 6<=A<=64, 2<=Z<=A-2");
  if (!g.tab.captured) {
    copy_tables(t, g.tab);
    rc = upload_model();
    if (rc) { g.tab.captured = false; return rc; }
  } else if (!same_tables(t, g.tab)) {
    return fail(INC_E_TABLES, "tables differ from those captured by the first inc_init (call inc_shutdown first)");
  }
  int slot = -1;
  for (int i = 0; i < INC_MAX_TARGETS; ++i) if (!g.nuc[i].live) { slot = i; break; }
  if (slot < 0) return fail(INC_E_BADARG, "all 16 target slots are live");
  setup_nucleus(A, Z, g.tab, g.nuc[slot]);
  NucDev<real> d;
  fill_nucdev(g.nuc[slot], d);
  cudaError_t e = cudaMemcpy(&g.d_nuc[slot], &d, sizeof(d), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) { g.nuc[slot].live = false; return fail(INC_E_CUDA, std::string("upload nucleus: ") + cudaGetErrorString(e)); }
  return slot;
}

int inc_free_target(int id) {
  if (id < 0 || id >= INC_MAX_TARGETS || !g.nuc[id].live) return fail(INC_E_BADARG, "no such target");
  g.nuc[id].live = false;
  NucDev<real> d;
  std::memset(&d, 0, sizeof(d));
  CU_TRY(cudaMemcpy(&g.d_nuc[id], &d, sizeof(d), cudaMemcpyHostToDevice));
  return 0;
}

void inc_shutdown(void) {
  free_ws();
  void **p[] = {(void **)&g.d_tabS, (void **)&g.d_tabC, (void **)&g.d_bind, (void **)&g.d_evch, (void **)&g.d_ld, (void **)&g.d_ldrow, (void **)&g.d_gtab, (void **)&g.d_nuc,
                (void **)&g.d_ctr, (void **)&g.d_wtrace, (void **)&g.d_offsets, (void **)&g.d_tiles};
  for (auto q : p) { if (*q) cudaFree(*q); *q = nullptr; }
  g.offsets_cap = g.tiles_cap = 0;
  free_host_ring();
  if (g.hp.copy_stream) { cudaStreamDestroy(g.hp.copy_stream); g.hp.copy_stream = nullptr; }
  if (g.hp.h_tot) { cudaFreeHost(g.hp.h_tot); g.hp.h_tot = nullptr; }
  if (g.hp.h_err) { cudaFreeHost(g.hp.h_err); g.hp.h_err = nullptr; }
  for (auto &n : g.nuc) n.live = false;
  g.tab.captured = false;
  g.last_n = -1;
  g.event_offset = 0;
  g.ovf_all = false;
}

}  // extern "C"

namespace {
constexpr int64_t kQueueOverflow = -1000;   // internal: the wavefront kernel's track queues overflowed
constexpr int64_t kPoolOverflow = -1001;    // internal: more events than overflow rows had over kStageMain secondaries

int64_t simulate_once(int64_t n, const INC_REAL *E_in, const int32_t *tid, uint64_t seed, inc_secondaries *sec,
                      int32_t *counts, inc_residual *res);
int64_t simulate_host_once(int64_t n, const INC_REAL *E_in, const int32_t *tid, uint64_t seed, inc_secondaries *sec,
                           int32_t *counts, inc_residual *res);
int resolve_stage_times();
int64_t device_error(unsigned int err);

// A call that hits one of the two implementation limits of the default configuration is run again, and the rerun can
// hit the other one (the abandoned first run allocates fewer overflow rows than a complete one needs), so the two
// recoveries loop: at most three reruns, and an internal code never reaches the caller.
//  - kPoolOverflow: the staging overflow pool (a row for one event in 64) was too small for this batch: from now on
//    every event has a row.
//  - kQueueOverflow: the default cascade kernel keeps its tracks in fixed per-warp queues; a batch that overflows them
//    (never seen: it takes ~190 simultaneous tracks in one warp's ~80 events) is run with the lane-per-event kernel,
//    which has no such limit and gives the same events (R-R4: a track's fate depends only on its own draws).
template <typename F> int64_t run_with_recovery(F once) {
  const uint32_t f0 = g.flags;
  int64_t rc = once();
  for (int rerun = 0; rerun < 3 && (rc == kPoolOverflow || rc == kQueueOverflow); ++rerun) {
    if (rc == kPoolOverflow) { g.ovf_all = true; g.ovf_rows_user = 0; }
    else g.flags = (g.flags | INC_F_LANE_STATE_MACHINE) & ~INC_F_TEST_QUEUE_OVF;
    g.reruns++;
    rc = once();
  }
  g.flags = f0;
  if (rc == kPoolOverflow) rc = fail(INC_E_STATE, "staging overflow pool exhausted (results invalid)");
  if (rc == kQueueOverflow) rc = fail(INC_E_STATE, "internal track-queue overflow (results invalid)");
  g.projectile = nullptr;       // inc_set_projectiles applies to one call
  return rc;
}
}  // namespace

extern "C" {

int64_t inc_simulate(int64_t n, const INC_REAL *E_in, const int32_t *tid, uint64_t seed, inc_secondaries *sec,
                     int32_t *counts, inc_residual *res) {
  return run_with_recovery([&]() { return simulate_once(n, E_in, tid, seed, sec, counts, res); });
}

int64_t inc_get_rerun_count(void) { return g.reruns; }

}  // extern "C"

namespace {

// stage times of the call from the events recorded around the kernels (INC_F_TIMING); the stream has been synchronised
int resolve_stage_times() {
  for (size_t c = 0; c + 4 < g.pending_events.size(); c += 5) {
    const int nl[4] = {1, 1, 3, 1};
    for (int i = 0; i < 4; ++i) {
      float ms = 0;
      CU_TRY(cudaEventElapsedTime(&ms, g.pending_events[c + i], g.pending_events[c + i + 1]));
      g.stage_ms[i] += ms; g.stage_launches[i] += nl[i];
    }
  }
  for (auto e : g.pending_events) cudaEventDestroy(e);
  g.pending_events.clear();
  return 0;
}

// the device error word of a finished call -> 0, kQueueOverflow, or a negative INC_E_* code with its message
int64_t device_error(unsigned int err) {
  if (err & 16u) return fail(INC_E_STATE, "watchdog: a warp of the wavefront cascade kernel made no progress (results invalid)");
  if (err & 4u) return kQueueOverflow;       // (before bit 32: the launch was given up, the call is run again with the lane kernel)
  if (err & 32u) return fail(INC_E_STATE, "checked build: an index of the wavefront kernel's queues was out of range (results invalid)");
  if (err & 64u) return kPoolOverflow;
  if (err) {
    return fail(INC_E_BADARG, std::string("device-side input check failed:") + ((err & 1u) ? " E_in outside [20,250] MeV" : "") +
                                  ((err & 2u) ? " target_id not initialised" : "") + ((err & 8u) ? " projectile not 0 or 1" : ""));
  }
  return 0;
}

int64_t simulate_once(int64_t n, const INC_REAL *E_in, const int32_t *tid, uint64_t seed, inc_secondaries *sec,
                      int32_t *counts, inc_residual *res) {
  if (!g.tab.captured) return fail(INC_E_STATE, "inc_simulate before inc_init");
  if (n < 0 || !sec || !res || (n > 0 && (!E_in || !tid || !counts))) return fail(INC_E_BADARG, "null argument or n < 0");
  if (n > 0 && (!res->A || !res->Z || !res->Estar || !res->px || !res->py || !res->pz || !res->status))
    return fail(INC_E_BADARG, "null residual array");
  if (sec->capacity < 0 || (sec->capacity > 0 && (!sec->species || !sec->T || !sec->ux || !sec->uy || !sec->uz)))
    return fail(INC_E_BADARG, "null secondary array");
  const size_t chunk_max = g.chunk_events;
  const size_t chunk = (size_t)n < chunk_max ? (size_t)(n > 0 ? n : 1) : chunk_max;
  int rc = ensure_ws(chunk, (size_t)n);
  if (rc) return rc;
  CU_TRY(cudaMemsetAsync(g.d_ctr, 0, sizeof(DevCounters), g.stream));
  if (int rk_rc = set_round_keys(seed)) return rk_rc;
  for (auto e : g.pending_events) cudaEventDestroy(e);
  g.pending_events.clear();
  for (int i = 0; i < 4; ++i) { g.stage_ms[i] = 0; g.stage_launches[i] = 0; }
  const bool stats = (g.flags & INC_F_STATS) != 0;
  State::Lane l0 = lane0();
  g.cur = &l0;
  for (long long e0 = 0; e0 < n; e0 += (long long)chunk) {
    const int nc = (int)((n - e0) < (long long)chunk ? (n - e0) : (long long)chunk);
    inc_residual r = *res;
    r.A += e0; r.Z += e0; r.Estar += e0; r.px += e0; r.py += e0; r.pz += e0; r.status += e0;
    const uint8_t *pj = g.projectile ? g.projectile + e0 : nullptr;
    rc = stats ? launch_chunk<true>(e0, nc, E_in + e0, tid + e0, pj, seed, sec, counts + e0, &r, g.d_offsets + e0)
               : launch_chunk<false>(e0, nc, E_in + e0, tid + e0, pj, seed, sec, counts + e0, &r, g.d_offsets + e0);
    if (rc) return rc;
  }
  CU_TRY(cudaMemcpyAsync(g.d_offsets + n, &g.d_ctr->total_sec, sizeof(long long), cudaMemcpyDeviceToDevice, g.stream));
  struct { unsigned long long total; unsigned int err, pad; } tail;
  CU_TRY(cudaMemcpyAsync(&tail, &g.d_ctr->total_sec, 16, cudaMemcpyDeviceToHost, g.stream));
  CU_TRY(cudaStreamSynchronize(g.stream));
  if (int rt = resolve_stage_times()) return rt;
  g.last_n = n; g.last_total = (long long)tail.total;
  g.last_chunks = (int)((n + (long long)chunk - 1) / (long long)chunk);
  g.last_offsets_valid = true;
  if (int64_t er = device_error(tail.err)) return er;
  if ((long long)tail.total > sec->capacity) {
    char buf[160];
    std::snprintf(buf, sizeof buf, "secondary capacity %lld too small, need %llu", (long long)sec->capacity, tail.total);
    return fail(INC_E_CAPACITY, buf);
  }
  return (int64_t)tail.total;
}

}  // namespace

extern "C" {

int inc_get_offsets(int64_t *dev_offsets) {
  if (g.last_n < 0) return fail(INC_E_STATE, "no previous inc_simulate");
  if (!g.last_offsets_valid) return fail(INC_E_STATE, "the last call was a multi-chunk inc_simulate_host: its offsets are per chunk (take the prefix sum of out_counts)");
  if (!dev_offsets) return fail(INC_E_BADARG, "null pointer");
  CU_TRY(cudaMemcpyAsync(dev_offsets, g.d_offsets, (size_t)(g.last_n + 1) * sizeof(long long), cudaMemcpyDeviceToDevice, g.stream));
  CU_TRY(cudaStreamSynchronize(g.stream));
  return 0;
}

int inc_get_cascade_stage(int32_t *A, int32_t *Z, INC_REAL *Es, INC_REAL *px, INC_REAL *py, INC_REAL *pz, int32_t *ncs) {
  if (g.last_n < 0) return fail(INC_E_STATE, "no previous inc_simulate");
  if (g.last_chunks > 1) return fail(INC_E_STATE, "cascade stage is only kept for single-chunk calls (n <= the chunk size, inc_set_chunk_events)");
  const long long n = g.last_n;
  if (n > 0) {
    unpack_cascade_kernel<real><<<(unsigned)((n + 255) / 256), 256, 0, g.stream>>>(g.ws.crec, n, A, Z, Es, px, py, pz, ncs);
    CU_TRY(cudaGetLastError());
  }
  CU_TRY(cudaStreamSynchronize(g.stream));
  return 0;
}

int inc_get_stats(inc_stats *out) {
  if (!out) return fail(INC_E_BADARG, "null pointer");
  if (g.last_n < 0) return fail(INC_E_STATE, "no previous inc_simulate");
  DevCounters c;
  CU_TRY(cudaMemcpy(&c, g.d_ctr, sizeof(c), cudaMemcpyDeviceToHost));
  out->events = c.stats[S_EVENTS]; out->failed = c.stats[S_FAILED]; out->attempts = c.stats[S_ATTEMPTS];
  out->segments = c.stats[S_SEG]; out->boundaries = c.stats[S_BND]; out->reflections = c.stats[S_REFL];
  out->escapes = c.stats[S_ESC]; out->collisions = c.stats[S_COLL]; out->blocked = c.stats[S_BLOCKED];
  out->allowed = c.stats[S_ALLOWED]; out->absorbed = c.stats[S_ABSORBED];
  out->evap_steps = c.stats[S_EVSTEPS]; out->evap_trials = c.stats[S_EVTRIALS]; out->evap_emitted = c.stats[S_EVEMIT];
  out->warp_iters_seg = c.stats[S_WI_SEG]; out->warp_iters_coll = c.stats[S_WI_COLL]; out->warp_iters_epi = c.stats[S_WI_EPI];
  out->lane_slots_seg = c.stats[S_LS_SEG]; out->lane_slots_coll = c.stats[S_LS_COLL]; out->lane_slots_epi = c.stats[S_LS_EPI];
  return 0;
}

int inc_get_drain_timeline(double ms[4]) {
  if (!ms) return fail(INC_E_BADARG, "null pointer");
  if (g.last_n < 0) return fail(INC_E_STATE, "no previous inc_simulate");
  DevCounters c;
  CU_TRY(cudaMemcpy(&c, g.d_ctr, sizeof(c), cudaMemcpyDeviceToHost));
  ms[0] = ms[1] = ms[2] = ms[3] = 0;
  if (c.tl[4] == 0) return 0;
  const double t0 = (double)(~c.tl[0]), nw = (double)c.tl[4];
  ms[0] = ((double)c.tl[1] / nw - t0) * 1e-6;
  ms[1] = ((double)c.tl[2] / nw - t0) * 1e-6;
  ms[2] = ((double)c.tl[3] - t0) * 1e-6;
  ms[3] = ((double)(~c.tl[5]) - t0) * 1e-6;
  return 0;
}

int inc_get_warp_trace(uint32_t *out, int32_t max_warps) {
  if (!out || max_warps < 0) return fail(INC_E_BADARG, "null pointer");
  if (g.last_n < 0 || !g.d_wtrace) return 0;
  const int n = g.wtrace_warps < max_warps ? g.wtrace_warps : max_warps;
  CU_TRY(cudaMemcpy(out, g.d_wtrace, sizeof(uint32_t) * kWTrace * (size_t)n, cudaMemcpyDeviceToHost));
  return n;
}

int inc_get_stage_times(float ms[4], int32_t launches[4]) {
  if (g.last_n < 0) return fail(INC_E_STATE, "no previous inc_simulate");
  for (int i = 0; i < 4; ++i) { if (ms) ms[i] = g.stage_ms[i]; if (launches) launches[i] = g.stage_launches[i]; }
  return 0;
}

int inc_get_nucleus(int id, int32_t *A, int32_t *Z, int32_t *ns, double *R, double *EC, double *EBp, double *EBn,
                    double *r, double *rho_p, double *rho_n, double *pF_p, double *pF_n, double *EF_p, double *EF_n,
                    double *V_p, double *V_n) {
  if (id < 0 || id >= INC_MAX_TARGETS || !g.nuc[id].live) return fail(INC_E_BADARG, "no such target");
  const HostNucleus &h = g.nuc[id];
  if (A) *A = h.A; if (Z) *Z = h.Z; if (ns) *ns = h.ns; if (R) *R = h.R; if (EC) *EC = h.EC;
  if (EBp) *EBp = h.EB_p; if (EBn) *EBn = h.EB_n;
  auto cp = [](double *dst, const std::vector<double> &v) { if (dst) std::memcpy(dst, v.data(), v.size() * sizeof(double)); };
  cp(r, h.r); cp(rho_p, h.rho_p); cp(rho_n, h.rho_n); cp(pF_p, h.pF_p); cp(pF_n, h.pF_n);
  cp(EF_p, h.EF_p); cp(EF_n, h.EF_n); cp(V_p, h.V_p); cp(V_n, h.V_n);
  return 0;
}

int inc_set_vote_thresholds(int coll, int epi) {
  if (coll < 1 || coll > 32 || epi < 1 || epi > 32) return fail(INC_E_BADARG, "thresholds must be 1..32");
  g.vote_coll = coll; g.vote_epi = epi;
  return 0;
}

int inc_set_projectiles(const uint8_t *projectile) {
  g.projectile = projectile;
  return 0;
}

int inc_set_chunk_events(int64_t n) {
  if (n < 0 || (n > 0 && n < 1024) || n > ((int64_t)1 << 24)) return fail(INC_E_BADARG, "chunk size must be 0 (default) or 1024 .. 2^24");
  g.chunk_events = n == 0 ? ((size_t)1 << 22) : (size_t)n;
  return 0;
}

int inc_set_segments_per_pass(int n) {
  if (n < 0 || n > 8) return fail(INC_E_BADARG, "segments per pass must be 0 (automatic) or 1..8");
  g.seg_per_pass = n;
  return 0;
}

int inc_set_stage_overflow_rows(int64_t rows) {
  if (rows < 0) return fail(INC_E_BADARG, "rows must be >= 0");
  g.ovf_rows_user = rows;
  return 0;
}

int inc_set_event_taper(int min_events_per_warp) {
  if (min_events_per_warp < -1 || min_events_per_warp > 128) return fail(INC_E_BADARG, "taper minimum must be -1 (automatic), 0 (off) .. 128");
  g.taper_min = min_events_per_warp;
  return 0;
}

int inc_set_long_track_threshold(int n_segments) {
  if (n_segments < 0) return fail(INC_E_BADARG, "threshold must be >= 0");
  g.long_seg = n_segments == 0 ? kLongSegDefault : n_segments;
  return 0;
}

int inc_measure_issue_peak(double *out, double *clock_mhz) {
  if (!out) return fail(INC_E_BADARG, "null pointer");
  int dev = 0, sms = 0, khz = 0;
  CU_TRY(cudaGetDevice(&dev));
  CU_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  CU_TRY(cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev));
  real *d = nullptr;
  CU_TRY(cudaMalloc((void **)&d, sizeof(real)));
  const int blocks = sms * 8, iters = 4096;
  cudaEvent_t a, b;
  CU_TRY(cudaEventCreate(&a)); CU_TRY(cudaEventCreate(&b));
  double best = 0;
  for (int rep = 0; rep < 5; ++rep) {
    CU_TRY(cudaEventRecord(a, g.stream));
    fma_peak_kernel<real><<<blocks, 256, 0, g.stream>>>(d, iters, (real)0.999, (real)0.001);
    CU_TRY(cudaEventRecord(b, g.stream));
    CU_TRY(cudaEventSynchronize(b));
    float ms = 0;
    CU_TRY(cudaEventElapsedTime(&ms, a, b));
    const double ops = (double)blocks * 256.0 * iters * 16.0 * 8.0;
    const double rate = ops / (ms * 1e-3);
    if (rep > 0 && rate > best) best = rate;
  }
  cudaEventDestroy(a); cudaEventDestroy(b); cudaFree(d);
  *out = best;
  if (clock_mhz) *clock_mhz = khz / 1000.0;
  return 0;
}

int inc_tally(int64_t n, const inc_secondaries *sec, const int32_t *counts, const int64_t *offsets,
              const inc_residual *res, const inc_tally_spec *spec, const inc_tallies *out) {
  if (n < 0 || !sec || !res || !spec || !out) return fail(INC_E_BADARG, "null pointer or n < 0");
  if (spec->n_T < 1 || spec->n_cos < 1 || spec->mult_max < 0 || spec->A_max < 0 || spec->Z_max < 0 || !(spec->T_max > 0.0))
    return fail(INC_E_BADARG, "tally spec: bin counts must be positive");
  if (!out->dd || !out->mult || !out->nuclide || !out->yield) return fail(INC_E_BADARG, "null tally pointer");
  if (n == 0) return 0;
  if (!counts || !offsets || !sec->species || !sec->T || !sec->uz || !res->A || !res->Z) return fail(INC_E_BADARG, "null pointer");
  TallyParams<real> tp;
  tp.species = sec->species; tp.T = sec->T; tp.uz = sec->uz; tp.counts = counts;
  tp.offsets = reinterpret_cast<const long long *>(offsets); tp.rA = res->A; tp.rZ = res->Z; tp.n_events = n;
  tp.n_T = spec->n_T; tp.n_cos = spec->n_cos; tp.mult_max = spec->mult_max; tp.A_max = spec->A_max; tp.Z_max = spec->Z_max;
  tp.T_scale = (real)((double)spec->n_T / spec->T_max); tp.cos_scale = (real)((double)spec->n_cos / 2.0);
  tp.dd = out->dd; tp.mult = out->mult; tp.nuclide = out->nuclide; tp.yield = out->yield;
  const size_t bins = (size_t)3 * spec->n_cos * (spec->n_T + 1) + (size_t)4 * (spec->mult_max + 1) +
                      (size_t)(spec->A_max + 1) * (spec->Z_max + 1) + 12;
  const size_t smem = bins * sizeof(unsigned int);
  tp.smem = smem <= 96 * 1024 ? 1 : 0;
  auto kern = tally_kernel<real>;
  if (tp.smem && smem > 48 * 1024) CU_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  long long blocks = (n + 255) / 256;
  const long long cap = (long long)g.sm_count * 4;
  if (g.sm_count > 0 && blocks > cap) blocks = cap;
  kern<<<(unsigned)blocks, 256, tp.smem ? smem : 0, g.stream>>>(tp);
  CU_TRY(cudaGetLastError());
  return 0;
}

int inc_philox_blocks(const uint32_t *ctr, uint64_t seed, uint32_t *out, int64_t n) {
  if (n < 0 || (n > 0 && (!ctr || !out))) return fail(INC_E_BADARG, "bad argument");
  if (n == 0) return 0;
  if (int rc = set_round_keys(seed)) return rc;
  philox_blocks_kernel<<<(unsigned)((n + 255) / 256), 256, 0, g.stream>>>(ctr, out, n);
  CU_TRY(cudaGetLastError());
  CU_TRY(cudaStreamSynchronize(g.stream));
  return 0;
}

int64_t inc_simulate_host(int64_t n, const INC_REAL *E_in, const int32_t *tid, uint64_t seed, inc_secondaries *sec,
                          int32_t *counts, inc_residual *res) {
  return run_with_recovery([&]() { return simulate_host_once(n, E_in, tid, seed, sec, counts, res); });
}

}  // extern "C"

namespace {

void free_host_ring() {
  State::HostPath &h = g.hp;
  for (auto &sl : h.slot) {
    void **p[] = {(void **)&sl.E, (void **)&sl.tid, (void **)&sl.counts, (void **)&sl.A, (void **)&sl.Z, (void **)&sl.Es,
                  (void **)&sl.px, (void **)&sl.py, (void **)&sl.pz, (void **)&sl.status, (void **)&sl.sp, (void **)&sl.T,
                  (void **)&sl.ux, (void **)&sl.uy, (void **)&sl.uz};
    for (auto q : p) { if (*q) cudaFree(*q); *q = nullptr; }
    if (sl.computed) { cudaEventDestroy(sl.computed); sl.computed = nullptr; }
    if (sl.copied) { cudaEventDestroy(sl.copied); sl.copied = nullptr; }
  }
  h.chunk_cap = 0;
}

int ensure_host_ring(size_t chunk) {
  State::HostPath &h = g.hp;
  if (!h.copy_stream) CU_TRY(cudaStreamCreateWithFlags(&h.copy_stream, cudaStreamNonBlocking));
  if (!h.h_tot) CU_TRY(cudaMallocHost((void **)&h.h_tot, State::kRing * sizeof(unsigned long long)));
  if (!h.h_err) CU_TRY(cudaMallocHost((void **)&h.h_err, sizeof(unsigned int)));
  if (chunk <= h.chunk_cap) return 0;
  free_host_ring();
  const size_t m = chunk, k = chunk * (size_t)kMaxSec;
  for (auto &sl : h.slot) {
    CU_TRY(cudaMalloc((void **)&sl.E, m * sizeof(real))); CU_TRY(cudaMalloc((void **)&sl.tid, m * 4));
    CU_TRY(cudaMalloc((void **)&sl.counts, m * 4)); CU_TRY(cudaMalloc((void **)&sl.A, m * 4)); CU_TRY(cudaMalloc((void **)&sl.Z, m * 4));
    CU_TRY(cudaMalloc((void **)&sl.Es, m * sizeof(real))); CU_TRY(cudaMalloc((void **)&sl.px, m * sizeof(real)));
    CU_TRY(cudaMalloc((void **)&sl.py, m * sizeof(real))); CU_TRY(cudaMalloc((void **)&sl.pz, m * sizeof(real)));
    CU_TRY(cudaMalloc((void **)&sl.status, m * 4));
    CU_TRY(cudaMalloc((void **)&sl.sp, k)); CU_TRY(cudaMalloc((void **)&sl.T, k * sizeof(real)));
    CU_TRY(cudaMalloc((void **)&sl.ux, k * sizeof(real))); CU_TRY(cudaMalloc((void **)&sl.uy, k * sizeof(real)));
    CU_TRY(cudaMalloc((void **)&sl.uz, k * sizeof(real)));
    CU_TRY(cudaEventCreateWithFlags(&sl.computed, cudaEventDisableTiming));
    CU_TRY(cudaEventCreateWithFlags(&sl.copied, cudaEventDisableTiming));
  }
  h.chunk_cap = chunk;
  return 0;
}

// Streaming: the call runs in chunks; chunk c lives in ring slot c % kRing (inputs, per-event
// outputs, up to kMaxSec secondaries per event, numbered from 0 inside the chunk), is computed on the caller's stream,
// and its outputs travel to the host on a second stream while the next chunks compute.  Device memory does not depend
// on n.  The host learns each chunk's number of secondaries (8 bytes, pinned) behind an event: that fixes where its
// list goes in the caller's arrays.
int64_t simulate_host_chunks(int64_t n, const INC_REAL *E_in, const int32_t *tid, uint64_t seed, inc_secondaries *sec,
                             int32_t *counts, inc_residual *res);

// Every exit, the error exits included, waits for both streams: asynchronous copies into the caller's host buffers and
// kernels on the ring slots must not be in flight when the caller gets control back and may free or reuse its buffers.
int64_t simulate_host_once(int64_t n, const INC_REAL *E_in, const int32_t *tid, uint64_t seed, inc_secondaries *sec,
                           int32_t *counts, inc_residual *res) {
  const int64_t rc = simulate_host_chunks(n, E_in, tid, seed, sec, counts, res);
  if (rc < 0) {
    const std::string msg = g.err;           // (keep the first failure's message)
    cudaStreamSynchronize(g.stream);
    if (g.hp.copy_stream) cudaStreamSynchronize(g.hp.copy_stream);
    g.err = msg;
  }
  return rc;
}

int64_t simulate_host_chunks(int64_t n, const INC_REAL *E_in, const int32_t *tid, uint64_t seed, inc_secondaries *sec,
                             int32_t *counts, inc_residual *res) {
  if (!g.tab.captured) return fail(INC_E_STATE, "inc_simulate_host before inc_init");
  if (n < 0 || !sec || !res || (n > 0 && (!E_in || !tid || !counts))) return fail(INC_E_BADARG, "null argument or n < 0");
  if (n > 0 && (!res->A || !res->Z || !res->Estar || !res->px || !res->py || !res->pz || !res->status))
    return fail(INC_E_BADARG, "null residual array");
  if (sec->capacity < 0 || (sec->capacity > 0 && (!sec->species || !sec->T || !sec->ux || !sec->uy || !sec->uz)))
    return fail(INC_E_BADARG, "null secondary array");
  // 2^19 events per chunk, 2^20 for long calls (a chunk costs one tail of the cascade kernel, so chunks should not be
  // smaller than hiding the copies needs); never more than inc_set_chunk_events
  size_t chunk = (size_t)n > ((size_t)1 << 21) ? 2 * g.host_chunk_events : g.host_chunk_events;
  if (chunk > g.chunk_events) chunk = g.chunk_events;
  if ((size_t)n < chunk) chunk = (size_t)(n > 0 ? n : 1);
  int rc = ensure_ws(chunk, chunk);
  if (rc) return rc;
  rc = ensure_host_ring(chunk);
  if (rc) return rc;
  State::HostPath &h = g.hp;
  const long long n_chunks = (n + (long long)chunk - 1) / (long long)chunk;
  State::Lane L = lane0();
  g.cur = &L;
  CU_TRY(cudaMemsetAsync(g.d_ctr, 0, sizeof(DevCounters), g.stream));
  if (int rk_rc = set_round_keys(seed)) return rk_rc;
  for (auto e : g.pending_events) cudaEventDestroy(e);
  g.pending_events.clear();
  for (int i = 0; i < 4; ++i) { g.stage_ms[i] = 0; g.stage_launches[i] = 0; }
  const bool stats = (g.flags & INC_F_STATS) != 0;
  unsigned long long host_total = 0;                       // secondaries of the chunks copied so far
  const unsigned long long cap = (unsigned long long)sec->capacity;
  cudaStream_t cs = h.copy_stream;
  // outputs of chunk c -> host (its kernels have been enqueued before)
  auto copy_out = [&](long long c) -> int {
    State::HostSlot &sl = h.slot[c % State::kRing];
    const size_t o = (size_t)c * chunk;
    const size_t m = (size_t)(n - (long long)o) < chunk ? (size_t)(n - (long long)o) : chunk;
    CU_TRY(cudaEventSynchronize(sl.computed));
    const unsigned long long t = h.h_tot[c % State::kRing];
    CU_TRY(cudaMemcpyAsync(counts + o, sl.counts, m * 4, cudaMemcpyDeviceToHost, cs));
    CU_TRY(cudaMemcpyAsync(res->A + o, sl.A, m * 4, cudaMemcpyDeviceToHost, cs));
    CU_TRY(cudaMemcpyAsync(res->Z + o, sl.Z, m * 4, cudaMemcpyDeviceToHost, cs));
    CU_TRY(cudaMemcpyAsync(res->Estar + o, sl.Es, m * sizeof(real), cudaMemcpyDeviceToHost, cs));
    CU_TRY(cudaMemcpyAsync(res->px + o, sl.px, m * sizeof(real), cudaMemcpyDeviceToHost, cs));
    CU_TRY(cudaMemcpyAsync(res->py + o, sl.py, m * sizeof(real), cudaMemcpyDeviceToHost, cs));
    CU_TRY(cudaMemcpyAsync(res->pz + o, sl.pz, m * sizeof(real), cudaMemcpyDeviceToHost, cs));
    CU_TRY(cudaMemcpyAsync(res->status + o, sl.status, m * 4, cudaMemcpyDeviceToHost, cs));
    const unsigned long long a0 = host_total < cap ? host_total : cap;                 // nothing is written past the capacity
    const unsigned long long a1 = host_total + t < cap ? host_total + t : cap;
    if (a1 > a0) {
      const size_t k = (size_t)(a1 - a0), f = (size_t)a0;
      CU_TRY(cudaMemcpyAsync(sec->species + f, sl.sp, k, cudaMemcpyDeviceToHost, cs));
      CU_TRY(cudaMemcpyAsync(sec->T + f, sl.T, k * sizeof(real), cudaMemcpyDeviceToHost, cs));
      CU_TRY(cudaMemcpyAsync(sec->ux + f, sl.ux, k * sizeof(real), cudaMemcpyDeviceToHost, cs));
      CU_TRY(cudaMemcpyAsync(sec->uy + f, sl.uy, k * sizeof(real), cudaMemcpyDeviceToHost, cs));
      CU_TRY(cudaMemcpyAsync(sec->uz + f, sl.uz, k * sizeof(real), cudaMemcpyDeviceToHost, cs));
    }
    host_total += t;
    CU_TRY(cudaEventRecord(sl.copied, cs));
    return 0;
  };
  for (long long c = 0; c < n_chunks; ++c) {
    State::HostSlot &sl = h.slot[c % State::kRing];
    const long long e0 = c * (long long)chunk;
    const int nc = (int)((n - e0) < (long long)chunk ? (n - e0) : (long long)chunk);
    // the slot is free once the copies of chunk c - kRing are done (they were enqueued two iterations ago)
    if (c >= State::kRing) CU_TRY(cudaStreamWaitEvent(L.stream, sl.copied, 0));
    CU_TRY(cudaMemcpyAsync(sl.E, E_in + e0, (size_t)nc * sizeof(real), cudaMemcpyHostToDevice, L.stream));
    CU_TRY(cudaMemcpyAsync(sl.tid, tid + e0, (size_t)nc * 4, cudaMemcpyHostToDevice, L.stream));
    CU_TRY(cudaMemsetAsync(&L.ctr->total_sec, 0, sizeof(unsigned long long), L.stream));     // chunk-local offsets
    inc_secondaries ds; ds.species = sl.sp; ds.T = sl.T; ds.ux = sl.ux; ds.uy = sl.uy; ds.uz = sl.uz;
    ds.capacity = (int64_t)chunk * kMaxSec;
    inc_residual dr; dr.A = sl.A; dr.Z = sl.Z; dr.Estar = sl.Es; dr.px = sl.px; dr.py = sl.py; dr.pz = sl.pz; dr.status = sl.status;
    const uint8_t *pj = g.projectile ? g.projectile + e0 : nullptr;
    rc = stats ? launch_chunk<true>(e0, nc, sl.E, sl.tid, pj, seed, &ds, sl.counts, &dr, L.offsets)
               : launch_chunk<false>(e0, nc, sl.E, sl.tid, pj, seed, &ds, sl.counts, &dr, L.offsets);
    if (rc) return rc;
    CU_TRY(cudaMemcpyAsync(&h.h_tot[c % State::kRing], &L.ctr->total_sec, sizeof(unsigned long long), cudaMemcpyDeviceToHost, L.stream));
    CU_TRY(cudaEventRecord(sl.computed, L.stream));
    // chunk c is enqueued: now wait for chunk c - 1 and send its outputs home while c computes
    if (c >= 1) { rc = copy_out(c - 1); if (rc) return rc; }
  }
  if (n_chunks >= 1) { rc = copy_out(n_chunks - 1); if (rc) return rc; }
  CU_TRY(cudaMemcpyAsync(h.h_err, &L.ctr->error_word, sizeof(unsigned int), cudaMemcpyDeviceToHost, L.stream));
  CU_TRY(cudaStreamSynchronize(L.stream));
  CU_TRY(cudaStreamSynchronize(cs));
  if (int rt = resolve_stage_times()) return rt;
  g.last_n = n; g.last_total = (long long)host_total;
  g.last_chunks = (int)n_chunks;
  g.last_offsets_valid = n_chunks <= 1;
  if (int64_t er = device_error(n > 0 ? *h.h_err : 0u)) return er;
  if (host_total > cap) {
    char buf[160];
    std::snprintf(buf, sizeof buf, "secondary capacity %lld too small, need %llu", (long long)sec->capacity, host_total);
    return fail(INC_E_CAPACITY, buf);
  }
  return (int64_t)host_total;
}

}  // namespace

// =================================================================================================
// inc_scan_counts_static: the prefix sum of the per-event counts for callers that must not allocate (include/inc.h).
// The scan's scratch -- one partial sum per tile of kScanTile events, then the running total -- lives in the array
// below instead of a cudaMalloc'ed buffer.  It is part of the library image: every GPU that loads the library carries
// these 64.25 KB from the load until the process ends, whether or not the entry point is ever called.
// =================================================================================================
constexpr int kStaticScanTiles = INC_SCAN_STATIC_MAX_EVENTS / kScanTile;        // 8192 tiles of 2048 events
static_assert(kStaticScanTiles * kScanTile == INC_SCAN_STATIC_MAX_EVENTS, "the maximum is a whole number of tiles");
// [0, kStaticScanTiles): tile sums, each rewritten by every call that uses the tile; [kStaticScanTiles]: the running
// total, which a call must find at zero and therefore clears itself (the array keeps what the previous call left)
static __device__ __align__(256) long long s_scan_scratch[kStaticScanTiles + 32];

namespace {

// In host code `s_scan_scratch` names a host-side shadow of the array, NOT device memory: handing it to a kernel would
// fault (or, on a system whose GPU can read host memory, quietly scan into the wrong place).  The device address comes
// from cudaGetSymbolAddress, asked once per device with that device current, and is kept here by device ordinal.
constexpr int kMaxDevices = 64;
long long *g_scan_scratch_dev[kMaxDevices] = {};

int static_scan_scratch(long long **out) {
  int dev = -1;
  CU_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return fail(INC_E_CUDA, "inc_scan_counts_static: device ordinal beyond 63");
  if (!g_scan_scratch_dev[dev]) {
    void *p = nullptr;
    CU_TRY(cudaGetSymbolAddress(&p, s_scan_scratch));
    if (!p) return fail(INC_E_CUDA, "inc_scan_counts_static: cudaGetSymbolAddress gave no address");
    g_scan_scratch_dev[dev] = static_cast<long long *>(p);
  }
  *out = g_scan_scratch_dev[dev];
  return 0;
}

}  // namespace

extern "C" {

int inc_scan_counts_static(int64_t n, const int32_t *counts, int64_t *offsets) {
  if (n < 0 || !offsets || (n > 0 && !counts)) return fail(INC_E_BADARG, "inc_scan_counts_static: null pointer or n < 0");
  if (n > (int64_t)INC_SCAN_STATIC_MAX_EVENTS) {
    char buf[200];
    std::snprintf(buf, sizeof buf, "inc_scan_counts_static: n = %lld is beyond the %d events its fixed scratch array holds "
                  "(split the call, or use inc_get_offsets)", (long long)n, (int)INC_SCAN_STATIC_MAX_EVENTS);
    return fail(INC_E_BADARG, buf);
  }
  long long *scratch = nullptr;
  if (int rc = static_scan_scratch(&scratch)) return rc;
  long long *total = scratch + kStaticScanTiles;
  long long *off = reinterpret_cast<long long *>(offsets);
  CU_TRY(cudaMemsetAsync(total, 0, sizeof(long long), g.stream));                 // the previous call's total is still there
  if (n > 0) {
    const int tiles = (int)((n + kScanTile - 1) / kScanTile);
    scan_tile_sums<<<tiles, kScanBlock, 0, g.stream>>>(counts, (int)n, scratch);
    scan_tiles<<<1, kScanBlock, 0, g.stream>>>(scratch, tiles, reinterpret_cast<unsigned long long *>(total));
    scan_write_offsets<<<tiles, kScanBlock, 0, g.stream>>>(counts, (int)n, scratch, off);
    CU_TRY(cudaGetLastError());
  }
  CU_TRY(cudaMemcpyAsync(off + n, total, sizeof(long long), cudaMemcpyDeviceToDevice, g.stream));
  CU_TRY(cudaStreamSynchronize(g.stream));
  return 0;
}

}  // extern "C"
