// inc_device.cuh — sm_100a device code of the INC + evaporation hot path (arXiv:1309.7963).
//
// Shares nothing with oracle/.  Templated on the real type R (float: production build,
// double: parity build compiled with -fmad=false).  Citations: P:NN = PAPER.md line,
// R-xx = reading in DESIGN.md section 3.
//
// Kernels
//   cascade_kernel   persistent warps; every lane owns one event at a time and runs a small
//                    state machine {SEG, COLL, EPI}.  Each warp pass executes ONE phase, chosen
//                    by warp vote, so the expensive rare steps (collision, epilogue+entry) are
//                    deferred until several lanes need them instead of diverging every pass.
//   evap_kernel      persistent lanes, one Weisskopf-Ewing emission step per pass.
//   scan_* / compact_kernel   exclusive prefix sum of counts, canonical-order SoA output.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/inc.h"

namespace inc {

constexpr int kMaxShells = 32;
constexpr int kMaxSeg = 1024;      // R-C2
constexpr int kMaxAttempt = 256;   // R-C6
constexpr int kMaxTrial = 64;      // R-E4
constexpr int kMaxSec = INC_MAX_SEC;
constexpr int kStackCap = 16;      // pending tracks per event (implementation limit, INC_ST_QUEUE_OVF)
constexpr int kAmax = 72;          // binding / channel tables cover 0..kAmax-1
constexpr int kZmax = 40;
constexpr unsigned kFull = 0xFFFFFFFFu;

// ---- physical constants (standard values; R-K) -----------------------------------------
template <typename R> struct K {
  static constexpr R mp = R(938.27208816);
  static constexpr R mn = R(939.56542052);
  static constexpr R two_pi = R(6.283185307179586476925286766559);
};

// ---- device-resident model data ----------------------------------------------------------
template <typename R> struct ShellDev {   // one constant-density shell
  R rho_p, rho_n;      // fm^-3
  R pF_p, pF_n;        // Fermi momenta, MeV/c
  R pF2_p, pF2_n;      // Pauli threshold on |p'|^2  (T' > E_F  <=>  p'^2 > pF^2)
  R pc2_p, pc2_n;      // cutoff threshold on |p'|^2 (T' - V <= cut <=> p'^2 <= pc2)
  R V_p, V_n;          // well depth E_F + E_B, MeV
  R pad0, pad1;
};

template <typename R> struct NucDev {
  int32_t A, Z, ns, live;
  R Rn, dr, Bt, pad;                       // radius, shell thickness, target binding energy
  ShellDev<R> sh[kMaxShells + 1];          // [ns] = outside: V = 0
};

template <typename R> struct EvChan {        // per (A_d, Z_d, channel j): R-E1/E2 constants
  R V;        // Coulomb barrier of the channel
  R pref;     // g_j M_j A_d^(2/3) alpha_j   (0 => channel closed: daughter invalid)
  R beta;     // Dostrovsky beta (neutron) or 0
  R BdBj;     // B(A_d,Z_d) + B_j, so that X = E* - B(parent) + BdBj - V
};

template <typename R> struct ModelDev {
  const R *tabS;          // [n_xs][4]  {sig_pp, dsig_pp, sig_np, dsig_np} in fm^2 (mb * 0.1)
  const R *tabC;          // [n_xs][8]  {B_pp, dB_pp, B_np, dB_np, a_np, da_np, 0, 0}
  const R *bind;          // [kAmax][kZmax] binding energy, MeV; < -1e29 => no such nucleus
  const EvChan<R> *evch;  // [kAmax][kZmax][6]
  const NucDev<R> *nuc;   // [INC_MAX_TARGETS]
  int32_t n_xs;
  R inv_dp;               // 1 / (grid step in MeV/c)
  R a_div;                // level density a = A_d / a_div
};

template <typename R> struct Workspace {   // per-chunk internal buffers (DEVICE)
  uint32_t *st_code;      // [chunk][kMaxSec]  path code | type << 24 | evap << 31 (evap: species<<24 | seq)
  R *st_T, *st_ux, *st_uy, *st_uz;
  int32_t *cA, *cZ;       // post-cascade nucleus ("SoA of excited nuclei")
  R *cE, *cPx, *cPy, *cPz;
  uint32_t *cmeta;        // n_casc | attempt << 8 | failed << 16
  uint32_t *cstatus;
};

struct DevCounters {       // device scalars
  unsigned long long next_event_casc, next_event_evap;
  unsigned long long total_sec;
  unsigned int error_word;   // bit0: E_in out of range, bit1: bad target id
  unsigned int pad;
  unsigned long long stats[24];
};

enum StatIdx { S_EVENTS = 0, S_FAILED, S_ATTEMPTS, S_SEG, S_BND, S_REFL, S_ESC, S_COLL, S_BLOCKED,
               S_ALLOWED, S_ABSORBED, S_EVSTEPS, S_EVTRIALS, S_EVEMIT, S_WI_SEG, S_WI_COLL, S_WI_EPI,
               S_LS_SEG, S_LS_COLL, S_LS_EPI, S_NSTAT };

// ---- math wrappers: exact library calls for double, fast intrinsics for float ---------------
template <typename R> struct M;
template <> struct M<double> {
  static __device__ __forceinline__ double sqrt_(double x) { return sqrt(x); }
  static __device__ __forceinline__ double rsqrt_(double x) { return 1.0 / sqrt(x); }
  static __device__ __forceinline__ double log_(double x) { return log(x); }
  static __device__ __forceinline__ double exp_(double x) { return exp(x); }
  static __device__ __forceinline__ double cbrt_(double x) { return cbrt(x); }
  static __device__ __forceinline__ double log1p_(double x) { return log1p(x); }
  static __device__ __forceinline__ double expm1_(double x) { return expm1(x); }
  static __device__ __forceinline__ void sincos2pi(double u, double *s, double *c) {
    sincos(6.283185307179586476925286766559 * u, s, c);
  }
  static __device__ __forceinline__ double div_(double a, double b) { return a / b; }
  static __device__ __forceinline__ double u01(uint32_t x) {   // R-R3 (fp64): (x + 1/2) 2^-32
    return ((double)x + 0.5) * (1.0 / 4294967296.0);
  }
  static __device__ __forceinline__ double floor_(double x) { return floor(x); }
  static constexpr int kSeriesTerms = 24;
};
template <> struct M<float> {
  static __device__ __forceinline__ float sqrt_(float x) { return __fsqrt_rn(x); }
  static __device__ __forceinline__ float rsqrt_(float x) { return rsqrtf(x); }
  static __device__ __forceinline__ float log_(float x) { return __logf(x); }
  static __device__ __forceinline__ float exp_(float x) { return __expf(x); }
  static __device__ __forceinline__ float cbrt_(float x) { return cbrtf(x); }
  static __device__ __forceinline__ float log1p_(float x) { return log1pf(x); }
  static __device__ __forceinline__ float expm1_(float x) { return expm1f(x); }
  static __device__ __forceinline__ void sincos2pi(float u, float *s, float *c) {
    float a = 6.283185307179586f * u;
    *s = __sinf(a);
    *c = __cosf(a);
  }
  static __device__ __forceinline__ float div_(float a, float b) { return __fdividef(a, b); }
  static __device__ __forceinline__ float u01(uint32_t x) {    // R-R3 (fp32): ((x>>9) + 1/2) 2^-23, exact
    return ((float)(x >> 9) + 0.5f) * (1.0f / 8388608.0f);
  }
  static __device__ __forceinline__ float floor_(float x) { return floorf(x); }
  static constexpr int kSeriesTerms = 13;
};

// ---- R-R1: Philox4x32-10 ---------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    c0 = hi1 ^ c1 ^ k0;
    c1 = lo1;
    c2 = hi0 ^ c3 ^ k1;
    c3 = lo0;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  return make_uint4(c0, c1, c2, c3);
}

struct RngKey {
  uint32_t k0, k1;   // seed
  uint32_t e0, e1;   // global event index (counter words 2, 3)
};

// R-R2: block k of stream (attempt, path code pi)
template <typename R>
__device__ __forceinline__ void draw4(const RngKey &g, uint32_t attempt, uint32_t pi, uint32_t k, R u[4]) {
  uint4 o = philox4x32_10(k, (attempt << 24) | pi, g.e0, g.e1, g.k0, g.k1);
  u[0] = M<R>::u01(o.x); u[1] = M<R>::u01(o.y); u[2] = M<R>::u01(o.z); u[3] = M<R>::u01(o.w);
}

// ---- table lookup (R-N7): y_k + f (y_{k+1} - y_k), clamped to the grid -------------------------
template <typename R>
__device__ __forceinline__ void grid_pos(R plab_mev, R inv_dp, int n_xs, int &k, R &f) {
  R x = plab_mev * inv_dp;
  R xmax = R(n_xs - 1);
  x = x > xmax ? xmax : x;
  int kk = (int)x;            // x >= 0
  kk = kk > n_xs - 2 ? n_xs - 2 : kk;
  k = kk;
  f = x - R(kk);
}

template <typename R> __device__ __forceinline__ R nucleon_mass(int type) { return type ? K<R>::mp : K<R>::mn; }

// momentum of particle 1 (mass m1, kinetic T1, momentum vector dotted with partner direction = pn)
// in the rest frame of a partner of momentum magnitude q along n (mass m2), MeV/c.  Equivalent to
// sqrt(E_lab^2 - m1^2) with E_lab = (s - m1^2 - m2^2)/(2 m2), written without cancellation.
template <typename R>
__device__ __forceinline__ R plab_of(R m1, R T1, R pn, R q, R m2) {
  R q2 = q * q;
  R E2 = M<R>::sqrt_(q2 + m2 * m2);
  R T2 = M<R>::div_(q2, E2 + m2);
  R Tlab = M<R>::div_(m1 * T2 + m2 * T1 + T1 * T2 - q * pn, m2);
  R a = Tlab * (Tlab + R(2) * m1);
  a = a > R(0) ? a : R(0);
  return M<R>::sqrt_(a);
}

// ---- lane state ------------------------------------------------------------------------------
enum LaneState : int { ST_SEG = 0, ST_COLL = 1, ST_EPI = 2, ST_DONE = 3 };

template <typename R> struct TrackRec {   // pending track (local-memory stack)
  R x, y, z, px, py, pz;
  uint32_t pi;
  uint32_t meta;   // type | shell << 1
};

template <typename R> struct CascadeParams {
  ModelDev<R> model;
  Workspace<R> ws;
  DevCounters *ctr;
  const R *E_in;            // chunk base
  const int32_t *target_id; // chunk base
  long long e_base;         // global index of the chunk's first event
  int n_chunk;
  uint32_t seed_lo, seed_hi;
  uint32_t flags;
  int vote_coll, vote_epi;  // phase-vote thresholds
  int n_live_nuc;           // nuclei slots to stage into shared memory (0..INC_MAX_TARGETS)
};

// shared-memory layout: [NucDev x INC_MAX_TARGETS (only live ones filled)] [tabS n_xs*4]
template <typename R> __host__ __device__ inline size_t cascade_smem_bytes(int n_xs) {
  return sizeof(NucDev<R>) * INC_MAX_TARGETS + sizeof(R) * 4 * (size_t)n_xs;
}

template <typename R, bool STATS>
__global__ void __launch_bounds__(256, 2) cascade_kernel(const CascadeParams<R> P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  NucDev<R> *s_nuc = reinterpret_cast<NucDev<R> *>(smem_raw);
  R *s_tabS = reinterpret_cast<R *>(smem_raw + sizeof(NucDev<R>) * INC_MAX_TARGETS);

  // ---- stage the model into shared memory (read-only afterwards) ----
  {
    const int nw = (int)(sizeof(NucDev<R>) / 4);
    for (int t = 0; t < INC_MAX_TARGETS; ++t) {
      if (!P.model.nuc[t].live) { if (threadIdx.x == 0) s_nuc[t].live = 0; continue; }
      const uint32_t *src = reinterpret_cast<const uint32_t *>(&P.model.nuc[t]);
      uint32_t *dst = reinterpret_cast<uint32_t *>(&s_nuc[t]);
      for (int i = threadIdx.x; i < nw; i += blockDim.x) dst[i] = src[i];
    }
    const int nt = P.model.n_xs * 4;
    for (int i = threadIdx.x; i < nt; i += blockDim.x) s_tabS[i] = P.model.tabS[i];
  }
  __syncthreads();

  const int lane = threadIdx.x & 31;
  const int n_xs = P.model.n_xs;
  const R inv_dp = P.model.inv_dp;
  const bool keep_transparent = (P.flags & INC_F_KEEP_TRANSPARENT) != 0;
  const bool same_stream = (P.flags & INC_F_SAME_STREAM) != 0;

  // ---- lane registers ----
  int state = ST_EPI;
  int ev = -1;                  // chunk-local event index
  int tgt = 0;
  uint32_t attempt = 0;
  R E_in = R(0);
  RngKey g;
  g.k0 = P.seed_lo; g.k1 = P.seed_hi; g.e0 = 0; g.e1 = 0;
  // current track
  R x = 0, y = 0, z = 0, px = 0, py = 0, pz = 0;
  uint32_t pi = 0, kblk = 0;
  int type = 0, shell = 0, nseg = 0;
  // event accumulators
  R Eavail = 0, Prx = 0, Pry = 0, Prz = 0;
  int n_esc = 0, n_p = 0, n_real = 0;
  uint32_t st_try = 0;
  // pending stack
  TrackRec<R> stack[kStackCap];
  int sp = 0;
  // carry from SEG to COLL
  R c_f = 0, c_nx = 0, c_ny = 0, c_nz = 0, c_Sp = 0, c_Sig = 0;
  // stats
  unsigned long long stc[S_NSTAT];
  if (STATS) {
#pragma unroll
    for (int i = 0; i < S_NSTAT; ++i) stc[i] = 0;
  }

  for (;;) {
    __syncwarp();
    // ---- phase vote ----
    const unsigned mS = __ballot_sync(kFull, state == ST_SEG);
    const unsigned mC = __ballot_sync(kFull, state == ST_COLL);
    const unsigned mE = __ballot_sync(kFull, state == ST_EPI);
    const int nS = __popc(mS), nC = __popc(mC), nE = __popc(mE);
    if ((nS | nC | nE) == 0) break;
    int phase;
    if (nC >= P.vote_coll || (nS == 0 && nC > 0 && nC >= nE)) phase = ST_COLL;
    else if (nE >= P.vote_epi || (nS == 0 && nE > 0)) phase = ST_EPI;
    else phase = ST_SEG;

    if (phase == ST_SEG) {
      if (STATS && lane == 0) { stc[S_WI_SEG]++; stc[S_LS_SEG] += nS; }
      if (state == ST_SEG) {
        bool dead = false;
        const NucDev<R> &nu = s_nuc[tgt];
        if (nseg >= kMaxSeg) {                       // R-C2 cap
          st_try |= INC_ST_SEG_CAP;
          if (STATS) stc[S_ABSORBED]++;
          dead = true;
        } else {
          nseg++;
          if (STATS) stc[S_SEG]++;
          // ---------- C2: segment (R-Q8 partner first, then the path) ----------
          R u[4];
          draw4<R>(g, attempt, pi, kblk++, u);
          const ShellDev<R> &sh = nu.sh[shell];
          const R m1 = nucleon_mass<R>(type);
          const R p1sq = px * px + py * py + pz * pz;
          const R E1 = M<R>::sqrt_(p1sq + m1 * m1);
          const R T1 = M<R>::div_(p1sq, E1 + m1);
          // partner direction and magnitude fraction ("quadratic distribution")
          const R cth = R(2) * u[1] - R(1);
          R s2 = R(1) - cth * cth;
          s2 = s2 > R(0) ? s2 : R(0);
          const R sth = M<R>::sqrt_(s2);
          R sph, cph;
          M<R>::sincos2pi(u[2], &sph, &cph);
          const R nx = sth * cph, ny = sth * sph, nz = cth;
          const R f = M<R>::cbrt_(u[0]);
          const R pn = px * nx + py * ny + pz * nz;
          // cross sections against a proton and a neutron partner (same n, f: R-C2)
          const R plab_p = plab_of<R>(m1, T1, pn, sh.pF_p * f, K<R>::mp);
          const R plab_n = plab_of<R>(m1, T1, pn, sh.pF_n * f, K<R>::mn);
          int kp, kn; R fp, fn;
          grid_pos<R>(plab_p, inv_dp, n_xs, kp, fp);
          grid_pos<R>(plab_n, inv_dp, n_xs, kn, fn);
          // tabS row: {sig_pp, d, sig_np, d}; vs proton: pp if type==1 else np; vs neutron: opposite
          const R *rp = s_tabS + 4 * kp + (type ? 0 : 2);
          const R *rn = s_tabS + 4 * kn + (type ? 2 : 0);
          const R sig_p = rp[0] + fp * rp[1];
          const R sig_n = rn[0] + fn * rn[1];
          const R Sp = sh.rho_p * sig_p, Sn = sh.rho_n * sig_n;
          const R Sig = Sp + Sn;
          const R d_coll = Sig > R(0) ? M<R>::div_(-M<R>::log_(u[3]), Sig) : R(1e30);
          // geometry: distances to the shell spheres along the flight direction
          const R ip = M<R>::rsqrt_(p1sq);
          const R dx = px * ip, dy = py * ip, dz = pz * ip;
          const R beta = x * dx + y * dy + z * dz;
          const R r2 = x * x + y * y + z * z;
          const R r_in = R(shell) * nu.dr, r_out = R(shell + 1) * nu.dr;
          R disc_out = beta * beta - r2 + r_out * r_out;
          disc_out = disc_out > R(0) ? disc_out : R(0);
          const R d_out = -beta + M<R>::sqrt_(disc_out);
          R d_in = R(1e30);
          if (shell > 0 && beta < R(0)) {
            const R D = beta * beta - r2 + r_in * r_in;
            if (D > R(0)) d_in = -beta - M<R>::sqrt_(D);
          }
          const bool inward = d_in < d_out;
          const R d_min = inward ? d_in : d_out;
          if (d_coll < d_min) {
            // collision point reached first: defer the collision to the COLL phase
            x += d_coll * dx; y += d_coll * dy; z += d_coll * dz;
            c_f = f; c_nx = nx; c_ny = ny; c_nz = nz; c_Sp = Sp; c_Sig = Sig;
            state = ST_COLL;
          } else {
            // ---------- C4: shell boundary, potential step (P:49 refraction/reflection) ----------
            if (STATS) stc[S_BND]++;
            const int j = inward ? shell - 1 : shell + 1;
            const R rb = inward ? r_in : r_out;
            x += d_min * dx; y += d_min * dy; z += d_min * dz;
            const R irr = M<R>::rsqrt_(x * x + y * y + z * z);
            const R ux = x * irr, uy = y * irr, uz = z * irr;   // outward normal
            x = ux * rb; y = uy * rb; z = uz * rb;                // renormalise onto the sphere
            const R pr = px * ux + py * uy + pz * uz;
            const R Vi = type ? sh.V_p : sh.V_n;
            const R Vj = type ? nu.sh[j].V_p : nu.sh[j].V_n;
            const R dV = Vj - Vi;
            const R Tj = T1 + dV;
            const R prj2 = pr * pr + dV * (T1 + Tj + R(2) * m1);  // p_j^2 - p_t^2
            if (Tj <= R(0) || prj2 <= R(0)) {
              if (STATS) stc[S_REFL]++;
              const R t2 = R(2) * pr;
              px -= t2 * ux; py -= t2 * uy; pz -= t2 * uz;         // specular reflection
            } else {
              const R prj = pr >= R(0) ? M<R>::sqrt_(prj2) : -M<R>::sqrt_(prj2);
              const R dp = prj - pr;
              px += dp * ux; py += dp * uy; pz += dp * uz;
              shell = j;
              if (j == nu.ns) {
                // escape: append to the event's list ("SoA ... exiting particles")
                if (STATS) stc[S_ESC]++;
                dead = true;
                if (n_esc < kMaxSec) {
                  const R ipj = M<R>::rsqrt_(px * px + py * py + pz * pz);
                  const size_t o = (size_t)ev * kMaxSec + n_esc;
                  P.ws.st_code[o] = pi | ((uint32_t)type << 24);
                  P.ws.st_T[o] = Tj;
                  P.ws.st_ux[o] = px * ipj; P.ws.st_uy[o] = py * ipj; P.ws.st_uz[o] = pz * ipj;
                  n_esc++; n_p += type;
                  Eavail -= Tj; Prx -= px; Pry -= py; Prz -= pz;
                } else {
                  st_try |= INC_ST_SEC_TRUNC;
                }
              }
            }
          }
        }
        if (dead) {
          if (sp > 0) {
            const TrackRec<R> &t = stack[--sp];
            x = t.x; y = t.y; z = t.z; px = t.px; py = t.py; pz = t.pz;
            pi = t.pi; type = t.meta & 1; shell = (int)(t.meta >> 1);
            kblk = 0; nseg = 0;
          } else {
            state = ST_EPI;
          }
        }
      }
    } else if (phase == ST_COLL) {
      if (STATS && lane == 0) { stc[S_WI_COLL]++; stc[S_LS_COLL] += nC; }
      if (state == ST_COLL) {
        // ---------- C3: collision ----------
        if (STATS) stc[S_COLL]++;
        const NucDev<R> &nu = s_nuc[tgt];
        const ShellDev<R> &sh = nu.sh[shell];
        R u[4];
        draw4<R>(g, attempt, pi, kblk++, u);
        const int t2 = (u[0] * c_Sig < c_Sp) ? 1 : 0;
        const R m1 = nucleon_mass<R>(type), m2 = nucleon_mass<R>(t2);
        const R q = (t2 ? sh.pF_p : sh.pF_n) * c_f;
        const R p2x = q * c_nx, p2y = q * c_ny, p2z = q * c_nz;
        const R p1sq = px * px + py * py + pz * pz;
        const R E1 = M<R>::sqrt_(p1sq + m1 * m1);
        const R T1 = M<R>::div_(p1sq, E1 + m1);
        const R E2 = M<R>::sqrt_(q * q + m2 * m2);
        const R pn = px * c_nx + py * c_ny + pz * c_nz;
        const R plab = plab_of<R>(m1, T1, pn, q, m2);
        int kk; R ff;
        grid_pos<R>(plab, inv_dp, n_xs, kk, ff);
        const bool same = (t2 == type);
        const R *row = P.model.tabC + 8 * kk;
        const R B = same ? (__ldg(row + 0) + ff * __ldg(row + 1)) : (__ldg(row + 2) + ff * __ldg(row + 3));
        const R ab = same ? R(0) : (__ldg(row + 4) + ff * __ldg(row + 5));
        // boost to the CM frame
        const R Px = px + p2x, Py = py + p2y, Pz = pz + p2z;
        const R E = E1 + E2;
        const R s = E * E - (Px * Px + Py * Py + Pz * Pz);
        const R iE = R(1) / E;
        const R bx = Px * iE, by = Py * iE, bz = Pz * iE;
        const R gam = E * M<R>::rsqrt_(s);
        const R gfac = gam * gam / (gam + R(1));        // (gamma - 1) / beta^2
        const R pb = px * bx + py * by + pz * bz;
        const R fb = gfac * pb - gam * E1;
        const R qx = px + fb * bx, qy = py + fb * by, qz = pz + fb * bz;   // p1 in the CM frame
        const R pcm2 = qx * qx + qy * qy + qz * qz;
        const R ipcm = M<R>::rsqrt_(pcm2);
        const R pcm = pcm2 * ipcm;
        // scattering angle: dsigma/dt ~ exp(B t), t in (GeV/c)^2 (R-Q10)
        const R pg2 = pcm2 * R(1e-6);
        const R tmin = R(-4) * pg2;
        R t;
        if (B * (-tmin) < R(1e-9)) t = u[1] * tmin;
        else t = M<R>::log1p_(-u[1] * (-M<R>::expm1_(B * tmin))) / B;
        R ct = R(1) + t / (R(2) * pg2);
        ct = ct < R(-1) ? R(-1) : (ct > R(1) ? R(1) : ct);
        if (!same && u[2] * (R(1) + ab) < ab) ct = -ct;       // np backward term
        R st2 = R(1) - ct * ct;
        const R stt = M<R>::sqrt_(st2 > R(0) ? st2 : R(0));
        R sphi, cphi;
        M<R>::sincos2pi(u[3], &sphi, &cphi);
        // rotation frame around n = q/|q|
        const R n0 = qx * ipcm, n1 = qy * ipcm, n2 = qz * ipcm;
        const R q2 = n0 * n0 + n1 * n1;
        R e1x, e1y, e1z, e2x, e2y;
        if (q2 > R(1e-24)) {
          const R iq = M<R>::rsqrt_(q2);
          e1x = n0 * n2 * iq; e1y = n1 * n2 * iq; e1z = -q2 * iq;
          e2x = -n1 * iq; e2y = n0 * iq;
        } else {
          e1x = R(1); e1y = R(0); e1z = R(0);
          e2x = R(0); e2y = n2 >= R(0) ? R(1) : R(-1);
        }
        const R a1 = stt * cphi, a2 = stt * sphi;
        const R w1x = pcm * (a1 * e1x + a2 * e2x + ct * n0);
        const R w1y = pcm * (a1 * e1y + a2 * e2y + ct * n1);
        const R w1z = pcm * (a1 * e1z + ct * n2);
        // boost back; partner by momentum conservation
        const R E1cm = M<R>::sqrt_(pcm2 + m1 * m1);
        const R wb = w1x * bx + w1y * by + w1z * bz;
        const R fo = gfac * wb + gam * E1cm;
        const R o1x = w1x + fo * bx, o1y = w1y + fo * by, o1z = w1z + fo * bz;
        const R o2x = Px - o1x, o2y = Py - o1y, o2z = Pz - o1z;
        const R o1sq = o1x * o1x + o1y * o1y + o1z * o1z;
        const R o2sq = o2x * o2x + o2y * o2y + o2z * o2z;
        // Pauli blocking: both products above their Fermi energies (strict, R-Q12)
        const R pF2_1 = type ? sh.pF2_p : sh.pF2_n;
        const R pF2_2 = t2 ? sh.pF2_p : sh.pF2_n;
        if (!(o1sq > pF2_1 && o2sq > pF2_2)) {
          if (STATS) stc[S_BLOCKED]++;
          state = ST_SEG;                                  // projectile continues unchanged (R-Q13)
        } else {
          n_real++;
          if (STATS) stc[S_ALLOWED]++;
          bool keep1 = false, keep2 = false;
          if (2u * pi + 1u >= (1u << 24)) {                // depth cap (R-C3)
            st_try |= INC_ST_DEPTH_CAP;
            if (STATS) stc[S_ABSORBED] += 2;
          } else {
            // cutoff: E_F + E_B (n), E_F + E_B + E_C (p)
            keep1 = o1sq > (type ? sh.pc2_p : sh.pc2_n);
            keep2 = o2sq > (t2 ? sh.pc2_p : sh.pc2_n);
            if (STATS) stc[S_ABSORBED] += (keep1 ? 0 : 1) + (keep2 ? 0 : 1);
          }
          const uint32_t pi0 = 2u * pi, pi1 = 2u * pi + 1u;
          if (keep1 && keep2) {
            if (sp < kStackCap) {
              TrackRec<R> &t = stack[sp++];
              t.x = x; t.y = y; t.z = z; t.px = o2x; t.py = o2y; t.pz = o2z;
              t.pi = pi1; t.meta = (uint32_t)t2 | ((uint32_t)shell << 1);
            } else {
              st_try |= INC_ST_QUEUE_OVF;
            }
          }
          if (keep1) {
            px = o1x; py = o1y; pz = o1z; pi = pi0; kblk = 0; nseg = 0;
            state = ST_SEG;
          } else if (keep2) {
            px = o2x; py = o2y; pz = o2z; pi = pi1; type = t2; kblk = 0; nseg = 0;
            state = ST_SEG;
          } else if (sp > 0) {
            const TrackRec<R> &t = stack[--sp];
            x = t.x; y = t.y; z = t.z; px = t.px; py = t.py; pz = t.pz;
            pi = t.pi; type = t.meta & 1; shell = (int)(t.meta >> 1);
            kblk = 0; nseg = 0;
            state = ST_SEG;
          } else {
            state = ST_EPI;
          }
        }
      }
    } else {  // ---------- EPI phase: epilogue of the finished attempt, then entry of the next ----------
      if (STATS && lane == 0) { stc[S_WI_EPI]++; stc[S_LS_EPI] += nE; }
      bool want_event = false;
      if (state == ST_EPI) {
        if (ev >= 0) {
          // ---------- C6: epilogue ("excitation energy ... through energy conservation") ----------
          const NucDev<R> &nu = s_nuc[tgt];
          const int A_res = nu.A + 1 - n_esc, Z_res = nu.Z + 1 - n_p;
          bool ok = (n_real > 0) || keep_transparent;
          R Estar = R(0);
          if (ok) {
            R Bres = R(-1e30);
            if (A_res >= 1 && A_res < kAmax && Z_res >= 0 && Z_res < kZmax) Bres = __ldg(P.model.bind + A_res * kZmax + Z_res);
            if (Bres < R(-1e29)) ok = false;                 // no such nucleus: retry
            else {
              // E_res - M_res = X, with the nucleon masses cancelled analytically
              const R X = Eavail + Bres - nu.Bt;
              const R Mres = R(Z_res) * K<R>::mp + R(A_res - Z_res) * K<R>::mn - Bres;
              const R P2 = Prx * Prx + Pry * Pry + Prz * Prz;
              const R Er = Mres + X;
              const R M2 = Er * Er - P2;
              const R Mstar = M2 > R(0) ? M<R>::sqrt_(M2) : R(0);
              Estar = (R(2) * Mres * X + X * X - P2) / (Mstar + Mres);
              if (Estar < R(0) && !(keep_transparent && n_real == 0)) ok = false;
            }
          }
          if (ok) {
            P.ws.cA[ev] = A_res; P.ws.cZ[ev] = Z_res; P.ws.cE[ev] = Estar;
            P.ws.cPx[ev] = Prx; P.ws.cPy[ev] = Pry; P.ws.cPz[ev] = Prz;
            P.ws.cmeta[ev] = (uint32_t)n_esc | (attempt << 8);
            const uint32_t used = attempt + 1u > 255u ? 255u : attempt + 1u;
            P.ws.cstatus[ev] = st_try | used;
            ev = -1;
          } else {
            attempt++;
            if (attempt >= (uint32_t)kMaxAttempt) {          // FAILED: count 0, target at rest
              P.ws.cA[ev] = nu.A; P.ws.cZ[ev] = nu.Z; P.ws.cE[ev] = R(0);
              P.ws.cPx[ev] = R(0); P.ws.cPy[ev] = R(0); P.ws.cPz[ev] = R(0);
              P.ws.cmeta[ev] = (1u << 16);
              P.ws.cstatus[ev] = INC_ST_FAILED | 0xFFu;
              if (STATS) stc[S_FAILED]++;
              ev = -1;
            }
          }
        }
        want_event = (ev < 0);
      }
      // ---- warp-aggregated event fetch (convergent) ----
      const unsigned need = __ballot_sync(kFull, want_event);
      if (need) {
        const int leader = __ffs(need) - 1;
        unsigned long long base = 0;
        if (lane == leader) base = atomicAdd(&P.ctr->next_event_casc, (unsigned long long)__popc(need));
        base = __shfl_sync(kFull, base, leader);
        if (want_event) {
          const unsigned long long mine = base + (unsigned long long)__popc(need & ((1u << lane) - 1u));
          if (mine < (unsigned long long)P.n_chunk) {
            ev = (int)mine;
            attempt = 0;
            E_in = P.E_in[ev];
            tgt = P.target_id[ev];
            unsigned err = 0;
            if (!(E_in >= R(INC_E_MIN) && E_in <= R(INC_E_MAX))) err |= 1u;
            if (tgt < 0 || tgt >= INC_MAX_TARGETS || !s_nuc[tgt < 0 ? 0 : (tgt >= INC_MAX_TARGETS ? 0 : tgt)].live) err |= 2u;
            if (err) {
              atomicOr(&P.ctr->error_word, err);
              // neutral outputs; the call returns INC_E_BADARG
              P.ws.cA[ev] = 0; P.ws.cZ[ev] = 0; P.ws.cE[ev] = R(0);
              P.ws.cPx[ev] = R(0); P.ws.cPy[ev] = R(0); P.ws.cPz[ev] = R(0);
              P.ws.cmeta[ev] = (1u << 16); P.ws.cstatus[ev] = INC_ST_FAILED;
              ev = -1;
              state = ST_EPI;    // try again for another event on the next EPI pass
            } else {
              const unsigned long long ge = same_stream ? 0ull : (unsigned long long)(P.e_base + ev);
              g.e0 = (uint32_t)ge; g.e1 = (uint32_t)(ge >> 32);
              if (STATS) stc[S_EVENTS]++;
            }
          } else {
            state = ST_DONE;
          }
        }
      }
      if (state == ST_EPI && ev >= 0) {
        // ---------- C0: entry — uniform disc, beam along +z (R-Q15) ----------
        if (STATS) stc[S_ATTEMPTS]++;
        const NucDev<R> &nu = s_nuc[tgt];
        R u[4];
        draw4<R>(g, attempt, 1u, 0u, u);
        const R b = nu.Rn * M<R>::sqrt_(u[0]);
        R sb, cb;
        M<R>::sincos2pi(u[1], &sb, &cb);
        x = b * cb; y = b * sb;
        R zz = nu.Rn * nu.Rn - b * b;
        z = -M<R>::sqrt_(zz > R(0) ? zz : R(0));
        const R p_in = M<R>::sqrt_(E_in * (E_in + R(2) * K<R>::mp));
        // potential step into the outermost shell (cannot reflect: V rises inward)
        const R ir = R(1) / nu.Rn;
        const R ux = x * ir, uy = y * ir, uz = z * ir;
        const R pr = p_in * uz;
        const R dV = nu.sh[nu.ns - 1].V_p;
        const R Tj = E_in + dV;
        const R prj2 = pr * pr + dV * (E_in + Tj + R(2) * K<R>::mp);
        const R prj = -M<R>::sqrt_(prj2 > R(0) ? prj2 : R(0));
        const R dp = prj - pr;
        px = dp * ux; py = dp * uy; pz = p_in + dp * uz;
        type = 1; shell = nu.ns - 1; pi = 1u; kblk = 1u; nseg = 0;
        Eavail = E_in; Prx = R(0); Pry = R(0); Prz = p_in;
        n_esc = 0; n_p = 0; n_real = 0; st_try = 0; sp = 0;
        state = ST_SEG;
      }
    }
  }

  if (STATS) {
#pragma unroll
    for (int i = 0; i < S_NSTAT; ++i) {
      unsigned long long v = stc[i];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
      if (lane == 0 && v) atomicAdd(&P.ctr->stats[i], v);
    }
  }
}

// =================================================================================================
// Evaporation: Weisskopf-Ewing emission of n, p, d, t, 3He, 4He until no channel is
// open.  One lane = one nucleus at a time; one emission step per warp pass; lanes refill.
// =================================================================================================
__constant__ int c_evA[6] = {1, 1, 2, 3, 3, 4};
__constant__ int c_evZ[6] = {0, 1, 1, 1, 2, 2};

template <typename R> struct EvapParams {
  ModelDev<R> model;
  Workspace<R> ws;
  DevCounters *ctr;
  long long e_base;
  int n_chunk;
  uint32_t seed_lo, seed_hi;
  uint32_t flags;
  // final outputs (caller arrays, chunk base)
  int32_t *out_counts;
  int32_t *rA, *rZ;
  R *rE, *rPx, *rPy, *rPz;
  uint32_t *rstatus;
};

// G_n(s) e^{-s_ref} with G_n(s) = int_0^s t^n e^t dt, n = 1 or 3 (closed forms of R-E2)
template <typename R>
__device__ __forceinline__ void G13_scaled(R s, R s_ref, R &g1, R &g3) {
  if (s < R(1)) {
    // series sum_k s^(n+1+k) / (k! (n+1+k)); the closed forms cancel catastrophically here
    R term = s * s;   // s^(2+k)/k!
    R a1 = R(0), a3 = R(0);
#pragma unroll 1
    for (int k = 0; k < M<R>::kSeriesTerms; ++k) {
      a1 += term / R(k + 2);
      a3 += term * s * s / R(k + 4);
      term *= s / R(k + 1);
    }
    const R e = M<R>::exp_(-s_ref);
    g1 = a1 * e; g3 = a3 * e;
  } else {
    const R e1 = M<R>::exp_(s - s_ref), e0 = M<R>::exp_(-s_ref);
    g1 = (s - R(1)) * e1 + e0;
    g3 = (((s - R(3)) * s + R(6)) * s - R(6)) * e1 + R(6) * e0;
  }
}

template <typename R, bool STATS>
__global__ void __launch_bounds__(256, 2) evap_kernel(const EvapParams<R> P) {
  const int lane = threadIdx.x & 31;
  const bool cascade_only = (P.flags & INC_F_CASCADE_ONLY) != 0;
  const bool same_stream = (P.flags & INC_F_SAME_STREAM) != 0;
  int ev = -1;
  int A = 0, Z = 0, count = 0;
  R Es = 0, Px = 0, Py = 0, Pz = 0;
  uint32_t status = 0, attempt = 0, kblk = 0;
  RngKey g;
  g.k0 = P.seed_lo; g.k1 = P.seed_hi; g.e0 = 0; g.e1 = 0;
  bool exhausted = false;
  unsigned long long n_steps = 0, n_trials = 0, n_emit = 0;

  for (;;) {
    __syncwarp();
    // ---- refill idle lanes ----
    const unsigned need = __ballot_sync(kFull, ev < 0 && !exhausted);
    if (need) {
      const int leader = __ffs(need) - 1;
      unsigned long long base = 0;
      if (lane == leader) base = atomicAdd(&P.ctr->next_event_evap, (unsigned long long)__popc(need));
      base = __shfl_sync(kFull, base, leader);
      if (ev < 0 && !exhausted) {
        const unsigned long long mine = base + (unsigned long long)__popc(need & ((1u << lane) - 1u));
        if (mine < (unsigned long long)P.n_chunk) {
          ev = (int)mine;
          A = P.ws.cA[ev]; Z = P.ws.cZ[ev]; Es = P.ws.cE[ev];
          Px = P.ws.cPx[ev]; Py = P.ws.cPy[ev]; Pz = P.ws.cPz[ev];
          const uint32_t meta = P.ws.cmeta[ev];
          count = (int)(meta & 0xFFu); attempt = (meta >> 8) & 0xFFu;
          status = P.ws.cstatus[ev];
          kblk = 0;
          const unsigned long long ge = same_stream ? 0ull : (unsigned long long)(P.e_base + ev);
          g.e0 = (uint32_t)ge; g.e1 = (uint32_t)(ge >> 32);
          if ((meta >> 16) & 1u) count = 0;   // FAILED or rejected input
        } else {
          exhausted = true;
        }
      }
    }
    if (__ballot_sync(kFull, ev >= 0) == 0) break;
    if (ev < 0) continue;

    bool finish = cascade_only || !(Es > R(0)) || (status & INC_ST_FAILED);
    if (!finish) {
      // ---------- E1/E2: channel widths ----------
      const R Bpar = __ldg(P.model.bind + A * kZmax + Z);
      R Xj[6], sj[6], aj[6];
      EvChan<R> ch[6];
      R s_ref = R(0);
      bool any = false;
#pragma unroll
      for (int j = 0; j < 6; ++j) {
        const int Ad = A - c_evA[j], Zd = Z - c_evZ[j];
        Xj[j] = R(-1); sj[j] = R(0); aj[j] = R(1);
        ch[j].pref = R(0); ch[j].V = R(0); ch[j].beta = R(0); ch[j].BdBj = R(0);
        if (Ad >= 1 && Zd >= 0 && Zd <= Ad) {
          const EvChan<R> c = P.model.evch[(Ad * kZmax + Zd) * 6 + j];
          if (c.pref > R(0)) {
            const R X = Es - Bpar + c.BdBj - c.V;
            if (X > R(0)) {
              ch[j] = c;
              Xj[j] = X;
              aj[j] = R(Ad) / P.model.a_div;
              sj[j] = R(2) * M<R>::sqrt_(aj[j] * X);
              s_ref = sj[j] > s_ref ? sj[j] : s_ref;
              any = true;
            }
          }
        }
      }
      if (!any) finish = true;
      else if (count >= kMaxSec) { status |= INC_ST_SEC_TRUNC; finish = true; }
      else {
        if (STATS) n_steps++;
        R W[6];
        R Wsum = R(0);
#pragma unroll
        for (int j = 0; j < 6; ++j) {
          W[j] = R(0);
          if (Xj[j] > R(0)) {
            R g1, g3;
            G13_scaled<R>(sj[j], s_ref, g1, g3);
            const R I0 = g1 / (R(2) * aj[j]);
            const R I1 = Xj[j] * I0 - g3 / (R(8) * aj[j] * aj[j]);
            R w = ch[j].pref * (I1 + ch[j].beta * I0);
            W[j] = w > R(0) ? w : R(0);
            Wsum += W[j];
          }
        }
        if (!(Wsum > R(0))) finish = true;
        else {
          // ---------- E3: choose the channel ----------
          R u[4];
          draw4<R>(g, attempt, 0u, kblk++, u);
          int jsel = -1;
          R cum = R(0);
          const R thr = u[0] * Wsum;
          bool done = false;
#pragma unroll
          for (int j = 0; j < 6; ++j) {
            if (!done && W[j] > R(0)) { cum += W[j]; jsel = j; if (thr < cum) done = true; }
          }
          R X = R(0), a = R(1), beta = R(0), V = R(0), BdBj = R(0);
#pragma unroll
          for (int j = 0; j < 6; ++j) if (j == jsel) { X = Xj[j]; a = aj[j]; beta = ch[j].beta; V = ch[j].V; BdBj = ch[j].BdBj; }
          // ---------- E4: rejection sampling of x (two envelopes, R-E4) ----------
          const R s = R(2) * M<R>::sqrt_(a * X);
          const R T = M<R>::sqrt_(X / a);
          const R areaA = T * (T + beta), areaB = R(0.5) * X * X + beta * X;
          R xs = R(-1);
#pragma unroll 1
          for (int n = 0; n < kMaxTrial; ++n) {
            R v[4];
            draw4<R>(g, attempt, 0u, kblk++, v);
            if (STATS) n_trials++;
            R xx;
            if (areaB < areaA) {
              xx = -beta + M<R>::sqrt_(beta * beta + v[1] * (X * X + R(2) * beta * X));
              R rem = X - xx;
              rem = rem > R(0) ? rem : R(0);
              if (M<R>::log_(v[3]) < R(2) * M<R>::sqrt_(a * rem) - s) { xs = xx < X ? xx : X; break; }
            } else {
              if (v[0] * (T + beta) < T) xx = -T * M<R>::log_(v[1] * v[2]);
              else xx = -T * M<R>::log_(v[1]);
              if (xx < X && M<R>::log_(v[3]) < R(2) * M<R>::sqrt_(a * (X - xx)) - s + xx / T) { xs = xx; break; }
            }
          }
          if (xs < R(0)) { status |= INC_ST_TRIAL_CAP; finish = true; }
          else {
            // ---------- E5: two-body decay in the parent rest frame, isotropic, boost to lab ----------
            const int Aj = c_evA[jsel], Zj = c_evZ[jsel];
            const int Ad = A - Aj, Zd = Z - Zj;
            const R Bj = __ldg(P.model.bind + Aj * kZmax + Zj);
            const R Mj = R(Zj) * K<R>::mp + R(Aj - Zj) * K<R>::mn - Bj;
            const R Bd = BdBj - Bj;
            const R Esd = X - xs;
            const R Mds = R(Zd) * K<R>::mp + R(Ad - Zd) * K<R>::mn - Bd + Esd;
            const R Mpar = R(Z) * K<R>::mp + R(A - Z) * K<R>::mn - Bpar + Es;
            const R eps = V + xs;   // total kinetic energy released in the parent frame
            const R p2 = eps * (R(2) * Mpar - eps) * (R(2) * Mds + eps) * (R(2) * Mj + eps) / (R(4) * Mpar * Mpar);
            const R pm = M<R>::sqrt_(p2 > R(0) ? p2 : R(0));
            const R Ej = M<R>::sqrt_(p2 + Mj * Mj);
            const R cth = R(2) * u[1] - R(1);
            R s2 = R(1) - cth * cth;
            const R sth = M<R>::sqrt_(s2 > R(0) ? s2 : R(0));
            R sph, cph;
            M<R>::sincos2pi(u[2], &sph, &cph);
            const R qx = pm * sth * cph, qy = pm * sth * sph, qz = pm * cth;
            const R Epar = M<R>::sqrt_(Mpar * Mpar + Px * Px + Py * Py + Pz * Pz);
            const R iEp = R(1) / Epar;
            const R bx = Px * iEp, by = Py * iEp, bz = Pz * iEp;
            const R gam = Epar / Mpar;
            const R gfac = gam * gam / (gam + R(1));
            const R fo = gfac * (qx * bx + qy * by + qz * bz) + gam * Ej;
            const R lx = qx + fo * bx, ly = qy + fo * by, lz = qz + fo * bz;
            const R l2 = lx * lx + ly * ly + lz * lz;
            const R El = M<R>::sqrt_(l2 + Mj * Mj);
            const R Tl = l2 / (El + Mj);
            const R il = M<R>::rsqrt_(l2);
            const size_t o = (size_t)ev * kMaxSec + count;
            P.ws.st_code[o] = 0x80000000u | ((uint32_t)jsel << 24) | (uint32_t)count;
            P.ws.st_T[o] = Tl;
            P.ws.st_ux[o] = lx * il; P.ws.st_uy[o] = ly * il; P.ws.st_uz[o] = lz * il;
            count++;
            if (STATS) n_emit++;
            A = Ad; Z = Zd; Es = Esd;
            Px -= lx; Py -= ly; Pz -= lz;
          }
        }
      }
    }
    if (finish) {
      P.out_counts[ev] = count;
      P.rA[ev] = A; P.rZ[ev] = Z; P.rE[ev] = Es;
      P.rPx[ev] = Px; P.rPy[ev] = Py; P.rPz[ev] = Pz;
      P.rstatus[ev] = status;
      ev = -1;
    }
  }
  if (STATS) {
    unsigned long long v[3] = {n_steps, n_trials, n_emit};
#pragma unroll
    for (int i = 0; i < 3; ++i) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v[i] += __shfl_xor_sync(kFull, v[i], o);
      if (lane == 0 && v[i]) atomicAdd(&P.ctr->stats[S_EVSTEPS + i], v[i]);
    }
  }
}

// =================================================================================================
// Output: exclusive prefix sum of the per-event counts, then canonical-order SoA compaction
// (BASELINE.json north_star "prefix-sum compaction of variable-length secondary lists into
// coalesced SoA buffers").
// =================================================================================================
constexpr int kScanBlock = 256;
constexpr int kScanItems = 8;                       // per thread
constexpr int kScanTile = kScanBlock * kScanItems;  // 2048 events per block

__device__ __forceinline__ long long block_exclusive_scan(long long v, long long *s_warp, long long &block_total) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  long long incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    long long t = __shfl_up_sync(kFull, incl, o);
    if (lane >= o) incl += t;
  }
  if (lane == 31) s_warp[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    long long w = lane < (kScanBlock / 32) ? s_warp[lane] : 0;
    long long wi = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      long long t = __shfl_up_sync(kFull, wi, o);
      if (lane >= o) wi += t;
    }
    if (lane < (kScanBlock / 32)) s_warp[lane] = wi - w;
    if (lane == (kScanBlock / 32) - 1) s_warp[kScanBlock / 32] = wi;
  }
  __syncthreads();
  block_total = s_warp[kScanBlock / 32];
  return incl - v + s_warp[wid];
}

// pass 1: per-tile sums
__global__ void __launch_bounds__(kScanBlock) scan_tile_sums(const int32_t *counts, int n, long long *tile_sums) {
  __shared__ long long s_warp[kScanBlock / 32 + 1];
  const int base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
  long long v = 0;
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) if (base + i < n) v += counts[base + i];
  long long total;
  block_exclusive_scan(v, s_warp, total);
  if (threadIdx.x == 0) tile_sums[blockIdx.x] = total;
}

// pass 2: one block scans the tile sums (n_tiles <= 2^20/2048 * ... loop) and adds the running base
__global__ void __launch_bounds__(kScanBlock) scan_tiles(long long *tile_sums, int n_tiles, unsigned long long *running_total) {
  __shared__ long long s_warp[kScanBlock / 32 + 1];
  __shared__ long long s_carry;
  if (threadIdx.x == 0) s_carry = (long long)*running_total;
  __syncthreads();
  for (int b = 0; b < n_tiles; b += kScanBlock) {
    const int i = b + threadIdx.x;
    const long long v = i < n_tiles ? tile_sums[i] : 0;
    long long total;
    const long long ex = block_exclusive_scan(v, s_warp, total);
    const long long carry = s_carry;
    if (i < n_tiles) tile_sums[i] = carry + ex;
    __syncthreads();
    if (threadIdx.x == 0) s_carry = carry + total;
    __syncthreads();
  }
  if (threadIdx.x == 0) *running_total = (unsigned long long)s_carry;
}

// pass 3: offsets[e] = tile base + exclusive scan inside the tile
__global__ void __launch_bounds__(kScanBlock) scan_write_offsets(const int32_t *counts, int n, const long long *tile_sums,
                                                                 long long *offsets) {
  __shared__ long long s_warp[kScanBlock / 32 + 1];
  const int base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
  int c[kScanItems];
  long long v = 0;
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) { c[i] = base + i < n ? counts[base + i] : 0; v += c[i]; }
  long long total;
  long long ex = block_exclusive_scan(v, s_warp, total) + tile_sums[blockIdx.x];
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) {
    if (base + i < n) offsets[base + i] = ex;
    ex += c[i];
  }
}

template <typename R> struct CompactParams {
  Workspace<R> ws;
  const long long *offsets;   // chunk-local array of global output offsets
  const int32_t *counts;
  int n_chunk;
  uint8_t *species;
  R *T, *ux, *uy, *uz;
  long long capacity;
};

// One warp per group of 32 events; lanes sweep the records of each event so that the stores of a
// warp cover one contiguous span of the output arrays.  Cascade records are placed by the rank of
// their path code (canonical order), evaporation records keep their emission order.
template <typename R>
__global__ void __launch_bounds__(256) compact_kernel(const CompactParams<R> P) {
  const int lane = threadIdx.x & 31;
  const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int e0 = warp * 32;
  if (e0 >= P.n_chunk) return;
  const int e = e0 + lane;
  long long off = 0;
  int cnt = 0;
  if (e < P.n_chunk) { off = P.offsets[e]; cnt = P.counts[e]; }
  // flatten (event, record) pairs of the 32 events over the lanes
  int incl = cnt;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int t = __shfl_up_sync(kFull, incl, o);
    if (lane >= o) incl += t;
  }
  const int total = __shfl_sync(kFull, incl, 31);
  const int excl = incl - cnt;
  for (int i0 = 0; i0 < total; i0 += 32) {
    const int i = i0 + lane;
    // find the event: largest l with excl_l <= i  (binary search over the 32 lanes' excl via shuffles)
    int lo = 0;
#pragma unroll
    for (int step = 16; step > 0; step >>= 1) {
      const int cand = lo + step;
      const int ex_c = __shfl_sync(kFull, excl, cand & 31);
      if (cand < 32 && ex_c <= i) lo = cand;
    }
    const int ex_l = __shfl_sync(kFull, excl, lo);
    const long long off_l = __shfl_sync(kFull, off, lo);
    if (i < total) {
      const int el = e0 + lo;
      const int j = i - ex_l;
      const size_t sbase = (size_t)el * kMaxSec;
      const uint32_t code = P.ws.st_code[sbase + j];
      int rank = j;
      uint8_t sp;
      if (code & 0x80000000u) {
        sp = (uint8_t)(0x80u | ((code >> 24) & 0x7u));
      } else {
        sp = (uint8_t)((code >> 24) & 1u);
        const uint32_t key = code & 0xFFFFFFu;
        const int n_casc = (int)(P.ws.cmeta[el] & 0xFFu);
        rank = 0;
        for (int l = 0; l < n_casc; ++l) rank += ((P.ws.st_code[sbase + l] & 0xFFFFFFu) < key) ? 1 : 0;
      }
      const long long dst = off_l + rank;
      if (dst < P.capacity) {
        P.species[dst] = sp;
        P.T[dst] = P.ws.st_T[sbase + j];
        P.ux[dst] = P.ws.st_ux[sbase + j];
        P.uy[dst] = P.ws.st_uy[sbase + j];
        P.uz[dst] = P.ws.st_uz[sbase + j];
      }
    }
  }
}

// ---- issue-peak microbenchmark: 8 independent FMA chains per thread ------------------------------
template <typename R>
__global__ void __launch_bounds__(256) fma_peak_kernel(R *out, int iters, R a, R b) {
  R v0 = R(threadIdx.x) * R(1e-3), v1 = v0 + R(1), v2 = v0 + R(2), v3 = v0 + R(3);
  R v4 = v0 + R(4), v5 = v0 + R(5), v6 = v0 + R(6), v7 = v0 + R(7);
#pragma unroll 1
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      v0 = fma(v0, a, b); v1 = fma(v1, a, b); v2 = fma(v2, a, b); v3 = fma(v3, a, b);
      v4 = fma(v4, a, b); v5 = fma(v5, a, b); v6 = fma(v6, a, b); v7 = fma(v7, a, b);
    }
  }
  R s = v0 + v1 + v2 + v3 + v4 + v5 + v6 + v7;
  if (s == R(123456.789)) out[0] = s;
}

__global__ void philox_blocks_kernel(const uint32_t *ctr, uint32_t k0, uint32_t k1, uint32_t *out, long long n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint4 o = philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], k0, k1);
  out[4 * i] = o.x; out[4 * i + 1] = o.y; out[4 * i + 2] = o.z; out[4 * i + 3] = o.w;
}

}  // namespace inc
