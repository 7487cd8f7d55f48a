// inc_common.cuh — constants, device-resident model data, staging / nucleus records, completion-list primitives, math
// wrappers (exact for double, MUFU-based for float), Philox4x32-10, table lookup, track state.  Part of inc_device.cuh.
#pragma once

namespace inc {

constexpr int kMaxShells = 32;
constexpr int kMaxSeg = 1024;      // R-C2
constexpr int kMaxAttempt = 256;   // R-C6
constexpr int kMaxTrial = 64;      // R-E4
constexpr int kMaxSec = INC_MAX_SEC;
constexpr int kStackCap = 16;      // lane kernel: pending tracks per event (INC_ST_QUEUE_OVF beyond)
constexpr int kAmax = 72;          // binding / channel tables cover 0..kAmax-1
constexpr int kZmax = 66;          // (inc_init accepts Z <= 62; the residual may carry one charge more)
constexpr unsigned kFull = 0xFFFFFFFFu;

// ---- physical constants (standard values; R-K) -----------------------------------------
template <typename R> struct K {
  static constexpr R mp = R(938.27208816);
  static constexpr R mn = R(939.56542052);
  static constexpr R imp = R(1.0 / 938.27208816);
  static constexpr R imn = R(1.0 / 939.56542052);
};

// ---- device-resident model data ----------------------------------------------------------
template <typename R> struct ShellDev {   // one constant-density shell; 16 reals
  R rho_p, rho_n;      // fm^-3
  R pF_p, pF_n;        // Fermi momenta, MeV/c
  R pF2_p, pF2_n;      // Pauli threshold on |p'|^2  (T' > E_F  <=>  p'^2 > pF^2)
  R pc2_p, pc2_n;      // cutoff threshold on |p'|^2 (T' - V <= cut <=> p'^2 <= pc2)
  R V_p, V_n;          // well depth E_F + E_B, MeV
  R r_in, r_out;       // shell radii i*dr, (i+1)*dr
  R ir_in, ir_out;     // reciprocals (ir_in = 0 for the innermost shell)
  R pad0, pad1;
};

template <typename R> struct NucDev {
  int32_t A, Z, ns, live;
  R Rn, dr, Bt, iRn;                       // radius, shell thickness, target binding energy, 1/R
  ShellDev<R> sh[kMaxShells + 1];          // [ns] = outside: V = 0
};

template <typename R> struct __align__(16) EvChan {        // per (A_d, Z_d, channel j): R-E1/E2 constants
  R V;        // Coulomb barrier of the channel
  R pref;     // g_j M_j A_d^(2/3) alpha_j   (0 => channel closed: daughter invalid)
  R beta;     // Dostrovsky beta (neutron) or 0
  R BdBj;     // B(A_d,Z_d) + B_j, so that X = E* - B(parent) + BdBj - V
};

// NEXT-2 (GEM level density, R-G2..G4): constants of one daughter nucleus; a = 0 => no level density (channel closed)
template <typename R> struct __align__(16) LdDev {
  R a, delta;     // level-density parameter MeV^-1, pairing energy MeV
  R Ux, Ex;       // matching energy U_x = 150/A_d + 2.5 and E_x = U_x + delta
  R T, E0;        // constant-temperature branch below E_x: rho = exp((U - E0)/T)/T
  R lnT, lna4;    // ln T, (1/4) ln a
};
template <typename R> struct GaussNodes { R x[16], w[16]; };
template <typename R> struct __align__(16) GemNode { R l0, d0, l1, d1; };
#ifndef INC_GEM_POINTS
#define INC_GEM_POINTS 1281             // (the checked test build uses 121, so that most steps take the direct-quadrature fallback)
#endif
constexpr int kGemPoints = INC_GEM_POINTS;   // table points per daughter nucleus: X = E_x .. E_x + 320 MeV
#define INC_GEM_STEP 0.25               // MeV
__constant__ GaussNodes<INC_REAL> c_gl;     // 16-point Gauss-Legendre on [-1, 1] (width integral of the GEM mode)

template <typename R> struct ModelDev {
  const R *tabS;          // [n_xs][4]  {sig_pp, dsig_pp, sig_np, dsig_np} in fm^2 (mb * 0.1)
  const R *tabC;          // [n_xs][8]  {B_pp, dB_pp, B_np, dB_np, a_np, da_np, 0, 0}
  const R *bind;          // [kAmax][kZmax] binding energy, MeV; < -1e29 => no such nucleus
  const EvChan<R> *evp;   // [kAmax][kZmax][8] by PARENT (A, Z): entries 0-5 the channels' constants (of the daughters
                          // (A - A_j, Z - Z_j); pref = 0: channel closed), entry 6: V = B(A, Z), entry 7 unused
  const LdDev<R> *ld;     // [kAmax][kZmax]  (level_density = 1 only)
  // GEM width integrals (R-G5) as tables built at inc_init: for daughter row r = ldrow[A_d * kZmax + Z_d] (-1: none) and
  // X_k = E_x + k * kGemStep, gtab[r * kGemPoints + k] = {ln J0, d ln J0 / dX, ln J1, d ln J1 / dX} with
  // J0(X) = int_0^X rho(U) dU and J1(X) = int_0^X (X - U) rho(U) dU, so that int_0^X (x + beta) rho(X - x) dx = J1 + beta J0
  const int32_t *ldrow;
  const GemNode<R> *gtab;
  const NucDev<R> *nuc;   // [INC_MAX_TARGETS]
  int32_t n_xs;
  R inv_dp;               // 1 / (grid step in MeV/c)
  R a_div;                // level density a = A_d / a_div
};

// One staged secondary.  f32: 32 bytes = one DRAM sector, so an event with n secondaries touches n sectors when it
// is written (cascade escapes, evaporation emissions) and when the compaction kernel reads it back; the earlier
// layout (five [chunk][64] arrays) touched 5-10 sectors per event and made the compaction the one HBM-bound kernel.
template <typename R> struct __align__(16) StageRec {
  R T, ux, uy, uz;
  uint32_t code;          // path code | type << 24 ; evaporation: 1 << 31 | species << 24 | sequence number
  uint32_t pad[3];
};

// One nucleus record per event: 32 bytes in the f32 build (one DRAM sector), 48 in f64.  Events finish, and are
// evaporated, in an order unrelated to their index, so a record that is one sector costs one sector of traffic
// where eight parallel arrays cost eight.  crec: post-cascade nucleus (the paper's "SoA of excited nuclei"),
// meta = n_casc | attempt << 8 | failed << 16.  frec: final residual, meta = number of secondaries | n_casc << 8; the
// compaction kernel, which walks the events in index order, transposes it into the caller's arrays.
template <typename R> struct __align__(16) NucRec {
  R E, Px, Py, Pz;
  int32_t A, Z;
  uint32_t meta, status;
};

// Staged secondaries: an event's first kStageMain records sit in its own row; an event that has more (R-C5 allows 64, the
// mean is 4-6) gets one row of the overflow pool for records kStageMain..63, its number kept in ovf_id[event].  The rows
// are then a quarter of what 64 records per event would take (2.1 GB instead of 8.6 GB at 2^22 events per chunk).
// (Of 6e4 250 MeV p-48Ti events none has more than 16 secondaries; the checked test build uses 4 per row.)
#ifndef INC_STAGE_MAIN
#define INC_STAGE_MAIN 16      // (the checked test build uses 4, so that the overflow rows are in constant use)
#endif
constexpr int kStageMain = INC_STAGE_MAIN;
constexpr int kStageOvf = kMaxSec - kStageMain;

template <typename R> struct Workspace {   // per-chunk internal buffers (DEVICE)
  StageRec<R> *st;        // [chunk][kStageMain] staged secondaries, one record per secondary
  StageRec<R> *ovf;       // [ovf_rows][kStageOvf] overflow pool
  int32_t *ovf_id;        // [chunk] overflow row of the event, -1 = none (-2 = being allocated)
  int32_t ovf_rows;
  NucRec<R> *crec;        // [chunk] post-cascade nuclei
  NucRec<R> *frec;        // [chunk] final residuals
  // Completion list: the cascade kernel appends the chunk-local index of every event whose post-cascade record is
  // complete; the evaporation kernel, which may start while the cascade kernel's last CTAs are still draining
  // (programmatic dependent launch), consumes the entries in order.  kNotDone = not written yet.
  uint32_t *done_list;    // [chunk]
};
constexpr uint32_t kNotDone = 0xFFFFFFFFu;

// release / acquire pair of the completion list (gpu scope)
__device__ __forceinline__ uint32_t ld_acquire_u32(const uint32_t *p) {
  uint32_t v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
// Warp-collective: publishes the events of the lanes with `pub` set.  Every lane's earlier global writes (post-cascade
// record; staged escapes, written by lanes of this warp in earlier passes and ordered by the __syncwarp()s since) are
// made visible before the entry (fence + release store).
__device__ __forceinline__ void publish_done(bool pub, int ev, unsigned long long *n_done, uint32_t *done_list, int lane) {
  const unsigned mp = __ballot_sync(kFull, pub);
  if (mp == 0u) return;
  const int leader = __ffs(mp) - 1;
  unsigned long long base = 0;
  if (lane == leader) base = atomicAdd(n_done, (unsigned long long)__popc(mp));
  base = __shfl_sync(kFull, base, leader);
  __threadfence();
  if (pub) *(volatile uint32_t *)(done_list + base + (unsigned long long)__popc(mp & ((1u << lane) - 1u))) = (uint32_t)ev;
}

template <typename R>
__device__ __forceinline__ void stage_write(StageRec<R> *dst, R T, R ux, R uy, R uz, uint32_t code) {
  StageRec<R> r;
  r.T = T; r.ux = ux; r.uy = uy; r.uz = uz; r.code = code; r.pad[0] = 0u; r.pad[1] = 0u; r.pad[2] = 0u;
  *dst = r;               // 16-byte vector stores
}

struct DevCounters {       // device scalars
  unsigned long long next_event_casc, next_event_evap;
  unsigned long long n_done;          // entries of the completion list handed out (cascade -> evaporation)
  unsigned long long ovf_next;        // rows of the staging overflow pool handed out
  unsigned long long total_sec;
  unsigned int error_word;   // bit0: E_in out of range, bit1: bad target id
  unsigned int pad;
  unsigned long long stats[24];
  // drain timeline of the wavefront kernel (INC_F_TIMING), %globaltimer ns (low 40 bits): [0] max of ~start
  // (= ~earliest start), [1] sum over warps of the time the event counter ran out for them, [2] sum of warp
  // exit times, [3] latest warp exit, [4] number of warps, [5] max of ~exit (= ~earliest exit)
  unsigned long long tl[6];
};

// Where record `idx` of event `ev` is staged.  Records beyond the event's own row go to its overflow row, allocated by
// whoever needs it first.  The cascade escapes of one event are written by lanes of ONE warp, possibly in the same pass:
// one claims the row (compare-and-swap -1 -> -2), the others wait for its number (independent thread scheduling lets
// lanes of a warp wait for each other; the wait is bounded all the same).  Returns nullptr if the pool is exhausted
// (error bit 64: the library runs the call again with a pool that has a row for every event).
// (the overflow part is a real function call: as inline code in the cascade kernel's escape block it cost the steady
// state 1.2 % without ever running)
template <typename R>
__device__ __noinline__ StageRec<R> *stage_slot_overflow(StageRec<R> *ovf, int32_t *ovf_id, int32_t ovf_rows, DevCounters *ctr, int ev, int idx) {
  Workspace<R> ws;
  ws.ovf = ovf; ws.ovf_id = ovf_id; ws.ovf_rows = ovf_rows;
  volatile int32_t *pid = ws.ovf_id + ev;
  int id = *pid;
  if (id < 0) {
    const int prev = atomicCAS(ws.ovf_id + ev, -1, -2);
    if (prev == -1) {
      const unsigned long long r = atomicAdd(&ctr->ovf_next, 1ull);
      id = r < (unsigned long long)ws.ovf_rows ? (int)r : 0x7FFFFFFF;
      if (id == 0x7FFFFFFF) atomicOr(&ctr->error_word, 64u);
      __threadfence();
      *pid = id;
    } else if (prev >= 0) {
      id = prev;
    } else {
      unsigned spins = 0;
      while ((id = *pid) < 0) { if (++spins > (1u << 26)) { atomicOr(&ctr->error_word, 16u); return nullptr; } }
    }
  }
  if (id == 0x7FFFFFFF) return nullptr;
  return ws.ovf + (size_t)id * kStageOvf + (idx - kStageMain);
}
template <typename R>
__device__ __forceinline__ StageRec<R> *stage_slot(const Workspace<R> &ws, DevCounters *ctr, int ev, int idx) {
  if (idx < kStageMain) return ws.st + (size_t)ev * kStageMain + idx;
  return stage_slot_overflow<R>(ws.ovf, ws.ovf_id, ws.ovf_rows, ctr, ev, idx);
}
// the same for a reader: the row exists
template <typename R>
__device__ __forceinline__ const StageRec<R> *stage_at(const Workspace<R> &ws, int ev, int idx, int ovf_row) {
  return idx < kStageMain ? ws.st + (size_t)ev * kStageMain + idx : ws.ovf + (size_t)ovf_row * kStageOvf + (idx - kStageMain);
}

__device__ __forceinline__ unsigned long long global_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
  return t & 0xFFFFFFFFFFull;     // 40 bits (18 minutes): sums over a few thousand warps stay far below 2^64
}

enum StatIdx { S_EVENTS = 0, S_FAILED, S_ATTEMPTS, S_SEG, S_BND, S_REFL, S_ESC, S_COLL, S_BLOCKED,
               S_ALLOWED, S_ABSORBED, S_EVSTEPS, S_EVTRIALS, S_EVEMIT, S_WI_SEG, S_WI_COLL, S_WI_EPI,
               S_LS_SEG, S_LS_COLL, S_LS_EPI, S_NSTAT };

template <bool ON> struct LaneStats {
  unsigned long long c[ON ? S_NSTAT : 1];
  __device__ __forceinline__ void clear() {
    if (ON) {
#pragma unroll
      for (int i = 0; i < S_NSTAT; ++i) c[i] = 0;
    }
  }
  __device__ __forceinline__ void add(int i, unsigned long long v = 1) { if (ON) c[i] += v; }
  __device__ __forceinline__ void flush(DevCounters *ctr, int lane) {
    if (ON) {
#pragma unroll
      for (int i = 0; i < S_NSTAT; ++i) {
        unsigned long long v = c[i];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
        if (lane == 0 && v) atomicAdd(&ctr->stats[i], v);
      }
    }
  }
};

// ---- math wrappers: exact library calls for double, MUFU-based approximations for float ------
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
  static __device__ __forceinline__ double rcp_(double a) { return 1.0 / a; }
  static __device__ __forceinline__ double u01(uint32_t x) {   // R-R3 (fp64): (x + 1/2) 2^-32
    return ((double)x + 0.5) * (1.0 / 4294967296.0);
  }
  // x >= 0 -> integer part k (clamped to kmax) and fraction
  static __device__ __forceinline__ void split(double x, int kmax, int &k, double &f) {
    int kk = (int)x;
    kk = kk > kmax ? kmax : kk;
    k = kk; f = x - (double)kk;
  }
  static constexpr int kSeriesTerms = 24;
  static __device__ __forceinline__ double series_below() { return 1.0; }
  // pinned arithmetic: never re-contracted by the compiler, so an inlined function gives the same bits at every
  // call site.  fp64: product and sum rounded separately, like the oracle (-ffp-contract=off).
  static __device__ __forceinline__ double mul_(double a, double b) { return __dmul_rn(a, b); }
  static __device__ __forceinline__ double add_(double a, double b) { return __dadd_rn(a, b); }
  static __device__ __forceinline__ double sub_(double a, double b) { return __dsub_rn(a, b); }
  static __device__ __forceinline__ double fma_(double a, double b, double c) { return __dadd_rn(__dmul_rn(a, b), c); }
};
template <> struct M<float> {
  static __device__ __forceinline__ float sqrt_(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
  static __device__ __forceinline__ float rsqrt_(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
  static __device__ __forceinline__ float lg2_(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
  static __device__ __forceinline__ float ex2_(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
  static __device__ __forceinline__ float log_(float x) { return __fmul_rn(0.6931471805599453f, lg2_(x)); }
  static __device__ __forceinline__ float exp_(float x) { return ex2_(1.4426950408889634f * x); }
  static __device__ __forceinline__ float cbrt_(float x) { return ex2_(__fmul_rn(0.3333333333f, lg2_(x))); }   // x in (0,1)
  static __device__ __forceinline__ float log1p_(float x) { return log1pf(x); }
  static __device__ __forceinline__ float expm1_(float x) { return expm1f(x); }
  static __device__ __forceinline__ void sincos2pi(float u, float *s, float *c) {
    // sin.approx / cos.approx scale their argument by 1/(2 pi) before MUFU: feed radians
    float a = __fmul_rn(6.283185307179586f, u);
    float ss, cc;
    asm("sin.approx.ftz.f32 %0, %1;" : "=f"(ss) : "f"(a));
    asm("cos.approx.ftz.f32 %0, %1;" : "=f"(cc) : "f"(a));
    *s = ss; *c = cc;
  }
  static __device__ __forceinline__ float rcp_(float a) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(a)); return y; }
  static __device__ __forceinline__ float div_(float a, float b) { return __fmul_rn(a, rcp_(b)); }
  static __device__ __forceinline__ float u01(uint32_t x) {
    // R-R3 (fp32): ((x>>9) + 1/2) 2^-23, built from the mantissa bits (no int->float conversion)
    return __uint_as_float(0x3F800000u | (x >> 9)) - 0.99999994f;
  }
  static __device__ __forceinline__ void split(float x, int kmax, int &k, float &f) {
    // round-to-nearest of (x - 1/2) by the 2^23 trick: stays on the FMA/ALU pipes.  A knot that is
    // mis-assigned by one ulp gives f just outside [0,1]; the interpolant is continuous there.
    float y = (x - 0.49999997f) + 8388608.0f;
    int kk = __float_as_int(y) - 0x4B000000;
    kk = kk < 0 ? 0 : (kk > kmax ? kmax : kk);
    k = kk; f = x - (y - 8388608.0f);
    f = kk == kmax ? x - (float)kmax : f;
  }
  static constexpr int kSeriesTerms = 13;
  // below this s the closed forms of G_1, G_3 are replaced by their series; at 0.25 the closed G_3 still has 3 of
  // f32's 7 digits (it only weighs channels that are 6 keV from closing), and the 13-iteration series loop, which
  // a single lane imposes on its whole warp, runs in 5 % instead of 84 % of the passes
  static __device__ __forceinline__ float series_below() { return 0.25f; }
  static __device__ __forceinline__ float mul_(float a, float b) { return __fmul_rn(a, b); }
  static __device__ __forceinline__ float add_(float a, float b) { return __fadd_rn(a, b); }
  static __device__ __forceinline__ float sub_(float a, float b) { return __fsub_rn(a, b); }
  static __device__ __forceinline__ float fma_(float a, float b, float c) { return __fmaf_rn(a, b, c); }
};

// ---- R-R1: Philox4x32-10 ---------------------------------------------------------------------
// The key is the call's seed for every block, so the ten round keys (key + r * Weyl constants) are the same for
// the whole call: the host writes them to constant memory once per call and the rounds read them as constant-bank
// operands, which takes the 20 key additions out of every block (4 % of the issue slots of a segment pass).
struct RoundKeys { uint32_t k0[10], k1[10]; };
__constant__ RoundKeys c_rk;

__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const unsigned long long p0 = (unsigned long long)0xD2511F53u * c0;   // one IMAD.WIDE each
    const unsigned long long p1 = (unsigned long long)0xCD9E8D57u * c2;
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    c0 = hi1 ^ c1 ^ c_rk.k0[r];
    c1 = lo1;
    c2 = hi0 ^ c3 ^ c_rk.k1[r];
    c3 = lo0;
  }
  return make_uint4(c0, c1, c2, c3);
}

struct RngKey {
  uint32_t k0, k1;   // seed (the rounds use its expansion c_rk)
  uint32_t e0, e1;   // global event index (counter words 2, 3)
};

// R-R2: block k of stream (attempt, path code pi)
template <typename R>
__device__ __forceinline__ void draw4(const RngKey &g, uint32_t attempt, uint32_t pi, uint32_t k, R u[4]) {
  uint4 o = philox4x32_10(k, (attempt << 24) | pi, g.e0, g.e1);
  u[0] = M<R>::u01(o.x); u[1] = M<R>::u01(o.y); u[2] = M<R>::u01(o.z); u[3] = M<R>::u01(o.w);
}

// ---- table lookup (R-N7): y_k + f (y_{k+1} - y_k), clamped to the grid -------------------------
template <typename R>
__device__ __forceinline__ void grid_pos(R plab_mev, R inv_dp, int n_xs, int &k, R &f) {
  R x = M<R>::mul_(plab_mev, inv_dp);
  const R xmax = R(n_xs - 1);
  x = x > xmax ? xmax : x;
  M<R>::split(x, n_xs - 2, k, f);
}

template <typename R> __device__ __forceinline__ R nucleon_mass(int type) { return type ? K<R>::mp : K<R>::mn; }
template <typename R> __device__ __forceinline__ R nucleon_imass(int type) { return type ? K<R>::imp : K<R>::imn; }

// Momentum of particle 1 (mass m1, total energy E1) in the rest frame of a partner with momentum q n
// (mass m2, 1/m2 = im2); pn = p1 . n.  E_lab = (E1 E2 - p1.p2)/m2 is the invariant s expression
// (s - m1^2 - m2^2)/(2 m2) of R-C2; p_lab = sqrt(T_lab (T_lab + 2 m1)), MeV/c.
template <typename R>
__device__ __forceinline__ R plab_of(R m1, R E1, R pn, R q, R m2, R im2) {
  const R E2 = M<R>::sqrt_(q * q + m2 * m2);
  const R Tlab = (E1 * E2 - q * pn) * im2 - m1;
  R a = Tlab * (Tlab + R(2) * m1);
  a = a > R(0) ? a : R(0);
  return M<R>::sqrt_(a);
}

// ---- track state ---------------------------------------------------------------------------------
template <typename R> struct Track {
  R x, y, z;          // position, fm
  R px, py, pz;       // momentum, MeV/c
  R T;                // kinetic energy, MeV (kept consistent with |p|)
  uint32_t pi;        // path code (R-R2)
  uint32_t k;         // next Philox block of this track's stream
  int nseg;           // segments done (R-C2 cap)
  int type, shell;    // 1 = proton, 0 = neutron; shell index
};

template <typename R> struct CollCarry { R f, nx, ny, nz, Sp, Sig; };   // SEG -> COLL hand-over
template <typename R> struct Escape { R T, ux, uy, uz; };

enum SegOutcome : int { SEG_REFLECT = -1, SEG_CONT = 0, SEG_COLLIDE = 1, SEG_ESCAPE = 2, SEG_CAP = 3 };

}  // namespace inc
