// inc_evap.cuh — evaporation: Weisskopf-Ewing widths (and the GEM level density), channel choice, rejection sampler,
// two-body emission; EvapLanes + evap_kernel.  Part of inc_device.cuh.
#pragma once

namespace inc {

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
  int32_t *out_counts;      // caller array, chunk base (the residual goes to ws.frec, see compact_kernel)
};

// G_n(s) e^{-s_ref} with G_n(s) = int_0^s t^n e^t dt, n = 1 or 3 (closed forms of R-E2)
template <typename R>
__device__ __forceinline__ void G13_scaled(R s, R s_ref, R &g1, R &g3) {
  if (s < M<R>::series_below()) {
    // series sum_k s^(n+1+k) / (k! (n+1+k)); the closed forms cancel catastrophically here
    R term = s * s;   // s^(2+k)/k!
    R a1 = R(0), a3 = R(0);
#pragma unroll 1
    for (int k = 0; k < M<R>::kSeriesTerms; ++k) {
      a1 += M<R>::div_(term, R(k + 2));
      a3 += M<R>::div_(term * s * s, R(k + 4));
      term *= M<R>::div_(s, R(k + 1));
    }
    const R e = M<R>::exp_(-s_ref);
    g1 = a1 * e; g3 = a3 * e;
  } else {
    const R e1 = M<R>::exp_(s - s_ref), e0 = M<R>::exp_(-s_ref);
    g1 = (s - R(1)) * e1 + e0;
    g3 = (((s - R(3)) * s + R(6)) * s - R(6)) * e1 + R(6) * e0;
  }
}

// ---- NEXT-2: GEM level density (DESIGN.md R-G1..G6) ----
// ln rho(U): Fermi gas with the pre-exponential factor above E_x, constant temperature below (R-G1, R-G5)
template <typename R>
__device__ __forceinline__ R gem_lnrho(const LdDev<R> &ld, R U) {
  if (U >= ld.Ex) {
    const R u = U - ld.delta;
    return R(2) * M<R>::sqrt_(ld.a * u) - ld.lna4 - R(1.25) * M<R>::log_(u);
  }
  return M<R>::div_(U - ld.E0, ld.T) - ld.lnT;
}

// int_x0^x1 (x + beta) rho(X - x) e^(-lref) dx: panels of at most 8 MeV, 16 Gauss-Legendre nodes each (R-G5: the
// definition, evaluated by quadrature)
template <typename R>
__device__ __forceinline__ R gem_range(const LdDev<R> &ld, R X, R beta, R x0, R x1, R lref) {
  if (!(x1 > x0)) return R(0);
  int np = (int)ceil((double)((x1 - x0) * R(0.125)));
  np = np < 1 ? 1 : np;
  const R h = M<R>::div_(x1 - x0, R(np));
  R sum = R(0);
#pragma unroll 1
  for (int p = 0; p < np; ++p) {
    const R a0 = x0 + h * R(p);
#pragma unroll 1
    for (int q = 0; q < 16; ++q) {
      const R x = a0 + R(0.5) * h * (c_gl.x[q] + R(1));
      R U = X - x;
      U = U < R(0) ? R(0) : U;
      sum += R(0.5) * h * c_gl.w[q] * (x + beta) * M<R>::exp_(gem_lnrho<R>(ld, U) - lref);
    }
  }
  return sum;
}

template <typename R>
__device__ __forceinline__ R gem_integral(const LdDev<R> &ld, R X, R beta, R lref) {
  const R xs = X - ld.Ex;                         // x below xs: daughter above E_x (Fermi gas)
  if (xs <= R(0) || xs >= X) return gem_range<R>(ld, X, beta, R(0), X, lref);      // one branch on all of [0, X] (R-G7: E_x <= 0)
  return gem_range<R>(ld, X, beta, R(0), xs, lref) + gem_range<R>(ld, X, beta, xs, X, lref);
}

enum EvapMode : int { kEvapKernel = 0, kEvapHelper = 1, kEvapDrainOnly = 2 };

// The persistent-lane evaporation loop as an object, so that two hosts can run it: the evaporation kernel (one pass after
// the other until the completion list is exhausted) and the idle warps of the cascade kernel (a pass whenever they have
// nothing else to do: DESIGN.md section 6).  State = one nucleus per lane + the warp's pool of completion-list entries.
// ln J0(X), ln J1(X) of a daughter nucleus (R-G5; ModelDev::gtab): elementary below E_x (constant temperature), cubic
// Hermite interpolation of the tables built at inc_init above.  Returns false if X lies beyond the table (the caller then
// integrates directly).  The interpolation error (~1e-8 in the logarithm at a 0.25 MeV step) only enters the channel
// choice; emission energies come from the sampler, which uses ln rho itself.
template <typename R>
__device__ __forceinline__ bool gem_lnJ(const ModelDev<R> &md, const LdDev<R> &ld, int row, R X, R &l0, R &l1) {
  const R Xs = ld.Ex > R(0) ? ld.Ex : R(0);
  if (X <= Xs) {
    const R z = M<R>::div_(X, ld.T);
    const R em = M<R>::expm1_(z);                      // e^z - 1
    R em2 = em - z;                                    // e^z - 1 - z (series where the difference cancels)
    if (z < R(0.5)) em2 = R(0.5) * z * z * (R(1) + z * R(1.0 / 3.0) * (R(1) + z * R(0.25) * (R(1) + z * R(0.2) * (R(1) + z * R(1.0 / 6.0) *
                          (R(1) + z * R(1.0 / 7.0) * (R(1) + z * R(0.125) * (R(1) + z * R(1.0 / 9.0) * (R(1) + z * R(0.1)))))))));
    const R base = -M<R>::div_(ld.E0, ld.T);
    l0 = base + M<R>::log_(em);
    l1 = base + ld.lnT + M<R>::log_(em2);
    return true;
  }
  if (row < 0) return false;
  const R t = (X - Xs) * R(1.0 / INC_GEM_STEP);
  const int k = (int)t;
  if (k >= kGemPoints - 1) return false;
  // R-G7: a table of a nucleus with E_x <= 0 starts at X = 0, where J0 = J1 = 0 have no logarithm: its first interval is
  // integrated directly
  if (k == 0 && !(ld.Ex > R(0))) return false;
  const R f = t - R(k);
  const GemNode<R> n0 = md.gtab[(size_t)row * kGemPoints + k], n1 = md.gtab[(size_t)row * kGemPoints + k + 1];
  const R f2 = f * f, f3 = f2 * f;
  const R h00 = R(2) * f3 - R(3) * f2 + R(1), h10 = (f3 - R(2) * f2 + f) * R(INC_GEM_STEP);
  const R h01 = R(3) * f2 - R(2) * f3, h11 = (f3 - f2) * R(INC_GEM_STEP);
  l0 = h00 * n0.l0 + h10 * n0.d0 + h01 * n1.l0 + h11 * n1.d0;
  l1 = h00 * n0.l1 + h10 * n0.d1 + h01 * n1.l1 + h11 * n1.d1;
  return true;
}

template <typename R, bool STATS, bool GEM>
struct EvapLanes {
  static constexpr int kTrialsPerPass = 2;
  int lane;
  bool cascade_only, same_stream;
  int ev;
  unsigned long long pbase;      // the warp's pool of completion-list entries: [pbase + ph, pbase + pn) not handed out yet
  int pn, ph;
  uint32_t pent;
  int A, Z, count, n_casc;     // n_casc: cascade secondaries of the event (passed on to the compaction kernel)
  R Es, Px, Py, Pz;
  uint32_t status, attempt, kblk;
  RngKey g;
  bool exhausted;
  unsigned long long n_steps, n_trials, n_emit;
  // state of an emission step whose rejection sampling is not finished yet: at most kTrialsPerPass trials run per
  // pass, a lane that has not accepted by then keeps its step (channel, X, ...) and goes on in the next pass
  // without computing the widths again -- the loop's trip count is the maximum over the warp's lanes (4.7 for a
  // mean of 1.6 trials), and it was 37 % of the kernel's instructions at 6 lanes
  bool sampling;
  int jsel, ntrial;
  R Bpar, X, a, beta, V, BdBj, s, T, areaA, areaB;
  R u1, u2;
  LdDev<R> ldsel;           // GEM mode: level density of the chosen channel's daughter

  __device__ __forceinline__ void init(const EvapParams<R> &P) {
    lane = threadIdx.x & 31;
    cascade_only = (P.flags & INC_F_CASCADE_ONLY) != 0;
    same_stream = (P.flags & INC_F_SAME_STREAM) != 0;
    ev = -1; pbase = 0; pn = 0; ph = 0; pent = kNotDone;
    A = 0; Z = 0; count = 0; n_casc = 0; Es = 0; Px = 0; Py = 0; Pz = 0;
    status = 0; attempt = 0; kblk = 0;
    g.k0 = P.seed_lo; g.k1 = P.seed_hi; g.e0 = 0; g.e1 = 0;
    exhausted = false;
    n_steps = 0; n_trials = 0; n_emit = 0;
    sampling = false; jsel = -1; ntrial = 0;
    Bpar = R(0); X = R(0); a = R(1); beta = R(0); V = R(0); BdBj = R(0); s = R(0); T = R(1); areaA = R(0); areaB = R(0);
    u1 = R(0); u2 = R(0);
    ldsel.a = ldsel.delta = ldsel.Ux = ldsel.Ex = ldsel.T = ldsel.E0 = ldsel.lnT = ldsel.lna4 = R(0);
  }
  __device__ __forceinline__ bool busy() const { return __ballot_sync(kFull, ev >= 0) != 0u; }

  // One pass: refill, one emission step (or up to kTrialsPerPass sampler trials of a pending one) per lane.  Returns
  // false when there is nothing (more) to do: kernel mode -- the list is exhausted; helper modes -- no lane has an event.
  __device__ __forceinline__ bool pass(const EvapParams<R> &P, const int mode) {
    __syncwarp();
    // ---- refill idle lanes from the warp's pool of consecutive entries of the cascade kernel's completion list
    // (lane i holds entry pbase + i).  Kernel mode: a pool is 32 tickets taken blindly (one global atomic and one
    // coalesced load per 32 events), entries not published yet are polled.  Helper mode (idle warps of the cascade
    // kernel): only entries that are published already are taken (compare-and-swap on the ticket counter), so that a
    // helper never holds a ticket it would have to wait for. ----
    const bool want = ev < 0;
    const unsigned need = __ballot_sync(kFull, want);
    if (need && mode != kEvapDrainOnly) {
      if (ph == pn && !exhausted) {
        if (mode == kEvapKernel) {
          unsigned long long base = 0;
          if (lane == 0) base = atomicAdd(&P.ctr->next_event_evap, 32ull);
          base = __shfl_sync(kFull, base, 0);
          if (base >= (unsigned long long)P.n_chunk) exhausted = true;
          else {
            pbase = base; ph = 0; pent = kNotDone;
            const unsigned long long left = (unsigned long long)P.n_chunk - base;
            pn = left < 32ull ? (int)left : 32;
          }
        } else {
          unsigned long long cur = 0;
          if (lane == 0) cur = *(volatile unsigned long long *)&P.ctr->next_event_evap;
          cur = __shfl_sync(kFull, cur, 0);
          if (cur >= (unsigned long long)P.n_chunk) exhausted = true;
          else {
            const bool in = cur + (unsigned long long)lane < (unsigned long long)P.n_chunk;
            const uint32_t v = in ? ld_acquire_u32(P.ws.done_list + cur + lane) : kNotDone;
            const unsigned gap0 = ~__ballot_sync(kFull, v != kNotDone);
            const int k = gap0 ? __ffs(gap0) - 1 : 32;
            int ok = 0;
            if (k > 0 && lane == 0) ok = atomicCAS(&P.ctr->next_event_evap, cur, cur + (unsigned long long)k) == cur;
            ok = __shfl_sync(kFull, ok, 0);
            if (ok) { pbase = cur; pn = k; ph = 0; pent = v; }
          }
        }
      }
      if (ph < pn) {
        // (the cascade kernel may still be running: poll the entries not seen yet; acquire = their events' records)
        const bool mine = lane >= ph && lane < pn;
        if (mine && pent == kNotDone) pent = ld_acquire_u32(P.ws.done_list + pbase + lane);
        const unsigned rdy = __ballot_sync(kFull, mine && pent != kNotDone);
        const unsigned gap = ~rdy & (kFull << ph);                    // first entry from ph on that is not there yet
        const int nready = (gap ? __ffs(gap) - 1 : 32) - ph;
        const int r = __popc(need & ((1u << lane) - 1u));
        int give = __popc(need);
        give = give < nready ? give : nready;
        const uint32_t d = __shfl_sync(kFull, pent, (ph + r) & 31);
        if (want && r < give) {
          ev = (int)d;
          const NucRec<R> rec = P.ws.crec[ev];
          A = rec.A; Z = rec.Z; Es = rec.E; Px = rec.Px; Py = rec.Py; Pz = rec.Pz;
          const uint32_t meta = rec.meta;
          count = (int)(meta & 0xFFu); attempt = (meta >> 8) & 0xFFu;
          status = rec.status;
          kblk = 0;
          const unsigned long long ge = same_stream ? 0ull : (unsigned long long)(P.e_base + ev);
          g.e0 = (uint32_t)ge; g.e1 = (uint32_t)(ge >> 32);
          if ((meta >> 16) & 1u) count = 0;   // FAILED or rejected input
          n_casc = count;
        }
        ph += give;
      }
    }
    if (__ballot_sync(kFull, ev >= 0) == 0) {
      if (mode != kEvapKernel) return false;             // nothing to do right now
      if (exhausted && ph == pn) return false;
      // every lane waits for the cascade kernel -- unless that has given up (queue overflow, watchdog, failed index
      // check): its unfinished events never reach the list, and the call fails or is run again anyway
      unsigned int err = 0;
      if (lane == 0) err = *(volatile unsigned int *)&P.ctr->error_word;
      if (__shfl_sync(kFull, err, 0) & (4u | 16u | 32u)) return false;
      __nanosleep(200);
      return true;
    }
    // The step is written as stages that every lane of the warp walks through, each under its own predicate, with
    // the rejection loop ended by a vote: the warp is converged again before the two-body kinematics.  (With the
    // loop left by `break`, the compiler ran everything behind it once per group of lanes that left the loop
    // together: 2.9 executions per pass at 6 lanes instead of one at 20.)
    const bool have = ev >= 0;
    const bool carry = sampling;      // a step from the previous pass is still being sampled
    bool finish = have && !carry && (cascade_only || !(Es > R(0)) || (status & INC_ST_FAILED));
    if (have && !finish && !carry) {
      jsel = -1;
      // ---------- E1/E2: channel widths ----------
      // one 128-byte row per PARENT nucleus: the six channels' constants and the parent's binding energy (a step then
      // touches one cache line instead of seven scattered ones; the loads were 10 % of the kernel's stall samples)
      const EvChan<R> *prow = P.model.evp + ((size_t)(A * kZmax + Z) << 3);
      Bpar = prow[6].V;
      R Xj[6], sj[6], aj[6];
      EvChan<R> ch[6];
      R s_ref = R(0);
      bool any = false;
      bool direct = false;          // GEM mode: some channel's X lies beyond its table
#pragma unroll
      for (int j = 0; j < 6; ++j) {
        const int Ad = A - c_evA[j], Zd = Z - c_evZ[j];
        Xj[j] = R(-1); sj[j] = R(0); aj[j] = R(1);
        ch[j].pref = R(0); ch[j].V = R(0); ch[j].beta = R(0); ch[j].BdBj = R(0);
        if (Ad >= 1 && Zd >= 0 && Zd <= Ad) {
          const EvChan<R> c = prow[j];
          if (c.pref > R(0)) {
            const R Xc = Es - Bpar + c.BdBj - c.V;
            if (GEM) {
              // (GEM mode: sj = ln rho(X) of the daughter, the largest value of the integrand's density; s_ref, their
              // maximum, scales the f32 integrals like e^{-s_max} does in the Weisskopf-Ewing mode)
              if (Xc > R(0)) {
                const LdDev<R> ld = P.model.ld[Ad * kZmax + Zd];
                if (ld.a > R(0)) {
                  ch[j] = c;
                  Xj[j] = Xc;
                  // sj, aj = ln J0, ln J1 from the tables; a channel beyond its table makes the step integrate directly
                  R l0, l1;
                  if (!gem_lnJ<R>(P.model, ld, P.model.ldrow[Ad * kZmax + Zd], Xc, l0, l1)) { direct = true; l0 = l1 = R(0); }
                  sj[j] = l0; aj[j] = l1;
                  const R lm = l0 > l1 ? l0 : l1;
                  s_ref = (!any || lm > s_ref) ? lm : s_ref;
                  any = true;
                }
              }
            } else if (Xc > R(0)) {
              ch[j] = c;
              Xj[j] = Xc;
              aj[j] = M<R>::div_(R(Ad), P.model.a_div);
              sj[j] = R(2) * M<R>::sqrt_(aj[j] * Xc);
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
        R dref = R(0);              // direct GEM quadrature in f32: common scale = the largest ln rho_j(X_j)
        if (GEM && direct && sizeof(R) == 4) {
          bool first = true;
#pragma unroll
          for (int j = 0; j < 6; ++j) {
            if (Xj[j] > R(0)) {
              const R l = gem_lnrho<R>(P.model.ld[((A - c_evA[j]) * kZmax + (Z - c_evZ[j]))], Xj[j]);
              dref = (first || l > dref) ? l : dref;
              first = false;
            }
          }
        }
#pragma unroll
        for (int j = 0; j < 6; ++j) {
          W[j] = R(0);
          if (GEM) {
            if (Xj[j] > R(0)) {
              // R-G5: W_j = g_j M_j A_d^(2/3) alpha_j int_0^X (x + beta) rho(X - x) dx = ... (J1 + beta J0), from the
              // tables (scaled by the largest ln J of the step); by direct quadrature if a channel is beyond its table
              R w;
              if (direct) {
                const LdDev<R> ld = P.model.ld[((A - c_evA[j]) * kZmax + (Z - c_evZ[j]))];
                w = ch[j].pref * gem_integral<R>(ld, Xj[j], ch[j].beta, sizeof(R) == 4 ? gem_lnrho<R>(ld, Xj[j]) : R(0));
                if (sizeof(R) == 4) w *= M<R>::exp_(gem_lnrho<R>(ld, Xj[j]) - dref);
              } else {
                w = ch[j].pref * (M<R>::exp_(aj[j] - s_ref) + ch[j].beta * M<R>::exp_(sj[j] - s_ref));
              }
              W[j] = w > R(0) ? w : R(0);
              Wsum += W[j];
            }
          } else if (Xj[j] > R(0)) {
            R g1, g3;
            G13_scaled<R>(sj[j], s_ref, g1, g3);
            const R I0 = M<R>::div_(g1, R(2) * aj[j]);
            const R I1 = Xj[j] * I0 - M<R>::div_(g3, R(8) * aj[j] * aj[j]);
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
          u1 = u[1]; u2 = u[2];
          R cum = R(0);
          const R thr = u[0] * Wsum;
          bool done = false;
#pragma unroll
          for (int j = 0; j < 6; ++j) {
            if (!done && W[j] > R(0)) { cum += W[j]; jsel = j; if (thr < cum) done = true; }
          }
#pragma unroll
          for (int j = 0; j < 6; ++j) if (j == jsel) { X = Xj[j]; a = aj[j]; beta = ch[j].beta; V = ch[j].V; BdBj = ch[j].BdBj; }
          if (GEM) {
            // R-G6: envelope slope = the smallest slope of ln rho on [0, X]: 1/T of the constant-temperature branch,
            // or the Fermi-gas slope at X if that is smaller; s holds ln rho(X)
            ldsel = P.model.ld[((A - c_evA[jsel]) * kZmax + (Z - c_evZ[jsel]))];
            R mm = M<R>::div_(R(1), ldsel.T);
            if (X > ldsel.Ex) {
              const R uu = X - ldsel.delta;
              const R sfg = M<R>::sqrt_(M<R>::div_(ldsel.a, uu)) - M<R>::div_(R(1.25), uu);
              mm = sfg < mm ? sfg : mm;
            }
            T = M<R>::div_(R(1), mm);
            s = gem_lnrho<R>(ldsel, X);
          } else {
            s = R(2) * M<R>::sqrt_(a * X);
            T = M<R>::sqrt_(M<R>::div_(X, a));
          }
          areaA = T * (T + beta); areaB = R(0.5) * X * X + beta * X;
          sampling = true; ntrial = 0;
        }
      }
    }
    // ---------- E4: rejection sampling of x (two envelopes, R-E4); warp-uniform loop ----------
    R xs = R(-1);
    bool pending = sampling;
#pragma unroll 1
    for (int n = 0; n < kTrialsPerPass; ++n) {
      if (__ballot_sync(kFull, pending) == 0u) break;
      if (pending && ntrial >= kMaxTrial) pending = false;      // trial cap (R-E4): xs stays < 0
      if (pending) {
        R v[4];
        draw4<R>(g, attempt, 0u, kblk++, v);
        ntrial++;
        if (STATS) n_trials++;
        R xx;
        if (areaB < areaA) {
          xx = -beta + M<R>::sqrt_(beta * beta + v[1] * (X * X + R(2) * beta * X));
          R rem = X - xx;
          rem = rem > R(0) ? rem : R(0);
          const R lr = GEM ? gem_lnrho<R>(ldsel, rem) : R(2) * M<R>::sqrt_(a * rem);
          if (M<R>::log_(v[3]) < lr - s) { xs = xx < X ? xx : X; pending = false; }
        } else {
          if (v[0] * (T + beta) < T) xx = -T * M<R>::log_(v[1] * v[2]);
          else xx = -T * M<R>::log_(v[1]);
          if (xx < X) {
            const R lr = GEM ? gem_lnrho<R>(ldsel, X - xx) : R(2) * M<R>::sqrt_(a * (X - xx));
            if (M<R>::log_(v[3]) < lr - s + M<R>::div_(xx, T)) { xs = xx; pending = false; }
          }
        }
      }
    }
    __syncwarp();
    if (sampling && !(pending && ntrial < kMaxTrial)) {      // accepted, or the cap was reached
      sampling = false;
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
        const R p2 = M<R>::div_(eps * (R(2) * Mpar - eps) * (R(2) * Mds + eps) * (R(2) * Mj + eps), R(4) * Mpar * Mpar);
        const R pm = M<R>::sqrt_(p2 > R(0) ? p2 : R(0));
        const R Ej = M<R>::sqrt_(p2 + Mj * Mj);
        const R cth = R(2) * u1 - R(1);
        R s2 = R(1) - cth * cth;
        const R sth = M<R>::sqrt_(s2 > R(0) ? s2 : R(0));
        R sph, cph;
        M<R>::sincos2pi(u2, &sph, &cph);
        const R qx = pm * sth * cph, qy = pm * sth * sph, qz = pm * cth;
        const R Epar = M<R>::sqrt_(Mpar * Mpar + Px * Px + Py * Py + Pz * Pz);
        const R iEp = M<R>::rcp_(Epar);
        const R bx = Px * iEp, by = Py * iEp, bz = Pz * iEp;
        const R gam = M<R>::div_(Epar, Mpar);
        const R gfac = M<R>::div_(gam * gam, gam + R(1));
        const R fo = gfac * (qx * bx + qy * by + qz * bz) + gam * Ej;
        const R lx = qx + fo * bx, ly = qy + fo * by, lz = qz + fo * bz;
        const R l2 = lx * lx + ly * ly + lz * lz;
        const R El = M<R>::sqrt_(l2 + Mj * Mj);
        const R Tl = M<R>::div_(l2, El + Mj);
        const R il = M<R>::rsqrt_(l2);
        StageRec<R> *dst = stage_slot<R>(P.ws, P.ctr, ev, count);
        if (dst) stage_write<R>(dst, Tl, lx * il, ly * il, lz * il, 0x80000000u | ((uint32_t)jsel << 24) | (uint32_t)count);
        count++;
        if (STATS) n_emit++;
        A = Ad; Z = Zd; Es = Esd;
        Px -= lx; Py -= ly; Pz -= lz;
      }
    }
    if (finish) {
      P.out_counts[ev] = count;
      NucRec<R> r;
      r.E = Es; r.Px = Px; r.Py = Py; r.Pz = Pz; r.A = A; r.Z = Z; r.meta = (uint32_t)count | ((uint32_t)n_casc << 8); r.status = status;
      P.ws.frec[ev] = r;
      ev = -1;
    }
    return true;
  }

  __device__ __forceinline__ void flush_stats(const EvapParams<R> &P) {
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
};

template <typename R, bool STATS, bool GEM>
__global__ void __launch_bounds__(256, sizeof(R) == 4 ? 3 : 2) evap_kernel(const EvapParams<R> P) {
  EvapLanes<R, STATS, GEM> L;
  L.init(P);
  while (L.pass(P, kEvapKernel)) { }
  L.flush_stats(P);
}

}  // namespace inc
