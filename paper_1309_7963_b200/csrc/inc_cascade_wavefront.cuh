// inc_cascade_wavefront.cuh — cascade kernel B (default): per-warp wavefront over shared-memory track queues, drain
// helpers, completion list.  Part of inc_device.cuh.
#pragma once

namespace inc {

// =================================================================================================
// Cascade kernel B (default): per-warp wavefront with shared-memory queues
// =================================================================================================

// ---- drain helpers ---------------------------------------------------------------------------------
// A track that orbits in the outer shells (nearly tangential, reflected at every surface hit, short chords,
// hardly any collision) runs up to kMaxSeg = 1024 segments, one per pass of its warp; the last such tracks of a
// launch kept single lanes busy for ~0.5 ms while the rest of the GPU idled.  Between collisions the path is
// deterministic, so a warp that has finished its own events (a "helper") takes such a track over: every lane
// walks the collision-free path (seg_geometry + seg_boundary only) and lane j keeps the state at the start of
// segment j; then the 32 lanes run seg_step on their segments in parallel.  If all 32 simply continue, the track
// has advanced 32 segments in one pass; otherwise the state at the start of the first segment that does not
// continue (collision, escape, cap) goes back to the owner, which runs that segment in the ordinary way.  The
// owner's bookkeeping is never touched by a helper.  seg_step is written in pinned arithmetic, so the helper's
// path is bit-identical to the owner's: results do not depend on whether, or when, a track was helped.
constexpr int kCtaLongQ = 32;      // hand-over queue owners -> helpers (per CTA)
constexpr int kRetQ = 8;           // returns helpers -> owner (per warp) = max tracks an owner has out at a time
constexpr int kLongSegDefault = 48;

template <typename R> struct CtaLong {
  int credits;              // free entries of q (producers reserve with atomicSub, consumers give back)
  int avail;                // published, not yet taken entries
  uint32_t tail, head;      // producer / consumer tickets
  uint32_t n_helpers;       // warps that have finished their own events
  uint32_t lock;            // consumers take entries one at a time, in ticket order: the ring frees in order, so a
                            // producer that holds a credit always finds the entry of its ticket free
  int idle;                 // helpers waiting for an entry: owners hand a track over only to a helper that is free
  uint32_t pad;
  uint32_t valid[kCtaLongQ];
  R q[7][kCtaLongQ];        // x y z px py pz T
  uint32_t qi[5][kCtaLongQ];   // pi, k | nseg << 16, meta (type | shell << 1 | slot << 8), event, attempt | tgt << 8 | owner << 16
};

template <typename R, int NS, int QS, int QC> struct WarpMem {
  // event slots (32 B each in the f32 build)
  int32_t ev[NS];
  uint32_t info[NS];        // n_esc | n_p << 8 | attempt << 16 | tgt << 24 (7 bits) | projectile type << 31
  uint32_t cnt[NS];         // pending tracks of the attempt (low 16) | real collisions (high 16)
  uint32_t status[NS];
  typename Fx<R>::T acc[4][NS];   // fixed-point E_in - sum T, p_in - sum p (x, y, z)
  // segment queue (structure of arrays: lane-consecutive addresses)
  R qx[QS], qy[QS], qz[QS], qpx[QS], qpy[QS], qpz[QS], qT[QS];
  uint32_t qpi[QS], qkn[QS], qmeta[QS];   // qkn = k | nseg << 16 ; qmeta = type | shell << 1 | slot << 8
  // collision queue
  R cx[QC], cy[QC], cz[QC], cpx[QC], cpy[QC], cpz[QC], cT[QC];
  uint32_t cpi[QC], ckn[QC], cmeta[QC];
  R cf[QC], cnx[QC], cny[QC], cnz[QC], cSp[QC], cSig[QC];
  // slot lists
  uint8_t epi_q[NS], free_q[NS];
  // finished events waiting to be published in the completion list (a batch costs one fence and one global atomic)
  uint32_t pub_q[96];
  // tracks coming back from the drain helpers
  uint32_t r_tail;
  uint32_t r_valid[kRetQ];
  R rq[7][kRetQ];
  uint32_t rqi[3][kRetQ];
};

// Defaults per build; -DINC_WNS= -DINC_WQS= -DINC_WQC= -DINC_WWARPS= (all four) override them for the build's real type:
// tuning experiments and the small-queue test build, which exercises the capacity guards.  Needs QS >= 64, QC >= 33.
#ifdef INC_WNS
static_assert(INC_WQS >= 64 && INC_WQC >= 33 && INC_WNS <= 128 && INC_WNS >= 32, "wavefront queue sizes");
template <typename R> struct WaveCfg { static constexpr int NS = INC_WNS, QS = INC_WQS, QC = INC_WQC, WARPS = INC_WWARPS; };
#else
template <typename R> struct WaveCfg;
template <> struct WaveCfg<float> { static constexpr int NS = 80, QS = 128, QC = 64, WARPS = 16; };
template <> struct WaveCfg<double> { static constexpr int NS = 64, QS = 128, QC = 64, WARPS = 8; };
#endif

template <typename R> __host__ __device__ inline size_t wave_smem_bytes(int n_xs, int n_stage, int n_shells) {
  typedef WaveCfg<R> C;
  return model_smem_bytes<R>(n_xs, n_stage, n_shells) + 32 + sizeof(CtaLong<R>) + sizeof(WarpMem<R, C::NS, C::QS, C::QC>) * C::WARPS;
}

// One warp, done with its own events, serves the CTA's hand-over queue until every warp of the CTA is done.
template <typename R, typename WM, typename TAB>
__device__ __forceinline__ void help_long_tracks(const CascadeParams<R> &P, const TAB &s_nuc, const R *s_tabS, WM *wm,
                                              CtaLong<R> &cq, int n_warps) {
  const int lane = threadIdx.x & 31;
  const bool same_stream = (P.flags & INC_F_SAME_STREAM) != 0;
  LaneStats<false> st;      // the STATS build never hands tracks over (its counters would see the speculative lanes)
  bool idle = false;
  for (;;) {
    // ---- take an entry (under the CTA's consumer lock) ----
    int h = -1;
    if (lane == 0) {
      if (atomicSub(&cq.avail, 1) > 0) {
        // (both waits are a few instructions of another warp long; the bound turns a protocol bug into error bit 16 --
        // INC_E_STATE -- instead of a hung device)
        unsigned spins = 0;
        while (atomicCAS(&cq.lock, 0u, 1u) != 0u) { if (++spins > (1u << 26)) { atomicOr(&P.ctr->error_word, 16u); break; } }
        h = (int)(*(volatile uint32_t *)&cq.head & (kCtaLongQ - 1));
        spins = 0;
        while (((volatile uint32_t *)cq.valid)[h] == 0u) {         // its producer is just publishing it
          if (++spins > (1u << 26)) { atomicOr(&P.ctr->error_word, 16u); break; }
        }
      } else {
        atomicAdd(&cq.avail, 1);
      }
    }
    h = __shfl_sync(kFull, h, 0);
    if (h < 0) {
      if (*(volatile uint32_t *)&cq.n_helpers == (uint32_t)n_warps) break;     // nobody has a track out any more
      if (!idle) { idle = true; if (lane == 0) atomicAdd(&cq.idle, 1); }
      __nanosleep(64);
      continue;
    }
    if (idle) { idle = false; if (lane == 0) atomicSub(&cq.idle, 1); }
    __threadfence_block();
    Track<R> cur;
    cur.x = cq.q[0][h]; cur.y = cq.q[1][h]; cur.z = cq.q[2][h]; cur.px = cq.q[3][h]; cur.py = cq.q[4][h]; cur.pz = cq.q[5][h];
    cur.T = cq.q[6][h]; cur.pi = cq.qi[0][h];
    const uint32_t kn = cq.qi[1][h], mt = cq.qi[2][h], ev = cq.qi[3][h], ao = cq.qi[4][h];
    cur.k = kn & 0xFFFFu; cur.nseg = (int)(kn >> 16);
    cur.type = mt & 1u; cur.shell = (int)((mt >> 1) & 0x7Fu);
    __syncwarp();
    if (lane == 0) {
      ((volatile uint32_t *)cq.valid)[h] = 0u;
      *(volatile uint32_t *)&cq.head = *(volatile uint32_t *)&cq.head + 1u;
      __threadfence_block();
      atomicAdd(&cq.credits, 1);
      atomicExch(&cq.lock, 0u);
    }
    const uint32_t attempt = ao & 0xFFu;
    const NucDev<R> &nu = s_nuc[(ao >> 8) & 0xFFu];
    RngKey g;
    const unsigned long long ge = same_stream ? 0ull : (unsigned long long)(P.e_base + (long long)ev);
    g.k0 = P.seed_lo; g.k1 = P.seed_hi; g.e0 = (uint32_t)ge; g.e1 = (uint32_t)(ge >> 32);
    // ---- advance it up to 32 segments per pass while every segment just continues (8 in the first pass: a
    // track that has only just become long often collides within a few segments) ----
    int depth = 8;
    for (;;) {
      Track<R> mine = cur;
      int n_look = depth;
#pragma unroll 1
      for (int j = 0; j < depth; ++j) {
        if (j == lane) mine = cur;
        if (cur.nseg >= kMaxSeg) { n_look = j + 1; break; }       // segment j ends at the cap
        cur.nseg++; cur.k++;
        const ShellDev<R> &sh = nu.sh[cur.shell];
        SegGeom<R> gm;
        Escape<R> e;
        seg_geometry<R>(cur, sh, gm);
        if (seg_boundary<R>(cur, nu, sh, gm, e) == SEG_ESCAPE) { n_look = j + 1; break; }   // segment j ends outside
      }
      int out = -1;
      if (lane < n_look) {
        Track<R> post = mine;
        CollCarry<R> cc;
        Escape<R> esc;
        out = seg_step<R, false>(post, nu, s_tabS, P.model.n_xs, P.model.inv_dp, g, attempt, cc, esc, st);
      }
      const unsigned ended = __ballot_sync(kFull, out > SEG_CONT);
      if (ended == 0u && n_look == depth) { depth = 32; continue; }     // cur = the state after `depth` continuing segments
      // the start of the first segment that does not continue goes back to the owner (were the walk and seg_step
      // ever to disagree about an escape or the cap, the start of the last walked segment does)
      const int f = ended ? __ffs(ended) - 1 : n_look - 1;
      if (lane == f) {
        WM &o = wm[ao >> 16];
        const int i = (int)(atomicAdd(&o.r_tail, 1u) & (kRetQ - 1));
        o.rq[0][i] = mine.x; o.rq[1][i] = mine.y; o.rq[2][i] = mine.z; o.rq[3][i] = mine.px; o.rq[4][i] = mine.py; o.rq[5][i] = mine.pz;
        o.rq[6][i] = mine.T; o.rqi[0][i] = mine.pi; o.rqi[1][i] = mine.k | ((uint32_t)mine.nseg << 16);
        o.rqi[2][i] = (uint32_t)mine.type | ((uint32_t)mine.shell << 1) | (mt & 0xFFFFFF00u);
        __threadfence_block();
        ((volatile uint32_t *)o.r_valid)[i] = 1u;
      }
      break;
    }
  }
}

// The kernel's pass lambda has three call sites (two of its steady-state instance).  Left to its heuristics the compiler
// stopped inlining that instance in the f64 build (round 2, 48e33cc..3045f81): the warp's state moved from registers to
// a 1000-byte stack frame and the fp64 parity build ran 2.4 times slower (5.1e7 instead of 1.2e8 events/s on config 2),
// so there the lambda is always_inline.  The f32 build inlines it anyway, and the attribute costs it 3 % there (another
// register allocation, 1.55 -> 1.61 ms), so it is left alone.
#ifdef INC_REAL_IS_DOUBLE
#define INC_PASS_INLINE __attribute__((always_inline))
#else
#define INC_PASS_INLINE
#endif

// NSH: shells per staged nucleus record (15: the paper's value and the default tables'; 32: any other table)
template <typename R, bool STATS, int NSH>
__global__ void __launch_bounds__(WaveCfg<R>::WARPS * 32, 1) cascade_wavefront_kernel(const CascadeParams<R> P) {
  typedef WaveCfg<R> C;
  typedef WarpMem<R, C::NS, C::QS, C::QC> WM;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  NucTab<R, NSH> s_nuc;
  s_nuc.base = smem_raw; s_nuc.stride = P.nuc_stride;
  R *s_tabS = reinterpret_cast<R *>(smem_raw + (size_t)P.nuc_stride * P.n_stage);
  const size_t off = ((size_t)P.nuc_stride * P.n_stage + sizeof(R) * 4 * (size_t)P.model.n_xs + 15) & ~(size_t)15;
  CtaLong<R> &cq = *reinterpret_cast<CtaLong<R> *>(smem_raw + off);
  WM *wm = reinterpret_cast<WM *>(smem_raw + off + ((sizeof(CtaLong<R>) + 15) & ~(size_t)15));
  WM &w = wm[threadIdx.x >> 5];
  const int lane = threadIdx.x & 31;
  if (lane < kRetQ) w.r_valid[lane] = 0u;
  if (lane == 0) w.r_tail = 0u;
  if (threadIdx.x < kCtaLongQ) cq.valid[threadIdx.x] = 0u;
  if (threadIdx.x == 0) { cq.credits = kCtaLongQ; cq.avail = 0; cq.tail = 0u; cq.head = 0u; cq.n_helpers = 0u; cq.lock = 0u; cq.idle = 0; }
  stage_model<R>(P.model, P.n_stage, P.nuc_stride, smem_raw, s_tabS);      // ends with __syncthreads()
  // programmatic dependent launch: the evaporation kernel may be scheduled as soon as every CTA of this grid is
  // resident (it then fills the SMs whose CTA has finished); it takes its events from the completion list
  asm volatile("griddepcontrol.launch_dependents;");

  const unsigned lt = (1u << lane) - 1u;
  const int n_xs = P.model.n_xs;
  const R inv_dp = P.model.inv_dp;
  const bool keep_transparent = (P.flags & INC_F_KEEP_TRANSPARENT) != 0;
  const bool same_stream = (P.flags & INC_F_SAME_STREAM) != 0;
  const int spp = P.seg_per_pass;
  LaneStats<STATS> st;
  st.clear();

  // warp-uniform queue sizes (every queue operation is warp-collective, so all lanes agree)
  int nSeg = 0, nColl = 0, nEpi = 0, nFree = C::NS;
  // Taper (P.taper_min > 0): a warp holds at most `quota` events, its share of the events not handed out yet (never
  // fewer than taper_min).  While the chunk has more than NS events per warp left that is NS and changes nothing; then
  // the last events are spread over all warps instead of sitting 80 deep in the warps that asked first, and a small
  // batch is spread over the whole grid from the start.  Scheduling only: results never depend on it (R-R4).
  const float inv_warps = 1.0f / (float)(gridDim.x * C::WARPS);
  int quota = C::NS;
  if (P.taper_min > 0) {
    const int q = __float2int_ru((float)P.n_chunk * inv_warps);
    quota = q < P.taper_min ? P.taper_min : (q > C::NS ? C::NS : q);
  }
  bool exhausted = false;
  // drain helpers: a track with long_seg segments behind it is handed to a warp that has finished its own events
  // (if there is one).  The STATS build keeps every track (a helper's speculative lanes would be counted).
  const bool helpers_on = !STATS && (P.flags & INC_F_NO_DRAIN_HELPERS) == 0;
  const int long_seg = helpers_on ? P.long_seg : (1 << 30);
  int n_out = 0;              // tracks of ours that are with helpers
  uint32_t r_head = 0u;       // returns consumed
  for (int i = lane; i < C::NS; i += 32) { w.free_q[i] = (uint8_t)i; w.ev[i] = -1; }
  __syncwarp();
  const bool timeline = (P.flags & INC_F_TIMING) != 0;
  if (timeline && lane == 0) { atomicMax(&P.ctr->tl[0], ~global_ns()); atomicAdd(&P.ctr->tl[4], 1ull); }
  // per-warp drain trace (diagnostic, INC_F_TIMING only)
  uint32_t *wt = (timeline && P.wtrace) ? P.wtrace + (size_t)kWTrace * (blockIdx.x * C::WARPS + (threadIdx.x >> 5)) : nullptr;
  uint32_t tr_pass = 0, tr_seg = 0, tr_lanes = 0, tr_att = 0, tr_out = 0, tr_wait = 0;
  if (wt && lane == 0) wt[7] = (uint32_t)global_ns();

  auto load_key = [&](int slot, RngKey &g, uint32_t &attempt, int &tgt, int &ev) {
    ev = w.ev[slot];
    const uint32_t m = w.info[slot];
    attempt = (m >> 16) & 0xFFu; tgt = (int)((m >> 24) & 0x7Fu);
    const unsigned long long ge = same_stream ? 0ull : (unsigned long long)(P.e_base + ev);
    g.k0 = P.seed_lo; g.k1 = P.seed_hi; g.e0 = (uint32_t)ge; g.e1 = (uint32_t)(ge >> 32);
  };
  auto push_seg = [&](bool pred, const Track<R> &t, int slot) {
    const unsigned m = __ballot_sync(kFull, pred);
    if (pred) {
      const int i = nSeg + __popc(m & lt);
      INC_CHECK(i >= 0 && i < C::QS && slot >= 0 && slot < C::NS);
      w.qx[i] = t.x; w.qy[i] = t.y; w.qz[i] = t.z; w.qpx[i] = t.px; w.qpy[i] = t.py; w.qpz[i] = t.pz; w.qT[i] = t.T;
      w.qpi[i] = t.pi; w.qkn[i] = t.k | ((uint32_t)t.nseg << 16);
      w.qmeta[i] = (uint32_t)t.type | ((uint32_t)t.shell << 1) | ((uint32_t)slot << 8);
    }
    nSeg += __popc(m);
  };
  // Completion list: finished events are collected per warp and published in batches.
  int nPub = 0;
  auto push_pub = [&](bool pred, int ev) {
    const unsigned m = __ballot_sync(kFull, pred);
    INC_CHECK(!pred || (nPub + __popc(m & lt) < 96 && ev >= 0 && ev < P.n_chunk));
    if (pred) w.pub_q[nPub + __popc(m & lt)] = (uint32_t)ev;
    nPub += __popc(m);
  };
  auto flush_pub = [&]() {
    if (nPub == 0) return;
    unsigned long long base = 0;
    if (lane == 0) base = atomicAdd(&P.ctr->n_done, (unsigned long long)nPub);
    base = __shfl_sync(kFull, base, 0);
    __syncwarp();
    __threadfence();          // every lane: its records (and, through the __syncwarp()s since, the warp's) before the entries
    for (int i = lane; i < nPub; i += 32) *(volatile uint32_t *)(P.ws.done_list + base + i) = w.pub_q[i];
    nPub = 0;
  };
  auto push_epi = [&](bool pred, int slot) {
    const unsigned m = __ballot_sync(kFull, pred);
    INC_CHECK(!pred || (nEpi + __popc(m & lt) < C::NS && slot >= 0 && slot < C::NS));
    if (pred) w.epi_q[nEpi + __popc(m & lt)] = (uint8_t)slot;
    nEpi += __popc(m);
  };

  // lane-resident segment track: stays in registers across consecutive segment passes; only lanes whose
  // track left the segment state (collision, escape, cap) touch the queues
  Track<R> rt;
  rt.x = rt.y = rt.z = rt.px = rt.py = rt.pz = rt.T = R(0); rt.pi = 0; rt.k = 0; rt.nseg = 0; rt.type = 0; rt.shell = 0;
  int rslot = 0, rev = 0, rtgt = 0;
  uint32_t rattempt = 0, rge0 = 0, rge1 = 0;
  bool rhas = false;
  int nRes = 0;   // warp-uniform count of resident tracks

  // One pass of the warp (returns true when the warp has nothing left to do).  Two instances: the steady state,
  // and the drain phase (after the event counter has run out for this warp), which alone carries the hand-over
  // of long tracks to drain helpers -- so that code costs the steady-state loop nothing (registers, uniform
  // registers, instructions).
  auto pass = [&](auto drain_tag) INC_PASS_INLINE -> bool {
    constexpr bool DRAIN = decltype(drain_tag)::value;
    __syncwarp();
    if (DRAIN && n_out > 0) {
      // ---- a track back from a helper: it continues here, at the segment that ends its collision-free run ----
      const int i = (int)(r_head & (kRetQ - 1));
      // (votes make the loaded flags warp-uniform for the compiler as well)
      const bool back = __ballot_sync(kFull, ((volatile uint32_t *)w.r_valid)[i] != 0u) == kFull;
      if (back && nSeg + nRes < C::QS) {
        __threadfence_block();
        Track<R> t;
        t.x = w.rq[0][i]; t.y = w.rq[1][i]; t.z = w.rq[2][i]; t.px = w.rq[3][i]; t.py = w.rq[4][i]; t.pz = w.rq[5][i];
        t.T = w.rq[6][i]; t.pi = w.rqi[0][i];
        const uint32_t kn = w.rqi[1][i], mt = w.rqi[2][i];
        t.k = kn & 0xFFFFu; t.nseg = (int)(kn >> 16);
        t.type = mt & 1u; t.shell = (int)((mt >> 1) & 0x7Fu);
        __syncwarp();
        if (lane == 0) ((volatile uint32_t *)w.r_valid)[i] = 0u;
        push_seg(lane == 0, t, (int)(mt >> 8));
        r_head++; n_out--;
      }
    }
    // ---- choose the kind of step of this pass (warp-uniform) ----
    // Queue invariants: a segment pass adds at most one collision item per running lane, a collision pass at most two
    // segment tracks per item, an entry pass one per item.  kCollTrig: from this many waiting collisions on a full
    // segment pass might not fit into the collision queue, so a collision pass runs first.
    constexpr int kCollTrig = C::QC - 31 < 32 ? C::QC - 31 : 32;
    constexpr int kAdmit = (C::QS + C::QC) / 3;       // admission control: no new attempts while more tracks wait
    const int nSegT = nSeg + nRes;
    int freeU = quota - (C::NS - nFree);           // free slots the taper lets this warp fill (all of them while quota = NS)
    freeU = freeU < 0 ? 0 : freeU;
    const int availE = nEpi + (exhausted ? 0 : freeU);
    int phase = ST_SEG;
    int lim = 32;                                 // tracks the refill of a segment pass may take
    if (!(nColl < kCollTrig && nSegT >= 32)) {        // (the common case needs none of what follows)
      if (nColl >= kCollTrig) phase = ST_COLL;
      else if (availE >= 32) phase = ST_EPI;
      else {
        // nothing fills a whole pass: take the fullest queue (ties: entry first, it creates work)
        if (availE > 0 && availE >= nSegT && availE >= nColl) phase = ST_EPI;
        else if (nColl > 0 && nColl >= nSegT) phase = ST_COLL;
        else if (nSegT > 0) phase = ST_SEG;
        else if (DRAIN && n_out > 0) { __nanosleep(100); tr_wait++; return false; }      // our last tracks are with helpers
        else return true;
      }
      if (phase == ST_EPI && nSegT + nColl > kAdmit) phase = nSegT > 0 ? ST_SEG : ST_COLL;   // admission control
      // While a full collision pass does not fit into the segment queue, segment passes make room first (nSegT > 0
      // then, because QS >= 64); as long as the collision queue can take a full segment pass they are ordinary ones,
      // beyond that a partial collision pass runs if it can (m >= 1), else a segment pass of at most QC - nColl lanes:
      // the resident tracks go back to the queue and the refill takes no more than that.  So some pass can always run
      // unless both queues are full (error bit 4: inc_simulate reruns the call with the lane kernel).
      if (phase == ST_COLL && nSegT + 2 * (nColl < 32 ? nColl : 32) > C::QS) {
        if (nColl <= C::QC - 32) phase = ST_SEG;
        else if (C::QS - nSegT < 2 && nColl < C::QC) {
          push_seg(rhas, rt, rslot);
          rhas = false; nRes = 0;
          phase = ST_SEG; lim = C::QC - nColl;
        }
      }
    }

    if (phase == ST_SEG) {
      // refill lanes without a resident track from the top of the segment queue
      {
        const bool need = !rhas;
        const unsigned mk = __ballot_sync(kFull, need);
        int take = __popc(mk);
        take = take < nSeg ? take : nSeg;
        take = take < lim ? take : lim;
        const int r = __popc(mk & lt);
        if (need && r < take) {
          const int i = nSeg - 1 - r;
          INC_CHECK(i >= 0 && i < C::QS);
          rt.x = w.qx[i]; rt.y = w.qy[i]; rt.z = w.qz[i]; rt.px = w.qpx[i]; rt.py = w.qpy[i]; rt.pz = w.qpz[i]; rt.T = w.qT[i];
          rt.pi = w.qpi[i];
          const uint32_t kn = w.qkn[i], mt = w.qmeta[i];
          rt.k = kn & 0xFFFFu; rt.nseg = (int)(kn >> 16);
          rt.type = mt & 1u; rt.shell = (int)((mt >> 1) & 0x7Fu); rslot = (int)(mt >> 8);
          rev = w.ev[rslot];
          {
            const unsigned long long ge = same_stream ? 0ull : (unsigned long long)(P.e_base + rev);
            rge0 = (uint32_t)ge; rge1 = (uint32_t)(ge >> 32);       // counter words 2, 3 of this track's event
          }
          const uint32_t inf = w.info[rslot];
          rattempt = (inf >> 16) & 0xFFu; rtgt = (int)((inf >> 24) & 0x7Fu);
          rhas = true;
        }
        nSeg -= take; nRes += take;
      }
      if (lane == 0) { st.add(S_WI_SEG); st.add(S_LS_SEG, nRes); }
      if (DRAIN && wt) { tr_seg++; tr_lanes += (uint32_t)nRes; }
      int out = -1;
      CollCarry<R> cc;
      Escape<R> esc;
      // Several segment steps per pass (P.seg_per_pass): a track continues in ~87 % of its segments (16O; 76 % in
      // 48Ti), so a second and third step still run at most of the lanes, and the refill, the hand-over of the tracks
      // that leave and the scheduling are paid once per pass instead of once per step.  (Config 2, cascade kernel:
      // 1 step 1.78 ms, 2 steps 1.63, 3 steps 1.57; 48Ti: 1.88, 1.74, 1.77.)
      {
        RngKey g;
        g.k0 = P.seed_lo; g.k1 = P.seed_hi; g.e0 = rge0; g.e1 = rge1;
        bool act = rhas;
#pragma unroll 1
        for (int it = 0; it < spp; ++it) {
          if (STATS && it > 0) {
            const int na = __popc(__ballot_sync(kFull, act));
            if (lane == 0) { st.add(S_WI_SEG); st.add(S_LS_SEG, na); }
          }
          if (act) out = seg_step<R, STATS>(rt, s_nuc[rtgt], s_tabS, n_xs, inv_dp, g, rattempt, cc, esc, st);
          act = act && out == SEG_CONT;
        }
      }
      {
        // long tracks go to a helper, if there is one and its queue and our return queue have room
        // ... and only tracks that have hardly collided so far (k - nseg = collisions <= nseg / 16): those are the
        // orbits whose collision-free runs are long enough for a helper to pay off
        const bool wl = DRAIN && rhas && out == SEG_CONT && rt.nseg >= long_seg && ((int)rt.k - rt.nseg) * 16 <= rt.nseg;
        const unsigned ml = __ballot_sync(kFull, wl);
        if (ml) {
          bool moved = false;
          // only to helpers that are free right now: a track never waits in the queue behind another one
          const int free_helpers = *(volatile int *)&cq.idle - *(volatile int *)&cq.avail;
          const int room = free_helpers < kRetQ - n_out ? free_helpers : kRetQ - n_out;
          if (wl && __popc(ml & lt) < room) {
            if (atomicSub(&cq.credits, 1) > 0) {
              const int i = (int)(atomicAdd(&cq.tail, 1u) & (kCtaLongQ - 1));
              cq.q[0][i] = rt.x; cq.q[1][i] = rt.y; cq.q[2][i] = rt.z; cq.q[3][i] = rt.px; cq.q[4][i] = rt.py; cq.q[5][i] = rt.pz;
              cq.q[6][i] = rt.T; cq.qi[0][i] = rt.pi; cq.qi[1][i] = rt.k | ((uint32_t)rt.nseg << 16);
              cq.qi[2][i] = (uint32_t)rt.type | ((uint32_t)rt.shell << 1) | ((uint32_t)rslot << 8);
              cq.qi[3][i] = (uint32_t)rev;
              cq.qi[4][i] = rattempt | ((uint32_t)rtgt << 8) | ((uint32_t)(threadIdx.x >> 5) << 16);
              __threadfence_block();
              ((volatile uint32_t *)cq.valid)[i] = 1u;
              atomicAdd(&cq.avail, 1);
              moved = true;
            } else {
              atomicAdd(&cq.credits, 1);
            }
          }
          const unsigned mm = __ballot_sync(kFull, moved);
          if (moved) rhas = false;
          nRes -= __popc(mm); n_out += __popc(mm);
          if (wt) tr_out += (uint32_t)__popc(mm);
        }
      }
      const unsigned left = __ballot_sync(kFull, out > SEG_CONT);     // tracks that leave the segment state
      if (left) {
        {   // collisions -> collision queue
          const bool pc = out == SEG_COLLIDE;
          const unsigned mk = __ballot_sync(kFull, pc);
          if (pc) {
            const int i = nColl + __popc(mk & lt);
            INC_CHECK(i >= 0 && i < C::QC && rslot >= 0 && rslot < C::NS);
            w.cx[i] = rt.x; w.cy[i] = rt.y; w.cz[i] = rt.z; w.cpx[i] = rt.px; w.cpy[i] = rt.py; w.cpz[i] = rt.pz; w.cT[i] = rt.T;
            w.cpi[i] = rt.pi; w.ckn[i] = rt.k | ((uint32_t)rt.nseg << 16);
            w.cmeta[i] = (uint32_t)rt.type | ((uint32_t)rt.shell << 1) | ((uint32_t)rslot << 8);
            w.cf[i] = cc.f; w.cnx[i] = cc.nx; w.cny[i] = cc.ny; w.cnz[i] = cc.nz; w.cSp[i] = cc.Sp; w.cSig[i] = cc.Sig;
          }
          nColl += __popc(mk);
        }
        bool finished = false;
        if (out == SEG_ESCAPE || out == SEG_CAP) {
          if (out == SEG_ESCAPE) {
            const uint32_t old = atomicAdd(&w.info[rslot], 1u + ((uint32_t)rt.type << 8));
            const int idx = (int)(old & 0xFFu);
            typedef typename Fx<R>::U FU;
            if (idx < kStageMain) {
              INC_CHECK(rev >= 0 && rev < P.n_chunk && rslot >= 0 && rslot < C::NS && w.ev[rslot] == rev);
              const size_t o = (size_t)rev * kStageMain + idx;
              stage_write<R>(P.ws.st + o, esc.T, esc.ux, esc.uy, esc.uz, rt.pi | ((uint32_t)rt.type << 24));
              atomicAdd((FU *)&w.acc[0][rslot], (FU)(-Fx<R>::to(esc.T)));
              atomicAdd((FU *)&w.acc[1][rslot], (FU)(-Fx<R>::to(rt.px)));
              atomicAdd((FU *)&w.acc[2][rslot], (FU)(-Fx<R>::to(rt.py)));
              atomicAdd((FU *)&w.acc[3][rslot], (FU)(-Fx<R>::to(rt.pz)));
            } else if (idx < kMaxSec) {
              // (rare: the record goes to the event's overflow row; kept apart so that the common branch is the code
              // it was before there were overflow rows)
              StageRec<R> *dst = stage_slot_overflow<R>(P.ws.ovf, P.ws.ovf_id, P.ws.ovf_rows, P.ctr, rev, idx);
              if (dst) stage_write<R>(dst, esc.T, esc.ux, esc.uy, esc.uz, rt.pi | ((uint32_t)rt.type << 24));
              atomicAdd((FU *)&w.acc[0][rslot], (FU)(-Fx<R>::to(esc.T)));
              atomicAdd((FU *)&w.acc[1][rslot], (FU)(-Fx<R>::to(rt.px)));
              atomicAdd((FU *)&w.acc[2][rslot], (FU)(-Fx<R>::to(rt.py)));
              atomicAdd((FU *)&w.acc[3][rslot], (FU)(-Fx<R>::to(rt.pz)));
            } else {
              atomicSub(&w.info[rslot], 1u + ((uint32_t)rt.type << 8));
              atomicOr(&w.status[rslot], INC_ST_SEC_TRUNC);
            }
          } else {
            atomicOr(&w.status[rslot], INC_ST_SEG_CAP);
          }
          finished = (atomicSub(&w.cnt[rslot], 1u) & 0xFFFFu) == 1u;
        }
        push_epi(finished, rslot);
        if (out > SEG_CONT) rhas = false;
        nRes -= __popc(left);
      }
      return false;
    }

    // any other pass: park the resident tracks in the segment queue first
    if (nRes > 0) {
      push_seg(rhas, rt, rslot);
      rhas = false; nRes = 0;
    }

    if (phase == ST_COLL) {
      int m = nColl < 32 ? nColl : 32;
      if (2 * m > C::QS - nSeg) m = (C::QS - nSeg) / 2;
      if (m <= 0) {   // both queues full: implementation limit exceeded -> fail loudly, never hang
        if (lane == 0) atomicOr(&P.ctr->error_word, 4u);
        return true;
      }
      if (lane == 0) { st.add(S_WI_COLL); st.add(S_LS_COLL, m); }
      const bool has = lane < m;
      Track<R> t, c2;
      CollCarry<R> cc;
      int slot = 0;
      if (has) {
        const int i = nColl - 1 - lane;
        INC_CHECK(i >= 0 && i < C::QC);
        t.x = w.cx[i]; t.y = w.cy[i]; t.z = w.cz[i]; t.px = w.cpx[i]; t.py = w.cpy[i]; t.pz = w.cpz[i]; t.T = w.cT[i];
        t.pi = w.cpi[i];
        const uint32_t kn = w.ckn[i], mt = w.cmeta[i];
        t.k = kn & 0xFFFFu; t.nseg = (int)(kn >> 16);
        t.type = mt & 1u; t.shell = (int)((mt >> 1) & 0x7Fu); slot = (int)(mt >> 8);
        cc.f = w.cf[i]; cc.nx = w.cnx[i]; cc.ny = w.cny[i]; cc.nz = w.cnz[i]; cc.Sp = w.cSp[i]; cc.Sig = w.cSig[i];
      }
      nColl -= m;
      __syncwarp();
      bool keep1 = false, keep2 = false, allowed = false, finished = false;
      if (has) {
        RngKey g;
        uint32_t attempt;
        int tgt, ev;
        load_key(slot, g, attempt, tgt, ev);
        uint32_t stbits = 0;
        allowed = coll_step<R, STATS>(t, cc, s_nuc[tgt], P.model.tabC, n_xs, inv_dp, g, attempt, c2, keep1, keep2, stbits, st);
        if (stbits) atomicOr(&w.status[slot], stbits);
        if (allowed) {
          // one real collision (high half) and the change of the pending count (low half) in one atomic
          const uint32_t delta = (1u << 16) + (keep1 ? 1u : 0u) + (keep2 ? 1u : 0u) - 1u;
          finished = ((atomicAdd(&w.cnt[slot], delta) + delta) & 0xFFFFu) == 0u;
        } else {
          keep1 = true;   // blocked: the projectile continues from the collision point
        }
      }
      push_seg(has && keep1, t, slot);
      push_seg(has && allowed && keep2, c2, slot);
      push_epi(finished, slot);
      return false;
    }

    // ---------- EPI pass: epilogue of finished attempts, event fetch, entry ----------
    {
      int m = availE < 32 ? availE : 32;
      if (m > C::QS - nSeg) m = C::QS - nSeg;
      const int mE = nEpi < m ? nEpi : m;          // finished slots first, then free slots
      const int mF = m - mE;
      if (lane == 0) { st.add(S_WI_EPI); st.add(S_LS_EPI, m); }
      const bool has = lane < m;
      int slot = 0;
      INC_CHECK(!has || (lane < mE ? (nEpi - 1 - lane >= 0 && nEpi - 1 - lane < C::NS) : (nFree - 1 - (lane - mE) >= 0 && nFree - 1 - (lane - mE) < C::NS)));
      if (has) slot = lane < mE ? w.epi_q[nEpi - 1 - lane] : w.free_q[nFree - 1 - (lane - mE)];
      INC_CHECK(slot >= 0 && slot < C::NS);
      nEpi -= mE; nFree -= mF;
      __syncwarp();
      bool want_event = has && lane >= mE;
      bool do_entry = false;
      bool done_now = false;
      int ev_done = 0;
      int ev = -1, tgt = 0, ptype = 1;
      uint32_t attempt = 0;
      R E_in = R(0);
      if (has && lane < mE) {
        ev = w.ev[slot];
        const uint32_t ne = w.info[slot];
        attempt = (ne >> 16) & 0xFFu; tgt = (int)((ne >> 24) & 0x7Fu); ptype = (int)(ne >> 31);
        E_in = P.E_in[ev];
        const NucDev<R> &nu = s_nuc[tgt];
        const int n_esc = (int)(ne & 0xFFu), n_p = (int)((ne >> 8) & 0xFFu);
        const R Eavail = Fx<R>::from(w.acc[0][slot]);
        const R Prx = Fx<R>::from(w.acc[1][slot]), Pry = Fx<R>::from(w.acc[2][slot]), Prz = Fx<R>::from(w.acc[3][slot]);
        int A_res, Z_res;
        R Estar;
        const bool ok = epilogue_eval<R>(nu, P.model.bind, ptype, n_esc, n_p, (int)(w.cnt[slot] >> 16), Eavail, Prx, Pry, Prz, keep_transparent, A_res, Z_res, Estar);
        if (ok) {
          const uint32_t used = attempt + 1u > 255u ? 255u : attempt + 1u;
          write_cascade_result<R>(P.ws, ev, A_res, Z_res, Estar, Prx, Pry, Prz, (uint32_t)n_esc | (attempt << 8), w.status[slot] | used);
          want_event = true; done_now = true; ev_done = ev;
        } else if (attempt + 1u >= (uint32_t)kMaxAttempt) {    // FAILED: count 0, target at rest
          write_cascade_result<R>(P.ws, ev, nu.A, nu.Z, R(0), R(0), R(0), R(0), (1u << 16), INC_ST_FAILED | 0xFFu);
          st.add(S_FAILED);
          want_event = true; done_now = true; ev_done = ev;
        } else {
          attempt++;
          do_entry = true;
        }
      }
      push_pub(done_now, ev_done);                 // finished events -> evaporation kernel
      // ---- warp-aggregated event fetch ----
      const unsigned need = __ballot_sync(kFull, want_event && !exhausted);
      bool got_none = false;
      if (need) {
        bool rejected = false;
        int ev_rej = 0;
        const int leader = __ffs(need) - 1;
        unsigned long long base = 0;
        if (lane == leader) base = atomicAdd(&P.ctr->next_event_casc, (unsigned long long)__popc(need));
        base = __shfl_sync(kFull, base, leader);
        if (P.taper_min > 0) {
          const int left = P.n_chunk - (int)(base < (unsigned long long)P.n_chunk ? base : (unsigned long long)P.n_chunk);
          const int q = __float2int_ru((float)left * inv_warps);
          quota = q < P.taper_min ? P.taper_min : (q > C::NS ? C::NS : q);
        }
        if (want_event) {
          const unsigned long long mine = base + (unsigned long long)__popc(need & lt);
          if (mine < (unsigned long long)P.n_chunk) {
            ev = (int)mine;
            attempt = 0;
            E_in = P.E_in[ev];
            tgt = P.target_id[ev];
            ptype = P.projectile ? (int)P.projectile[ev] : 1;
            if (check_inputs<R, NucTab<R, NSH>>(P, s_nuc, ev, E_in, tgt, ptype)) { do_entry = true; st.add(S_EVENTS); }
            else { rejected = true; ev_rej = ev; }
          } else {
            got_none = true;
          }
        }
        push_pub(rejected, ev_rej);               // (neutral outputs are complete results too)
      }
      // a batch is more than a pass's worth (one fence + one global atomic round trip each); the rest goes out when
      // the warp has finished its own events
      if (nPub > 32) flush_pub();
      const bool ran_out = __ballot_sync(kFull, got_none) != 0u;
      if (timeline && ran_out && !exhausted && lane == 0) { atomicAdd(&P.ctr->tl[1], global_ns()); if (wt) wt[0] = (uint32_t)global_ns(); }
      if (DRAIN && wt) { const uint32_t am = __reduce_max_sync(kFull, do_entry ? attempt : 0u); tr_att = am > tr_att ? am : tr_att; }
      if (ran_out) exhausted = true;
      // slots that did not get work go back to the free list
      {
        const bool fr = has && !do_entry;
        const unsigned mk = __ballot_sync(kFull, fr);
        INC_CHECK(!fr || nFree + __popc(mk & lt) < C::NS);
        if (fr) { w.free_q[nFree + __popc(mk & lt)] = (uint8_t)slot; w.ev[slot] = -1; }
        nFree += __popc(mk);
      }
      Track<R> t;
      if (do_entry) {
        st.add(S_ATTEMPTS);
        RngKey g;
        const unsigned long long ge = same_stream ? 0ull : (unsigned long long)(P.e_base + ev);
        g.k0 = P.seed_lo; g.k1 = P.seed_hi; g.e0 = (uint32_t)ge; g.e1 = (uint32_t)(ge >> 32);
        R p_in;
        entry_step<R>(t, s_nuc[tgt], E_in, ptype, g, attempt, p_in);
        w.ev[slot] = ev; w.info[slot] = (attempt << 16) | ((uint32_t)tgt << 24) | ((uint32_t)ptype << 31);
        w.cnt[slot] = 1u; w.status[slot] = 0;
        w.acc[0][slot] = Fx<R>::to(E_in); w.acc[1][slot] = 0; w.acc[2][slot] = 0; w.acc[3][slot] = Fx<R>::to(p_in);
      }
      push_seg(do_entry, t, slot);
    }
    return false;
  };
  bool done = false;
  // test hook: one warp fetches its first events, reports a queue overflow and abandons them, as a real overflow
  // would: the evaporation kernel must not wait for them, and inc_simulate must run the call again.  (The hook makes a
  // second call site of the steady-state instance of `pass`: see INC_PASS_INLINE.)
  if ((P.flags & INC_F_TEST_QUEUE_OVF) && blockIdx.x == 0 && (threadIdx.x >> 5) == 0) {
    pass(std::false_type());
    if (lane == 0) atomicOr(&P.ctr->error_word, 4u);
    done = true; exhausted = true;
  }
  while (!exhausted && !done) done = pass(std::false_type());
  // watchdog: a drain phase is a few hundred passes (thousands with waits for helpers); 2^24 means a scheduling bug:
  // fail loudly (error bit 16 -> INC_E_STATE) instead of hanging the device
  while (!done) {
    done = pass(std::true_type());
    if (++tr_pass > (1u << 24)) {
      if (wt) {   // (debug dump of the stuck state)
        const unsigned mh = __ballot_sync(kFull, rhas);
        const int fl = mh ? __ffs(mh) - 1 : 0;
        const uint32_t ns = (uint32_t)__shfl_sync(kFull, rt.nseg, fl), sl = (uint32_t)__shfl_sync(kFull, rslot, fl), kk = __shfl_sync(kFull, rt.k, fl), pp = __shfl_sync(kFull, rt.pi, fl);
        if (lane == 0) { wt[0] = mh; wt[1] = ns | (kk << 16); wt[6] = w.status[sl]; wt[7] = tr_seg; wt[3] = (uint32_t)nSeg | ((uint32_t)nRes << 16); }
      }
      if (lane == 0) {
        atomicOr(&P.ctr->error_word, 16u);
        if (wt) { wt[2] = tr_pass; wt[4] = (uint32_t)nColl | ((uint32_t)nEpi << 16); wt[5] = (uint32_t)nFree | ((uint32_t)n_out << 16); }
      }
      break;
    }
  }
  if (wt && lane == 0 && tr_pass <= (1u << 24)) { wt[1] = (uint32_t)global_ns(); wt[2] = tr_pass; wt[3] = tr_seg; wt[4] = tr_lanes; wt[5] = tr_att | (tr_wait << 8); wt[6] = tr_out; }
  if (timeline && lane == 0) {
    const unsigned long long t = global_ns();
    atomicAdd(&P.ctr->tl[2], t); atomicMax(&P.ctr->tl[3], t); atomicMax(&P.ctr->tl[5], ~t);
  }
  // every slot came back -- unless the launch was given up (queue overflow, watchdog): a warp that leaves that way
  // still holds tracks, and the call is run again or fails with its own message, not with an index-check error
  INC_CHECK((nSeg == 0 && nColl == 0 && nEpi == 0 && nRes == 0 && n_out == 0 && nFree == C::NS) ||
            (*(volatile unsigned int *)&P.ctr->error_word & (4u | 16u)) != 0u);
  flush_pub();
  st.flush(P.ctr, lane);
  if (helpers_on) {
    if (lane == 0) { __threadfence_block(); atomicAdd(&cq.n_helpers, 1u); }
    help_long_tracks<R, WM, NucTab<R, NSH>>(P, s_nuc, s_tabS, wm, cq, C::WARPS);
  }
}

}  // namespace inc
