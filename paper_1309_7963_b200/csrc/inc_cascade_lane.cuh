// inc_cascade_lane.cuh — cascade kernel A: one lane owns one event (the paper's layout, and its warp-voted state
// machine variant); cross-check, and the fallback when the wavefront kernel's queues overflow.  Part of inc_device.cuh.
#pragma once

namespace inc {

// =================================================================================================
// Cascade kernel A: lane-per-event state machine with warp-voted phases
// =================================================================================================
enum LaneState : int { ST_SEG = 0, ST_COLL = 1, ST_EPI = 2, ST_DONE = 3 };

template <typename R> struct TrackRec {   // pending track (local-memory stack)
  R x, y, z, px, py, pz, T;
  uint32_t pi;
  uint32_t meta;   // type | shell << 1
};

template <typename R, bool STATS>
__global__ void __launch_bounds__(256, 2) cascade_lane_kernel(const CascadeParams<R> P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  NucTab<R, 0> s_nuc;
  s_nuc.base = smem_raw; s_nuc.stride = P.nuc_stride;
  R *s_tabS = reinterpret_cast<R *>(smem_raw + (size_t)P.nuc_stride * P.n_stage);
  stage_model<R>(P.model, P.n_stage, P.nuc_stride, smem_raw, s_tabS);
  // programmatic dependent launch: the evaporation kernel may be scheduled as soon as every CTA of this grid is
  // resident; it takes its events from the completion list, never from stream order
  asm volatile("griddepcontrol.launch_dependents;");

  const int lane = threadIdx.x & 31;
  const int n_xs = P.model.n_xs;
  const R inv_dp = P.model.inv_dp;
  const bool keep_transparent = (P.flags & INC_F_KEEP_TRANSPARENT) != 0;
  const bool same_stream = (P.flags & INC_F_SAME_STREAM) != 0;

  int state = ST_EPI;
  int ev = -1, tgt = 0, ptype = 1;
  uint32_t attempt = 0;
  R E_in = R(0);
  RngKey g;
  g.k0 = P.seed_lo; g.k1 = P.seed_hi; g.e0 = 0; g.e1 = 0;
  Track<R> t;
  t.x = t.y = t.z = t.px = t.py = t.pz = t.T = R(0); t.pi = 0; t.k = 0; t.nseg = 0; t.type = 0; t.shell = 0;
  typename Fx<R>::T fxE = 0, fxX = 0, fxY = 0, fxZ = 0;   // fixed-point E_in - sum T, p_in - sum p
  int n_esc = 0, n_p = 0, n_real = 0;
  uint32_t st_try = 0;
  TrackRec<R> stack[kStackCap];
  int sp = 0;
  CollCarry<R> cc;
  cc.f = cc.nx = cc.ny = cc.nz = cc.Sp = cc.Sig = R(0);
  LaneStats<STATS> st;
  st.clear();

  auto pop_or_finish = [&]() {
    if (sp > 0) {
      const TrackRec<R> &r = stack[--sp];
      t.x = r.x; t.y = r.y; t.z = r.z; t.px = r.px; t.py = r.py; t.pz = r.pz; t.T = r.T;
      t.pi = r.pi; t.type = r.meta & 1; t.shell = (int)(r.meta >> 1);
      t.k = 0; t.nseg = 0;
      state = ST_SEG;
    } else {
      state = ST_EPI;
    }
  };

  for (;;) {
    __syncwarp();
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
      if (lane == 0) { st.add(S_WI_SEG); st.add(S_LS_SEG, nS); }
      if (state == ST_SEG) {
        Escape<R> esc;
        const int out = seg_step<R, STATS>(t, s_nuc[tgt], s_tabS, n_xs, inv_dp, g, attempt, cc, esc, st);
        if (out == SEG_COLLIDE) state = ST_COLL;
        else if (out == SEG_ESCAPE) {
          if (n_esc < kMaxSec) {
            StageRec<R> *dst = stage_slot<R>(P.ws, P.ctr, ev, n_esc);
            if (dst) stage_write<R>(dst, esc.T, esc.ux, esc.uy, esc.uz, t.pi | ((uint32_t)t.type << 24));
            n_esc++; n_p += t.type;
            fxE -= Fx<R>::to(esc.T); fxX -= Fx<R>::to(t.px); fxY -= Fx<R>::to(t.py); fxZ -= Fx<R>::to(t.pz);
          } else {
            st_try |= INC_ST_SEC_TRUNC;
          }
          pop_or_finish();
        } else if (out == SEG_CAP) {
          st_try |= INC_ST_SEG_CAP;
          pop_or_finish();
        }
      }
    } else if (phase == ST_COLL) {
      if (lane == 0) { st.add(S_WI_COLL); st.add(S_LS_COLL, nC); }
      if (state == ST_COLL) {
        Track<R> c2;
        bool keep1 = false, keep2 = false;
        const bool allowed = coll_step<R, STATS>(t, cc, s_nuc[tgt], P.model.tabC, n_xs, inv_dp, g, attempt, c2, keep1, keep2, st_try, st);
        if (!allowed) state = ST_SEG;
        else {
          n_real++;
          if (keep1 && keep2) {
            if (sp < kStackCap) {
              TrackRec<R> &r = stack[sp++];
              r.x = c2.x; r.y = c2.y; r.z = c2.z; r.px = c2.px; r.py = c2.py; r.pz = c2.pz; r.T = c2.T;
              r.pi = c2.pi; r.meta = (uint32_t)c2.type | ((uint32_t)c2.shell << 1);
            } else {
              st_try |= INC_ST_QUEUE_OVF;
            }
            state = ST_SEG;
          } else if (keep1) state = ST_SEG;
          else if (keep2) { t = c2; state = ST_SEG; }
          else pop_or_finish();
        }
      }
    } else {  // EPI phase: epilogue of the finished attempt, then entry of the next attempt / event
      if (lane == 0) { st.add(S_WI_EPI); st.add(S_LS_EPI, nE); }
      bool want_event = false;
      bool done_now = false;
      int ev_done = ev;
      if (state == ST_EPI) {
        if (ev >= 0) {
          const NucDev<R> &nu = s_nuc[tgt];
          int A_res, Z_res;
          R Estar;
          const R Eavail = Fx<R>::from(fxE), Prx = Fx<R>::from(fxX), Pry = Fx<R>::from(fxY), Prz = Fx<R>::from(fxZ);
          const bool ok = epilogue_eval<R>(nu, P.model.bind, ptype, n_esc, n_p, n_real, Eavail, Prx, Pry, Prz, keep_transparent, A_res, Z_res, Estar);
          if (ok) {
            const uint32_t used = attempt + 1u > 255u ? 255u : attempt + 1u;
            write_cascade_result<R>(P.ws, ev, A_res, Z_res, Estar, Prx, Pry, Prz, (uint32_t)n_esc | (attempt << 8), st_try | used);
            ev = -1;
            done_now = true;
          } else {
            attempt++;
            if (attempt >= (uint32_t)kMaxAttempt) {          // FAILED: count 0, target at rest
              write_cascade_result<R>(P.ws, ev, nu.A, nu.Z, R(0), R(0), R(0), R(0), (1u << 16), INC_ST_FAILED | 0xFFu);
              st.add(S_FAILED);
              ev = -1;
              done_now = true;
            }
          }
        }
        want_event = (ev < 0);
      }
      publish_done(done_now, ev_done, &P.ctr->n_done, P.ws.done_list, lane);
      const unsigned need = __ballot_sync(kFull, want_event);
      if (need) {
        bool rejected = false;
        int ev_rej = 0;
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
            ptype = P.projectile ? (int)P.projectile[ev] : 1;
            if (!check_inputs<R, NucTab<R, 0>>(P, s_nuc, ev, E_in, tgt, ptype)) { rejected = true; ev_rej = ev; ev = -1; tgt = 0; }
            else {
              const unsigned long long ge = same_stream ? 0ull : (unsigned long long)(P.e_base + ev);
              g.e0 = (uint32_t)ge; g.e1 = (uint32_t)(ge >> 32);
              st.add(S_EVENTS);
            }
          } else {
            state = ST_DONE;
          }
        }
        publish_done(rejected, ev_rej, &P.ctr->n_done, P.ws.done_list, lane);   // (neutral outputs are complete results too)
      }
      if (state == ST_EPI && ev >= 0) {
        st.add(S_ATTEMPTS);
        R p_in;
        entry_step<R>(t, s_nuc[tgt], E_in, ptype, g, attempt, p_in);
        fxE = Fx<R>::to(E_in); fxX = 0; fxY = 0; fxZ = Fx<R>::to(p_in);
        n_esc = 0; n_p = 0; n_real = 0; st_try = 0; sp = 0;
        state = ST_SEG;
      }
    }
  }
  st.flush(P.ctr, lane);
}

}  // namespace inc
