// inc_physics.cuh — the physics steps as device functions (entry C0, segment C2 + boundary C4, collision C3, epilogue C6),
// kernel parameters, model staging, fixed-point sums.  Part of inc_device.cuh.
#pragma once

namespace inc {

// ---------- C0: entry — uniform disc, beam along +z (R-Q15), potential step into the last shell ----------
template <typename R>
__device__ __forceinline__ void entry_step(Track<R> &t, const NucDev<R> &nu, R E_in, int ptype, const RngKey &g,
                                           uint32_t attempt, R &p_in) {
  R u[4];
  draw4<R>(g, attempt, 1u, 0u, u);
  const R b = nu.Rn * M<R>::sqrt_(u[0]);
  R sb, cb;
  M<R>::sincos2pi(u[1], &sb, &cb);
  t.x = b * cb; t.y = b * sb;
  const R zz = nu.Rn * nu.Rn - b * b;
  t.z = -M<R>::sqrt_(zz > R(0) ? zz : R(0));
  // the incident nucleon: proton (ptype 1, the paper's case P:9) or neutron (NEXT-3), with its own mass and potential
  const R m0 = nucleon_mass<R>(ptype);
  p_in = M<R>::sqrt_(E_in * (E_in + R(2) * m0));
  // potential step (cannot reflect: V rises inward)
  const R ux = t.x * nu.iRn, uy = t.y * nu.iRn, uz = t.z * nu.iRn;
  const R pr = p_in * uz;
  const R dV = ptype ? nu.sh[nu.ns - 1].V_p : nu.sh[nu.ns - 1].V_n;
  const R Tj = E_in + dV;
  const R prj2 = pr * pr + dV * (E_in + Tj + R(2) * m0);
  const R prj = -M<R>::sqrt_(prj2 > R(0) ? prj2 : R(0));
  const R dp = prj - pr;
  t.px = dp * ux; t.py = dp * uy; t.pz = p_in + dp * uz;
  t.T = Tj;
  t.type = ptype; t.shell = nu.ns - 1; t.pi = 1u; t.k = 1u; t.nseg = 0;
}

// ---------- C2 + C4: one segment (R-Q8 partner first, then the path) ----------
// Written in pinned arithmetic (M<R>::fma_/mul_/add_/sub_, never re-contracted): the wavefront kernel runs a
// segment at two call sites (its own segment pass and the drain helpers' look-ahead), and both must give the
// same bits in the f32 build too.  The f64 operation order is the oracle's.
template <typename R> struct SegGeom { R dx, dy, dz, d_min; bool inward; };

// R-C2 geometry: distances to the shell spheres along the flight direction
template <typename R>
__device__ __forceinline__ void seg_geometry(const Track<R> &t, const ShellDev<R> &sh, SegGeom<R> &gm) {
  typedef M<R> m;
  const R p1sq = m::fma_(t.pz, t.pz, m::fma_(t.py, t.py, m::mul_(t.px, t.px)));
  const R ip = m::rsqrt_(p1sq);
  gm.dx = m::mul_(t.px, ip); gm.dy = m::mul_(t.py, ip); gm.dz = m::mul_(t.pz, ip);
  const R beta = m::fma_(t.z, gm.dz, m::fma_(t.y, gm.dy, m::mul_(t.x, gm.dx)));
  const R r2 = m::fma_(t.z, t.z, m::fma_(t.y, t.y, m::mul_(t.x, t.x)));
  const R bb = m::sub_(m::mul_(beta, beta), r2);
  R disc_out = m::fma_(sh.r_out, sh.r_out, bb);
  disc_out = disc_out > R(0) ? disc_out : R(0);
  const R d_out = m::sub_(m::sqrt_(disc_out), beta);
  R d_in = R(1e30);
  if (t.shell > 0 && beta < R(0)) {
    const R D = m::fma_(sh.r_in, sh.r_in, bb);
    if (D > R(0)) d_in = m::sub_(-beta, m::sqrt_(D));
  }
  gm.inward = d_in < d_out;
  gm.d_min = gm.inward ? d_in : d_out;
}

// R-C4 shell boundary, potential step (P:49 refraction / reflection).  Returns SEG_CONT (refracted into the
// next shell), SEG_REFLECT (total reflection, shell unchanged) or SEG_ESCAPE (left the nucleus; esc filled).
// Straight-line code: both outcomes are computed and selected (the lanes of a warp take both anyway), so that the
// compiler can overlap this chain, which needs no random number, with the cross-section chain of seg_step.
template <typename R>
__device__ __forceinline__ int seg_boundary(Track<R> &t, const NucDev<R> &nu, const ShellDev<R> &sh, const SegGeom<R> &gm,
                                            Escape<R> &esc) {
  typedef M<R> m;
  const int j = gm.inward ? t.shell - 1 : t.shell + 1;
  const R irb = gm.inward ? sh.ir_in : sh.ir_out;
  const R m1 = nucleon_mass<R>(t.type);
  R x = m::fma_(gm.d_min, gm.dx, t.x), y = m::fma_(gm.d_min, gm.dy, t.y), z = m::fma_(gm.d_min, gm.dz, t.z);
  // renormalise onto the sphere: one Newton step of 1/sqrt around |x|^2 = rb^2 (|x| is within rounding of rb)
  const R rr = m::fma_(z, z, m::fma_(y, y, m::mul_(x, x)));
  const R corr = m::sub_(R(1.5), m::mul_(m::mul_(m::mul_(R(0.5), rr), irb), irb));
  x = m::mul_(x, corr); y = m::mul_(y, corr); z = m::mul_(z, corr);
  t.x = x; t.y = y; t.z = z;
  const R ux = m::mul_(x, irb), uy = m::mul_(y, irb), uz = m::mul_(z, irb);              // outward normal
  const R pr = m::fma_(t.pz, uz, m::fma_(t.py, uy, m::mul_(t.px, ux)));
  const R Vi = t.type ? sh.V_p : sh.V_n;
  const R Vj = t.type ? nu.sh[j].V_p : nu.sh[j].V_n;
  const R dV = m::sub_(Vj, Vi);
  const R Tj = m::add_(t.T, dV);
  const R prj2 = m::fma_(dV, m::add_(m::add_(t.T, Tj), m::mul_(R(2), m1)), m::mul_(pr, pr));   // p_j^2 - p_t^2
  const bool refl = (Tj <= R(0) || prj2 <= R(0));
  // specular reflection: p -= 2 p_r u; refraction: p_r -> sign(p_r) sqrt(p_rj^2)  (one is selected; a reflecting
  // lane's square root is of a non-positive number and is not used)
  const R sq = m::sqrt_(prj2);
  const R dp = refl ? m::mul_(R(-2), pr) : m::sub_(pr >= R(0) ? sq : -sq, pr);
  t.px = m::fma_(dp, ux, t.px); t.py = m::fma_(dp, uy, t.py); t.pz = m::fma_(dp, uz, t.pz);
  t.T = refl ? t.T : Tj;
  t.shell = refl ? t.shell : j;
  // escape ("exiting particles"): direction of the refracted momentum
  const R ipj = m::rsqrt_(m::mul_(Tj, m::fma_(R(2), m1, Tj)));
  esc.T = Tj; esc.ux = m::mul_(t.px, ipj); esc.uy = m::mul_(t.py, ipj); esc.uz = m::mul_(t.pz, ipj);
  return refl ? SEG_REFLECT : (j == nu.ns ? SEG_ESCAPE : SEG_CONT);
}

// momentum of the track in the rest frame of a partner with momentum q n (plab_of in pinned arithmetic)
template <typename R>
__device__ __forceinline__ R plab_pinned(R m1, R E1, R pn, R q, R m2, R im2) {
  typedef M<R> m;
  const R E2 = m::sqrt_(m::fma_(q, q, m::mul_(m2, m2)));
  const R Tlab = m::fma_(m::fma_(E1, E2, -m::mul_(q, pn)), im2, -m1);
  R a = m::mul_(Tlab, m::fma_(R(2), m1, Tlab));
  a = a > R(0) ? a : R(0);
  return m::sqrt_(a);
}

template <typename R, bool STATS>
__device__ __forceinline__ int seg_step(Track<R> &t, const NucDev<R> &nu, const R *s_tabS, int n_xs, R inv_dp,
                                        const RngKey &g, uint32_t attempt, CollCarry<R> &cc, Escape<R> &esc,
                                        LaneStats<STATS> &st) {
  typedef M<R> m;
  // Straight-line code: the collision point and the boundary step are both computed and one is selected.  The
  // geometry / boundary chain depends on the track only, the cross-section chain on the random numbers, so they
  // overlap; with a branch between them the second could not start before the first had ended.
  const bool cap = t.nseg >= kMaxSeg;                                // R-C2 cap: absorbed (the track is dead then)
  t.nseg++;
  if (!cap) st.add(S_SEG);
  R u[4];
  draw4<R>(g, attempt, t.pi, t.k++, u);
  const ShellDev<R> &sh = nu.sh[t.shell];
  const R m1 = nucleon_mass<R>(t.type);
  const R E1 = m::add_(t.T, m1);
  // partner direction and magnitude fraction ("quadratic distribution")
  const R cth = m::fma_(R(2), u[1], R(-1));
  R s2 = m::fma_(-cth, cth, R(1));
  s2 = s2 > R(0) ? s2 : R(0);
  const R sth = m::sqrt_(s2);
  R sph, cph;
  m::sincos2pi(u[2], &sph, &cph);
  const R nx = m::mul_(sth, cph), ny = m::mul_(sth, sph), nz = cth;
  const R f = m::cbrt_(u[0]);
  const R pn = m::fma_(t.pz, nz, m::fma_(t.py, ny, m::mul_(t.px, nx)));
  // cross sections against a proton and a neutron partner (same n, f: R-C2)
  const R plab_p = plab_pinned<R>(m1, E1, pn, m::mul_(sh.pF_p, f), K<R>::mp, K<R>::imp);
  const R plab_n = plab_pinned<R>(m1, E1, pn, m::mul_(sh.pF_n, f), K<R>::mn, K<R>::imn);
  int kp, kn; R fp, fn;
  grid_pos<R>(plab_p, inv_dp, n_xs, kp, fp);
  grid_pos<R>(plab_n, inv_dp, n_xs, kn, fn);
  // tabS row {sig_pp, d, sig_np, d}: vs a proton pp if the track is a proton else np; vs a neutron the opposite
  const R *rp = s_tabS + 4 * kp + (t.type ? 0 : 2);
  const R *rn = s_tabS + 4 * kn + (t.type ? 2 : 0);
  const R Sp = m::mul_(sh.rho_p, m::fma_(fp, rp[1], rp[0]));
  const R Sn = m::mul_(sh.rho_n, m::fma_(fn, rn[1], rn[0]));
  const R Sig = m::add_(Sp, Sn);
  const R nlu = -m::log_(u[3]);                  // d_coll = nlu / Sig
  SegGeom<R> gm;
  seg_geometry<R>(t, sh, gm);
  // ---------- C4: shell boundary, potential step (on a copy) ----------
  Track<R> tb = t;
  const int rb = seg_boundary<R>(tb, nu, sh, gm, esc);
  // ---------- collision point reached first (d_coll < d_min)?  Then hand over to the collision step ----------
  const bool coll = nlu < m::mul_(Sig, gm.d_min);
  const R d_coll = m::div_(nlu, Sig);
  cc.f = f; cc.nx = nx; cc.ny = ny; cc.nz = nz; cc.Sp = Sp; cc.Sig = Sig;
  t.x = coll ? m::fma_(d_coll, gm.dx, t.x) : tb.x;
  t.y = coll ? m::fma_(d_coll, gm.dy, t.y) : tb.y;
  t.z = coll ? m::fma_(d_coll, gm.dz, t.z) : tb.z;
  t.px = coll ? t.px : tb.px; t.py = coll ? t.py : tb.py; t.pz = coll ? t.pz : tb.pz;
  t.T = coll ? t.T : tb.T;
  t.shell = coll ? t.shell : tb.shell;
  if (STATS) {
    if (cap) st.add(S_ABSORBED);
    else if (!coll) { st.add(S_BND); if (rb == SEG_REFLECT) st.add(S_REFL); if (rb == SEG_ESCAPE) st.add(S_ESC); }
  }
  return cap ? SEG_CAP : (coll ? SEG_COLLIDE : (rb == SEG_ESCAPE ? SEG_ESCAPE : SEG_CONT));
}

// ---------- C3: collision.  Returns false if Pauli-blocked (track t continues, k advanced) ----------
template <typename R, bool STATS>
__device__ __forceinline__ bool coll_step(Track<R> &t, const CollCarry<R> &cc, const NucDev<R> &nu, const R *tabC,
                                          int n_xs, R inv_dp, const RngKey &g, uint32_t attempt,
                                          Track<R> &c2, bool &keep1, bool &keep2, uint32_t &status, LaneStats<STATS> &st) {
  st.add(S_COLL);
  const ShellDev<R> &sh = nu.sh[t.shell];
  R u[4];
  draw4<R>(g, attempt, t.pi, t.k++, u);
  const int t2 = (u[0] * cc.Sig < cc.Sp) ? 1 : 0;
  const R m1 = nucleon_mass<R>(t.type), m2 = nucleon_mass<R>(t2);
  const R q = (t2 ? sh.pF_p : sh.pF_n) * cc.f;
  const R p2x = q * cc.nx, p2y = q * cc.ny, p2z = q * cc.nz;
  const R E1 = t.T + m1;
  const R E2 = M<R>::sqrt_(q * q + m2 * m2);
  const R pn = t.px * cc.nx + t.py * cc.ny + t.pz * cc.nz;
  const R Tlab = (E1 * E2 - q * pn) * nucleon_imass<R>(t2) - m1;
  R pl2 = Tlab * (Tlab + R(2) * m1);
  const R plab = M<R>::sqrt_(pl2 > R(0) ? pl2 : R(0));
  int kk; R ff;
  grid_pos<R>(plab, inv_dp, n_xs, kk, ff);
  const bool same = (t2 == t.type);
  const R *row = tabC + 8 * kk;
  const R B = same ? (__ldg(row + 0) + ff * __ldg(row + 1)) : (__ldg(row + 2) + ff * __ldg(row + 3));
  const R ab = same ? R(0) : (__ldg(row + 4) + ff * __ldg(row + 5));
  // boost to the CM frame
  const R Px = t.px + p2x, Py = t.py + p2y, Pz = t.pz + p2z;
  const R E = E1 + E2;
  const R s = E * E - (Px * Px + Py * Py + Pz * Pz);
  const R iE = M<R>::rcp_(E);
  const R bx = Px * iE, by = Py * iE, bz = Pz * iE;
  const R gam = E * M<R>::rsqrt_(s);
  const R gfac = M<R>::div_(gam * gam, gam + R(1));      // (gamma - 1) / beta^2
  const R pb = t.px * bx + t.py * by + t.pz * bz;
  const R fb = gfac * pb - gam * E1;
  const R qx = t.px + fb * bx, qy = t.py + fb * by, qz = t.pz + fb * bz;   // p1 in the CM frame
  const R pcm2 = qx * qx + qy * qy + qz * qz;
  const R ipcm = M<R>::rsqrt_(pcm2);
  const R pcm = pcm2 * ipcm;
  // scattering angle: dsigma/dt ~ exp(B t), t in (GeV/c)^2 (R-Q10)
  const R pg2 = pcm2 * R(1e-6);
  const R tmin = R(-4) * pg2;
  R tt;
  if (B * (-tmin) < R(1e-9)) tt = u[1] * tmin;
  else tt = M<R>::div_(M<R>::log1p_(-u[1] * (-M<R>::expm1_(B * tmin))), B);
  R ct = R(1) + M<R>::div_(tt, R(2) * pg2);
  ct = ct < R(-1) ? R(-1) : (ct > R(1) ? R(1) : ct);
  if (!same && u[2] * (R(1) + ab) < ab) ct = -ct;       // np backward term
  const R st2 = R(1) - ct * ct;
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
  const R pF2_1 = t.type ? sh.pF2_p : sh.pF2_n;
  const R pF2_2 = t2 ? sh.pF2_p : sh.pF2_n;
  if (!(o1sq > pF2_1 && o2sq > pF2_2)) {
    st.add(S_BLOCKED);
    return false;                                     // projectile continues unchanged (R-Q13)
  }
  st.add(S_ALLOWED);
  keep1 = false; keep2 = false;
  if (2u * t.pi + 1u >= (1u << 24)) {                 // depth cap (R-C3)
    status |= INC_ST_DEPTH_CAP;
    st.add(S_ABSORBED, 2);
  } else {
    // cutoff: E_F + E_B (n), E_F + E_B + E_C (p)
    keep1 = o1sq > (t.type ? sh.pc2_p : sh.pc2_n);
    keep2 = o2sq > (t2 ? sh.pc2_p : sh.pc2_n);
    st.add(S_ABSORBED, (keep1 ? 0 : 1) + (keep2 ? 0 : 1));
  }
  // children: scattered projectile keeps the lane's track slot (pi' = 2 pi), recoil is c2 (pi' = 2 pi + 1)
  c2.x = t.x; c2.y = t.y; c2.z = t.z; c2.px = o2x; c2.py = o2y; c2.pz = o2z;
  c2.T = M<R>::div_(o2sq, M<R>::sqrt_(o2sq + m2 * m2) + m2);
  c2.pi = 2u * t.pi + 1u; c2.k = 0u; c2.nseg = 0; c2.type = t2; c2.shell = t.shell;
  t.px = o1x; t.py = o1y; t.pz = o1z;
  t.T = M<R>::div_(o1sq, M<R>::sqrt_(o1sq + m1 * m1) + m1);
  t.pi = 2u * t.pi; t.k = 0u; t.nseg = 0;
  return true;
}

// ---------- C6: epilogue ("excitation energy ... through energy conservation") ----------
// Eavail = E_in - sum T_k, (Prx,Pry,Prz) = p_in - sum p_k.  Returns true if the attempt is accepted.
template <typename R>
__device__ __forceinline__ bool epilogue_eval(const NucDev<R> &nu, const R *bind, int ptype, int n_esc, int n_p, int n_real,
                                              R Eavail, R Prx, R Pry, R Prz, bool keep_transparent,
                                              int &A_res, int &Z_res, R &Estar) {
  A_res = nu.A + 1 - n_esc; Z_res = nu.Z + ptype - n_p;   // (the nucleon masses cancel for either projectile)
  Estar = R(0);
  if (!((n_real > 0) || keep_transparent)) return false;       // transparent: not a non-elastic event
  R Bres = R(-1e30);
  if (A_res >= 1 && A_res < kAmax && Z_res >= 0 && Z_res < kZmax) Bres = __ldg(bind + A_res * kZmax + Z_res);
  if (Bres < R(-1e29)) return false;                            // no such nucleus
  // E_res - M_res = X with the nucleon masses cancelled analytically; E* = M* - M_res in rationalised form
  const R X = Eavail + Bres - nu.Bt;
  const R Mres = R(Z_res) * K<R>::mp + R(A_res - Z_res) * K<R>::mn - Bres;
  const R P2 = Prx * Prx + Pry * Pry + Prz * Prz;
  const R Er = Mres + X;
  const R M2 = Er * Er - P2;
  const R Mstar = M2 > R(0) ? M<R>::sqrt_(M2) : R(0);
  Estar = (R(2) * Mres * X + X * X - P2) / (Mstar + Mres);
  if (Estar < R(0) && !(keep_transparent && n_real == 0)) return false;
  return true;
}

// ---- kernel parameters ------------------------------------------------------------------------------
template <typename R> struct CascadeParams {
  ModelDev<R> model;
  Workspace<R> ws;
  DevCounters *ctr;
  const R *E_in;            // chunk base
  const int32_t *target_id; // chunk base
  const uint8_t *projectile; // chunk base; 0 = neutron, 1 = proton; nullptr = all protons
  long long e_base;         // global index of the chunk's first event
  int n_chunk;
  uint32_t seed_lo, seed_hi;
  uint32_t flags;
  int vote_coll, vote_epi;  // lane kernel: phase-vote thresholds
  int long_seg;             // wavefront kernel: tracks with this many segments behind them may go to a drain helper
  int taper_min;            // wavefront kernel: 0 = off; else a warp holds at most max(taper_min, events left / warps) events
  int seg_per_pass;         // wavefront kernel: segment steps per segment pass (1..8)
  int n_stage;              // nuclei slots staged into shared memory (target_id must be < n_stage)
  int nuc_stride;           // bytes of one staged nucleus (nuc_stride_bytes)
  uint32_t *wtrace;         // INC_F_TIMING: kWTrace words per warp of the wavefront kernel (inc_get_warp_trace), or nullptr
};
constexpr int kWTrace = 8;  // [0] ns (low 32 bits) when the event counter ran out for the warp, [1] ns at exit of its own work,
                            // [2] passes of the drain phase, [3] segment passes among them, [4] lanes summed over those,
                            // [5] highest attempt number started in the drain, [6] tracks handed to helpers, [7] ns at kernel entry

// shared-memory staging of the model: [NucDev x n_stage] [tabS n_xs*4]   (n_stage = highest live slot + 1)
// The staged copy of a nucleus is truncated after its last shell (header + ns + 1 shells of the 33 a NucDev has room
// for): 1056 instead of 2144 bytes in the f32 build at 15 shells, so that ten live targets fit beside the queues of the
// wavefront kernel instead of five.  All targets of a library state have the same number of shells.
template <typename R> __host__ __device__ inline int nuc_stride_bytes(int n_shells) {
  return (int)(sizeof(NucDev<R>) - sizeof(ShellDev<R>) * (size_t)(kMaxShells - n_shells));
}
// NSH > 0: the stride is that of NSH shells, known at compile time (the wavefront kernel's hot path: a run-time stride
// cost its steady state 2.5 %); NSH = 0: the run-time stride.
template <typename R, int NSH> struct NucTab {
  const unsigned char *base;
  int stride;
  __device__ __forceinline__ const NucDev<R> &operator[](int t) const {
    const size_t s = NSH > 0 ? sizeof(NucDev<R>) - sizeof(ShellDev<R>) * (size_t)(kMaxShells - NSH) : (size_t)stride;
    return *reinterpret_cast<const NucDev<R> *>(base + (size_t)t * s);
  }
};
template <typename R> __host__ __device__ inline size_t model_smem_bytes(int n_xs, int n_stage, int n_shells) {
  return (size_t)nuc_stride_bytes<R>(n_shells) * (size_t)n_stage + sizeof(R) * 4 * (size_t)n_xs;
}

template <typename R>
__device__ __forceinline__ void stage_model(const ModelDev<R> &model, int n_stage, int stride, unsigned char *s_nuc, R *s_tabS) {
  const int nw = stride / 4;
  for (int t = 0; t < n_stage; ++t) {
    uint32_t *dst = reinterpret_cast<uint32_t *>(s_nuc + (size_t)t * (size_t)stride);
    if (!model.nuc[t].live) { if (threadIdx.x == 0) reinterpret_cast<NucDev<R> *>(dst)->live = 0; continue; }
    const uint32_t *src = reinterpret_cast<const uint32_t *>(&model.nuc[t]);
    for (int i = threadIdx.x; i < nw; i += blockDim.x) dst[i] = src[i];
  }
  const int nt = model.n_xs * 4;
  for (int i = threadIdx.x; i < nt; i += blockDim.x) s_tabS[i] = model.tabS[i];
  __syncthreads();
}

// validate an event's inputs; on failure write neutral outputs and raise the device error word
template <typename R, typename TAB>
__device__ __forceinline__ bool check_inputs(const CascadeParams<R> &P, const TAB &s_nuc, int ev, R E_in, int tgt, int ptype) {
  unsigned err = 0;
  if (ptype != 0 && ptype != 1) err |= 8u;
  if (!(E_in >= R(INC_E_MIN) && E_in <= R(INC_E_MAX))) err |= 1u;
  if (tgt < 0 || tgt >= P.n_stage) err |= 2u;
  else if (!s_nuc[tgt].live) err |= 2u;
  if (!err) return true;
  atomicOr(&P.ctr->error_word, err);
  NucRec<R> r;
  r.E = R(0); r.Px = R(0); r.Py = R(0); r.Pz = R(0); r.A = 0; r.Z = 0; r.meta = (1u << 16); r.status = INC_ST_FAILED;
  P.ws.crec[ev] = r;
  return false;
}

template <typename R>
__device__ __forceinline__ void write_cascade_result(const Workspace<R> &ws, int ev, int A, int Z, R Es, R Px, R Py, R Pz,
                                                     uint32_t meta, uint32_t status) {
  NucRec<R> r;
  r.E = Es; r.Px = Px; r.Py = Py; r.Pz = Pz; r.A = A; r.Z = Z; r.meta = meta; r.status = status;
  ws.crec[ev] = r;          // 16-byte vector stores
}

// Order-independent sums (escaped energy and momentum): fixed point, so that any processing order of
// an event's tracks gives bit-identical residuals.  double: int64, unit 2^-40 MeV; float: int32, unit
// 2^-20 MeV (|values| < 2048 MeV, resolution below the fp32 rounding of the addends).
template <typename R> struct Fx;
template <> struct Fx<double> {
  typedef long long T; typedef unsigned long long U;
  static __device__ __forceinline__ T to(double v) { return __double2ll_rn(v * 1099511627776.0); }
  static __device__ __forceinline__ double from(T v) { return (double)v * (1.0 / 1099511627776.0); }
};
template <> struct Fx<float> {
  typedef int T; typedef unsigned int U;
  static __device__ __forceinline__ T to(float v) { return __float2int_rn(v * 1048576.0f); }
  static __device__ __forceinline__ float from(T v) { return (float)v * (1.0f / 1048576.0f); }
};

}  // namespace inc
