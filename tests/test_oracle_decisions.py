"""Pins of the oracle's DECISION LOGIC at event level ("What's weak 1"): the wiring inside
`cascade_attempt` (which sigma / B / a table a species pair reads, the partner-type draw, which species' E_F
and V a product is tested against, the E_C cutoff, the child path codes), the entry distribution C0, the three
retry rules of C6, the channel choice E3 and the interior branch of the Dostrovsky interpolation.

Each pin compares the oracle with something other than itself: a closed form, a structural consequence of a
zeroed table, a quadrature of independently written kinematics, numpy.interp, or a recount from the trace.
tests/test_pins_bite.py breaks the oracle in the way each pin is meant to notice and checks that it does.
P:49 = PAPER.md line 49 (cross sections, Pauli blocking, cutoff); P:53 evaporation; R-xx = DESIGN.md section 3.
"""
import ctypes as C

import numpy as np
import pytest
from scipy import integrate, stats

from helpers import blocked_indicator_independent

DP = C.POINTER(C.c_double)


def flat_tables(orc, sig_pp, sig_np, B_pp=0.0, B_np=0.0, a_np=0.0, **kw):
    """Tables whose NN arrays are constants: the collision rate then does not depend on the partner's momentum,
    so every closed form below is exact."""
    t = orc.Tables(**kw)
    n = t.n_xs
    t.sig_pp, t.sig_np = np.full(n, float(sig_pp)), np.full(n, float(sig_np))
    t.B_pp, t.B_np, t.a_np = np.full(n, float(B_pp)), np.full(n, float(B_np)), np.full(n, float(a_np))
    return t.refresh()


def traces(orc, t, target, E, n, seed=7, proj=1, attempt=0, flags=0):
    nu = orc.setup_nucleus(target[0], target[1], t)
    return [orc.cascade_trace(t, nu, seed, e, attempt, E, proj=proj, flags=flags) for e in range(n)]


def type_from_code(pi, proj, recoil_flips):
    """Species of the track with path code pi when every recoil (odd child, R-R2) has the opposite species of its
    parent (recoil_flips) or the same one; the scattered child (even) always keeps it."""
    bits = bin(int(pi))[3:]          # below the leading 1
    typ = proj
    for b in bits:
        if b == "1" and recoil_flips:
            typ = 1 - typ
    return typ


# ------------------------------------------------------------------ sigma table wiring (oracle C2)
def test_zeroed_sigma_table_fixes_the_partner_species(orc):
    """sigma_np = 0: like particles only, so a proton beam knocks out protons only and a neutron beam neutrons
    only (pp table also serves nn).  sigma_pp = 0: unlike partners only, so the species of every track
    follows from its path code.  A swap of the two tables for either track species breaks one of these."""
    t = orc.Tables()
    t.sig_np = np.zeros(t.n_xs)
    t.refresh()
    n = 1500
    for proj in (1, 0):
        r = orc.simulate(t, [(16, 8)], np.full(n, 200.0), np.zeros(n, dtype=np.int32), 3, flags=orc.F_CASCADE_ONLY,
                         projectile=np.full(n, proj, dtype=np.uint8))
        assert not np.any(r["status"] & orc.ST_FAILED)
        assert r["stats"]["allowed"] > n and np.sum(r["counts"] >= 2) > n // 4
        assert np.all(r["species"] == proj)
    t = orc.Tables()
    t.sig_pp = np.zeros(t.n_xs)
    t.refresh()
    n_coll = n_esc = 0
    for proj in (1, 0):
        for tr in traces(orc, t, (16, 8), 200.0, 600, seed=4, proj=proj):
            c = tr["coll"]
            assert np.all(c["type1"] != c["type2"])
            n_coll += len(c)
            for pi, typ in zip(tr["esc_pi"], tr["esc_type"]):
                assert typ == type_from_code(pi, proj, recoil_flips=True)
                n_esc += pi > 1
    assert n_coll > 1000 and n_esc > 300


# ------------------------------------------------------------------ Sigma, free path, entry disc, partner draw
@pytest.mark.parametrize("proj", [1, 0])
def test_flat_sigma_one_shell_closed_forms(orc, proj):
    """One constant-density shell, momentum-independent sigma_pp = 30 mb, sigma_np = 50 mb, 48Ti (N != Z).
    (i) An attempt has no collision with probability (2/R^2) int_0^R b db exp(-Sigma chord(b)): uniform disc
    (R-C0), exponential path with Sigma = rho_p sigma_.p + rho_n sigma_.n (R-C2), straight chord
    2 sqrt(R^2 - (b p_0/p_1)^2) inside the potential step (angular momentum b p_0 conserved, R-C4).
    (ii) The partner of a collision is a proton with probability rho_p sigma_.p / Sigma (R-C3)."""
    A, Z, E = 48, 22, 150.0
    s_pp, s_np = 30.0, 50.0
    t = flat_tables(orc, s_pp, s_np, n_shells=1)
    nu = orc.nucleus_arrays(orc.setup_nucleus(A, Z, t))
    R = nu["R"]
    vol = 4.0 / 3.0 * np.pi * R ** 3
    rho_p, rho_n = Z / vol, (A - Z) / vol                       # one shell: the mean density (R-N2)
    assert nu["rho_p"][0] == pytest.approx(rho_p, rel=1e-12) and nu["rho_n"][0] == pytest.approx(rho_n, rel=1e-12)
    sp, sn = (s_pp, s_np) if proj else (s_np, s_pp)              # against a proton / a neutron partner
    Sigma = 0.1 * (rho_p * sp + rho_n * sn)                      # mb -> fm^2
    m = orc.M_P if proj else orc.M_N
    V = (nu["V_p"] if proj else nu["V_n"])[0]
    p0, p1 = np.sqrt(E * (E + 2 * m)), np.sqrt((E + V) * (E + V + 2 * m))
    f = lambda b: b * np.exp(-Sigma * 2.0 * np.sqrt(max(R * R - (b * p0 / p1) ** 2, 0.0)))
    P0 = 2.0 / R ** 2 * integrate.quad(f, 0.0, R, epsabs=0, epsrel=1e-11)[0]
    n = 12000
    trs = traces(orc, t, (A, Z), E, n, seed=11, proj=proj)
    none = sum(len(tr["coll"]) == 0 for tr in trs)
    assert 0.1 < P0 < 0.9
    assert abs(none / n - P0) < 3.0 * np.sqrt(P0 * (1 - P0) / n), (none / n, P0)
    first = np.array([tr["coll"]["type2"][0] for tr in trs if len(tr["coll"])])   # the projectile's first collision
    share = 0.1 * rho_p * sp / Sigma
    assert abs(first.mean() - share) < 3.0 * np.sqrt(share * (1 - share) / len(first)), (first.mean(), share)
    # the logged macroscopic cross sections are these numbers
    c = np.concatenate([tr["coll"] for tr in trs])
    own = c[c["pi"] == 1]
    assert np.allclose(own["Sigma"], Sigma, rtol=1e-12) and np.allclose(own["Sp"], 0.1 * rho_p * sp, rtol=1e-12)


def test_entry_points_are_uniform_on_the_disc(orc):
    """R-C0: b = R sqrt(u), azimuth uniform.  One shell, sigma = 0, transparent attempts kept: the proton leaves
    deflected by Theta(b) = 2 [asin(b/R) - asin(b p_0/(p_1 R))] (monotone in b), in the plane of incidence; so
    the observed directions give b back, and (b/R)^2 and the azimuth must be uniform."""
    t = flat_tables(orc, 0.0, 0.0, n_shells=1)
    A, Z, E, n = 40, 20, 100.0, 4000
    nu = orc.nucleus_arrays(orc.setup_nucleus(A, Z, t))
    r = orc.simulate(t, [(A, Z)], np.full(n, E), np.zeros(n, dtype=np.int32), 5,
                     flags=orc.F_KEEP_TRANSPARENT | orc.F_CASCADE_ONLY)
    assert np.all(r["counts"] == 1) and np.allclose(r["T"], E, rtol=1e-12)
    p0 = np.sqrt(E * (E + 2 * orc.M_P))
    p1 = np.sqrt((E + nu["V_p"][0]) * (E + nu["V_p"][0] + 2 * orc.M_P))
    x = np.sin(np.linspace(0.0, np.pi / 2, 20001))                  # b/R, dense near 1
    theta_of_x = 2.0 * (np.arcsin(x) - np.arcsin(x * p0 / p1))
    assert np.all(np.diff(theta_of_x) > 0)
    theta = np.arccos(np.clip(r["uz"], -1, 1))
    xb = np.interp(theta, theta_of_x, x)
    assert stats.kstest(xb ** 2, "uniform").pvalue > 1e-3
    assert np.mean(xb ** 2) == pytest.approx(0.5, abs=4 * np.sqrt(1 / 12 / n))        # <b^2> = R^2/2
    phi = np.arctan2(-r["uy"], -r["ux"]) % (2 * np.pi)                             # bent towards the axis
    assert stats.kstest(phi, "uniform", args=(0, 2 * np.pi)).pvalue > 1e-3


# ------------------------------------------------------------------ Pauli blocking: whose E_F (R-Q12)
def test_blocked_fraction_of_projectile_collisions_vs_quadrature(orc):
    """48Ti (E_F,n != E_F,p), one shell, flat sigma and slope: every collision of the incident proton happens at
    T_1 = E_in + V_p against an unbiased Fermi-sea partner, so the blocked fraction per partner species equals a
    deterministic quadrature of the independently written kinematics (helpers.blocked_indicator_independent)
    with the proton's E_F for the projectile and the PARTNER species' p_F and E_F for the recoil."""
    A, Z, E, B = 48, 22, 10.0, 3.0      # slow projectile: both products end near their Fermi energies
    t = flat_tables(orc, 40.0, 40.0, B_pp=B, B_np=B, a_np=0.0, n_shells=1)
    nu = orc.nucleus_arrays(orc.setup_nucleus(A, Z, t))
    trs = traces(orc, t, (A, Z), E, 15000, seed=13)
    c = np.concatenate([tr["coll"] for tr in trs])
    own = c[c["pi"] == 1]
    T1 = E + nu["V_p"][0]
    assert np.allclose(own["T_in"], T1, rtol=1e-12)
    g = lambda k: (np.arange(k) + 0.5) / k
    umag, ucos, uphk, ut, uph = np.meshgrid(g(20), g(20), g(16), g(28), g(24), indexing="ij", sparse=True)
    shape = np.broadcast_shapes(umag.shape, ucos.shape, uphk.shape, ut.shape, uph.shape)
    for t2, m2, pF2, EF2 in ((1, orc.M_P, nu["pF_p"][0], nu["EF_p"][0]), (0, orc.M_N, nu["pF_n"][0], nu["EF_n"][0])):
        sel = own[own["type2"] == t2]
        ind = blocked_indicator_independent(T1, orc.M_P, m2, pF2, nu["EF_p"][0], EF2, B, np.cbrt(umag), 2 * ucos - 1,
                                            2 * np.pi * uphk, ut, 2 * np.pi * uph)
        fq = float(np.mean(np.broadcast_to(ind, shape)))
        fm = float(np.mean(sel["blocked"]))
        assert len(sel) > 3000 and 0.1 < fq < 0.9
        assert abs(fm - fq) < 3.0 * np.sqrt(fq * (1 - fq) / len(sel)) + 3e-3, (t2, fm, fq, len(sel))


# ------------------------------------------------------------------ cutoff: E_C for protons only, own V (R-Q7)
def test_cutoff_thresholds_show_in_the_escape_spectra(orc, otables):
    """eps = T - V is conserved between collisions (R-C4), so a nucleon created with eps leaves with T_out = eps:
    every cascade proton of an accepted event (path code >= 2) has T_out > E_C, every neutron T_out > 0, and
    both spectra start right at their threshold (populated first MeV)."""
    A, Z, n = 40, 20, 12000
    nu = orc.setup_nucleus(A, Z, otables)
    EC = nu.EC
    assert EC == pytest.approx(1.43996448 * Z / nu.R, rel=1e-12) and 3.0 < EC < 6.0
    r = orc.simulate(otables, [(A, Z)], np.full(n, 150.0), np.zeros(n, dtype=np.int32), 8, flags=orc.F_CASCADE_ONLY)
    Tp, Tn = r["T"][r["species"] == 1], r["T"][r["species"] == 0]
    assert Tp.min() > EC - 1e-9 and np.sum(Tp < EC + 1.0) > 100
    assert Tn.min() > 0.0 and np.sum(Tn < 2.0) > 30 and np.sum(Tn < EC) > 150
    # nothing is trapped behind a wrong well depth (a nucleon that passes the cutoff can always leave)
    assert r["stats"]["cap_seg"] <= 2


# ------------------------------------------------------------------ child path codes and species (R-R2, R-C3)
def test_track_tree_is_consistent(orc, otables):
    """Children of an allowed collision of track pi are 2 pi (the scattered projectile, same species) and
    2 pi + 1 (the recoil, the partner's species), k restarts; a blocked collision leaves the track alive; every
    track ends exactly once (escape, allowed collision, or absorption at creation)."""
    n_tracks = 0
    for tr in traces(orc, otables, (16, 8), 200.0, 400, seed=21):
        species = {1: 1}
        ended = set()
        last_k = {}
        for c in tr["coll"]:
            pi = int(c["pi"])
            assert pi in species and pi not in ended and species[pi] == c["type1"]
            assert last_k.get(pi, 0) < c["k"]                # blocks of a track are consumed in order
            last_k[pi] = int(c["k"])
            if not c["blocked"]:
                ended.add(pi)
                if c["keep1"]:
                    species[2 * pi] = int(c["type1"])
                if c["keep2"]:
                    species[2 * pi + 1] = int(c["type2"])
        assert tr["n_real"] == int(np.sum(tr["coll"]["blocked"] == 0))
        assert np.all(np.diff(tr["esc_pi"].astype(np.int64)) > 0)
        for pi, typ in zip(tr["esc_pi"], tr["esc_type"]):
            assert int(pi) in species and int(pi) not in ended and species[int(pi)] == typ
            ended.add(int(pi))
        if not (tr["status"] & (orc.ST_SEG_CAP | orc.ST_DEPTH_CAP)):
            assert ended == set(species)
        n_tracks += len(species)
    assert n_tracks > 800


# ------------------------------------------------------------------ B and a tables (R-C3)
def test_angular_tables_wiring(orc):
    """B_pp = 0 and no backward term for like pairs: isotropic in the CM frame.  Unlike pairs read B_np = 6 and
    a_np = 0.5: P(cos < 0) = q (1 - f) + (1 - q) f with the forward law's own backward share
    q = (e^{B t_min / 2} - e^{B t_min}) / (1 - e^{B t_min}) and the mirror probability f = a / (1 + a), summed
    over the collisions' own p_cm (from the logged p_lab by the invariant s)."""
    t = flat_tables(orc, 40.0, 40.0, B_pp=0.0, B_np=6.0, a_np=0.5)
    c = np.concatenate([tr["coll"] for tr in traces(orc, t, (16, 8), 220.0, 2500, seed=31)])
    like, unlike = c[c["type1"] == c["type2"]], c[c["type1"] != c["type2"]]
    assert len(like) > 2000 and len(unlike) > 2000
    assert stats.kstest(like["costheta"], "uniform", args=(-1, 2)).pvalue > 1e-3
    m1 = np.where(unlike["type1"] == 1, orc.M_P, orc.M_N)
    m2 = np.where(unlike["type2"] == 1, orc.M_P, orc.M_N)
    pl = unlike["plab"] * 1000.0
    s = m1 ** 2 + m2 ** 2 + 2 * m2 * np.sqrt(pl ** 2 + m1 ** 2)
    pcm2 = (s - (m1 + m2) ** 2) * (s - (m1 - m2) ** 2) / (4 * s) * 1e-6
    Bt = 6.0 * (-4.0 * pcm2)
    q = (np.exp(Bt / 2) - np.exp(Bt)) / (1 - np.exp(Bt))
    f = 0.5 / 1.5
    pback = q * (1 - f) + (1 - q) * f
    back = np.sum(unlike["costheta"] < 0)
    assert abs(back - pback.sum()) < 3.0 * np.sqrt(np.sum(pback * (1 - pback))), (back, pback.sum())


# ------------------------------------------------------------------ retry rules (R-C6 / R-Q18)
def test_retry_rules_recounted_from_traces(orc, otables):
    """The three retry conditions, in their order (transparent; residual not a nucleus; E* < 0), recounted
    attempt by attempt from the traces with the 4-momentum balance written out here, against orc_simulate's
    counters, its attempts-used status bits and its post-cascade residuals."""
    L = orc.lib()
    tp = C.byref(otables.c)
    light = {(1, 0), (1, 1), (2, 1), (3, 1), (3, 2), (4, 2)}
    cases = [((6, 3), 230.0, 400, 41), ((12, 6), 60.0, 400, 42)]
    tot = dict(t=0, i=0, e=0)
    for (A, Z), E, n, seed in cases:
        r = orc.simulate(otables, [(A, Z)], np.full(n, E), np.zeros(n, dtype=np.int32), seed, flags=orc.F_CASCADE_ONLY)
        nu = orc.setup_nucleus(A, Z, otables)
        Mt = L.orc_mass(A, Z, tp)
        p_in = np.sqrt(E * (E + 2 * orc.M_P))
        cnt = dict(t=0, i=0, e=0)
        for e in range(n):
            for a in range(256):
                tr = orc.cascade_trace(otables, nu, seed, e, a, E)
                ne, n_p = len(tr["esc_pi"]), int(np.sum(tr["esc_type"]))
                Ar, Zr = A + 1 - ne, Z + 1 - n_p
                if tr["n_real"] == 0:
                    cnt["t"] += 1
                    continue
                if not ((Ar, Zr) in light or (Ar >= 5 and 0 <= Zr <= Ar)):
                    cnt["i"] += 1
                    continue
                mk = np.where(tr["esc_type"] == 1, orc.M_P, orc.M_N)
                Er = E + orc.M_P + Mt - np.sum(tr["esc_T"] + mk)
                Pr = np.array([0.0, 0.0, p_in]) - tr["esc_p"].sum(axis=0)
                Es = np.sqrt(Er * Er - Pr @ Pr) - L.orc_mass(Ar, Zr, tp)
                if Es < 0.0:
                    cnt["e"] += 1
                    continue
                break
            assert (r["status"][e] & 0xFF) == a + 1, e
            assert (r["casc_A"][e], r["casc_Z"][e], r["casc_count"][e]) == (Ar, Zr, ne)
            assert r["casc_Estar"][e] == pytest.approx(Es, abs=1e-7)
        st = r["stats"]
        assert (st["retry_transparent"], st["retry_invalid"], st["retry_estar"]) == (cnt["t"], cnt["i"], cnt["e"])
        for k in cnt:
            tot[k] += cnt[k]
    assert tot["t"] > 100 and tot["i"] > 0 and tot["e"] > 5      # every rule was exercised


# ------------------------------------------------------------------ channel choice (R-E3)
@pytest.mark.parametrize("A,Z,Es", [(16, 8, 30.0), (48, 22, 80.0)])
def test_channel_choice_follows_the_widths(orc, otables, A, Z, Es):
    L = orc.lib()
    arrs = [(C.c_double * 6)() for _ in range(6)]
    Wsum = L.orc_evap_widths(A, Z, Es, C.byref(otables.c), *arrs)
    W = np.array(arrs[0][:])
    assert np.sum(W > 0) >= 4
    rng = np.random.default_rng(A)
    n = 100000
    picks = np.array([L.orc_evap_choose(arrs[0], Wsum, float(u)) for u in rng.random(n)])
    obs = np.bincount(picks, minlength=6).astype(float)
    exp = W / Wsum * n
    assert np.all(obs[W == 0] == 0)
    big = exp >= 10
    o = np.append(obs[big], obs[~big].sum())
    e = np.append(exp[big], exp[~big].sum())
    if e[-1] == 0:
        o, e = o[:-1], e[:-1]
    assert stats.chi2.sf(np.sum((o - e) ** 2 / e), len(e) - 1) > 1e-3, (obs, exp)
    # exact: u just below / above each cumulative boundary, in the E1 order n, p, d, t, 3He, 4He
    cum = np.cumsum(W) / Wsum
    open_j = np.nonzero(W > 0)[0]
    for a, j in enumerate(open_j[:-1]):
        assert L.orc_evap_choose(arrs[0], Wsum, float(cum[j]) * (1 - 1e-12)) == j
        assert L.orc_evap_choose(arrs[0], Wsum, float(cum[j]) * (1 + 1e-12)) == open_j[a + 1]
    assert L.orc_evap_choose(arrs[0], Wsum, 1.0 - 2.0 ** -33) == open_j[-1]
    assert L.orc_evap_choose(arrs[0], Wsum, 2.0 ** -33) == open_j[0]


# ------------------------------------------------------------------ Dostrovsky interpolation, interior (R-T)
def test_dostrovsky_interpolation_interior(orc, otables):
    L = orc.lib()
    zz = otables.ev_Z
    for name in ("ev_kp", "ev_cp", "ev_ka", "ev_ca"):
        y = getattr(otables, name)
        z = np.concatenate([np.arange(0, 81, dtype=float), [10.5, 19.999, 20.001, 49.5, 69.9]])
        got = np.array([L.orc_lerp_z(zz.ctypes.data_as(DP), y.ctypes.data_as(DP), len(zz), float(v)) for v in z])
        assert np.allclose(got, np.interp(z, zz, y), rtol=1e-14, atol=0)
    # Coulomb barriers and alpha_j = 1 + c_j at daughter charges 15, 20, 21 (configs 3-5 run up to Z_d = 22)
    e2 = 1.43996448
    arrs = [(C.c_double * 6)() for _ in range(6)]
    for (A, Z), kp, cp, ka, ca in (((32, 16), 0.50, 0.39, 0.75, 0.10),     # Z_d(p) = 15: halfway between rows 10 and 20
                                   ((42, 21), 0.58, 0.28, 0.82, 0.10),     # Z_d(p) = 20: on the knot
                                   ((46, 22), 0.59, 0.272, 0.829, 0.10)):  # Z_d(p) = 21
        Wsum = L.orc_evap_widths(A, Z, 120.0, C.byref(otables.c), *arrs)
        W, X, Q, V, beta, a = [np.array(x[:]) for x in arrs]
        Zd = Z - 1
        assert V[1] == pytest.approx(kp * e2 * Zd / (1.5 * (A - 1) ** (1 / 3)), rel=1e-12)
        assert V[2] == pytest.approx((kp + 0.06) * e2 * Zd / (1.5 * (A - 2) ** (1 / 3) + 1.2), rel=1e-12)
        assert V[3] == pytest.approx((kp + 0.12) * e2 * Zd / (1.5 * (A - 3) ** (1 / 3) + 1.2), rel=1e-12)
        # alpha_p from the width: W_p / (g M A_d^(2/3) int_0^X x e^{2 sqrt(a(X-x))} dx) = 1 + c_p(Z_d)
        s = 2 * np.sqrt(a[1] * X[1])
        I = integrate.quad(lambda x: x * np.exp(2 * np.sqrt(a[1] * (X[1] - x)) - s), 0, X[1], epsabs=0, epsrel=1e-13)[0] * np.exp(s)
        assert W[1] / (2 * orc.SPECIES_M[1] * (A - 1) ** (2 / 3) * I) == pytest.approx(1 + cp, rel=1e-9)
    # the alpha channel of (46,22) has Z_d = 20 (knot), its 3He channel too; (47,23) -> alpha daughter Z_d = 21
    Wsum = L.orc_evap_widths(47, 23, 120.0, C.byref(otables.c), *arrs)
    V = np.array(arrs[3][:])
    assert V[5] == pytest.approx(0.829 * e2 * 2 * 21 / (1.5 * 43 ** (1 / 3) + 1.2), rel=1e-12)
    assert V[4] == pytest.approx((0.829 - 0.06) * e2 * 2 * 21 / (1.5 * 44 ** (1 / 3) + 1.2), rel=1e-12)
