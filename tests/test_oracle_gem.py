"""Pins of the oracle's GEM level density ("we adopt the generalized evaporation model
(GEM) [18]"; DESIGN.md R-G1..G6): Gilbert-Cameron matching, constant-temperature branch, pre-exponential factor,
caller-supplied pairing and shell corrections.  It changes E2 (widths) and E4 (sampler) only."""
import ctypes as C

import numpy as np
import pytest
from scipy import integrate, stats

G = np.array([2, 2, 3, 2, 2, 1], dtype=float)


def gem_tables(orc, pairing=False, shells=False, **kw):
    """GEM mode; optional pairing 12/sqrt(A)-like table (even Z or N: 1.2 MeV, odd: 0) and a smooth fake shell
    correction -- the arrays are caller inputs of the model, any values will do for the pins."""
    pz = pn = sz = sn = None
    if pairing:
        pz = np.where(np.arange(40) % 2 == 0, 1.2, 0.0)
        pn = np.where(np.arange(40) % 2 == 0, 1.1, 0.0)
    if shells:
        sz = 3.0 * np.sin(np.arange(40) / 4.0)
        sn = -2.0 * np.cos(np.arange(40) / 5.0)
    return orc.Tables(level_density=1, pair_Z=pz, pair_N=pn, shell_Z=sz, shell_N=sn, **kw)


def _ld(orc, t, Ad, Zd):
    ld = orc.OrcLd()
    assert orc.lib().orc_gem_ld(Ad, Zd, C.byref(t.c), C.byref(ld)) == 0
    return ld


def _widths(orc, t, A, Z, Es):
    arrs = [(C.c_double * 6)() for _ in range(6)]
    tot = orc.lib().orc_evap_widths(A, Z, Es, C.byref(t.c), *arrs)
    return (tot,) + tuple(np.array(x[:]) for x in arrs)


def test_level_density_constants_and_matching(orc):
    """R-G2..G4: a = A_d (a0 + a1 S), delta from the pairing arrays, U_x = 150/A_d + 2.5; the two branches meet at
    E_x = U_x + delta with equal value, and the constant-temperature slope is the Fermi-gas slope minus 1/(4 U_x)
    (the matching of [18]: 1/T = sqrt(a/U_x) - 1.5/U_x against d/dU [2 sqrt(aU) - 5/4 ln U])."""
    L = orc.lib()
    t = gem_tables(orc, pairing=True, shells=True)
    for Ad, Zd in ((15, 7), (12, 6), (47, 22), (44, 20), (5, 2)):
        ld = _ld(orc, t, Ad, Zd)
        S = t.shell_Z[Zd] + t.shell_N[Ad - Zd]
        assert ld.a == pytest.approx(Ad * (0.125 + 0.00917 * S), rel=1e-14)
        assert ld.delta == pytest.approx(t.pair_Z[Zd] + t.pair_N[Ad - Zd], rel=1e-14)
        assert ld.Ux == pytest.approx(150.0 / Ad + 2.5, rel=1e-14) and ld.Ex == pytest.approx(ld.Ux + ld.delta, rel=1e-14)
        lo, hi = L.orc_gem_lnrho(C.byref(ld), ld.Ex * (1 - 1e-13)), L.orc_gem_lnrho(C.byref(ld), ld.Ex * (1 + 1e-13))
        assert lo == pytest.approx(hi, abs=1e-10)
        h = 1e-4
        s_ct = (L.orc_gem_lnrho(C.byref(ld), ld.Ex - h) - L.orc_gem_lnrho(C.byref(ld), ld.Ex - 3 * h)) / (2 * h)
        s_fg = (L.orc_gem_lnrho(C.byref(ld), ld.Ex + 3 * h) - L.orc_gem_lnrho(C.byref(ld), ld.Ex + h)) / (2 * h)
        assert s_ct == pytest.approx(np.sqrt(ld.a / ld.Ux) - 1.5 / ld.Ux, rel=1e-6)
        assert s_fg - s_ct == pytest.approx(0.25 / ld.Ux, rel=1e-3)
        # far above E_x the density is the Fermi gas with its pre-exponential factor: rho U^(5/4) a^(1/4) e^(-2 sqrt(aU)) = 1
        U = ld.delta + 90.0
        assert L.orc_gem_lnrho(C.byref(ld), U) + 1.25 * np.log(90.0) + 0.25 * np.log(ld.a) - 2 * np.sqrt(ld.a * 90.0) == pytest.approx(0.0, abs=1e-11)
    # pairing is a pure back-shift of the whole curve: rho(U; delta) = rho(U - delta; 0)
    t0 = gem_tables(orc, pairing=False, shells=True)
    for Ad, Zd in ((16, 8), (46, 22)):
        a, b = _ld(orc, t, Ad, Zd), _ld(orc, t0, Ad, Zd)
        assert a.delta > 2.0 and b.delta == 0.0 and a.a == b.a
        for U in (a.delta + 0.3, a.Ex - 0.1, a.Ex + 0.1, a.delta + 40.0):
            assert L.orc_gem_lnrho(C.byref(a), U) == pytest.approx(L.orc_gem_lnrho(C.byref(b), U - a.delta), abs=1e-11)
    # entries beyond the arrays count as zero; a <= 0 closes the channel
    short = orc.Tables(level_density=1, pair_Z=[0.0, 5.0], pair_N=[0.0, 0.0, 7.0])
    assert _ld(orc, short, 3, 1).delta == 12.0 and _ld(orc, short, 30, 15).delta == 0.0
    neg = orc.Tables(level_density=1, shell_Z=np.full(40, -20.0))
    assert L.orc_gem_ld(20, 10, C.byref(neg.c), C.byref(orc.OrcLd())) == -1
    assert _widths(orc, neg, 21, 10, 60.0)[1][0] == 0.0


@pytest.mark.parametrize("A,Z,Es", [(16, 8, 30.0), (17, 9, 200.0), (48, 22, 80.0), (12, 6, 22.0), (15, 7, 11.0), (41, 21, 250.0)])
@pytest.mark.parametrize("corr", [False, True])
def test_gem_widths_vs_numerical_integration(orc, A, Z, Es, corr):
    """W_j = g_j M_j A_d^(2/3) alpha_j int_0^X (x + beta_j) rho_d(X - x) dx against scipy.integrate.quad of the
    piecewise integrand written out here (break point at the daughter excitation E_x)."""
    L = orc.lib()
    t = gem_tables(orc, pairing=corr, shells=corr)
    tw = orc.Tables()                                   # mode 0: same Q, V, beta, X (E2's integrand is all that changes)
    tot, W, X, Q, V, beta, a = _widths(orc, t, A, Z, Es)
    tot0, W0, X0, Q0, V0, beta0, a0 = _widths(orc, tw, A, Z, Es)
    assert np.array_equal(X, X0) and np.array_equal(V, V0) and np.array_equal(beta, beta0)
    assert tot == pytest.approx(W.sum(), rel=1e-14)
    n_open = 0
    for j in range(6):
        if X[j] <= 0:
            assert W[j] == 0.0
            continue
        n_open += 1
        Ad, Zd = int(A - orc.SPECIES_A[j]), int(Z - orc.SPECIES_Z[j])
        at = lambda y, i: float(y[i]) if i < len(y) else 0.0
        S = at(t.shell_Z, Zd) + at(t.shell_N, Ad - Zd)
        aa = Ad * (0.125 + 0.00917 * S)
        delta = at(t.pair_Z, Zd) + at(t.pair_N, Ad - Zd)
        assert a[j] == pytest.approx(aa, rel=1e-14)
        Ux = 150.0 / Ad + 2.5
        Ex = Ux + delta
        T = 1.0 / (np.sqrt(aa / Ux) - 1.5 / Ux)
        E0 = Ex - T * (np.log(T) - 0.25 * np.log(aa) - 1.25 * np.log(Ux) + 2 * np.sqrt(aa * Ux))
        ref = 2 * np.sqrt(aa * max(X[j] - delta, Ux))        # scale of the exponent, to keep quad well conditioned

        def rho(U):
            if U >= Ex:
                return np.exp(2 * np.sqrt(aa * (U - delta)) - ref) / (aa ** 0.25 * (U - delta) ** 1.25)
            return np.exp((U - E0) / T - ref) / T
        f = lambda x: (x + beta[j]) * rho(X[j] - x)
        xs = X[j] - Ex
        if xs > 0:
            I = (integrate.quad(f, 0, xs, epsabs=0, epsrel=1e-13, limit=400)[0] +
                 integrate.quad(f, xs, X[j], epsabs=0, epsrel=1e-13, limit=400)[0])
        else:
            I = integrate.quad(f, 0, X[j], epsabs=0, epsrel=1e-13, limit=400)[0]
        Ad13 = Ad ** (1.0 / 3.0)
        # alpha_j as in mode 0 (pinned in test_oracle_evap / test_oracle_decisions): take it from the mode-0 width
        s0 = 2 * np.sqrt(a0[j] * X[j])
        I0 = integrate.quad(lambda x: (x + beta[j]) * np.exp(2 * np.sqrt(a0[j] * (X[j] - x)) - s0), 0, X[j], epsabs=0, epsrel=1e-13, limit=400)[0]
        alpha = W0[j] / (G[j] * orc.SPECIES_M[j] * Ad13 ** 2 * I0 * np.exp(s0))
        assert W[j] == pytest.approx(G[j] * orc.SPECIES_M[j] * Ad13 ** 2 * alpha * I * np.exp(ref), rel=2e-10), j
    assert n_open >= 1


@pytest.mark.parametrize("Ad,Zd,X,beta", [(15, 7, 25.0, 0.0), (15, 8, 3.0, 0.64), (46, 22, 60.0, 0.3), (12, 6, 16.5, 0.0), (30, 14, 9.0, 0.0)])
def test_gem_sampler_matches_pdf(orc, Ad, Zd, X, beta):
    """Histogram of sampled x vs the normalised (x + beta) rho(X - x): daughter entirely below E_x (pure constant
    temperature: X = 3), straddling the matching energy, and far above it."""
    L = orc.lib()
    t = gem_tables(orc, pairing=True, shells=True)
    ld = _ld(orc, t, Ad, Zd)
    n = 40000
    key = (C.c_uint32 * 2)(321, 654)
    k = C.c_uint32(0)
    tr = C.c_int(0)
    xs = np.array([L.orc_evap_sample_x_gem(C.byref(ld), X, beta, key, 7, i, 0, C.byref(k), C.byref(tr)) for i in range(n)])
    assert np.all((xs >= 0) & (xs <= X))
    assert tr.value / n < 1 / 0.25
    l0 = L.orc_gem_lnrho(C.byref(ld), X)
    f = lambda x: (x + beta) * np.exp(L.orc_gem_lnrho(C.byref(ld), max(X - x, 0.0)) - l0)
    nb = 25
    edges = np.linspace(0, X, nb + 1)
    brk = X - ld.Ex
    probs = np.array([integrate.quad(f, edges[i], edges[i + 1], points=[brk] if edges[i] < brk < edges[i + 1] else None)[0] for i in range(nb)])
    probs /= probs.sum()
    obs = np.histogram(xs, edges)[0]
    keep = probs * n >= 10
    o = np.append(obs[keep], obs[~keep].sum())
    e = np.append(probs[keep] * n, probs[~keep].sum() * n)
    if e[-1] == 0:
        o, e = o[:-1], e[:-1]
    assert stats.chi2.sf(np.sum((o - e) ** 2 / e), len(e) - 1) > 1e-3
    # the envelope really is one: ln rho(X - x) <= ln rho(X) - x m on a fine grid, m = the smallest slope
    m = 1.0 / ld.T
    if X > ld.Ex:
        m = min(m, np.sqrt(ld.a / (X - ld.delta)) - 1.25 / (X - ld.delta))
    xg = np.linspace(0, X, 4001)
    lr = np.array([L.orc_gem_lnrho(C.byref(ld), max(X - x, 0.0)) for x in xg])
    assert np.all(lr <= l0 - xg * m + 1e-9) and np.all(lr <= l0 + 1e-12)


def test_mode_zero_is_the_round_one_model(orc, otables):
    """level_density = 0 with the correction arrays present: the Weisskopf-Ewing model of R-Q19, bit for bit."""
    t = orc.Tables(level_density=0, pair_Z=np.full(40, 1.5), pair_N=np.full(40, 1.5), shell_Z=np.full(40, 2.0), shell_N=np.full(40, 2.0))
    n = 1500
    E, tid = np.full(n, 200.0), np.zeros(n, dtype=np.int32)
    a = orc.simulate(t, [(16, 8)], E, tid, 1)
    b = orc.simulate(otables, [(16, 8)], E, tid, 1)
    for k in ("species", "T", "ux", "uy", "uz", "counts", "A", "Z", "Estar", "px", "py", "pz", "status"):
        assert np.array_equal(a[k], b[k]), k
    assert a["stats"] == b["stats"]


@pytest.mark.parametrize("A,Z,E,corr", [(16, 8, 200.0, False), (48, 22, 250.0, True)])
def test_gem_events_conserve_and_differ(orc, otables, A, Z, E, corr):
    """Whole events in GEM mode: the cascade is untouched (same post-cascade nuclei), conservation holds exactly,
    and the evaporation chain is a different one (the pre-exponential factor favours ... whatever it favours)."""
    from test_oracle_events import _check_conservation
    t = gem_tables(orc, pairing=corr, shells=corr)
    n = 3000
    Ein, tid = np.full(n, E), np.zeros(n, dtype=np.int32)
    g = orc.simulate(t, [(A, Z)], Ein, tid, 9)
    w = orc.simulate(otables, [(A, Z)], Ein, tid, 9)
    assert not np.any(g["status"] & orc.ST_FAILED)
    for k in ("casc_A", "casc_Z", "casc_Estar", "casc_count"):
        assert np.array_equal(g[k], w[k]), k
    _check_conservation(orc, t, g, A, Z, np.float64(E))
    assert not np.array_equal(g["counts"], w["counts"])
    assert g["stats"]["evap_steps"] > 0.5 * n and g["stats"]["cap_trial"] == 0
    # every chain ends with a nucleus that cannot emit: all widths zero at the final state
    L = orc.lib()
    for e in range(0, n, 97):
        assert _widths(orc, t, int(g["A"][e]), int(g["Z"][e]), float(g["Estar"][e]))[0] == 0.0


def test_gem_degenerate_inputs(orc):
    """DESIGN.md R-G7: caller inputs that leave no constant-temperature branch (1/T <= 0 with a > 0) close the channel;
    a pairing input below -U_x (E_x <= 0) puts the daughter on the Fermi-gas branch everywhere, and the width integral is
    int_0^X (x + beta) rho_FG(X - x) dx over [0, X] only -- checked against scipy.integrate.quad of that integrand."""
    L = orc.lib()
    sz = np.zeros(40); sz[6] = -13.0                       # a = A_d (0.125 - 0.1192) > 0, sqrt(a/U_x) < 1.5/U_x
    t = orc.Tables(level_density=1, shell_Z=sz)
    ld = orc.OrcLd()
    assert L.orc_gem_ld(12, 6, C.byref(t.c), C.byref(ld)) == -1
    a, Ux = 12 * (0.125 + 0.00917 * -13.0), 150.0 / 12 + 2.5
    assert a > 0 and np.sqrt(a / Ux) - 1.5 / Ux < 0
    assert L.orc_gem_ld(12, 5, C.byref(t.c), C.byref(ld)) == 0          # the neighbours are untouched
    tot, W, X = _widths(orc, t, 13, 6, 40.0)[:3]
    assert W[0] == 0.0 and X[0] < 0 and W[1] > 0.0                      # n (daughter 12,6) closed, p (daughter 12,5) open
    pz = np.zeros(40); pz[7] = -20.0                       # E_x = U_x - 20 < 0 for Z_d = 7
    t2 = orc.Tables(level_density=1, pair_Z=pz)
    ld = _ld(orc, t2, 15, 7)
    assert ld.Ex < 0
    for Xv, beta in ((0.1, 0.0), (3.0, 1.5), (25.0, -0.8), (60.0, 2.0)):
        f = lambda x: (x + beta) * np.exp(2 * np.sqrt(ld.a * (Xv - x - ld.delta)) - 0.25 * np.log(ld.a) - 1.25 * np.log(Xv - x - ld.delta))
        want = integrate.quad(f, 0.0, Xv, epsabs=0, epsrel=1e-12, limit=200)[0]
        assert L.orc_gem_integral(C.byref(ld), Xv, beta) == pytest.approx(want, rel=1e-9)
