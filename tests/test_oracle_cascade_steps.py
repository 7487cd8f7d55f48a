"""Pins for the single cascade steps C2-C4: Fermi-sea partner, geometry,
relativistic two-body scatter, Pauli blocking rate vs brute force, potential step."""
import ctypes as C

import numpy as np
import pytest
from scipy import stats

DP = C.POINTER(C.c_double)


def _arr(v):
    return (C.c_double * len(v))(*[float(x) for x in v])


def _collide(L, p1, m1, p2, m2, B, a, same, ut, ub, uphi):
    o1, o2, ct = (C.c_double * 3)(), (C.c_double * 3)(), C.c_double()
    L.orc_collide(_arr(p1), m1, _arr(p2), m2, B, a, int(same), ut, ub, uphi, o1, o2, C.byref(ct))
    return np.array(o1[:]), np.array(o2[:]), ct.value


# ---------------------------------------------------------------- partner
def test_partner_is_fermi_gas(orc):
    """|p2|/pF has CDF x^3 ("quadratic distribution"), <p^2> = 3/5 pF^2, isotropic."""
    L = orc.lib()
    rng = np.random.default_rng(1)
    pF = 251.6
    n = 20000
    u = rng.random((n, 3))
    out = (C.c_double * 3)()
    P = np.empty((n, 3))
    for i in range(n):
        L.orc_partner(pF, u[i, 0], u[i, 1], u[i, 2], out)
        P[i] = out[:]
    mag = np.linalg.norm(P, axis=1)
    assert mag.max() <= pF
    assert stats.kstest(mag / pF, lambda x: np.clip(x, 0, 1) ** 3).pvalue > 1e-3
    assert np.mean(mag ** 2) == pytest.approx(0.6 * pF ** 2, rel=0.01)
    cosz = P[:, 2] / mag
    assert stats.kstest(cosz, "uniform", args=(-1, 2)).pvalue > 1e-3
    phi = np.arctan2(P[:, 1], P[:, 0]) % (2 * np.pi)
    assert stats.kstest(phi, "uniform", args=(0, 2 * np.pi)).pvalue > 1e-3
    # exact special values: u_mag = 1/8 -> |p| = pF/2 ; u_cos = 1 -> along +z
    L.orc_partner(pF, 0.125, 1.0, 0.3, out)
    assert np.allclose(out[:], [0, 0, pF / 2], atol=1e-9)


def test_plab_textbook_cases(orc):
    """Partner at rest: p_lab = |p1|.  Head-on equal momenta: closed form from s."""
    L = orc.lib()
    m = orc.M_P
    p1 = [30.0, -40.0, 500.0]
    assert L.orc_plab(_arr(p1), m, _arr([0, 0, 0]), orc.M_N) * 1000 == pytest.approx(np.linalg.norm(p1), rel=1e-12)
    # head-on, equal masses, momenta +-q: s = 4(q^2+m^2); T_lab = (s - 4m^2)/(2m) = 2q^2/m
    q = 300.0
    Tlab = 2 * q * q / m
    plab = np.sqrt(Tlab * (Tlab + 2 * m))
    assert L.orc_plab(_arr([0, 0, q]), m, _arr([0, 0, -q]), m) * 1000 == pytest.approx(plab, rel=1e-12)
    # symmetric in exchange for equal masses
    a, b = [10.0, 200.0, 50.0], [-70.0, 20.0, 100.0]
    assert L.orc_plab(_arr(a), m, _arr(b), m) == pytest.approx(L.orc_plab(_arr(b), m, _arr(a), m), rel=1e-12)


# ---------------------------------------------------------------- geometry
def test_shell_distances(orc):
    L = orc.lib()
    din, dout = C.c_double(), C.c_double()
    # centre-directed ray from r = 2.5 in shell [2,3]: hits inner sphere after 0.5
    L.orc_shell_distances(_arr([0, 0, 2.5]), _arr([0, 0, -1]), 2.0, 3.0, 1, C.byref(din), C.byref(dout))
    assert din.value == pytest.approx(0.5, rel=1e-14)
    assert dout.value == pytest.approx(5.5, rel=1e-14)   # far side of the outer sphere
    # outward radial ray: d_out = r_out - r, never hits the inner sphere
    L.orc_shell_distances(_arr([0, 2.5, 0]), _arr([0, 1, 0]), 2.0, 3.0, 1, C.byref(din), C.byref(dout))
    assert dout.value == pytest.approx(0.5, rel=1e-14) and np.isinf(din.value)
    # random rays: the end points lie on the spheres
    rng = np.random.default_rng(2)
    for _ in range(500):
        r = rng.uniform(2.0, 3.0)
        x = rng.normal(size=3); x *= r / np.linalg.norm(x)
        d = rng.normal(size=3); d /= np.linalg.norm(d)
        L.orc_shell_distances(_arr(x), _arr(d), 2.0, 3.0, 1, C.byref(din), C.byref(dout))
        assert dout.value > 0
        assert np.linalg.norm(x + dout.value * d) == pytest.approx(3.0, rel=1e-12)
        if np.isfinite(din.value):
            assert 0 < din.value < dout.value
            assert np.linalg.norm(x + din.value * d) == pytest.approx(2.0, rel=1e-12)
        else:
            # the ray misses the inner sphere: closest approach >= 2 or moving outward
            tca = -np.dot(x, d)
            assert tca <= 0 or np.linalg.norm(x + tca * d) >= 2.0 - 1e-12
    # on the outer sphere moving inward: far root, not 0
    x = np.array([0.0, 0.0, 3.0]); d = np.array([np.sin(0.3), 0, -np.cos(0.3)])
    L.orc_shell_distances(_arr(x), _arr(d), 2.0, 3.0, 0, C.byref(din), C.byref(dout))
    assert dout.value == pytest.approx(2 * 3.0 * np.cos(0.3), rel=1e-13) and np.isinf(din.value)


# ---------------------------------------------------------------- collision
def test_collision_conserves_four_momentum(orc):
    L = orc.lib()
    rng = np.random.default_rng(3)
    for _ in range(2000):
        m1, m2 = rng.choice([orc.M_P, orc.M_N], 2)
        p1 = rng.normal(size=3) * 300
        p2 = rng.normal(size=3) * 120
        B = rng.uniform(0, 8)
        a = rng.uniform(0, 1)
        same = bool(rng.integers(0, 2))
        q1, q2, ct = _collide(L, p1, m1, p2, m2, B, a, same, *rng.random(3))
        E_in = np.hypot(np.linalg.norm(p1), m1) + np.hypot(np.linalg.norm(p2), m2)
        E_out = np.hypot(np.linalg.norm(q1), m1) + np.hypot(np.linalg.norm(q2), m2)
        assert E_out == pytest.approx(E_in, rel=1e-12)
        assert np.allclose(q1 + q2, p1 + p2, rtol=0, atol=1e-9)
        # the invariant momentum transfer reproduces cos(theta_cm): t = (p1 - q1)^2
        E1, E1o = np.hypot(np.linalg.norm(p1), m1), np.hypot(np.linalg.norm(q1), m1)
        t = (E1 - E1o) ** 2 - np.sum((p1 - q1) ** 2)
        s = E_in ** 2 - np.sum((p1 + p2) ** 2)
        pcm2 = (s - (m1 + m2) ** 2) * (s - (m1 - m2) ** 2) / (4 * s)
        assert 1 + t / (2 * pcm2) == pytest.approx(ct, abs=1e-9)


def test_collision_angular_law(orc):
    """t = -2 pcm^2 (1 - cos) is distributed as exp(B t) on [tmin, 0] (analytic CDF);
    B = 0 is isotropic; the np backward branch mirrors cos with probability a/(1+a);
    azimuth uniform about the incoming CM direction."""
    L = orc.lib()
    rng = np.random.default_rng(4)
    m = orc.M_P
    p1, p2 = np.array([40.0, -30.0, 600.0]), np.array([100.0, 50.0, -80.0])
    n = 8000
    for B in (0.0, 3.0, 7.5):
        cts = np.empty(n)
        phis = np.empty(n)
        U = rng.random((n, 3))
        # CM frame quantities, independently
        E = np.hypot(np.linalg.norm(p1), m) + np.hypot(np.linalg.norm(p2), m)
        s = E ** 2 - np.sum((p1 + p2) ** 2)
        pcm2 = s / 4 - m * m
        for i in range(n):
            q1, q2, ct = _collide(L, p1, m, p2, m, B, 0.0, True, U[i, 0], 0.5, U[i, 2])
            cts[i] = ct
        tmin = -4 * pcm2 * 1e-6
        t = -2 * pcm2 * 1e-6 * (1 - cts)
        if B == 0.0:
            assert stats.kstest(cts, "uniform", args=(-1, 2)).pvalue > 1e-3
        else:
            cdf = lambda x: (np.exp(B * x) - np.exp(B * tmin)) / (1 - np.exp(B * tmin))
            assert stats.kstest(t, cdf).pvalue > 1e-3
            assert np.mean(cts) > 0   # forward peaked
    # backward term: fraction a/(1+a) of np events have cos -> -cos
    a = 0.6
    flips = 0
    for i in range(n):
        u = rng.random(3)
        _, _, c_np = _collide(L, p1, orc.M_P, p2, orc.M_N, 5.0, a, False, u[0], u[1], u[2])
        _, _, c_ref = _collide(L, p1, orc.M_P, p2, orc.M_N, 5.0, 0.0, False, u[0], u[1], u[2])
        assert abs(c_np) == pytest.approx(abs(c_ref), abs=1e-12)
        flips += (np.sign(c_np) != np.sign(c_ref))
    assert flips / n == pytest.approx(a / (1 + a), abs=4 * np.sqrt(0.25 / n))


def test_collision_forward_limit_and_azimuth(orc):
    L = orc.lib()
    m = orc.M_P
    p1, p2 = np.array([0.0, 0.0, 500.0]), np.array([0.0, 0.0, 0.0])
    # u_t -> 0 gives t = 0: no scattering at all
    q1, q2, ct = _collide(L, p1, m, p2, m, 4.0, 0.0, True, 1e-15, 0.5, 0.25)
    assert ct == pytest.approx(1.0, abs=1e-12)
    assert np.allclose(q1, p1, atol=1e-3) and np.allclose(q2, p2, atol=1e-3)
    # target at rest, equal masses: outgoing lab momenta are perpendicular-ish
    # (exactly: q1.q2 = (E1'-m)(E2'-m) for equal masses) and azimuth follows u_phi
    rng = np.random.default_rng(5)
    phis = []
    for _ in range(3000):
        u = rng.random(3)
        q1, q2, ct = _collide(L, p1, m, p2, m, 2.0, 0.0, True, u[0], 0.5, u[2])
        T1, T2 = np.hypot(np.linalg.norm(q1), m) - m, np.hypot(np.linalg.norm(q2), m) - m
        assert np.dot(q1, q2) == pytest.approx(T1 * T2, rel=1e-9, abs=1e-6)
        phis.append(np.arctan2(q1[1], q1[0]) % (2 * np.pi))
    assert stats.kstest(phis, "uniform", args=(0, 2 * np.pi)).pvalue > 1e-3


# ---------------------------------------------------------------- Pauli
from helpers import blocked_indicator_independent as _blocked_indicator_independent


@pytest.mark.parametrize("T1,B", [(60.0, 2.0), (150.0, 5.0)])
def test_pauli_blocking_rate_vs_brute_force(orc, otables, T1, B):
    """Blocked fraction from the oracle's collision routine (Monte Carlo over its own
    uniform inputs) against a deterministic 5-D midpoint quadrature of an independent
    scalar restatement of the kinematics, for a one-shell 'tiny nucleus'."""
    L = orc.lib()
    nu = orc.nucleus_arrays(orc.setup_nucleus(16, 8, otables))
    pF, EFp, EFn = nu["pF_n"][0], nu["EF_p"][0], nu["EF_n"][0]
    m1, m2 = orc.M_P, orc.M_N
    p1 = np.array([0, 0, np.sqrt(T1 * (T1 + 2 * m1))])
    rng = np.random.default_rng(6)
    n = 60000
    U = rng.random((n, 6))
    blocked = 0
    out = (C.c_double * 3)()
    for i in range(n):
        L.orc_partner(pF, U[i, 0], U[i, 1], U[i, 2], out)
        q1, q2, _ = _collide(L, p1, m1, np.array(out[:]), m2, B, 0.0, False, U[i, 3], 0.9, U[i, 4])
        T1o = np.hypot(np.linalg.norm(q1), m1) - m1
        T2o = np.hypot(np.linalg.norm(q2), m2) - m2
        blocked += not (T1o > EFp and T2o > EFn)
    frac_mc = blocked / n
    # quadrature: midpoints in (u_mag, u_cos, phi_k, u_t, phi)
    g = lambda k: (np.arange(k) + 0.5) / k
    umag, ucos, uphk, ut, uph = np.meshgrid(g(20), g(20), g(16), g(28), g(24), indexing="ij", sparse=True)
    ind = _blocked_indicator_independent(T1, m1, m2, pF, EFp, EFn, B, np.cbrt(umag), 2 * ucos - 1,
                                         2 * np.pi * uphk, ut, 2 * np.pi * uph)
    frac_q = np.mean(np.broadcast_to(ind, np.broadcast_shapes(umag.shape, ucos.shape, uphk.shape, ut.shape, uph.shape)))
    sigma = np.sqrt(frac_q * (1 - frac_q) / n)
    assert 0.05 < frac_q < 0.95
    assert abs(frac_mc - frac_q) < 3 * sigma + 4e-3, (frac_mc, frac_q)


# ---------------------------------------------------------------- boundary
def test_boundary_potential_step(orc):
    L = orc.lib()
    rng = np.random.default_rng(7)
    m = orc.M_N
    n_refl = n_refr = 0
    for _ in range(3000):
        x = rng.normal(size=3); x *= 3.0 / np.linalg.norm(x)
        p = rng.normal(size=3) * 150
        Vf, Vt = rng.uniform(0, 45, 2)
        nrm = x / 3.0
        pr = np.dot(p, nrm); pt = p - pr * nrm
        T = np.hypot(np.linalg.norm(p), m) - m
        pp = _arr(p); Tn = C.c_double()
        refl = L.orc_boundary(_arr(x), pp, m, Vf, Vt, C.byref(Tn))
        q = np.array(pp[:])
        qr = np.dot(q, nrm); qt = q - qr * nrm
        assert np.allclose(qt, pt, atol=1e-9)                    # tangential momentum conserved
        Tj = T + Vt - Vf
        should_reflect = Tj <= 0 or Tj * (Tj + 2 * m) - np.dot(pt, pt) <= 0
        assert bool(refl) == bool(should_reflect)
        if refl:
            n_refl += 1
            assert qr == pytest.approx(-pr, rel=1e-12)
            assert np.linalg.norm(q) == pytest.approx(np.linalg.norm(p), rel=1e-13)
            assert Tn.value == pytest.approx(T, rel=1e-12)
        else:
            n_refr += 1
            assert np.sign(qr) == np.sign(pr)
            assert Tn.value == pytest.approx(Tj, rel=1e-13)
            assert np.hypot(np.linalg.norm(q), m) - m == pytest.approx(Tj, rel=1e-10)   # energy step
    assert n_refl > 100 and n_refr > 100
    # Delta V = 0 is the identity
    x, p = [0.0, 3.0, 0.0], [10.0, 200.0, -50.0]
    pp = _arr(p)
    assert L.orc_boundary(_arr(x), pp, m, 20.0, 20.0, None) == 0
    assert np.allclose(pp[:], p, rtol=1e-13)
    # radial exit: |p| from T - V only
    pp = _arr([0.0, 300.0, 0.0])
    T = np.hypot(300.0, m) - m
    assert L.orc_boundary(_arr(x), pp, m, 30.0, 0.0, None) == 0
    assert pp[1] == pytest.approx(np.sqrt((T - 30) * (T - 30 + 2 * m)), rel=1e-13)
