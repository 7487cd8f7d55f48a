"""Default model-input tables for inc_init (the caller-supplied `inc_tables`).

The paper fixes the nuclear-model constants and names its NN input only by
citation ("parameterizations of Cugnon et al. [17]"; Dostrovsky [16] for the
evaporation barriers).  This module is the PRODUCT's table builder; the oracle has
its own, written separately (oracle/oracle.py) and tests compare the two.
Units: momentum GeV/c, cross sections mb, slopes (GeV/c)^-2.
"""
from __future__ import annotations

import numpy as np

N_XS = 1025
PLAB_MAX = 2.048            # GeV/c -> 2 MeV/c grid step
P_FLOOR = 0.1               # GeV/c: the low-momentum cross sections are held constant below this
WS_C0, WS_DELTA, WS_RPAD, N_SHELLS = 1.07, 0.545, 2.5, 15
SEMF = (15.75, 17.8, 0.711, 23.7, 11.18)                       # a_v a_s a_c a_a a_p, MeV
EVAP_R0, EVAP_RJ, EVAP_A_DIV = 1.5, 1.2, 8.0


def _piecewise(p, edges, funcs):
    out = np.empty_like(p)
    lo = -np.inf
    for hi, f in zip(list(edges) + [np.inf], funcs):
        m = (p >= lo) & (p < hi)
        out[m] = f(p[m])
        lo = hi
    return out


def nn_tables(n_xs: int = N_XS, plab_max: float = PLAB_MAX) -> dict:
    """Elastic NN cross sections and angular-distribution parameters on the p_lab grid."""
    p = np.arange(n_xs, dtype=np.float64) * (plab_max / (n_xs - 1))
    # low-momentum branches of ref. [17] below 0.44 (pp) / 0.45 (np) GeV/c, where they meet the next branch to
    # ~1 %; both diverge for p -> 0, so knots below P_FLOOR carry the value at P_FLOOR (T_lab ~ 5 MeV)
    sig_pp = _piecewise(p, [0.44, 0.8, 2.0], [
        lambda q: 34.0 * (np.maximum(q, P_FLOOR) / 0.4) ** -2.104,
        lambda q: 23.5 + 1000.0 * (q - 0.7) ** 4,
        lambda q: 1250.0 / (q + 50.0) - 4.0 * (q - 1.3) ** 2,
        lambda q: 77.0 / (q + 1.5)])
    sig_np = _piecewise(p, [0.45, 0.8, 2.0], [
        lambda q: 6.3555 * np.maximum(q, P_FLOOR) ** -3.2481 * np.exp(-0.377 * np.log(np.maximum(q, P_FLOOR)) ** 2),
        lambda q: 33.0 + 196.0 * np.abs(q - 0.95) ** 2.5,
        lambda q: 31.0 / np.sqrt(q),
        lambda q: 77.0 / (q + 1.5)])
    b_pp_lo = lambda q: 5.5 * q ** 8 / (7.7 + q ** 8)
    b_pp_hi = lambda q: 5.334 + 0.67 * (q - 2.0)
    B_pp = _piecewise(p, [2.0], [b_pp_lo, b_pp_hi])
    B_np = _piecewise(p, [0.225, 0.6, 1.6, 2.0], [
        lambda q: np.zeros_like(q),
        lambda q: 16.53 * (q - 0.225),
        lambda q: -1.63 * q + 7.16,
        b_pp_lo, b_pp_hi])
    a_np = _piecewise(p, [0.8], [lambda q: np.ones_like(q), lambda q: 0.64 / (q * q)])
    return dict(plab=p, sig_pp=sig_pp, sig_np=sig_np, B_pp=B_pp, B_np=B_np, a_np=a_np)


def evap_tables() -> dict:
    """Dostrovsky et al. Coulomb-barrier (k) and inverse-cross-section (c) parameters."""
    return dict(ev_Z=np.array([10.0, 20.0, 30.0, 50.0, 70.0]),
                ev_kp=np.array([0.42, 0.58, 0.68, 0.77, 0.80]),
                ev_cp=np.array([0.50, 0.28, 0.20, 0.15, 0.10]),
                ev_ka=np.array([0.68, 0.82, 0.91, 0.97, 0.98]),
                ev_ca=np.array([0.10, 0.10, 0.10, 0.08, 0.06]))


def default_tables(**overrides) -> dict:
    """Everything inc_init needs, as a plain dict (see binding.IncTables)."""
    t = dict(version=2, n_xs=N_XS, plab_max=PLAB_MAX, n_shells=N_SHELLS,
             ws_c0=WS_C0, ws_delta=WS_DELTA, ws_rpad=WS_RPAD, semf=SEMF,
             evap_r0=EVAP_R0, evap_rj=EVAP_RJ, evap_a_div=EVAP_A_DIV,
             # level density of the evaporation stage (inc.h, version 2 block): 0 = the frozen Weisskopf-Ewing model;
             # 1 = GEM level density with the caller's pairing energies and shell corrections (none by default)
             level_density=0, pair_Z=None, pair_N=None, shell_Z=None, shell_N=None, gc_a0=0.125, gc_a1=0.00917)
    t.update(nn_tables(t["n_xs"], t["plab_max"]))
    t.update(evap_tables())
    t.update(overrides)
    return t
