"""ctypes front-end of the CPU fp64 oracle (oracle/inc_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  Never imported by paper_1309_7963_b200.

Also holds the oracle's OWN restatement of the model-input tables (Cugnon NN
parameterisations, P:49 ref. [17]; Dostrovsky k/c, P:173 ref. [16]) — written
independently of paper_1309_7963_b200/tables.py; tests compare the two.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# INC_ORACLE_SRC / INC_ORACLE_LIB: tests/test_pins_bite.py points them at a deliberately broken copy of the
# oracle to prove that the pins notice it
_SRC = os.environ.get("INC_ORACLE_SRC", os.path.join(_HERE, "inc_oracle.c"))
_LIB = os.environ.get("INC_ORACLE_LIB", os.path.join(_HERE, "libinc_oracle.so"))

MAX_SHELLS = 32
MAX_SEC = 64

ST_FAILED = 1 << 8
ST_SEC_TRUNC = 1 << 9
ST_DEPTH_CAP = 1 << 10
ST_SEG_CAP = 1 << 11
ST_TRIAL_CAP = 1 << 12

F_CASCADE_ONLY = 1
F_KEEP_TRANSPARENT = 2
F_FIFO = 4

M_P = 938.27208816
M_N = 939.56542052
SPECIES_A = np.array([1, 1, 2, 3, 3, 4])
SPECIES_Z = np.array([0, 1, 1, 1, 2, 2])
LIGHT_B = np.array([0.0, 0.0, 2.224566, 8.481798, 7.718043, 28.29566])
SPECIES_M = SPECIES_Z * M_P + (SPECIES_A - SPECIES_Z) * M_N - LIGHT_B


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 -ffp-contract=off (no fast-math)."""
    hdr = os.path.join(_HERE, "inc_oracle.h")
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= max(os.path.getmtime(_SRC), os.path.getmtime(hdr))):
        return _LIB
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC",
           "-I", _HERE, "-o", _LIB, _SRC, "-lm"]
    subprocess.check_call(cmd)
    return _LIB


class OrcTables(C.Structure):
    _fields_ = [
        ("version", C.c_int32), ("n_xs", C.c_int32), ("plab_max", C.c_double),
        ("sig_pp", C.POINTER(C.c_double)), ("sig_np", C.POINTER(C.c_double)),
        ("B_pp", C.POINTER(C.c_double)), ("B_np", C.POINTER(C.c_double)),
        ("a_np", C.POINTER(C.c_double)),
        ("n_evz", C.c_int32),
        ("ev_Z", C.POINTER(C.c_double)), ("ev_kp", C.POINTER(C.c_double)),
        ("ev_cp", C.POINTER(C.c_double)), ("ev_ka", C.POINTER(C.c_double)),
        ("ev_ca", C.POINTER(C.c_double)),
        ("ws_c0", C.c_double), ("ws_delta", C.c_double), ("ws_rpad", C.c_double),
        ("n_shells", C.c_int32),
        ("semf", C.c_double * 5),
        ("evap_r0", C.c_double), ("evap_rj", C.c_double), ("evap_a_div", C.c_double),
        ("level_density", C.c_int32), ("n_ldZ", C.c_int32), ("n_ldN", C.c_int32),
        ("pair_Z", C.POINTER(C.c_double)), ("pair_N", C.POINTER(C.c_double)),
        ("shell_Z", C.POINTER(C.c_double)), ("shell_N", C.POINTER(C.c_double)),
        ("gc_a0", C.c_double), ("gc_a1", C.c_double),
    ]


class OrcLd(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("a", "delta", "Ux", "Ex", "T", "E0")]


class OrcNucleus(C.Structure):
    _fields_ = [
        ("A", C.c_int32), ("Z", C.c_int32), ("n_shells", C.c_int32),
        ("c", C.c_double), ("R", C.c_double), ("delta_r", C.c_double),
        ("r", C.c_double * (MAX_SHELLS + 1)),
        ("rho", C.c_double * MAX_SHELLS),
        ("rho_p", C.c_double * MAX_SHELLS), ("rho_n", C.c_double * MAX_SHELLS),
        ("pF_p", C.c_double * MAX_SHELLS), ("pF_n", C.c_double * MAX_SHELLS),
        ("EF_p", C.c_double * MAX_SHELLS), ("EF_n", C.c_double * MAX_SHELLS),
        ("V_p", C.c_double * (MAX_SHELLS + 1)), ("V_n", C.c_double * (MAX_SHELLS + 1)),
        ("EB_p", C.c_double), ("EB_n", C.c_double), ("EC", C.c_double), ("M", C.c_double),
    ]


_STAT_FIELDS = ["events", "failed", "attempts", "retry_transparent", "retry_invalid",
                "retry_estar", "segments", "boundaries", "reflections", "escapes",
                "collisions", "blocked", "allowed", "absorbed", "evap_steps", "evap_trials",
                "evap_emitted", "cap_seg", "cap_depth", "cap_sec", "cap_trial", "philox_blocks"]


class OrcCollRec(C.Structure):
    _fields_ = [("pi", C.c_uint32), ("k", C.c_uint32), ("shell", C.c_int32), ("type1", C.c_int32), ("type2", C.c_int32),
                ("blocked", C.c_int32), ("keep1", C.c_int32), ("keep2", C.c_int32),
                ("T_in", C.c_double), ("plab", C.c_double), ("B", C.c_double), ("a_back", C.c_double),
                ("Sp", C.c_double), ("Sigma", C.c_double), ("T1", C.c_double), ("T2", C.c_double), ("costheta", C.c_double)]


COLL_DTYPE = np.dtype([(n, np.uint32 if t is C.c_uint32 else np.int32 if t is C.c_int32 else np.float64)
                       for n, t in OrcCollRec._fields_], align=True)


class OrcStats(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in _STAT_FIELDS]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n in _STAT_FIELDS}


_lib = None


def lib():
    global _lib
    if _lib is not None:
        return _lib
    build()
    L = C.CDLL(_LIB)
    dp = C.POINTER(C.c_double)
    L.orc_setup_nucleus.argtypes = [C.c_int, C.c_int, C.POINTER(OrcTables), C.POINTER(OrcNucleus)]
    L.orc_setup_nucleus.restype = C.c_int
    L.orc_simulate.restype = C.c_int64
    L.orc_simulate.argtypes = [
        C.POINTER(OrcTables), C.POINTER(OrcNucleus), C.c_int, C.c_int64, C.c_int64,
        C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32,
        C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p,
        C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
        C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(OrcStats), C.c_void_p]
    L.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
    L.orc_philox4x32_10.restype = None
    L.orc_u01.argtypes = [C.c_uint32]
    L.orc_u01.restype = C.c_double
    L.orc_valid_nucleus.argtypes = [C.c_int, C.c_int]
    L.orc_valid_nucleus.restype = C.c_int
    L.orc_binding.argtypes = [C.c_int, C.c_int, C.POINTER(OrcTables)]
    L.orc_binding.restype = C.c_double
    L.orc_mass.argtypes = [C.c_int, C.c_int, C.POINTER(OrcTables)]
    L.orc_mass.restype = C.c_double
    L.orc_lerp_table.argtypes = [dp, C.c_int, C.c_double, C.c_double]
    L.orc_lerp_table.restype = C.c_double
    L.orc_partner.argtypes = [C.c_double] * 4 + [dp]
    L.orc_partner.restype = None
    L.orc_plab.argtypes = [dp, C.c_double, dp, C.c_double]
    L.orc_plab.restype = C.c_double
    L.orc_shell_distances.argtypes = [dp, dp, C.c_double, C.c_double, C.c_int, dp, dp]
    L.orc_shell_distances.restype = None
    L.orc_collide.argtypes = [dp, C.c_double, dp, C.c_double, C.c_double, C.c_double, C.c_int,
                              C.c_double, C.c_double, C.c_double, dp, dp, dp]
    L.orc_collide.restype = None
    L.orc_boundary.argtypes = [dp, dp, C.c_double, C.c_double, C.c_double, dp]
    L.orc_boundary.restype = C.c_int
    L.orc_evap_widths.argtypes = [C.c_int, C.c_int, C.c_double, C.POINTER(OrcTables)] + [dp] * 6
    L.orc_evap_widths.restype = C.c_double
    L.orc_evap_sample_x.argtypes = [C.c_double, C.c_double, C.c_double, C.POINTER(C.c_uint32),
                                    C.c_uint32, C.c_uint32, C.c_uint32,
                                    C.POINTER(C.c_uint32), C.POINTER(C.c_int)]
    L.orc_evap_sample_x.restype = C.c_double
    L.orc_evap_emit.argtypes = [C.c_int, C.c_int, C.c_double, dp, C.c_int, C.c_double, C.c_double,
                                C.c_double, C.c_double, C.POINTER(OrcTables), dp, dp, dp]
    L.orc_evap_emit.restype = None
    L.orc_gem_ld.argtypes = [C.c_int, C.c_int, C.POINTER(OrcTables), C.POINTER(OrcLd)]
    L.orc_gem_ld.restype = C.c_int
    L.orc_gem_lnrho.argtypes = [C.POINTER(OrcLd), C.c_double]
    L.orc_gem_lnrho.restype = C.c_double
    L.orc_gem_integral.argtypes = [C.POINTER(OrcLd), C.c_double, C.c_double]
    L.orc_gem_integral.restype = C.c_double
    L.orc_evap_sample_x_gem.argtypes = [C.POINTER(OrcLd), C.c_double, C.c_double, C.POINTER(C.c_uint32),
                                        C.c_uint32, C.c_uint32, C.c_uint32, C.POINTER(C.c_uint32), C.POINTER(C.c_int)]
    L.orc_evap_sample_x_gem.restype = C.c_double
    L.orc_lerp_z.argtypes = [dp, dp, C.c_int, C.c_double]
    L.orc_lerp_z.restype = C.c_double
    L.orc_evap_choose.argtypes = [dp, C.c_double, C.c_double]
    L.orc_evap_choose.restype = C.c_int
    L.orc_cascade_trace.argtypes = [C.POINTER(OrcTables), C.POINTER(OrcNucleus), C.c_uint64, C.c_uint64, C.c_uint32,
                                    C.c_double, C.c_int, C.c_uint32, C.c_int, C.c_void_p, C.POINTER(C.c_int),
                                    C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_int),
                                    C.POINTER(C.c_uint32)]
    L.orc_cascade_trace.restype = C.c_int
    _lib = L
    return L


# ----------------------------------------------------------------------------------
# Oracle's own model-input tables (R-T in DESIGN.md).  p in GeV/c, sigma in mb.
# ----------------------------------------------------------------------------------
SIGMA_P_FLOOR = 0.1   # GeV/c; the p -> 0 divergence of the lowest branches is cut here (R-T)


def cugnon_sigma_pp(p):
    p = np.asarray(p, dtype=np.float64)
    pc = np.clip(p, SIGMA_P_FLOOR, None)
    vlo = 34.0 * (pc / 0.4) ** (-2.104)                       # p < 0.44
    lo = 23.5 + 1000.0 * (p - 0.7) ** 4                       # 0.44 <= p < 0.8
    mid = 1250.0 / (p + 50.0) - 4.0 * (p - 1.3) ** 2
    hi = 77.0 / (p + 1.5)
    return np.where(p < 0.44, vlo, np.where(p < 0.8, lo, np.where(p < 2.0, mid, hi)))


def cugnon_sigma_np(p):
    p = np.asarray(p, dtype=np.float64)
    pc = np.clip(p, SIGMA_P_FLOOR, None)
    vlo = 6.3555 * pc ** (-3.2481) * np.exp(-0.377 * np.log(pc) ** 2)   # p < 0.45
    lo = 33.0 + 196.0 * np.abs(p - 0.95) ** 2.5                         # 0.45 <= p < 0.8
    mid = 31.0 / np.sqrt(np.maximum(p, 0.8))
    hi = 77.0 / (p + 1.5)
    return np.where(p < 0.45, vlo, np.where(p < 0.8, lo, np.where(p < 2.0, mid, hi)))


def cugnon_B_pp(p):
    p = np.asarray(p, dtype=np.float64)
    p8 = p ** 8
    return np.where(p < 2.0, 5.5 * p8 / (7.7 + p8), 5.334 + 0.67 * (p - 2.0))


def cugnon_B_np(p):
    p = np.asarray(p, dtype=np.float64)
    return np.where(p < 0.225, 0.0,
                    np.where(p < 0.6, 16.53 * (p - 0.225),
                             np.where(p < 1.6, -1.63 * p + 7.16, cugnon_B_pp(p))))


def cugnon_a_np(p):
    p = np.asarray(p, dtype=np.float64)
    return np.where(p < 0.8, 1.0, 0.64 / np.maximum(p, 0.8) ** 2)


class Tables:
    """Holds the numpy arrays alive and exposes the ctypes struct."""

    def __init__(self, n_xs=1025, plab_max=2.048, n_shells=15, semf=(15.75, 17.8, 0.711, 23.7, 11.18),
                 ws=(1.07, 0.545, 2.5), evap=(1.5, 1.2, 8.0), sigma_scale=1.0, B_scale=1.0,
                 level_density=0, pair_Z=None, pair_N=None, shell_Z=None, shell_N=None, gc=(0.125, 0.00917)):
        p = np.arange(n_xs, dtype=np.float64) * (plab_max / (n_xs - 1))
        self.plab = p
        self.sig_pp = np.ascontiguousarray(cugnon_sigma_pp(p) * sigma_scale)
        self.sig_np = np.ascontiguousarray(cugnon_sigma_np(p) * sigma_scale)
        self.B_pp = np.ascontiguousarray(cugnon_B_pp(p) * B_scale)
        self.B_np = np.ascontiguousarray(cugnon_B_np(p) * B_scale)
        self.a_np = np.ascontiguousarray(cugnon_a_np(p))
        self.ev_Z = np.array([10.0, 20.0, 30.0, 50.0, 70.0])
        self.ev_kp = np.array([0.42, 0.58, 0.68, 0.77, 0.80])
        self.ev_cp = np.array([0.50, 0.28, 0.20, 0.15, 0.10])
        self.ev_ka = np.array([0.68, 0.82, 0.91, 0.97, 0.98])
        self.ev_ca = np.array([0.10, 0.10, 0.10, 0.08, 0.06])
        self.n_xs, self.plab_max, self.n_shells = n_xs, plab_max, n_shells
        self.semf, self.ws, self.evap = tuple(semf), tuple(ws), tuple(evap)
        # NEXT-2 (version 2 block): level-density mode and the caller-supplied pairing / shell-correction arrays
        self.level_density, self.gc = int(level_density), tuple(gc)
        nz = max(len(x) for x in (pair_Z, shell_Z) if x is not None) if (pair_Z is not None or shell_Z is not None) else 1
        nn = max(len(x) for x in (pair_N, shell_N) if x is not None) if (pair_N is not None or shell_N is not None) else 1
        pad = lambda x, n: np.concatenate([np.asarray(x, dtype=np.float64), np.zeros(n - len(x))]) if x is not None else np.zeros(n)
        self.pair_Z, self.shell_Z = pad(pair_Z, nz), pad(shell_Z, nz)
        self.pair_N, self.shell_N = pad(pair_N, nn), pad(shell_N, nn)
        self.refresh()

    def refresh(self):
        dp = C.POINTER(C.c_double)
        s = OrcTables()
        s.version = 2
        s.n_xs = self.n_xs
        s.plab_max = self.plab_max
        for name in ("sig_pp", "sig_np", "B_pp", "B_np", "a_np", "ev_Z", "ev_kp", "ev_cp", "ev_ka", "ev_ca",
                     "pair_Z", "pair_N", "shell_Z", "shell_N"):
            arr = np.ascontiguousarray(getattr(self, name), dtype=np.float64)
            setattr(self, name, arr)
            setattr(s, name, arr.ctypes.data_as(dp))
        s.n_evz = len(self.ev_Z)
        s.ws_c0, s.ws_delta, s.ws_rpad = self.ws
        s.n_shells = self.n_shells
        for i in range(5):
            s.semf[i] = self.semf[i]
        s.evap_r0, s.evap_rj, s.evap_a_div = self.evap
        s.level_density, s.n_ldZ, s.n_ldN = self.level_density, len(self.pair_Z), len(self.pair_N)
        assert len(self.shell_Z) == len(self.pair_Z) and len(self.shell_N) == len(self.pair_N)
        s.gc_a0, s.gc_a1 = self.gc
        self.c = s
        return self


def setup_nucleus(A, Z, tables: Tables) -> OrcNucleus:
    nu = OrcNucleus()
    rc = lib().orc_setup_nucleus(int(A), int(Z), C.byref(tables.c), C.byref(nu))
    if rc != 0:
        raise ValueError(f"orc_setup_nucleus({A},{Z}) -> {rc}")
    return nu


def nucleus_arrays(nu: OrcNucleus) -> dict:
    ns = nu.n_shells
    out = {k: getattr(nu, k) for k in ("A", "Z", "n_shells", "c", "R", "delta_r", "EB_p", "EB_n", "EC", "M")}
    for k in ("rho", "rho_p", "rho_n", "pF_p", "pF_n", "EF_p", "EF_n"):
        out[k] = np.array(getattr(nu, k)[:ns])
    for k in ("r", "V_p", "V_n"):
        out[k] = np.array(getattr(nu, k)[:ns + 1])
    return out


def simulate(tables: Tables, nuclei, E_in, target, seed, e0=0, flags=0, want_stats=True, projectile=None):
    """Run the oracle on events e0..e0+n-1.  nuclei: list of (A,Z) or OrcNucleus.
    projectile: None (protons, the paper's case) or per-event uint8 array, 0 = neutron, 1 = proton (NEXT-3)."""
    L = lib()
    nus = (OrcNucleus * len(nuclei))()
    for i, nz in enumerate(nuclei):
        nus[i] = nz if isinstance(nz, OrcNucleus) else setup_nucleus(nz[0], nz[1], tables)
    E_in = np.ascontiguousarray(E_in, dtype=np.float64)
    if projectile is not None:
        projectile = np.ascontiguousarray(projectile, dtype=np.uint8)
        assert len(projectile) == len(E_in)
    target = np.ascontiguousarray(target, dtype=np.int32)
    n = len(E_in)
    cap = n * MAX_SEC
    cap = min(cap, max(64, n * 24))
    while True:
        sp = np.zeros(cap, dtype=np.uint8)
        T = np.zeros(cap); ux = np.zeros(cap); uy = np.zeros(cap); uz = np.zeros(cap)
        counts = np.zeros(n, dtype=np.int32)
        rA = np.zeros(n, dtype=np.int32); rZ = np.zeros(n, dtype=np.int32)
        rE = np.zeros(n); rpx = np.zeros(n); rpy = np.zeros(n); rpz = np.zeros(n)
        status = np.zeros(n, dtype=np.uint32)
        cA = np.zeros(n, dtype=np.int32); cZ = np.zeros(n, dtype=np.int32)
        cE = np.zeros(n); cP = np.zeros((n, 3)); cN = np.zeros(n, dtype=np.int32)
        st = OrcStats()
        vp = lambda a: a.ctypes.data_as(C.c_void_p)
        tot = L.orc_simulate(C.byref(tables.c), nus, len(nuclei), int(e0), int(n), vp(E_in), vp(target),
                             C.c_uint64(int(seed)), C.c_uint32(int(flags)),
                             vp(sp), vp(T), vp(ux), vp(uy), vp(uz), int(cap), vp(counts),
                             vp(rA), vp(rZ), vp(rE), vp(rpx), vp(rpy), vp(rpz), vp(status),
                             vp(cA), vp(cZ), vp(cE), vp(cP), vp(cN), C.byref(st),
                             None if projectile is None else vp(projectile))
        if tot == -3 and cap < n * MAX_SEC:
            cap = n * MAX_SEC
            continue
        break
    if tot < 0:
        raise RuntimeError(f"orc_simulate -> {tot}")
    offsets = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(counts, out=offsets[1:])
    return dict(species=sp[:tot], T=T[:tot], ux=ux[:tot], uy=uy[:tot], uz=uz[:tot], counts=counts,
                offsets=offsets, A=rA, Z=rZ, Estar=rE, px=rpx, py=rpy, pz=rpz, status=status,
                casc_A=cA, casc_Z=cZ, casc_Estar=cE, casc_P=cP, casc_count=cN,
                stats=st.as_dict() if want_stats else None, total=int(tot))


def cascade_trace(tables: Tables, nucleus, seed, event, attempt, E_in, proj=1, flags=0, cap_coll=512):
    """One cascade attempt of one event with its collision log (numpy structured array, COLL_DTYPE) and its
    escaped particles in ascending path code.  nucleus: (A, Z) or OrcNucleus."""
    assert C.sizeof(OrcCollRec) == COLL_DTYPE.itemsize
    nu = nucleus if isinstance(nucleus, OrcNucleus) else setup_nucleus(nucleus[0], nucleus[1], tables)
    coll = np.zeros(cap_coll, dtype=COLL_DTYPE)
    pi = np.zeros(MAX_SEC, dtype=np.uint32); typ = np.zeros(MAX_SEC, dtype=np.int32)
    T = np.zeros(MAX_SEC); p = np.zeros((MAX_SEC, 3))
    nc, ne, st = C.c_int(0), C.c_int(0), C.c_uint32(0)
    vp = lambda a: a.ctypes.data_as(C.c_void_p)
    n_real = lib().orc_cascade_trace(C.byref(tables.c), C.byref(nu), C.c_uint64(int(seed)), C.c_uint64(int(event)),
                                     C.c_uint32(int(attempt)), float(E_in), int(proj), C.c_uint32(int(flags)), cap_coll,
                                     vp(coll), C.byref(nc), vp(pi), vp(typ), vp(T), vp(p), C.byref(ne), C.byref(st))
    if n_real < 0:
        raise ValueError("orc_cascade_trace: bad arguments")
    assert nc.value <= cap_coll, "collision log truncated: raise cap_coll"
    k = ne.value
    return dict(n_real=n_real, coll=coll[:nc.value], esc_pi=pi[:k], esc_type=typ[:k], esc_T=T[:k], esc_p=p[:k], status=st.value)


def tally_reference(species, T, uz, counts, A_res, Z_res, n_T=50, T_max=250.0, n_cos=20, mult_max=24,
                    A_max=72, Z_max=36, real=np.float64):
    """The tallies of include/inc.h `inc_tally` written out as the
    plain definition: histograms over the outputs of a simulate call.  Classes 0 = n, 1 = p, 2 = composites.
    `real` is the precision in which the two bin coordinates are formed (one rounding per operation, as the
    library does): np.float64 for the parity build and the oracle, np.float32 for the production build."""
    species = np.asarray(species); counts = np.asarray(counts)
    code = (species & 0x7).astype(np.int64)
    origin = (species >> 7).astype(np.int64)
    cls = np.minimum(code, 2)
    cos_scale = real(n_cos / 2.0)
    T_scale = real(n_T / T_max)
    a = ((np.asarray(uz, dtype=real) + real(1)) * cos_scale).astype(np.int64)      # truncation, like the (int) cast
    a = np.clip(a, 0, n_cos - 1)
    tt = np.asarray(T, dtype=real) * T_scale
    t = np.where(tt >= real(n_T), n_T, tt.astype(np.int64))
    t = np.maximum(t, 0)
    dd = np.zeros((3, n_cos, n_T + 1), dtype=np.int64)
    np.add.at(dd, (cls, a, t), 1)
    n = len(counts)
    ev = np.repeat(np.arange(n), counts)
    mult = np.zeros((4, mult_max + 1), dtype=np.int64)
    for c in range(3):
        m = np.bincount(ev[cls == c], minlength=n)
        mult[c] = np.bincount(np.minimum(m, mult_max), minlength=mult_max + 1)
    mult[3] = np.bincount(np.minimum(counts, mult_max), minlength=mult_max + 1)
    nuclide = np.zeros((A_max + 1, Z_max + 1), dtype=np.int64)
    A_res = np.asarray(A_res); Z_res = np.asarray(Z_res)
    ok = (A_res >= 0) & (A_res <= A_max) & (Z_res >= 0) & (Z_res <= Z_max)
    np.add.at(nuclide, (A_res[ok], Z_res[ok]), 1)
    yields = np.zeros((6, 2), dtype=np.int64)
    ok6 = code < 6
    np.add.at(yields, (code[ok6], origin[ok6]), 1)
    return dict(dd=dd, mult=mult, nuclide=nuclide, yields=yields)
