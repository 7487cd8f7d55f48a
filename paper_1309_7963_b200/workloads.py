"""Seeded synthetic input generators for the five BASELINE.json configs.

Shared by the CUDA path, the tests and the oracle legs of bench.py.  Holds NONE of the
method's arithmetic: only (E_in[], target_id[], list of (A,Z), seed) per config, drawn
with numpy PCG64(seed) — independent of the Philox event streams.
The paper measures on no public dataset (fixed energy, single target); these
synthetic inputs ARE the paper's workload shape.
"""
from __future__ import annotations

import numpy as np

# id -> (n_events, E_lo, E_hi (MeV; equal = constant), [(A,Z)...], weights, seed)
CONFIGS = {
    1: dict(n=10**4, E=(200.0, 200.0), targets=[(16, 8)], weights=[1.0], seed=1,
            name="1e4 x 200 MeV p-16O"),
    2: dict(n=10**6, E=(200.0, 200.0), targets=[(16, 8)], weights=[1.0], seed=2,
            name="1e6 x 200 MeV p-16O (headline)"),
    3: dict(n=10**6, E=(20.0, 250.0), targets=[(40, 20)], weights=[1.0], seed=3,
            name="1e6 x U[20,250] MeV p-40Ca"),
    4: dict(n=10**7, E=(70.0, 250.0),
            targets=[(12, 6), (14, 7), (16, 8), (31, 15), (40, 20)],
            weights=[0.20, 0.04, 0.70, 0.02, 0.04], seed=4,
            name="1e7 x U[70,250] MeV mixed tissue/bone"),
    5: dict(n=10**6, E=(250.0, 250.0), targets=[(48, 22)], weights=[1.0], seed=5,
            name="1e6 x 250 MeV p-48Ti"),
}


def make_inputs(config_id: int, n: int | None = None):
    """Return (E_in float64[n], target_id int32[n], targets [(A,Z)], seed, name).

    target_id indexes `targets` (the caller maps it onto inc_init slots).  Energies and targets
    come from two independent streams of the config's seed, so a prefix of a config (n smaller
    than the config's) is the prefix of the full arrays and slices are consistent with full runs.
    """
    c = CONFIGS[config_id]
    n_full = c["n"]
    n = n_full if n is None else int(n)
    rng = np.random.Generator(np.random.PCG64(c["seed"]))
    lo, hi = c["E"]
    m = max(n, 0)
    if hi > lo:
        E = lo + (hi - lo) * rng.random(m)
    else:
        E = np.full(m, lo, dtype=np.float64)
    if len(c["targets"]) > 1:
        w = np.asarray(c["weights"], dtype=np.float64)
        cdf = np.cumsum(w / w.sum())
        rng_t = np.random.Generator(np.random.PCG64(np.random.SeedSequence(c["seed"], spawn_key=(1,))))
        tid = np.minimum(np.searchsorted(cdf, rng_t.random(m), side="right"), len(w) - 1).astype(np.int32)
    else:
        tid = np.zeros(m, dtype=np.int32)
    return E, tid, list(c["targets"]), c["seed"], c["name"]
