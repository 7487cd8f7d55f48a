"""Writes tests/golden/oracle_config1_first64.json by calling ONLY oracle/ (plus the
seeded input generator, which holds no method arithmetic).  Run from the repo root:
    python tests/golden/make_golden.py
The stored values are the oracle's own (regression guard), never the CUDA path's.
"""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import oracle as O  # noqa: E402
import paper_1309_7963_b200.workloads as W  # noqa: E402

E, tid, targets, seed, name = W.make_inputs(1, 64)
r = O.simulate(O.Tables(), targets, E, tid, seed)
out = dict(source="oracle/inc_oracle.c via tests/golden/make_golden.py", config=name, seed=seed,
           counts=r["counts"].tolist(), A=r["A"].tolist(), Z=r["Z"].tolist(),
           species=r["species"].tolist(), T=[float(x) for x in r["T"]],
           Estar=[float(x) for x in r["Estar"]])
with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_config1_first64.json"), "w") as f:
    json.dump(out, f)
print("wrote", len(out["T"]), "secondaries of 64 events")
