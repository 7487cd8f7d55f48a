"""CPU tests (`-m "not gpu"`): the C-ABI library loads and exports every symbol include/inc.h
declares, the ctypes structs match the C layout, product tables equal the oracle's own,
workload generators, sharding (world_size-2 gloo), and the statistics helpers."""
import ctypes as C
import os
import re
import subprocess
import sys
import tempfile

import numpy as np
import pytest

import helpers as H

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    import paper_1309_7963_b200.binding as B
    hdr = open(os.path.join(ROOT, "include", "inc.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(inc_[a-z_0-9]+)\s*\(", hdr))
    assert {"inc_init", "inc_simulate", "inc_simulate_host", "inc_get_offsets"} <= declared
    for variant in ("f32", "f64", "f64q"):
        lib = B.load(variant)
        for name in sorted(declared):
            assert hasattr(lib.lib, name), (variant, name)
        assert variant[:3] in lib.build_info()
    assert declared == set(B.EXPORTS)


def test_ctypes_structs_match_c_layout():
    """Compile a probe against include/inc.h with gcc and compare sizeof/offsetof."""
    import paper_1309_7963_b200.binding as B
    src = r'''
#include <stdio.h>
#include <stddef.h>
#include "inc.h"
int main(void){
 printf("%zu %zu %zu %zu %zu %zu\n", sizeof(inc_tables), offsetof(inc_tables, n_evz), offsetof(inc_tables, ws_c0),
        offsetof(inc_tables, semf), offsetof(inc_tables, evap_a_div), offsetof(inc_tables, plab_max));
 printf("%zu %zu %zu %zu\n", sizeof(inc_secondaries), offsetof(inc_secondaries, capacity), sizeof(inc_residual), sizeof(inc_stats));
 return 0; }'''
    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "probe.c"); exe = os.path.join(d, "probe")
        open(c, "w").write(src)
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), c, "-o", exe])
        a, b = subprocess.check_output([exe]).decode().split("\n")[:2]
    a = [int(x) for x in a.split()]; b = [int(x) for x in b.split()]
    T = B.IncTables
    assert a == [C.sizeof(T), T.n_evz.offset, T.ws_c0.offset, T.semf.offset, T.evap_a_div.offset, T.plab_max.offset]
    assert b == [C.sizeof(B.IncSecondaries), B.IncSecondaries.capacity.offset, C.sizeof(B.IncResidual), C.sizeof(B.IncStats)]


def test_no_cpu_fallback():
    """Without a CUDA device the product fails loudly (INC_E_CUDA), it never computes on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_1309_7963_b200.binding as B
    import paper_1309_7963_b200.tables as T
    lib = B.load("f32")
    with pytest.raises(B.IncError) as ei:
        lib.inc_init(16, 8, T.default_tables())
    assert ei.value.code == B.INC_E_CUDA
    # the product package never imports the oracle
    for f in os.listdir(os.path.join(ROOT, "paper_1309_7963_b200")):
        if f.endswith(".py"):
            txt = open(os.path.join(ROOT, "paper_1309_7963_b200", f)).read()
            assert "import oracle" not in txt and "from oracle" not in txt, f


def test_product_tables_equal_oracle_tables(orc, otables):
    """Two independently written generators of the model inputs agree (DESIGN.md R-T)."""
    import paper_1309_7963_b200.tables as T
    t = T.default_tables()
    for k in ("sig_pp", "sig_np", "B_pp", "B_np", "a_np", "ev_Z", "ev_kp", "ev_cp", "ev_ka", "ev_ca"):
        assert np.allclose(t[k], getattr(otables, k), rtol=1e-13, atol=0), k
    assert t["n_xs"] == otables.n_xs and t["plab_max"] == otables.plab_max and t["n_shells"] == otables.n_shells
    assert tuple(t["semf"]) == tuple(otables.semf)
    assert (t["ws_c0"], t["ws_delta"], t["ws_rpad"]) == tuple(otables.ws)
    assert (t["evap_r0"], t["evap_rj"], t["evap_a_div"]) == tuple(otables.evap)


def test_workloads_match_baseline_configs():
    import paper_1309_7963_b200.workloads as W
    assert [W.CONFIGS[i]["n"] for i in (1, 2, 3, 4, 5)] == [10**4, 10**6, 10**6, 10**7, 10**6]
    E, tid, targets, seed, _ = W.make_inputs(2, 1000)
    assert np.all(E == 200.0) and targets == [(16, 8)] and seed == 2 and np.all(tid == 0)
    E, tid, targets, seed, _ = W.make_inputs(3, 50000)
    assert targets == [(40, 20)] and 20.0 <= E.min() and E.max() < 250.0 and abs(E.mean() - 135.0) < 1.5
    E, tid, targets, seed, _ = W.make_inputs(4, 200000)
    frac = np.bincount(tid, minlength=5) / len(tid)
    assert np.allclose(frac, [0.20, 0.04, 0.70, 0.02, 0.04], atol=0.004)
    assert targets == [(12, 6), (14, 7), (16, 8), (31, 15), (40, 20)] and E.min() >= 70.0
    E5, _, targets5, _, _ = W.make_inputs(5, 10)
    assert np.all(E5 == 250.0) and targets5 == [(48, 22)]
    # deterministic, and a shorter request is a prefix of a longer one
    Ea, ta, *_ = W.make_inputs(4, 5000)
    Eb, tb, *_ = W.make_inputs(4, 100)
    assert np.array_equal(Ea[:100], Eb) and np.array_equal(ta[:100], tb) and len(np.unique(ta[:100])) > 1
    Ec, tc, *_ = W.make_inputs(4, 5000)
    assert np.array_equal(Ea, Ec) and np.array_equal(ta, tc)


def test_shard_ranges_cover_exactly():
    from paper_1309_7963_b200.sharding import shard_range
    for n in (0, 1, 7, 10**6, 10**7 + 3):
        for w in (1, 2, 3, 8):
            r = [shard_range(n, k, w) for k in range(w)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(r[i][1] == r[i + 1][0] for i in range(w - 1))
            assert max(b - a for a, b in r) - min(b - a for a, b in r) <= 1


_WORKER = r'''
import os, sys, json
sys.path.insert(0, sys.argv[1])
import numpy as np, torch, torch.distributed as dist
from paper_1309_7963_b200.sharding import shard_range, gather_secondary_bases
import paper_1309_7963_b200.workloads as W
from oracle import oracle as O
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%s" % sys.argv[2], rank=int(sys.argv[3]), world_size=2)
rank = dist.get_rank()
n = 600
E, tid, targets, seed, _ = W.make_inputs(4, n)
lo, hi = shard_range(n, rank, 2)
r = O.simulate(O.Tables(), targets, E[lo:hi], tid[lo:hi], seed, e0=lo)   # stand-in for the per-GPU call
base, total = gather_secondary_bases(r["total"])
json.dump(dict(lo=lo, hi=hi, base=base, total=total, counts=r["counts"].tolist(), T=r["T"].tolist()), open(sys.argv[4], "w"))
dist.barrier(); dist.destroy_process_group()
'''


def test_two_rank_sharding_gloo(orc, otables):
    """world_size 2 on CPU (gloo): each rank runs its event range with the global event offset;
    the concatenation equals the single-process run and the gathered bases are the offsets."""
    import paper_1309_7963_b200.workloads as W
    import socket
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    with tempfile.TemporaryDirectory() as d:
        w = os.path.join(d, "w.py"); open(w, "w").write(_WORKER)
        outs = [os.path.join(d, f"o{r}.json") for r in range(2)]
        ps = [subprocess.Popen([sys.executable, w, ROOT, str(port), str(r), outs[r]]) for r in range(2)]
        for p in ps:
            assert p.wait(timeout=240) == 0
        import json
        res = [json.load(open(o)) for o in outs]
    E, tid, targets, seed, _ = W.make_inputs(4, 600)
    full = orc.simulate(otables, targets, E, tid, seed)
    assert res[0]["counts"] + res[1]["counts"] == full["counts"].tolist()
    assert np.array_equal(np.array(res[0]["T"] + res[1]["T"]), full["T"])
    assert res[0]["base"] == 0 and res[1]["base"] == res[0]["total"] - len(res[1]["T"]) == len(res[0]["T"])
    assert res[0]["total"] == res[1]["total"] == full["total"]


def test_statistics_helpers():
    rng = np.random.default_rng(0)
    a = rng.multinomial(100000, np.ones(30) / 30)
    b = rng.multinomial(120000, np.ones(30) / 30)
    assert H.chi2_two_sample(a, b) > 1e-3
    p = np.ones(30); p[3] = 1.25
    c = rng.multinomial(120000, p / p.sum())
    assert H.chi2_two_sample(a, c) < 1e-6
    sp = np.array([0, 1, 0x85, 1, 0x80], dtype=np.uint8)
    h = H.histograms(sp, np.array([10.0, 30, 5, 260, 2]), np.array([0.1, -0.5, 0.9, 0.3, 0]), np.array([3, 2]), np.array([14, 15]))
    assert h["T_n"].sum() == 2 and h["T_p"].sum() == 1 and h["T_over_p"] == 1 and h["T_comp"].sum() == 1
    assert h["mult_all"][3] == 1 and h["mult_all"][2] == 1 and h["A_res"][14] == 1
    assert not H.compare_histograms(h, h)


def test_bench_gpus_flag_never_underreports():
    """bench.py --gpus N: without a torchrun environment it starts N ranks itself, and it refuses to run when
    fewer than N devices are visible or when WORLD_SIZE disagrees -- it can never print n_gpus: 1 for a run asked for N."""
    import bench
    assert bench.check_world(1, None) is False
    assert bench.check_world(2, None, visible=2) is True          # plain `python bench.py --gpus 2` on a 2-GPU node
    assert bench.check_world(2, "2") is False                     # a rank under torchrun
    with pytest.raises(SystemExit, match="only 1 CUDA device"):
        bench.check_world(2, None, visible=1)
    with pytest.raises(SystemExit, match="must agree"):
        bench.check_world(8, "2")
    # the rank arithmetic: disjoint event ranges, the slowest rank's time, the whole job's events
    sh = [bench.rank_share(r, 4, 1000, [1.0, 3.5, 2.0, 1.5]) for r in range(4)]
    assert [x["event_offset"] for x in sh] == [0, 1000, 2000, 3000]
    assert all(x["ms"] == 3.5 and x["events"] == 4000 for x in sh)
    # and as the driver would start it here (no GPU): a loud failure, not a line
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="")
    env.pop("WORLD_SIZE", None)
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1"], env=env,
                       capture_output=True, text=True, timeout=300)
    assert r.returncode != 0 and "n_gpus" not in r.stdout and "CUDA device" in r.stderr
