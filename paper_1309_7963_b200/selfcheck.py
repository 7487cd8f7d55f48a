"""Product-only self-check of an installation: one small batch through the C ABI, checked against the
conservation laws that hold for every event (BASELINE.json criterion (1)) -- no oracle involved.

    python -m paper_1309_7963_b200.selfcheck [--config C] [--events N] [--variant f32|f64]
                                             [--long-seg S] [--chunk M] [--host]

It was written as the target of compute-sanitizer runs:

    compute-sanitizer --tool memcheck  python -m paper_1309_7963_b200.selfcheck --config 1 --long-seg 2
    compute-sanitizer --tool racecheck python -m paper_1309_7963_b200.selfcheck --config 1 --long-seg 2

No such run exists under profiles/: the GPU pool this was developed on refuses the tool.  The substitute that does run
is the checked small-queue build (libinc_f64q.so, -DINC_CHECKED: every queue, ring and slot index verified on the
device), exercised by tests/test_gpu_parity.py::test_small_queue_build_and_overflow_rerun.

(--long-seg 2 makes almost every drain-phase track go through the drain helpers' shared-memory rings.)
"""
from __future__ import annotations

import argparse
import sys

import numpy as np

SPECIES_A = np.array([1, 1, 2, 3, 3, 4])
SPECIES_Z = np.array([0, 1, 1, 1, 2, 2])


def main(argv=None) -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--events", type=int, default=None)
    ap.add_argument("--variant", default="f32", choices=["f32", "f64"])
    ap.add_argument("--long-seg", type=int, default=0, help="inc_set_long_track_threshold (0 = default)")
    ap.add_argument("--chunk", type=int, default=0, help="inc_set_chunk_events (0 = default)")
    ap.add_argument("--flags", type=int, default=0)
    ap.add_argument("--host", action="store_true", help="go through inc_simulate_host")
    a = ap.parse_args(argv)

    import torch
    if not torch.cuda.is_available():
        print("selfcheck: no CUDA device (the product has no CPU path)", file=sys.stderr)
        return 2
    from . import binding as B, tables as T, workloads as W
    E, tid, targets, seed, name = W.make_inputs(a.config, a.events)
    n = len(E)
    lib = B.load(a.variant)
    lib.inc_shutdown()
    tables = T.default_tables()
    slots = np.array([lib.inc_init(A, Z, tables) for A, Z in targets], dtype=np.int32)
    lib.inc_set_stream()
    lib.inc_set_flags(a.flags)
    lib.inc_set_long_track_threshold(a.long_seg)
    lib.inc_set_chunk_events(a.chunk)
    cap = max(64, 24 * n)
    if a.host:
        out = lib.alloc_outputs(n, cap, device="cpu")
        total = lib.inc_simulate_host(torch.as_tensor(E.astype(lib.real)).pin_memory(),
                                      torch.as_tensor(slots[tid]).pin_memory(), seed, out)
    else:
        out = lib.alloc_outputs(n, cap)
        total = lib.inc_simulate(torch.as_tensor(E.astype(lib.real), device="cuda"),
                                 torch.as_tensor(slots[tid], device="cuda"), seed, out)
    torch.cuda.synchronize()
    r = {k: v.cpu().numpy() for k, v in out.items()}
    counts = r["counts"].astype(np.int64)
    assert counts.sum() == total, (counts.sum(), total)
    code = r["species"][:total] & 0x7F
    ev = np.repeat(np.arange(n), counts)
    At = np.array([A for A, Z in targets])[tid]
    Zt = np.array([Z for A, Z in targets])[tid]
    ok = (r["status"].view(np.uint32) & B.ST_FAILED) == 0
    dA = np.bincount(ev, weights=SPECIES_A[code], minlength=n) + r["A"] - (At + 1)
    dZ = np.bincount(ev, weights=SPECIES_Z[code], minlength=n) + r["Z"] - (Zt + 1)
    bad = int(np.sum((dA != 0) & ok) + np.sum((dZ != 0) & ok))
    flagged = int(np.sum((r["status"].view(np.uint32) & ~np.uint32(0xFF)) != 0))
    print(f"selfcheck {a.variant} config {a.config} ({name}), {n} events: {total} secondaries, "
          f"{bad} conservation violations, {flagged} events with status flags")
    lib.inc_set_long_track_threshold(0)
    lib.inc_set_chunk_events(0)
    lib.inc_shutdown()
    return 1 if bad else 0


if __name__ == "__main__":
    sys.exit(main())
