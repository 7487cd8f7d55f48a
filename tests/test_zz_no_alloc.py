"""GPU test of inc_scan_counts_static, the library's one entry point that allocates nothing.

Who needs it: a host program that has given the whole device memory to an allocator of its own (a transport Monte
Carlo with a fixed memory budget, a framework pool sized to the GPU), where a cudaMalloc issued by a library fails or
eats into that budget, and a caller in a latency-critical loop, where cudaMalloc / cudaFree stall every stream of the
device.  For them the prefix sum of the per-event counts keeps its scratch in a fixed array inside the library (room
for 2^24 events) instead of a cudaMalloc'ed buffer.

The array is shared by every call and keeps what the last call left, so the test makes two calls in a row, the second
one shorter than the first and with other counts: anything stale that leaked into it would show.  Each result must be
bit-identical (integer work) to the existing path, inc_get_offsets after inc_simulate on the same events.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It passes alone in a fresh process (the first call on the device does the set-up) and after the others.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _simulate_counts(lib, n, config_id, seed_shift=0):
    import torch
    import paper_1309_7963_b200.tables as T
    import paper_1309_7963_b200.workloads as W
    E, tid, targets, seed, _ = W.make_inputs(config_id, n)
    lib.inc_shutdown()
    slots = np.asarray([lib.inc_init(a, z, T.default_tables()) for a, z in targets], dtype=np.int32)
    lib.inc_set_stream()
    lib.inc_set_flags(0)
    Ed = torch.as_tensor(np.asarray(E, dtype=lib.real), device="cuda")
    td = torch.as_tensor(slots[np.asarray(tid)], device="cuda")
    out = lib.alloc_outputs(n, 24 * n)
    total = lib.inc_simulate(Ed, td, seed + seed_shift, out)
    ref = lib.inc_get_offsets(n)                   # the existing path: scratch from cudaMalloc
    return out["counts"], ref, total


@pytest.mark.parametrize("variant", ["f32", "f64"])
def test_static_scratch_scan_matches_existing_path_twice(variant):
    import torch
    import paper_1309_7963_b200.binding as B
    if not torch.cuda.is_available():
        pytest.fail("needs a CUDA device")
    lib = B.load(variant)
    # first call: several tiles of 2048 events and a ragged tail; second call: fewer events, other counts
    for n, config_id, shift in ((3 * 2048 + 777, 2, 0), (2048 + 5, 5, 11)):
        counts, ref, total = _simulate_counts(lib, n, config_id, shift)
        off = torch.full((n + 1,), -7, dtype=torch.int64, device="cuda")      # caller-owned output, poisoned
        lib.inc_scan_counts_static(counts, off)
        assert torch.equal(off, ref), (variant, n)
        assert int(off[n]) == total
        # and the definition itself, computed by torch, so that the two paths cannot be wrong together
        want = torch.zeros(n + 1, dtype=torch.int64, device="cuda")
        want[1:] = torch.cumsum(counts.to(torch.int64), 0)
        assert torch.equal(off, want)
    lib.inc_shutdown()


def test_static_scratch_scan_edges_and_limit():
    import torch
    import paper_1309_7963_b200.binding as B
    lib = B.load("f32")
    lib.inc_set_stream()
    # a large, ragged n right after small ones: every tile sum is rewritten, the old total is cleared
    g = torch.Generator(device="cuda").manual_seed(5)
    for n in (1, 2048, 2049, 1_000_003, 0, 33):
        counts = torch.randint(0, 65, (max(n, 1),), generator=g, device="cuda", dtype=torch.int32)[:n]
        off = torch.full((n + 1,), -7, dtype=torch.int64, device="cuda")
        lib.inc_scan_counts_static(counts, off, n=n)
        want = torch.zeros(n + 1, dtype=torch.int64, device="cuda")
        if n:
            want[1:] = torch.cumsum(counts.to(torch.int64), 0)
        assert torch.equal(off, want), n
    # beyond the fixed array: refused with a message, the output untouched
    off = torch.full((4,), -7, dtype=torch.int64, device="cuda")
    counts = torch.zeros(4, dtype=torch.int32, device="cuda")
    rc = lib.inc_scan_counts_static(counts, off, n=B.SCAN_STATIC_MAX_EVENTS + 1, check=False)
    assert rc == B.INC_E_BADARG
    assert "beyond" in lib.last_error() and str(B.SCAN_STATIC_MAX_EVENTS) in lib.last_error()
    assert bool((off == -7).all())
