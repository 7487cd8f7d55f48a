#!/usr/bin/env python
"""bench.py — headline benchmark: 200 MeV p-16O non-elastic events/s on B200 (BASELINE.json).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C]

A "step" is one pass of the whole hot path (entry, segment, boundary, collision, epilogue,
evaporation, prefix sum, compaction: SURVEY 8(a)) over one batch of synthetic events — config 2
(1e6 x 200 MeV p-16O, seed 2) unless --config says otherwise.  Inputs are resident in HBM for
`value`; `e2e` goes through inc_simulate_host with pinned host buffers (H2D + D2H inside the
timed region).  N > 1 (torchrun): weak scaling, every rank runs the same batch size on its own
global event range; no data-path collective (events are independent).

--impl reference times the CPU oracle as it stands on the host cores (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "200 MeV p-16O non-elastic events/sec on 1 B200; % of FP32 issue roofline"
UNIT = "events/s"

# Algorithmic work model: lane-instructions per step kind, hand-counted
# from the formulas (FMA = 1, MUFU = 1, Philox block = 72), times the per-event step counts
# measured by the work counters.  Queue management, addressing and votes are NOT counted.
WORK = dict(segment=190.0, boundary=42.0, collision=255.0, epilogue=135.0, evap_step=430.0, evap_trial=90.0)


def work_per_event(stats: dict) -> dict:
    n = float(stats["events"])
    casc = (stats["segments"] * WORK["segment"] + stats["boundaries"] * WORK["boundary"] +
            stats["collisions"] * WORK["collision"] + stats["attempts"] * WORK["epilogue"]) / n
    evap = (stats["evap_steps"] * WORK["evap_step"] + stats["evap_trials"] * WORK["evap_trial"]) / n
    return dict(cascade=casc, evap=evap, total=casc + evap)


class ClockSampler:
    """SM clock and throttle reasons DURING the timed region (B200_PROFILING.md).  The timed region of the default run is
    ~20 ms, so the recipe's `nvidia-smi -lms 200` would see it once at best: this polls NVML from a thread every
    millisecond instead (same counters), and falls back to nvidia-smi if NVML cannot be loaded."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc, self.nvml, self.stop_flag = index, [], None, None, False

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            # CUDA_VISIBLE_DEVICES may renumber: take the NVML handle by the PCI bus id of the torch device
            import torch
            bus = torch.cuda.get_device_properties(self.index).pci_bus_id if hasattr(torch.cuda.get_device_properties(self.index), "pci_bus_id") else None
            self.h = pynvml.nvmlDeviceGetHandleByIndex(self.index) if bus is None else pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.nvml = pynvml
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.th = threading.Thread(target=self._poll, daemon=True)
            self.th.start()
            return
        except Exception:
            self.nvml = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "20", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _poll(self):
        n = self.nvml
        R = {"hw_slowdown": n.nvmlClocksEventReasonHwSlowdown if hasattr(n, "nvmlClocksEventReasonHwSlowdown") else 0x8,
             "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}
        get_reasons = getattr(n, "nvmlDeviceGetCurrentClocksEventReasons", None) or getattr(n, "nvmlDeviceGetCurrentClocksThrottleReasons")
        while not self.stop_flag:
            try:
                sm = float(n.nvmlDeviceGetClockInfo(self.h, n.NVML_CLOCK_SM))
                mask = int(get_reasons(self.h))
                pw = n.nvmlDeviceGetPowerUsage(self.h) / 1000.0
                self.rows.append((time.time(), sm, pw, [k for k, bit in R.items() if mask & bit]))
            except Exception:
                pass
            time.sleep(0.001)

    def _read(self):
        for line in self.proc.stdout:
            r = [x.strip() for x in line.split(",")]
            if len(r) >= 9:
                names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
                self.rows.append((time.time(), float(r[1]), float(r[3]), [k for k, v in zip(names, r[5:9]) if v.lower().startswith("active")]))
                self.sm_max = float(r[2])

    def stop(self, t0, t1):
        self.stop_flag = True
        if self.nvml is None and not self.proc:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["no NVML, no nvidia-smi"])
        time.sleep(0.03)
        if self.proc:
            self.proc.terminate()
        rows = [r for r in self.rows if t0 <= r[0] <= t1]
        loaded = [r for r in self.rows if r[0] <= t1]
        if not rows:
            rows = loaded[-3:]
        if not rows:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["no samples"])
        sm = sorted(r[1] for r in rows)
        reasons = sorted({k for r in rows for k in r[3]})
        return dict(sm_mhz=sm[len(sm) // 2], sm_min_mhz=sm[0], sm_max_mhz=getattr(self, "sm_max", None), power_w_max=max(r[2] for r in rows),
                    samples=len(rows), samples_warmup_and_timed=len(loaded), source="NVML polled every ms" if self.nvml else "nvidia-smi -lms 20",
                    reasons=reasons)


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def _oracle_shard(job):
    """One process of the all-core oracle leg: events [a, b) of the config (counter-keyed RNG: shards are exact)."""
    cfg, n, a, b = job
    from oracle import oracle as O
    import paper_1309_7963_b200.workloads as W
    E, tid, targets, seed, _ = W.make_inputs(cfg, n)
    t = O.Tables()
    nuclei = [O.setup_nucleus(A, Z, t) for A, Z in targets]
    t0 = time.perf_counter()
    O.simulate(t, nuclei, E[a:b], tid[a:b], seed, e0=a, want_stats=False)
    return time.perf_counter() - t0


def oracle_baseline(cfg, n, one_thread_events, per_core_events):
    """The oracle as it stands on the host cores: one thread, then one process per core on disjoint event ranges."""
    import multiprocessing as mp
    m1 = min(one_thread_events, n)
    dt1 = _oracle_shard((cfg, n, 0, m1))
    P = os.cpu_count() or 1
    per = max(1000, min(per_core_events, n // P))
    jobs = [(cfg, n, i * per, (i + 1) * per) for i in range(P)]
    t0 = time.perf_counter()
    with mp.get_context("spawn").Pool(P) as pool:
        pool.map(_oracle_shard, jobs[:P])            # (first map also pays the workers' start-up and library load)
        t1 = time.perf_counter()
        pool.map(_oracle_shard, jobs)
        dtP = time.perf_counter() - t1
    return dict(value=P * per / dtP, unit=UNIT, cores=P, kind="oracle", cpu_model=cpu_model(),
                single_thread=dict(value=m1 / dt1, events=m1, seconds=round(dt1, 2)),
                sample=f"config {cfg}: {P} processes x {per} events each in {dtP:.1f} s (aggregate = value); one thread: first {m1} events in "
                       f"{dt1:.1f} s; oracle/inc_oracle.c as it stands, gcc -O2 -ffp-contract=off")


def run_reference(args, rank, world):
    """The oracle as it stands, single thread, on a bounded sample per step."""
    if rank != 0:
        return
    import numpy as np
    from oracle import oracle as O
    import paper_1309_7963_b200.workloads as W
    cfg = args.config
    sample = args.ref_events
    E, tid, targets, seed, name = W.make_inputs(cfg, sample)
    t = O.Tables()
    nuclei = [O.setup_nucleus(a, z, t) for a, z in targets]
    for _ in range(args.warmup):
        O.simulate(t, nuclei, E[:2000], tid[:2000], seed, want_stats=False)
    t0 = time.perf_counter()
    for k in range(args.steps):
        O.simulate(t, nuclei, E, tid, seed, e0=k * sample, want_stats=False)
    dt = time.perf_counter() - t0
    v = args.steps * sample / dt
    line = dict(metric=METRIC, value=v, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=1e3 * dt / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f64", data="synthetic", impl="reference",
                config=dict(workload=f"config {cfg}: {name}", events_per_step=sample,
                            note="bounded sample of the workload per step; oracle/inc_oracle.c, gcc -O2 -ffp-contract=off"),
                cpu_baseline=dict(value=v, unit=UNIT, cores=1, kind="oracle", sample=f"{sample} events/step x {args.steps} steps of config {cfg}"),
                e2e=dict(value=v, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))


def check_world(gpus: int, world_env, visible=None) -> bool:
    """--gpus N against the launch: returns True if this process must start N ranks itself (N > 1 and no torchrun
    environment), False if it is a rank (or N = 1) and the numbers agree.  Anything else stops the run: a line that says
    n_gpus: 1 for a run asked to use N GPUs, or N ranks sharing fewer than N devices, is never printed."""
    if world_env is None:
        if gpus <= 1:
            return False
        if visible is None:
            import torch
            visible = torch.cuda.device_count()
        if visible < gpus:
            raise SystemExit(f"bench.py --gpus {gpus}: only {visible} CUDA device(s) visible; not reporting a {gpus}-GPU number from fewer")
        return True
    if int(world_env) != gpus:
        raise SystemExit(f"bench.py --gpus {gpus} launched with WORLD_SIZE={world_env}: the two must agree")
    return False


def rank_share(rank: int, world: int, n: int, ms_by_rank) -> dict:
    """The multi-GPU arithmetic of the bench (events are independent): rank r owns global events
    [r n, (r + 1) n) -- no collective on the data path -- and the job's time is the slowest rank's."""
    return dict(event_offset=rank * n, ms=max(ms_by_rank), events=world * n)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--events", type=int, default=None, help="override the config's event count")
    ap.add_argument("--ref-events", type=int, default=100000, help="events per step of --impl reference")
    ap.add_argument("--cpu-events", type=int, default=400000, help="oracle sample of the cpu_baseline leg: one thread; a quarter of it per core for the all-core leg")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the one-line-per-config block (configs 1-5, f32 and f64)")
    ap.add_argument("--variant", default="f32", choices=["f32", "f64"])
    ap.add_argument("--flags", type=int, default=0)
    ap.add_argument("--vote", type=int, nargs=2, default=None)
    ap.add_argument("--taper", type=int, default=None, help="inc_set_event_taper (scheduling experiment)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "ours":
        relaunch = check_world(args.gpus, os.environ.get("WORLD_SIZE"))
        if relaunch:
            # started as plain `python bench.py --gpus N`: start the N ranks ourselves (one process per GPU)
            import socket
            with socket.socket() as sk:
                sk.bind(("127.0.0.1", 0))
                port = sk.getsockname()[1]
            cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
                   "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
            os.execv(sys.executable, cmd)

    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import numpy as np
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    import paper_1309_7963_b200.binding as B
    import paper_1309_7963_b200.tables as T
    import paper_1309_7963_b200.workloads as W

    cfg = args.config
    n = args.events or W.CONFIGS[cfg]["n"]
    E, tid, targets, seed, name = W.make_inputs(cfg, n)
    lib = B.load(args.variant)
    tables = T.default_tables()
    lib.inc_shutdown()
    slots = np.array([lib.inc_init(a, z, tables) for a, z in targets], dtype=np.int32)
    lib.inc_set_stream()
    if args.vote:
        lib.inc_set_vote_thresholds(*args.vote)
    if args.taper is not None:
        lib.inc_set_event_taper(args.taper)
    real_t = lib.torch_real()
    E_d = torch.as_tensor(E.astype(lib.real), device="cuda")
    tid_d = torch.as_tensor(slots[tid], device="cuda")
    cap = n * 16
    out = lib.alloc_outputs(n, cap)
    lib.inc_set_event_offset(rank_share(rank, world, n, [0.0])["event_offset"])      # weak scaling: rank r owns global events [r n, (r+1) n)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- work counters: one untimed pass with INC_F_STATS ----
    lib.inc_set_flags(args.flags | B.F_STATS)
    total = lib.inc_simulate(E_d, tid_d, seed, out)
    stats = lib.inc_get_stats()
    wpe = work_per_event(stats)

    # ---- the timed region: K steps in the production configuration (the evaporation kernel overlaps the cascade
    # kernel's tail, no events between the stages), CUDA events around it on the launching stream ----
    lib.inc_set_flags(args.flags)
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    for _ in range(args.warmup):
        lib.inc_simulate(E_d, tid_d, seed, out)
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    step_ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    t_wall0 = time.time()
    ev0.record()
    step_ev[0].record()
    for k in range(args.steps):
        lib.inc_simulate(E_d, tid_d, seed + k, out)
        step_ev[k + 1].record()
    ev1.record()
    barrier()
    t_wall1 = time.time()
    ms_total = ev0.elapsed_time(ev1)
    tmax = torch.tensor([ms_total], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    ms_total = float(tmax.item())
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None
    value = world * n * args.steps / (ms_total * 1e-3)
    per_step = sorted(step_ev[k].elapsed_time(step_ev[k + 1]) for k in range(args.steps))
    chunks = -(-n // (1 << 22))
    launches = args.steps * chunks * 6          # cascade, evaporation, three scan kernels, compaction per chunk

    # ---- per-kernel durations: the same K steps again with INC_F_TIMING, which puts CUDA events between the stages
    # and therefore runs them one after the other (the roofline of a kernel needs a duration of its own) ----
    lib.inc_set_flags(args.flags | B.F_TIMING)
    lib.inc_simulate(E_d, tid_d, seed, out)
    stage = dict(cascade=0.0, evap=0.0, scan=0.0, compact=0.0)
    sv0, sv1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sv0.record()
    for k in range(args.steps):
        lib.inc_simulate(E_d, tid_d, seed + k, out)
        ms, nl = lib.inc_get_stage_times()
        for kk in stage:
            stage[kk] += ms[kk]
    sv1.record()
    torch.cuda.synchronize()
    serial_ms = sv0.elapsed_time(sv1) / args.steps
    timeline = lib.inc_get_drain_timeline()

    # ---- extras (outside the timed region) ----
    # divergence-free ceiling: every event draws the random stream of event 0
    lib.inc_set_flags(args.flags | B.F_SAME_STREAM)
    lib.inc_simulate(E_d, tid_d, seed, out)
    pev0, pev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    pev0.record()
    lib.inc_simulate(E_d, tid_d, seed, out)
    pev1.record()
    torch.cuda.synchronize()
    same_stream_ms = pev0.elapsed_time(pev1)
    # on-device tallies
    lib.inc_set_flags(args.flags)
    lib.inc_simulate(E_d, tid_d, seed + args.steps - 1, out)
    off_d = lib.inc_get_offsets(n)
    tspec, tall = lib.alloc_tallies()
    lib.inc_tally(out, off_d, tspec, tall)
    tev0, tev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    tev0.record()
    for _ in range(5):
        lib.inc_tally(out, off_d, tspec, tall)
    tev1.record()
    torch.cuda.synchronize()
    tally_ms = tev0.elapsed_time(tev1) / 5

    # ---- end to end through the host-buffer entry point (pinned host memory) ----
    E_h = torch.as_tensor(E.astype(lib.real)).pin_memory()
    tid_h = torch.as_tensor(slots[tid]).pin_memory()
    out_h = lib.alloc_outputs(n, cap, device="cpu")
    lib.inc_simulate_host(E_h, tid_h, seed, out_h)
    e2e_steps = max(2, min(args.steps, 5))
    barrier()
    t0 = time.perf_counter()
    tot_h = 0
    for k in range(e2e_steps):
        tot_h = lib.inc_simulate_host(E_h, tid_h, seed + k, out_h)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    tm = torch.tensor([dt], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(tm, op=dist.ReduceOp.MAX)
    e2e_value = world * n * e2e_steps / float(tm.item())
    # the host link itself: one 256 MB device-to-host copy into pinned memory, timed (the floor of the e2e number)
    lk_d = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    lk_h = torch.empty(256 << 20, dtype=torch.uint8).pin_memory()
    lk_h.copy_(lk_d, non_blocking=True)
    torch.cuda.synchronize()
    l0, l1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0.record()
    lk_h.copy_(lk_d, non_blocking=True)
    l1.record()
    torch.cuda.synchronize()
    d2h_GBps = (256 << 20) / (l0.elapsed_time(l1) * 1e-3) / 1e9
    del lk_d, lk_h
    rb = E_h.element_size()
    h2d = n * (rb + 4)
    d2h = n * (4 + 4 + 4 + 4 * rb + 4) + tot_h * (1 + 4 * rb)
    del out_h, E_h, tid_h

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (cascade): plain-ALU issue bound ----
    peak, clk = lib.inc_measure_issue_peak()
    casc_ms = stage["cascade"] / args.steps
    achieved = wpe["cascade"] * n / (casc_ms * 1e-3)
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "roofline_traffic.json")
    if os.path.exists(tpath):
        try:
            traffic = json.load(open(tpath)).get("cascade_dram_bytes_per_launch")
        except Exception:
            traffic = None
    roofline = dict(bound="alu", kernel="cascade_wavefront_kernel", achieved=achieved / 1e12, peak=peak / 1e12, unit="T lane-instr/s",
                    frac=achieved / peak, traffic=traffic,
                    peak_source=f"measured in this run: {'FFMA' if args.variant == 'f32' else 'DFMA'} chain microbenchmark (inc_measure_issue_peak)",
                    work_lane_instr_per_event=wpe, kernel_ms=dict((k, v / args.steps) for k, v in stage.items()),
                    kernel_ms_note="stages run one after the other (INC_F_TIMING) over the same K steps; in the timed region the evaporation kernel overlaps the cascade kernel's tail",
                    serialized_ms_per_step=serial_ms,
                    kernel_share=dict((k, v / max(sum(stage.values()), 1e-9)) for k, v in stage.items()),
                    evap_frac=wpe["evap"] * n / (stage["evap"] / args.steps * 1e-3) / peak,
                    whole_step_frac=wpe["total"] * n / (ms_total / args.steps * 1e-3) / peak)

    # ---- every config of BASELINE.json, one line each (outside the timed region): production build, events/s of the
    # whole step, cascade roofline fraction; and the fp64 parity build's events/s ----
    per_config = None
    if not args.no_per_config and world == 1 and args.variant == "f32":
        per_config = {}
        del out
        for c in (1, 2, 3, 4, 5):
            per_config[str(c)] = config_line(c, peak, B, T, W, np, torch, oracle=not args.no_cpu_baseline)
        # the same headline workload with the GEM level density (NEXT-2; no pairing / shell arrays: the uncorrected a = A/8)
        per_config["2_gem"] = config_line(2, peak, B, T, W, np, torch, oracle=False, tables_kw=dict(level_density=1))
        lib.inc_shutdown()

    cpu_baseline = None
    if not args.no_cpu_baseline:
        cpu_baseline = oracle_baseline(cfg, n, args.cpu_events, args.cpu_events // 4)

    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
                ms_per_step=ms_total / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype=args.variant, data="synthetic",
                config=dict(workload=f"config {cfg}: {name}", events_per_step_per_gpu=n, seed=seed,
                            secondaries_per_step=int(total), build=lib.build_info(),
                            l2="no flush: each step writes and re-reads ~0.3 GB (staging records, nucleus records, outputs; new seed every step), above the 126 MB L2",
                            parallelism=f"dp{world} (independent event ranges, no collective)"),
                clocks=clocks, e2e=dict(value=e2e_value, unit=UNIT, h2d_bytes_per_step=int(h2d), d2h_bytes_per_step=int(d2h),
                                        steps=e2e_steps, d2h_link_GBps=d2h_GBps,
                                        link_floor_events_per_s=n / (d2h / (d2h_GBps * 1e9)),
                                        note="link: one 256 MB device-to-pinned-host copy timed in this run; floor = the step's D2H bytes at that rate"),
                gpu_launches=int(launches), roofline=roofline, cpu_baseline=cpu_baseline,
                per_step_ms=dict(best=per_step[0], median=per_step[len(per_step) // 2]),
                per_config=per_config,
                same_stream_probe=dict(ms=same_stream_ms, events_per_s=n / (same_stream_ms * 1e-3),
                                       note="INC_F_SAME_STREAM: all events identical, no divergence (the paper's probe, P:73-75)"),
                paper_time_split="GTX680, 200 MeV p-16O: INC 72 %, evaporation 23 %, RNG init 3 % (P:142); see roofline.kernel_share",
                cascade_drain_timeline_ms=timeline,
                tally=dict(ms=tally_ms, note="inc_tally over the step's outputs (dd spectra 3x20x51, multiplicities, nuclide chart, yields); not part of the step"),
                work_counters_per_event={k: stats[k] / max(stats["events"], 1) for k in
                                         ("attempts", "segments", "boundaries", "collisions", "allowed", "evap_steps", "evap_trials")},
                lane_utilisation=dict(seg=stats["lane_slots_seg"] / max(32 * stats["warp_iters_seg"], 1),
                                      coll=stats["lane_slots_coll"] / max(32 * stats["warp_iters_coll"], 1),
                                      epi=stats["lane_slots_epi"] / max(32 * stats["warp_iters_epi"], 1)))
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def config_line(c, peak, B, T, W, np, torch, steps=3, oracle=True, tables_kw=None):
    """One BASELINE.json config: events/s of the whole step (production build, device-resident, `steps` steps after two
    warm-ups), the cascade kernel's roofline fraction (INC_F_TIMING steps), and the fp64 parity build's events/s."""
    n = W.CONFIGS[c]["n"]
    E, tid, targets, seed, name = W.make_inputs(c, n)
    tables = T.default_tables(**(tables_kw or {}))
    res = dict(workload=name + (" [GEM level density]" if tables_kw else ""), events=n)
    for variant in ("f32", "f64"):
        lib = B.load(variant)
        lib.inc_shutdown()
        slots = np.array([lib.inc_init(a, z, tables) for a, z in targets], dtype=np.int32)
        lib.inc_set_stream()
        m = n if variant == "f32" else min(n, 1000000)
        E_d = torch.as_tensor(E[:m].astype(lib.real), device="cuda")
        tid_d = torch.as_tensor(slots[tid[:m]], device="cuda")
        out = lib.alloc_outputs(m, m * 12)
        if variant == "f32":
            lib.inc_set_flags(B.F_STATS)
            lib.inc_simulate(E_d, tid_d, seed, out)
            st = lib.inc_get_stats()
            wpe = work_per_event(st)
            res["lanes_per_segment_step"] = st["lane_slots_seg"] / max(st["warp_iters_seg"], 1)
        lib.inc_set_flags(0)
        for _ in range(2):
            lib.inc_simulate(E_d, tid_d, seed, out)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for k in range(steps):
            lib.inc_simulate(E_d, tid_d, seed + k, out)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / steps
        if variant == "f32":
            lib.inc_set_flags(B.F_TIMING)
            casc = 0.0
            for k in range(steps):
                lib.inc_simulate(E_d, tid_d, seed + k, out)
                casc += lib.inc_get_stage_times()[0]["cascade"] / steps
            res.update(events_per_s=m / (ms * 1e-3), ms_per_step=ms, cascade_ms=casc,
                       roofline_frac=wpe["cascade"] * m / (casc * 1e-3) / peak,
                       whole_step_frac=wpe["total"] * m / (ms * 1e-3) / peak)
        else:
            # the parity build against ITS roofline: the same algorithmic lane-instructions, the DFMA issue peak measured
            # with this library's own chain microbenchmark
            peak64, _ = lib.inc_measure_issue_peak()
            res.update(f64_events_per_s=m / (ms * 1e-3), f64_events=m, f64_ms_per_step=ms, f64_dfma_peak_T_lane_instr_per_s=peak64 / 1e12,
                       f64_roofline_frac=wpe["total"] * m / (ms * 1e-3) / peak64)
        lib.inc_set_flags(0)
        lib.inc_shutdown()
        del out, E_d, tid_d
        torch.cuda.empty_cache()
    if oracle:
        # the oracle on this config: one thread on 5e4 events, then every core on 2e4 events each
        ob = oracle_baseline(c, n, min(n, 50000), 20000)
        res.update(oracle_events_per_s_1thread=ob["single_thread"]["value"], oracle_events_per_s_allcores=ob["value"], oracle_cores=ob["cores"])
    return res


if __name__ == "__main__":
    main()
