/* inc.h — C ABI of the B200-native intranuclear-cascade + evaporation Monte Carlo
 * (hot path of arXiv:1309.7963; citations "P:NN" are /root/reference/PAPER.md lines,
 * "R-xx" are the readings frozen in DESIGN.md section 3).
 *
 * One source, two shared libraries with identical symbol names:
 *     libinc_f32.so   INC_REAL = float    production build ("floating point precision")
 *     libinc_f64.so   INC_REAL = double   parity build, compiled with -fmad=false
 * Define INC_REAL_IS_DOUBLE before including this header to describe libinc_f64.so.
 *
 * Conventions
 *  - Every function returns 0 (or a non-negative value where stated) on success and a
 *    negative INC_E_* code on failure.  Nothing throws or aborts; inc_last_error() gives
 *    a human-readable message for the last failure.
 *  - The library has ONE process-wide state (targets, tables, workspace, stream, flags) bound to the CUDA
 *    device that was current at the first inc_init: it is not thread-safe, and concurrent callers must
 *    serialise their calls.  One process drives one GPU (one process per GPU).
 *  - "DEVICE" pointers are CUDA device pointers owned by the caller (e.g. torch tensors);
 *    the library never frees or reallocates them.  "HOST" pointers are ordinary host
 *    memory.  The library owns only its internal workspace and the device copies of the
 *    model tables.
 *  - All work is enqueued on the stream given to inc_set_stream() (default: stream 0).
 *    inc_simulate() ends with ONE small synchronous device-to-host copy (total number of
 *    secondaries + error word), so on return the outputs are complete.
 *  - Determinism: results depend only on (seed, global event index e = 0..n-1, E_in[e],
 *    target_id[e], tables) — not on chunking, launch shape or GPU (R-R4).
 *  - Units: MeV, MeV/c, fm.  Beam along +z (R-Q15); the caller rotates.
 *  - There is NO CPU fallback: without a CUDA device every compute call returns INC_E_CUDA.
 */
#ifndef INC_H
#define INC_H
#include <stdint.h>

#ifdef INC_REAL_IS_DOUBLE
typedef double INC_REAL;
#else
typedef float INC_REAL;
#endif

#ifdef __cplusplus
extern "C" {
#endif

/* ---- error codes ------------------------------------------------------------------ */
#define INC_OK 0
#define INC_E_BADARG (-1)   /* null pointer, n < 0, unsupported (A,Z), E_in outside [20,250] MeV
                               (found on device and reported, not clamped), unknown target_id */
#define INC_E_TABLES (-2)   /* wrong version, non-monotone grid, or tables differ from the
                               ones captured by the first inc_init                       */
#define INC_E_CAPACITY (-3) /* out_secondaries->capacity too small: nothing is written past
                               capacity, out_counts / residual are still complete, and
                               inc_last_error() reports the needed size                   */
#define INC_E_CUDA (-4)     /* a CUDA call failed; message in inc_last_error()            */
#define INC_E_STATE (-5)    /* call order: inc_simulate before any inc_init, etc.         */

/* ---- per-event status word (out_residual->status) ----------------------------------- */
#define INC_ST_ATTEMPTS_MASK 0xFFu  /* bits 0-7: cascade attempts used (R-C6), saturating    */
#define INC_ST_FAILED (1u << 8)     /* 256 attempts without a valid non-elastic event:
                                       count = 0, residual = target at rest              */
#define INC_ST_SEC_TRUNC (1u << 9)  /* more than INC_MAX_SEC secondaries: extra dropped (R-C5) */
#define INC_ST_DEPTH_CAP (1u << 10) /* path code would exceed 24 bits (R-C3)              */
#define INC_ST_SEG_CAP (1u << 11)   /* a track hit 1024 segments and was absorbed (R-C2)  */
#define INC_ST_TRIAL_CAP (1u << 12) /* evaporation sampler hit 64 trials; chain stopped (R-E4) */
#define INC_ST_QUEUE_OVF (1u << 13) /* implementation limit: pending-track storage overflowed;
                                       never expected, tests assert it is never set       */

#define INC_MAX_SEC 64        /* R-C5 */
#define INC_MAX_TARGETS 16
#define INC_E_MIN 20.0        /* P:9 "between 20 and 250 MeV" */
#define INC_E_MAX 250.0

/* ---- flags for inc_set_flags ---------------------------------------------------------- */
#define INC_F_CASCADE_ONLY 1u      /* stop after the cascade epilogue: outputs are the cascade
                                      secondaries and the post-cascade residual ("SoA of
                                      excited nuclei")                                     */
#define INC_F_KEEP_TRANSPARENT 2u  /* debug: accept attempts without a real collision       */
#define INC_F_SAME_STREAM 4u       /* divergence probe of P:73-75: every event draws the random
                                      stream of event 0                                     */
#define INC_F_STATS 8u             /* accumulate the work counters of inc_get_stats         */
#define INC_F_TIMING 32u           /* record CUDA events around each stage (inc_get_stage_times) */
#define INC_F_LANE_PER_EVENT 16u   /* scheduling variant: one lane runs one event straight through,
                                      no phase voting (the layout of P:61, for comparison)  */
#define INC_F_LANE_STATE_MACHINE 64u /* scheduling variant: lane-per-event state machine with
                                      warp-voted phases instead of the default per-warp
                                      wavefront queues.  Results never depend on the variant. */

#define INC_F_NO_OVERLAP 512u       /* scheduling variant: the evaporation kernel starts only after the cascade kernel
                                      has finished (no programmatic dependent launch).  Results never depend on it. */
#define INC_F_TEST_QUEUE_OVF 1024u  /* test hook: one warp of the wavefront kernel reports a track-queue overflow and
                                      abandons its events, as a real overflow would; exercises the library's rerun of
                                      the call with the lane kernel                                                  */
#define INC_F_NO_DRAIN_HELPERS 256u /* scheduling variant: every track stays with the warp that owns its
                                      event (no drain helpers).  Results never depend on it.   */

/* ---- model inputs ("precalculated ... tables and other read-only input data") ----- */
typedef struct inc_tables {   /* HOST memory, caller-owned, copied during inc_init           */
  int32_t version;            /* 1: the fields up to evap_a_div; 2: also the level-density block at the end */
  int32_t n_xs;               /* NN grid points (<= 4096); plab_k = k*plab_max/(n_xs-1) GeV/c */
  double plab_max;
  const double *sig_pp, *sig_np;    /* [n_xs] elastic NN cross sections, mb (pp also for nn) */
  const double *B_pp, *B_np, *a_np; /* [n_xs] slope of exp(B t), (GeV/c)^-2; np backward weight    */
  int32_t n_evz;                    /* Dostrovsky grid points (<= 16)                        */
  const double *ev_Z, *ev_kp, *ev_cp, *ev_ka, *ev_ca; /* [n_evz] k, c vs daughter charge      */
  double ws_c0, ws_delta, ws_rpad;  /* 1.07, 0.545, 2.5 (Eq. (1))                      */
  int32_t n_shells;                 /* 15; 1..32                                      */
  double semf[5];                   /* a_v a_s a_c a_a a_p, MeV ("semi-empirical mass formula") */
  double evap_r0, evap_rj, evap_a_div; /* 1.5 fm, 1.2 fm, 8 (R-E1)                           */
  /* ---- version 2: level density of the evaporation stage ("we adopt the generalized
   * evaporation model (GEM) [18]").  level_density = 0 is the frozen Weisskopf-Ewing model rho ~ exp(2 sqrt(a U)),
   * a = A_d / evap_a_div (R-Q19); level_density = 1 is the GEM level density (DESIGN.md R-G1..G6): Fermi gas with
   * the pre-exponential factor, rho(U) = exp(2 sqrt(a (U - delta))) / (a^(1/4) (U - delta)^(5/4)), above the
   * Gilbert-Cameron matching energy E_x = U_x + delta, U_x = 150/A_d + 2.5 MeV, and the constant-temperature form
   * exp((U - E_0)/T)/T below it, with T, E_0 from continuity of value and slope convention of [18]
   * (1/T = sqrt(a/U_x) - 1.5/U_x).  Pairing energies and shell corrections are CALLER INPUTS like the NN tables
   * (the paper prints none): delta = pair_Z[Z_d] + pair_N[N_d]; a = A_d (gc_a0 + gc_a1 (shell_Z[Z_d] + shell_N[N_d]));
   * indices beyond the arrays count as 0; a <= 0 closes the channel.  It changes the emission widths (E2) and the
   * energy sampler (E4) only.  inc_init then also builds per-nucleus tables of the width integrals (about a second of
   * host time and 55 MB (f32) / 110 MB (f64) of device memory). */
  int32_t level_density;
  int32_t n_ldZ, n_ldN;              /* lengths of the arrays below (may be 0 with NULL pointers)            */
  const double *pair_Z, *pair_N;     /* [n_ldZ], [n_ldN] pairing energies, MeV                               */
  const double *shell_Z, *shell_N;   /* [n_ldZ], [n_ldN] shell corrections, MeV                              */
  double gc_a0, gc_a1;               /* 1/8 MeV^-1 and 0.00917 MeV^-2 in [18]                                */
} inc_tables;

/* inc_init — nuclear setup for one target (Woods-Saxon -> n_shells constant-density
 * shells, Fermi momenta/energies, V = E_F + E_B, Coulomb barrier) done in fp64 on the host,
 * uploaded once.  The first call also captures the NN / evaporation tables.
 * Supported: 6 <= A <= 64, 2 <= Z <= A-2 (the separation energies need valid A-1 nuclei; the library's binding-energy
 * and evaporation-channel tables cover every nucleus a cascade on such a target can leave).  Returns target_id >= 0 (slot, < INC_MAX_TARGETS).
 * Performance note: the default (wavefront) cascade kernel stages the records of all live target slots in shared memory
 * beside its track queues, which leaves room for slots 0..9 in the f32 build with tables of at most 15 shells (0..4 with
 * more shells); while a higher slot is live the library uses the lane-per-event cascade kernel instead (same results,
 * about half the throughput).  Free unused targets. */
int inc_init(int A, int Z, const inc_tables *tables /*HOST*/);
int inc_free_target(int target_id);
void inc_shutdown(void);       /* frees every target, the tables and the workspace          */

int inc_set_stream(void *cuda_stream /* cudaStream_t, e.g. torch.cuda.current_stream().cuda_stream */);
int inc_set_flags(uint32_t flags);
/* Scheduling knob of the cascade kernel: a warp runs the collision phase when at least `coll`
 * lanes wait for it, the epilogue+entry phase when at least `epi` lanes wait (1..32; default 8, 8).
 * Results never depend on it. */
int inc_set_vote_thresholds(int coll, int epi);
/* Incident nucleon species (the paper's model is a "nucleon-nucleus" one, and is
 * applied to protons, P:9): projectile[i] = 1 proton, 0 neutron for event i of the NEXT inc_simulate /
 * inc_simulate_host call only (the pointer is dropped when that call returns, so a stale pointer is never read).
 * DEVICE array, caller-owned, at least as long as that call's n_events.  NULL (the default) = all protons.  A neutron enters with its own mass
 * and feels the neutron potential; the residual then has charge Z - n_p instead of Z + 1 - n_p.  Any other
 * value is an input error (INC_E_BADARG, found on the device like E_in out of range). */
int inc_set_projectiles(const uint8_t *projectile /*DEVICE [n] or NULL*/);
/* A call is processed in chunks of at most `n` events (default 2^22; 0 restores it; 1024 .. 2^24): the
 * library's staging workspace is sized for one chunk (16 records of 32 bytes per event in the f32
 * build plus an overflow pool and two 32-byte nucleus records: 2.4 GB at the default) and every chunk is one
 * launch of each kernel, so large chunks mean few tails of the persistent cascade kernel.  Results never
 * depend on it (R-R4). */
int inc_set_chunk_events(int64_t n);
/* Staging overflow pool: an event's first 16 secondaries are staged in its own row, an event with more (up to
 * INC_MAX_SEC) takes one row of a pool that has, by default, a row for one event in 64.  A batch that needs more makes
 * inc_simulate run the call again with a row for every event (inc_get_rerun_count counts it) and keeps that size.
 * `rows` > 0 fixes the pool size (tests use 1 to force that path); 0 restores the default.  Results never depend on it. */
int inc_set_stage_overflow_rows(int64_t rows);
/* Scheduling knob of the default (wavefront) cascade kernel: a track that has run `n_segments`
 * segments may be handed to a warp that has finished its own events, which evaluates 32 consecutive
 * segments of the one track per pass along its collision-free path (drain helpers, DESIGN.md
 * section 6).  0 restores the default (48).  Results never depend on it. */
int inc_set_long_track_threshold(int n_segments);
/* Scheduling knob of the default (wavefront) cascade kernel: a segment pass advances its 32 resident tracks by up to
 * `n` segments (1..8) before the tracks that collided, escaped or were absorbed are handed over and the lanes are
 * refilled.  0 (the default) lets the library choose: 3 while every live target has A <= 20 (a track then continues
 * in ~87 % of its segments), otherwise 2.  Results never depend on it. */
int inc_set_segments_per_pass(int n);
/* Scheduling knob of the default (wavefront) cascade kernel: with `min_events_per_warp` > 0 a warp holds at most its
 * share of the events of the chunk that have not been handed out yet (at least that minimum, at most its slot count), so
 * the last events of a chunk are spread over all warps instead of queueing in the warps that asked first, and a batch
 * smaller than the GPU's slot count (~1.9e5 events) is spread over all SMs from the start.  0 switches it off (every warp
 * fills all its slots while events remain); -1 (the default) lets the library choose: 8 for chunks below 1e5 events (1e4
 * events: 0.51 -> 0.44 ms), off above, where it was measured to change nothing.  Results never depend on it (R-R4). */
int inc_set_event_taper(int min_events_per_warp);
/* Global index of the first event of the following inc_simulate calls (default 0): event i of a
 * call uses the random stream of global event e = offset + i.  This is how a job is sharded over
 * several GPUs or calls with bit-identical per-event results (R-R4). */
int inc_set_event_offset(int64_t first_event);

/* ---- outputs ---------------------------------------------------------------------------- */
typedef struct inc_secondaries { /* DEVICE pointers, caller-owned, structure of arrays  */
  uint8_t *species;              /* 0=n 1=p 2=d 3=t 4=3He 5=4He; bit 7 set = from evaporation */
  INC_REAL *T;                   /* kinetic energy, MeV, lab                                  */
  INC_REAL *ux, *uy, *uz;        /* unit direction                                            */
  int64_t capacity;              /* elements available in each array                          */
} inc_secondaries;

typedef struct inc_residual {    /* DEVICE, structure of arrays of length n_events             */
  int32_t *A, *Z;                /* final residual nucleus                                    */
  INC_REAL *Estar;               /* leftover excitation, MeV (no photon model)          */
  INC_REAL *px, *py, *pz;        /* lab momentum, MeV/c                                       */
  uint32_t *status;              /* INC_ST_* bits                                             */
} inc_residual;

/* inc_simulate — the whole hot path for a batch (INC kernel, evaporation kernel;
 * BASELINE.json north_star: entry, segment, boundary, collision, epilogue, evaporation,
 * prefix-sum compaction).  Event e is a proton of kinetic energy E_in[e] on target
 * target_id[e].  Secondaries of all events are written back to back in event order, inside
 * an event in canonical order: cascade nucleons by ascending path code, then evaporation
 * products in emission order.  out_counts[e] is the number of secondaries of event e.
 * Returns the total number of secondaries (>= 0) or a negative INC_E_* code. */
int64_t inc_simulate(int64_t n_events, const INC_REAL *E_in /*DEVICE, MeV*/,
                     const int32_t *target_id /*DEVICE*/, uint64_t seed,
                     inc_secondaries *out_secondaries /*HOST struct of DEVICE ptrs*/,
                     int32_t *out_counts /*DEVICE [n_events]*/,
                     inc_residual *out_residual /*HOST struct of DEVICE ptrs*/);

/* inc_simulate_host — same computation with HOST buffers (every pointer, including those
 * inside the two structs, is host memory).  It streams: the call runs in chunks of at most
 * 2^19 events (2^20 for calls above 2^21 events; or inc_set_chunk_events, if smaller); chunk c lives in slot c mod 3
 * of a ring of chunk-sized device buffers (inputs, per-event outputs, room for INC_MAX_SEC secondaries per event), so
 * device memory is O(chunk) whatever n_events is; while chunks compute on the caller's stream the outputs of the
 * previous one travel to the host on a second stream, so a long call costs about max(compute, copy) instead of
 * their sum.  Pinned host memory is what makes the copies asynchronous; pageable memory works, without the overlap.
 * After a call of more than one chunk inc_get_offsets and inc_get_cascade_stage return INC_E_STATE (the device holds
 * per-chunk data only; the offsets are the prefix sum of out_counts). */
int64_t inc_simulate_host(int64_t n_events, const INC_REAL *E_in /*HOST*/,
                          const int32_t *target_id /*HOST*/, uint64_t seed,
                          inc_secondaries *out_secondaries /*HOST ptrs*/,
                          int32_t *out_counts /*HOST*/, inc_residual *out_residual /*HOST ptrs*/);

/* Exclusive prefix sum of out_counts of the last inc_simulate: dev_offsets[e] is the index of
 * the first secondary of event e, dev_offsets[n_events] the total. */
int inc_get_offsets(int64_t *dev_offsets /*DEVICE [n_events+1]*/);

/* inc_scan_counts_static — the same exclusive prefix sum (the "prefix-sum" step of the compaction, BASELINE.json
 * north_star) as an entry point that allocates nothing, for callers who cannot let this library call
 * cudaMalloc.  Those are: a host program that has handed all of the device's memory to an arena of its own (a transport
 * Monte Carlo with a fixed budget, or a framework allocator holding the whole GPU), where a cudaMalloc from a library
 * fails or steals from that budget; and a caller inside a latency-critical loop, because cudaMalloc and cudaFree
 * synchronise the whole device and stall every other stream.  (inc_simulate sizes its workspace with cudaMalloc when it
 * first sees a batch size; this call never does, and calls no cudaFree or other allocating routine either.)
 *   counts  DEVICE [n]      per-event numbers of secondaries (e.g. out_counts of inc_simulate), caller-owned, read only;
 *                           a value outside [0, INC_MAX_SEC] is read as the nearer end of that range, as everywhere in the library
 *   offsets DEVICE [n + 1]  caller-owned; offsets[e] = counts[0] + ... + counts[e-1], offsets[n] = the total
 * The scan's scratch (one partial sum per 2048 events and the running total) is a fixed array inside the library,
 * 64.25 KB of device memory that every GPU which loads the library holds until the process exits.  Hence the limit:
 * n <= INC_SCAN_STATIC_MAX_EVENTS; a larger n is refused with INC_E_BADARG and a message, nothing is written.
 * The first call on a device looks up the array's device address (once per device, with the device that is current at
 * the call): make that first call before any stream capture begins.  All calls share the one array and it keeps the
 * previous call's contents (the call clears the one word that must start at zero), so two calls whose kernels
 * overlap on the GPU (issued from two host threads, say) race on it and both results are garbage: serialise them.
 * Work is enqueued on the inc_set_stream stream and the call returns when it has finished.  Needs no
 * inc_init.  Returns 0, INC_E_BADARG or INC_E_CUDA. */
#define INC_SCAN_STATIC_MAX_EVENTS (1 << 24)
int inc_scan_counts_static(int64_t n, const int32_t *counts /*DEVICE [n]*/, int64_t *offsets /*DEVICE [n+1]*/);

/* Post-cascade nuclei of the last inc_simulate (the paper's "SoA of excited nuclei", P:69,
 * P:83), for stage-level tests: any pointer may be NULL; n_cascade_secondaries[e] is the number of
 * cascade nucleons of event e.  Only after a call that ran as ONE chunk (n_events <= the chunk size):
 * the records are per chunk, so after a multi-chunk call this returns INC_E_STATE. */
int inc_get_cascade_stage(int32_t *A /*DEVICE [n]*/, int32_t *Z, INC_REAL *Estar,
                          INC_REAL *px, INC_REAL *py, INC_REAL *pz, int32_t *n_cascade_secondaries);

typedef struct inc_stats {     /* work counters of the last inc_simulate (needs INC_F_STATS)   */
  uint64_t events, failed, attempts, segments, boundaries, reflections, escapes;
  uint64_t collisions, blocked, allowed, absorbed;
  uint64_t evap_steps, evap_trials, evap_emitted;
  uint64_t warp_iters_seg, warp_iters_coll, warp_iters_epi; /* scheduling: phase passes    */
  uint64_t lane_slots_seg, lane_slots_coll, lane_slots_epi; /* active lanes summed over passes */
} inc_stats;
int inc_get_stats(inc_stats *host_out /*HOST*/);

/* Device time of the stages of the last inc_simulate, summed over its chunks, in milliseconds:
 * ms[0] cascade kernel, ms[1] evaporation kernel, ms[2] prefix-sum kernels, ms[3] compaction
 * kernel; launches[0..3] the number of kernel launches of each stage.  Needs INC_F_TIMING. */
int inc_get_stage_times(float ms[4] /*HOST*/, int32_t launches[4] /*HOST*/);

/* Drain timeline of the cascade kernel of the last inc_simulate (last chunk; needs INC_F_TIMING),
 * in milliseconds after the first warp started: ms[0] mean over warps of the moment the event
 * counter ran out for the warp, ms[1] mean warp exit, ms[2] last warp exit, ms[3] first warp
 * exit.  Diagnostic for the tail of the persistent kernel; wavefront
 * kernel only, zeros otherwise. */
int inc_get_drain_timeline(double ms[4] /*HOST*/);

/* Per-warp drain trace of the cascade kernel of the last inc_simulate (last chunk; needs INC_F_TIMING; wavefront
 * kernel only): 8 words per warp -- [0] %globaltimer ns (low 32 bits) when the event counter ran out for the warp,
 * [1] ns when its own work was finished, [2] passes of its drain phase, [3] segment passes among them, [4] active
 * lanes summed over those, [5] highest attempt number started in the drain, [6] tracks handed to drain helpers,
 * [7] ns at kernel entry.  Returns the number of warps written (<= max_warps), 0 if none was recorded.  Diagnostic. */
int inc_get_warp_trace(uint32_t *out /*HOST [8 * max_warps]*/, int32_t max_warps);

/* How many inc_simulate calls so far were run a second time: with the lane-per-event cascade kernel because the
 * wavefront kernel's per-warp track queues overflowed, or with a larger staging overflow pool (implementation limits
 * of the default configuration, never a property of the result: the events are the same).  Diagnostic; expected to
 * stay 0. */
int64_t inc_get_rerun_count(void);

/* Nuclear-setup record of a target, for tests of inc_init (all HOST, fp64, length n_shells
 * except r, V_p, V_n which have n_shells+1; pointers may be NULL). */
int inc_get_nucleus(int target_id, int32_t *A, int32_t *Z, int32_t *n_shells, double *R,
                    double *E_C, double *EB_p, double *EB_n, double *r, double *rho_p,
                    double *rho_n, double *pF_p, double *pF_n, double *EF_p, double *EF_n,
                    double *V_p, double *V_n);

/* Measured peak of the plain-ALU roofline: runs an FFMA (f32) or DFMA (f64) chain kernel at
 * full occupancy on the current stream and returns lane-instructions per second (one FMA =
 * one lane-instruction).  Used by bench.py for roofline.peak. */
int inc_measure_issue_peak(double *lane_instr_per_s /*HOST*/, double *sm_clock_mhz /*HOST, may be NULL*/);

/* Philox4x32-10 block, exposed for the RNG parity test (R-R1): out[4*i..] for counters
 * ctr[4*i..] (DEVICE arrays of n blocks), key = (seed lo, seed hi). */
int inc_philox_blocks(const uint32_t *ctr /*DEVICE [4n]*/, uint64_t seed, uint32_t *out /*DEVICE [4n]*/, int64_t n);

/* ---- on-device tallies --------------------------------------------------
 * The quantities the paper shows for its results: secondary yields and double-differential
 * spectra ("double differential yields at 7.5, 30, 60 and 150 degrees", Figs. 1-2)
 * and the residual nuclides, whose positron emitters are the paper's named application ("very
 * fast calculation of the yield of positron emitters for range verification").  inc_tally
 * reduces the outputs of an inc_simulate call on the device, so that a study needs O(bins) instead
 * of O(events) to come back to the host.  All tallies are unsigned 64-bit counts in DEVICE memory,
 * caller-owned, and are ACCUMULATED into (the caller zeroes them once and may call inc_tally after
 * every batch).  Classes: 0 = neutrons, 1 = protons, 2 = composites (d, t, 3He, 4He).
 *   dd[c][a][t]     c < 3, a < n_cos, t <= n_T : secondaries of class c with
 *                   a = min(floor((uz + 1) * n_cos / 2), n_cos - 1)   (uz = cos of the polar angle to the beam)
 *                   t = min(floor(T * n_T / T_max), n_T)               (t = n_T: overflow T >= T_max)
 *                   both products evaluated in INC_REAL, one rounding each.
 *   mult[c][m]      c < 4 (3 = all secondaries), m <= mult_max: events with min(multiplicity of class c, mult_max) = m
 *   nuclide[A][Z]   A <= A_max, Z <= Z_max: events whose final residual is (A, Z); others are not counted
 *   yield[s][o]     s < 6 species, o = 0 cascade / 1 evaporation (bit 7 of the species byte)
 * Events are all n_events of the call; offsets = exclusive prefix sum of counts ([n_events + 1], e.g. from
 * inc_get_offsets).  Returns 0 or INC_E_BADARG (null pointer, n < 0, non-positive bin counts) / INC_E_CUDA. */
typedef struct inc_tally_spec {
  int32_t n_T; double T_max;     /* energy bins of width T_max / n_T, MeV, plus one overflow bin */
  int32_t n_cos;                 /* bins of cos(theta) on [-1, 1]                                */
  int32_t mult_max;              /* multiplicities are clamped to this                           */
  int32_t A_max, Z_max;          /* extent of the nuclide chart                                  */
} inc_tally_spec;
typedef struct inc_tallies {     /* DEVICE pointers, caller-owned, accumulated                   */
  unsigned long long *dd;        /* [3][n_cos][n_T + 1]                                          */
  unsigned long long *mult;      /* [4][mult_max + 1]                                            */
  unsigned long long *nuclide;   /* [A_max + 1][Z_max + 1]                                       */
  unsigned long long *yield;     /* [6][2]                                                       */
} inc_tallies;
int inc_tally(int64_t n_events, const inc_secondaries *sec /*HOST struct of DEVICE pointers*/,
              const int32_t *counts /*DEVICE [n]*/, const int64_t *offsets /*DEVICE [n+1]*/,
              const inc_residual *res /*HOST struct of DEVICE pointers*/, const inc_tally_spec *spec /*HOST*/,
              const inc_tallies *out /*HOST struct of DEVICE pointers*/);

const char *inc_last_error(void);
const char *inc_build_info(void);   /* "f32 fast-math sm_100a ..." */

#ifdef __cplusplus
}
#endif
#endif
