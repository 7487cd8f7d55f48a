// inc_device.cuh — sm_100a device code of the INC + evaporation hot path (arXiv:1309.7963).
//
// Shares nothing with oracle/.  Templated on the real type R (float: production build,
// double: parity build compiled with -fmad=false).  Citations: P:NN = PAPER.md line,
// R-xx = reading in DESIGN.md section 3.
//
// Physics steps (device functions, used by both cascade kernels)
//   entry_step      C0  uniform-disc entry, potential step into the outermost shell
//   seg_step        C2  Fermi-sea partner, NN cross sections, exponential path, shell geometry,
//                   C4  refraction / reflection / escape at the shell boundary
//   coll_step       C3  relativistic two-body scatter, Pauli blocking, cutoff
//   epilogue_eval   C6  residual nucleus and excitation energy from 4-momentum balance
// Kernels
//   cascade_wavefront_kernel  DEFAULT.  Per-warp wavefront: tracks of ~80 events in flight live in
//                   per-warp shared-memory queues, sorted by the kind of step they need next
//                   (segment / collision / epilogue+entry).  Every warp pass pops up to 32 items of
//                   ONE kind, so lanes execute the same step; queue indices come from warp votes
//                   (__ballot_sync + popc), per-event bookkeeping from shared-memory integer atomics.
//   cascade_lane_kernel       INC_F_LANE_STATE_MACHINE.  One lane owns one event at a time and runs a
//                   {SEG, COLL, EPI} state machine; the warp votes which phase to run each pass.
//   evap_kernel     persistent lanes, one Weisskopf-Ewing emission step per pass.
//   scan_* / compact_kernel   exclusive prefix sum of counts, canonical-order SoA output.
// Files: inc_common.cuh (model data, records, math, Philox), inc_physics.cuh (the steps), inc_cascade_lane.cuh,
// inc_cascade_wavefront.cuh, inc_evap.cuh, inc_output.cuh; this header includes them in that order.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <type_traits>

#include "../../include/inc.h"

// -DINC_CHECKED: every index into the wavefront kernel's shared-memory queues, rings and slot lists is checked and a
// violation raises error bit 32 (inc_simulate -> INC_E_STATE).  compute-sanitizer is closed on the GPU pool this was
// developed on, so the checked small-queue build (libinc_f64q.so) is the memory check of the queue code.
#ifdef INC_CHECKED
#define INC_CHECK(cond) do { if (!(cond)) atomicOr(&P.ctr->error_word, 32u); } while (0)
#else
#define INC_CHECK(cond) do { } while (0)
#endif


#include "inc_common.cuh"
#include "inc_physics.cuh"
#include "inc_cascade_lane.cuh"
#include "inc_cascade_wavefront.cuh"
#include "inc_evap.cuh"
#include "inc_output.cuh"
