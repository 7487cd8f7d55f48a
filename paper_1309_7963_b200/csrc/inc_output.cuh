// inc_output.cuh — exclusive prefix sum of the counts, canonical-order compaction, on-device tallies, the unpack kernel
// of inc_get_cascade_stage, the issue-peak microbenchmark and the Philox test hook.  Part of inc_device.cuh.
#pragma once

namespace inc {

// =================================================================================================
// Output: exclusive prefix sum of the per-event counts, then canonical-order SoA compaction
// (BASELINE.json north_star "prefix-sum compaction of variable-length secondary lists into
// coalesced SoA buffers").
// =================================================================================================
constexpr int kScanBlock = 256;
constexpr int kScanItems = 8;                       // per thread
constexpr int kScanTile = kScanBlock * kScanItems;  // 2048 events per block

// A per-event count as the scan and the compaction read it: the counts array is caller memory, and a value outside
// [0, kMaxSec] (an event the evaporation kernel never reached after an abandoned cascade launch, a caller's stale
// buffer) must not turn into a huge or negative offset: those would send the compaction outside the staging workspace
// or in front of the caller's arrays.
__device__ __forceinline__ int clamp_count(int c) { return c < 0 ? 0 : (c > kMaxSec ? kMaxSec : c); }

__device__ __forceinline__ long long block_exclusive_scan(long long v, long long *s_warp, long long &block_total) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  long long incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    long long t = __shfl_up_sync(kFull, incl, o);
    if (lane >= o) incl += t;
  }
  if (lane == 31) s_warp[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    long long w = lane < (kScanBlock / 32) ? s_warp[lane] : 0;
    long long wi = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      long long t = __shfl_up_sync(kFull, wi, o);
      if (lane >= o) wi += t;
    }
    if (lane < (kScanBlock / 32)) s_warp[lane] = wi - w;
    if (lane == (kScanBlock / 32) - 1) s_warp[kScanBlock / 32] = wi;
  }
  __syncthreads();
  block_total = s_warp[kScanBlock / 32];
  return incl - v + s_warp[wid];
}

// pass 1: per-tile sums
__global__ void __launch_bounds__(kScanBlock) scan_tile_sums(const int32_t *counts, int n, long long *tile_sums) {
  __shared__ long long s_warp[kScanBlock / 32 + 1];
  const int base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
  long long v = 0;
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) if (base + i < n) v += clamp_count(counts[base + i]);
  long long total;
  block_exclusive_scan(v, s_warp, total);
  if (threadIdx.x == 0) tile_sums[blockIdx.x] = total;
}

// pass 2: one block scans the tile sums (n_tiles <= 2^20/2048 * ... loop) and adds the running base
__global__ void __launch_bounds__(kScanBlock) scan_tiles(long long *tile_sums, int n_tiles, unsigned long long *running_total) {
  __shared__ long long s_warp[kScanBlock / 32 + 1];
  __shared__ long long s_carry;
  if (threadIdx.x == 0) s_carry = (long long)*running_total;
  __syncthreads();
  for (int b = 0; b < n_tiles; b += kScanBlock) {
    const int i = b + threadIdx.x;
    const long long v = i < n_tiles ? tile_sums[i] : 0;
    long long total;
    const long long ex = block_exclusive_scan(v, s_warp, total);
    const long long carry = s_carry;
    if (i < n_tiles) tile_sums[i] = carry + ex;
    __syncthreads();
    if (threadIdx.x == 0) s_carry = carry + total;
    __syncthreads();
  }
  if (threadIdx.x == 0) *running_total = (unsigned long long)s_carry;
}

// pass 3: offsets[e] = tile base + exclusive scan inside the tile
__global__ void __launch_bounds__(kScanBlock) scan_write_offsets(const int32_t *counts, int n, const long long *tile_sums,
                                                                 long long *offsets) {
  __shared__ long long s_warp[kScanBlock / 32 + 1];
  const int base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
  int c[kScanItems];
  long long v = 0;
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) { c[i] = base + i < n ? clamp_count(counts[base + i]) : 0; v += c[i]; }
  long long total;
  long long ex = block_exclusive_scan(v, s_warp, total) + tile_sums[blockIdx.x];
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) {
    if (base + i < n) offsets[base + i] = ex;
    ex += c[i];
  }
}

template <typename R> struct CompactParams {
  Workspace<R> ws;
  const long long *offsets;   // chunk-local array of global output offsets
  const int32_t *counts;
  int n_chunk;
  uint8_t *species;
  R *T, *ux, *uy, *uz;
  long long capacity;
  // residual of the caller (chunk base): transposed from ws.frec
  int32_t *rA, *rZ;
  R *rE, *rPx, *rPy, *rPz;
  uint32_t *rstatus;
};

// One warp per group of 32 events; lanes sweep the records of each event so that the stores of a
// warp cover one contiguous span of the output arrays.  Cascade records are placed by the rank of
// their path code (canonical order), evaporation records keep their emission order.
template <typename R>
__global__ void __launch_bounds__(256) compact_kernel(const CompactParams<R> P) {
  const int lane = threadIdx.x & 31;
  const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int e0 = warp * 32;
  if (e0 >= P.n_chunk) return;
  const int e = e0 + lane;
  long long off = 0;
  int cnt = 0, ncs = 0, oid = -1;
  if (e < P.n_chunk) {
    off = P.offsets[e]; cnt = clamp_count(P.counts[e]);
    if (cnt > kStageMain) oid = P.ws.ovf_id[e];     // records beyond the event's own row sit in its overflow row
    const NucRec<R> r = P.ws.frec[e];
    ncs = (int)((r.meta >> 8) & 0xFFu);             // cascade secondaries of event e (frec.meta = count | n_casc << 8)
    P.rA[e] = r.A; P.rZ[e] = r.Z; P.rE[e] = r.E; P.rPx[e] = r.Px; P.rPy[e] = r.Py; P.rPz[e] = r.Pz; P.rstatus[e] = r.status;
  }
  // flatten (event, record) pairs of the 32 events over the lanes
  int incl = cnt;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int t = __shfl_up_sync(kFull, incl, o);
    if (lane >= o) incl += t;
  }
  const int total = __shfl_sync(kFull, incl, 31);
  const int excl = incl - cnt;
  for (int i0 = 0; i0 < total; i0 += 32) {
    const int i = i0 + lane;
    // find the event: largest l with excl_l <= i  (binary search over the 32 lanes' excl via shuffles)
    int lo = 0;
#pragma unroll
    for (int step = 16; step > 0; step >>= 1) {
      const int cand = lo + step;
      const int ex_c = __shfl_sync(kFull, excl, cand & 31);
      if (cand < 32 && ex_c <= i) lo = cand;
    }
    const int ex_l = __shfl_sync(kFull, excl, lo);
    const long long off_l = __shfl_sync(kFull, off, lo);
    const int n_casc = __shfl_sync(kFull, ncs, lo);
    int oid_l = __shfl_sync(kFull, oid, lo);
    // (a missing overflow row -- pool exhausted, error bit 64, the call is run again -- reads row 0: nothing faults)
    oid_l = (oid_l >= 0 && oid_l < P.ws.ovf_rows) ? oid_l : 0;
    if (i < total) {
      const int el = e0 + lo;
      const int j = i - ex_l;
      const StageRec<R> rec = *stage_at<R>(P.ws, el, j, oid_l);
      const uint32_t code = rec.code;
      int rank = j;
      uint8_t sp;
      if (code & 0x80000000u) {
        sp = (uint8_t)(0x80u | ((code >> 24) & 0x7u));
      } else {
        sp = (uint8_t)((code >> 24) & 1u);
        const uint32_t key = code & 0xFFFFFFu;
        rank = 0;
        for (int l = 0; l < n_casc; ++l) rank += ((stage_at<R>(P.ws, el, l, oid_l)->code & 0xFFFFFFu) < key) ? 1 : 0;
      }
      const long long dst = off_l + rank;
      if (dst >= 0 && dst < P.capacity) {
        P.species[dst] = sp;
        P.T[dst] = rec.T; P.ux[dst] = rec.ux; P.uy[dst] = rec.uy; P.uz[dst] = rec.uz;
      }
    }
  }
}

// =================================================================================================
// On-device tallies (inc_tally): double-differential spectra per
// class, multiplicities, residual nuclide chart, yields.  One thread per event (grid-stride); each block
// histograms into 32-bit shared-memory bins and adds its non-zero bins to the caller's 64-bit tallies at the end
// (smem = 0: straight to the global tallies, for bin counts that do not fit in shared memory).
// =================================================================================================
template <typename R> struct TallyParams {
  const uint8_t *species; const R *T, *uz;
  const int32_t *counts; const long long *offsets;
  const int32_t *rA, *rZ;
  long long n_events;
  int n_T, n_cos, mult_max, A_max, Z_max;
  R T_scale, cos_scale;          // n_T / T_max and n_cos / 2, rounded once to R
  unsigned long long *dd, *mult, *nuclide, *yield;
  int smem;                      // 1 = shared-memory bins
};

template <typename R>
__global__ void __launch_bounds__(256) tally_kernel(const TallyParams<R> P) {
  extern __shared__ unsigned int s_bins[];
  const int n_dd = 3 * P.n_cos * (P.n_T + 1), n_mult = 4 * (P.mult_max + 1), n_nuc = (P.A_max + 1) * (P.Z_max + 1);
  const int o_mult = n_dd, o_nuc = n_dd + n_mult, o_y = o_nuc + n_nuc, n_all = o_y + 12;
  if (P.smem) {
    for (int i = threadIdx.x; i < n_all; i += blockDim.x) s_bins[i] = 0u;
    __syncthreads();
  }
  auto bump = [&](int bin) {
    if (P.smem) atomicAdd(&s_bins[bin], 1u);
    else {
      unsigned long long *g = bin < o_mult ? P.dd + bin : bin < o_nuc ? P.mult + (bin - o_mult)
                            : bin < o_y ? P.nuclide + (bin - o_nuc) : P.yield + (bin - o_y);
      atomicAdd(g, 1ull);
    }
  };
  for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < P.n_events; e += (long long)gridDim.x * blockDim.x) {
    const long long b = P.offsets[e];
    const int n = P.counts[e];
    int m[3] = {0, 0, 0};
    for (int k = 0; k < n; ++k) {
      const unsigned sp = P.species[b + k];
      const int code = (int)(sp & 0x7u);
      const int c = code < 2 ? code : 2;
      m[c]++;
      int a = (int)((P.uz[b + k] + R(1)) * P.cos_scale);
      a = a < 0 ? 0 : (a > P.n_cos - 1 ? P.n_cos - 1 : a);
      const R tt = P.T[b + k] * P.T_scale;
      int t = tt >= R(P.n_T) ? P.n_T : (int)tt;
      t = t < 0 ? 0 : t;
      bump((c * P.n_cos + a) * (P.n_T + 1) + t);
      if (code < 6) bump(o_y + code * 2 + (int)(sp >> 7));
    }
    const int mm = P.mult_max;
    bump(o_mult + 0 * (mm + 1) + (m[0] < mm ? m[0] : mm));
    bump(o_mult + 1 * (mm + 1) + (m[1] < mm ? m[1] : mm));
    bump(o_mult + 2 * (mm + 1) + (m[2] < mm ? m[2] : mm));
    bump(o_mult + 3 * (mm + 1) + (n < mm ? n : mm));
    const int A = P.rA[e], Z = P.rZ[e];
    if (A >= 0 && A <= P.A_max && Z >= 0 && Z <= P.Z_max) bump(o_nuc + A * (P.Z_max + 1) + Z);
  }
  if (P.smem) {
    __syncthreads();
    for (int i = threadIdx.x; i < n_all; i += blockDim.x) {
      const unsigned int v = s_bins[i];
      if (v) {
        unsigned long long *g = i < o_mult ? P.dd + i : i < o_nuc ? P.mult + (i - o_mult)
                              : i < o_y ? P.nuclide + (i - o_nuc) : P.yield + (i - o_y);
        atomicAdd(g, (unsigned long long)v);
      }
    }
  }
}

// post-cascade records -> parallel arrays (inc_get_cascade_stage); any pointer may be null
template <typename R>
__global__ void unpack_cascade_kernel(const NucRec<R> *rec, long long n, int32_t *A, int32_t *Z, R *E, R *px, R *py, R *pz, int32_t *ncs) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const NucRec<R> r = rec[i];
  if (A) A[i] = r.A;
  if (Z) Z[i] = r.Z;
  if (E) E[i] = r.E;
  if (px) px[i] = r.Px;
  if (py) py[i] = r.Py;
  if (pz) pz[i] = r.Pz;
  if (ncs) ncs[i] = (int32_t)(r.meta & 0xFFu);
}

// ---- issue-peak microbenchmark: 8 independent FMA chains per thread ------------------------------
template <typename R>
__global__ void __launch_bounds__(256) fma_peak_kernel(R *out, int iters, R a, R b) {
  R v0 = R(threadIdx.x) * R(1e-3), v1 = v0 + R(1), v2 = v0 + R(2), v3 = v0 + R(3);
  R v4 = v0 + R(4), v5 = v0 + R(5), v6 = v0 + R(6), v7 = v0 + R(7);
#pragma unroll 1
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      v0 = fma(v0, a, b); v1 = fma(v1, a, b); v2 = fma(v2, a, b); v3 = fma(v3, a, b);
      v4 = fma(v4, a, b); v5 = fma(v5, a, b); v6 = fma(v6, a, b); v7 = fma(v7, a, b);
    }
  }
  R s = v0 + v1 + v2 + v3 + v4 + v5 + v6 + v7;
  if (s == R(123456.789)) out[0] = s;
}

__global__ void philox_blocks_kernel(const uint32_t *ctr, uint32_t *out, long long n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint4 o = philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3]);
  out[4 * i] = o.x; out[4 * i + 1] = o.y; out[4 * i + 2] = o.z; out[4 * i + 3] = o.w;
}

}  // namespace inc
