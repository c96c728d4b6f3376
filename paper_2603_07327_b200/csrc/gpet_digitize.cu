// gpet_digitize.cu -- singles digitizer and coincidence sorter (S11..S14 of DESIGN.md section 1).
// PAPER.md:33,37 (single-event readout at crystal / module / panel level), PAPER.md:61 (energy resolution,
// coincidence timing window), PAPER.md:65 (list-mode coincidences).  Readings [R16], [R24]-[R27].
//
// Sort / segmented-scan structure (all hand-written, no CUB/Thrust):
//   1. sort of the hits by history id: per 512-pair chunk in shared memory (chunked hit layout: gpet_simulate writes the hits
//      of a chunk into the chunk's own region), or, for hits in any order, a counting sort through HBM (histogram by L2
//      atomics whose return value is the hit's rank in its history, single-pass look-back scan, scatter of 32-byte records);
//   2. adder: one thread per hit, the leader of each (history, readout unit) group sums the group in order-free fixed
//      point, then blur, window, absolute time -> kept singles;
//   3. time sort.  Coarse buckets (the batch's decay times are uniform over its time range [R16]): a kept single goes
//      straight into the region of its bucket, a scan of the fill counts gives the offsets, one block per group of buckets
//      sorts the regions in shared memory.  Fine buckets (any distribution): counted by the adder, scanned, scattered,
//      ranked inside the bucket;
//   4. coincidences: a thread per cluster start (gap >= tau) walks its cluster with the window rule [R27] and flags the
//      accepted pairs, counted per tile; scan over the tiles; block scan + one list-mode record per flagged single.
// Every stage is deterministic: the output does not depend on the order of the hit buffer.
#include <cmath>
#include <cstring>
#include <mutex>
#include "../../include/gpet.h"
#include "gpet_internal.h"

namespace gpet {

constexpr int kItems = 16;       // elements per thread of a scan tile (four 16-byte loads)
constexpr int kTile = 256 * kItems;

// ---------------------------------------------------------------- device-wide exclusive scan (u32)
template <int NW>
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t *total) {
  __shared__ uint32_t warp_sum[NW];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint32_t inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o); if (lane >= o) inc += t; }
  __syncthreads();                         // protect warp_sum reuse across calls
  if (lane == 31) warp_sum[wid] = inc;
  __syncthreads();
  uint32_t base = 0, tot = 0;
#pragma unroll
  for (int w = 0; w < NW; ++w) { const uint32_t s = warp_sum[w]; if (w < wid) base += s; tot += s; }
  *total = tot;
  return base + inc - v;
}
__device__ __forceinline__ uint32_t block_exclusive_scan_256(uint32_t v, uint32_t *total) { return block_exclusive_scan<8>(v, total); }

// Decoupled look-back of one tile, run by warp 0 of the tile's block: publishes the tile's aggregate `tot` (flag 1), adds up
// the aggregates of the preceding tiles 32 at a time until one that already knows its inclusive prefix (flag 2), publishes
// this tile's inclusive prefix and returns the exclusive one.  state: [0] ticket counter, [1 + tile] = flag << 62 | value.
__device__ __forceinline__ uint32_t lookback_prefix(unsigned long long *state, uint32_t tile, uint32_t tot) {
  volatile unsigned long long *st = state + 1;
  const int lane = threadIdx.x & 31;
  uint32_t prefix = 0;
  if (tile > 0) {
    if (lane == 0) st[tile] = (1ull << 62) | tot;
    for (int j = (int)tile - 1;; j -= 32) {
      const int jj = j - lane;
      unsigned long long w = 2ull << 62;                              // before tile 0: an inclusive prefix of 0
      if (jj >= 0) do { w = st[jj]; } while ((w >> 62) == 0ull);
      const unsigned incl = __ballot_sync(0xFFFFFFFFu, (w >> 62) == 2ull);
      const int first = incl ? __ffs(incl) - 1 : 31;                  // nearest predecessor that already knows its prefix
      uint32_t part = lane <= first ? (uint32_t)w : 0u;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xFFFFFFFFu, part, o);
      prefix += part;
      if (incl) break;
    }
  }
  if (lane == 0) st[tile] = (2ull << 62) | (unsigned long long)(prefix + tot);
  return prefix;
}

// Single-pass exclusive scan with decoupled look-back (one read and one write of the data).  Tiles take tickets
// from an atomic counter, so a tile only ever waits for tiles that are already running or done; a tile publishes
// its aggregate (flag 1) as soon as it is known and its inclusive prefix (flag 2) after the look-back.
// out[i] = sum of in[0..i), out[n] = total; n = min(*n_dev, n_host) when n_dev is given (lengths known only on
// the device).  state: [0] ticket counter, [1 + tile] = flag << 62 | value; zeroed by the caller.
__global__ void __launch_bounds__(256) scan_lookback_kernel(const uint32_t *in, uint64_t n_host, const uint32_t *n_dev, uint32_t *out,
                                                            unsigned long long *state, unsigned long long *total_out) {
  __shared__ uint32_t s_tile, s_prefix;
  if (threadIdx.x == 0) s_tile = (uint32_t)atomicAdd(&state[0], 1ull);
  __syncthreads();
  const uint32_t tile = s_tile;
  uint64_t n = n_host;
  if (n_dev) { const uint64_t nd = *n_dev; if (nd < n) n = nd; }
  const uint32_t ntiles = n ? (uint32_t)((n + kTile - 1) / kTile) : 1u;
  if (tile >= ntiles) return;
  const uint64_t base = (uint64_t)tile * kTile + (uint64_t)threadIdx.x * kItems;
  uint32_t v[kItems], s = 0;
  if (base + kItems <= n) {
#pragma unroll
    for (int q = 0; q < kItems / 4; ++q) {
      const uint4 a = *reinterpret_cast<const uint4 *>(in + base + 4 * q);
      v[4 * q] = a.x; v[4 * q + 1] = a.y; v[4 * q + 2] = a.z; v[4 * q + 3] = a.w;
    }
  } else {
#pragma unroll
    for (int k = 0; k < kItems; ++k) v[k] = base + k < n ? in[base + k] : 0u;
  }
#pragma unroll
  for (int k = 0; k < kItems; ++k) s += v[k];
  uint32_t tot; uint32_t ex = block_exclusive_scan_256(s, &tot);
  if (threadIdx.x < 32) {                                            // warp 0: publish, then look back 32 tiles at a time
    const uint32_t prefix = lookback_prefix(state, tile, tot);
    if (threadIdx.x == 0) {
      s_prefix = prefix;
      if (tile == ntiles - 1) { out[n] = prefix + tot; if (total_out) *total_out = prefix + tot; }
    }
  }
  __syncthreads();
  ex += s_prefix;
  if (base + kItems <= n) {
#pragma unroll
    for (int q = 0; q < kItems / 4; ++q) {
      uint4 a;
      a.x = ex; ex += v[4 * q]; a.y = ex; ex += v[4 * q + 1]; a.z = ex; ex += v[4 * q + 2]; a.w = ex; ex += v[4 * q + 3];
      *reinterpret_cast<uint4 *>(out + base + 4 * q) = a;
    }
  } else {
#pragma unroll
    for (int k = 0; k < kItems; ++k) { if (base + k < n) out[base + k] = ex; ex += v[k]; }
  }
}

static cudaError_t exclusive_scan(const uint32_t *in, uint64_t n_host, const uint32_t *n_dev, uint32_t *out, unsigned long long *state,
                                  unsigned long long *total_out, cudaStream_t st) {
  const uint32_t nb = n_host ? (uint32_t)((n_host + kTile - 1) / kTile) : 1u;
  scan_lookback_kernel<<<nb, 256, 0, st>>>(in, n_host, n_dev, out, state, total_out);
  count_launch(1);
  return cudaGetLastError();
}

// ---------------------------------------------------------------- records
// Both intermediate record types are 32 bytes = one DRAM sector, so that the scattered accesses of the two
// counting sorts move whole sectors and every later pass reads contiguous memory.
struct HitRec { uint32_t ids; float x, y, z; float e, tof; uint32_t idx, pad; };            // one hit, grouped by history (pad = history - first)
struct SinRec { double t; uint32_t history, ids; float x, y, z, e; };                      // one kept single
static_assert(sizeof(HitRec) == 32 && sizeof(SinRec) == 32, "records must be one 32-byte sector");

__device__ __forceinline__ void store_rec(void *dst, const void *src) {
  const uint4 *s = reinterpret_cast<const uint4 *>(src); uint4 *d = reinterpret_cast<uint4 *>(dst);
  d[0] = s[0]; d[1] = s[1];
}

// ---------------------------------------------------------------- stage 1: counting sort by history
__device__ __forceinline__ uint32_t valid_hits(const HitBuf &H, uint32_t bound) {
  const unsigned long long n = *H.n_hits, c = H.capacity < bound ? H.capacity : bound;
  return (uint32_t)(n < c ? n : c);
}
// the atomic's return value is the hit's rank inside its history: kept (coalesced) so that the scatter needs no atomics
__global__ void __launch_bounds__(256) count_hits_kernel(HitBuf H, uint32_t bound, uint32_t first_lo, uint32_t n_pairs, uint32_t *cnt, uint32_t *hrank) {
  const uint32_t n_hits = valid_hits(H, bound); const uint32_t *history = H.history;
  for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < n_hits; i += gridDim.x * 256u) {
    const uint32_t h = history[i] - first_lo;
    if (h < n_pairs) hrank[i] = atomicAdd(&cnt[h], 1u);
  }
}
// reads the struct-of-arrays hit buffer coalesced, writes each hit as one sector into its history's segment
__global__ void __launch_bounds__(256) scatter_hits_kernel(HitBuf H, uint32_t bound, uint32_t first_lo, uint32_t n_pairs,
                                                           const uint32_t *off, const uint32_t *hrank, HitRec *rec) {
  const uint32_t n_hits = valid_hits(H, bound);
  for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < n_hits; i += gridDim.x * 256u) {
    const uint32_t h = H.history[i] - first_lo;
    if (h >= n_pairs) continue;
    HitRec r; r.ids = H.ids[i]; r.x = H.x[i]; r.y = H.y[i]; r.z = H.z[i]; r.e = H.e[i]; r.tof = H.tof[i]; r.idx = i; r.pad = h;
    store_rec(&rec[off[h] + hrank[i]], &r);
  }
}

// ---------------------------------------------------------------- stage 2: adder + blur + window + time
// Time buckets of a batch: nb equal intervals of [t_lo, t_hi).  Two uses.  FINE buckets (cap = 0; about one kept single
// each): counted while the adder appends its singles, then a counting sort (scan, scatter, rank inside the bucket).
// COARSE buckets (cap > 0; the decay times of a batch are uniform by construction [R16], so a bucket sized for a mean of
// kCoarseMean singles never sees more than cap): the adder writes each kept single straight into its bucket's region of
// cap records, and one block per group of buckets sorts the regions in shared memory -- no scatter pass through HBM.
struct Buckets { double t_lo, scale; uint32_t nb, cap; uint32_t *dropped; };   // dropped: kept singles that found their coarse bucket full (zeroed per call)
constexpr uint32_t kCoarseMean = 512, kCoarseCap = 832, kSubBuckets = 1024;   // cap = mean + 14 sigma of a Poisson count
__device__ __forceinline__ double bucket_coord(const Buckets &B, double t) { return __dmul_rn(__dsub_rn(t, B.t_lo), B.scale); }   // monotonic in t
__device__ __forceinline__ uint32_t bucket_of(const Buckets &B, double t) {
  const double x = bucket_coord(B, t);
  if (!(x > 0.0)) return 0u;
  return x >= (double)(B.nb - 1) ? B.nb - 1 : (uint32_t)x;
}

// [R34] ln(z), z in (0, 1], and ln(1 - y), y in [0, 1), from IEEE +, -, *, / only (round-to-nearest intrinsics: no FMA
// contraction, no library logarithm), operation for operation what the fp64 reference definition does, so that decay
// times come out bit-identical on both sides.  z = m 2^e, m in [sqrt(1/2), sqrt(2)); ln m = 2 atanh((m-1)/(m+1)).
__host__ __device__ inline double det_series(double s) {
#ifdef __CUDA_ARCH__
  const double s2 = __dmul_rn(s, s); double p = 1.0 / 25.0;
  for (int k = 23; k >= 1; k -= 2) p = __dadd_rn(__dmul_rn(p, s2), 1.0 / (double)k);
  return __dmul_rn(__dmul_rn(2.0, s), p);
#else
  volatile double s2 = s * s; volatile double p = 1.0 / 25.0;       // volatile: keep the host compiler from contracting
  for (int k = 23; k >= 1; k -= 2) { volatile double t = p * s2; p = t + 1.0 / (double)k; }
  volatile double t2 = 2.0 * s; return t2 * p;
#endif
}
__host__ __device__ inline double det_log(double z) {
#ifdef __CUDA_ARCH__
  unsigned long long bits = (unsigned long long)__double_as_longlong(z);
#else
  unsigned long long bits; memcpy(&bits, &z, 8);
#endif
  int e = (int)((bits >> 52) & 0x7FF) - 1022;
  bits = (bits & 0x000FFFFFFFFFFFFFull) | 0x3FE0000000000000ull;
#ifdef __CUDA_ARCH__
  double m = __longlong_as_double((long long)bits);
  if (m < 0.70710678118654752440) { m = __dmul_rn(m, 2.0); e -= 1; }
  const double s = __ddiv_rn(__dsub_rn(m, 1.0), __dadd_rn(m, 1.0));
  return __dadd_rn(__dmul_rn((double)e, 0.69314718055994530942), det_series(s));
#else
  double m; memcpy(&m, &bits, 8);
  if (m < 0.70710678118654752440) { m = m * 2.0; e -= 1; }
  volatile double num = m - 1.0, den = m + 1.0; volatile double s = num / den;
  volatile double a = (double)e * 0.69314718055994530942; return a + det_series(s);
#endif
}
__host__ __device__ inline double det_log1m(double y) {
  if (y < 0.25) {
#ifdef __CUDA_ARCH__
    return det_series(__ddiv_rn(-y, __dsub_rn(2.0, y)));
#else
    volatile double den = 2.0 - y; volatile double s = -y / den; return det_series(s);
#endif
  }
#ifdef __CUDA_ARCH__
  return det_log(__dsub_rn(1.0, y));
#else
  volatile double z = 1.0 - y; return det_log(z);
#endif
}
// [R16] t0 = (slice + u53) B / A; [R34] with a half-life: t0 = -ln(1 - q P) / lambda, q = (slice + u53 f) B / N, f = 1 but
// for a last slice cut short by the end of the run, which covers only (N mod B) / B of a slice (q <= 1, t0 <= T)
__host__ __device__ inline double decay_time_of(const DigiParams &P, double slice_plus_u) {
#ifdef __CUDA_ARCH__
  if (P.lambda > 0.0) return __ddiv_rn(-det_log1m(__dmul_rn(__dmul_rn(slice_plus_u, P.q_scale), P.pfrac)), P.lambda);
  return __dmul_rn(slice_plus_u, P.slice_s);
#else
  if (P.lambda > 0.0) { volatile double q = slice_plus_u * P.q_scale; volatile double y = q * P.pfrac; return -det_log1m(y) / P.lambda; }
  return slice_plus_u * P.slice_s;
#endif
}
// u53 of [R16]: words 8, 9 of the history's source stream (block 2)
__device__ __forceinline__ double decay_u53(const DigiParams &P, uint64_t history) {
  const uint4 w = philox4x32_10(make_uint4((uint32_t)history, (uint32_t)(history >> 32), 0u, 2u), P.keys);
  const uint64_t bits = (((uint64_t)w.x << 32) | (uint64_t)w.y) >> 11;
  return __dmul_rn(__dadd_rn((double)bits, 0.5), 1.0 / 9007199254740992.0);
}
__device__ __forceinline__ double slice_plus_u(const DigiParams &P, uint64_t slice, double u53) {
  const double f = (P.lambda > 0.0 && slice == P.cut_slice) ? P.cut_frac : 1.0;    // u53 * 1.0 is exact: full slices as before
  return __dadd_rn((double)slice, __dmul_rn(u53, f));
}
__device__ __forceinline__ double decay_time(const DigiParams &P, uint64_t history) {
  const uint64_t B = P.pairs_per_slice;
  const uint64_t slice = history < B ? 0ull : history / B;
  return decay_time_of(P, slice_plus_u(P, slice, decay_u53(P, history)));
}

// [R25] standard normal by Box-Muller.  The blurred energy must stay within 1e-3 keV of the fp64 oracle's: sigma is
// ~33 keV, so n needs 3e-5 absolute.  lg2.approx is good to ~1e-7 absolute in ln u, i.e. 0.7e-7 / sqrt(|ln u|) in n:
// fine below u = 0.999, and the accurate logf takes the rest (1 draw in 1000); cos.approx on [-pi, pi] is good to 4e-7.
__device__ __forceinline__ float box_muller(float u0, float u1) {
  const float l = u0 < 0.999f ? __logf(u0) : logf(u0);
  float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(-2.0f * l));
  return -r * __cosf(6.283185307179586f * (u1 - 0.5f));              // cos(2 pi u) = -cos(2 pi u - pi)
}

// a deposit in 2^-40 keV fixed point: e 2^40 is exact in fp32 (a power-of-two scaling), so the rounding to an integer is
// the only one -- the same value the fp64 product rounds to
__device__ __forceinline__ long long deposit_fixed(float e) { return __float2ll_rn(e * 1099511627776.0f); }

// coarse buckets: the kept single goes to the next free record of its bucket's region.  A region does not fill while the
// batch's times are uniform over its range (see Buckets); if one does, the single is dropped, the fill count put back (the
// later passes see min(fill, cap)) and the drop COUNTED: the call then reports both list lengths as UINT64_MAX (gpet.h).
__device__ __forceinline__ void emit_coarse(const Buckets &B, const SinRec &s, SinRec *regions, uint32_t *fill) {
  const uint32_t b = bucket_of(B, s.t), pos = atomicAdd(&fill[b], 1u);
  if (pos < B.cap) store_rec(&regions[(size_t)b * B.cap + pos], &s);
  else { atomicSub(&fill[b], 1u); atomicAdd(B.dropped, 1u); }
}

// records per block of the adder / bucket-scatter pair: the same split in both kernels, a multiple of the block size
__device__ __forceinline__ uint32_t region_size(uint32_t n, uint32_t blocks) {
  return (uint32_t)(((((unsigned long long)n + blocks - 1) / blocks) + 255ull) & ~255ull);
}

// One thread per hit record (a thread per history would idle on the ~54 % of histories without hits).  The record with
// the smallest (ids, position) of its (history, readout unit) group is the group's leader: one pass over the history's
// segment gives it the energy sum, the largest deposit (tie: lowest (photon, seq)) and the earliest time [R24].  The
// sum is formed in 2^-40 keV fixed point (int64): exact integer addition, so it does not depend on the order of the
// hit buffer, and it differs from the exact sum by < 2^-36 keV.  Leaders then blur [R25], window [R26] and time
// [R16] their single.  Block b owns the records [b R, (b+1) R) and appends its kept singles at sing[b R ...] through a
// shared-memory counter (one shared atomic per warp, no block barrier in the loop, no global append counter); the
// per-block counts go to kcnt[].  Each kept single is counted into its time bucket (the atomic's return value is its
// rank in the bucket).  The append order is free: the bucket sort fixes it.
__global__ void __launch_bounds__(256) adder_kernel(DigiParams P, Buckets B, uint64_t first_history, const uint32_t *off, const uint32_t *n_rec,
                                                    const HitRec *rec, SinRec *sing, uint32_t *srank, uint32_t *kcnt, uint32_t *bcnt) {
  __shared__ uint32_t s_cnt;
  const uint32_t n = *n_rec, R = region_size(n, gridDim.x), r0 = blockIdx.x * R;
  const int lane = threadIdx.x & 31;
  if (threadIdx.x == 0) s_cnt = 0;
  __syncthreads();
  for (uint32_t it = 0; it < R && r0 + it < n; it += 256u) {
    const uint32_t i = r0 + it + threadIdx.x;
    bool keep = false; SinRec s;
    if (i < n) {
      const uint4 me = *reinterpret_cast<const uint4 *>(&rec[i]);      // ids, x, y, z
      const uint4 m2 = *(reinterpret_cast<const uint4 *>(&rec[i]) + 1);  // e, tof, idx, history - first
      const uint32_t my_ids = me.x, h = m2.w, b = off[h], k = off[h + 1] - b, unit = my_ids >> P.shift;
      bool leader = true; uint32_t best = i;
      float e_sum = __uint_as_float(m2.x), tof_min = __uint_as_float(m2.y);
      if (k > 1) {
        const uint64_t my_key = ((uint64_t)my_ids << 32) | i;
        long long isum = 0; float e_best = -1.0f; uint32_t best_ord = 0;
        for (uint32_t j = b; j < b + k; ++j) {
          const uint4 r = *reinterpret_cast<const uint4 *>(&rec[j]);
          if ((r.x >> P.shift) != unit) continue;
          if ((((uint64_t)r.x << 32) | j) < my_key) { leader = false; break; }
          const float2 et = *reinterpret_cast<const float2 *>(&rec[j].e);
          isum += deposit_fixed(et.x);
          const uint32_t ord = r.x & 31u;
          if (et.x > e_best || (et.x == e_best && ord < best_ord)) { e_best = et.x; best = j; best_ord = ord; }
          tof_min = fminf(tof_min, et.y);
        }
        e_sum = (float)((double)isum * (1.0 / 1099511627776.0));
      }
      if (leader) {
        const uint64_t history = first_history + h;
        const uint4 w = philox4x32_10(make_uint4((uint32_t)history, 0u, 3u, unit), P.keys);        // Box-Muller on words 0,1
        const float nrm = box_muller(u01(w.x), u01(w.y));
        const float sigma = P.sigma_scale * (P.ref_keV > 0.0f ? sqrtf(P.ref_keV * e_sum) : e_sum);
        const float e_b = fmaf(sigma, nrm, e_sum);
        keep = e_b >= P.e_lo && e_b < P.e_hi;
        if (keep) {
          const uint4 r = best == i ? me : *reinterpret_cast<const uint4 *>(&rec[best]);
          s.t = __dadd_rn(decay_time(P, history), __dmul_rn((double)tof_min, 1e-9));
          s.history = (uint32_t)history; s.ids = r.x; s.x = __uint_as_float(r.y); s.y = __uint_as_float(r.z); s.z = __uint_as_float(r.w); s.e = e_b;
        }
      }
    }
    if (B.cap) { if (keep) emit_coarse(B, s, sing, bcnt); continue; }   // coarse buckets: straight into the bucket's region
    const unsigned mk = __ballot_sync(0xFFFFFFFFu, keep);
    if (mk) {
      uint32_t o = 0;
      if (lane == 0) o = atomicAdd(&s_cnt, (uint32_t)__popc(mk));
      o = r0 + __shfl_sync(0xFFFFFFFFu, o, 0) + __popc(mk & ((1u << lane) - 1u));
      if (keep) {
        store_rec(&sing[o], &s);
        srank[o] = atomicAdd(&bcnt[bucket_of(B, s.t)], 1u);          // rank inside its time bucket (any order will do)
      }
    }
  }
  __syncthreads();
  if (threadIdx.x == 0) kcnt[blockIdx.x] = s_cnt;
}

// ---------------------------------------------------------------- stages 1 + 2 for the chunked hit layout
// One block per chunk of 512 pairs (gpet.h: gpet_hits.chunk_fill): the chunk's hits (~400, at most 2048) are already
// together, so the sort by history is a counting sort in SHARED memory -- histogram with shared atomics, block scan,
// order array -- followed by the same adder, blur, window and time as adder_kernel on the staged copies.  No count
// pass, no global scan, no scatter of records through HBM; the hit buffer is read once, coalesced.
constexpr int kChunkThreads = 128;   // small blocks: many chunks resident per SM hide the barriers of each
__global__ void __launch_bounds__(kChunkThreads, 12) chunk_adder_kernel(DigiParams P, Buckets B, uint64_t first_history, HitBuf H, SinRec *sing, uint32_t *srank,
                                                          uint32_t *kcnt, uint32_t *bcnt) {
  extern __shared__ __align__(16) unsigned char chunk_smem[];       // 18 bytes per region entry (cap rounded up to 8): sized at launch
  __shared__ uint32_t s_cnt[kHitChunkPairs], s_off[kHitChunkPairs];
  __shared__ uint32_t s_kept;
  const uint32_t c = blockIdx.x, cap = H.chunk_cap, cap8 = (cap + 7u) & ~7u, fill = H.chunk_fill[c], n = fill < cap ? fill : cap;
  uint32_t *s_ids = reinterpret_cast<uint32_t *>(chunk_smem);
  float *s_e = reinterpret_cast<float *>(s_ids + cap8), *s_tof = s_e + cap8;
  uint16_t *s_h = reinterpret_cast<uint16_t *>(s_tof + cap8), *s_rk = s_h + cap8, *s_ord = s_rk + cap8;
  const unsigned long long g0 = (unsigned long long)c * cap;
  const uint32_t first_lo = (uint32_t)first_history + c * kHitChunkPairs;
  const int lane = threadIdx.x & 31;
  // [R16] slice of a history = history / B: one 64-bit division per chunk, then a compare per history (B >= 512)
  const uint64_t h0 = first_history + (uint64_t)c * kHitChunkPairs, Bs = P.pairs_per_slice;
  const uint64_t slice0 = h0 < Bs ? 0ull : h0 / Bs, rem0 = h0 - slice0 * Bs;
  for (int q = threadIdx.x; q < (int)kHitChunkPairs; q += kChunkThreads) s_cnt[q] = 0;
  if (threadIdx.x == 0) s_kept = 0;
  __syncthreads();
  for (uint32_t i = threadIdx.x; i < n; i += kChunkThreads) {        // stage keys and values, histogram by local history
    const uint32_t h = H.history[g0 + i] - first_lo;
    s_ids[i] = H.ids[g0 + i]; s_e[i] = H.e[g0 + i]; s_tof[i] = H.tof[g0 + i];
    s_h[i] = (uint16_t)(h & (kHitChunkPairs - 1));
    s_rk[i] = (uint16_t)atomicAdd(&s_cnt[h & (kHitChunkPairs - 1)], 1u);
  }
  __syncthreads();
  {
    constexpr int kPer = kHitChunkPairs / kChunkThreads;               // consecutive bins per thread
    uint32_t v[kPer], sum = 0;
#pragma unroll
    for (int q = 0; q < kPer; ++q) { v[q] = s_cnt[kPer * threadIdx.x + q]; sum += v[q]; }
    uint32_t tot; uint32_t ex = block_exclusive_scan<kChunkThreads / 32>(sum, &tot);
#pragma unroll
    for (int q = 0; q < kPer; ++q) { s_off[kPer * threadIdx.x + q] = ex; ex += v[q]; }
  }
  __syncthreads();
  for (uint32_t i = threadIdx.x; i < n; i += kChunkThreads) s_ord[s_off[s_h[i]] + s_rk[i]] = (uint16_t)i;
  __syncthreads();
  // inside a history (a handful of hits) order by (ids, position): the hits of a readout unit become contiguous and the
  // smallest key of a group -- its leader -- comes first.  The ranks go to s_rk, whose arrival ranks are no longer needed.
  uint16_t *s_grp = s_rk;
  for (uint32_t j = threadIdx.x; j < n; j += kChunkThreads) {
    const uint32_t i = s_ord[j], h = s_h[i], b = s_off[h], k = s_cnt[h];
    uint32_t r = 0;
    if (k > 1) {
      const uint64_t my_key = ((uint64_t)s_ids[i] << 32) | i;
      for (uint32_t q = b; q < b + k; ++q) { const uint32_t i2 = s_ord[q]; r += ((((uint64_t)s_ids[i2] << 32) | i2) < my_key) ? 1u : 0u; }
    }
    s_grp[b + r] = (uint16_t)i;
  }
  __syncthreads();
  for (uint32_t j0 = 0; j0 < n; j0 += kChunkThreads) {               // adder: one thread per hit, in (history, ids) order
    const uint32_t j = j0 + threadIdx.x;
    bool keep = false; SinRec s;
    if (j < n) {
      const uint32_t i = s_grp[j], h = s_h[i], b = s_off[h], k = s_cnt[h], my_ids = s_ids[i], unit = my_ids >> P.shift;
      const bool leader = j == b || (s_ids[s_grp[j - 1]] >> P.shift) != unit;
      uint32_t best = i;
      float e_sum = s_e[i], tof_min = s_tof[i];
      if (leader && j + 1 < b + k && (s_ids[s_grp[j + 1]] >> P.shift) == unit) {   // the group has more members: they follow
        long long isum = deposit_fixed(e_sum); float e_best = e_sum; uint32_t best_ord = my_ids & 31u;
        for (uint32_t q = j + 1; q < b + k; ++q) {
          const uint32_t i2 = s_grp[q], ids2 = s_ids[i2];
          if ((ids2 >> P.shift) != unit) break;
          const float e2 = s_e[i2];
          isum += deposit_fixed(e2);
          const uint32_t ord = ids2 & 31u;
          if (e2 > e_best || (e2 == e_best && ord < best_ord)) { e_best = e2; best = i2; best_ord = ord; }
          tof_min = fminf(tof_min, s_tof[i2]);
        }
        e_sum = (float)((double)isum * (1.0 / 1099511627776.0));
      }
      __syncwarp(__activemask());                                    // one copy of the blur and time code below, run by all leaders together
      if (leader) {
        const uint64_t history = h0 + h;
        const uint4 w = philox4x32_10(make_uint4((uint32_t)history, 0u, 3u, unit), P.keys);        // Box-Muller on words 0,1
        const float nrm = box_muller(u01(w.x), u01(w.y));
        const float sigma = P.sigma_scale * (P.ref_keV > 0.0f ? sqrtf(P.ref_keV * e_sum) : e_sum);
        const float e_b = fmaf(sigma, nrm, e_sum);
        keep = e_b >= P.e_lo && e_b < P.e_hi;
        if (keep) {
          uint64_t slice = slice0;
          if (Bs >= kHitChunkPairs) slice += rem0 + h >= Bs ? 1ull : 0ull; else slice = history / Bs;
          s.t = __dadd_rn(decay_time_of(P, slice_plus_u(P, slice, decay_u53(P, history))), __dmul_rn((double)tof_min, 1e-9));
          s.history = (uint32_t)history; s.ids = s_ids[best]; s.x = H.x[g0 + best]; s.y = H.y[g0 + best]; s.z = H.z[g0 + best]; s.e = e_b;
        }
      }
    }
    if (B.cap) { if (keep) emit_coarse(B, s, sing, bcnt); continue; }   // coarse buckets: straight into the bucket's region
    const unsigned mk = __ballot_sync(0xFFFFFFFFu, keep);
    if (mk) {
      uint32_t o = 0;
      if (lane == 0) o = atomicAdd(&s_kept, (uint32_t)__popc(mk));
      o = (uint32_t)g0 + __shfl_sync(0xFFFFFFFFu, o, 0) + __popc(mk & ((1u << lane) - 1u));
      if (keep) {
        store_rec(&sing[o], &s);
        srank[o] = atomicAdd(&bcnt[bucket_of(B, s.t)], 1u);
      }
    }
  }
  __syncthreads();
  if (threadIdx.x == 0) kcnt[c] = s_kept;
}

// ---------------------------------------------------------------- stage 3: time-bucket counting sort
// region = records per block (0: derived from *n_rec as in adder_kernel)
__global__ void __launch_bounds__(256) bucket_scatter_kernel(const SinRec *sing, const uint32_t *srank, const uint32_t *n_rec, uint32_t region,
                                                             const uint32_t *kcnt, Buckets B, const uint32_t *boff, SinRec *srt) {
  const uint32_t r0 = blockIdx.x * (region ? region : region_size(*n_rec, gridDim.x)), m = kcnt[blockIdx.x];   // this block's kept singles
  for (uint32_t i = r0 + threadIdx.x; i < r0 + m; i += 256u) {
    SinRec s; store_rec(&s, &sing[i]);
    store_rec(&srt[boff[bucket_of(B, s.t)] + srank[i]], &s);
  }
}
__device__ __forceinline__ bool single_less(const SinRec &a, const SinRec &b, int shift) {             // (t, history, unit)
  if (a.t != b.t) return a.t < b.t;
  if (a.history != b.history) return a.history < b.history;
  return (a.ids >> shift) < (b.ids >> shift);
}
// one thread per single (bucket order): rank inside its bucket (~1-3 singles) by counting, then the final time-ordered
// record and the caller's arrays
__global__ void __launch_bounds__(256) bucket_sort_kernel(const SinRec *srt, int shift, const uint32_t *n_ptr, Buckets B, const uint32_t *boff, SinRec *fin, SinglesBuf S) {
  const uint32_t n = *n_ptr;
  for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < n; i += gridDim.x * 256u) {
    SinRec a; store_rec(&a, &srt[i]);
    const uint32_t b = bucket_of(B, a.t), s = boff[b], m = boff[b + 1] - s;
    uint32_t rank = 0;
    for (uint32_t q = s; q < s + m; ++q) {
      if (q == i) continue;
      SinRec c; store_rec(&c, &srt[q]);
      if (single_less(c, a, shift) || (!single_less(a, c, shift) && q < i)) ++rank;
    }
    const uint32_t o = s + rank;
    store_rec(&fin[o], &a);
    if (S.history && o < S.capacity) { S.history[o] = a.history; S.ids[o] = a.ids; S.x[o] = a.x; S.y[o] = a.y; S.z[o] = a.z; S.e[o] = a.e; S.t[o] = a.t; }
  }
}

// ---------------------------------------------------------------- stage 3 with coarse buckets: one block sorts a group of buckets
// The records of kSortGroup consecutive buckets (together at most kCoarseCap, ~560 on C1) are staged in shared memory and
// ordered by (t, history, unit) with a counting sort over kSubBuckets equal time intervals (shared atomics give each record
// its rank of arrival, a block scan the offsets) and a rank by comparison among the records of the same sub-bucket (rarely
// more than one).  The time-ordered records leave as whole sectors, coalesced, at the group's offset in the final array.
#ifndef GPET_SORT_THREADS
#define GPET_SORT_THREADS 256
#endif
constexpr int kSortThreads = GPET_SORT_THREADS;
constexpr uint32_t kSortGroup = 4;   // buckets per block: their records are sorted together when they fit (the regions are sized for
                                     // the worst case -- every hit a kept single -- and are a quarter full on C1), else one by one
// sorts the records of buckets [b0, b0 + nbk) (together at most kCoarseCap) and writes them at boff[b0]
__device__ __forceinline__ void sort_span(const SinRec *regions, const uint32_t *fill, const uint32_t *boff, const Buckets &B, int shift, SinRec *fin, const SinglesBuf &S,
                                          uint32_t b0, uint32_t nbk, uint32_t n, uint4 *s_a, uint32_t *s_src, uint32_t *s_cnt, uint32_t *s_off,
                                          uint16_t *s_sb, uint16_t *s_rk, uint16_t *s_idx, uint16_t *s_fin) {
  const uint32_t base = boff[b0];
  const double sub_scale = (double)(kSubBuckets / kSortGroup) * (double)(kSortGroup / nbk);   // nbk = 1 or kSortGroup
  for (int q = threadIdx.x; q < (int)kSubBuckets; q += kSortThreads) s_cnt[q] = 0;
  __syncthreads();
  static_assert(kSortGroup == 4, "the flat loop below splits a span of four buckets");
  uint32_t e1 = 0, e2 = 0, e3 = 0;                                    // records of the span's first 1, 2, 3 buckets
  if (nbk > 1) {
    const uint32_t f0 = fill[b0], f1 = fill[b0 + 1], f2 = fill[b0 + 2];
    e1 = f0 < B.cap ? f0 : B.cap; e2 = e1 + (f1 < B.cap ? f1 : B.cap); e3 = e2 + (f2 < B.cap ? f2 : B.cap);
  }
  for (uint32_t i = threadIdx.x; i < n; i += kSortThreads) {         // one flat loop over the records of all the span's buckets
    uint32_t k = 0, q = i;
    if (nbk > 1) { k = (i >= e1 ? 1u : 0u) + (i >= e2 ? 1u : 0u) + (i >= e3 ? 1u : 0u); q = i - (k == 0 ? 0u : (k == 1 ? e1 : (k == 2 ? e2 : e3))); }
    const uint32_t src = (b0 + k) * B.cap + q;
    const uint4 ra = reinterpret_cast<const uint4 *>(regions + src)[0];
    s_a[i] = ra; s_src[i] = src;                                      // the payload {x, y, z, e} is fetched when the record leaves
    const double t = __longlong_as_double((long long)(((unsigned long long)ra.y << 32) | ra.x));
    const double x = __dmul_rn(__dsub_rn(bucket_coord(B, t), (double)b0), sub_scale);   // monotonic in t
    const uint32_t sb = !(x > 0.0) ? 0u : (x >= (double)(kSubBuckets - 1) ? kSubBuckets - 1 : (uint32_t)x);
    s_sb[i] = (uint16_t)sb; s_rk[i] = (uint16_t)atomicAdd(&s_cnt[sb], 1u);
  }
  __syncthreads();
  {
    constexpr int kPer = kSubBuckets / kSortThreads;
    uint32_t v[kPer], sum = 0;
#pragma unroll
    for (int q = 0; q < kPer; ++q) { v[q] = s_cnt[kPer * threadIdx.x + q]; sum += v[q]; }
    uint32_t tot; uint32_t ex = block_exclusive_scan<kSortThreads / 32>(sum, &tot);
#pragma unroll
    for (int q = 0; q < kPer; ++q) { s_off[kPer * threadIdx.x + q] = ex; ex += v[q]; }
  }
  __syncthreads();
  for (uint32_t i = threadIdx.x; i < n; i += kSortThreads) s_idx[s_off[s_sb[i]] + s_rk[i]] = (uint16_t)i;
  __syncthreads();
  for (uint32_t p = threadIdx.x; p < n; p += kSortThreads) {         // rank inside the sub-bucket by (t, history, unit)
    const uint32_t i = s_idx[p], sb = s_sb[i], s0 = s_off[sb], m = s_cnt[sb];
    uint32_t rank = 0;
    if (m > 1) {
      const uint4 me = s_a[i];
      const double tm = __longlong_as_double((long long)(((unsigned long long)me.y << 32) | me.x));
      for (uint32_t q = s0; q < s0 + m; ++q) {
        if (q == p) continue;
        const uint4 o = s_a[s_idx[q]];
        const double to = __longlong_as_double((long long)(((unsigned long long)o.y << 32) | o.x));
        const bool o_less = to != tm ? to < tm : (o.z != me.z ? o.z < me.z : (o.w >> shift) < (me.w >> shift));
        const bool m_less = to != tm ? tm < to : (o.z != me.z ? me.z < o.z : (me.w >> shift) < (o.w >> shift));
        if (o_less || (!m_less && q < p)) ++rank;
      }
    }
    s_fin[s0 + rank] = (uint16_t)i;
  }
  __syncthreads();
  uint4 *out = reinterpret_cast<uint4 *>(fin + base);
  for (uint32_t p = threadIdx.x; p < n; p += kSortThreads) {
    const uint32_t i = s_fin[p];
    const uint4 ra = s_a[i], rb = reinterpret_cast<const uint4 *>(regions + s_src[i])[1];
    out[2 * p] = ra; out[2 * p + 1] = rb;
    const unsigned long long o = (unsigned long long)base + p;
    if (S.history && o < S.capacity) {
      S.history[o] = ra.z; S.ids[o] = ra.w; S.x[o] = __uint_as_float(rb.x); S.y[o] = __uint_as_float(rb.y); S.z[o] = __uint_as_float(rb.z);
      S.e[o] = __uint_as_float(rb.w); S.t[o] = __longlong_as_double((long long)(((unsigned long long)ra.y << 32) | ra.x));
    }
  }
  __syncthreads();                                                   // the arrays are reused by the next span
}
__global__ void __launch_bounds__(kSortThreads) bucket_sort_coarse_kernel(const SinRec *regions, const uint32_t *fill, const uint32_t *boff, Buckets B, int shift,
                                                                          SinRec *fin, SinglesBuf S) {
  __shared__ uint4 s_a[kCoarseCap];                                  // {t, history, ids}
  __shared__ uint32_t s_src[kCoarseCap], s_cnt[kSubBuckets], s_off[kSubBuckets];
  __shared__ uint16_t s_sb[kCoarseCap], s_rk[kCoarseCap], s_idx[kCoarseCap], s_fin[kCoarseCap];
  const uint32_t b0 = blockIdx.x * kSortGroup, nbk = B.nb - b0 < kSortGroup ? B.nb - b0 : kSortGroup;
  uint32_t n = 0;
  for (uint32_t k = 0; k < nbk; ++k) { const uint32_t f = fill[b0 + k]; n += f < B.cap ? f : B.cap; }
  if (n == 0) return;
  if (n <= B.cap && nbk == kSortGroup) { sort_span(regions, fill, boff, B, shift, fin, S, b0, nbk, n, s_a, s_src, s_cnt, s_off, s_sb, s_rk, s_idx, s_fin); return; }
  for (uint32_t k = 0; k < nbk; ++k) {
    const uint32_t f = fill[b0 + k], nk = f < B.cap ? f : B.cap;
    if (nk) sort_span(regions, fill, boff, B, shift, fin, S, b0 + k, 1u, nk, s_a, s_src, s_cnt, s_off, s_sb, s_rk, s_idx, s_fin);
  }
}

// ---------------------------------------------------------------- stage 4: coincidence windows [R27], two passes
// Pass 1, a thread per single of the time-ordered array: a single that starts a cluster (gap >= tau to its predecessor)
// walks the cluster with the window rule -- an unconsumed single opens a window, the members are the following singles
// within tau of the opener, exactly two members on different panels make a coincidence -- and writes the flag of EVERY
// member (1 = this single opens an accepted pair with its successor), so `flag` needs no clearing; every pair is counted
// in the tile (kCoTile singles) of its opener (tile_cnt is zeroed by the caller).  A scan over the tiles gives every
// tile its offset in the list-mode output, in time order.  Pass 2: block scan of the tile's flags, one record per
// flagged single.
// (Measured alternatives: one kernel with a decoupled look-back over the tiles -- with ~600 short tiles in flight every
// tile looks back over the whole wave, 120 us; a second walk in pass 2 instead of the flags -- re-reads the times from
// HBM, 52 us for that pass.)
constexpr int kCoTile = 256;
__global__ void __launch_bounds__(kCoTile) coincidence_flag_kernel(const SinRec *fin, const uint32_t *n_ptr, double tau, uint8_t *flag, uint32_t *tile_cnt) {
  __shared__ uint32_t s_sum;
  const uint32_t n = *n_ptr;
  for (uint32_t tile = blockIdx.x; (unsigned long long)tile * kCoTile < n; tile += gridDim.x) {
  if (threadIdx.x == 0) s_sum = 0u;
  __syncthreads();
  const uint32_t i = tile * kCoTile + threadIdx.x;
  uint32_t cnt = 0;
  if (i < n && (i == 0 || !(__dsub_rn(fin[i].t, fin[i - 1].t) < tau))) {
    uint32_t o = i;
    for (;;) {                                                       // o opens a window
      const double to = fin[o].t;
      uint32_t j = o + 1;
      double tl = to;                                                // time of single j - 1
      while (j < n) { const double tj = fin[j].t; if (!(__dsub_rn(tj, to) < tau)) break; flag[j] = 0; tl = tj; ++j; }
      const bool pair = j - o == 2 && (fin[o].ids >> 26) != (fin[o + 1].ids >> 26);
      flag[o] = pair ? 1 : 0;
      if (pair) { if (o / kCoTile == tile) ++cnt; else atomicAdd(&tile_cnt[o / kCoTile], 1u); }   // (a cluster may run past its tile)
      if (j >= n || !(__dsub_rn(fin[j].t, tl) < tau)) break;         // the next opener starts a new cluster (its own thread)
      o = j;
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xFFFFFFFFu, cnt, o);
  if ((threadIdx.x & 31) == 0 && cnt) atomicAdd(&s_sum, cnt);
  __syncthreads();
  if (threadIdx.x == 0 && s_sum) atomicAdd(&tile_cnt[tile], s_sum);
  __syncthreads();
  }
}
__global__ void __launch_bounds__(kCoTile) coincidence_write_kernel(const SinRec *fin, const uint32_t *n_ptr, const uint8_t *flag, const uint32_t *tile_off, CoincBuf C,
                                                                    const uint32_t *dropped, unsigned long long *n_singles_out) {
  // last kernel of the call: if the time sort dropped singles both lists are incomplete -- say so where every caller looks
  if (blockIdx.x == 0 && threadIdx.x == 0 && *dropped) { *C.n = ~0ull; if (n_singles_out) *n_singles_out = ~0ull; }
  const uint32_t n = *n_ptr;
  for (uint32_t tile = blockIdx.x; (unsigned long long)tile * kCoTile < n; tile += gridDim.x) {
  const unsigned long long w0 = tile_off[tile];
  if (tile_off[tile + 1] == (uint32_t)w0) continue;                  // no pair opens in this tile
  const uint32_t i = tile * kCoTile + threadIdx.x;
  const uint32_t f = i < n ? flag[i] : 0u;
  uint32_t tot; const uint32_t ex = block_exclusive_scan<kCoTile / 32>(f, &tot);
  const unsigned long long w = w0 + ex;
  if (f && w < C.capacity) {
    SinRec a, b; store_rec(&a, &fin[i]); store_rec(&b, &fin[i + 1]);
    C.ids_a[w] = a.ids; C.ids_b[w] = b.ids; C.history_a[w] = a.history; C.history_b[w] = b.history;
    C.e_a[w] = a.e; C.e_b[w] = b.e;
    C.dt_ns[w] = (float)__dmul_rn(__dsub_rn(b.t, a.t), 1e9); C.t[w] = a.t;
  }
  }
}

// ---------------------------------------------------------------- scratch layout + driver
namespace {
struct Layout { size_t kcnt, cnt, off, ctl, ctl_bytes, st1, st2, bcnt, boff, tcnt, toff, flag, hrank, srank, rec, sing, fin, total; uint64_t nb, nb_coarse; };
Layout layout(uint64_t N, uint64_t M) {
  Layout L; size_t o = 0; const uint64_t Mx = M ? M : 1;
  auto take = [&](size_t bytes) { o = (o + 255) & ~(size_t)255; size_t r = o; o += bytes; return r; };
  L.nb = (Mx + 1) / 2;              // fine time buckets: kept singles are ~0.4 per hit, so ~1 per bucket
  L.nb_coarse = (Mx + kCoarseMean - 1) / kCoarseMean;   // coarse ones: at most kCoarseMean on average even if every hit became a single
  L.kcnt = take(4 * (148 * 16 + N / kHitChunkPairs + 2));   // kept singles per adder block (dense) or per chunk (chunked layout)
  L.cnt = take(4 * N); L.off = take(4 * (N + 1));
  // control block, cleared by one memset per call: the look-back state of the three scans (hits per history, singles per
  // bucket, coincidences per tile) and the accepted pairs per tile of the time-ordered singles
  const size_t s0 = 16 * (N / kTile / 2 + 2), s1 = 16 * (L.nb / kTile / 2 + 2), s2 = 16 * (Mx / kCoTile / kTile / 2 + 2), s3 = 4 * (Mx / kCoTile + 4);   // (16-byte aligned: the scan reads uint4)
  L.ctl = take(256 + s0 + s1 + s2 + s3); L.st1 = L.ctl + 256 + s0; L.st2 = L.st1 + s1; L.tcnt = L.st2 + s2; L.ctl_bytes = 256 + s0 + s1 + s2 + s3;
  L.bcnt = take(4 * L.nb); L.boff = take(4 * (L.nb + 1));
  L.toff = take(4 * (Mx / kCoTile + 2)); L.flag = take(Mx);
  L.hrank = take(4 * Mx); L.srank = take(4 * Mx);   // rank of a hit in its history / of a kept single in its time bucket
  L.rec = take(32 * Mx);            // hit records by history; reused for the bucket-ordered singles
  const size_t coarse = 32 * (size_t)kCoarseCap * L.nb_coarse;
  L.sing = take(coarse > 32 * Mx ? coarse : 32 * Mx);   // kept singles: append order, or the regions of the coarse buckets
  L.fin = take(32 * Mx);            // kept singles, time order
  L.total = o + 256; return L;
}
inline int grid_for(uint64_t n) { const uint64_t b = (n + 255) / 256; return (int)(b < 1 ? 1 : (b > 148ull * 16 ? 148ull * 16 : b)); }
}  // namespace

size_t digitize_scratch_bytes(uint64_t n_pairs, uint64_t n_hits) { return layout(n_pairs, n_hits).total; }

cudaError_t launch_digitize(const DigiParams &P, const HitBuf &H, uint64_t first_history, uint64_t n_pairs, uint64_t n_hits,
                            void *scratch, size_t scratch_bytes, const SinglesBuf &S, const CoincBuf &C, cudaStream_t st) {
  (void)scratch_bytes;
  const uint64_t N = n_pairs, M = n_hits ? n_hits : 1;
  const Layout L = layout(N, n_hits);
  char *s = (char *)scratch;
  uint32_t *cnt = (uint32_t *)(s + L.cnt), *off = (uint32_t *)(s + L.off), *kcnt = (uint32_t *)(s + L.kcnt);
  unsigned long long *st0 = (unsigned long long *)(s + L.ctl + 256), *st1 = (unsigned long long *)(s + L.st1), *st2 = (unsigned long long *)(s + L.st2);
  uint32_t *bcnt = (uint32_t *)(s + L.bcnt), *boff = (uint32_t *)(s + L.boff);
  uint32_t *hrank = (uint32_t *)(s + L.hrank), *srank = (uint32_t *)(s + L.srank), *tcnt = (uint32_t *)(s + L.tcnt), *toff = (uint32_t *)(s + L.toff);
  uint8_t *flag = (uint8_t *)(s + L.flag);
  HitRec *rec = (HitRec *)(s + L.rec); SinRec *srt = (SinRec *)(s + L.rec), *sing = (SinRec *)(s + L.sing), *fin = (SinRec *)(s + L.fin);
  const bool chunked = H.chunk_fill != nullptr;
  const uint64_t B = P.pairs_per_slice;
  const uint64_t slice_first = first_history / B, slice_last = (first_history + n_pairs - 1) / B;
  Buckets bk;
  bk.dropped = (uint32_t *)(s + L.ctl);                               // first word of the control block (cleared below)
  bk.t_lo = decay_time_of(P, (double)slice_first);                  // the batch's time slices cover [t_lo, t_hi) [R16, R34]
  const double t_hi = decay_time_of(P, fmin((double)slice_last + 1.0, P.lambda > 0.0 ? 1.0 / P.q_scale : 1e300)) + 2e-6;
  // Coarse buckets need times that are uniform over [t_lo, t_hi): the batch lies inside one time slice, or covers whole
  // slices (a last slice cut short by the end of the run only lowers the density), and the decay law [R34] changes the
  // rate by less than 10 % across it.  Anything else takes the fine buckets, which count before they place.
  const bool whole = first_history % B == 0 && ((first_history + n_pairs) % B == 0 || first_history + n_pairs == P.n_pairs_total);
  const bool coarse = (slice_first == slice_last || whole) && P.lambda * (t_hi - bk.t_lo) < 0.1;
  bk.nb = (uint32_t)(coarse ? L.nb_coarse : L.nb); bk.cap = coarse ? kCoarseCap : 0u;
  bk.scale = (double)bk.nb / (t_hi - bk.t_lo);
  cudaError_t e;
  if (!chunked && (e = cudaMemsetAsync(cnt, 0, 4 * N, st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(s + L.ctl, 0, L.ctl_bytes, st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(bcnt, 0, 4 * (size_t)bk.nb, st)) != cudaSuccess) return e;
  const uint32_t nh = (uint32_t)n_hits, np = (uint32_t)N, first_lo = (uint32_t)first_history;
  const int ga = grid_for(M);                                         // adder and bucket scatter share the block -> region split
  if (chunked) {
    // 1 + 2. per chunk in shared memory: sort by history, adder, blur, window, time
    chunk_adder_kernel<<<H.n_chunks, kChunkThreads, 18 * (size_t)((H.chunk_cap + 7u) & ~7u), st>>>(P, bk, first_history, H, sing, srank, kcnt, bcnt); count_launch();
  } else {
    // 1. counting sort by history
    if (nh) { count_hits_kernel<<<grid_for(nh), 256, 0, st>>>(H, nh, first_lo, np, cnt, hrank); count_launch(); }
    if ((e = exclusive_scan(cnt, N, nullptr, off, st0, nullptr, st)) != cudaSuccess) return e;
    if (nh) { scatter_hits_kernel<<<grid_for(nh), 256, 0, st>>>(H, nh, first_lo, np, off, hrank, rec); count_launch(); }
    // 2. adder, blur, window, time; kept singles appended and counted into time buckets
    adder_kernel<<<ga, 256, 0, st>>>(P, bk, first_history, off, off + N, rec, sing, srank, kcnt, bcnt); count_launch();
  }
  // 3. time order: offsets of the buckets (the total is the number of kept singles), then the order inside each bucket
  if ((e = exclusive_scan(bcnt, bk.nb, nullptr, boff, st1, S.n, st)) != cudaSuccess) return e;
  const uint32_t *n_singles = boff + bk.nb;
  if (coarse) {
    bucket_sort_coarse_kernel<<<(bk.nb + kSortGroup - 1) / kSortGroup, kSortThreads, 0, st>>>(sing, bcnt, boff, bk, P.shift, fin, S); count_launch();
  } else {
    bucket_scatter_kernel<<<chunked ? (int)H.n_chunks : ga, 256, 0, st>>>(sing, srank, off + N, chunked ? H.chunk_cap : 0u, kcnt, bk, boff, srt); count_launch();
    bucket_sort_kernel<<<grid_for(M / 2 + 1), 256, 0, st>>>(srt, P.shift, n_singles, bk, boff, fin, S); count_launch();
  }
  // 4. coincidences (the number of singles is known on the device only: tiles past it return at once)
  const unsigned co_tiles = (unsigned)((M + kCoTile - 1) / kCoTile);
  const unsigned co_grid = co_tiles < 148u * 8u ? co_tiles : 148u * 8u;   // blocks stride over the tiles up to the device-side count
  coincidence_flag_kernel<<<co_grid, kCoTile, 0, st>>>(fin, n_singles, P.window_s, flag, tcnt); count_launch();
  if ((e = exclusive_scan(tcnt, co_tiles, nullptr, toff, st2, C.n, st)) != cudaSuccess) return e;
  coincidence_write_kernel<<<co_grid, kCoTile, 0, st>>>(fin, n_singles, flag, toff, C, bk.dropped, S.n); count_launch();
  return cudaGetLastError();
}

// ---------------------------------------------------------------- built-in scratch (gpet_digitize_static, gpet.h)
// Scratch for callers that may not allocate device memory: one fixed array in the library's device image.  It exists once
// per GPU that loads these kernels, from that load until the process exits, whether or not anyone uses it.  In HOST code
// the name below is only a handle for the runtime -- it is not a device address and must never be given to a kernel; the
// address the kernels of this file receive comes from cudaGetSymbolAddress, asked once per device with that device current.
static __device__ __align__(256) unsigned char g_static_scratch[GPET_STATIC_SCRATCH_BYTES];

cudaError_t static_digitize_scratch(void **ptr, size_t *bytes) {
  constexpr int kMaxDevices = 64;
  static std::mutex lock;
  static void *addr[kMaxDevices] = {};
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lk(lock);
  if (!addr[dev]) {                                                   // set-up, first call on this device
    void *p = nullptr;
    if ((e = cudaGetSymbolAddress(&p, g_static_scratch)) != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    addr[dev] = p;
  }
  *ptr = addr[dev]; *bytes = sizeof g_static_scratch;
  return cudaSuccess;
}

}  // namespace gpet
