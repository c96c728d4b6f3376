// gpet_digitize.cu -- singles digitizer and coincidence sorter (S11..S14 of DESIGN.md section 1).
// PAPER.md:33,37 (single-event readout at crystal / module / panel level), PAPER.md:61 (energy resolution,
// coincidence timing window), PAPER.md:65 (list-mode coincidences).  Readings [R16], [R24]-[R27].
//
// Sort / segmented-scan structure (all hand-written, no CUB/Thrust):
//   1. counting sort of the hits by history id (dense integer keys: histogram by atomics in L2,
//      exclusive scan, scatter of 32-byte hit records) -> one contiguous run of sectors per history;
//   2. one thread per history: canonical in-segment order by repeated min-selection (segments hold
//      ~1-4 hits), adder per readout unit, blur, window, absolute time -> kept singles appended as
//      32-byte records and counted into time buckets;
//   3. counting sort of the kept singles by time bucket (decay times are uniform by construction
//      [R16], so buckets hold ~0.4 singles on average), in-bucket rank sort by (t, history, unit);
//   4. head-flag pass: a thread per cluster start (gap >= tau) walks its cluster with the window rule
//      [R27]; exclusive scan of the pair flags; compaction into list-mode output.
// Every stage is deterministic: the output does not depend on the order of the hit buffer.
#include "gpet_internal.h"

namespace gpet {

constexpr int kTile = 2048;      // elements per scan block (256 threads x 8)

// ---------------------------------------------------------------- device-wide exclusive scan (u32)
__device__ __forceinline__ uint32_t block_exclusive_scan_256(uint32_t v, uint32_t *total) {
  __shared__ uint32_t warp_sum[8];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint32_t inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o); if (lane >= o) inc += t; }
  __syncthreads();                         // protect warp_sum reuse across calls
  if (lane == 31) warp_sum[wid] = inc;
  __syncthreads();
  uint32_t base = 0, tot = 0;
#pragma unroll
  for (int w = 0; w < 8; ++w) { const uint32_t s = warp_sum[w]; if (w < wid) base += s; tot += s; }
  *total = tot;
  return base + inc - v;
}

__global__ void __launch_bounds__(256) scan_reduce_kernel(const uint32_t *in, uint64_t n, uint32_t *bsum) {
  const uint64_t base = (uint64_t)blockIdx.x * kTile;
  uint32_t s = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) { const uint64_t i = base + (uint64_t)k * 256 + threadIdx.x; if (i < n) s += in[i]; }
  uint32_t tot; block_exclusive_scan_256(s, &tot);
  if (threadIdx.x == 0) bsum[blockIdx.x] = tot;
}
// single block: exclusive scan of the block sums in place; total -> bsum[nb] and (optionally) a u64 counter
__global__ void __launch_bounds__(256) scan_bsums_kernel(uint32_t *bsum, uint32_t nb, unsigned long long *total_out) {
  uint32_t carry = 0;
  for (uint32_t start = 0; start < nb; start += 256) {
    const uint32_t i = start + threadIdx.x;
    const uint32_t v = i < nb ? bsum[i] : 0u;
    uint32_t tot; const uint32_t ex = block_exclusive_scan_256(v, &tot);
    if (i < nb) bsum[i] = carry + ex;
    carry += tot;
  }
  if (threadIdx.x == 0) { bsum[nb] = carry; if (total_out) *total_out = carry; }
}
// out[i] = exclusive prefix of in; out[n] = total (out has n+1 entries; may alias in only if out == in and n+1 fits)
__global__ void __launch_bounds__(256) scan_apply_kernel(const uint32_t *in, uint64_t n, const uint32_t *bsum, uint32_t nb, uint32_t *out) {
  const uint64_t base = (uint64_t)blockIdx.x * kTile + (uint64_t)threadIdx.x * 8;
  uint32_t v[8], s = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) { v[k] = base + k < n ? in[base + k] : 0u; s += v[k]; }
  uint32_t tot; uint32_t ex = block_exclusive_scan_256(s, &tot) + bsum[blockIdx.x];
#pragma unroll
  for (int k = 0; k < 8; ++k) { if (base + k < n) out[base + k] = ex; ex += v[k]; }
  if (blockIdx.x == 0 && threadIdx.x == 0) out[n] = bsum[nb];
}

static cudaError_t exclusive_scan(const uint32_t *in, uint64_t n, uint32_t *out, uint32_t *bsum, unsigned long long *total_out, cudaStream_t st) {
  const uint32_t nb = (uint32_t)((n + kTile - 1) / kTile);
  scan_reduce_kernel<<<nb, 256, 0, st>>>(in, n, bsum);
  scan_bsums_kernel<<<1, 256, 0, st>>>(bsum, nb, total_out);
  scan_apply_kernel<<<nb, 256, 0, st>>>(in, n, bsum, nb, out);
  count_launch(3);
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
__global__ void __launch_bounds__(256) count_hits_kernel(HitBuf H, uint32_t bound, uint32_t first_lo, uint32_t n_pairs, uint32_t *cnt) {
  const uint32_t n_hits = valid_hits(H, bound); const uint32_t *history = H.history;
  for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < n_hits; i += gridDim.x * 256u) {
    const uint32_t h = history[i] - first_lo;
    if (h < n_pairs) atomicAdd(&cnt[h], 1u);
  }
}
// reads the struct-of-arrays hit buffer coalesced, writes each hit as one sector into its history's segment
__global__ void __launch_bounds__(256) scatter_hits_kernel(HitBuf H, uint32_t bound, uint32_t first_lo, uint32_t n_pairs,
                                                           const uint32_t *off, uint32_t *cnt, HitRec *rec) {
  const uint32_t n_hits = valid_hits(H, bound);
  for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < n_hits; i += gridDim.x * 256u) {
    const uint32_t h = H.history[i] - first_lo;
    if (h >= n_pairs) continue;
    HitRec r; r.ids = H.ids[i]; r.x = H.x[i]; r.y = H.y[i]; r.z = H.z[i]; r.e = H.e[i]; r.tof = H.tof[i]; r.idx = i; r.pad = h;
    store_rec(&rec[off[h] + atomicSub(&cnt[h], 1u) - 1u], &r);
  }
}

// ---------------------------------------------------------------- stage 2: adder + blur + window + time
struct Buckets { double t_lo, scale; uint32_t nb; };
__device__ __forceinline__ uint32_t bucket_of(const Buckets &B, double t) {
  const double x = (t - B.t_lo) * B.scale;
  if (!(x > 0.0)) return 0u;
  return x >= (double)(B.nb - 1) ? B.nb - 1 : (uint32_t)x;
}

__device__ __forceinline__ double decay_time(const DigiParams &P, uint64_t history) {     // [R16]
  const uint2 key = make_uint2((uint32_t)P.seed, (uint32_t)(P.seed >> 32));
  const uint4 w = philox4x32_10(make_uint4((uint32_t)history, (uint32_t)(history >> 32), 0u, 2u), key);
  const uint64_t bits = (((uint64_t)w.x << 32) | (uint64_t)w.y) >> 11;
  const double u53 = __dmul_rn(__dadd_rn((double)bits, 0.5), 1.0 / 9007199254740992.0);
  const uint64_t B = P.pairs_per_slice;
  const uint64_t slice = history < B ? 0ull : history / B;
  return __dmul_rn(__dadd_rn((double)slice, u53), P.slice_s);                               // slice_s = B / A
}

// blur [R25], window [R26], absolute time [R16]; a kept single goes to the next slot of its history's segment
// (no global append counter: slots not used are marked invalid by the caller) and is counted into its time bucket
__device__ __forceinline__ void emit_single(const DigiParams &P, const Buckets &B, uint64_t history, uint32_t unit, float e_sum,
                                            const HitRec &best, float tof_min, SinRec *sing, uint32_t &slot, uint32_t *bcnt) {
  const uint2 key = make_uint2((uint32_t)P.seed, (uint32_t)(P.seed >> 32));
  const uint4 w = philox4x32_10(make_uint4((uint32_t)history, 0u, 3u, unit), key);           // Box-Muller on words 0,1
  const float nrm = sqrtf(-2.0f * logf(u01(w.x))) * cospif(2.0f * u01(w.y));
  const float sigma = P.sigma_scale * (P.ref_keV > 0.0f ? sqrtf(P.ref_keV * e_sum) : e_sum);
  const float e_b = fmaf(sigma, nrm, e_sum);
  if (!(e_b >= P.e_lo && e_b < P.e_hi)) return;
  SinRec s; s.t = __dadd_rn(decay_time(P, history), __dmul_rn((double)tof_min, 1e-9));
  s.history = (uint32_t)history; s.ids = best.ids; s.x = best.x; s.y = best.y; s.z = best.z; s.e = e_b;
  store_rec(&sing[slot++], &s);
  atomicAdd(&bcnt[bucket_of(B, s.t)], 1u);
}

// One thread per hit record (all lanes busy; a thread per history would idle on the ~54 % of histories without
// hits).  The record with the smallest (ids, position) of its (history, readout unit) group is the group's
// leader: it sums the group in ascending (ids, position) order -- canonical, so the fp32 sum does not depend
// on the hit buffer's order -- picks the largest deposit and the earliest time [R24], and emits the single
// into its own slot; every other slot is marked unused.
__global__ void __launch_bounds__(256) adder_kernel(DigiParams P, Buckets B, uint64_t first_history, const uint32_t *off, const uint32_t *n_rec,
                                                    const HitRec *rec, SinRec *sing, uint32_t *bcnt) {
  const uint32_t n = *n_rec;
  for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < n; i += gridDim.x * 256u) {
    HitRec me; store_rec(&me, &rec[i]);
    const uint32_t h = me.pad, b = off[h], k = off[h + 1] - b, unit = me.ids >> P.shift;
    const uint64_t my_key = ((uint64_t)me.ids << 32) | i;
    bool leader = true;
    float e_sum = me.e, tof_min = me.tof; HitRec best = me;
    if (k > 1) {
      uint32_t members = 0;
      for (uint32_t j = b; j < b + k; ++j) {
        const uint32_t ids = rec[j].ids;
        if ((ids >> P.shift) != unit) continue;
        ++members;
        if ((((uint64_t)ids << 32) | j) < my_key) leader = false;
      }
      if (leader && members > 1) {                                   // ascending (ids, position) after the leader itself
        uint64_t prev = my_key; float e_best = me.e; uint32_t best_ord = me.ids & 31u;
        for (uint32_t m = 1; m < members; ++m) {
          uint64_t sel = ~0ull;
          for (uint32_t j = b; j < b + k; ++j) {
            const uint32_t ids = rec[j].ids;
            const uint64_t key = ((uint64_t)ids << 32) | j;
            if ((ids >> P.shift) == unit && key > prev && key < sel) sel = key;
          }
          prev = sel;
          HitRec r; store_rec(&r, &rec[(uint32_t)sel]);
          const uint32_t ord = r.ids & 31u;
          e_sum += r.e;
          if (r.e > e_best || (r.e == e_best && ord < best_ord)) { e_best = r.e; best = r; best_ord = ord; }
          tof_min = fminf(tof_min, r.tof);
        }
      }
    }
    uint32_t slot = i;
    if (leader) emit_single(P, B, first_history + h, unit, e_sum, best, tof_min, sing, slot, bcnt);
    if (slot == i) sing[i].ids = kNone;                              // not a leader, or outside the energy window
  }
}

// ---------------------------------------------------------------- stage 3: time-bucket counting sort
__global__ void __launch_bounds__(256) bucket_scatter_kernel(const SinRec *sing, const uint32_t *n_slots, Buckets B,
                                                             const uint32_t *boff, uint32_t *bcnt, SinRec *srt) {
  const uint32_t n = *n_slots;                                       // = number of hits: one slot per hit
  for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < n; i += gridDim.x * 256u) {
    SinRec s; store_rec(&s, &sing[i]);
    if (s.ids == kNone) continue;
    const uint32_t b = bucket_of(B, s.t);
    store_rec(&srt[boff[b] + atomicSub(&bcnt[b], 1u) - 1u], &s);
  }
}
__device__ __forceinline__ bool single_less(const SinRec &a, const SinRec &b, int shift) {             // (t, history, unit)
  if (a.t != b.t) return a.t < b.t;
  if (a.history != b.history) return a.history < b.history;
  return (a.ids >> shift) < (b.ids >> shift);
}
// one thread per bucket (~0-3 singles): rank by counting, write the final time-ordered records and the caller's arrays
__global__ void __launch_bounds__(256) bucket_sort_kernel(const SinRec *srt, int shift, uint32_t nb, const uint32_t *boff, SinRec *fin, SinglesBuf S) {
  for (uint32_t b = blockIdx.x * 256u + threadIdx.x; b < nb; b += gridDim.x * 256u) {
    const uint32_t s = boff[b], m = boff[b + 1] - s;
    for (uint32_t j = 0; j < m; ++j) {
      SinRec a; store_rec(&a, &srt[s + j]);
      uint32_t rank = 0;
      for (uint32_t q = 0; q < m; ++q) {
        if (q == j) continue;
        SinRec c; store_rec(&c, &srt[s + q]);
        if (single_less(c, a, shift) || (!single_less(a, c, shift) && q < j)) ++rank;
      }
      const uint32_t o = s + rank;
      store_rec(&fin[o], &a);
      if (S.history && o < S.capacity) { S.history[o] = a.history; S.ids[o] = a.ids; S.x[o] = a.x; S.y[o] = a.y; S.z[o] = a.z; S.e[o] = a.e; S.t[o] = a.t; }
    }
  }
}

// ---------------------------------------------------------------- stage 4: coincidence windows [R27]
__global__ void __launch_bounds__(256) coincidence_flag_kernel(const SinRec *fin, const uint32_t *n_ptr, double tau, uint32_t *flag) {
  const uint32_t n = *n_ptr;
  for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < n; i += gridDim.x * 256u) {
    uint32_t f = 0;
    if (i == 0 || !(__dsub_rn(fin[i].t, fin[i - 1].t) < tau)) {      // cluster start: this thread walks the cluster
      uint32_t o = i;
      for (;;) {                                                     // o opens a window
        const double to = fin[o].t;
        uint32_t j = o + 1;
        while (j < n && __dsub_rn(fin[j].t, to) < tau) ++j;
        const uint32_t pair = (j - o == 2 && (fin[o].ids >> 26) != (fin[o + 1].ids >> 26)) ? 1u : 0u;
        if (o == i) f = pair; else flag[o] = pair;
        if (j >= n || !(__dsub_rn(fin[j].t, fin[j - 1].t) < tau)) break;   // the next opener starts a new cluster (its own thread)
        o = j;
      }
      flag[i] = f;
    }
  }
}
__global__ void __launch_bounds__(256) coincidence_write_kernel(const SinRec *fin, const uint32_t *n_ptr, const uint32_t *flag, const uint32_t *coff, CoincBuf C) {
  const uint32_t n = *n_ptr;
  for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < n; i += gridDim.x * 256u) {
    if (!flag[i]) continue;
    const uint32_t o = coff[i];
    if (o >= C.capacity) continue;
    SinRec a, b; store_rec(&a, &fin[i]); store_rec(&b, &fin[i + 1]);
    C.ids_a[o] = a.ids; C.ids_b[o] = b.ids; C.history_a[o] = a.history; C.history_b[o] = b.history;
    C.e_a[o] = a.e; C.e_b[o] = b.e;
    C.dt_ns[o] = (float)__dmul_rn(__dsub_rn(b.t, a.t), 1e9); C.t[o] = a.t;
  }
}

// ---------------------------------------------------------------- scratch layout + driver
namespace {
struct Layout { size_t cnt, off, bsum, bcnt, boff, flag, coff, rec, sing, fin, total; };
Layout layout(uint64_t N, uint64_t M) {
  Layout L; size_t o = 0; const uint64_t Mx = M ? M : 1;
  auto take = [&](size_t bytes) { o = (o + 255) & ~(size_t)255; size_t r = o; o += bytes; return r; };
  L.cnt = take(4 * N); L.off = take(4 * (N + 1));
  const uint64_t big = N > Mx ? N : Mx;
  L.bsum = take(4 * (big / kTile + 3));
  L.bcnt = take(4 * Mx); L.boff = take(4 * (Mx + 1));
  L.flag = take(4 * Mx); L.coff = take(4 * (Mx + 1));
  L.rec = take(32 * Mx);            // hit records by history; reused for the bucket-ordered singles
  L.sing = take(32 * Mx);           // kept singles, append order
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
  uint32_t *cnt = (uint32_t *)(s + L.cnt), *off = (uint32_t *)(s + L.off), *bsum = (uint32_t *)(s + L.bsum);
  uint32_t *bcnt = (uint32_t *)(s + L.bcnt), *boff = (uint32_t *)(s + L.boff), *flag = (uint32_t *)(s + L.flag), *coff = (uint32_t *)(s + L.coff);
  HitRec *rec = (HitRec *)(s + L.rec); SinRec *srt = (SinRec *)(s + L.rec), *sing = (SinRec *)(s + L.sing), *fin = (SinRec *)(s + L.fin);
  cudaError_t e;
  if ((e = cudaMemsetAsync(cnt, 0, 4 * N, st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(bcnt, 0, 4 * M, st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(flag, 0, 4 * M, st)) != cudaSuccess) return e;
  const uint32_t nh = (uint32_t)n_hits, np = (uint32_t)N, first_lo = (uint32_t)first_history;
  // 1. counting sort by history
  if (nh) { count_hits_kernel<<<grid_for(nh), 256, 0, st>>>(H, nh, first_lo, np, cnt); count_launch(); }
  if ((e = exclusive_scan(cnt, N, off, bsum, nullptr, st)) != cudaSuccess) return e;
  if (nh) { scatter_hits_kernel<<<grid_for(nh), 256, 0, st>>>(H, nh, first_lo, np, off, cnt, rec); count_launch(); }
  // 2. adder, blur, window, time; kept singles counted into time buckets
  const uint64_t B = P.pairs_per_slice;
  const double slice_s = (double)B / P.activity_bq;
  Buckets bk; bk.nb = (uint32_t)M;
  bk.t_lo = (double)(first_history / B) * slice_s;
  const double t_hi = ((double)((first_history + n_pairs - 1) / B) + 1.0) * slice_s + 2e-6;
  bk.scale = (double)bk.nb / (t_hi - bk.t_lo);
  adder_kernel<<<grid_for(M), 256, 0, st>>>(P, bk, first_history, off, off + N, rec, sing, bcnt); count_launch();
  // 3. time-bucket counting sort
  if ((e = exclusive_scan(bcnt, M, boff, bsum, S.n, st)) != cudaSuccess) return e;
  bucket_scatter_kernel<<<grid_for(M), 256, 0, st>>>(sing, off + N, bk, boff, bcnt, srt); count_launch();
  bucket_sort_kernel<<<grid_for(M), 256, 0, st>>>(srt, P.shift, bk.nb, boff, fin, S); count_launch();
  // 4. coincidences
  const uint32_t *n_singles = boff + M;
  coincidence_flag_kernel<<<grid_for(M), 256, 0, st>>>(fin, n_singles, P.window_s, flag); count_launch();
  if ((e = exclusive_scan(flag, M, coff, bsum, C.n, st)) != cudaSuccess) return e;
  coincidence_write_kernel<<<grid_for(M), 256, 0, st>>>(fin, n_singles, flag, coff, C); count_launch();
  return cudaGetLastError();
}

}  // namespace gpet
