// gpet_digitize.cu -- singles digitizer and coincidence sorter (S11..S14 of DESIGN.md section 1).
// PAPER.md:33,37 (single-event readout at crystal / module / panel level), PAPER.md:61 (energy resolution,
// coincidence timing window), PAPER.md:65 (list-mode coincidences).  Readings [R16], [R24]-[R27].
//
// Sort / segmented-scan structure (all hand-written, no CUB/Thrust):
//   1. counting sort of the hits by history id (dense integer keys: histogram by atomics in L2,
//      exclusive scan, scatter) -> one contiguous segment per history;
//   2. one thread per history: canonical in-segment order by repeated min-selection (segments hold
//      ~1-4 hits), adder per readout unit, blur, window, absolute time -> candidate singles;
//   3. counting sort of the kept singles by time bucket (decay times are uniform by construction
//      [R16], so buckets hold ~0.4 singles on average), in-bucket selection sort by (t, history, unit);
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
__global__ void __launch_bounds__(256) scatter_hits_kernel(HitBuf H, uint32_t bound, uint32_t first_lo, uint32_t n_pairs,
                                                           const uint32_t *off, uint32_t *cnt, uint32_t *idx) {
  const uint32_t n_hits = valid_hits(H, bound); const uint32_t *history = H.history;
  for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < n_hits; i += gridDim.x * 256u) {
    const uint32_t h = history[i] - first_lo;
    if (h < n_pairs) idx[off[h] + atomicSub(&cnt[h], 1u) - 1u] = i;
  }
}

// ---------------------------------------------------------------- stage 2: adder + blur + window + time
struct Tmp { uint32_t *history, *ids; float *x, *y, *z, *e; double *t; };

__device__ __forceinline__ double decay_time(const DigiParams &P, uint64_t history) {     // [R16]
  const uint2 key = make_uint2((uint32_t)P.seed, (uint32_t)(P.seed >> 32));
  const uint4 w = philox4x32_10(make_uint4((uint32_t)history, (uint32_t)(history >> 32), 0u, 2u), key);
  const uint64_t bits = (((uint64_t)w.x << 32) | (uint64_t)w.y) >> 11;
  const double u53 = __dmul_rn(__dadd_rn((double)bits, 0.5), 1.0 / 9007199254740992.0);
  const uint64_t B = P.pairs_per_slice;
  return __dmul_rn(__dadd_rn((double)(history / B), u53), __ddiv_rn((double)B, P.activity_bq));
}

__device__ __forceinline__ void emit_single(const DigiParams &P, const HitBuf &H, const Tmp &T, uint32_t slot, uint64_t history,
                                            uint32_t unit, float e_sum, uint32_t best, float tof_min) {
  // [R25] blur: Box-Muller on words 0,1 of Philox(counter = (history lo, 0, 3, unit))
  const uint2 key = make_uint2((uint32_t)P.seed, (uint32_t)(P.seed >> 32));
  const uint4 w = philox4x32_10(make_uint4((uint32_t)history, 0u, 3u, unit), key);
  const float nrm = sqrtf(-2.0f * logf(u01(w.x))) * cospif(2.0f * u01(w.y));
  const float sigma = P.sigma_scale * (P.ref_keV > 0.0f ? sqrtf(P.ref_keV * e_sum) : e_sum);
  const float e_b = fmaf(sigma, nrm, e_sum);
  if (!(e_b >= P.e_lo && e_b < P.e_hi)) return;                      // [R26]
  T.history[slot] = (uint32_t)history; T.ids[slot] = H.ids[best];
  T.x[slot] = H.x[best]; T.y[slot] = H.y[best]; T.z[slot] = H.z[best]; T.e[slot] = e_b;
  T.t[slot] = __dadd_rn(decay_time(P, history), __dmul_rn((double)tof_min, 1e-9));
}

__global__ void __launch_bounds__(256) adder_kernel(DigiParams P, HitBuf H, uint64_t first_history, uint32_t n_pairs,
                                                    const uint32_t *off, const uint32_t *idx, Tmp T) {
  for (uint32_t h = blockIdx.x * 256u + threadIdx.x; h < n_pairs; h += gridDim.x * 256u) {
    const uint32_t b = off[h], k = off[h + 1] - b;
    if (k == 0) continue;
    const uint64_t history = first_history + h;
    // canonical order = ascending (ids, buffer index) by repeated min-selection (k is ~1-4)      [R24]
    uint64_t prev = 0; bool first = true;
    uint32_t cur_unit = 0, best = 0, best_ord = 0, slot = b; float e_sum = 0.0f, e_best = -1.0f, tof_min = INFINITY; bool open = false;
    for (uint32_t m = 0; m < k; ++m) {
      uint64_t sel = ~0ull;
      for (uint32_t j = 0; j < k; ++j) {
        const uint32_t i = idx[b + j];
        const uint64_t key = ((uint64_t)H.ids[i] << 32) | i;
        if ((first || key > prev) && key < sel) sel = key;
      }
      prev = sel; first = false;
      const uint32_t i = (uint32_t)sel, ids = (uint32_t)(sel >> 32), unit = ids >> P.shift;
      if (open && unit != cur_unit) { emit_single(P, H, T, slot++, history, cur_unit, e_sum, best, tof_min); open = false; }
      if (!open) { open = true; cur_unit = unit; e_sum = 0.0f; e_best = -1.0f; tof_min = INFINITY; }
      const float e = H.e[i]; const uint32_t ord = ids & 31u;
      e_sum += e;
      if (e > e_best || (e == e_best && ord < best_ord)) { e_best = e; best = i; best_ord = ord; }
      tof_min = fminf(tof_min, H.tof[i]);
    }
    if (open) emit_single(P, H, T, slot, history, cur_unit, e_sum, best, tof_min);
  }
}

// ---------------------------------------------------------------- stage 3: time-bucket counting sort
struct Buckets { double t_lo, scale; uint32_t nb; };
__device__ __forceinline__ uint32_t bucket_of(const Buckets &B, double t) {
  const double x = (t - B.t_lo) * B.scale;
  if (!(x > 0.0)) return 0u;
  return x >= (double)(B.nb - 1) ? B.nb - 1 : (uint32_t)x;
}
__global__ void __launch_bounds__(256) bucket_count_kernel(Tmp T, uint32_t n, Buckets B, uint32_t *bcnt) {
  for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < n; i += gridDim.x * 256u)
    if (T.ids[i] != kNone) atomicAdd(&bcnt[bucket_of(B, T.t[i])], 1u);
}
__global__ void __launch_bounds__(256) bucket_scatter_kernel(Tmp T, uint32_t n, Buckets B, const uint32_t *boff, uint32_t *bcnt, uint32_t *sidx) {
  for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < n; i += gridDim.x * 256u)
    if (T.ids[i] != kNone) { const uint32_t b = bucket_of(B, T.t[i]); sidx[boff[b] + atomicSub(&bcnt[b], 1u) - 1u] = i; }
}
__device__ __forceinline__ bool single_less(const Tmp &T, int shift, uint32_t a, uint32_t b) {      // (t, history, unit)
  const double ta = T.t[a], tb = T.t[b];
  if (ta != tb) return ta < tb;
  const uint32_t ha = T.history[a], hb = T.history[b];
  if (ha != hb) return ha < hb;
  return (T.ids[a] >> shift) < (T.ids[b] >> shift);
}
// one thread per bucket: r-th smallest by rank counting (buckets hold ~0-3 singles), write final arrays
__global__ void __launch_bounds__(256) bucket_sort_kernel(Tmp T, int shift, uint32_t nb, const uint32_t *boff, const uint32_t *sidx,
                                                          Tmp F, SinglesBuf S) {
  for (uint32_t b = blockIdx.x * 256u + threadIdx.x; b < nb; b += gridDim.x * 256u) {
    const uint32_t s = boff[b], m = boff[b + 1] - s;
    for (uint32_t j = 0; j < m; ++j) {
      const uint32_t a = sidx[s + j]; uint32_t rank = 0;
      for (uint32_t q = 0; q < m; ++q) { const uint32_t c = sidx[s + q]; if (q != j && (single_less(T, shift, c, a) || (!single_less(T, shift, a, c) && q < j))) ++rank; }
      const uint32_t o = s + rank;
      const uint32_t hi = T.history[a], id = T.ids[a]; const float x = T.x[a], y = T.y[a], z = T.z[a], e = T.e[a]; const double t = T.t[a];
      F.history[o] = hi; F.ids[o] = id; F.x[o] = x; F.y[o] = y; F.z[o] = z; F.e[o] = e; F.t[o] = t;
      if (S.history && o < S.capacity) { S.history[o] = hi; S.ids[o] = id; S.x[o] = x; S.y[o] = y; S.z[o] = z; S.e[o] = e; S.t[o] = t; }
    }
  }
}

// ---------------------------------------------------------------- stage 4: coincidence windows [R27]
__global__ void __launch_bounds__(256) coincidence_flag_kernel(Tmp F, const uint32_t *n_ptr, double tau, uint32_t *flag) {
  const uint32_t n = *n_ptr;
  for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < n; i += gridDim.x * 256u) {
    if (i > 0 && __dsub_rn(F.t[i], F.t[i - 1]) < tau) continue;      // not a cluster start
    uint32_t o = i;
    for (;;) {                                                       // o opens a window
      const double to = F.t[o];
      uint32_t j = o + 1;
      while (j < n && __dsub_rn(F.t[j], to) < tau) ++j;
      if (j - o == 2 && (F.ids[o] >> 26) != (F.ids[o + 1] >> 26)) flag[o] = 1u;
      if (j >= n || !(__dsub_rn(F.t[j], F.t[j - 1]) < tau)) break;   // next opener starts a new cluster: its own thread handles it
      o = j;
    }
  }
}
__global__ void __launch_bounds__(256) coincidence_write_kernel(Tmp F, const uint32_t *n_ptr, const uint32_t *flag, const uint32_t *coff, CoincBuf C) {
  const uint32_t n = *n_ptr;
  for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < n; i += gridDim.x * 256u) {
    if (!flag[i]) continue;
    const uint32_t o = coff[i];
    if (o >= C.capacity) continue;
    C.ids_a[o] = F.ids[i]; C.ids_b[o] = F.ids[i + 1]; C.history_a[o] = F.history[i]; C.history_b[o] = F.history[i + 1];
    C.e_a[o] = F.e[i]; C.e_b[o] = F.e[i + 1];
    C.dt_ns[o] = (float)__dmul_rn(__dsub_rn(F.t[i + 1], F.t[i]), 1e9); C.t[o] = F.t[i];
  }
}

// ---------------------------------------------------------------- scratch layout + driver
namespace {
struct Layout {
  size_t cnt, off, idx, bsum, bcnt, boff, sidx, flag, coff, tmp_u32, tmp_f32, tmp_t, fin_u32, fin_f32, fin_t, total;
};
Layout layout(uint64_t N, uint64_t M) {
  Layout L; size_t o = 0; const uint64_t Mx = M ? M : 1;
  auto take = [&](size_t bytes) { o = (o + 255) & ~(size_t)255; size_t r = o; o += bytes; return r; };
  L.cnt = take(4 * N); L.off = take(4 * (N + 1)); L.idx = take(4 * Mx);
  const uint64_t big = N > Mx ? N : Mx;
  L.bsum = take(4 * (big / kTile + 3));
  L.bcnt = take(4 * Mx); L.boff = take(4 * (Mx + 1)); L.sidx = take(4 * Mx);
  L.flag = take(4 * Mx); L.coff = take(4 * (Mx + 1));
  L.tmp_u32 = take(8 * Mx); L.tmp_f32 = take(16 * Mx); L.tmp_t = take(8 * Mx);
  L.fin_u32 = take(8 * Mx); L.fin_f32 = take(16 * Mx); L.fin_t = take(8 * Mx);
  L.total = o + 256; return L;
}
Tmp view(char *s, size_t u32, size_t f32, size_t t, uint64_t M) {
  Tmp T; T.history = (uint32_t *)(s + u32); T.ids = T.history + M;
  T.x = (float *)(s + f32); T.y = T.x + M; T.z = T.y + M; T.e = T.z + M; T.t = (double *)(s + t); return T;
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
  uint32_t *cnt = (uint32_t *)(s + L.cnt), *off = (uint32_t *)(s + L.off), *idx = (uint32_t *)(s + L.idx), *bsum = (uint32_t *)(s + L.bsum);
  uint32_t *bcnt = (uint32_t *)(s + L.bcnt), *boff = (uint32_t *)(s + L.boff), *sidx = (uint32_t *)(s + L.sidx);
  uint32_t *flag = (uint32_t *)(s + L.flag), *coff = (uint32_t *)(s + L.coff);
  Tmp T = view(s, L.tmp_u32, L.tmp_f32, L.tmp_t, M), F = view(s, L.fin_u32, L.fin_f32, L.fin_t, M);
  cudaError_t e;
  if ((e = cudaMemsetAsync(cnt, 0, 4 * N, st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(bcnt, 0, 4 * M, st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(flag, 0, 4 * M, st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(T.ids, 0xFF, 4 * M, st)) != cudaSuccess) return e;
  const uint32_t nh = (uint32_t)n_hits, np = (uint32_t)(N == (1ull << 32) ? 0xFFFFFFFFu : N), first_lo = (uint32_t)first_history;
  // 1. counting sort by history
  if (nh) { count_hits_kernel<<<grid_for(nh), 256, 0, st>>>(H, nh, first_lo, np, cnt); count_launch(); }
  if ((e = exclusive_scan(cnt, N, off, bsum, nullptr, st)) != cudaSuccess) return e;
  if (nh) { scatter_hits_kernel<<<grid_for(nh), 256, 0, st>>>(H, nh, first_lo, np, off, cnt, idx); count_launch(); }
  // 2. adder, blur, window, time
  adder_kernel<<<grid_for(N), 256, 0, st>>>(P, H, first_history, np, off, idx, T); count_launch();
  // 3. time-bucket counting sort
  const uint64_t B = P.pairs_per_slice;
  const double slice_s = (double)B / P.activity_bq;
  Buckets bk; bk.nb = (uint32_t)M;
  bk.t_lo = (double)(first_history / B) * slice_s;
  const double t_hi = ((double)((first_history + n_pairs - 1) / B) + 1.0) * slice_s + 2e-6;
  bk.scale = (double)bk.nb / (t_hi - bk.t_lo);
  bucket_count_kernel<<<grid_for(M), 256, 0, st>>>(T, (uint32_t)M, bk, bcnt); count_launch();
  if ((e = exclusive_scan(bcnt, M, boff, bsum, S.n, st)) != cudaSuccess) return e;
  bucket_scatter_kernel<<<grid_for(M), 256, 0, st>>>(T, (uint32_t)M, bk, boff, bcnt, sidx); count_launch();
  bucket_sort_kernel<<<grid_for(M), 256, 0, st>>>(T, P.shift, bk.nb, boff, sidx, F, S); count_launch();
  // 4. coincidences
  const uint32_t *n_singles = boff + M;
  coincidence_flag_kernel<<<grid_for(M), 256, 0, st>>>(F, n_singles, P.window_s, flag); count_launch();
  if ((e = exclusive_scan(flag, M, coff, bsum, C.n, st)) != cudaSuccess) return e;
  coincidence_write_kernel<<<grid_for(M), 256, 0, st>>>(F, n_singles, flag, coff, C); count_launch();
  return cudaGetLastError();
}

}  // namespace gpet
