// gpet_transport.cu -- photon transport (S2..S10 of DESIGN.md section 1) as ONE persistent wavefront kernel.
// PAPER.md:33 (panel transfer by ray/plane crossing, global->local), PAPER.md:43 (Woodcock tracking in the
// panel frame, layer selection from the local depth, run until exit or cutoff).
//
// Design.  One CTA of 24 warps per SM, persistent.  Every warp owns a pool of 128 photon
// SLOTS in shared memory (48-byte records that never move) and one index list per NEXT EVENT: SEARCH (needs a panel
// search), STEP (Woodcock step in a panel), KN (Klein-Nishina trial), RAY (Rayleigh deflection), PHANTOM (Woodcock
// step in the voxel grid), plus the FREE list.  A pass pops up to 32 slot indices from ONE list, runs that event for
// all of them at full SIMD width, writes the changed fields back and pushes every index onto the list of its next
// event (ballot + prefix popcount).  The scheduler runs the list with the most ready photons; when no list fills a
// pass, a GEN pass samples one annihilation pair per lane (S3) and queues both photons, so a warp is never short of
// work before the end.  This is the "regroup live photons by next event" of the north star, done per warp: no
// block-level barrier, no atomics except the chunked work counter and the hit counter.  Every event's code appears
// exactly once, and the kernel is specialised on phantom / source kind / search variant to stay small.  Geometry
// descriptor and interleaved float4 mu tables live in shared memory; hits are staged per warp in shared memory and
// flushed 32 at a time: one atomicAdd per 32 hits and seven fully coalesced 128-byte stores (SoA).
#include "gpet_internal.h"

namespace gpet {

// Launch shape and pool sizes (measured on B200, C1-C4; -D overrides are for experiments only).
#ifndef GPET_THREADS
#define GPET_THREADS 768              // one CTA of 24 warps per SM: the tables are staged once, each warp gets 8.7 KB
#endif
#ifndef GPET_SLOTS
#define GPET_SLOTS 128                // photon slots per warp (20 x 160 and 28 x 104 run within 2 % of 24 x 128)
#endif
#ifndef GPET_MIN_GEN
#define GPET_MIN_GEN 24               // the source refills only when at least this many pairs fit (2 free slots each)
#endif
constexpr int kThreads = GPET_THREADS;
constexpr int kWarps = kThreads / 32;
constexpr int kStage = 64;            // staged hits per warp (ring buffer)
// the parity builds (HASH) also keep an 8-byte hash per slot and get by with 16 slots fewer
template <bool HASH> constexpr int kSlotsOf = HASH ? GPET_SLOTS - 16 : GPET_SLOTS;
constexpr uint32_t kChunk = 512;      // pairs a warp reserves at a time
constexpr int kMinGen = GPET_MIN_GEN;

enum : int { L_FREE = 0, L_SEARCH, L_STEP, L_KN, L_RAY, L_PHANTOM, kLists, L_NONE = kLists, L_GEN };

struct HitStage { uint32_t w[7][kStage]; };      // history, ids, x, y, z, e, tof

// One warp's private memory.  A photon record is 48 bytes in three 16-byte planes (one LDS.128 / STS.128 each).
template <bool HASH> struct WarpMem {
  static constexpr int kSlots = kSlotsOf<HASH>;
  float4 a[kSlots];                    // x, y, z, dx
  float4 b[kSlots];                    // dy, dz, E, path
  uint4 c[kSlots];                     // pair, meta, ids of the pending interaction, inv_mu bits
  uint2 hh[HASH ? kSlots : 1];         // outcome hash (parity builds only)
  uint8_t list[kLists][kSlots];        // slot indices by next event (stacks)
  HitStage stage;
};

// dynamic shared memory: [WarpMem x warps of the CTA][mu: n_staged x n_energies float4][DevPanel x n_panels]
template <bool HASH> struct SmemLayout {
  __host__ __device__ static size_t mu_off(int warps) { return sizeof(WarpMem<HASH>) * (size_t)warps; }
  __host__ __device__ static size_t geom_off(int warps, int n_mu) { return mu_off(warps) + sizeof(float4) * (size_t)n_mu; }
};

// ---------------------------------------------------------------- fast math with bounded error
__device__ __forceinline__ float rcp_fast(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float sqrt_fast(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
// 1/d with a zero component treated as +tiny: an inside point then sees (-inf, +inf), an outside one misses [R32]
__device__ __forceinline__ float rcp_dir(float d) { return rcp_fast(d == 0.0f ? 1e-30f : d); }
// (sin, cos) of a small angle (acolinearity, ~4e-3 rad): Taylor to x^7 / x^8 below 0.25 rad (error < 1e-9)
__device__ __forceinline__ void sincos_small(float x, float &s, float &c) {
  if (x < 0.25f) {
    const float x2 = x * x;
    s = x * fmaf(x2, fmaf(x2, fmaf(x2, -1.984126984e-4f, 8.333333333e-3f), -0.1666666667f), 1.0f);
    c = fmaf(x2, fmaf(x2, fmaf(x2, fmaf(x2, 2.48015873e-5f, -1.388888889e-3f), 4.166666667e-2f), -0.5f), 1.0f);
  } else { s = __sinf(x); c = __cosf(x); }   // > 14 degrees of acolinearity: unphysical, kept finite and cheap
}
// (sin, cos)(2 pi u), u in (0,1): argument folded to [-pi, pi] where sin.approx / cos.approx are good to 2^-21
__device__ __forceinline__ void sincos_2pi(float u, float &s, float &c) {
  const float a = 6.283185307179586f * (u - 0.5f);
  s = -__sinf(a); c = -__cosf(a);
}

// [R11] linear interpolation on the energy grid: {mu_pe, mu_pe+mu_C, mu_tot, mu_maj}
__device__ __forceinline__ float4 mu_lookup(const float4 *mu, const DevTables &T, int m, float E) {
  const float x = (E - T.e_min) * T.inv_step;
  int i = min(__float2int_rd(x), T.n_energies - 2); i = max(i, 0);
  const float f = x - (float)i;
  const int row = ((T.matmap >> (4 * m)) & 15u) * T.n_energies + i;           // staged slot of material m
  const float4 a = mu[row], b = mu[row + 1];
  return make_float4(fmaf(f, b.x - a.x, a.x), fmaf(f, b.y - a.y, a.y), fmaf(f, b.z - a.z, a.z), fmaf(f, b.w - a.w, a.w));
}

// ---------------------------------------------------------------- photon state
struct Photon {
  float x[3], d[3];        // global frame while searching / in the phantom, panel frame in STEP / KN / RAY
  float E, path, inv_mu;   // inv_mu = 1 / majorant(E) of the medium the photon is tracked in
  uint32_t pair;           // history - first_history
  uint32_t meta;           // bit0 photon, bits1-4 seq, bits5-10 panel (current, or just left; 63 = none), bit11 in
                           // phantom, bits12-17 Klein-Nishina trial counter, bits18-31 Philox blocks consumed from
                           // this photon's stream [R4] (16383 events per photon: never reached, the energy falls)
  uint32_t ids;            // lattice result of the pending interaction (KN / RAY)
};
__device__ __forceinline__ int ph_panel(const Photon &p) { return (p.meta >> 5) & 63u; }
__device__ __forceinline__ void ph_set_panel(Photon &p, int panel) { p.meta = (p.meta & ~(63u << 5)) | ((uint32_t)panel << 5); }
__device__ __forceinline__ bool ph_in_phantom(const Photon &p) { return (p.meta >> 11) & 1u; }

template <bool HASH>
__device__ __forceinline__ void slot_store(WarpMem<HASH> &W, int slot, const Photon &p, uint64_t h) {
  W.a[slot] = make_float4(p.x[0], p.x[1], p.x[2], p.d[0]);
  W.b[slot] = make_float4(p.d[1], p.d[2], p.E, p.path);
  W.c[slot] = make_uint4(p.pair, p.meta, p.ids, __float_as_uint(p.inv_mu));
  if (HASH) W.hh[slot] = make_uint2((uint32_t)h, (uint32_t)(h >> 32));
}
template <bool HASH>
__device__ __forceinline__ void slot_load(const WarpMem<HASH> &W, int slot, Photon &p, uint64_t &h) {
  const float4 a = W.a[slot], b = W.b[slot]; const uint4 c = W.c[slot];
  p.x[0] = a.x; p.x[1] = a.y; p.x[2] = a.z; p.d[0] = a.w; p.d[1] = b.x; p.d[2] = b.y; p.E = b.z; p.path = b.w;
  p.pair = c.x; p.meta = c.y; p.ids = c.z; p.inv_mu = __uint_as_float(c.w);
  if (HASH) { const uint2 v = W.hh[slot]; h = ((uint64_t)v.y << 32) | v.x; }
}

// write one staged hit (slot of this warp's ring buffer) to the global struct-of-arrays buffer
__device__ __forceinline__ void store_hit(const HitBuf &H, unsigned long long o, const HitStage &stage, uint32_t slot) {
  if (o < H.capacity) {
    H.history[o] = stage.w[0][slot]; H.ids[o] = stage.w[1][slot];
    H.x[o] = __uint_as_float(stage.w[2][slot]); H.y[o] = __uint_as_float(stage.w[3][slot]); H.z[o] = __uint_as_float(stage.w[4][slot]);
    H.e[o] = __uint_as_float(stage.w[5][slot]); H.tof[o] = __uint_as_float(stage.w[6][slot]);
  }
}
// Flush up to 32 staged hits (lane < count has one, in ring slot `slot`).  Dense layout: one atomicAdd on the global
// counter, seven coalesced stores.  Chunked layout: the hits go to the region of their 512-pair chunk; lanes of the same
// chunk (almost always all of them) share one atomicAdd on that chunk's fill counter and write consecutive entries.
__device__ __forceinline__ void flush_hits(const HitBuf &H, uint32_t first_lo, const HitStage &stage, uint32_t slot, uint32_t count, int lane) {
  const bool act = (uint32_t)lane < count;
  if (H.chunk_fill == nullptr) {
    unsigned long long base = 0;
    if (lane == 0) base = atomicAdd(H.n_hits, (unsigned long long)count);
    base = __shfl_sync(0xFFFFFFFFu, base, 0);
    if (act) store_hit(H, base + lane, stage, slot);
  } else {
    if (lane == 0) atomicAdd(H.n_hits, (unsigned long long)count);                    // total produced (no return value needed)
    const uint32_t chunk = act ? (stage.w[0][slot] - first_lo) >> kHitChunkShift : 0xFFFFFFFFu;
    const unsigned grp = __match_any_sync(0xFFFFFFFFu, chunk);
    const int leader = __ffs(grp) - 1;
    uint32_t base = 0;
    if (act && lane == leader && chunk < H.n_chunks) base = atomicAdd(&H.chunk_fill[chunk], (uint32_t)__popc(grp));
    base = __shfl_sync(0xFFFFFFFFu, base, leader);
    if (act && chunk < H.n_chunks) {
      const uint32_t pos = base + __popc(grp & ((1u << lane) - 1u));
      if (pos < H.chunk_cap) store_hit(H, (unsigned long long)chunk * H.chunk_cap + pos, stage, slot);
      else atomicAdd(&H.chunk_fill[H.n_chunks], 1u);                                   // dropped: this chunk's region is full
    }
  }
}

// [R20] Rayleigh: Thomson pdf by closed-form inversion of the cdf, then a rotation about d
__device__ __noinline__ float3 rayleigh_dir(float dx, float dy, float dz, float u_polar, float u_azimuth) {
  const float a = 4.0f * u_polar - 2.0f, q = sqrtf(a * a + 1.0f);
  const float ct = cbrtf(a + q) - cbrtf(q - a);
  float sp, cp; sincos_2pi(u_azimuth, sp, cp);
  float d[3] = { dx, dy, dz };
  rotate(d, ct, sqrtf(fmaxf(0.0f, 1.0f - ct * ct)), cp, sp);
  return make_float3(d[0], d[1], d[2]);
}
__device__ __forceinline__ void rayleigh(float d[3], float u_polar, float u_azimuth) {
  const float3 r = rayleigh_dir(d[0], d[1], d[2], u_polar, u_azimuth);
  d[0] = r.x; d[1] = r.y; d[2] = r.z;
}

// [R13] decay site from the activity map: voxel by the integer cdf (word 0), uniform point inside (words 1-3)
__device__ __forceinline__ void decay_site(const DevSource &src, uint4 w, float x[3]) {
  const uint64_t Wl = src.w_total & 0xFFFFFFFFull, Wh = src.w_total >> 32;          // floor(w.x * W / 2^32), exact
  const uint64_t target = (uint64_t)w.x * Wh + (((uint64_t)w.x * Wl) >> 32);
  uint32_t lo = 0, hi = src.n_active - 1;
  while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (src.act_cdf[mid] > target) hi = mid; else lo = mid + 1; }
  const uint32_t vi = src.act_index[lo], nx = (uint32_t)src.dims[0], ny = (uint32_t)src.dims[1];
  x[0] = src.origin[0] + ((float)(vi % nx) + u01(w.y)) * src.voxel[0];
  x[1] = src.origin[1] + ((float)((vi / nx) % ny) + u01(w.z)) * src.voxel[1];
  x[2] = src.origin[2] + ((float)(vi / (nx * ny)) + u01(w.w)) * src.voxel[2];
}

// ---------------------------------------------------------------- acceptance pre-test (planar detectors)
// Every panel point lies at least bore_r from the z axis and inside the common axial range [blo[1], bhi[1]) (z is the
// axial coordinate of every panel of a planar detector).  A photon inside the bore needs at least (bore_r - r0) / |d_xy|
// of path to reach that radius; if by then it has already passed an axial end, moving away from it, it can meet no
// panel: the search of [R6] would return "escapes".  Half of the photons of a centred source leave this way.
__device__ __forceinline__ bool misses_detector(const DevGeomHead &g, const float x[3], const float d[3]) {
  if (!(g.bore_r > 0.0f)) return false;
  const float r0sq = fmaf(x[0], x[0], x[1] * x[1]);
  if (r0sq >= g.bore_r * g.bore_r) return false;
  const float t = (g.bore_r - sqrt_fast(r0sq)) * rcp_fast(sqrt_fast(fmaf(d[0], d[0], d[1] * d[1])) + 1e-30f) * 0.9999f;
  const float z1 = fmaf(d[2], t, x[2]);                              // axial position when the bore radius can first be reached
  return (d[2] > 0.0f && z1 > g.bhi[1] + 1e-3f) || (d[2] < 0.0f && z1 < g.blo[1] - 1e-3f);
}

// ---------------------------------------------------------------- [R6] panel search
// Nearest-entry panel over all panels but `excl`; ties keep the lowest index; -1 = escapes.
// Two steps.  (1) Cull: a panel stays a candidate only if the ray passes the circle (planar detectors) or
// sphere about its box, ahead of the photon -- 6 / 11 operations per panel instead of a slab test; the bound
// carries a margin far above fp32 rounding, so no panel the slab test would accept is ever dropped.  (2) The
// surviving panels (about one per photon) take the slab test of [R6] in ascending index order, so the
// decision -- including ties -- is the one the loop over all panels makes.
// "planar" detectors (every panel has v = +z, u_z = w_z = o_z = 0: any ring built in repetition mode,
// PAPER.md:33) share the axial slab and need only the 2-D part of each pose; the arithmetic on the
// surviving terms is the generic one (the dropped terms are exact zeros).
template <int PLANAR>
__device__ __forceinline__ int panel_search(const DevGeomHead &g, const DevPanel *pan, const float x[3], const float d[3], int excl, float &t_enter) {
  float bt = INFINITY; int bp = -1;
  if (PLANAR < 0 ? g.planar != 0 : PLANAR != 0) {
    const float iz = rcp_dir(d[2]);
    const float z1 = (g.blo[1] - x[2]) * iz, z2 = (g.bhi[1] - x[2]) * iz;
    const float tnz = fmaxf(fminf(z1, z2), 0.0f), tfz = fmaxf(z1, z2);
    // circle test in the form cross = c x d - L, dot = c . d - M with L = x x d, M = x . d (four FMAs per panel); the
    // 1e-4 mm of absolute slack covers the cancellation error of that form for nearly axial rays
    const float sr = fmaf(g.cull_r2, sqrt_fast(fmaf(d[0], d[0], d[1] * d[1])), 1e-4f);
    const float Lz = fmaf(x[0], d[1], -x[1] * d[0]), Mz = fmaf(x[0], d[0], x[1] * d[1]);
    const bool axial_ok = tfz > tnz;
    for (int base = 0; base < g.n_panels; base += 32) {
      const int nq = min(32, g.n_panels - base);
      uint32_t cand = 0, bit = 1u;
#pragma unroll 4
      for (int q = 0; q < nq; ++q, bit <<= 1) {
        const float cx = g.ctr[base + q][0], cy = g.ctr[base + q][1];
        const float cross = fmaf(cx, d[1], fmaf(-cy, d[0], -Lz)), dot = fmaf(cx, d[0], fmaf(cy, d[1], -Mz));
        if (fmaxf(fabsf(cross), -dot) <= sr) cand |= bit;                  // |cross| <= sr and dot >= -sr
      }
      if ((unsigned)(excl - base) < 32u) cand &= ~(1u << (excl - base));
      if (!axial_ok) cand = 0;
      while (cand) {
        const int q = base + __ffs(cand) - 1; cand &= cand - 1;
        const float *P = pan[q].pose;
        const float r0 = x[0] - P[0], r1 = x[1] - P[1];
        const float a = r0 * P[3] + r1 * P[4], c = r0 * P[9] + r1 * P[10];
        const float ia = rcp_dir(d[0] * P[3] + d[1] * P[4]), ic = rcp_dir(d[0] * P[9] + d[1] * P[10]);
        const float a1 = (g.blo[0] - a) * ia, a2 = (g.bhi[0] - a) * ia, c1 = (g.blo[2] - c) * ic, c2 = (g.bhi[2] - c) * ic;
        const float tn = fmaxf(tnz, fmaxf(fminf(a1, a2), fminf(c1, c2)));
        const float tf = fminf(tfz, fminf(fmaxf(a1, a2), fmaxf(c1, c2)));
        if (tf > tn && tn < bt) { bt = tn; bp = q; }
      }
    }
  } else {
    for (int base = 0; base < g.n_panels; base += 32) {
      const int nq = min(32, g.n_panels - base);
      uint32_t cand = 0;
#pragma unroll 2
      for (int q = 0; q < nq; ++q) {
        const float rx = g.ctr[base + q][0] - x[0], ry = g.ctr[base + q][1] - x[1], rz = g.ctr[base + q][2] - x[2];
        const float b = fmaf(rx, d[0], fmaf(ry, d[1], rz * d[2]));                  // |d| = 1
        const float r2 = fmaf(rx, rx, fmaf(ry, ry, rz * rz));
        if (r2 - b * b <= g.cull_r3 * g.cull_r3 * 1.0001f && b >= -g.cull_r3) cand |= 1u << q;
      }
      if ((unsigned)(excl - base) < 32u) cand &= ~(1u << (excl - base));
      while (cand) {
        const int q = base + __ffs(cand) - 1; cand &= cand - 1;
        float xl[3], dl[3];
        to_local(pan[q].pose, x, d, xl, dl);
        float tn = 0.0f, tf = INFINITY;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          const float inv = rcp_dir(dl[k]);
          const float t1 = (g.blo[k] - xl[k]) * inv, t2 = (g.bhi[k] - xl[k]) * inv;
          tn = fmaxf(tn, fminf(t1, t2)); tf = fminf(tf, fmaxf(t1, t2));
        }
        if (tf > tn && tn < bt) { bt = tn; bp = q; }
      }
    }
  }
  t_enter = bt; return bp;
}

// ---------------------------------------------------------------- the kernel
// Specialisations keep the kernel small (at ~3000 SASS instructions it is sensitive to instruction-cache misses: dropping
// the phantom code alone made the ring configs 10 % faster).  PHANTOM: the source is a voxel map with a phantom
// [R17]; KIND: source kind (0 point, 1 voxel map, -1 = read src.kind); PLANAR: panel search variant (-1 = read g.planar);
// PRETEST: fresh photons take the acceptance pre-test (misses_detector) before they get a slot.
template <bool HASH, bool PHANTOM, int KIND, int PLANAR, bool PRETEST>
__global__ void __launch_bounds__(kThreads, 1)
transport_wavefront_kernel(const __grid_constant__ DevGeomHead g, const DevPanel *panels, DevTables T, DevSource src, uint64_t first_history, uint64_t n_pairs,
                           const __grid_constant__ PhiloxKeys key, HitBuf H, uint64_t *hash_out, unsigned long long *work_counter) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n_mu = T.n_staged * T.n_energies;
  float4 *mu_s = reinterpret_cast<float4 *>(smem_raw + SmemLayout<HASH>::mu_off(blockDim.x >> 5));
  DevPanel *pan = reinterpret_cast<DevPanel *>(smem_raw + SmemLayout<HASH>::geom_off(blockDim.x >> 5, n_mu));
  const int lane = threadIdx.x & 31;
  WarpMem<HASH> &W = reinterpret_cast<WarpMem<HASH> *>(smem_raw)[threadIdx.x >> 5];
  {
    const uint32_t *gs = reinterpret_cast<const uint32_t *>(panels);
    uint32_t *gd = reinterpret_cast<uint32_t *>(pan);
    const int words = (int)(sizeof(DevPanel) / 4) * g.n_panels;
    for (int i = threadIdx.x; i < words; i += blockDim.x) gd[i] = gs[i];
    for (int i = threadIdx.x; i < n_mu; i += blockDim.x) mu_s[i] = T.mu[i];
    for (int i = lane; i < kSlotsOf<HASH>; i += 32) W.list[L_FREE][i] = (uint8_t)i;
    __syncthreads();
  }
  const float4 *mu = mu_s;
  HitStage &stage = W.stage;
  const unsigned lt_mask = (1u << lane) - 1u;
  constexpr bool use_phantom = PHANTOM;
  const int kind = KIND < 0 ? src.kind : KIND;

  uint64_t w_next = 0, w_end = 0;          // this warp's reserved pairs [w_next, w_end)
  bool exhausted = false;                  // the global counter ran past n_pairs
  uint32_t stage_head = 0, stage_cnt = 0;  // ring buffer of staged hits (warp-uniform)
  int cF = kSlotsOf<HASH>, cS = 0, cT = 0, cK = 0, cR = 0, cP = 0;   // list fill levels (warp-uniform)

  // [R4] every transport event consumes one whole Philox block of the photon's stream
  auto block_at = [&](const Photon &p, uint32_t blk) -> uint4 {
    const uint64_t history = first_history + p.pair;
    return philox4x32_10(make_uint4((uint32_t)history, (uint32_t)(history >> 32), 1u + (p.meta & 1u), blk), key);
  };
  auto next_block = [&](Photon &p) -> uint4 { const uint4 w = block_at(p, p.meta >> 18); p.meta += 1u << 18; return w; };
  // stage one hit per lane that has one; flush 32 staged hits with one atomic + coalesced stores (S10)
  auto stage_hits = [&](bool has, uint32_t pair, uint32_t hit_ids, const float xg[3], float e, float tof) {
    const unsigned who = __ballot_sync(0xFFFFFFFFu, has);
    if (who == 0) return;
    if (has) {
      const uint32_t slot = (stage_head + stage_cnt + __popc(who & lt_mask)) & (kStage - 1);
      stage.w[0][slot] = (uint32_t)(first_history + pair); stage.w[1][slot] = hit_ids;
      stage.w[2][slot] = __float_as_uint(xg[0]); stage.w[3][slot] = __float_as_uint(xg[1]); stage.w[4][slot] = __float_as_uint(xg[2]);
      stage.w[5][slot] = __float_as_uint(e); stage.w[6][slot] = __float_as_uint(tof);
    }
    stage_cnt += __popc(who);
    __syncwarp();
    if (stage_cnt >= 32) {
      flush_hits(H, (uint32_t)first_history, stage, (stage_head + lane) & (kStage - 1), 32u, lane);
      stage_head = (stage_head + 32) & (kStage - 1); stage_cnt -= 32;
      __syncwarp();
    }
  };
  // push the slot index of every lane with `pred` onto list L (ballot + prefix popcount)
  auto push = [&](int L, int &cnt, bool pred, int idx) {
    const unsigned m = __ballot_sync(0xFFFFFFFFu, pred);
    if (pred) W.list[L][cnt + __popc(m & lt_mask)] = (uint8_t)idx;
    cnt += __popc(m);
  };

#pragma unroll 1
  for (;;) {
    // ================================================ scheduler: the list with the most ready photons; when no list
    // fills a pass, the source refills the SEARCH list with up to 32 fresh pairs (two free slots each)
    const bool more_src = !exhausted || w_next < w_end;
    int phase = L_SEARCH, best = cS;
    if (cT > 0 && cT >= best) { phase = L_STEP; best = cT; }
    if (cK > best) { phase = L_KN; best = cK; }
    if (PHANTOM && cP > best) { phase = L_PHANTOM; best = cP; }
    if (cR > best) { phase = L_RAY; best = cR; }
    const int np = more_src ? min(32, cF >> 1) : 0;
    if (best < 32 && np >= kMinGen) phase = L_GEN;
    else if (best == 0) { if (np > 0) phase = L_GEN; else break; }      // nothing in flight: last pairs, or done

    if (phase == L_GEN) {
      // ---------------------------------------------- GEN: one annihilation pair per lane (S3) [R13-R16]: both photons
      // get a slot and wait for their panel search (or, born inside a phantom, for their first phantom step [R17])
      if (w_next >= w_end && !exhausted) {
        unsigned long long b = 0;
        if (lane == 0) b = atomicAdd(work_counter, (unsigned long long)kChunk);
        b = __shfl_sync(0xFFFFFFFFu, b, 0);
        if (b >= n_pairs) { exhausted = true; w_next = w_end = 0; }
        else { w_next = b; w_end = min((uint64_t)(b + kChunk), n_pairs); }
      }
      const uint64_t j = w_next + (uint64_t)lane;
      const int ng = (int)min((uint64_t)np, w_end - w_next);           // pairs generated in this pass (warp-uniform)
      w_next += (uint64_t)ng;
      Photon qa = {}, qb = {}; bool fa = false, fb = false;
      if (lane < ng) {
        Photon q = {};
        q.pair = (uint32_t)j; q.meta = 63u << 5; q.ids = kNone; q.E = 511.0f; q.path = 0.0f; q.inv_mu = 0.0f;
        const uint64_t history = first_history + j;
        const uint32_t h_lo = (uint32_t)history, h_hi = (uint32_t)(history >> 32);
        q.x[0] = src.pos[0]; q.x[1] = src.pos[1]; q.x[2] = src.pos[2];
        if (kind == 1) decay_site(src, philox4x32_10(make_uint4(h_lo, h_hi, 0u, 0u), key), q.x);
        const uint4 w = philox4x32_10(make_uint4(h_lo, h_hi, 0u, 1u), key);
        if (kind == 2) { q.d[0] = src.beam[0]; q.d[1] = src.beam[1]; q.d[2] = src.beam[2]; }
        else {
          const float u = u01(w.x), ct = 1.0f - 2.0f * u, sth = 2.0f * sqrtf(u * (1.0f - u));   // sin^2 = (1-ct)(1+ct)
          float sp, cp; sincospif(2.0f * u01(w.y), &sp, &cp);
          q.d[0] = sth * cp; q.d[1] = sth * sp; q.d[2] = ct;
        }
        if (use_phantom) { q.meta |= 1u << 11; q.inv_mu = rcp_fast(mu_lookup(mu, T, src.ph_major, q.E).z); }
        auto make_b = [&]() {                                       // photon B: opposite, plus acolinearity
          q.d[0] = -q.d[0]; q.d[1] = -q.d[1]; q.d[2] = -q.d[2];
          if (src.acol_sigma > 0.0f) {
            const float rho = src.acol_sigma * sqrt_fast(-2.0f * __logf(u01(w.z)));
            float sr, cr; sincos_small(rho, sr, cr);
            float sp, cp; sincos_2pi(u01(w.w), sp, cp);               // azimuth of a ~4e-3 rad deviation: 2^-21 is ample
            rotate(q.d, cr, sr, cp, sp);
          }
          q.meta |= 1u;
        };
        if (!PRETEST) {                                               // both photons take a slot: SEARCH, or PHANTOM when born there [R17]
          uint8_t *dst = use_phantom ? &W.list[L_PHANTOM][cP] : &W.list[L_SEARCH][cS];
          const int ia = W.list[L_FREE][cF - 1 - 2 * lane], ib = W.list[L_FREE][cF - 2 - 2 * lane];
          slot_store(W, ia, q, 0xCBF29CE484222325ull);
          make_b();
          slot_store(W, ib, q, 0xCBF29CE484222325ull);
          dst[2 * lane] = (uint8_t)ia; dst[2 * lane + 1] = (uint8_t)ib;
        } else {
          // a photon that cannot reach the detector ends here (ESCAPE); the others take a slot and wait for their search
          fa = !misses_detector(g, q.x, q.d);
          if (HASH && !fa) { uint64_t ha = 0xCBF29CE484222325ull; hash_ev(ha, EV_ESCAPE, 0); hash_out[2ull * q.pair] = ha; }
          qa = q;
          make_b();
          fb = !misses_detector(g, q.x, q.d);
          if (HASH && !fb) { uint64_t hb2 = 0xCBF29CE484222325ull; hash_ev(hb2, EV_ESCAPE, 0); hash_out[2ull * q.pair + 1] = hb2; }
          qb = q;
        }
      }
      if (!PRETEST) { cF -= 2 * ng; if (use_phantom) cP += 2 * ng; else cS += 2 * ng; }
      else {
        const unsigned mA = __ballot_sync(0xFFFFFFFFu, fa), mB = __ballot_sync(0xFFFFFFFFu, fb);
        const int ra = __popc(mA & lt_mask), na = __popc(mA), rb = __popc(mB & lt_mask), nb = __popc(mB);
        if (fa) { const int ia = W.list[L_FREE][cF - 1 - ra]; slot_store(W, ia, qa, 0xCBF29CE484222325ull); W.list[L_SEARCH][cS + ra] = (uint8_t)ia; }
        if (fb) { const int ib = W.list[L_FREE][cF - 1 - na - rb]; slot_store(W, ib, qb, 0xCBF29CE484222325ull); W.list[L_SEARCH][cS + na + rb] = (uint8_t)ib; }
        cF -= na + nb; cS += na + nb;
      }
      __syncwarp();
      continue;
    }
    if (phase == L_SEARCH) {
      // ---------------------------------------------- SEARCH: nearest panel ahead [R6], entry transform [R18]
      // (repeated without a trip through the scheduler while the list still fills a whole pass: a GEN pass leaves two)
      do {
      const int n = min(cS, 32); const bool act = lane < n;
      Photon q = {}; uint64_t hq = 0; int idx = 0;
      if (act) { idx = W.list[L_SEARCH][cS - 1 - lane]; slot_load(W, idx, q, hq); }
      cS -= n;
      int dest = L_NONE;
      if (act) {
        float bt; const int bp = panel_search<PLANAR>(g, pan, q.x, q.d, ph_panel(q), bt);
        if (bp < 0) {
          if (HASH) { hash_ev(hq, EV_ESCAPE, 0); hash_out[2ull * q.pair + (q.meta & 1u)] = hq; }
          dest = L_FREE;
        } else {
          if (HASH) hash_ev(hq, EV_ENTER, (uint32_t)bp);
          float xl[3], dl[3];
          to_local(pan[bp].pose, q.x, q.d, xl, dl);
#pragma unroll
          for (int k = 0; k < 3; ++k) { q.x[k] = fmaf(bt, dl[k], xl[k]); q.d[k] = dl[k]; }   // [R18]
          q.path += bt; ph_set_panel(q, bp);
          q.inv_mu = rcp_fast(mu_lookup(mu, T, 0, q.E).w);
          dest = L_STEP;
          slot_store(W, idx, q, hq);
        }
      }
      push(L_FREE, cF, dest == L_FREE, idx);
      push(L_STEP, cT, dest == L_STEP, idx);
      __syncwarp();
      } while (cS >= 32);
      continue;
    }
    if (phase == L_STEP) {
      // ---------------------------------------------- STEP: Woodcock step, layer selection, lattice lookup [R19]
      const int n = min(cT, 32); const bool act = lane < n;
      Photon p = {}; uint64_t h = 0; int idx = 0;
      if (act) { idx = W.list[L_STEP][cT - 1 - lane]; slot_load(W, idx, p, h); }
      cT -= n;
      int dest = L_NONE; bool hit = false; float xg[3] = {0.f, 0.f, 0.f};
      if (act) {
        const uint4 w = next_block(p);                                // [R4] free path, outcome, Rayleigh polar + azimuth
        const float s = -__logf(u01(w.x)) * p.inv_mu;
        float te[3];
#pragma unroll
        for (int k = 0; k < 3; ++k)                                   // distance to the box exit [R32]
          te[k] = ((p.d[k] >= 0.0f ? g.bhi[k] : g.blo[k]) - p.x[k]) * rcp_dir(p.d[k]);
        float tf = fminf(te[0], fminf(te[1], te[2]));
        const int panel = ph_panel(p);
        if (s >= tf) {                                                // leaves the panel [R33]
          // Exit face = the axis that limits tf.  If no other panel has a point beyond that face (precomputed per panel
          // and face at create time: true for the back and axial faces of any ring), the search of [R6] cannot find
          // anything: the photon escapes here, with the same EXIT, ESCAPE events, and skips transform and search.
          const int kx = te[0] <= tf ? 0 : (te[1] <= tf ? 1 : 2);
          const float dk = kx == 0 ? p.d[0] : (kx == 1 ? p.d[1] : p.d[2]);
          const bool open = (pan[panel].open_faces >> (2 * kx + (dk >= 0.0f ? 1 : 0))) & 1u;
          if (HASH) hash_ev(h, EV_EXIT, (uint32_t)panel);
          if (open) {
            if (HASH) { hash_ev(h, EV_ESCAPE, 0); hash_out[2ull * p.pair + (p.meta & 1u)] = h; }
            dest = L_FREE;
          } else {
            tf = fmaxf(tf, 0.0f);
            const float xl[3] = { fmaf(tf, p.d[0], p.x[0]), fmaf(tf, p.d[1], p.x[1]), fmaf(tf, p.d[2], p.x[2]) };
            const float dl[3] = { p.d[0], p.d[1], p.d[2] };
            p.path += tf;
            point_to_global(pan[panel].pose, xl, p.x); dir_to_global(pan[panel].pose, dl, p.d);   // back to the global frame
            dest = L_SEARCH;
          }
        } else {
#pragma unroll
          for (int k = 0; k < 3; ++k) p.x[k] = fmaf(s, p.d[k], p.x[k]);
          p.path += s;
          uint32_t id;                                                // depth -> layer -> crystal
          const int mat = lattice_lookup(g, __float2int_rd(p.x[0] * kQ) + g.hWq, __float2int_rd(p.x[1] * kQ) + g.hHq,
                                         __float2int_rd(p.x[2] * kQ), id);
          dest = L_STEP;
          if (mat < 0) { if (HASH) hash_ev(h, EV_STEP_VACUUM, 0); }
          else {
            if (id != kNone) id |= (uint32_t)panel << 26;
            const float4 m4 = mu_lookup(mu, T, mat, p.E);
            const float t = u01(w.y) * m4.w;                          // [R20] one draw picks the outcome
            p.ids = id;
            if (t < m4.x) {                                           // photoelectric: deposit E, end
              if (HASH) { hash_ev(h, EV_PE, id); hash_out[2ull * p.pair + (p.meta & 1u)] = h; }
              if (id != kNone) { hit = true; point_to_global(pan[panel].pose, p.x, xg); }
              dest = L_FREE;
            } else if (t < m4.y) dest = L_KN;
            else if (t < m4.z) { dest = L_RAY; if (HASH) hash_ev(h, EV_RAYLEIGH, id); }   // deflected in its own pass
            else if (HASH) hash_ev(h, EV_VIRTUAL, id);
          }
        }
      }
      stage_hits(hit, p.pair, p.ids | ((p.meta & 1u) << 4) | ((p.meta >> 1) & 15u), xg, p.E, p.path * kInvC);
      if (act && dest != L_FREE) slot_store(W, idx, p, h);
      push(L_STEP, cT, dest == L_STEP, idx);
      push(L_KN, cK, dest == L_KN, idx);
      push(L_FREE, cF, dest == L_FREE, idx);
      if (__any_sync(0xFFFFFFFFu, dest == L_SEARCH || dest == L_RAY)) {   // the rare destinations share one vote
        push(L_SEARCH, cS, dest == L_SEARCH, idx);
        push(L_RAY, cR, dest == L_RAY, idx);
      }
    } else if (phase == L_KN) {
      // ---------------------------------------------- KN: one Klein-Nishina trial per visit [R20]
      const int n = min(cK, 32); const bool act = lane < n;
      Photon p = {}; uint64_t h = 0; int idx = 0;
      if (act) { idx = W.list[L_KN][cK - 1 - lane]; slot_load(W, idx, p, h); }
      cK -= n;
      int dest = L_NONE; bool hit = false; float xg[3] = {0.f, 0.f, 0.f}, e_dep = 0.f; uint32_t hit_ids = 0;
      if (act) {
        const bool in_ph = PHANTOM && ph_in_phantom(p);
        const float k = p.E * (1.0f / kMec2), e0 = rcp_fast(1.0f + 2.0f * k), e02 = e0 * e0;
        const float a1 = -__logf(e0), a2 = 0.5f * (1.0f - e02);
        const uint4 w = next_block(p);                                // [R4] u_a, u_b, u_c, azimuth
        const float ua = u01(w.x), ub = u01(w.y), uc = u01(w.z);
        // om = 1 - eps and em = eps - eps0 are formed without cancellation, so that sin^2 = t (2 - t) keeps
        // full relative accuracy at both poles (t = om/(k eps), 2 - t = em/(eps0 k eps)); plain fp32 loses
        // 3-4 digits of small scattering angles and moves later hits by micrometres
        float eps, om, em;
        if (ua * (a1 + a2) < a1) {
          if (ub < 0.5f) { om = -expm1f(-a1 * ub); eps = 1.0f - om; em = eps - e0; }
          else { em = e0 * expm1f(a1 * (1.0f - ub)); eps = e0 + em; om = 1.0f - eps; }
        } else {
          eps = sqrt_fast(fmaf(1.0f - e02, ub, e02));
          om = (1.0f - e02) * (1.0f - ub) * rcp_fast(1.0f + eps); em = (1.0f - e02) * ub * rcp_fast(eps + e0);
        }
        const float ike = rcp_fast(k * eps);
        const float t = om * ike, tm = em * ike * (1.0f + 2.0f * k);
        const float gr = 1.0f - eps * t * tm * rcp_fast(1.0f + eps * eps);
        dest = L_KN;
        if (gr >= uc || ((p.meta >> 12) & 63u) >= 63u) {              // accepted [R22: the 64th trial always is]
          p.meta &= ~(63u << 12);
          float sp, cp; sincos_2pi(u01(w.w), sp, cp);
          rotate(p.d, 1.0f - t, sqrt_fast(fmaxf(t * tm, 0.0f)), cp, sp);
          const float dep = om * p.E, E2 = p.E - dep;
          const bool cut = E2 < kCutoff;                              // [R12]
          if (in_ph) {
            if (HASH) { hash_ev(h, EV_PH_COMPTON, 0); if (cut) hash_ev(h, EV_PH_CUTOFF, 0); }
            if (!cut) { p.E = E2; p.inv_mu = rcp_fast(mu_lookup(mu, T, src.ph_major, p.E).z); dest = L_PHANTOM; }
          } else {
            if (HASH) { hash_ev(h, EV_COMPTON, p.ids); if (cut) hash_ev(h, EV_CUTOFF, p.ids); }
            if (p.ids != kNone) {
              hit = true; e_dep = cut ? p.E : dep; point_to_global(pan[ph_panel(p)].pose, p.x, xg);
              const uint32_t seq = (p.meta >> 1) & 15u;
              hit_ids = p.ids | ((p.meta & 1u) << 4) | seq;
              if (seq < 15u) p.meta += 2u;                            // [R9] 4-bit saturating hit counter
            }
            if (!cut) { p.E = E2; p.inv_mu = rcp_fast(mu_lookup(mu, T, 0, p.E).w); dest = L_STEP; }
          }
          if (cut) { if (HASH) hash_out[2ull * p.pair + (p.meta & 1u)] = h; dest = L_FREE; }
        } else p.meta += 1u << 12;
      }
      stage_hits(hit, p.pair, hit_ids, xg, e_dep, p.path * kInvC);
      if (act && dest != L_FREE) slot_store(W, idx, p, h);
      push(L_KN, cK, dest == L_KN, idx);
      push(L_STEP, cT, dest == L_STEP, idx);
      push(L_FREE, cF, dest == L_FREE, idx);
      if (use_phantom) push(L_PHANTOM, cP, dest == L_PHANTOM, idx);
    } else if (phase == L_RAY) {
      // ---------------------------------------------- RAY: Rayleigh deflection with words 2-3 of the step's block [R4, R20]
      const int n = min(cR, 32); const bool act = lane < n;
      Photon p = {}; uint64_t h = 0; int idx = 0;
      if (act) { idx = W.list[L_RAY][cR - 1 - lane]; slot_load(W, idx, p, h); }
      cR -= n;
      int dest = L_NONE;
      if (act) {
        const uint4 w = block_at(p, (p.meta >> 18) - 1u);             // the block its Woodcock step drew (rare event: recomputed)
        rayleigh(p.d, u01(w.z), u01(w.w));
        dest = (PHANTOM && ph_in_phantom(p)) ? L_PHANTOM : L_STEP;
        slot_store(W, idx, p, h);
      }
      push(L_STEP, cT, dest == L_STEP, idx);
      if (use_phantom) push(L_PHANTOM, cP, dest == L_PHANTOM, idx);
    } else if (PHANTOM) {
      // ---------------------------------------------- PHANTOM: Woodcock tracking in the voxel grid [R17]
      const int n = min(cP, 32); const bool act = lane < n;
      Photon p = {}; uint64_t h = 0; int idx = 0;
      if (act) { idx = W.list[L_PHANTOM][cP - 1 - lane]; slot_load(W, idx, p, h); }
      cP -= n;
      int dest = L_NONE;
      if (act) {
        const uint4 w = next_block(p);                                // [R4]
        const float s = -__logf(u01(w.x)) * p.inv_mu;
        int v[3]; bool out = false; float xt[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          xt[k] = fmaf(s, p.d[k], p.x[k]);
          v[k] = __float2int_rd((xt[k] - src.origin[k]) * src.inv_voxel[k]);
          out = out || v[k] < 0 || v[k] >= src.dims[k];
        }
        // tentative point outside the grid: the photon leaves along its line of flight from where it is [R17]
        if (out) {
          if (HASH) hash_ev(h, EV_PH_LEAVE, 0);
          p.meta &= ~(1u << 11); dest = L_SEARCH;
          if (misses_detector(g, p.x, p.d)) {                         // cannot reach the detector: ESCAPE without a search
            if (HASH) { hash_ev(h, EV_ESCAPE, 0); hash_out[2ull * p.pair + (p.meta & 1u)] = h; }
            dest = L_FREE;
          }
        }
        else {
          p.x[0] = xt[0]; p.x[1] = xt[1]; p.x[2] = xt[2]; p.path += s;
          dest = L_PHANTOM;
          const int mat = (int)src.phantom[((size_t)v[2] * src.dims[1] + v[1]) * src.dims[0] + v[0]] - 1;
          if (mat >= 0) {
            const float4 m4 = mu_lookup(mu, T, mat, p.E);
            const float t = u01(w.y) * mu_lookup(mu, T, src.ph_major, p.E).z;
            if (t < m4.x) { if (HASH) { hash_ev(h, EV_PH_ABSORBED, 0); hash_out[2ull * p.pair + (p.meta & 1u)] = h; } dest = L_FREE; }
            else if (t < m4.y) dest = L_KN;
            else if (t < m4.z) { dest = L_RAY; if (HASH) hash_ev(h, EV_PH_RAYLEIGH, 0); }
          }
        }
        if (dest != L_FREE) slot_store(W, idx, p, h);
      }
      push(L_PHANTOM, cP, dest == L_PHANTOM, idx);
      push(L_SEARCH, cS, dest == L_SEARCH, idx);
      push(L_KN, cK, dest == L_KN, idx);
      push(L_FREE, cF, dest == L_FREE, idx);
      push(L_RAY, cR, dest == L_RAY, idx);
    }
    __syncwarp();
  }

  // ------------------------------------------------ drain the staged hits (fewer than 32 per warp)
  if (stage_cnt) flush_hits(H, (uint32_t)first_history, stage, (stage_head + lane) & (kStage - 1), stage_cnt, lane);
}

static int g_transport_warps = kWarps;             // warps per CTA (one CTA per SM); fewer leave room for other streams' kernels
void set_transport_warps(int warps) { g_transport_warps = warps < 1 ? kWarps : (warps > kWarps ? kWarps : warps); }
int transport_warps() { return g_transport_warps; }

size_t transport_smem_bytes(const DevTables &T, int n_panels, bool hash) {
  const int n_mu = T.n_staged * T.n_energies, w = g_transport_warps;
  return (hash ? SmemLayout<true>::geom_off(w, n_mu) : SmemLayout<false>::geom_off(w, n_mu)) + panel_bytes(n_panels);
}

cudaError_t launch_transport(const DevGeom &host_geom, const DevGeom *geom, const DevTables &T, const DevSource &src,
                             uint64_t first_history, uint64_t n_pairs, uint64_t seed, const HitBuf &H, uint64_t *hash_out,
                             unsigned long long *work_counter, int sm_count, cudaStream_t stream) {
  const int n_panels = host_geom.n_panels, planar_hint = host_geom.planar;
  const DevGeomHead &head = host_geom;
  const DevPanel *panels = reinterpret_cast<const DevPanel *>(reinterpret_cast<const char *>(geom) +
                                                            (reinterpret_cast<const char *>(&host_geom.panel[0]) - reinterpret_cast<const char *>(&host_geom)));
  const size_t smem = transport_smem_bytes(T, n_panels, hash_out != nullptr);
  const int threads = 32 * g_transport_warps;
  const uint64_t want = (2 * n_pairs + threads - 1) / threads;
  const uint64_t resident = (uint64_t)sm_count;                      // persistent grid: one CTA per SM
  PhiloxKeys key;                                                     // [R1] round keys: key + r * Weyl constants
  for (int r = 0; r < 10; ++r) { key.k[2 * r] = (uint32_t)seed + (uint32_t)r * 0x9E3779B9u; key.k[2 * r + 1] = (uint32_t)(seed >> 32) + (uint32_t)r * 0xBB67AE85u; }
  const int blocks = (int)(want < resident ? (want ? want : 1) : resident);
  cudaError_t e = cudaMemsetAsync(work_counter, 0, sizeof(unsigned long long), stream);
  if (e != cudaSuccess) return e;
  const bool phantom = src.kind == 1 && src.phantom != nullptr;
  // acceptance pre-test at the source (misses_detector): worth its instructions when a fair share of the photons leaves
  // through the axial ends -- for a point source, when the bore is wide compared with the axial margin (slope < 2:
  // more than 10 % of an isotropic source); always for voxel sources without a phantom (positions vary)
  int pretest = 0;
  if (!phantom && host_geom.bore_r > 0.0f) {
    if (src.kind == 1) pretest = 1;
    else {
      const double r0 = hypot((double)src.pos[0], (double)src.pos[1]);
      const double zm = fmin((double)host_geom.bhi[1] - src.pos[2], (double)src.pos[2] - host_geom.blo[1]);
      pretest = r0 < host_geom.bore_r && (zm <= 0.0 || zm < 2.0 * (host_geom.bore_r - r0));
    }
  }
  auto launch = [&](auto kernel) -> cudaError_t {
    cudaError_t le = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (le != cudaSuccess) return le;
    kernel<<<blocks, threads, smem, stream>>>(head, panels, T, src, first_history, n_pairs, key, H, hash_out, work_counter);
    return cudaSuccess;
  };
  // specialised builds for the shapes the five configs use (point source or voxel map + phantom, planar ring);
  // anything else runs the generic build of the same code
  const bool planar = planar_hint != 0;
#define GPET_DISPATCH(H)                                                                                              \
  do {                                                                                                                \
    if (!phantom && src.kind == 0 && planar && pretest) e = launch(transport_wavefront_kernel<H, false, 0, 1, true>);  \
    else if (!phantom && src.kind == 0 && planar) e = launch(transport_wavefront_kernel<H, false, 0, 1, false>);      \
    else if (phantom && planar) e = launch(transport_wavefront_kernel<H, true, 1, 1, false>);                         \
    else if (phantom) e = launch(transport_wavefront_kernel<H, true, 1, -1, false>);                                  \
    else if (pretest) e = launch(transport_wavefront_kernel<H, false, -1, -1, true>);                                 \
    else e = launch(transport_wavefront_kernel<H, false, -1, -1, false>);                                             \
  } while (0)
  if (hash_out) GPET_DISPATCH(true); else GPET_DISPATCH(false);
#undef GPET_DISPATCH
  if (e != cudaSuccess) return e;
  count_launch();
  return cudaGetLastError();
}

// ---------------------------------------------------------------- locate (indexing test entry)
// fp64 global->local transform of the fp32 point (products of two fp32 values are exact in fp64), then
// the same integer lattice code as the transport kernel.
__global__ void locate_kernel(const DevGeom *geom, int64_t n, const float *xyz, uint32_t *ids) {
  __shared__ DevGeom g;
  {
    const uint32_t *src = reinterpret_cast<const uint32_t *>(geom);
    uint32_t *dst = reinterpret_cast<uint32_t *>(&g);
    for (int i = threadIdx.x; i < (int)(sizeof(DevGeom) / 4); i += blockDim.x) dst[i] = src[i];
    __syncthreads();
  }
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    uint32_t out = kNone;
    for (int p = 0; p < g.n_panels; ++p) {
      const float *P = g.panel[p].pose;
      const double r0 = (double)xyz[3 * i] - (double)P[0], r1 = (double)xyz[3 * i + 1] - (double)P[1], r2 = (double)xyz[3 * i + 2] - (double)P[2];
      const double a = r0 * P[3] + r1 * P[4] + r2 * P[5], b = r0 * P[6] + r1 * P[7] + r2 * P[8], c = r0 * P[9] + r1 * P[10] + r2 * P[11];
      const long long qa = (long long)floor(a * 1048576.0) + g.hWq, qb = (long long)floor(b * 1048576.0) + g.hHq, qc = (long long)floor(c * 1048576.0);
      if (qa < 0 || qa >= g.Wq || qb < 0 || qb >= g.Hq || qc < 0 || qc >= g.Dq) continue;
      lattice_lookup(g, (int)qa, (int)qb, (int)qc, out);
      if (out != kNone) out |= (uint32_t)p << 26;
      break;
    }
    ids[i] = out;
  }
}

cudaError_t launch_locate(const DevGeom *geom, int64_t n, const float *xyz_dev, uint32_t *ids_dev, cudaStream_t stream) {
  if (n <= 0) return cudaSuccess;
  const int blocks = (int)((n + 255) / 256 < 1184 ? (n + 255) / 256 : 1184);
  locate_kernel<<<blocks, 256, 0, stream>>>(geom, n, xyz_dev, ids_dev);
  count_launch();
  return cudaGetLastError();
}

}  // namespace gpet
