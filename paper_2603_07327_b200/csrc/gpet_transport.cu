// gpet_transport.cu -- photon transport (S2..S10 of DESIGN.md section 1) as ONE persistent wavefront kernel.
// PAPER.md:33 (panel transfer by ray/plane crossing, global->local), PAPER.md:43 (Woodcock tracking in the
// panel frame, layer selection from the local depth, run until exit or cutoff).
//
// Design.  One CTA of 20 warps per SM, persistent.  Every warp owns a pool of 160 photon
// SLOTS in shared memory (48-byte records that never move) and one index list per NEXT EVENT: SEARCH (needs a panel
// search), STEP (Woodcock step in a panel), KN (Klein-Nishina trial), RAY (Rayleigh deflection), PHANTOM (Woodcock
// step in the voxel grid), HIT (a deposit waiting to be written), plus the FREE list (phantom runs in a ring keep a second
// search list: SEARCH takes the polygon shortcut, SEARCHF the search over all panels).  A pass pops up to 32 slot indices
// from ONE list, runs that event for all of them at full SIMD width, writes the changed fields back and pushes every
// index onto the list of its next event (ballot + prefix popcount).  The pass bodies are written without divergent
// branches: every lane runs the same instructions and the outcome is selected at the end.  The scheduler runs any list
// that fills a pass; when none does, the source refills the pool.  For a point source inside the bore of a ring the
// source works in two stages: GEN1 draws the pair's Philox block and drops, from cos(theta) alone, the pairs that
// leave through the axial ends (half of them for a centred source); GEN2 gives the survivors their directions and
// takes each photon straight to its entry point in the panel whose polygon edge it crosses (ring_entry_fast), so the
// first panel search costs no pass of its own.  This is the "regroup live photons by next event" of the north star,
// done per warp: no block-level barrier, no atomics except the work counter and the hit counters.  Geometry header in
// the constant bank, per-panel and per-layer records and the interleaved float4 mu tables in shared memory; hits are
// written 32 at a time by the HIT pass: one atomicAdd per 32 hits and seven fully coalesced 128-byte stores (SoA).
#include <cstdio>
#include "gpet_internal.h"

namespace gpet {

// Launch shape and pool sizes (measured on B200, C1-C4; -D overrides are for experiments only).
#ifndef GPET_THREADS
#define GPET_THREADS 640              // one CTA of 20 warps per SM: the tables are staged once, each warp gets ~10.5 KB
#endif
#ifndef GPET_SLOTS
#define GPET_SLOTS 160                // photon slots per warp (measured on C1 / C3 / C4: 20 x 160 beats 24 x 128 and 22 x 144 by 1-5 %)
#endif
#ifndef GPET_MIN_GEN
#define GPET_MIN_GEN 32               // the one-stage source (voxel map, beam) refills only when a full pass of pairs fits (measured on C4: 16 / 24 / 32 -> 8.89 / 8.73 / 8.64 ms)
#endif
#ifndef GPET_GRAB
#define GPET_GRAB 128                 // pairs a warp reserves at a time (multiple of 32): short tails at the end of a launch
#endif
constexpr int kThreads = GPET_THREADS;
constexpr int kWarps = kThreads / 32;
constexpr int kQueue = 64;            // pair queue between the two source stages
constexpr int kReserve = 32;          // free slots kept for the deposits of a Klein-Nishina pass
// the parity builds (HASH) also keep an 8-byte hash per slot and get by with 16 slots fewer
template <bool HASH> constexpr int kSlotsOf = HASH ? GPET_SLOTS - 16 : GPET_SLOTS;
constexpr uint32_t kGrab = GPET_GRAB;
constexpr int kMinGen = GPET_MIN_GEN;
constexpr uint64_t kHash0 = 0xCBF29CE484222325ull;

enum : int { L_FREE = 0, L_SEARCH, L_STEP, L_KN, L_RAY, L_PHANTOM, L_HIT, kLists, L_SEARCHF = kLists, L_NONE = kLists + 1 };   // L_SEARCHF: builds without the pair queue only

// One warp's private memory.  A photon record is 48 bytes in three 16-byte planes (one LDS.128 / STS.128 each).
// (QUEUE: the build has the two-stage point source and its pair queue; the others leave that memory to the tables)
template <bool HASH, bool QUEUE> struct WarpMem {
  static constexpr int kSlots = kSlotsOf<HASH>;
  float4 a[kSlots];                    // x, y, z, path      (panel frame in STEP / KN / RAY / HIT and after an exit, else global)
  float4 b[kSlots];                    // dx, dy, dz, E
  uint4 c[kSlots];                     // pair, meta, ids of the pending interaction, 1/mu_maj bits (HIT: deposited energy bits)
  uint2 hh[HASH ? kSlots : 1];         // outcome hash (parity builds only)
  uint4 qw[QUEUE ? kQueue : 1];        // pair queue: the pair's source block [R3] ...
  uint32_t qp[QUEUE ? kQueue : 1];     // ... its index in the batch ...
  float2 qd[QUEUE ? kQueue : 1];                   // ... and, once photon A is placed, the transverse part of its direction (photon B starts from -d)
  uint8_t list[kLists + (QUEUE ? 0 : 1)][kSlots];   // slot indices by next event (stacks)
};

// dynamic shared memory: [WarpMem x warps of the CTA][mu: n_staged x n_energies float4][DevLayer x 4][DevPanel x (n_panels + 1)]
template <bool HASH, bool QUEUE> struct SmemLayout {
  __host__ __device__ static size_t mu_off(int warps) { return sizeof(WarpMem<HASH, QUEUE>) * (size_t)warps; }
  __host__ __device__ static size_t layer_off(int warps, int n_mu) { return mu_off(warps) + sizeof(float4) * (size_t)n_mu; }
  __host__ __device__ static size_t geom_off(int warps, int n_mu) { return layer_off(warps, n_mu) + sizeof(DevLayer) * kMaxLayers; }
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
// exp(x) - 1 for |x| <= 0.55 (Klein-Nishina: |x| <= ln(3)/2): Taylor to x^11, relative error below one ulp
__device__ __forceinline__ float expm1_small(float x) {
  float p = 2.505210839e-8f;                                           // 1/11!
  p = fmaf(p, x, 2.755731922e-7f); p = fmaf(p, x, 2.755731922e-6f); p = fmaf(p, x, 2.480158730e-5f);
  p = fmaf(p, x, 1.984126984e-4f); p = fmaf(p, x, 1.388888889e-3f); p = fmaf(p, x, 8.333333333e-3f);
  p = fmaf(p, x, 4.166666667e-2f); p = fmaf(p, x, 0.1666666667f); p = fmaf(p, x, 0.5f);
  return fmaf(p * x, x, x);
}
// atan2 good to ~1e-3 rad (it only proposes the first candidate panel of ring_entry_fast)
__device__ __forceinline__ float atan2_coarse(float y, float x) {
  const float ax = fabsf(x), ay = fabsf(y), mx = fmaxf(ax, ay), mn = fminf(ax, ay);
  const float q = mn * rcp_fast(mx + 1e-30f), q2 = q * q;
  float r = q * fmaf(q2, fmaf(q2, 0.0793f, -0.2883f), 0.9954f);       // atan(q), q in [0, 1]
  r = ay > ax ? 1.5707963f - r : r;
  r = x < 0.0f ? 3.1415927f - r : r;
  return y < 0.0f ? -r : r;
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

// [R19] 1 / majorant of the region the photon is tracked in.  One region (all of BASELINE's configs): the whole-detector
// majorant tabulated in .w.  Several regions (layers of different materials): the interpolation of the pointwise maximum
// of mu_tot over the region's crystal and gap material.
template <bool MULTI>
__device__ __forceinline__ float inv_majorant(const float4 *mu, const DevTables &T, const DevGeomHead &g, int reg, float E) {
  if (!MULTI) return rcp_fast(mu_lookup(mu, T, 0, E).w);
  const float x = (E - T.e_min) * T.inv_step;
  int i = min(__float2int_rd(x), T.n_energies - 2); i = max(i, 0);
  const float f = x - (float)i;
  const uint32_t mats = g.reg_mats[reg];                              // crystal material | gap material << 4 (the same when there is none)
  const int ra = ((T.matmap >> (4 * (mats & 15u))) & 15u) * T.n_energies + i, rb = ((T.matmap >> (4 * (mats >> 4))) & 15u) * T.n_energies + i;
  const float lo = fmaxf(mu[ra].z, mu[rb].z), hi = fmaxf(mu[ra + 1].z, mu[rb + 1].z);
  return rcp_fast(fmaf(f, hi - lo, lo));
}

// ---------------------------------------------------------------- photon state
struct Photon {
  float x[3], d[3];        // global frame while searching (fresh photons) / in the phantom, panel frame in STEP / KN / RAY
  float E, path, inv_mu;   // inv_mu = 1 / majorant(E) of the medium the photon is tracked in
  uint32_t pair;           // history - first_history
  uint32_t meta;           // bit0 photon, bits1-4 seq, bits5-10 panel (current, or just left; 63 = none), bit11 in
                           // phantom, bits12-17 Klein-Nishina trial counter, bits18-19 majorant region [R19], bits20-31
                           // Philox blocks consumed from this photon's stream [R4] (4095 events per photon: never
                           // reached, the energy falls)
  uint32_t ids;            // lattice result of the pending interaction (KN / RAY / HIT), panel bits included
};
constexpr uint32_t kNoPanel = 63u;
constexpr int kRegShift = 18, kBlkShift = 20;
__device__ __forceinline__ int ph_panel(uint32_t meta) { return (meta >> 5) & 63u; }
__device__ __forceinline__ uint32_t ph_with_panel(uint32_t meta, int panel) { return (meta & ~(63u << 5)) | ((uint32_t)panel << 5); }

template <bool HASH, bool QUEUE>
__device__ __forceinline__ void slot_store(WarpMem<HASH, QUEUE> &W, int slot, const Photon &p, uint64_t h) {
  W.a[slot] = make_float4(p.x[0], p.x[1], p.x[2], p.path);
  W.b[slot] = make_float4(p.d[0], p.d[1], p.d[2], p.E);
  W.c[slot] = make_uint4(p.pair, p.meta, p.ids, __float_as_uint(p.inv_mu));
  if (HASH) W.hh[slot] = make_uint2((uint32_t)h, (uint32_t)(h >> 32));
}
template <bool HASH, bool QUEUE>
__device__ __forceinline__ void slot_load(const WarpMem<HASH, QUEUE> &W, int slot, Photon &p, uint64_t &h) {
  const float4 a = W.a[slot], b = W.b[slot]; const uint4 c = W.c[slot];
  p.x[0] = a.x; p.x[1] = a.y; p.x[2] = a.z; p.path = a.w; p.d[0] = b.x; p.d[1] = b.y; p.d[2] = b.z; p.E = b.w;
  p.pair = c.x; p.meta = c.y; p.ids = c.z; p.inv_mu = __uint_as_float(c.w);
  if (HASH) { const uint2 v = W.hh[slot]; h = ((uint64_t)v.y << 32) | v.x; }
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

// [R13] decay site from the activity map: voxel by the integer cdf (word 0), uniform point inside (words 1-3)
__device__ __forceinline__ void decay_site(const DevSource &src, uint4 w, float x[3]) {
  const uint64_t Wl = src.w_total & 0xFFFFFFFFull, Wh = src.w_total >> 32;          // floor(w.x * W / 2^32), exact
  const uint64_t target = (uint64_t)w.x * Wh + (((uint64_t)w.x * Wl) >> 32);
  uint32_t lo = src.act_guide[w.x >> (32 - kActGuideBits)], hi = src.act_guide[(w.x >> (32 - kActGuideBits)) + 1];   // brackets the answer
  while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (src.act_cdf[mid] > target) hi = mid; else lo = mid + 1; }
  // voxel index -> (ix, iy, iz): exact multiply-high divisions (QDiv; magic = 0 stands for a divisor of 1)
  const uint32_t vi = src.act_index[lo], nx = (uint32_t)src.dims[0], nxy = nx * (uint32_t)src.dims[1];
  const uint32_t iz = src.div_nxy.magic ? __umulhi(vi, src.div_nxy.magic) >> src.div_nxy.shift : vi, r = vi - iz * nxy;
  const uint32_t iy = src.div_nx.magic ? __umulhi(r, src.div_nx.magic) >> src.div_nx.shift : r, ix = r - iy * nx;
  x[0] = src.origin[0] + ((float)ix + u01(w.y)) * src.voxel[0];
  x[1] = src.origin[1] + ((float)iy + u01(w.z)) * src.voxel[1];
  x[2] = src.origin[2] + ((float)iz + u01(w.w)) * src.voxel[2];
}

// ---------------------------------------------------------------- acceptance pre-test (planar detectors)
// Every panel point lies at least bore_r from the z axis and inside the common axial range [blo[1], bhi[1]) (z is the
// axial coordinate of every panel of a planar detector).  A photon inside the bore needs at least (bore_r - r0) / |d_xy|
// of path to reach that radius; if by then it has already passed an axial end, moving away from it, it can meet no
// panel: the search of [R6] would return "escapes".  Half of the photons of a centred source leave this way.
// Form used by both callers: r0 = distance of the start point from the axis (< bore_r), z0 its axial coordinate,
// sxy <= |d_xy| is NOT required -- pass an upper bound of |d_xy| and a lower bound of |d_z| for a conservative answer.
__device__ __forceinline__ bool misses_axially(const DevGeomHead &g, float r0, float z0, float sxy, float dz) {
  const float t = (g.bore_r - r0) * rcp_fast(sxy + 1e-30f) * 0.9999f;  // path needed to reach the bore radius, at least
  const float z1 = fmaf(dz, t, z0);                                    // axial position by then
  const float lim = dz > 0.0f ? g.bhi[1] + 1e-3f : g.blo[1] - 1e-3f;
  return dz > 0.0f ? z1 > lim : (dz < 0.0f && z1 < lim);
}
__device__ __forceinline__ bool misses_detector(const DevGeomHead &g, const float x[3], const float d[3]) {
  const float r0sq = fmaf(x[0], x[0], x[1] * x[1]);
  const bool inside = g.bore_r > 0.0f && r0sq < g.bore_r * g.bore_r;
  return inside && misses_axially(g, sqrt_fast(r0sq), x[2], sqrt_fast(fmaf(d[0], d[0], d[1] * d[1])), d[2]);
}

// ---------------------------------------------------------------- first panel of a photon inside the bore of a ring
// Repetition-mode rings: the front faces of the n panels lie on the edges of a regular polygon about the
// z axis (extended beyond the vertices when panels are wider than an edge, short of them when there are gaps), and every
// panel box lies outside the open polygon.  A ray that starts inside the inscribed circle crosses the polygon boundary
// exactly once; if that crossing lies on the front face of panel k, inside the edge, then panel k is the one the search
// of [R6] returns: no other box has a point the ray reaches earlier.  So: estimate k from the azimuth of the point where
// the ray leaves the inscribed circle, take the slab test of [R6] on that one panel (the same arithmetic as the search),
// accept when the ray enters through the front face inside the edge (1 um clear of the vertices, where two overlapping
// panels tie: those rays go to the full search and its lowest-index rule), otherwise step to the neighbour the crossing
// point indicates and try once more.  Anything else -- gaps between panels, entries through side or end faces, rays that
// leave through the axial ends -- is left to the full search (the caller queues the photon for a SEARCH pass).
// Called by all 32 lanes (`active` = this lane has a photon to place): the early exit is a full-warp vote.
// `hint_turns` >= 0 (the same choice in every lane): the ray's azimuth in turns is already known -- a source on the axis
// draws it [R14] -- and replaces the circle crossing as the estimate.
__device__ __forceinline__ bool ring_entry_fast(const DevGeomHead &g, const DevPanel *pan, const float x[3], const float d[3], bool active, float hint_turns, int &bp, float &bt) {
  int k;
  if (hint_turns >= 0.0f) {
    float kf = hint_turns - g.ring_phi0 * 0.15915494f; kf -= floorf(kf);
    k = __float2int_rn(kf * (float)g.n_panels); k = k >= g.n_panels ? 0 : k;
  } else {
    const float dxy2 = fmaf(d[0], d[0], d[1] * d[1]);
    const float b = fmaf(x[0], d[0], x[1] * d[1]);
    const float cc = fmaf(g.bore_r, g.bore_r, -fmaf(x[0], x[0], x[1] * x[1]));               // > 0: the photon is inside the bore
    const float tc = (sqrt_fast(fmaf(dxy2, cc, b * b)) - b) * rcp_fast(dxy2 + 1e-30f);     // leaves the inscribed circle here
    const float phi = atan2_coarse(fmaf(tc, d[1], x[1]), fmaf(tc, d[0], x[0]));
    k = __float2int_rn((phi - g.ring_phi0) * g.ring_kscale);
    k += k < 0 ? g.n_panels : 0; k -= k >= g.n_panels ? g.n_panels : 0;
  }
  const float iz = rcp_dir(d[2]);
  const float z1 = (g.blo[1] - x[2]) * iz, z2 = (g.bhi[1] - x[2]) * iz;
  const float tnz = fmaxf(fminf(z1, z2), 0.0f), tfz = fmaxf(z1, z2);
  bool done = !active, ok = false;
#pragma unroll 1
  for (int it = 0; it < 2; ++it) {
    const float *P = pan[k].pose;
    const float r0 = x[0] - P[0], r1 = x[1] - P[1];
    const float a = r0 * P[3] + r1 * P[4], c = r0 * P[9] + r1 * P[10];
    const float da = d[0] * P[3] + d[1] * P[4], dc = d[0] * P[9] + d[1] * P[10];
    const float ia = rcp_dir(da), ic = rcp_dir(dc);
    const float a1 = (g.blo[0] - a) * ia, a2 = (g.bhi[0] - a) * ia, c1 = (g.blo[2] - c) * ic, c2 = (g.bhi[2] - c) * ic;
    const float an = fminf(a1, a2), cn = fminf(c1, c2);
    const float tn = fmaxf(tnz, fmaxf(an, cn)), tf = fminf(tfz, fminf(fmaxf(a1, a2), fmaxf(c1, c2)));
    const float af = fmaf(c1, da, a);                                  // tangential coordinate where the ray meets the front plane
    const bool heading = dc > 0.0f && c < 0.0f;                        // towards the front face, from in front of it
    const bool within = fabsf(af) <= g.ring_edge_h;
    const bool front = tf > tn && cn >= tnz && cn >= an && c1 <= c2;   // enters, and through the front face
    if (!done) {
      if (heading && within) { done = true; ok = front; bp = k; bt = tn; }
      else if (!heading) done = true;                                  // the estimate is off by more than a neighbour: full search
      else { k += af > 0.0f ? 1 : -1; k += k < 0 ? g.n_panels : 0; k -= k >= g.n_panels ? g.n_panels : 0; }
    }
    if (__all_sync(0xFFFFFFFFu, done)) break;
  }
  return ok;
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
// Specialisations keep the kernel small (it is sensitive to instruction-cache misses: dropping the phantom code alone
// made the ring configs 10 % faster).  PHANTOM: the source is a voxel map with a phantom [R17]; KIND: source kind
// (0 point, 1 voxel map, -1 = read src.kind); PLANAR: panel search variant (-1 = read g.planar); PRETEST: fresh photons
// take the acceptance pre-test (misses_detector) before they get a slot -- with KIND = 0 as a stage of its own (GEN1);
// FAST: repetition-mode ring, photons inside the bore find their first panel by ring_entry_fast; MULTI: the layers form
// several majorant regions [R19] (mixed-material stacks).
template <bool HASH, bool PHANTOM, int KIND, int PLANAR, bool PRETEST, bool FAST, bool MULTI>
__global__ void __launch_bounds__(kThreads, 1)
transport_wavefront_kernel(const __grid_constant__ DevGeomHead g, const DevPanel *panels, DevTables T, DevSource src, uint64_t first_history, uint64_t n_pairs,
                           const __grid_constant__ PhiloxKeys key, HitBuf H, uint64_t *hash_out, unsigned long long *work_counter, uint32_t grab_pairs) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n_mu = T.n_staged * T.n_energies;
  constexpr bool QUEUE = KIND == 0 && !PHANTOM;                               // the two-stage point source
  float4 *mu_s = reinterpret_cast<float4 *>(smem_raw + SmemLayout<HASH, QUEUE>::mu_off(blockDim.x >> 5));
  DevLayer *lay = reinterpret_cast<DevLayer *>(smem_raw + SmemLayout<HASH, QUEUE>::layer_off(blockDim.x >> 5, n_mu));
  DevPanel *pan = reinterpret_cast<DevPanel *>(smem_raw + SmemLayout<HASH, QUEUE>::geom_off(blockDim.x >> 5, n_mu));
  const int lane = threadIdx.x & 31;
  WarpMem<HASH, QUEUE> &W = reinterpret_cast<WarpMem<HASH, QUEUE> *>(smem_raw)[threadIdx.x >> 5];
  constexpr int kSlots = kSlotsOf<HASH>;
  {
    const uint32_t *gs = reinterpret_cast<const uint32_t *>(panels);
    uint32_t *gd = reinterpret_cast<uint32_t *>(pan);
    const int words = (int)(sizeof(DevPanel) / 4) * g.n_panels;
    for (int i = threadIdx.x; i < words; i += blockDim.x) gd[i] = gs[i];
    // record n_panels: the identity pose (a photon that has no panel yet is "in the frame" of this one: global = local)
    for (int i = threadIdx.x; i < (int)(sizeof(DevPanel) / 4); i += blockDim.x)
      gd[words + i] = (i == 3 || i == 7 || i == 11) ? 0x3F800000u : 0u;
    for (int i = threadIdx.x; i < (int)(sizeof(DevLayer) / 4) * kMaxLayers; i += blockDim.x)
      reinterpret_cast<uint32_t *>(lay)[i] = reinterpret_cast<const uint32_t *>(&g.layer[0])[i];
    for (int i = threadIdx.x; i < n_mu; i += blockDim.x) mu_s[i] = T.mu[i];
    for (int i = lane; i < kSlots; i += 32) W.list[L_FREE][i] = (uint8_t)i;
    __syncthreads();
  }
  const float4 *mu = mu_s;
  const unsigned lt_mask = (1u << lane) - 1u;
  const unsigned FULL = 0xFFFFFFFFu;
  const int kind = KIND < 0 ? src.kind : KIND;
  constexpr bool kPointSrc = KIND == 0 && !PHANTOM;                           // GEN1 (draw, filter) + GEN2 (one photon per lane)
  const float src_r0 = sqrt_fast(fmaf(src.pos[0], src.pos[0], src.pos[1] * src.pos[1]));   // distance of a point source from the axis
  // the fused first search needs every fresh photon inside the bore of the ring: point sources only (uniform test)
  const bool fused = FAST && KIND == 0 && !PHANTOM && g.ring_edge_h > 0.0f &&
                     fmaf(src.pos[0], src.pos[0], src.pos[1] * src.pos[1]) < g.bore_r * g.bore_r;

  uint32_t w_next = 0, w_end = 0;          // this warp's reserved pairs [w_next, w_end)
  bool exhausted = false;                  // the global counter ran past n_pairs
  int cF = kSlots, cS = 0, cT = 0, cK = 0, cR = 0, cP = 0, cH = 0, cQ = 0, cX = 0;   // list / queue fill levels (warp-uniform)
  // SPLIT (phantom runs in a ring): photons that have left the phantom take the polygon shortcut in the SEARCH pass; the
  // few it cannot place, and every photon that leaves a panel towards another, wait in L_SEARCHF for the search over all
  // panels -- so neither pass pays for the other's lanes
  constexpr bool SPLIT = FAST && PHANTOM;
  constexpr int L_FULL = SPLIT ? L_SEARCHF : L_SEARCH;
  int &cFull = SPLIT ? cX : cS;

  auto history_of = [&](uint32_t pair) -> uint64_t { return first_history + pair; };
  // [R4] every transport event consumes one whole Philox block of the photon's stream
  auto block_at = [&](uint32_t pair, uint32_t meta, uint32_t blk) -> uint4 {
    const uint64_t history = history_of(pair);
    return philox4x32_10(make_uint4((uint32_t)history, (uint32_t)(history >> 32), 1u + (meta & 1u), blk), key);
  };
  // push the slot index of every lane with `pred` onto list L (ballot + prefix popcount)
  auto push = [&](int L, int &cnt, bool pred, int idx) {
    const unsigned m = __ballot_sync(FULL, pred);
    if (pred) W.list[L][cnt + __popc(m & lt_mask)] = (uint8_t)idx;
    cnt += __popc(m);
  };
  auto end_hash = [&](uint32_t pair, uint32_t meta, uint64_t h) { hash_out[2ull * pair + (meta & 1u)] = h; };
  auto grab = [&]() {                      // reserve the next pairs of the batch (one atomic per grab)
    if (w_next >= w_end && !exhausted) {
      unsigned long long b = 0;
      if (lane == 0) b = atomicAdd(work_counter, (unsigned long long)grab_pairs);
      b = __shfl_sync(FULL, b, 0);
      if (b >= n_pairs) { exhausted = true; w_next = w_end = 0; }
      else { w_next = (uint32_t)b; w_end = (uint32_t)min((uint64_t)(b + grab_pairs), n_pairs); }
    }
  };
  // fresh photon -> entry point of its first panel (fused search) or the SEARCH / PHANTOM list
  // returns the destination list; q is updated to the panel frame on success
  // 1 / majorant at 511 keV: every fresh photon enters its first panel with it (one region)
  const float inv_mu_511 = MULTI ? 0.0f : inv_majorant<MULTI>(mu, T, g, 0, 511.0f);
  const float inv_mu_ph511 = PHANTOM ? rcp_fast(mu_lookup(mu, T, src.ph_major, 511.0f).z) : 0.0f;   // ... and its first phantom step
  auto enter_panel = [&](Photon &q, uint64_t &hq, int bp, float bt, bool fresh) {
    if (HASH) hash_ev(hq, EV_ENTER, (uint32_t)bp);
    float xl[3], dl[3];
    to_local(pan[bp].pose, q.x, q.d, xl, dl);
#pragma unroll
    for (int k = 0; k < 3; ++k) { q.x[k] = fmaf(bt, dl[k], xl[k]); q.d[k] = dl[k]; }   // [R18]
    q.path += bt; q.meta = ph_with_panel(q.meta, bp);
    if (MULTI) {
      const int reg = (q.x[2] >= g.reg_lo[1] ? 1 : 0) + (q.x[2] >= g.reg_lo[2] ? 1 : 0) + (q.x[2] >= g.reg_lo[3] ? 1 : 0);   // [R19] by the entry depth (unused: +inf)
      q.meta = (q.meta & ~(3u << kRegShift)) | ((uint32_t)reg << kRegShift);
      q.inv_mu = inv_majorant<MULTI>(mu, T, g, reg, q.E);
    } else q.inv_mu = fresh ? inv_mu_511 : inv_majorant<MULTI>(mu, T, g, 0, q.E);   // one region: the bits stay 0
  };

#ifdef GPET_STATS
  unsigned st_pass[10] = {0,0,0,0,0,0,0,0,0,0}, st_lane[10] = {0,0,0,0,0,0,0,0,0,0};
#define GPET_STAT(i, n) do { st_pass[i]++; st_lane[i] += (unsigned)(n); } while (0)
#else
#define GPET_STAT(i, n) do { } while (0)
#endif
  int gen_b = 0, gen_nb = 0;               // point sources: photons A of the top gen_nb queued pairs are placed, their photons B come next

#pragma unroll 1
  for (;;) {
    // ================================================ scheduler: a list that fills a pass runs (cheap cascade, STEP first);
    // when none does, the source refills the pool; when it cannot, the fullest list runs short
    int phase = L_NONE, gen = 0;                                          // gen 1: GEN1 (draw + filter), 2: GEN2 / GEN
    if (cT >= 32) phase = L_STEP;
    else if (cH >= 32 || cF < kReserve) phase = L_HIT;                    // cF + cH >= kReserve always: a low free list means deposits wait
    else if (cK >= 32) phase = L_KN;
    else if (cS >= 32) phase = L_SEARCH;
    else if (SPLIT && cX >= 32) phase = L_SEARCHF;
    else if (PHANTOM && cP >= 32) phase = L_PHANTOM;
    else if (cR >= 32) phase = L_RAY;
    else {
      const bool more_src = !exhausted || w_next < w_end;
      const int room = cF - kReserve;                                     // photons that fit
      if (kPointSrc) {
        const int want = gen_b ? gen_nb : min(32, cQ);
        if (want > 0 && (gen_b || cQ >= 32 || !more_src) && room >= want) gen = 2;
        else if (!gen_b && more_src && cQ < 32) gen = 1;
      } else if (more_src && (room >> 1) >= kMinGen) gen = 2;
      if (!gen) {
        int best = 0;
        if (cT > 0) { phase = L_STEP; best = cT; }
        if (cK > best) { phase = L_KN; best = cK; }
        if (cS > best) { phase = L_SEARCH; best = cS; }
        if (SPLIT && cX > best) { phase = L_SEARCHF; best = cX; }
        if (PHANTOM && cP > best) { phase = L_PHANTOM; best = cP; }
        if (cR > best) { phase = L_RAY; best = cR; }
        if (best == 0) {
          if (cH > 0) phase = L_HIT;
          else if (!kPointSrc && more_src) gen = 2;                       // nothing in flight: take what fits
          else break;                                                     // (point sources: room >= 32 holds when nothing is in flight)
        }
      }
    }

    if (gen == 1) {
      // ---------------------------------------------- GEN1 (point source): the pair's source block [R3].  With PRETEST, cos(theta)
      // decides whether BOTH photons leave through the axial ends (misses_axially for photon A, and for photon B with any
      // acolinearity deviation it can draw [R15]); both tests are monotonic in u, so the host turns them into two integer
      // bounds on the 23 bits of u (pretest_bounds, with extra margin: a pair kept here is tested again, exactly, in
      // GEN2).  Pairs outside the bounds end here (two ESCAPEs); the others are queued for GEN2.
      grab();
      const int ng = (int)min(32u, w_end - w_next);
      const uint32_t j = w_next + (uint32_t)lane;
      w_next += (uint32_t)ng;
      GPET_STAT(7, ng);
      bool keep = false; uint4 w = make_uint4(0, 0, 0, 0);
      if (lane < ng) {
        const uint64_t history = history_of(j);
        w = philox4x32_10(make_uint4((uint32_t)history, (uint32_t)(history >> 32), 0u, 1u), key);
        keep = true;
        if (PRETEST) {
          const uint32_t kq = w.x >> 9;                                // [R2] the 23 bits of u: cos(theta) = 1 - 2u is monotonic in them
          keep = kq >= src.pre_klo && kq <= src.pre_khi;
          if (HASH && !keep) { uint64_t he = kHash0; hash_ev(he, EV_ESCAPE, 0); hash_out[2ull * j] = he; hash_out[2ull * j + 1] = he; }
        }
      }
      const unsigned mk = __ballot_sync(FULL, keep);
      if (keep) { const int o = cQ + __popc(mk & lt_mask); W.qw[o] = w; W.qp[o] = j; }
      cQ += __popc(mk);
      __syncwarp();
      continue;
    }
    if (gen == 2 && kPointSrc) {
      // ---------------------------------------------- GEN2 (point source): one photon per lane, in two half-passes over the same
      // queued pairs -- photons A, then photons B (opposite direction plus acolinearity [R15]) -- so that a pass needs
      // 32 free slots, not 64, and runs at full width.  A photon that may reach the detector gets a slot: at its entry
      // point in the STEP list when the fused search succeeds, else in the SEARCH list.
      const int nb = gen_b ? gen_nb : min(32, cQ);
      const bool have = lane < nb;
      GPET_STAT(8, nb);
      Photon q = {};
      q.meta = (kNoPanel << 5) | (uint32_t)gen_b; q.ids = kNone; q.E = 511.0f; q.path = 0.0f; q.inv_mu = 0.0f;
      q.x[0] = src.pos[0]; q.x[1] = src.pos[1]; q.x[2] = src.pos[2];
      q.d[0] = 1.0f; q.d[1] = 0.0f; q.d[2] = 0.0f;
      float sxy = 1.0f, hint = 0.0f;                                   // |d_xy|; azimuth in turns (exact for a source on the axis)
      if (have) {
        const uint4 w = W.qw[cQ - 1 - lane]; q.pair = W.qp[cQ - 1 - lane];
        hint = u01(w.y) + (gen_b ? 0.5f : 0.0f);
        const float u = u01(w.x), ct = 1.0f - 2.0f * u;
        if (!gen_b) {
          const float sth = 2.0f * sqrtf(u * (1.0f - u));             // sin^2 = (1-ct)(1+ct)
          float sp, cp; sincospif(2.0f * u01(w.y), &sp, &cp);
          q.d[0] = sth * cp; q.d[1] = sth * sp; q.d[2] = ct; sxy = sth;
          W.qd[cQ - 1 - lane] = make_float2(q.d[0], q.d[1]);
        } else {
          const float2 dA = W.qd[cQ - 1 - lane];                      // photon A's direction, as its half-pass computed it
          q.d[0] = -dA.x; q.d[1] = -dA.y; q.d[2] = -ct; sxy = sqrt_fast(fmaf(dA.x, dA.x, dA.y * dA.y));
          if (src.acol_sigma > 0.0f) {
            const float rho = src.acol_sigma * sqrt_fast(-2.0f * __logf(u01(w.z)));
            float sr, cr; sincos_small(rho, sr, cr);
            float sa, ca; sincos_2pi(u01(w.w), sa, ca);               // azimuth of a ~4e-3 rad deviation: 2^-21 is ample
            rotate(q.d, cr, sr, ca, sa);
            sxy = sqrt_fast(fmaf(q.d[0], q.d[0], q.d[1] * q.d[1]));
          }
        }
      }
      bool alive = have;
      uint64_t hq = kHash0;
      if (PRETEST) {
        alive = have && !misses_axially(g, src_r0, src.pos[2], sxy, q.d[2]);
        if (HASH && have && !alive) { uint64_t he = kHash0; hash_ev(he, EV_ESCAPE, 0); end_hash(q.pair, q.meta, he); }
      }
      int bp = 0; float bt = 0.0f; bool entered = false;
      if (FAST && fused) {
        entered = ring_entry_fast(g, pan, q.x, q.d, alive, src_r0 == 0.0f ? hint : -1.0f, bp, bt);
        if (entered) enter_panel(q, hq, bp, bt, true);
      }
      const unsigned ma = __ballot_sync(FULL, alive);
      const int idx = alive ? W.list[L_FREE][cF - 1 - __popc(ma & lt_mask)] : 0;
      cF -= __popc(ma);
      if (alive) slot_store(W, idx, q, hq);
      push(L_STEP, cT, alive && entered, idx);
      push(L_SEARCH, cS, alive && !entered, idx);
      if (gen_b) { cQ -= nb; gen_b = 0; } else { gen_b = 1; gen_nb = nb; }
      __syncwarp();
      continue;
    }
    if (gen == 2) {
      // ---------------------------------------------- GEN (voxel / beam sources): one annihilation pair per lane (S3) [R13-R16].
      // Each photon that may reach the detector gets a slot in the SEARCH list (or, born inside a phantom, in the
      // PHANTOM list for its first phantom step [R17]).
      const int room = max((cF - kReserve) >> 1, (cT | cK | cS | cP | cR | cH) == 0 ? 1 : 0);
      grab();
      const int ng = (int)min((uint32_t)min(32, room), w_end - w_next);
      const uint32_t j = w_next + (uint32_t)lane;
      w_next += (uint32_t)ng;
      const bool have = lane < ng;
      Photon q = {};
      q.pair = j; q.meta = kNoPanel << 5; q.ids = kNone; q.E = 511.0f; q.path = 0.0f; q.inv_mu = 0.0f;
      q.x[0] = src.pos[0]; q.x[1] = src.pos[1]; q.x[2] = src.pos[2];
      q.d[0] = 1.0f; q.d[1] = 0.0f; q.d[2] = 0.0f;
      uint4 w = make_uint4(0, 0, 0, 0);
      if (have) {
        const uint64_t history = history_of(j);
        const uint32_t h_lo = (uint32_t)history, h_hi = (uint32_t)(history >> 32);
        if (kind == 1) decay_site(src, philox4x32_10(make_uint4(h_lo, h_hi, 0u, 0u), key), q.x);
        if (src.positron_sigma > 0.0f) {                             // [R35] positron range: words 12-15 of the source stream
          const uint4 w3 = philox4x32_10(make_uint4(h_lo, h_hi, 0u, 3u), key);
          const float r1 = src.positron_sigma * sqrtf(-2.0f * logf(u01(w3.x))), r2 = src.positron_sigma * sqrtf(-2.0f * logf(u01(w3.z)));
          float s1, c1, s2, c2; sincospif(2.0f * u01(w3.y), &s1, &c1); sincospif(2.0f * u01(w3.w), &s2, &c2);
          q.x[0] = fmaf(r1, c1, q.x[0]); q.x[1] = fmaf(r1, s1, q.x[1]); q.x[2] = fmaf(r2, c2, q.x[2]);
        }
        w = philox4x32_10(make_uint4(h_lo, h_hi, 0u, 1u), key);
        if (kind == 2) { q.d[0] = src.beam[0]; q.d[1] = src.beam[1]; q.d[2] = src.beam[2]; }
        else {
          const float u = u01(w.x), ct = 1.0f - 2.0f * u, sth = 2.0f * sqrtf(u * (1.0f - u));   // sin^2 = (1-ct)(1+ct)
          float sp, cp; sincospif(2.0f * u01(w.y), &sp, &cp);
          q.d[0] = sth * cp; q.d[1] = sth * sp; q.d[2] = ct;
        }
        if (PHANTOM) { q.meta |= 1u << 11; q.inv_mu = inv_mu_ph511; }
      }
#pragma unroll 1
      for (int ph = 0; ph < 2; ++ph) {
        if (ph == 1 && have) {                                        // photon B: opposite, plus acolinearity [R15]
          q.d[0] = -q.d[0]; q.d[1] = -q.d[1]; q.d[2] = -q.d[2];
          if (src.acol_sigma > 0.0f) {
            const float rho = src.acol_sigma * sqrt_fast(-2.0f * __logf(u01(w.z)));
            float sr, cr; sincos_small(rho, sr, cr);
            float sp, cp; sincos_2pi(u01(w.w), sp, cp);               // azimuth of a ~4e-3 rad deviation: 2^-21 is ample
            rotate(q.d, cr, sr, cp, sp);
          }
          q.meta |= 1u;
        }
        bool alive = have;
        if (PRETEST && !PHANTOM) {
          alive = have && !misses_detector(g, q.x, q.d);
          if (HASH && have && !alive) { uint64_t he = kHash0; hash_ev(he, EV_ESCAPE, 0); end_hash(q.pair, q.meta, he); }
        }
        const unsigned ma = __ballot_sync(FULL, alive);
        const int idx = alive ? W.list[L_FREE][cF - 1 - __popc(ma & lt_mask)] : 0;
        cF -= __popc(ma);
        if (alive) slot_store(W, idx, q, kHash0);
        if (PHANTOM) push(L_PHANTOM, cP, alive, idx);
        else push(L_SEARCH, cS, alive, idx);
      }
      __syncwarp();
      continue;
    }

    if (SPLIT && phase == L_SEARCH) {
      // ---------------------------------------------- SEARCH, shortcut only (phantom runs in a ring): photons that have just left
      // the phantom are in the global frame, inside the bore; the polygon edge they cross names their panel
      const int n = min(cS, 32); const bool act = lane < n;
      Photon q = {}; uint64_t hq = 0; int idx = 0;
      if (act) { idx = W.list[L_SEARCH][cS - 1 - lane]; slot_load(W, idx, q, hq); }
      cS -= n;
      int bp = -1; float bt = 0.0f;
      const bool found = ring_entry_fast(g, pan, q.x, q.d, act && fmaf(q.x[0], q.x[0], q.x[1] * q.x[1]) < g.bore_r * g.bore_r, -1.0f, bp, bt);
      if (found) { enter_panel(q, hq, bp, bt, false); slot_store(W, idx, q, hq); }
      push(L_STEP, cT, found, idx);
      push(L_SEARCHF, cX, act && !found, idx);                         // unchanged, to the search over all panels
    } else if (phase == L_FULL) {
      // ---------------------------------------------- SEARCH: nearest panel ahead [R6], entry transform [R18].  A photon that has
      // just left a panel arrives in that panel's frame (record n_panels is the identity: fresh photons are global)
      const int n = min(cFull, 32); const bool act = lane < n;
      GPET_STAT(L_SEARCH, n);
      Photon q = {}; uint64_t hq = 0; int idx = 0;
      if (act) { idx = W.list[L_FULL][cFull - 1 - lane]; slot_load(W, idx, q, hq); }
      cFull -= n;
      int dest = L_NONE;
      const int excl = ph_panel(q.meta);
      if (act) {
        const float *P = pan[excl == (int)kNoPanel ? g.n_panels : excl].pose;
        const float xl[3] = { q.x[0], q.x[1], q.x[2] }, dl[3] = { q.d[0], q.d[1], q.d[2] };
        point_to_global(P, xl, q.x); dir_to_global(P, dl, q.d);
      }
      int bp = -1; float bt = 0.0f; bool found = false;
      if (FAST && PHANTOM && !SPLIT && g.ring_edge_h > 0.0f)          // (kept for builds that search in one pass)
        found = ring_entry_fast(g, pan, q.x, q.d, act && excl == (int)kNoPanel && fmaf(q.x[0], q.x[0], q.x[1] * q.x[1]) < g.bore_r * g.bore_r, -1.0f, bp, bt);
      if (act) {
        if (!found) bp = panel_search<PLANAR>(g, pan, q.x, q.d, excl, bt);
        if (bp < 0) {
          if (HASH) { hash_ev(hq, EV_ESCAPE, 0); end_hash(q.pair, q.meta, hq); }
          dest = L_FREE;
        } else {
          enter_panel(q, hq, bp, bt, false);
          dest = L_STEP;
          slot_store(W, idx, q, hq);
        }
      }
      push(L_FREE, cF, dest == L_FREE, idx);
      push(L_STEP, cT, dest == L_STEP, idx);
    } else if (phase == L_STEP) {
      // ---------------------------------------------- STEP: Woodcock step, layer selection, lattice lookup [R19], outcome [R20].
      // No divergent branches: every lane draws, advances to the collision point or to the exit face, looks the point up
      // and selects its next event.
      const int n = min(cT, 32); const bool act = lane < n;
      GPET_STAT(L_STEP, n);
      const int idx = W.list[L_STEP][max(cT - 1 - lane, 0)];
      cT -= n;
      float4 A = W.a[idx]; const float4 B = W.b[idx]; uint4 C = W.c[idx];
      uint64_t h = 0;
      if (HASH) { const uint2 v = W.hh[idx]; h = ((uint64_t)v.y << 32) | v.x; }
      const uint4 w = block_at(C.x, C.y, C.y >> kBlkShift);                  // [R4] free path, outcome, Rayleigh polar + azimuth
      C.y += 1u << kBlkShift;
      const float s = -__logf(u01(w.x)) * __uint_as_float(C.w);
      const float te0 = ((B.x >= 0.0f ? g.bhi[0] : g.blo[0]) - A.x) * rcp_dir(B.x);   // distance to the box exit [R32]
      const float te1 = ((B.y >= 0.0f ? g.bhi[1] : g.blo[1]) - A.y) * rcp_dir(B.y);
      constexpr bool multi = MULTI;                                    // [R19] several majorant regions: the depth slab is the region's
      int reg = (C.y >> kRegShift) & 3u;
      const float chi = multi ? g.reg_hi[reg] : g.bhi[2], clo = multi ? g.reg_lo[reg] : g.blo[2];
      const float te2 = ((B.z >= 0.0f ? chi : clo) - A.z) * rcp_dir(B.z);
      const float tf = fminf(te0, fminf(te1, te2));
      const int panel = ph_panel(C.y);
      const bool leaves = s >= tf;                                     // reaches a face of the (region's) slab first [R33]
      // Exit face = the axis that limits tf.  If no other panel has a point beyond that face (precomputed per panel and
      // face at create time: true for the back and axial faces of any ring), the search of [R6] cannot find anything:
      // the photon escapes here, with the same EXIT, ESCAPE events, and needs no search.
      const int kx = te0 <= tf ? 0 : (te1 <= tf ? 1 : 2);
      const float dk = kx == 0 ? B.x : (kx == 1 ? B.y : B.z);
      const bool open = (pan[panel].open_faces >> (2 * kx + (dk >= 0.0f ? 1 : 0))) & 1u;
      // a depth face that is not a face of the panel box: the photon crosses into the next region and draws afresh there
      const bool cross = multi && leaves && kx == 2 && (B.z >= 0.0f ? reg + 1 < g.n_regions : reg > 0);
      const bool exits = leaves && !cross;
      const float step = leaves ? fmaxf(tf, 0.0f) : s;
      A.x = fmaf(step, B.x, A.x); A.y = fmaf(step, B.y, A.y); A.z = fmaf(step, B.z, A.z); A.w += step;
      uint32_t id;                                                     // depth -> layer -> crystal
      const int mat = lattice_lookup(g, lay, __float2int_rd(A.x * kQ) + g.hWq, __float2int_rd(A.y * kQ) + g.hHq, __float2int_rd(A.z * kQ), id);
      if (id != kNone) id |= (uint32_t)panel << 26;
      const bool matter = !leaves && mat >= 0;
      const float4 m4 = mu_lookup(mu, T, mat < 0 ? 0 : mat, B.w);
      const float t = u01(w.y) * (multi ? rcp_fast(__uint_as_float(C.w)) : m4.w);   // [R20] one draw picks the outcome: u x the majorant the step was drawn with
      const bool pe = matter && t < m4.x, kn = matter && !pe && t < m4.y, ray = matter && !pe && !kn && t < m4.z;
      int dest = L_STEP;
      if (ray) dest = L_RAY;                                           // deflected in its own pass
      if (kn) dest = L_KN;
      if (pe) dest = id != kNone ? L_HIT : L_FREE;                     // photoelectric: deposit E, end
      if (exits) dest = open ? L_FREE : L_FULL;
      if (multi && cross) {                                            // (uniform test first: single-region detectors never get here)
        reg += B.z >= 0.0f ? 1 : -1;
        C.y = (C.y & ~(3u << kRegShift)) | ((uint32_t)reg << kRegShift);
        C.w = __float_as_uint(inv_majorant<MULTI>(mu, T, g, reg, B.w));
      }
      if (!act) dest = L_NONE;
      if (HASH && act) {
        if (cross) hash_ev(h, EV_REGION, (uint32_t)reg);
        else if (exits) { hash_ev(h, EV_EXIT, (uint32_t)panel); if (open) hash_ev(h, EV_ESCAPE, 0); }
        else if (mat < 0) hash_ev(h, EV_STEP_VACUUM, 0);
        else if (pe) hash_ev(h, EV_PE, id);
        else if (kn) { }                                               // hashed when a trial is accepted
        else if (ray) hash_ev(h, EV_RAYLEIGH, id);
        else hash_ev(h, EV_VIRTUAL, id);
        if (dest == L_FREE || dest == L_HIT) end_hash(C.x, C.y, h);
      }
      if (matter) C.z = id;
      if (pe) C.w = __float_as_uint(B.w);                              // the HIT pass reads the deposit here
      if (dest != L_FREE && dest != L_NONE) {
        W.a[idx] = A; W.c[idx] = C;
        if (HASH) W.hh[idx] = make_uint2((uint32_t)h, (uint32_t)(h >> 32));
      }
      push(L_STEP, cT, dest == L_STEP, idx);
      push(L_KN, cK, dest == L_KN, idx);
      push(L_FREE, cF, dest == L_FREE, idx);
      push(L_HIT, cH, dest == L_HIT, idx);
      if (__any_sync(FULL, dest == L_FULL || dest == L_RAY)) {         // the rare destinations share one vote
        push(L_FULL, cFull, dest == L_FULL, idx);
        push(L_RAY, cR, dest == L_RAY, idx);
      }
    } else if (phase == L_KN) {
      // ---------------------------------------------- KN: one Klein-Nishina trial per visit [R20].  A deposit in a crystal is
      // copied into a free slot and queued for the HIT pass; the photon itself goes on.
      const int n = min(min(cK, 32), cF); const bool act = lane < n;
      GPET_STAT(L_KN, n);
      const int idx = W.list[L_KN][max(cK - 1 - lane, 0)];
      cK -= n;
      const float4 A = W.a[idx]; float4 B = W.b[idx]; uint4 C = W.c[idx];
      uint64_t h = 0;
      if (HASH) { const uint2 v = W.hh[idx]; h = ((uint64_t)v.y << 32) | v.x; }
      const bool in_ph = PHANTOM && ((C.y >> 11) & 1u);
      const float E = B.w;
      const float k = E * (1.0f / kMec2), e0 = rcp_fast(1.0f + 2.0f * k), e02 = e0 * e0;
      const float a1 = -__logf(e0), a2 = 0.5f * (1.0f - e02);
      const uint4 w = block_at(C.x, C.y, C.y >> kBlkShift);                  // [R4] u_a, u_b, u_c, azimuth
      C.y += 1u << kBlkShift;
      const float ua = u01(w.x), ub = u01(w.y), uc = u01(w.z);
      // om = 1 - eps and em = eps - eps0 are formed without cancellation, so that sin^2 = t (2 - t) keeps
      // full relative accuracy at both poles (t = om/(k eps), 2 - t = em/(eps0 k eps)); plain fp32 loses
      // 3-4 digits of small scattering angles and moves later hits by micrometres
      const bool lowhalf = ub < 0.5f;
      const float v = expm1_small(lowhalf ? -a1 * ub : a1 * (1.0f - ub));
      const float om_x = lowhalf ? -v : 1.0f - fmaf(e0, v, e0);       // eps = exp(-a1 ub)
      const float em_x = lowhalf ? (1.0f + v) - e0 : e0 * v;
      const float eps_x = lowhalf ? 1.0f + v : fmaf(e0, v, e0);
      const float eps_s = sqrt_fast(fmaf(1.0f - e02, ub, e02));       // eps = sqrt(eps0^2 + (1 - eps0^2) ub)
      const float om_s = (1.0f - e02) * (1.0f - ub) * rcp_fast(1.0f + eps_s), em_s = (1.0f - e02) * ub * rcp_fast(eps_s + e0);
      const bool expo = ua * (a1 + a2) < a1;
      const float eps = expo ? eps_x : eps_s, om = expo ? om_x : om_s, em = expo ? em_x : em_s;
      const float ike = rcp_fast(k * eps);
      const float t = om * ike, tm = em * ike * (1.0f + 2.0f * k);
      const float gr = 1.0f - eps * t * tm * rcp_fast(1.0f + eps * eps);
      const bool accept = gr >= uc || ((C.y >> 12) & 63u) >= 63u;     // [R22: the 64th trial always is]
      float sp, cp; sincos_2pi(u01(w.w), sp, cp);
      float dn[3] = { B.x, B.y, B.z };
      rotate(dn, 1.0f - t, sqrt_fast(fmaxf(t * tm, 0.0f)), cp, sp);
      const float dep = om * E, E2 = E - dep;
      const bool cut = E2 < kCutoff;                                   // [R12]
      const bool hit = act && accept && !in_ph && C.z != kNone;
      // the deposit: its own record {x, y, z, path}, {pair, meta, ids, energy}, in a fresh slot, for the HIT pass
      const unsigned mh = __ballot_sync(FULL, hit);
      if (mh) {
        const int rk = __popc(mh & lt_mask);
        if (hit) {
          const int i2 = W.list[L_FREE][cF - 1 - rk];
          W.a[i2] = A; W.c[i2] = make_uint4(C.x, C.y, C.z, __float_as_uint(cut ? E : dep));
          W.list[L_HIT][cH + rk] = (uint8_t)i2;
        }
        cF -= __popc(mh); cH += __popc(mh);
      }
      int dest = L_KN;
      if (accept) {
        if (HASH && act) {
          if (in_ph) { hash_ev(h, EV_PH_COMPTON, 0); if (cut) hash_ev(h, EV_PH_CUTOFF, 0); }
          else { hash_ev(h, EV_COMPTON, C.z); if (cut) hash_ev(h, EV_CUTOFF, C.z); }
          if (cut) end_hash(C.x, C.y, h);
        }
        C.y &= ~(63u << 12);
        if (hit && ((C.y >> 1) & 15u) < 15u) C.y += 2u;                // [R9] 4-bit saturating hit counter
        B.x = dn[0]; B.y = dn[1]; B.z = dn[2]; B.w = E2;
        const float e_new = cut ? E : E2;
        C.w = __float_as_uint(in_ph ? rcp_fast(mu_lookup(mu, T, src.ph_major, e_new).z) : inv_majorant<MULTI>(mu, T, g, (C.y >> kRegShift) & 3u, e_new));
        dest = cut ? L_FREE : (in_ph ? L_PHANTOM : L_STEP);
      } else C.y += 1u << 12;
      if (!act) dest = L_NONE;
      if (dest != L_FREE && dest != L_NONE) {
        W.b[idx] = B; W.c[idx] = C;
        if (HASH) W.hh[idx] = make_uint2((uint32_t)h, (uint32_t)(h >> 32));
      }
      push(L_KN, cK, dest == L_KN, idx);
      push(L_STEP, cT, dest == L_STEP, idx);
      push(L_FREE, cF, dest == L_FREE, idx);
      if (PHANTOM) push(L_PHANTOM, cP, dest == L_PHANTOM, idx);
    } else if (phase == L_HIT) {
      // ---------------------------------------------- HIT (S10): up to 32 deposits -> global frame [R22] -> the hit buffer.  Dense
      // layout: one atomicAdd on the global counter, seven coalesced stores.  Chunked layout: the hits go to the region
      // of their 512-pair chunk; lanes of the same chunk (almost always all of them) share one atomicAdd on that chunk's
      // fill counter and write consecutive entries.
      const int n = min(cH, 32); const bool act = lane < n;
      GPET_STAT(L_HIT, n);
      const int idx = W.list[L_HIT][max(cH - 1 - lane, 0)];
      cH -= n;
      const float4 A = W.a[idx]; const uint4 C = W.c[idx];
      const float xl[3] = { A.x, A.y, A.z }; float xg[3];
      point_to_global(pan[C.z >> 26].pose, xl, xg);
      const uint32_t hist = (uint32_t)history_of(C.x), ids = C.z | ((C.y & 1u) << 4) | ((C.y >> 1) & 15u);
      const float tof = A.w * kInvC;
      unsigned long long o = 0; bool ok = false;
      if (H.chunk_fill == nullptr) {
        unsigned long long base = 0;
        if (lane == 0) base = atomicAdd(H.n_hits, (unsigned long long)n);
        base = __shfl_sync(FULL, base, 0);
        o = base + lane; ok = act && o < H.capacity;
      } else {
        if (lane == 0) atomicAdd(H.n_hits, (unsigned long long)n);     // total produced (no return value needed)
        const uint32_t chunk = act ? C.x >> kHitChunkShift : 0xFFFFFFFFu;
        const unsigned grp = __match_any_sync(FULL, chunk);
        const int leader = __ffs(grp) - 1;
        uint32_t base = 0;
        if (act && lane == leader && chunk < H.n_chunks) base = atomicAdd(&H.chunk_fill[chunk], (uint32_t)__popc(grp));
        base = __shfl_sync(FULL, base, leader);
        if (act && chunk < H.n_chunks) {
          const uint32_t pos = base + __popc(grp & lt_mask);
          if (pos < H.chunk_cap) { ok = true; o = (unsigned long long)chunk * H.chunk_cap + pos; }
          else atomicAdd(&H.chunk_fill[H.n_chunks], 1u);               // dropped: this chunk's region is full
        }
      }
      if (ok) {
        H.history[o] = hist; H.ids[o] = ids; H.x[o] = xg[0]; H.y[o] = xg[1]; H.z[o] = xg[2];
        H.e[o] = __uint_as_float(C.w); H.tof[o] = tof;
      }
      push(L_FREE, cF, act, idx);
    } else if (phase == L_RAY) {
      // ---------------------------------------------- RAY: Rayleigh deflection with words 2-3 of the step's block [R4, R20]
      const int n = min(cR, 32); const bool act = lane < n;
      Photon p = {}; uint64_t h = 0; int idx = 0;
      if (act) { idx = W.list[L_RAY][cR - 1 - lane]; slot_load(W, idx, p, h); }
      cR -= n;
      int dest = L_NONE;
      if (act) {
        const uint4 w = block_at(p.pair, p.meta, (p.meta >> kBlkShift) - 1u);   // the block its Woodcock step drew (rare event: recomputed)
        const float3 r = rayleigh_dir(p.d[0], p.d[1], p.d[2], u01(w.z), u01(w.w));
        p.d[0] = r.x; p.d[1] = r.y; p.d[2] = r.z;
        dest = (PHANTOM && ((p.meta >> 11) & 1u)) ? L_PHANTOM : L_STEP;
        slot_store(W, idx, p, h);
      }
      push(L_STEP, cT, dest == L_STEP, idx);
      if (PHANTOM) push(L_PHANTOM, cP, dest == L_PHANTOM, idx);
    } else if (PHANTOM && phase == L_PHANTOM) {
      // ---------------------------------------------- PHANTOM: Woodcock tracking in the voxel grid [R17].  No divergent branches:
      // every lane draws, advances to the tentative point, reads its voxel (clamped when the point lies outside the grid),
      // interpolates mu and selects its next event.
      const int n = min(cP, 32); const bool act = lane < n;
      const int idx = W.list[L_PHANTOM][max(cP - 1 - lane, 0)];
      cP -= n;
      float4 A = W.a[idx]; const float4 B = W.b[idx]; uint4 C = W.c[idx];
      uint64_t h = 0;
      if (HASH) { const uint2 v = W.hh[idx]; h = ((uint64_t)v.y << 32) | v.x; }
      const uint4 w = block_at(C.x, C.y, C.y >> kBlkShift);                  // [R4] free path, outcome
      C.y += 1u << kBlkShift;
      const float s = -__logf(u01(w.x)) * __uint_as_float(C.w);
      const float x0[3] = { A.x, A.y, A.z }, d0[3] = { B.x, B.y, B.z };
      const float xt0 = fmaf(s, B.x, A.x), xt1 = fmaf(s, B.y, A.y), xt2 = fmaf(s, B.z, A.z);
      const int v0 = __float2int_rd((xt0 - src.origin[0]) * src.inv_voxel[0]), v1 = __float2int_rd((xt1 - src.origin[1]) * src.inv_voxel[1]),
                v2 = __float2int_rd((xt2 - src.origin[2]) * src.inv_voxel[2]);
      // tentative point outside the grid: the photon leaves along its line of flight from where it is [R17]
      const bool out = (unsigned)v0 >= (unsigned)src.dims[0] || (unsigned)v1 >= (unsigned)src.dims[1] || (unsigned)v2 >= (unsigned)src.dims[2];
      const bool gone = out && misses_detector(g, x0, d0);            // cannot reach the detector: ESCAPE without a search
      const int c0 = min(max(v0, 0), src.dims[0] - 1), c1 = min(max(v1, 0), src.dims[1] - 1), c2 = min(max(v2, 0), src.dims[2] - 1);
      const int mat = out ? -1 : (int)src.phantom[((size_t)c2 * src.dims[1] + c1) * src.dims[0] + c0] - 1;
      const float4 m4 = mu_lookup(mu, T, mat < 0 ? 0 : mat, B.w);
      const float t = u01(w.y) * mu_lookup(mu, T, src.ph_major, B.w).z;
      const bool matter = mat >= 0;
      const bool pe = matter && t < m4.x, kn = matter && !pe && t < m4.y, ray = matter && !pe && !kn && t < m4.z;
      int dest = L_PHANTOM;
      if (ray) dest = L_RAY;
      if (kn) dest = L_KN;
      if (pe) dest = L_FREE;
      if (out) dest = gone ? L_FREE : L_SEARCH;
      if (!act) dest = L_NONE;
      if (HASH && act) {
        if (out) { hash_ev(h, EV_PH_LEAVE, 0); if (gone) hash_ev(h, EV_ESCAPE, 0); }
        else if (pe) hash_ev(h, EV_PH_ABSORBED, 0);
        else if (ray) hash_ev(h, EV_PH_RAYLEIGH, 0);
        if (dest == L_FREE) end_hash(C.x, C.y, h);
      }
      if (out) C.y &= ~(1u << 11);
      else { A.x = xt0; A.y = xt1; A.z = xt2; A.w += s; }
      if (kn) C.z = kNone;
      if (dest != L_FREE && dest != L_NONE) {
        W.a[idx] = A; W.c[idx] = C;
        if (HASH) W.hh[idx] = make_uint2((uint32_t)h, (uint32_t)(h >> 32));
      }
      push(L_PHANTOM, cP, dest == L_PHANTOM, idx);
      push(L_SEARCH, cS, dest == L_SEARCH, idx);
      push(L_FREE, cF, dest == L_FREE, idx);
      if (__any_sync(FULL, dest == L_KN || dest == L_RAY)) {           // scatters in the phantom are the rare destinations
        push(L_KN, cK, dest == L_KN, idx);
        push(L_RAY, cR, dest == L_RAY, idx);
      }
    }
    __syncwarp();
  }
#ifdef GPET_STATS
  if (blockIdx.x == 3 && lane == 0 && (threadIdx.x >> 5) < 4)
    printf("warp %d: SEARCH %u/%u STEP %u/%u KN %u/%u HIT %u/%u GEN1 %u/%u GEN2 %u/%u\n", threadIdx.x >> 5, st_lane[L_SEARCH], st_pass[L_SEARCH], st_lane[L_STEP], st_pass[L_STEP],
           st_lane[L_KN], st_pass[L_KN], st_lane[L_HIT], st_pass[L_HIT], st_lane[7], st_pass[7], st_lane[8], st_pass[8]);
#endif
}

static int g_transport_warps = kWarps;             // warps per CTA (one CTA per SM); fewer leave room for other streams' kernels
void set_transport_warps(int warps) { g_transport_warps = warps < 1 ? kWarps : (warps > kWarps ? kWarps : warps); }
int transport_warps() { return g_transport_warps; }

// which build a run takes (see the dispatch in launch_transport): point source in a repetition-mode ring -> two-stage source
static bool is_phantom_run(const DevSource &src) { return src.kind == 1 && src.phantom != nullptr; }
static bool is_ring(const DevGeom &g) { return g.planar != 0 && g.ring != 0 && g.ring_edge_h > 0.0f; }
static bool uses_pair_queue(const DevGeom &g, const DevSource &src) {
  return !is_phantom_run(src) && src.kind == 0 && !(src.positron_sigma > 0.0f) && is_ring(g);
}
static size_t smem_for(const DevTables &T, int n_panels, bool hash, bool queue, int warps) {
  const int n_mu = T.n_staged * T.n_energies;
  const size_t pools = hash ? (queue ? SmemLayout<true, true>::geom_off(warps, n_mu) : SmemLayout<true, false>::geom_off(warps, n_mu))
                            : (queue ? SmemLayout<false, true>::geom_off(warps, n_mu) : SmemLayout<false, false>::geom_off(warps, n_mu));
  return pools + panel_bytes(n_panels + 1);
}

// The tables are staged in shared memory next to the per-warp pools: with many materials or a fine energy grid the CTA
// gives up warps until everything fits (0 = it cannot fit at all).
int transport_warps_that_fit(const DevGeom &host_geom, const DevTables &T, const DevSource &src, bool hash, size_t smem_limit) {
  int w = g_transport_warps;
  const int floor_w = w < 4 ? w : 4;                 // a caller who asked for 1..3 warps gets them; nobody is cut below 4 silently
  const bool queue = uses_pair_queue(host_geom, src);
  while (w > floor_w && smem_for(T, host_geom.n_panels, hash, queue, w) > smem_limit) --w;
  return smem_for(T, host_geom.n_panels, hash, queue, w) <= smem_limit ? w : 0;
}

// Point-source pre-test as two integer bounds on k = (polar word >> 9), u = (k + 0.5) 2^-23 [R2].  A pair may be dropped in
// GEN1 only when misses_axially holds for photon A (d_z = 1 - 2u) AND for photon B with any acolinearity deviation it can
// draw [R15] (polar deviation at most rho_max: |d_z| >= |ct| cos(rho) - sth sin(rho), |d_xy| <= sth cos(rho) + |ct| sin(rho)).
// Both tests are monotonic in u on each side of u = 1/2, so the dropped pairs are k < k_lo and k > k_hi.  The bounds come
// from the same inequality evaluated in fp64 with wider margins than the kernel's fp32 form (path to the bore radius
// x 0.999 instead of 0.9999, the axial limit 2 um further out instead of 1 um, |d_xy| bounds + 0.1 %) and are then moved 64
// counts (7.6e-6 in u) towards the ends: every pair dropped here fails the exact tests of GEN2 too, the few extra pairs kept
// are dropped there.
static void pretest_bounds(const DevGeomHead &g, const DevSource &src, uint32_t &k_lo, uint32_t &k_hi) {
  const double r0 = hypot((double)src.pos[0], (double)src.pos[1]), z0 = src.pos[2];
  const double sr = src.acol_sin_max, cr = src.acol_cos_max;
  auto misses = [&](double sxy, double dz) -> bool {
    const double t = ((double)g.bore_r - r0) / (sxy + 1e-30) * 0.999, z1 = z0 + dz * t;
    return dz > 0.0 ? z1 > (double)g.bhi[1] + 2e-3 : (dz < 0.0 && z1 < (double)g.blo[1] - 2e-3);
  };
  auto drop = [&](uint32_t k) -> bool {
    const double u = ((double)k + 0.5) * (1.0 / 8388608.0), ct = 1.0 - 2.0 * u, sth = 2.0 * sqrt(u * (1.0 - u));
    const double bz = fabs(ct) * cr - sth * sr, bxy = (sth * cr + fabs(ct) * sr) * 1.001;
    return misses(sth * 1.001, ct) && bz > 0.0 && misses(bxy, ct > 0.0 ? -bz : bz);
  };
  const uint32_t half = 1u << 22;                                     // k < half: photon A goes up (+z)
  uint32_t lo = 0, hi = half;                                         // first k in [0, half] that is not dropped
  while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (drop(mid)) lo = mid + 1; else hi = mid; }
  k_lo = lo > 64u ? lo - 64u : 0u;
  lo = half; hi = (1u << 23);                                         // first k in [half, 2^23] from which all are dropped
  while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (drop(mid)) hi = mid; else lo = mid + 1; }
  k_hi = lo + 63u < (1u << 23) ? lo + 63u : (1u << 23) - 1u;
}

cudaError_t launch_transport(const DevGeom &host_geom, const DevGeom *geom, const DevTables &T, const DevSource &src,
                             uint64_t first_history, uint64_t n_pairs, uint64_t seed, const HitBuf &H, uint64_t *hash_out,
                             unsigned long long *work_counter, int sm_count, int warps, cudaStream_t stream) {
  const int n_panels = host_geom.n_panels;
  const DevGeomHead &head = host_geom;
  const DevPanel *panels = reinterpret_cast<const DevPanel *>(reinterpret_cast<const char *>(geom) +
                                                            (reinterpret_cast<const char *>(&host_geom.panel[0]) - reinterpret_cast<const char *>(&host_geom)));
  const size_t smem = smem_for(T, n_panels, hash_out != nullptr, uses_pair_queue(host_geom, src), warps);
  const int threads = 32 * warps;
  const uint64_t want = (2 * n_pairs + threads - 1) / threads;
  const uint64_t resident = (uint64_t)sm_count;                      // persistent grid: one CTA per SM
  PhiloxKeys key;                                                     // [R1] round keys: key + r * Weyl constants
  for (int r = 0; r < 10; ++r) { key.k[2 * r] = (uint32_t)seed + (uint32_t)r * 0x9E3779B9u; key.k[2 * r + 1] = (uint32_t)(seed >> 32) + (uint32_t)r * 0xBB67AE85u; }
  const int blocks = (int)(want < resident ? (want ? want : 1) : resident);
  // pairs a warp reserves at a time: kGrab for long runs, less when every warp gets only a few grabs (short tails: a warp
  // that draws the last grab works alone for one grab's time), never less than one GEN1 pass
  uint32_t grab_pairs = (uint32_t)(n_pairs / ((uint64_t)blocks * warps * 8));
  grab_pairs = grab_pairs >= kGrab ? kGrab : (grab_pairs < 32u ? 32u : grab_pairs & ~31u);
  cudaError_t e = cudaMemsetAsync(work_counter, 0, sizeof(unsigned long long), stream);
  if (e != cudaSuccess) return e;
  const bool phantom = is_phantom_run(src);
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
  DevSource srcp = src;
  srcp.pre_klo = 0u; srcp.pre_khi = 0xFFFFFFFFu;
  if (pretest && src.kind == 0) pretest_bounds(head, src, srcp.pre_klo, srcp.pre_khi);
  auto launch = [&](auto kernel) -> cudaError_t {
    cudaError_t le = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (le != cudaSuccess) return le;
    kernel<<<blocks, threads, smem, stream>>>(head, panels, T, srcp, first_history, n_pairs, key, H, hash_out, work_counter, grab_pairs);
    return cudaSuccess;
  };
  // specialised builds for the shapes the five configs use (point source or voxel map + phantom, in a repetition-mode
  // ring); anything else runs the generic build of the same code
  const bool ring = is_ring(host_geom);
  const bool point = !phantom && src.kind == 0 && !(src.positron_sigma > 0.0f);   // every pair starts at src.pos
#define GPET_DISPATCH(H, M)                                                                                                 \
  do {                                                                                                                      \
    if (point && ring && pretest) e = launch(transport_wavefront_kernel<H, false, 0, 1, true, true, M>);                     \
    else if (point && ring) e = launch(transport_wavefront_kernel<H, false, 0, 1, false, true, M>);                         \
    else if (phantom && ring) e = launch(transport_wavefront_kernel<H, true, 1, 1, false, true, M>);                        \
    else if (phantom) e = launch(transport_wavefront_kernel<H, true, 1, -1, false, false, M>);                              \
    else if (pretest) e = launch(transport_wavefront_kernel<H, false, -1, -1, true, false, M>);                             \
    else e = launch(transport_wavefront_kernel<H, false, -1, -1, false, false, M>);                                         \
  } while (0)
  const bool multi = host_geom.n_regions > 1;
  if (hash_out) { if (multi) GPET_DISPATCH(true, true); else GPET_DISPATCH(true, false); }
  else { if (multi) GPET_DISPATCH(false, true); else GPET_DISPATCH(false, false); }
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
      lattice_lookup(g, g.layer, (int)qa, (int)qb, (int)qc, out);
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
