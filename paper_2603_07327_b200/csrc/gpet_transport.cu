// gpet_transport.cu -- photon transport (S2..S10 of DESIGN.md section 1) as ONE persistent wavefront kernel.
// PAPER.md:33 (panel transfer by ray/plane crossing, global->local), PAPER.md:43 (Woodcock tracking in the
// panel frame, layer selection from the local depth, run until exit or cutoff).
//
// Design:
//  * unit of work = one photon (index j = 2*pair + photon); every lane of a persistent warp owns one photon
//    and a small state machine {REFILL, SEARCH, STEP, COMPTON, RAYLEIGH, PHANTOM};
//  * each pass of the warp's main loop ballots the lanes' next events and runs the ONE phase that most
//    lanes are waiting for (wavefront regrouping in time): its code is fetched once for all of them, the
//    other lanes keep their state in registers and wait; every phase appears exactly once in the kernel,
//    which keeps the SASS small enough for the instruction caches (v1's 107 KB of inlined code stalled
//    59 % of the time on instruction fetch);
//  * photon indices are handed out from a global counter in chunks of 1024 per warp;
//  * geometry descriptor and interleaved float4 mu tables live in shared memory; hits are staged per warp
//    in shared memory and flushed 32 at a time: one atomicAdd per 32 hits and seven fully coalesced
//    128-byte stores (struct of arrays).
#include <cstdlib>
#include "gpet_internal.h"

namespace gpet {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kStage = 64;            // staged hits per warp (ring buffer)
constexpr uint32_t kChunk = 1024;     // photon indices a warp reserves at a time

enum : int { ST_REFILL = 0, ST_SEARCH = 1, ST_STEP = 2, ST_COMPTON = 3, ST_RAYLEIGH = 4, ST_PHANTOM = 5, ST_IDLE = 6 };

struct HitStage { uint32_t w[7][kStage]; };      // history, ids, x, y, z, e, tof

struct Smem {
  DevGeom g;
  HitStage stage[kWarps];
  float4 mu[1];                        // [n_materials][n_energies], .w = detector majorant
};

// ---------------------------------------------------------------- fast math with bounded error
__device__ __forceinline__ float rcp_fast(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float sqrt_fast(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
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
  const float4 a = mu[m * T.n_energies + i], b = mu[m * T.n_energies + i + 1];
  return make_float4(fmaf(f, b.x - a.x, a.x), fmaf(f, b.y - a.y, a.y), fmaf(f, b.z - a.z, a.z), fmaf(f, b.w - a.w, a.w));
}

// ---------------------------------------------------------------- per-lane photon state
struct Photon {
  float x[3], d[3];        // global frame in SEARCH / PHANTOM, panel frame in STEP / COMPTON / RAYLEIGH
  float E, path, inv_mu;   // inv_mu = 1 / majorant(E) of the medium the photon is tracked in
  uint32_t pair;           // history - first_history
  uint32_t meta;           // bit0 photon, bits1-4 seq, bits5-10 panel (current, or just left; 63 = none),
                           // bit11 in phantom, bits12+ Klein-Nishina trial counter
  uint32_t ids;            // lattice result of the pending interaction
  uint32_t ndraw; uint4 blk;
};
__device__ __forceinline__ int ph_panel(const Photon &p) { return (p.meta >> 5) & 63u; }
__device__ __forceinline__ void ph_set_panel(Photon &p, int panel) { p.meta = (p.meta & ~(63u << 5)) | ((uint32_t)panel << 5); }

// write one staged hit (slot of this warp's ring buffer) to the global struct-of-arrays buffer
__device__ __forceinline__ void store_hit(const HitBuf &H, unsigned long long o, const HitStage &stage, uint32_t slot) {
  if (o < H.capacity) {
    H.history[o] = stage.w[0][slot]; H.ids[o] = stage.w[1][slot];
    H.x[o] = __uint_as_float(stage.w[2][slot]); H.y[o] = __uint_as_float(stage.w[3][slot]); H.z[o] = __uint_as_float(stage.w[4][slot]);
    H.e[o] = __uint_as_float(stage.w[5][slot]); H.tof[o] = __uint_as_float(stage.w[6][slot]);
  }
}

// ---------------------------------------------------------------- the kernel
template <bool HASH>
__global__ void __launch_bounds__(kThreads, 4)
transport_wavefront_kernel(const DevGeom *geom, DevTables T, const float *maj, DevSource src, uint64_t first_history, uint64_t n_photons,
                           uint64_t seed, HitBuf H, uint64_t *hash_out, unsigned long long *work_counter) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Smem *S = reinterpret_cast<Smem *>(smem_raw);
  {
    const uint32_t *gs = reinterpret_cast<const uint32_t *>(geom);
    uint32_t *gd = reinterpret_cast<uint32_t *>(&S->g);
    for (int i = threadIdx.x; i < (int)(sizeof(DevGeom) / 4); i += kThreads) gd[i] = gs[i];
    const int n = T.n_materials * T.n_energies;
    for (int i = threadIdx.x; i < n; i += kThreads) { float4 v = T.mu[i]; v.w = maj[i % T.n_energies]; S->mu[i] = v; }
    __syncthreads();
  }
  const DevGeom &g = S->g;
  const float4 *mu = S->mu;
  const int lane = threadIdx.x & 31;
  HitStage &stage = S->stage[threadIdx.x >> 5];
  const unsigned lt_mask = (1u << lane) - 1u;
  const uint2 key = make_uint2((uint32_t)seed, (uint32_t)(seed >> 32));
  const bool use_phantom = src.kind == 1 && src.phantom != nullptr;

  Photon p; p.meta = 0; p.ndraw = 0; p.E = 0.f; p.path = 0.f; p.inv_mu = 0.f; p.pair = 0; p.ids = kNone;
  p.blk = make_uint4(0, 0, 0, 0);
#pragma unroll
  for (int k = 0; k < 3; ++k) { p.x[k] = 0.f; p.d[k] = 0.f; }
  uint64_t h = 0;
  int st = ST_REFILL;
  uint64_t w_next = 0, w_end = 0;          // this warp's reserved photon indices [w_next, w_end)
  bool exhausted = false;                  // the global counter ran past n_photons
  uint32_t stage_head = 0, stage_cnt = 0;  // ring buffer of staged hits (warp-uniform)

  // next uniform of this photon's stream [R4]
  auto draw = [&]() -> float {
    const uint32_t j = p.ndraw & 3u;
    if (j == 0) {
      const uint64_t history = first_history + p.pair;
      p.blk = philox4x32_10(make_uint4((uint32_t)history, (uint32_t)(history >> 32), 1u + (p.meta & 1u), p.ndraw >> 2), key);
    }
    ++p.ndraw;
    return u01(j == 0 ? p.blk.x : (j == 1 ? p.blk.y : (j == 2 ? p.blk.z : p.blk.w)));
  };
  // stage one hit per lane that has one; flush 32 staged hits with one atomic + coalesced stores (S10)
  auto stage_hits = [&](bool has, uint32_t ids, const float xg[3], float e, float tof) {
    const unsigned who = __ballot_sync(0xFFFFFFFFu, has);
    if (who == 0) return;
    if (has) {
      const uint32_t slot = (stage_head + stage_cnt + __popc(who & lt_mask)) & (kStage - 1);
      stage.w[0][slot] = (uint32_t)(first_history + p.pair); stage.w[1][slot] = ids;
      stage.w[2][slot] = __float_as_uint(xg[0]); stage.w[3][slot] = __float_as_uint(xg[1]); stage.w[4][slot] = __float_as_uint(xg[2]);
      stage.w[5][slot] = __float_as_uint(e); stage.w[6][slot] = __float_as_uint(tof);
    }
    stage_cnt += __popc(who);
    __syncwarp();
    if (stage_cnt >= 32) {
      unsigned long long base = 0;
      if (lane == 0) base = atomicAdd(H.n_hits, 32ull);
      base = __shfl_sync(0xFFFFFFFFu, base, 0);
      store_hit(H, base + lane, stage, (stage_head + lane) & (kStage - 1));
      stage_head = (stage_head + 32) & (kStage - 1); stage_cnt -= 32;
      __syncwarp();
    }
  };
  auto finish = [&]() {                    // photon ended: publish its hash, ask for a new photon
    if (HASH) hash_out[2ull * p.pair + (p.meta & 1u)] = h;
    st = ST_REFILL;
  };

#pragma unroll 1
  for (;;) {
    // ------------------------------------------------ choose the phase most lanes are waiting for
    unsigned m_ref = __ballot_sync(0xFFFFFFFFu, st == ST_REFILL);
    if (m_ref && exhausted && w_next >= w_end) {      // nothing left to hand out: those lanes retire
      if (st == ST_REFILL) st = ST_IDLE;
      m_ref = 0;
    }
    int phase = ST_IDLE, best = __popc(m_ref);
    if (best) phase = ST_REFILL;
    { int c;
      c = __popc(__ballot_sync(0xFFFFFFFFu, st == ST_SEARCH));   if (c > best) { best = c; phase = ST_SEARCH; }
      c = __popc(__ballot_sync(0xFFFFFFFFu, st == ST_STEP));     if (c > best) { best = c; phase = ST_STEP; }
      c = __popc(__ballot_sync(0xFFFFFFFFu, st == ST_COMPTON));  if (c > best) { best = c; phase = ST_COMPTON; }
      c = __popc(__ballot_sync(0xFFFFFFFFu, st == ST_PHANTOM));  if (c > best) { best = c; phase = ST_PHANTOM; }
      c = __popc(__ballot_sync(0xFFFFFFFFu, st == ST_RAYLEIGH)); if (c > best) { best = c; phase = ST_RAYLEIGH; } }
    if (phase == ST_IDLE) break;

    if (phase == ST_REFILL) {
      // ------------------------------------------------ REFILL: new photon + source sampling (S3) [R13-R15]
      if (w_next >= w_end && !exhausted) {
        unsigned long long b = 0;
        if (lane == 0) b = atomicAdd(work_counter, (unsigned long long)kChunk);
        b = __shfl_sync(0xFFFFFFFFu, b, 0);
        if (b >= n_photons) { exhausted = true; w_next = w_end = 0; }
        else { w_next = b; w_end = min((uint64_t)(b + kChunk), n_photons); }
      }
      const uint64_t j = w_next + __popc(m_ref & lt_mask);
      const bool take = st == ST_REFILL && j < w_end;
      w_next = min(w_next + (uint64_t)__popc(m_ref), w_end);
      if (take) {
        p.pair = (uint32_t)(j >> 1); p.meta = (uint32_t)(j & 1u) | (63u << 5); p.ndraw = 0; p.E = 511.0f; p.path = 0.0f; p.ids = kNone;
        if (HASH) h = 0xCBF29CE484222325ull;
        const uint64_t history = first_history + p.pair;
        const uint32_t h_lo = (uint32_t)history, h_hi = (uint32_t)(history >> 32);
        p.x[0] = src.pos[0]; p.x[1] = src.pos[1]; p.x[2] = src.pos[2];
        if (src.kind == 1) {
          const uint4 w = philox4x32_10(make_uint4(h_lo, h_hi, 0u, 0u), key);
          const uint64_t Wl = src.w_total & 0xFFFFFFFFull, Wh = src.w_total >> 32;          // floor(w.x * W / 2^32), exact
          const uint64_t target = (uint64_t)w.x * Wh + (((uint64_t)w.x * Wl) >> 32);
          uint32_t lo = 0, hi = src.n_active - 1;
          while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (src.act_cdf[mid] > target) hi = mid; else lo = mid + 1; }
          const uint32_t vi = src.act_index[lo], nx = (uint32_t)src.dims[0], ny = (uint32_t)src.dims[1];
          p.x[0] = src.origin[0] + ((float)(vi % nx) + u01(w.y)) * src.voxel[0];
          p.x[1] = src.origin[1] + ((float)((vi / nx) % ny) + u01(w.z)) * src.voxel[1];
          p.x[2] = src.origin[2] + ((float)(vi / (nx * ny)) + u01(w.w)) * src.voxel[2];
        }
        const uint4 w = philox4x32_10(make_uint4(h_lo, h_hi, 0u, 1u), key);
        if (src.kind == 2) { p.d[0] = src.beam[0]; p.d[1] = src.beam[1]; p.d[2] = src.beam[2]; }
        else {
          const float u = u01(w.x), ct = 1.0f - 2.0f * u, sth = 2.0f * sqrtf(u * (1.0f - u));   // sin^2 = (1-ct)(1+ct)
          float sp, cp; sincospif(2.0f * u01(w.y), &sp, &cp);
          p.d[0] = sth * cp; p.d[1] = sth * sp; p.d[2] = ct;
        }
        if (p.meta & 1u) {                                            // photon B: opposite, plus acolinearity
          p.d[0] = -p.d[0]; p.d[1] = -p.d[1]; p.d[2] = -p.d[2];
          if (src.acol_sigma > 0.0f) {
            const float rho = src.acol_sigma * sqrtf(-2.0f * logf(u01(w.z)));
            float sr, cr; sincosf(rho, &sr, &cr);
            float sp, cp; sincospif(2.0f * u01(w.w), &sp, &cp);
            rotate(p.d, cr, sr, cp, sp);
          }
        }
        if (use_phantom) { p.meta |= 1u << 11; p.inv_mu = rcp_fast(mu_lookup(mu, T, src.ph_major, p.E).z); st = ST_PHANTOM; }
        else st = ST_SEARCH;
      }
      if (!use_phantom) phase = ST_SEARCH;                            // new photons go straight into the search
    }
    if (phase == ST_SEARCH) {
      // ------------------------------------------------ SEARCH: nearest-entry panel over all panels [R6]
      if (st == ST_SEARCH) {
        const int excl = ph_panel(p);
        // candidate panels: with a common axial axis v, a panel can only be hit if the ray passes within the
        // cross-section radius of its axis line (centre, v) and its bounding sphere is not entirely behind
        unsigned long long cand = (g.n_panels >= 64 ? ~0ull : (1ull << g.n_panels) - 1ull) & ~(1ull << excl);
        if (g.common_v) {
          const float nx = p.d[1] * g.vaxis[2] - p.d[2] * g.vaxis[1], ny = p.d[2] * g.vaxis[0] - p.d[0] * g.vaxis[2],
                      nz = p.d[0] * g.vaxis[1] - p.d[1] * g.vaxis[0];
          const float lim = (nx * nx + ny * ny + nz * nz) * g.cull_r2sq + 1e-12f;
          cand = 0;
#pragma unroll 1
          for (int q = 0; q < g.n_panels; ++q) {
            const float mx = g.centre[q][0] - p.x[0], my = g.centre[q][1] - p.x[1], mz = g.centre[q][2] - p.x[2];
            const float s1 = mx * nx + my * ny + mz * nz, s2 = mx * p.d[0] + my * p.d[1] + mz * p.d[2];
            if (s1 * s1 <= lim && s2 >= -g.cull_r3 && q != excl) cand |= 1ull << q;
          }
        }
        float bt = INFINITY; int bp = -1;
        while (cand) {                                               // ascending index: ties keep the lowest [R6]
          const int q = __ffsll((long long)cand) - 1; cand &= cand - 1ull;
          float xl[3], dl[3];
          to_local(g.pose[q], p.x, p.d, xl, dl);
          float tn = -INFINITY, tf = INFINITY;
#pragma unroll
          for (int k = 0; k < 3; ++k) {
            // a zero component behaves like +tiny: inside -> (-inf, +inf), outside -> miss [R32]
            const float inv = rcp_fast(dl[k] == 0.0f ? 1e-30f : dl[k]);
            const float t1 = (g.blo[k] - xl[k]) * inv, t2 = (g.bhi[k] - xl[k]) * inv;
            tn = fmaxf(tn, fminf(t1, t2)); tf = fminf(tf, fmaxf(t1, t2));
          }
          const float te = fmaxf(tn, 0.0f);
          if (tf > te && te < bt) { bt = te; bp = q; }
        }
        if (bp < 0) { if (HASH) hash_ev(h, EV_ESCAPE, 0); finish(); }
        else {
          if (HASH) hash_ev(h, EV_ENTER, (uint32_t)bp);
          float xl[3], dl[3];
          to_local(g.pose[bp], p.x, p.d, xl, dl);
#pragma unroll
          for (int k = 0; k < 3; ++k) { p.x[k] = fmaf(bt, dl[k], xl[k]); p.d[k] = dl[k]; }   // [R18]
          p.path += bt; ph_set_panel(p, bp);
          p.inv_mu = rcp_fast(mu_lookup(mu, T, 0, p.E).w);
          st = ST_STEP;
        }
      }
    } else if (phase == ST_STEP) {
      // ------------------------------------------------ STEP: Woodcock step, layer selection, lattice lookup [R19]
      bool hit = false; float xg[3] = {0.f, 0.f, 0.f}; uint32_t hit_ids = 0;
      if (st == ST_STEP) {
        const float s = -__logf(draw()) * p.inv_mu;
        float tf = INFINITY;
#pragma unroll
        for (int k = 0; k < 3; ++k) {                                 // distance to the box exit [R32]
          const float inv = rcp_fast(p.d[k] == 0.0f ? 1e-30f : p.d[k]);
          tf = fminf(tf, ((p.d[k] >= 0.0f ? g.bhi[k] : g.blo[k]) - p.x[k]) * inv);
        }
        const int panel = ph_panel(p);
        if (s >= tf) {                                                // leaves the panel: back to the global frame [R33]
          tf = fmaxf(tf, 0.0f);
          const float xl[3] = { fmaf(tf, p.d[0], p.x[0]), fmaf(tf, p.d[1], p.x[1]), fmaf(tf, p.d[2], p.x[2]) };
          const float dl[3] = { p.d[0], p.d[1], p.d[2] };
          p.path += tf; if (HASH) hash_ev(h, EV_EXIT, (uint32_t)panel);
          point_to_global(g.pose[panel], xl, p.x); dir_to_global(g.pose[panel], dl, p.d);
          st = ST_SEARCH;
        } else {
#pragma unroll
          for (int k = 0; k < 3; ++k) p.x[k] = fmaf(s, p.d[k], p.x[k]);
          p.path += s;
          uint32_t ids;                                               // depth -> layer -> crystal
          const int mat = lattice_lookup(g, __float2int_rd(p.x[0] * kQ) + g.hWq, __float2int_rd(p.x[1] * kQ) + g.hHq,
                                         __float2int_rd(p.x[2] * kQ), ids);
          if (mat < 0) { if (HASH) hash_ev(h, EV_STEP_VACUUM, 0); }
          else {
            if (ids != kNone) ids |= (uint32_t)panel << 26;
            const float4 m4 = mu_lookup(mu, T, mat, p.E);
            const float t = draw() * m4.w;                            // [R20] one draw picks the outcome
            if (t < m4.x) {                                           // photoelectric: deposit E, end
              if (HASH) hash_ev(h, EV_PE, ids);
              if (ids != kNone) { hit = true; hit_ids = ids; point_to_global(g.pose[panel], p.x, xg); }
              finish();
            } else if (t < m4.y) { p.ids = ids; st = ST_COMPTON; }
            else if (t < m4.z) { p.ids = ids; st = ST_RAYLEIGH; }
            else if (HASH) hash_ev(h, EV_VIRTUAL, ids);
          }
        }
      }
      stage_hits(hit, hit_ids | ((p.meta & 1u) << 4) | ((p.meta >> 1) & 15u), xg, p.E, p.path * kInvC);
    } else if (phase == ST_COMPTON) {
      // ------------------------------------------------ COMPTON: one Klein-Nishina trial per visit [R20]
      bool hit = false; float xg[3] = {0.f, 0.f, 0.f}, e_dep = 0.f;
      if (st == ST_COMPTON) {
        const bool in_ph = (p.meta >> 11) & 1u;
        const float k = p.E * (1.0f / kMec2), e0 = rcp_fast(1.0f + 2.0f * k), e02 = e0 * e0;
        const float a1 = -__logf(e0), a2 = 0.5f * (1.0f - e02);
        const float ua = draw(), ub = draw(), uc = draw();
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
        if (gr >= uc || (p.meta >> 12) >= 63u) {                      // accepted [R22: the 64th trial always is]
          p.meta &= 0xFFFu;
          float sp, cp; sincos_2pi(draw(), sp, cp);
          rotate(p.d, 1.0f - t, sqrt_fast(fmaxf(t * tm, 0.0f)), cp, sp);
          const float dep = om * p.E, E2 = p.E - dep;
          const bool cut = E2 < kCutoff;                              // [R12]
          if (in_ph) {
            if (HASH) hash_ev(h, EV_PH_COMPTON, 0);
            if (cut) { if (HASH) hash_ev(h, EV_PH_CUTOFF, 0); finish(); }
            else { p.E = E2; p.inv_mu = rcp_fast(mu_lookup(mu, T, src.ph_major, p.E).z); st = ST_PHANTOM; }
          } else {
            if (HASH) { hash_ev(h, EV_COMPTON, p.ids); if (cut) hash_ev(h, EV_CUTOFF, p.ids); }
            if (p.ids != kNone) { hit = true; e_dep = cut ? p.E : dep; point_to_global(g.pose[ph_panel(p)], p.x, xg); }
            if (cut) finish();
            else { p.E = E2; p.inv_mu = rcp_fast(mu_lookup(mu, T, 0, p.E).w); st = ST_STEP; }
          }
        } else p.meta += 1u << 12;
      }
      const uint32_t seq = (p.meta >> 1) & 15u;
      stage_hits(hit, p.ids | ((p.meta & 1u) << 4) | seq, xg, e_dep, p.path * kInvC);
      if (hit && seq < 15u) p.meta += 2u;                             // [R9] 4-bit saturating hit counter
    } else if (phase == ST_RAYLEIGH) {
      // ------------------------------------------------ RAYLEIGH: Thomson pdf by closed-form inversion [R20]
      if (st == ST_RAYLEIGH) {
        const float a = 4.0f * draw() - 2.0f, q = sqrtf(a * a + 1.0f);
        const float ct = cbrtf(a + q) - cbrtf(q - a);
        float sp, cp; sincos_2pi(draw(), sp, cp);
        rotate(p.d, ct, sqrtf(fmaxf(0.0f, 1.0f - ct * ct)), cp, sp);
        if ((p.meta >> 11) & 1u) { if (HASH) hash_ev(h, EV_PH_RAYLEIGH, 0); st = ST_PHANTOM; }
        else { if (HASH) hash_ev(h, EV_RAYLEIGH, p.ids); st = ST_STEP; }
      }
    } else if (phase == ST_PHANTOM) {
      // ------------------------------------------------ PHANTOM: Woodcock tracking in the voxel grid [R17]
      if (st == ST_PHANTOM) {
        const float s = -__logf(draw()) * p.inv_mu;
        int v[3]; bool out = false;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          p.x[k] = fmaf(s, p.d[k], p.x[k]);
          v[k] = __float2int_rd((p.x[k] - src.origin[k]) * src.inv_voxel[k]);
          out = out || v[k] < 0 || v[k] >= src.dims[k];
        }
        p.path += s;
        if (out) { if (HASH) hash_ev(h, EV_PH_LEAVE, 0); p.meta &= ~(1u << 11); st = ST_SEARCH; }
        else {
          const int mat = (int)src.phantom[((size_t)v[2] * src.dims[1] + v[1]) * src.dims[0] + v[0]] - 1;
          if (mat >= 0) {
            const float4 m4 = mu_lookup(mu, T, mat, p.E);
            const float t = draw() * mu_lookup(mu, T, src.ph_major, p.E).z;
            if (t < m4.x) { if (HASH) hash_ev(h, EV_PH_ABSORBED, 0); finish(); }
            else if (t < m4.y) st = ST_COMPTON;
            else if (t < m4.z) st = ST_RAYLEIGH;
          }
        }
      }
    }
  }

  // ------------------------------------------------ drain the staged hits (fewer than 32 per warp)
  if (stage_cnt) {
    unsigned long long base = 0;
    if (lane == 0) base = atomicAdd(H.n_hits, (unsigned long long)stage_cnt);
    base = __shfl_sync(0xFFFFFFFFu, base, 0);
    if ((uint32_t)lane < stage_cnt) store_hit(H, base + lane, stage, (stage_head + lane) & (kStage - 1));
  }
}

size_t transport_smem_bytes(const DevTables &T) {
  return sizeof(Smem) - sizeof(float4) + sizeof(float4) * (size_t)T.n_materials * T.n_energies + 16;
}

cudaError_t launch_transport(const DevGeom *geom, const DevTables &T, const float *maj, const DevSource &src,
                             uint64_t first_history, uint64_t n_pairs, uint64_t seed, const HitBuf &H, uint64_t *hash_out,
                             unsigned long long *work_counter, int sm_count, cudaStream_t stream) {
  const size_t smem = transport_smem_bytes(T);
  const uint64_t n_photons = 2 * n_pairs;
  const uint64_t want = (n_photons + kThreads - 1) / kThreads;
  static const int ctas_per_sm = getenv("GPET_CTAS_PER_SM") ? atoi(getenv("GPET_CTAS_PER_SM")) : 4;
  const uint64_t resident = (uint64_t)sm_count * ctas_per_sm;         // persistent grid
  const int blocks = (int)(want < resident ? (want ? want : 1) : resident);
  cudaError_t e = cudaMemsetAsync(work_counter, 0, sizeof(unsigned long long), stream);
  if (e != cudaSuccess) return e;
  if (hash_out) {
    e = cudaFuncSetAttribute(transport_wavefront_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    transport_wavefront_kernel<true><<<blocks, kThreads, smem, stream>>>(geom, T, maj, src, first_history, n_photons, seed, H, hash_out, work_counter);
  } else {
    e = cudaFuncSetAttribute(transport_wavefront_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    transport_wavefront_kernel<false><<<blocks, kThreads, smem, stream>>>(geom, T, maj, src, first_history, n_photons, seed, H, hash_out, work_counter);
  }
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
      const float *P = g.pose[p];
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
