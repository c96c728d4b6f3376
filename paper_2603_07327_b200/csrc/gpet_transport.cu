// gpet_transport.cu -- photon-pair transport kernels (S2..S10 of DESIGN.md section 1).
// PAPER.md:33 (panel transfer, global->local), PAPER.md:43 (Woodcock tracking, layer selection, exit/cutoff).
#include "gpet_internal.h"

namespace gpet {

// ---------------------------------------------------------------- shared-memory staging
struct Smem {
  DevGeom g;
  float4 mu[1];   // [n_materials][n_energies], .w = detector majorant
};

__device__ __forceinline__ void stage(Smem *s, const DevGeom *g, const DevTables &T, const float *maj) {
  const uint32_t *src = reinterpret_cast<const uint32_t *>(g);
  uint32_t *dst = reinterpret_cast<uint32_t *>(&s->g);
  for (int i = threadIdx.x; i < (int)(sizeof(DevGeom) / 4); i += blockDim.x) dst[i] = src[i];
  const int n = T.n_materials * T.n_energies;
  for (int i = threadIdx.x; i < n; i += blockDim.x) {
    float4 v = T.mu[i]; v.w = maj[i % T.n_energies]; s->mu[i] = v;
  }
  __syncthreads();
}

// [R11] linear interpolation on the energy grid: returns {mu_pe, mu_pe+mu_C, mu_tot, mu_maj}
__device__ __forceinline__ float4 mu_lookup(const float4 *mu, const DevTables &T, int m, float E) {
  const float x = (E - T.e_min) * T.inv_step;
  int i = min(__float2int_rd(x), T.n_energies - 2); i = max(i, 0);
  const float f = x - (float)i;
  const float4 a = mu[m * T.n_energies + i], b = mu[m * T.n_energies + i + 1];
  return make_float4(fmaf(f, b.x - a.x, a.x), fmaf(f, b.y - a.y, a.y), fmaf(f, b.z - a.z, a.z), fmaf(f, b.w - a.w, a.w));
}

// ---------------------------------------------------------------- hit output (S10)
// Warp-aggregated append: the lanes that reach this point together take one atomic.
__device__ __forceinline__ void append_hit(const HitBuf &H, uint32_t history, uint32_t ids, const float x[3], float e, float tof) {
  const unsigned mask = __activemask();
  const int lane = threadIdx.x & 31, leader = __ffs(mask) - 1;
  unsigned long long base = 0;
  if (lane == leader) base = atomicAdd(H.n_hits, (unsigned long long)__popc(mask));
  base = __shfl_sync(mask, base, leader);
  const unsigned long long i = base + __popc(mask & ((1u << lane) - 1u));
  if (i < H.capacity) {
    H.history[i] = history; H.ids[i] = ids; H.x[i] = x[0]; H.y[i] = x[1]; H.z[i] = x[2]; H.e[i] = e; H.tof[i] = tof;
  }
}

// ---------------------------------------------------------------- [R20] Klein-Nishina
// Returns om = 1 - eps (the deposited fraction).  Both om = 1 - eps and em = eps - eps0 are formed
// without cancellation (expm1 from the nearer end on the exponential branch, difference of squares on
// the other), so that sin^2(theta) = t (2 - t) with t = om/(k eps), 2 - t = em/(eps0 k eps) keeps full
// relative accuracy at both poles.  In plain fp32, small-angle and back-scatter events lose 3-4 digits
// of the scattering angle and move later hits by several micrometres.
__device__ __forceinline__ float kn_sample(Stream &r, float E, float &cos_t, float &sin2_t) {
  const float k = E / kMec2, e0 = 1.0f / (1.0f + 2.0f * k), e02 = e0 * e0;
  const float a1 = -logf(e0), a2 = 0.5f * (1.0f - e02), pa = a1 / (a1 + a2);
  float om = 0.0f, t = 0.0f, tm = 2.0f;
  for (int n = 1; n <= 64; ++n) {
    const float ua = r.next(), ub = r.next(), uc = r.next();
    float eps, em;
    if (ua < pa) {
      if (ub < 0.5f) { om = -expm1f(-a1 * ub); eps = 1.0f - om; em = eps - e0; }
      else { em = e0 * expm1f(a1 * (1.0f - ub)); eps = e0 + em; om = 1.0f - eps; }
    } else {
      eps = sqrtf(fmaf(1.0f - e02, ub, e02));
      om = (1.0f - e02) * (1.0f - ub) / (1.0f + eps); em = (1.0f - e02) * ub / (eps + e0);
    }
    const float ike = 1.0f / (k * eps);
    t = om * ike; tm = em * ike / e0;
    const float g = 1.0f - eps * t * tm / (1.0f + eps * eps);
    if (g >= uc) break;
  }
  cos_t = 1.0f - t; sin2_t = fmaxf(t * tm, 0.0f);
  return om;
}
// returns the deposited energy E - E' and rotates d
__device__ __forceinline__ float compton(Stream &r, float E, float d[3]) {
  float ct, s2; const float om = kn_sample(r, E, ct, s2);
  float sp, cp; sincospif(2.0f * r.next(), &sp, &cp);
  rotate(d, ct, sqrtf(s2), cp, sp);
  return om * E;
}
__device__ __forceinline__ void rayleigh(Stream &r, float d[3]) {
  const float a = 4.0f * r.next() - 2.0f, q = sqrtf(a * a + 1.0f);
  const float ct = cbrtf(a + q) - cbrtf(q - a);
  float sp, cp; sincospif(2.0f * r.next(), &sp, &cp);
  rotate(d, ct, sqrtf(fmaxf(0.0f, 1.0f - ct * ct)), cp, sp);
}

// ---------------------------------------------------------------- [R6] panel search over all panels
__device__ __forceinline__ int panel_search(const DevGeom &g, const float x[3], const float d[3], int excl, float &t_enter) {
  float best = INFINITY; int bp = -1;
  for (int p = 0; p < g.n_panels; ++p) {
    if (p == excl) continue;
    float xl[3], dl[3], tn, tf;
    to_local(g.pose[p], x, d, xl, dl);
    if (!slab(g.blo, g.bhi, xl, dl, tn, tf)) continue;
    const float te = fmaxf(tn, 0.0f);
    if (tf > te && te < best) { best = te; bp = p; }
  }
  t_enter = best; return bp;
}

// ---------------------------------------------------------------- one photon, run to completion
template <bool HASH>
__device__ void transport_photon(const Smem *S, const DevTables &T, const DevSource &src, const HitBuf &H, uint64_t seed,
                                 uint64_t history, int photon, float x[3], float d[3], bool in_phantom, uint64_t &h) {
  const DevGeom &g = S->g;
  Stream r; r.init(seed, history, photon ? 2u : 1u);
  float E = 511.0f, path = 0.0f; int seq = 0;

  if (in_phantom) {                                                  // [R17] Woodcock in the voxel grid
    for (;;) {
      const float mu_maj = mu_lookup(S->mu, T, src.ph_major, E).z;
      const float s = -logf(r.next()) / mu_maj;
      int v[3]; bool out = false;
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        x[k] = fmaf(s, d[k], x[k]);
        v[k] = __float2int_rd((x[k] - src.origin[k]) * src.inv_voxel[k]);
        out = out || v[k] < 0 || v[k] >= src.dims[k];
      }
      path += s;
      if (out) { if (HASH) hash_ev(h, EV_PH_LEAVE, 0); break; }
      const int mat = (int)src.phantom[((size_t)v[2] * src.dims[1] + v[1]) * src.dims[0] + v[0]] - 1;
      if (mat < 0) continue;
      const float4 mu = mu_lookup(S->mu, T, mat, E);
      const float t = r.next() * mu_maj;
      if (t < mu.x) { if (HASH) hash_ev(h, EV_PH_ABSORBED, 0); return; }
      else if (t < mu.y) {
        E -= compton(r, E, d); if (HASH) hash_ev(h, EV_PH_COMPTON, 0);
        if (E < kCutoff) { if (HASH) hash_ev(h, EV_PH_CUTOFF, 0); return; }
      } else if (t < mu.z) { rayleigh(r, d); if (HASH) hash_ev(h, EV_PH_RAYLEIGH, 0); }
    }
  }

  int excl = -1;
  for (;;) {
    float te;
    const int p = panel_search(g, x, d, excl, te);
    if (p < 0) { if (HASH) hash_ev(h, EV_ESCAPE, 0); return; }
    if (HASH) hash_ev(h, EV_ENTER, (uint32_t)p);
    const float *P = g.pose[p];
    float xl[3], dl[3];
    to_local(P, x, d, xl, dl);
#pragma unroll
    for (int k = 0; k < 3; ++k) xl[k] = fmaf(te, dl[k], xl[k]);     // [R18]
    path += te;
    bool alive = true;
    for (;;) {                                                       // [R19]
      const float mu_maj = mu_lookup(S->mu, T, 0, E).w;
      const float s = -logf(r.next()) / mu_maj;
      float tn, tf; slab(g.blo, g.bhi, xl, dl, tn, tf);
      if (s >= tf) {
        tf = fmaxf(tf, 0.0f);
#pragma unroll
        for (int k = 0; k < 3; ++k) xl[k] = fmaf(tf, dl[k], xl[k]);
        path += tf; if (HASH) hash_ev(h, EV_EXIT, (uint32_t)p); break;
      }
#pragma unroll
      for (int k = 0; k < 3; ++k) xl[k] = fmaf(s, dl[k], xl[k]);
      path += s;
      uint32_t ids;                                                  // PAPER.md:43 layer selection + lattice
      const int mat = lattice_lookup(g, __float2int_rd(xl[0] * kQ) + g.hWq, __float2int_rd(xl[1] * kQ) + g.hHq,
                                     __float2int_rd(xl[2] * kQ), ids);
      if (mat < 0) { if (HASH) hash_ev(h, EV_STEP_VACUUM, 0); continue; }
      if (ids != kNone) ids |= (uint32_t)p << 26;
      const float4 mu = mu_lookup(S->mu, T, mat, E);
      const float t = r.next() * mu_maj;                             // [R20] one draw picks the outcome
      if (t < mu.x) {
        if (HASH) hash_ev(h, EV_PE, ids);
        if (ids != kNone) {
          float xg[3]; point_to_global(P, xl, xg);
          append_hit(H, (uint32_t)history, ids | (photon << 4) | min(seq, 15), xg, E, path * kInvC); ++seq;
        }
        alive = false; break;
      } else if (t < mu.y) {
        const float dep = compton(r, E, dl), E2 = E - dep;
        if (HASH) hash_ev(h, EV_COMPTON, ids);
        const bool cut = E2 < kCutoff;                               // [R12]
        if (cut && HASH) hash_ev(h, EV_CUTOFF, ids);
        if (ids != kNone) {
          float xg[3]; point_to_global(P, xl, xg);
          append_hit(H, (uint32_t)history, ids | (photon << 4) | min(seq, 15), xg, cut ? E : dep, path * kInvC); ++seq;
        }
        if (cut) { alive = false; break; }
        E = E2;
      } else if (t < mu.z) {
        rayleigh(r, dl); if (HASH) hash_ev(h, EV_RAYLEIGH, ids);
      } else if (HASH) hash_ev(h, EV_VIRTUAL, ids);
    }
    if (!alive) return;
    point_to_global(P, xl, x); dir_to_global(P, dl, d);              // [R33]
    excl = p;
  }
}

// ---------------------------------------------------------------- source (S3) [R13-R15]
__device__ __forceinline__ void sample_pair(const DevSource &src, uint64_t seed, uint64_t history, float x0[3], float dA[3], float dB[3]) {
  const uint2 key = make_uint2((uint32_t)seed, (uint32_t)(seed >> 32));
  const uint32_t h_lo = (uint32_t)history, h_hi = (uint32_t)(history >> 32);
  x0[0] = src.pos[0]; x0[1] = src.pos[1]; x0[2] = src.pos[2];
  if (src.kind == 1) {
    const uint4 w = philox4x32_10(make_uint4(h_lo, h_hi, 0u, 0u), key);
    // target = floor(w.x * W_total / 2^32), exact: W_total = Wh*2^32 + Wl
    const uint64_t Wl = src.w_total & 0xFFFFFFFFull, Wh = src.w_total >> 32;
    const uint64_t target = (uint64_t)w.x * Wh + (((uint64_t)w.x * Wl) >> 32);
    uint32_t lo = 0, hi = src.n_active - 1;
    while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (src.act_cdf[mid] > target) hi = mid; else lo = mid + 1; }
    const uint32_t vi = src.act_index[lo];
    const uint32_t nx = (uint32_t)src.dims[0], ny = (uint32_t)src.dims[1];
    const int v[3] = { (int)(vi % nx), (int)((vi / nx) % ny), (int)(vi / (nx * ny)) };
    const float u[3] = { u01(w.y), u01(w.z), u01(w.w) };
#pragma unroll
    for (int k = 0; k < 3; ++k) x0[k] = src.origin[k] + ((float)v[k] + u[k]) * src.voxel[k];
  }
  const uint4 w = philox4x32_10(make_uint4(h_lo, h_hi, 0u, 1u), key);
  if (src.kind == 2) { dA[0] = src.beam[0]; dA[1] = src.beam[1]; dA[2] = src.beam[2]; }
  else {
    const float u = u01(w.x), ct = 1.0f - 2.0f * u, st = 2.0f * sqrtf(u * (1.0f - u));   // sin^2 = (1-ct)(1+ct), no cancellation
    float sp, cp; sincospif(2.0f * u01(w.y), &sp, &cp);
    dA[0] = st * cp; dA[1] = st * sp; dA[2] = ct;
  }
  dB[0] = -dA[0]; dB[1] = -dA[1]; dB[2] = -dA[2];
  if (src.acol_sigma > 0.0f) {
    const float rho = src.acol_sigma * sqrtf(-2.0f * logf(u01(w.z)));
    float sr, cr; sincosf(rho, &sr, &cr);
    float sp, cp; sincospif(2.0f * u01(w.w), &sp, &cp);
    rotate(dB, cr, sr, cp, sp);
  }
}

// ---------------------------------------------------------------- v1: one thread per pair, run to completion
template <bool HASH>
__global__ void __launch_bounds__(256) transport_pairs_kernel(const DevGeom *geom, DevTables T, const float *maj, DevSource src,
                                                              uint64_t first_history, uint64_t n_pairs, uint64_t seed,
                                                              HitBuf H, uint64_t *hash_out) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Smem *S = reinterpret_cast<Smem *>(smem_raw);
  stage(S, geom, T, maj);
  const bool in_ph = src.kind == 1 && src.phantom != nullptr;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_pairs; i += (uint64_t)gridDim.x * blockDim.x) {
    const uint64_t history = first_history + i;
    float x0[3], dA[3], dB[3];
    sample_pair(src, seed, history, x0, dA, dB);
    uint64_t h = 0xCBF29CE484222325ull;
    float xa[3] = { x0[0], x0[1], x0[2] };
    transport_photon<HASH>(S, T, src, H, seed, history, 0, xa, dA, in_ph, h);
    if (HASH) hash_ev(h, EV_PHOTON_B, 0);
    float xb[3] = { x0[0], x0[1], x0[2] };
    transport_photon<HASH>(S, T, src, H, seed, history, 1, xb, dB, in_ph, h);
    if (HASH) hash_out[i] = h;
  }
}

size_t transport_smem_bytes(const DevTables &T) {
  return sizeof(DevGeom) + sizeof(float4) * (size_t)T.n_materials * T.n_energies + 16;
}

cudaError_t launch_transport(const DevGeom *geom, const DevTables &T, const float *maj, const DevSource &src,
                             uint64_t first_history, uint64_t n_pairs, uint64_t seed, const HitBuf &H, uint64_t *hash_out,
                             int sm_count, cudaStream_t stream) {
  const size_t smem = transport_smem_bytes(T);
  const int threads = 256;
  const uint64_t want = (n_pairs + threads - 1) / threads;
  const int blocks = (int)(want < (uint64_t)sm_count * 8 ? (want ? want : 1) : (uint64_t)sm_count * 8);
  cudaError_t e;
  if (hash_out) {
    e = cudaFuncSetAttribute(transport_pairs_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    transport_pairs_kernel<true><<<blocks, threads, smem, stream>>>(geom, T, maj, src, first_history, n_pairs, seed, H, hash_out);
  } else {
    e = cudaFuncSetAttribute(transport_pairs_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    transport_pairs_kernel<false><<<blocks, threads, smem, stream>>>(geom, T, maj, src, first_history, n_pairs, seed, H, hash_out);
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
