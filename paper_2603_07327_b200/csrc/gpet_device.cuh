// gpet_device.cuh -- device-side building blocks shared by the transport, locate and digitizer kernels.
// sm_100a only.  "[Rn]" = reading n in DESIGN.md section 2; PAPER.md:<line> = the paper.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gpet {

constexpr int   kMaxPanels = 64;          // 63 usable (packed id 0xFFFFFFFF is reserved)
constexpr int   kMaxLayers = 4;
constexpr int   kMaxMaterials = 8;
constexpr float kQ = 1048576.0f;          // [R7] 2^20 quantisation units per mm
constexpr float kMec2 = 510.99895f;       // [R12]
constexpr float kInvC = 1.0f / 299.792458f;   // ns per mm
constexpr float kCutoff = 10.0f;          // [R12]
constexpr uint32_t kNone = 0xFFFFFFFFu;

// ---------------------------------------------------------------- descriptor as the kernels see it
// Exact division of a Q coordinate n (0 <= n < 2^31) by a Q pitch d >= 2 with one high multiply and a shift:
// floor(n / d) = umulhi(n, magic) >> shift, magic = floor(2^(32 + shift) / d) + 1, shift = ceil(log2 d) - 1.
// (magic d - 2^(32+shift) lies in (0, d] and d <= 2^(shift+1), so the error term n (magic d - 2^(32+shift)) / (d 2^(32+shift))
// stays below 1/d for n < 2^31: the quotient is exact.  Checked against plain division in tests/test_abi.py.)
struct QDiv { uint32_t magic, shift; };
__host__ __device__ inline QDiv qdiv_make(uint32_t d) {
  uint32_t sh = 0; while ((2ull << sh) < (unsigned long long)d) ++sh;        // 2^sh < d <= 2^(sh+1)
  QDiv q; q.shift = sh; q.magic = (uint32_t)((1ull << (32 + sh)) / d) + 1u; return q;
}

struct __align__(16) DevLayer {   // 64 bytes = four 16-byte rows: the transport kernel reads the record of a lane's layer from shared memory
  int c0, c1;                 // depth range [c0, c1) in Q units (unused layers: c0 = c1 = INT_MAX, never selected)
  int cmat, gmat;
  int n[2], pitch[2];
  int lo[2], hi[2];           // crystal occupies frac in [lo, hi) of each pitch cell
  int off[2];
  uint32_t magic[2];          // QDiv of the pitches ...
  // ... whose shifts ride in the top byte of n[] (n <= 8192)
};
struct __align__(16) DevPanel {
  float pose[12];             // front-face centre, u, v, w
  float cx, cy, cz;           // global position of the box centre (search culling)
  uint32_t open_faces;        // bit 2k + (outward along +axis k): no other panel has a point beyond that face of this box
  float skew[4];              // 80-byte stride: records of 8 consecutive panels start in 8 different 16-byte bank groups, so
};                            // lanes reading the poses of different panels (entry / exit / hit transforms) rarely conflict
// Header of the descriptor: everything the kernels read with the SAME address in every lane (extents, lattice
// parameters, box centres for the search cull).  The transport kernel receives it as a __grid_constant__ parameter, so
// these reads are constant-bank operands and do not load the shared-memory pipe; the per-panel records, read with a
// per-lane panel index, are staged into shared memory.
struct DevGeomHead {
  int n_panels, n_layers;
  int Wq, Hq, Dq, hWq, hHq;
  int nmod[2], msq[2], mpq[2];
  uint32_t mp_magic[2], mp_shift[2];   // QDiv of the module pitches
  float blo[3], bhi[3];       // panel box in the tracking frame (fp32 roundings of the Q extents)
  uint32_t det_mask;          // materials referenced by the layers
  int ring;                   // 1 = repetition mode
  int planar;                 // 1 = every panel has v = +z and u_z = w_z = o_z = 0: the search shares the axial slab
  float cull_r2, cull_r3;     // radius (+ margin) of the circle / sphere about a panel box: (a,c) plane / 3-D
  float bore_r;               // planar detectors: no panel has a point closer than this to the z axis (<= 0: unknown / not planar)
  // repetition-mode rings: the front faces lie on a regular polygon; a photon inside its inscribed circle
  // finds its first panel by the polygon edge it crosses (ring_entry_fast in gpet_transport.cu)
  float ring_phi0, ring_kscale;   // azimuth of panel 0 (rad); n_panels / (2 pi)
  float ring_edge_h;          // half length of a polygon edge minus 1 um (<= 0: shortcut off)
  // [R19] majorant regions: maximal runs of layers with the same crystal and gap material; region r spans the depths
  // [reg_lo[r], reg_hi[r]) (reg_lo past n_regions holds +inf); reg_mats = crystal material | gap material << 4
  int n_regions; float reg_lo[kMaxLayers], reg_hi[kMaxLayers]; uint32_t reg_mats[kMaxLayers];
  DevLayer layer[kMaxLayers];
  float ctr[kMaxPanels][3];   // global position of every box centre (same values as DevPanel::cx, cy, cz)
};
struct DevGeom : DevGeomHead {
  DevPanel panel[kMaxPanels]; // LAST member: kernels stage only the first n_panels records into shared memory
};
inline size_t panel_bytes(int n_panels) { return sizeof(DevPanel) * (size_t)n_panels; }
__host__ __device__ inline size_t geom_bytes(int n_panels) { return sizeof(DevGeom) - sizeof(DevPanel) * (size_t)(kMaxPanels - n_panels); }

struct DevTables {            // [R11] per staged material, per energy: {mu_pe, mu_pe+mu_C, mu_tot, detector majorant}
  int n_staged, n_energies;   // only the materials a run can touch are staged into shared memory
  float e_min, inv_step;
  uint32_t matmap;            // 4 bits per material id: its staged slot
  const float4 *mu;           // [n_staged][n_energies]
};

// ---------------------------------------------------------------- [R1] Philox4x32-10
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
    c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
    k.x += 0x9E3779B9u; k.y += 0xBB67AE85u;
  }
  return c;
}
// The same generator with the ten round keys precomputed on the host (they depend on the seed only): passed as a
// kernel parameter they are constant-bank operands of the XORs, so a round is two wide multiplies and two LOP3.
struct PhiloxKeys { uint32_t k[20]; };
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, const PhiloxKeys &K) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
    c = make_uint4(hi1 ^ c.y ^ K.k[2 * r], lo1, hi0 ^ c.w ^ K.k[2 * r + 1], lo0);
  }
  return c;
}
// [R2] u = ((x >> 9) + 0.5) * 2^-23, formed without an integer-to-float conversion: k = x >> 9 placed in the mantissa of
// 1.0 gives 1 + k 2^-23; subtracting 1 - 2^-24 leaves (2k + 1) 2^-24, which has 24 significant bits: every step is exact
__device__ __forceinline__ float u01(uint32_t x) { return __uint_as_float((x >> 9) | 0x3F800000u) - 0.99999994f; }

// ---------------------------------------------------------------- [R7] lattice lookup
// (qa, qb, qc) measured from the panel's low corner.  Returns the material (-1 vacuum) and the packed ids without
// panel/photon/seq bits (kNone when the point is in no crystal).  PAPER.md:43: the depth coordinate picks the layer,
// that layer's crystal parameters give material and index.  Written without early exits: every lane of a pass runs the
// same instructions (a point outside the box just ends as vacuum).  `lay` = the layer records (the header's own array,
// or the kernel's copy in shared memory: lanes in different layers then read different rows without serialising).
__device__ __forceinline__ int lattice_lookup(const DevGeomHead &g, const DevLayer *lay, int qa, int qb, int qc, uint32_t &ids) {
  bool ok = (unsigned)qa < (unsigned)g.Wq && (unsigned)qb < (unsigned)g.Hq && (unsigned)qc < (unsigned)g.Dq;
  const int mx = (int)(__umulhi((uint32_t)qa, g.mp_magic[0]) >> g.mp_shift[0]), ra = qa - mx * g.mpq[0];
  const int my = (int)(__umulhi((uint32_t)qb, g.mp_magic[1]) >> g.mp_shift[1]), rb = qb - my * g.mpq[1];
  ok = ok && ra < g.msq[0] && rb < g.msq[1];                         // else inter-module gap: vacuum
  // layers are stacked front to back: the last one that starts at or before qc is the only candidate
  const int l = (qc >= g.layer[1].c0 ? 1 : 0) + (qc >= g.layer[2].c0 ? 1 : 0) + (qc >= g.layer[3].c0 ? 1 : 0);   // unused layers hold INT_MAX
  const int4 r0 = reinterpret_cast<const int4 *>(&lay[l])[0];        // c0, c1, cmat, gmat
  const int4 r1 = reinterpret_cast<const int4 *>(&lay[l])[1];        // n0 | shift0 << 24, n1 | shift1 << 24, pitch0, pitch1
  const int4 r2 = reinterpret_cast<const int4 *>(&lay[l])[2];        // lo0, lo1, hi0, hi1
  const int4 r3 = reinterpret_cast<const int4 *>(&lay[l])[3];        // off0, off1, magic0, magic1
  ok = ok && qc >= r0.x && qc < r0.y;                                // else inter-layer gap: vacuum
  const int ea = ra - r3.x, eb = rb - r3.y;                          // negative: in front of the lattice (rim)
  const int n0 = r1.x & 0xFFFFFF, n1 = r1.y & 0xFFFFFF;
  const int ix = (int)(__umulhi((uint32_t)ea, (uint32_t)r3.z) >> ((uint32_t)r1.x >> 24)), fa = ea - ix * r1.z;
  const int iy = (int)(__umulhi((uint32_t)eb, (uint32_t)r3.w) >> ((uint32_t)r1.y >> 24)), fb = eb - iy * r1.w;
  const bool in = (ea | eb) >= 0 && ix < n0 && iy < n1 && fa >= r2.x && fa < r2.z && fb >= r2.y && fb < r2.w;
  ids = ok && in ? ((uint32_t)(mx + g.nmod[0] * my) << 20) | ((uint32_t)l << 18) | ((uint32_t)(ix + n0 * iy) << 5) : kNone;
  return ok ? (in ? r0.z : r0.w) : -1;
}

// PAPER.md:33 global -> local
__device__ __forceinline__ void to_local(const float *P, const float x[3], const float d[3], float xl[3], float dl[3]) {
  const float r0 = x[0] - P[0], r1 = x[1] - P[1], r2 = x[2] - P[2];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    xl[k] = r0 * P[3 + 3 * k] + r1 * P[4 + 3 * k] + r2 * P[5 + 3 * k];
    dl[k] = d[0] * P[3 + 3 * k] + d[1] * P[4 + 3 * k] + d[2] * P[5 + 3 * k];
  }
}
__device__ __forceinline__ void point_to_global(const float *P, const float xl[3], float x[3]) {
#pragma unroll
  for (int k = 0; k < 3; ++k) x[k] = P[k] + xl[0] * P[3 + k] + xl[1] * P[6 + k] + xl[2] * P[9 + k];
}
__device__ __forceinline__ void dir_to_global(const float *P, const float dl[3], float d[3]) {
#pragma unroll
  for (int k = 0; k < 3; ++k) d[k] = dl[0] * P[3 + k] + dl[1] * P[6 + k] + dl[2] * P[9 + k];
}

// ---------------------------------------------------------------- [R21] rotation
__device__ __forceinline__ void rotate(float d[3], float ct, float st, float cp, float sp) {
  const float sg = copysignf(1.0f, d[2]), a = -1.0f / (sg + d[2]), b = d[0] * d[1] * a;
  const float b1x = 1.0f + sg * d[0] * d[0] * a, b1y = sg * b, b1z = -sg * d[0];
  const float b2x = b, b2y = sg + d[1] * d[1] * a, b2z = -d[1];
  const float nx = ct * d[0] + st * (cp * b1x + sp * b2x);
  const float ny = ct * d[1] + st * (cp * b1y + sp * b2y);
  const float nz = ct * d[2] + st * (cp * b1z + sp * b2z);
  const float s = rsqrtf(nx * nx + ny * ny + nz * nz);
  d[0] = nx * s; d[1] = ny * s; d[2] = nz * s;
}

// ---------------------------------------------------------------- [R23] outcome hash
enum : uint32_t { EV_ENTER = 1, EV_STEP_VACUUM, EV_VIRTUAL, EV_PE, EV_COMPTON, EV_RAYLEIGH, EV_CUTOFF, EV_EXIT, EV_ESCAPE,
                  EV_PH_COMPTON, EV_PH_RAYLEIGH, EV_PH_ABSORBED, EV_PH_CUTOFF, EV_PH_LEAVE, EV_REGION };
__device__ __forceinline__ void hash_ev(uint64_t &h, uint32_t type, uint32_t payload) {
  h = (h ^ (uint64_t)type) * 0x100000001B3ull;
  h = (h ^ (uint64_t)payload) * 0x100000001B3ull;
}

}  // namespace gpet
