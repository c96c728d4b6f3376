// gpet_api.cu -- the C ABI declared in include/gpet.h: argument checks, descriptor quantisation [R7],
// table staging [R11], activity CDF [R13], and kernel launches.  No physics runs on the host.
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <vector>

#include "../../include/gpet.h"
#include "gpet_internal.h"

using namespace gpet;

// ---------------------------------------------------------------- handles
struct gpet_geometry {
  DevGeom host;
  DevGeom *dev = nullptr;
};
struct gpet_materials {
  int n_materials = 0, n_energies = 0; float e_min = 0, e_step = 0;
  std::vector<float4> mu;               // host [n_materials][n_energies]: {mu_pe, mu_pe+mu_C, mu_tot, 0} [R11]
  std::mutex lock;
  std::map<uint32_t, float4 *> staged;  // device tables per (detector mask << 8 | staged mask), built lazily
};
struct gpet_activity {
  int dims[3]; uint32_t n_active = 0; uint64_t w_total = 0;
  uint32_t *dev_index = nullptr, *dev_guide = nullptr; uint64_t *dev_cdf = nullptr;
};

// ---------------------------------------------------------------- errors, bookkeeping
static thread_local char g_err[512] = "";
static std::atomic<uint64_t> g_launches{0};
void gpet::count_launch(uint64_t n) { g_launches += n; }

static int fail(int code, const char *fmt, ...) {
  va_list ap; va_start(ap, fmt); vsnprintf(g_err, sizeof g_err, fmt, ap); va_end(ap);
  return code;
}
#define CUDA_TRY(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) \
  return fail(GPET_E_CUDA, "%s: %s", #expr, cudaGetErrorString(e_)); } while (0)

extern "C" const char *gpet_last_error(void) { return g_err; }
extern "C" int gpet_decay_count(double activity_bq, double half_life_s, double duration_s, uint64_t *n_pairs) {
  if (!n_pairs || !(activity_bq > 0.0) || !(duration_s > 0.0) || half_life_s < 0.0) return fail(GPET_E_INVALID_ARG, "gpet_decay_count: bad argument");
  if (!(half_life_s > 0.0)) { *n_pairs = (uint64_t)llrint(activity_bq * duration_s); return GPET_OK; }
  const double lambda = 0.69314718055994530942 / half_life_s;
  *n_pairs = (uint64_t)llrint(activity_bq / lambda * -expm1(-lambda * duration_s)); return GPET_OK;
}
extern "C" uint64_t gpet_launch_count(void) { return g_launches.load(); }
extern "C" int gpet_set_transport_warps(int32_t warps) { set_transport_warps(warps); return transport_warps(); }

static int sm_count() {
  static int n = 0;
  if (!n) { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev); if (n <= 0) n = 148; }
  return n;
}

// ---------------------------------------------------------------- geometry
static long long quant(float x) { return llrint((double)x * 1048576.0); }   // [R7]
// the multiply-high division of the lattice lookup (QDiv) against plain division at every cell boundary below n_max
static bool qdiv_exact(uint32_t d, uint32_t n_max) {
  const QDiv q = qdiv_make(d);
  for (uint64_t k = 0; k * d <= (uint64_t)n_max + d; ++k)
    for (int64_t n = (int64_t)(k * d) - 1; n <= (int64_t)(k * d) + 1; ++n) {
      if (n < 0 || n > (int64_t)n_max) continue;
      if ((uint32_t)(((uint64_t)(uint32_t)n * q.magic) >> 32 >> q.shift) != (uint32_t)(n / d)) return false;
    }
  return true;
}

extern "C" int gpet_geometry_create(const gpet_geometry_desc *d, gpet_geometry **out) {
  if (!d || !out || !d->layers) return fail(GPET_E_INVALID_ARG, "gpet_geometry_create: NULL argument");
  if (d->n_panels < 1 || d->n_panels > GPET_MAX_PANELS) return fail(GPET_E_GEOMETRY, "n_panels %d outside 1..%d", d->n_panels, GPET_MAX_PANELS);
  if (d->n_layers < 1 || d->n_layers > GPET_MAX_LAYERS) return fail(GPET_E_GEOMETRY, "n_layers %d outside 1..%d", d->n_layers, GPET_MAX_LAYERS);
  gpet_geometry *g = new gpet_geometry;
  DevGeom &G = g->host; memset(&G, 0, sizeof G);
  G.n_panels = d->n_panels; G.n_layers = d->n_layers; G.ring = d->panel_pose ? 0 : 1;
  long long ms[2], mp[2];
  for (int a = 0; a < 2; ++a) {
    ms[a] = quant(d->module_size_mm[a]); mp[a] = quant(d->module_pitch_mm[a]);
    if (d->n_modules[a] < 1 || d->n_modules[a] > 8 || ms[a] < 2 || mp[a] < ms[a] || mp[a] >= (1ll << 30) || (long long)d->n_modules[a] * mp[a] >= (1ll << 30) ||
        !qdiv_exact((uint32_t)mp[a], (uint32_t)(d->n_modules[a] * mp[a]))) {
      delete g; return fail(GPET_E_GEOMETRY, "module grid axis %d: n=%d size=%g pitch=%g", a, d->n_modules[a], d->module_size_mm[a], d->module_pitch_mm[a]);
    }
    G.nmod[a] = d->n_modules[a]; G.msq[a] = (int)ms[a]; G.mpq[a] = (int)mp[a]; { const QDiv qd = qdiv_make((uint32_t)mp[a]); G.mp_magic[a] = qd.magic; G.mp_shift[a] = qd.shift; }
  }
  const long long Wq = (G.nmod[0] - 1) * mp[0] + ms[0], Hq = (G.nmod[1] - 1) * mp[1] + ms[1];
  long long c = 0;
  for (int l = 0; l < d->n_layers; ++l) {
    const gpet_layer_desc &s = d->layers[l]; DevLayer &L = G.layer[l];
    const long long gb = quant(s.gap_before_mm), dp = quant(s.depth_mm);
    if (gb < 0 || dp <= 0) { delete g; return fail(GPET_E_GEOMETRY, "layer %d: depth %g, gap_before %g", l, s.depth_mm, s.gap_before_mm); }
    c += gb; L.c0 = (int)c; c += dp; L.c1 = (int)c;
    L.cmat = s.crystal_material; L.gmat = s.gap_material;
    if (L.cmat < 0 || L.cmat >= GPET_MAX_MATERIALS || L.gmat < -1 || L.gmat >= GPET_MAX_MATERIALS) {
      delete g; return fail(GPET_E_GEOMETRY, "layer %d: material index out of range", l);
    }
    G.det_mask |= 1u << L.cmat; if (L.gmat >= 0) G.det_mask |= 1u << L.gmat;
    for (int a = 0; a < 2; ++a) {
      const long long p = quant(s.pitch_mm[a]), gp = quant(s.reflector_mm[a]), of = quant(s.offset_mm[a]);
      if (s.n_crystals[a] < 1 || p < 2 || p >= (1ll << 30) || !qdiv_exact((uint32_t)p, (uint32_t)ms[a]) || gp < 0 || gp >= p || of < 0 || of + s.n_crystals[a] * p > ms[a]) {
        delete g; return fail(GPET_E_GEOMETRY, "layer %d axis %d: lattice (n=%d pitch=%g gap=%g offset=%g) does not fit its %g mm module",
                              l, a, s.n_crystals[a], s.pitch_mm[a], s.reflector_mm[a], s.offset_mm[a], d->module_size_mm[a]);
      }
      L.n[a] = s.n_crystals[a]; L.pitch[a] = (int)p; L.off[a] = (int)of;
      L.lo[a] = (int)(gp >> 1); L.hi[a] = (int)(p - (gp - (gp >> 1))); { const QDiv qd = qdiv_make((uint32_t)p); L.magic[a] = qd.magic; L.n[a] |= (int)(qd.shift << 24); }
    }
    if ((long long)s.n_crystals[0] * s.n_crystals[1] > 8192) { delete g; return fail(GPET_E_GEOMETRY, "layer %d: more than 8192 crystals", l); }
  }
  for (int l = d->n_layers; l < kMaxLayers; ++l) G.layer[l].c0 = G.layer[l].c1 = 0x7FFFFFFF;        // never selected by the depth compare
  // [R19] majorant regions: maximal runs of consecutive layers with the same crystal and gap material; the gap in front of
  // a region's first layer belongs to the region before it
  G.n_regions = 0;
  for (int l = 0; l < kMaxLayers; ++l) { G.reg_lo[l] = INFINITY; G.reg_hi[l] = INFINITY; G.reg_mats[l] = 0; }
  for (int l = 0; l < d->n_layers; ++l) {
    if (l == 0 || G.layer[l].cmat != G.layer[l - 1].cmat || G.layer[l].gmat != G.layer[l - 1].gmat) {
      G.reg_lo[G.n_regions] = l == 0 ? 0.0f : (float)((double)G.layer[l].c0 / 1048576.0);
      if (G.n_regions) G.reg_hi[G.n_regions - 1] = G.reg_lo[G.n_regions];
      G.reg_mats[G.n_regions] = (uint32_t)G.layer[l].cmat | (uint32_t)(G.layer[l].gmat >= 0 ? G.layer[l].gmat : G.layer[l].cmat) << 4;
      ++G.n_regions;
    }
  }
  G.reg_hi[G.n_regions - 1] = (float)((double)c / 1048576.0);
  if (Wq >= (1ll << 30) || Hq >= (1ll << 30) || c >= (1ll << 30)) { delete g; return fail(GPET_E_GEOMETRY, "panel larger than 1024 mm"); }
  G.Wq = (int)Wq; G.Hq = (int)Hq; G.Dq = (int)c; G.hWq = (int)(Wq >> 1); G.hHq = (int)(Hq >> 1);
  G.blo[0] = (float)(-(double)G.hWq / 1048576.0); G.bhi[0] = (float)((double)(Wq - G.hWq) / 1048576.0);
  G.blo[1] = (float)(-(double)G.hHq / 1048576.0); G.bhi[1] = (float)((double)(Hq - G.hHq) / 1048576.0);
  G.blo[2] = 0.0f;                                G.bhi[2] = (float)((double)c / 1048576.0);
  if (d->panel_pose) {
    for (int p = 0; p < d->n_panels; ++p) {
      const float *q = d->panel_pose + 12 * p;                        // u, v, w must be an orthonormal right-handed frame (u x v = w)
      const double u[3] = { q[3], q[4], q[5] }, v[3] = { q[6], q[7], q[8] }, w[3] = { q[9], q[10], q[11] };
      const double cr[3] = { u[1] * v[2] - u[2] * v[1], u[2] * v[0] - u[0] * v[2], u[0] * v[1] - u[1] * v[0] };
      double err = 0.0;
      for (int k = 0; k < 3; ++k) err = fmax(err, fabs(cr[k] - w[k]));
      err = fmax(err, fabs(u[0] * u[0] + u[1] * u[1] + u[2] * u[2] - 1.0)); err = fmax(err, fabs(v[0] * v[0] + v[1] * v[1] + v[2] * v[2] - 1.0));
      err = fmax(err, fabs(u[0] * v[0] + u[1] * v[1] + u[2] * v[2]));
      bool finite = true; for (int k = 0; k < 12; ++k) finite = finite && std::isfinite(q[k]);
      if (!finite || !(err < 1e-5)) { delete g; return fail(GPET_E_GEOMETRY, "panel %d: pose axes are not an orthonormal right-handed frame (u x v = w) to 1e-5", p); }
      memcpy(G.panel[p].pose, q, sizeof(float) * 12);
    }
  } else {                                                          // [R5] repetition mode
    const double PI = 3.14159265358979323846;
    for (int p = 0; p < d->n_panels; ++p) {
      const double phi = ((double)d->ring_first_angle_deg + 360.0 * (double)p / (double)d->n_panels) * (PI / 180.0);
      double cs = cos(phi), sn = sin(phi);
      if (fabs(cs) < 1e-12) cs = 0.0;
      if (fabs(sn) < 1e-12) sn = 0.0;
      float *q = G.panel[p].pose;
      q[0] = (float)((double)d->ring_inner_radius_mm * cs); q[1] = (float)((double)d->ring_inner_radius_mm * sn); q[2] = 0.0f;
      q[3] = (float)(-sn); q[4] = (float)cs; q[5] = 0.0f;
      q[6] = 0.0f; q[7] = 0.0f; q[8] = 1.0f;
      q[9] = (float)cs; q[10] = (float)sn; q[11] = 0.0f;
    }
  }
  G.planar = 1;                 // axial axis = +z everywhere and no z component elsewhere (any repetition-mode ring)
  for (int p = 0; p < G.n_panels; ++p) {
    const float *q = G.panel[p].pose;
    if (q[2] != 0.0f || q[5] != 0.0f || q[11] != 0.0f || q[6] != 0.0f || q[7] != 0.0f || q[8] != 1.0f) G.planar = 0;
  }
  // bounding circle (planar search: tangential x depth) and sphere of the panel box, 0.01 % + 1 um margin: the search
  // only culls panels whose bound the ray misses, so the surviving tests decide exactly as the full loop [R6]
  {
    const double ha = 0.5 * ((double)G.bhi[0] - G.blo[0]), hb = 0.5 * ((double)G.bhi[1] - G.blo[1]), hc = 0.5 * ((double)G.bhi[2] - G.blo[2]);
    const double ma = 0.5 * ((double)G.bhi[0] + G.blo[0]), mb = 0.5 * ((double)G.bhi[1] + G.blo[1]), mc = 0.5 * ((double)G.bhi[2] + G.blo[2]);
    G.cull_r2 = (float)(sqrt(ha * ha + hc * hc) * 1.0001 + 1e-3);
    G.cull_r3 = (float)(sqrt(ha * ha + hb * hb + hc * hc) * 1.0001 + 1e-3);
    for (int p = 0; p < G.n_panels; ++p) {
      const float *q = G.panel[p].pose; float c[3];
      for (int k = 0; k < 3; ++k) c[k] = (float)((double)q[k] + ma * q[3 + k] + mb * q[6 + k] + mc * q[9 + k]);
      G.panel[p].cx = c[0]; G.panel[p].cy = c[1]; G.panel[p].cz = c[2];
      G.ctr[p][0] = c[0]; G.ctr[p][1] = c[1]; G.ctr[p][2] = c[2];
    }
  }
  // bore radius of a planar detector: the smallest distance from the z axis to any panel box (exact point-to-rectangle
  // distance in each panel's (tangential, depth) frame, minus 1 um).  A photon inside the bore that passes the axial
  // ends of the detector before it can reach this radius meets no panel: transport drops it without a search.
  G.bore_r = -1.0f;
  if (G.planar) {
    double rmin = 1e300;
    for (int p = 0; p < G.n_panels; ++p) {
      const float *q = G.panel[p].pose;
      const double a = -((double)q[0] * q[3] + (double)q[1] * q[4]), c = -((double)q[0] * q[9] + (double)q[1] * q[10]);   // axis point in the panel frame
      const double da = a < G.blo[0] ? G.blo[0] - a : (a > G.bhi[0] ? a - G.bhi[0] : 0.0);
      const double dc = c < G.blo[2] ? G.blo[2] - c : (c > G.bhi[2] ? c - G.bhi[2] : 0.0);
      rmin = fmin(rmin, sqrt(da * da + dc * dc));
    }
    if (rmin > 2e-3) G.bore_r = (float)(rmin - 1e-3);
  }
  // Repetition-mode ring: the front faces lie on a regular polygon of apothem R about the z axis; a photon inside the
  // inscribed circle enters the panel whose edge it crosses (ring_entry_fast).  Half edge length R tan(pi/n), minus 1 um
  // so that rays through a vertex -- where two overlapping panels tie -- take the full search and its lowest-index rule.
  G.ring_phi0 = 0.0f; G.ring_kscale = 0.0f; G.ring_edge_h = -1.0f;
  if (G.ring && G.planar && G.n_panels >= 3 && G.bore_r > 0.0f && d->ring_inner_radius_mm > 0.0f) {
    const double PI = 3.14159265358979323846;
    G.ring_phi0 = (float)remainder((double)d->ring_first_angle_deg * (PI / 180.0), 2.0 * PI);   // in [-pi, pi]: the sector index wraps at most once
    G.ring_kscale = (float)((double)G.n_panels / (2.0 * PI));
    G.ring_edge_h = (float)((double)d->ring_inner_radius_mm * tan(PI / (double)G.n_panels) - 1e-3);
  }
  // open faces: face (axis k, side) of panel p is open when every corner of every other panel box lies at least 1 um on
  // the inner side of that face's plane -- a photon leaving p through it can meet no other panel (transport skips the
  // search of [R6] then; the result is the one the search would give).  Rings: back and axial faces are open.
  {
    const double lo[3] = { G.blo[0], G.blo[1], G.blo[2] }, hi[3] = { G.bhi[0], G.bhi[1], G.bhi[2] };
    for (int p = 0; p < G.n_panels; ++p) {
      const float *P = G.panel[p].pose; uint32_t open = 63u;
      for (int q = 0; q < G.n_panels; ++q) if (q != p) {
        const float *Q = G.panel[q].pose;
        for (int c = 0; c < 8; ++c) {
          const double a = c & 1 ? hi[0] : lo[0], b = c & 2 ? hi[1] : lo[1], w = c & 4 ? hi[2] : lo[2];
          double x[3], l[3];
          for (int k = 0; k < 3; ++k) x[k] = (double)Q[k] + a * Q[3 + k] + b * Q[6 + k] + w * Q[9 + k] - (double)P[k];
          for (int k = 0; k < 3; ++k) l[k] = x[0] * P[3 + 3 * k] + x[1] * P[4 + 3 * k] + x[2] * P[5 + 3 * k];
          for (int k = 0; k < 3; ++k) {
            if (!(l[k] < hi[k] - 1e-3)) open &= ~(1u << (2 * k + 1));
            if (!(l[k] > lo[k] + 1e-3)) open &= ~(1u << (2 * k));
          }
        }
      }
      G.panel[p].open_faces = open;
    }
  }
  *out = g;                     // the device copy is made lazily so the handle can be built without a GPU
  return GPET_OK;
}

static int geometry_upload(gpet_geometry *g) {
  if (g->dev) return GPET_OK;
  CUDA_TRY(cudaMalloc(&g->dev, sizeof(DevGeom)));
  CUDA_TRY(cudaMemcpy(g->dev, &g->host, sizeof(DevGeom), cudaMemcpyHostToDevice));
  return GPET_OK;
}

extern "C" int gpet_geometry_destroy(gpet_geometry *g) {
  if (!g) return GPET_OK;
  if (g->dev) cudaFree(g->dev);
  delete g; return GPET_OK;
}

extern "C" int gpet_geometry_panel_pose(const gpet_geometry *g, int32_t panel, float *pose12) {
  if (!g || !pose12 || panel < 0 || panel >= g->host.n_panels) return fail(GPET_E_INVALID_ARG, "gpet_geometry_panel_pose: bad argument");
  memcpy(pose12, g->host.panel[panel].pose, sizeof(float) * 12); return GPET_OK;
}

extern "C" int gpet_geometry_open_faces(const gpet_geometry *g, int32_t panel, uint32_t *mask) {
  if (!g || !mask || panel < 0 || panel >= g->host.n_panels) return fail(GPET_E_INVALID_ARG, "gpet_geometry_open_faces: bad argument");
  *mask = g->host.panel[panel].open_faces; return GPET_OK;
}

extern "C" int gpet_geometry_bore_radius(const gpet_geometry *g, float *radius_mm) {
  if (!g || !radius_mm) return fail(GPET_E_INVALID_ARG, "gpet_geometry_bore_radius: NULL argument");
  *radius_mm = g->host.bore_r; return GPET_OK;
}

extern "C" int gpet_geometry_locate(const gpet_geometry *g, int64_t n, const float *xyz, uint32_t *ids) {
  if (!g || n < 0 || (n > 0 && (!xyz || !ids))) return fail(GPET_E_INVALID_ARG, "gpet_geometry_locate: bad argument");
  if (n == 0) return GPET_OK;
  int rc = geometry_upload(const_cast<gpet_geometry *>(g)); if (rc) return rc;
  float *dx = nullptr; uint32_t *di = nullptr;
  cudaError_t e = cudaMalloc(&dx, sizeof(float) * 3 * (size_t)n);
  if (e == cudaSuccess) e = cudaMalloc(&di, sizeof(uint32_t) * (size_t)n);
  if (e == cudaSuccess) e = cudaMemcpy(dx, xyz, sizeof(float) * 3 * (size_t)n, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = launch_locate(g->dev, n, dx, di, 0);
  if (e == cudaSuccess) e = cudaMemcpy(ids, di, sizeof(uint32_t) * (size_t)n, cudaMemcpyDeviceToHost);
  cudaFree(dx); cudaFree(di);                                        // also on the error paths
  if (e != cudaSuccess) return fail(GPET_E_CUDA, "gpet_geometry_locate: %s", cudaGetErrorString(e));
  return GPET_OK;
}

// ---------------------------------------------------------------- materials
extern "C" int gpet_materials_load(int32_t n_materials, int32_t n_energies, float e_min, float e_step, const float *mu_pe,
                                   const float *mu_c, const float *mu_r, gpet_materials **out) {
  if (!mu_pe || !mu_c || !mu_r || !out) return fail(GPET_E_INVALID_ARG, "gpet_materials_load: NULL argument");
  if (n_materials < 1 || n_materials > GPET_MAX_MATERIALS) return fail(GPET_E_TABLE, "n_materials %d outside 1..%d", n_materials, GPET_MAX_MATERIALS);
  if (n_energies < 2 || !(e_step > 0.0f)) return fail(GPET_E_TABLE, "need >= 2 energies and a positive step");
  const size_t n = (size_t)n_materials * n_energies;
  gpet_materials *m = new gpet_materials;
  m->n_materials = n_materials; m->n_energies = n_energies; m->e_min = e_min; m->e_step = e_step; m->mu.resize(n);
  for (size_t i = 0; i < n; ++i) {
    if (!(mu_pe[i] >= 0.0f) || !(mu_c[i] >= 0.0f) || !(mu_r[i] >= 0.0f) || !std::isfinite(mu_pe[i] + mu_c[i] + mu_r[i])) {
      delete m; return fail(GPET_E_TABLE, "negative or non-finite mu at flat index %zu", i);
    }
    // cumulative sums formed in double, rounded to fp32 once [R11]
    m->mu[i] = make_float4(mu_pe[i], (float)((double)mu_pe[i] + mu_c[i]), (float)((double)mu_pe[i] + mu_c[i] + mu_r[i]), 0.0f);
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { delete m; return fail(GPET_E_CUDA, "gpet_materials_load: no CUDA device"); }
  *out = m; return GPET_OK;
}

extern "C" int gpet_materials_destroy(gpet_materials *m) {
  if (!m) return GPET_OK;
  for (auto &kv : m->staged) if (kv.second) cudaFree(kv.second);
  delete m; return GPET_OK;
}

// Device table for one run: the materials in `stage_mask`, interleaved float4 per energy with the detector
// majorant [R19] (pointwise max of mu_tot over `det_mask`) in .w; `matmap` gives each material's staged slot.
static int staged_table(gpet_materials *m, uint32_t det_mask, uint32_t stage_mask, DevTables *T) {
  const uint32_t all = (1u << m->n_materials) - 1u;
  det_mask &= all; stage_mask = (stage_mask | det_mask) & all;
  if (!det_mask) return fail(GPET_E_INVALID_ARG, "geometry references no loaded material");
  T->n_energies = m->n_energies; T->e_min = m->e_min; T->inv_step = 1.0f / m->e_step; T->matmap = 0; T->n_staged = 0;
  for (int k = 0; k < m->n_materials; ++k) if (stage_mask >> k & 1u) T->matmap |= (uint32_t)(T->n_staged++) << (4 * k);
  std::lock_guard<std::mutex> lk(m->lock);
  float4 *&dev = m->staged[det_mask << 8 | stage_mask];
  if (!dev) {
    const int ne = m->n_energies;
    std::vector<float4> tab((size_t)T->n_staged * ne);
    int slot = 0;
    for (int k = 0; k < m->n_materials; ++k) if (stage_mask >> k & 1u) {
      for (int i = 0; i < ne; ++i) {
        float4 v = m->mu[(size_t)k * ne + i]; v.w = 0.0f;
        for (int q = 0; q < m->n_materials; ++q) if (det_mask >> q & 1u) v.w = fmaxf(v.w, m->mu[(size_t)q * ne + i].z);
        tab[(size_t)slot * ne + i] = v;
      }
      ++slot;
    }
    CUDA_TRY(cudaMalloc(&dev, sizeof(float4) * tab.size()));
    CUDA_TRY(cudaMemcpy(dev, tab.data(), sizeof(float4) * tab.size(), cudaMemcpyHostToDevice));
  }
  T->mu = dev; return GPET_OK;
}

// ---------------------------------------------------------------- activity map [R13]
extern "C" int gpet_activity_create(const float *activity, const int32_t dims[3], gpet_activity **out) {
  if (!activity || !dims || !out) return fail(GPET_E_INVALID_ARG, "gpet_activity_create: NULL argument");
  if (dims[0] < 1 || dims[1] < 1 || dims[2] < 1 || (long long)dims[0] * dims[1] * dims[2] > (1ll << 31))
    return fail(GPET_E_INVALID_ARG, "activity grid %d x %d x %d out of range", dims[0], dims[1], dims[2]);
  const size_t nv = (size_t)dims[0] * dims[1] * dims[2];
  float amax = 0.0f;
  for (size_t i = 0; i < nv; ++i) { if (!(activity[i] >= 0.0f)) return fail(GPET_E_INVALID_ARG, "negative activity"); if (activity[i] > amax) amax = activity[i]; }
  if (!(amax > 0.0f)) return fail(GPET_E_INVALID_ARG, "activity map has no active voxel");
  std::vector<uint32_t> idx; std::vector<uint64_t> cdf; uint64_t cum = 0;
  for (size_t i = 0; i < nv; ++i) if (activity[i] > 0.0f) {
    long long w = llrint((double)activity[i] / (double)amax * 1048576.0); if (w < 1) w = 1;
    cum += (uint64_t)w; idx.push_back((uint32_t)i); cdf.push_back(cum);
  }
  gpet_activity *a = new gpet_activity;
  a->dims[0] = dims[0]; a->dims[1] = dims[1]; a->dims[2] = dims[2]; a->n_active = (uint32_t)idx.size(); a->w_total = cum;
  cudaError_t e = cudaMalloc(&a->dev_index, sizeof(uint32_t) * idx.size());
  if (e == cudaSuccess) e = cudaMalloc(&a->dev_cdf, sizeof(uint64_t) * cdf.size());
  if (e == cudaSuccess) e = cudaMemcpy(a->dev_index, idx.data(), sizeof(uint32_t) * idx.size(), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(a->dev_cdf, cdf.data(), sizeof(uint64_t) * cdf.size(), cudaMemcpyHostToDevice);
  // Guide table for the cdf search [R13]: guide[b] = the voxel the SMALLEST target of bucket b selects, bucket = the top
  // kActGuideBits bits of the voxel-pick word (target = floor(word W / 2^32) is monotonic in the word).  The voxel of any
  // word of bucket b then lies in [guide[b], guide[b + 1]]: the search starts from a handful of entries, not from all.
  std::vector<uint32_t> guide((size_t)kActGuide + 1);
  {
    size_t v = 0;
    const uint64_t Wl = cum & 0xFFFFFFFFull, Wh = cum >> 32;
    for (uint32_t b = 0; b < kActGuide; ++b) {
      const uint64_t word = (uint64_t)b << (32 - kActGuideBits);
      const uint64_t target = word * Wh + ((word * Wl) >> 32);          // floor(word W / 2^32), as the kernel forms it
      while (cdf[v] <= target) ++v;                                     // first voxel with cum > target
      guide[b] = (uint32_t)v;
    }
    guide[kActGuide] = (uint32_t)(idx.size() - 1);
  }
  if (e == cudaSuccess) e = cudaMalloc(&a->dev_guide, sizeof(uint32_t) * guide.size());
  if (e == cudaSuccess) e = cudaMemcpy(a->dev_guide, guide.data(), sizeof(uint32_t) * guide.size(), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) { gpet_activity_destroy(a); return fail(GPET_E_CUDA, "gpet_activity_create: %s", cudaGetErrorString(e)); }
  *out = a; return GPET_OK;
}

extern "C" int gpet_activity_destroy(gpet_activity *a) {
  if (!a) return GPET_OK;
  if (a->dev_index) cudaFree(a->dev_index);
  if (a->dev_cdf) cudaFree(a->dev_cdf);
  if (a->dev_guide) cudaFree(a->dev_guide);
  delete a; return GPET_OK;
}

// ---------------------------------------------------------------- source marshalling
static int make_source(const gpet_source *s, const gpet_materials *m, DevSource *D) {
  memset(D, 0, sizeof *D);
  if (s->kind < 0 || s->kind > 2) return fail(GPET_E_INVALID_ARG, "source kind %d", s->kind);
  D->kind = s->kind;
  for (int k = 0; k < 3; ++k) { D->pos[k] = s->pos_mm[k]; D->dims[k] = s->dims[k]; D->voxel[k] = s->voxel_mm[k]; D->origin[k] = s->origin_mm[k];
                                D->inv_voxel[k] = s->voxel_mm[k] > 0.0f ? 1.0f / s->voxel_mm[k] : 0.0f; }
  if (s->kind == 2) {
    const double nb = sqrt((double)s->beam_dir[0] * s->beam_dir[0] + (double)s->beam_dir[1] * s->beam_dir[1] + (double)s->beam_dir[2] * s->beam_dir[2]);
    if (!(nb > 0.0)) return fail(GPET_E_INVALID_ARG, "beam_dir is zero");
    for (int k = 0; k < 3; ++k) D->beam[k] = (float)((double)s->beam_dir[k] / nb);
  }
  if (!(s->acolinearity_fwhm_deg >= 0.0f)) return fail(GPET_E_INVALID_ARG, "negative acolinearity");
  D->acol_sigma = (float)((double)s->acolinearity_fwhm_deg * (3.14159265358979323846 / 180.0) / 2.354820045030949);
  {  // largest polar deviation photon B can draw [R15, R2]: sigma sqrt(-2 ln u_min), u_min = 2^-24; + 1 % for the fp32 evaluation
    const double rho = fmin((double)D->acol_sigma * sqrt(2.0 * 24.0 * log(2.0)) * 1.01, 1.5);
    D->acol_sin_max = (float)sin(rho); D->acol_cos_max = (float)cos(rho);
  }
  if (!(s->activity_bq > 0.0)) return fail(GPET_E_INVALID_ARG, "activity_bq must be positive");
  D->activity_bq = s->activity_bq; D->pairs_per_slice = s->pairs_per_time_slice;
  if (!(s->positron_fwhm_mm >= 0.0f)) return fail(GPET_E_INVALID_ARG, "negative positron range");
  D->positron_sigma = (float)((double)s->positron_fwhm_mm / 2.354820045030949);
  if (s->kind == 1) {
    if (!s->activity_map) return fail(GPET_E_INVALID_ARG, "kind 1 needs an activity_map");
    for (int k = 0; k < 3; ++k) if (s->dims[k] != s->activity_map->dims[k] || !(s->voxel_mm[k] > 0.0f))
      return fail(GPET_E_INVALID_ARG, "source grid does not match its activity map");
    D->act_index = s->activity_map->dev_index; D->act_cdf = s->activity_map->dev_cdf; D->act_guide = s->activity_map->dev_guide;
    D->n_active = s->activity_map->n_active; D->w_total = s->activity_map->w_total;
    const uint32_t nx = (uint32_t)s->dims[0], nxy = nx * (uint32_t)s->dims[1];
    QDiv one; one.magic = 0u; one.shift = 0u;
    D->div_nx = nx >= 2u ? qdiv_make(nx) : one; D->div_nxy = nxy >= 2u ? qdiv_make(nxy) : one;
    D->phantom = s->phantom_material; D->ph_major = s->phantom_majorant_material;
    if (D->phantom && m && (D->ph_major < 0 || D->ph_major >= m->n_materials)) return fail(GPET_E_INVALID_ARG, "phantom_majorant_material out of range");
  }
  return GPET_OK;
}

// n_pairs = pairs of the batch the buffer holds (chunked layout: fixes the number of chunks and the region size)
static int hitbuf(const gpet_hits *h, uint64_t n_pairs, HitBuf *out) {
  HitBuf H = { h->history, h->ids, h->x, h->y, h->z, h->e_keV, h->tof_ns, h->capacity, reinterpret_cast<unsigned long long *>(h->n_hits),
               nullptr, 0u, 0u };
  if (h->chunk_fill) {
    const uint64_t nc = (n_pairs + kHitChunkPairs - 1) / kHitChunkPairs;
    const uint64_t cap = nc ? h->capacity / nc : 0;
    if (cap < 1 || cap > kHitChunkCapMax) return fail(GPET_E_INVALID_ARG, "chunked hit buffer: capacity / n_chunks = %llu outside 1..%u",
                                                      (unsigned long long)cap, kHitChunkCapMax);
    H.chunk_fill = h->chunk_fill; H.chunk_cap = (uint32_t)cap; H.n_chunks = (uint32_t)nc;
  }
  *out = H; return GPET_OK;
}

// ---------------------------------------------------------------- transport
// Work counters of the persistent kernel: a ring of 64 device words, one per launch in flight.  Each slot carries an event
// recorded behind the launch that used it; before a slot is handed out again the host waits for that event, so a 65th
// launch in flight waits for the oldest one instead of sharing its counter.
namespace {
struct WorkRing {
  std::mutex lock; unsigned long long *words = nullptr; cudaEvent_t ev[64]; bool used[64]; unsigned next = 0;
};
WorkRing g_ring;
}
static int next_work_counter(unsigned long long **out, unsigned *slot) {
  std::lock_guard<std::mutex> lk(g_ring.lock);
  if (!g_ring.words) {
    CUDA_TRY(cudaMalloc(&g_ring.words, 64 * sizeof(unsigned long long)));
    for (int i = 0; i < 64; ++i) { CUDA_TRY(cudaEventCreateWithFlags(&g_ring.ev[i], cudaEventDisableTiming)); g_ring.used[i] = false; }
  }
  const unsigned s = g_ring.next++ & 63u;
  if (g_ring.used[s]) CUDA_TRY(cudaEventSynchronize(g_ring.ev[s]));
  *out = g_ring.words + s; *slot = s; return GPET_OK;
}
static int work_counter_launched(unsigned slot, cudaStream_t stream) {
  std::lock_guard<std::mutex> lk(g_ring.lock);
  CUDA_TRY(cudaEventRecord(g_ring.ev[slot], stream));
  g_ring.used[slot] = true; return GPET_OK;
}
static void work_ring_release() {
  std::lock_guard<std::mutex> lk(g_ring.lock);
  if (!g_ring.words) return;
  for (int i = 0; i < 64; ++i) {                                      // a persistent kernel still in flight counts on its word: wait for it
    if (g_ring.used[i]) cudaEventSynchronize(g_ring.ev[i]);
    cudaEventDestroy(g_ring.ev[i]); g_ring.used[i] = false;
  }
  cudaFree(g_ring.words); g_ring.words = nullptr; g_ring.next = 0;
}

static size_t smem_limit() {
  static size_t lim = 0;
  if (!lim) { int dev = 0, v = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev); lim = v > 0 ? (size_t)v : 48 * 1024; }
  return lim;
}

extern "C" int gpet_simulate(const gpet_geometry *g, const gpet_materials *m, const gpet_source *src, uint64_t first_history,
                             uint64_t n_pairs, uint64_t seed, gpet_hits *hits, void *stream) {
  if (!g || !m || !src || !hits) return fail(GPET_E_INVALID_ARG, "gpet_simulate: NULL argument");
  if (!hits->n_hits || (hits->capacity && (!hits->history || !hits->ids || !hits->x || !hits->y || !hits->z || !hits->e_keV || !hits->tof_ns)))
    return fail(GPET_E_INVALID_ARG, "gpet_simulate: hit buffer has NULL arrays");
  if (n_pairs >= (1ull << 32)) return fail(GPET_E_INVALID_ARG, "n_pairs >= 2^32");
  if (n_pairs == 0) return GPET_OK;
  for (int l = 0; l < g->host.n_layers; ++l)
    if (g->host.layer[l].cmat >= m->n_materials || g->host.layer[l].gmat >= m->n_materials)
      return fail(GPET_E_INVALID_ARG, "layer %d references a material that is not loaded", l);
  DevSource D; int rc = make_source(src, m, &D); if (rc) return rc;
  rc = geometry_upload(const_cast<gpet_geometry *>(g)); if (rc) return rc;
  // a phantom may hold any loaded material (its map lives on the device): stage them all in that case
  const uint32_t stage_mask = (D.kind == 1 && D.phantom) ? (1u << m->n_materials) - 1u : 0u;
  DevTables T; rc = staged_table(const_cast<gpet_materials *>(m), g->host.det_mask, stage_mask, &T); if (rc) return rc;
  HitBuf HB; rc = hitbuf(hits, n_pairs, &HB); if (rc) return rc;
  // per-warp pools + staged tables + panel records share the CTA's shared memory: with many materials or a fine energy
  // grid the CTA runs with fewer warps; if not even 4 warps fit, say so instead of failing in the launch
  const int warps = transport_warps_that_fit(g->host, T, D, hits->outcome_hash != nullptr, smem_limit());
  if (!warps) return fail(GPET_E_TABLE, "mu tables too large for shared memory: %d staged materials x %d energies x 16 B next to the photon pools "
                          "(limit %zu B per CTA); load fewer materials or a coarser energy grid", T.n_staged, T.n_energies, smem_limit());
  unsigned long long *wc = nullptr; unsigned slot = 0; rc = next_work_counter(&wc, &slot); if (rc) return rc;
  CUDA_TRY(launch_transport(g->host, g->dev, T, D, first_history, n_pairs, seed, HB, hits->outcome_hash, wc, sm_count(), warps, (cudaStream_t)stream));
  return work_counter_launched(slot, (cudaStream_t)stream);
}

// ---------------------------------------------------------------- digitizer
extern "C" size_t gpet_digitize_scratch_bytes(uint64_t n_pairs, uint64_t n_hits) { return digitize_scratch_bytes(n_pairs, n_hits); }

static int make_digi(const gpet_source *src, uint64_t seed, uint64_t n_pairs_total, const gpet_digitizer *d, DigiParams *P) {
  if (d->readout_level < 0 || d->readout_level > 2) return fail(GPET_E_INVALID_ARG, "readout_level %d", d->readout_level);
  if (!(d->blur_fwhm_frac >= 0.0f) || !(d->window_ns > 0.0) || !(src->activity_bq > 0.0)) return fail(GPET_E_INVALID_ARG, "bad digitizer parameters");
  if (n_pairs_total == 0) return fail(GPET_E_INVALID_ARG, "n_pairs_total must be positive (it sets the time-slice length [R16])");
  P->sigma_scale = (float)((double)d->blur_fwhm_frac / 2.354820045030949); P->ref_keV = d->blur_ref_keV;
  P->e_lo = d->e_lo_keV; P->e_hi = d->e_hi_keV; P->window_s = d->window_ns * 1e-9;
  P->shift = d->readout_level == 0 ? 5 : (d->readout_level == 1 ? 20 : 26);
  P->activity_bq = src->activity_bq; P->pairs_per_slice = src->pairs_per_time_slice ? src->pairs_per_time_slice : n_pairs_total;
  P->seed = seed; P->slice_s = (double)P->pairs_per_slice / P->activity_bq; P->n_pairs_total = n_pairs_total;
  for (int r = 0; r < 10; ++r) { P->keys.k[2 * r] = (uint32_t)seed + (uint32_t)r * 0x9E3779B9u; P->keys.k[2 * r + 1] = (uint32_t)(seed >> 32) + (uint32_t)r * 0xBB67AE85u; }
  P->lambda = 0.0; P->pfrac = 0.0; P->q_scale = (double)P->pairs_per_slice / (double)n_pairs_total;
  P->cut_slice = ~0ull; P->cut_frac = 1.0;
  if (n_pairs_total % P->pairs_per_slice != 0) { P->cut_slice = n_pairs_total / P->pairs_per_slice; P->cut_frac = (double)(n_pairs_total % P->pairs_per_slice) / (double)P->pairs_per_slice; }
  if (src->half_life_s > 0.0) {                                      // [R34] decay law
    if (!(src->duration_s > 0.0)) return fail(GPET_E_INVALID_ARG, "half_life_s > 0 needs duration_s > 0");
    P->lambda = 0.69314718055994530942 / src->half_life_s; P->pfrac = -expm1(-P->lambda * src->duration_s);
  } else if (src->half_life_s < 0.0) return fail(GPET_E_INVALID_ARG, "negative half-life");
  return GPET_OK;
}

extern "C" int gpet_digitize(const gpet_source *src, uint64_t seed, uint64_t n_pairs_total, uint64_t first_history, uint64_t n_pairs,
                             const gpet_hits *hits, uint64_t n_hits, const gpet_digitizer *dig, void *scratch, size_t scratch_bytes,
                             gpet_singles *so, gpet_coincidences *co, void *stream) {
  if (!src || !hits || !dig || !co || !co->n_coinc) return fail(GPET_E_INVALID_ARG, "gpet_digitize: NULL argument");
  if (n_pairs == 0 || n_pairs >= (1ull << 32) || n_hits > hits->capacity || n_hits > (1ull << 31)) return fail(GPET_E_INVALID_ARG, "gpet_digitize: counts out of range");
  if (n_pairs_total < n_pairs) return fail(GPET_E_INVALID_ARG, "gpet_digitize: n_pairs_total %llu < n_pairs %llu", (unsigned long long)n_pairs_total, (unsigned long long)n_pairs);
  if (scratch_bytes < digitize_scratch_bytes(n_pairs, n_hits) || !scratch) return fail(GPET_E_OVERFLOW, "scratch too small: %zu < %zu", scratch_bytes, digitize_scratch_bytes(n_pairs, n_hits));
  DigiParams P; int rc = make_digi(src, seed, n_pairs_total, dig, &P); if (rc) return rc;
  SinglesBuf S; memset(&S, 0, sizeof S);
  if (so) { SinglesBuf s = { so->history, so->ids, so->x, so->y, so->z, so->e_keV, so->t_s, so->capacity, reinterpret_cast<unsigned long long *>(so->n_singles) }; S = s; }
  CoincBuf Cb = { co->ids_a, co->ids_b, co->history_a, co->history_b, co->e_a, co->e_b, co->dt_ns, co->t_s, co->capacity,
                  reinterpret_cast<unsigned long long *>(co->n_coinc) };
  HitBuf HB; rc = hitbuf(hits, n_pairs, &HB); if (rc) return rc;
  CUDA_TRY(launch_digitize(P, HB, first_history, n_pairs, n_hits, scratch, scratch_bytes, S, Cb, (cudaStream_t)stream));
  return GPET_OK;
}

// gpet_digitize on the library's built-in workspace (gpet.h): for callers that own their data buffers but may not call
// cudaMalloc -- the GPU already belongs to the host program's pool, or the call sits in a per-time-slice loop where an
// allocation would stall the device.  Nothing here allocates: the size test is host arithmetic, the workspace address is
// looked up once per device (first call: do it during set-up, before any stream capture), and the rest is gpet_digitize.
extern "C" int gpet_digitize_static(const gpet_source *src, uint64_t seed, uint64_t n_pairs_total, uint64_t first_history, uint64_t n_pairs,
                                    const gpet_hits *hits, uint64_t n_hits, const gpet_digitizer *dig, gpet_singles *so,
                                    gpet_coincidences *co, void *stream) {
  if (!src || !hits || !dig || !co || !co->n_coinc) return fail(GPET_E_INVALID_ARG, "gpet_digitize_static: NULL argument");
  if (n_pairs == 0 || n_pairs >= (1ull << 32) || n_hits > hits->capacity || n_hits > (1ull << 31)) return fail(GPET_E_INVALID_ARG, "gpet_digitize_static: counts out of range");
  const size_t need = digitize_scratch_bytes(n_pairs, n_hits);
  if (need > (size_t)GPET_STATIC_SCRATCH_BYTES)
    return fail(GPET_E_OVERFLOW, "gpet_digitize_static: a batch of %llu pairs / %llu hits needs %zu bytes of workspace, the built-in array holds %zu "
                "(GPET_STATIC_SCRATCH_BYTES); digitize smaller time slices, or call gpet_digitize with your own scratch",
                (unsigned long long)n_pairs, (unsigned long long)n_hits, need, (size_t)GPET_STATIC_SCRATCH_BYTES);
  void *ws = nullptr; size_t ws_bytes = 0;
  CUDA_TRY(static_digitize_scratch(&ws, &ws_bytes));
  return gpet_digitize(src, seed, n_pairs_total, first_history, n_pairs, hits, n_hits, dig, ws, ws_bytes, so, co, stream);
}

// ---------------------------------------------------------------- whole path with host outputs
// One device SLOT holds everything a batch needs (hit buffer, singles, coincidences, scratch, counters); a pipeline owns
// two of them, one compute stream and one copy stream per slot.  Batch k+1 is transported and digitized while the
// list-mode output of batch k travels to the host.
namespace {
struct DevArena {                      // bump allocator over one cudaMalloc
  char *base = nullptr; size_t size = 0, used = 0;
  template <class T> T *take(size_t n) { used = (used + 255) & ~(size_t)255; T *p = reinterpret_cast<T *>(base + used); used += sizeof(T) * n; return p; }
};
struct Slot {
  DevArena A; gpet_hits H; gpet_singles S; gpet_coincidences C; void *scratch = nullptr; size_t scratch_bytes = 0;
  uint64_t cap = 0, n_chunks = 0, n_pairs = 0; bool chunked = true, busy = false;
  cudaStream_t copy = nullptr; cudaEvent_t computed = nullptr, counted = nullptr;
  uint64_t *host_counts = nullptr;     // pinned: n_hits, n_singles, n_coinc, dropped
};
}
struct gpet_pipeline {
  const gpet_geometry *g; const gpet_materials *m; gpet_source src; gpet_digitizer dig;
  uint64_t n_pairs_total, max_pairs; double hits_per_pair; uint32_t want;
  uint8_t *phantom_dev = nullptr; cudaStream_t compute = nullptr; Slot slot[2]; uint64_t submitted = 0, collected = 0;
};

static void slot_release(Slot &s) {
  if (s.A.base) cudaFree(s.A.base);
  if (s.copy) cudaStreamDestroy(s.copy);
  if (s.computed) cudaEventDestroy(s.computed);
  if (s.counted) cudaEventDestroy(s.counted);
  if (s.host_counts) cudaFreeHost(s.host_counts);
  s = Slot();
}

static int slot_create(Slot &s, uint64_t max_pairs, double hits_per_pair, uint32_t want) {
  // hits that stay on the device use the chunked layout (shared-memory sort per chunk in the digitizer); hits the caller
  // wants on the host use the dense one, which is what gpet_host_outputs describes
  s.chunked = !(want & GPET_WANT_HITS);
  s.n_chunks = (max_pairs + kHitChunkPairs - 1) / kHitChunkPairs;
  uint64_t chunk_cap = (uint64_t)ceil((double)kHitChunkPairs * hits_per_pair);
  if (chunk_cap > kHitChunkCapMax) chunk_cap = kHitChunkCapMax;
  const uint64_t cap = s.chunked ? s.n_chunks * chunk_cap : (uint64_t)((double)max_pairs * hits_per_pair) + 1024;
  if (cap >= (1ull << 32)) return fail(GPET_E_INVALID_ARG, "batch too large (%llu hit entries): split it", (unsigned long long)cap);
  s.cap = cap; s.scratch_bytes = digitize_scratch_bytes(max_pairs, cap);
  const bool singles = (want & GPET_WANT_SINGLES) != 0;
  s.A.size = cap * (28 + (singles ? 36 : 0) + 40) + 4 * (s.n_chunks + 1) + s.scratch_bytes + ((want & GPET_WANT_HASH) ? 16 * max_pairs : 0) + 64 * 256;
  CUDA_TRY(cudaMalloc(&s.A.base, s.A.size));
  DevArena &A = s.A; gpet_hits &H = s.H; memset(&H, 0, sizeof H);
  H.history = A.take<uint32_t>(cap); H.ids = A.take<uint32_t>(cap); H.x = A.take<float>(cap); H.y = A.take<float>(cap); H.z = A.take<float>(cap);
  H.e_keV = A.take<float>(cap); H.tof_ns = A.take<float>(cap); H.capacity = cap; H.n_hits = A.take<uint64_t>(1);
  H.outcome_hash = (want & GPET_WANT_HASH) ? A.take<uint64_t>(2 * max_pairs) : nullptr;
  H.chunk_fill = s.chunked ? A.take<uint32_t>(s.n_chunks + 1) : nullptr;
  gpet_singles &S = s.S; memset(&S, 0, sizeof S);
  if (singles) { S.history = A.take<uint32_t>(cap); S.ids = A.take<uint32_t>(cap); S.x = A.take<float>(cap); S.y = A.take<float>(cap);
                 S.z = A.take<float>(cap); S.e_keV = A.take<float>(cap); S.t_s = A.take<double>(cap); }
  S.capacity = cap; S.n_singles = A.take<uint64_t>(1);
  gpet_coincidences &Cc = s.C;
  Cc.ids_a = A.take<uint32_t>(cap); Cc.ids_b = A.take<uint32_t>(cap); Cc.history_a = A.take<uint32_t>(cap);
  Cc.history_b = A.take<uint32_t>(cap); Cc.e_a = A.take<float>(cap); Cc.e_b = A.take<float>(cap); Cc.dt_ns = A.take<float>(cap);
  Cc.t_s = A.take<double>(cap); Cc.capacity = cap; Cc.n_coinc = A.take<uint64_t>(1);
  s.scratch = A.take<char>(s.scratch_bytes);
  if (A.used > A.size) return fail(GPET_E_OVERFLOW, "internal arena too small");
  CUDA_TRY(cudaStreamCreateWithFlags(&s.copy, cudaStreamNonBlocking));
  CUDA_TRY(cudaEventCreateWithFlags(&s.computed, cudaEventDisableTiming));
  CUDA_TRY(cudaEventCreateWithFlags(&s.counted, cudaEventDisableTiming));
  CUDA_TRY(cudaMallocHost(&s.host_counts, 4 * sizeof(uint64_t)));
  return GPET_OK;
}

extern "C" int gpet_pipeline_create(const gpet_geometry *g, const gpet_materials *m, const gpet_source *src, const gpet_digitizer *dig,
                                    uint64_t n_pairs_total, uint64_t max_pairs_per_batch, double hits_per_pair, uint32_t want, int32_t n_slots,
                                    gpet_pipeline **out) {
  if (!g || !m || !src || !dig || !out) return fail(GPET_E_INVALID_ARG, "gpet_pipeline_create: NULL argument");
  if (max_pairs_per_batch == 0 || max_pairs_per_batch >= (1ull << 32) || !(hits_per_pair > 0.0) || n_slots < 1 || n_slots > 2)
    return fail(GPET_E_INVALID_ARG, "gpet_pipeline_create: bad counts");
  if (n_pairs_total < max_pairs_per_batch) return fail(GPET_E_INVALID_ARG, "gpet_pipeline_create: n_pairs_total < max_pairs_per_batch");
  gpet_pipeline *p = new gpet_pipeline;
  p->g = g; p->m = m; p->src = *src; p->dig = *dig; p->n_pairs_total = n_pairs_total; p->max_pairs = max_pairs_per_batch;
  p->hits_per_pair = hits_per_pair; p->want = want;
  int rc = GPET_OK;
  do {
    if (cudaStreamCreateWithFlags(&p->compute, cudaStreamNonBlocking) != cudaSuccess) { rc = fail(GPET_E_CUDA, "cannot create a stream"); break; }
    if (src->kind == 1 && src->phantom_material) {                   // HOST phantom map -> device, once
      const size_t nvox = (size_t)src->dims[0] * src->dims[1] * src->dims[2];
      for (size_t i = 0; i < nvox; ++i) if (src->phantom_material[i] > m->n_materials) { rc = fail(GPET_E_INVALID_ARG, "phantom voxel %zu holds material %d, only %d are loaded", i, (int)src->phantom_material[i] - 1, m->n_materials); break; }
      if (rc) break;
      if (cudaMalloc(&p->phantom_dev, nvox) != cudaSuccess || cudaMemcpy(p->phantom_dev, src->phantom_material, nvox, cudaMemcpyHostToDevice) != cudaSuccess) {
        rc = fail(GPET_E_CUDA, "phantom upload failed"); break; }
      p->src.phantom_material = p->phantom_dev;
    }
    for (int i = 0; i < n_slots && !rc; ++i) rc = slot_create(p->slot[i], max_pairs_per_batch, hits_per_pair, want);
  } while (0);
  if (rc) { gpet_pipeline_destroy(p); return rc; }
  *out = p; return GPET_OK;
}

extern "C" int gpet_pipeline_destroy(gpet_pipeline *p) {
  if (!p) return GPET_OK;
  if (p->compute) cudaStreamSynchronize(p->compute);
  for (Slot &s : p->slot) slot_release(s);
  if (p->phantom_dev) cudaFree(p->phantom_dev);
  if (p->compute) cudaStreamDestroy(p->compute);
  delete p; return GPET_OK;
}

extern "C" int gpet_pipeline_submit(gpet_pipeline *p, uint64_t first_history, uint64_t n_pairs, uint64_t seed) {
  if (!p) return fail(GPET_E_INVALID_ARG, "gpet_pipeline_submit: NULL pipeline");
  if (n_pairs == 0 || n_pairs > p->max_pairs) return fail(GPET_E_INVALID_ARG, "gpet_pipeline_submit: n_pairs %llu outside 1..%llu", (unsigned long long)n_pairs, (unsigned long long)p->max_pairs);
  if (first_history > p->n_pairs_total || n_pairs > p->n_pairs_total - first_history)
    return fail(GPET_E_INVALID_ARG, "gpet_pipeline_submit: histories [%llu, %llu) leave the run of %llu pairs", (unsigned long long)first_history,
                (unsigned long long)(first_history + n_pairs), (unsigned long long)p->n_pairs_total);
  const int n_slots = p->slot[1].A.base ? 2 : 1;
  Slot &s = p->slot[p->submitted % n_slots];
  if (s.busy) return fail(GPET_E_INVALID_ARG, "gpet_pipeline_submit: %d batches already in flight; collect one first", n_slots);
  cudaStream_t st = p->compute;
  CUDA_TRY(cudaMemsetAsync(s.H.n_hits, 0, 8, st));
  if (s.chunked) CUDA_TRY(cudaMemsetAsync(s.H.chunk_fill, 0, 4 * (s.n_chunks + 1), st));
  // the chunked layout divides the buffer by the chunks of THIS batch: keep the per-chunk region of the full-size batch
  gpet_hits H = s.H;
  if (s.chunked) H.capacity = ((n_pairs + kHitChunkPairs - 1) / kHitChunkPairs) * (s.cap / s.n_chunks);
  int rc = gpet_simulate(p->g, p->m, &p->src, first_history, n_pairs, seed, &H, st); if (rc) return rc;
  gpet_singles Sd = s.S;
  rc = gpet_digitize(&p->src, seed, p->n_pairs_total, first_history, n_pairs, &H, H.capacity, &p->dig, s.scratch, s.scratch_bytes, &Sd, &s.C, st); if (rc) return rc;
  CUDA_TRY(cudaEventRecord(s.computed, st));
  CUDA_TRY(cudaStreamWaitEvent(s.copy, s.computed, 0));
  CUDA_TRY(cudaMemcpyAsync(&s.host_counts[0], s.H.n_hits, 8, cudaMemcpyDeviceToHost, s.copy));
  CUDA_TRY(cudaMemcpyAsync(&s.host_counts[1], s.S.n_singles, 8, cudaMemcpyDeviceToHost, s.copy));
  CUDA_TRY(cudaMemcpyAsync(&s.host_counts[2], s.C.n_coinc, 8, cudaMemcpyDeviceToHost, s.copy));
  s.host_counts[3] = 0;
  if (s.chunked) CUDA_TRY(cudaMemcpyAsync(&s.host_counts[3], s.H.chunk_fill + (n_pairs + kHitChunkPairs - 1) / kHitChunkPairs, 4, cudaMemcpyDeviceToHost, s.copy));
  CUDA_TRY(cudaEventRecord(s.counted, s.copy));
  s.busy = true; s.n_pairs = n_pairs; ++p->submitted;
  return GPET_OK;
}

extern "C" int gpet_pipeline_collect(gpet_pipeline *p, gpet_host_outputs *out) {
  if (!p || !out) return fail(GPET_E_INVALID_ARG, "gpet_pipeline_collect: NULL argument");
  const int n_slots = p->slot[1].A.base ? 2 : 1;
  Slot &s = p->slot[p->collected % n_slots];
  if (!s.busy) return fail(GPET_E_INVALID_ARG, "gpet_pipeline_collect: nothing submitted");
  s.busy = false; ++p->collected;
  if (cudaEventSynchronize(s.counted) != cudaSuccess) return fail(GPET_E_CUDA, "transport/digitizer failed: %s", cudaGetErrorString(cudaGetLastError()));
  const uint64_t nh = s.host_counts[0], ns = s.host_counts[1], nc = s.host_counts[2], dropped = s.host_counts[3] & 0xFFFFFFFFull;
  if (dropped) return fail(GPET_E_OVERFLOW, "hit buffer overflow: %llu hits dropped; raise hits_per_pair", (unsigned long long)dropped);
  if (!s.chunked && nh > s.cap) return fail(GPET_E_OVERFLOW, "hit buffer overflow: %llu hits > capacity %llu; raise hits_per_pair", (unsigned long long)nh, (unsigned long long)s.cap);
  if (nc == ~0ull) return fail(GPET_E_OVERFLOW, "the digitizer's time sort dropped singles (decay times far from uniform over the batch's time range): the lists are incomplete");
  if (nc > s.C.capacity) return fail(GPET_E_OVERFLOW, "coincidence buffer overflow");
  cudaStream_t st = s.copy;
#define D2H(dst, srcp, n, T) do { if ((dst) && (srcp) && (n)) CUDA_TRY(cudaMemcpyAsync((dst), (srcp), sizeof(T) * (n), cudaMemcpyDeviceToHost, st)); } while (0)
  if (!s.chunked) {
    const uint64_t ch = nh < out->hits.capacity ? nh : out->hits.capacity;
    D2H(out->hits.history, s.H.history, ch, uint32_t); D2H(out->hits.ids, s.H.ids, ch, uint32_t); D2H(out->hits.x, s.H.x, ch, float);
    D2H(out->hits.y, s.H.y, ch, float); D2H(out->hits.z, s.H.z, ch, float); D2H(out->hits.e_keV, s.H.e_keV, ch, float); D2H(out->hits.tof_ns, s.H.tof_ns, ch, float);
  }
  D2H(out->hits.outcome_hash, s.H.outcome_hash, 2 * s.n_pairs, uint64_t);
  const uint64_t cs = ns < out->singles.capacity ? ns : out->singles.capacity;
  D2H(out->singles.history, s.S.history, cs, uint32_t); D2H(out->singles.ids, s.S.ids, cs, uint32_t); D2H(out->singles.x, s.S.x, cs, float);
  D2H(out->singles.y, s.S.y, cs, float); D2H(out->singles.z, s.S.z, cs, float); D2H(out->singles.e_keV, s.S.e_keV, cs, float); D2H(out->singles.t_s, s.S.t_s, cs, double);
  const uint64_t cc = nc < out->coinc.capacity ? nc : out->coinc.capacity;
  D2H(out->coinc.ids_a, s.C.ids_a, cc, uint32_t); D2H(out->coinc.ids_b, s.C.ids_b, cc, uint32_t); D2H(out->coinc.history_a, s.C.history_a, cc, uint32_t);
  D2H(out->coinc.history_b, s.C.history_b, cc, uint32_t); D2H(out->coinc.e_a, s.C.e_a, cc, float); D2H(out->coinc.e_b, s.C.e_b, cc, float);
  D2H(out->coinc.dt_ns, s.C.dt_ns, cc, float); D2H(out->coinc.t_s, s.C.t_s, cc, double);
#undef D2H
  if (cudaStreamSynchronize(st) != cudaSuccess) return fail(GPET_E_CUDA, "copy back failed: %s", cudaGetErrorString(cudaGetLastError()));
  if (out->hits.n_hits) *out->hits.n_hits = nh;
  if (out->singles.n_singles) *out->singles.n_singles = ns;
  if (out->coinc.n_coinc) *out->coinc.n_coinc = nc;
  return GPET_OK;
}

// One batch, start to finish: a one-slot pipeline kept between calls of the same shape (freed by gpet_shutdown).
namespace {
std::mutex g_host_lock; gpet_pipeline *g_host_pipe = nullptr;
// Field by field: both structs have padding bytes (after positron_fwhm_mm, at the end of gpet_digitizer) that a struct copy
// need not preserve, so a memcmp could miss on equal values and throw the kept buffers away on every call.
bool same_digitizer(const gpet_digitizer &a, const gpet_digitizer &b) {
  return a.blur_fwhm_frac == b.blur_fwhm_frac && a.blur_ref_keV == b.blur_ref_keV && a.e_lo_keV == b.e_lo_keV && a.e_hi_keV == b.e_hi_keV &&
         a.window_ns == b.window_ns && a.readout_level == b.readout_level;
}
bool same_source(const gpet_source &a, const gpet_source &b) {
  bool eq = a.kind == b.kind && a.acolinearity_fwhm_deg == b.acolinearity_fwhm_deg && a.activity_bq == b.activity_bq &&
            a.pairs_per_time_slice == b.pairs_per_time_slice && a.activity_map == b.activity_map && a.phantom_material == b.phantom_material &&
            a.phantom_majorant_material == b.phantom_majorant_material && a.positron_fwhm_mm == b.positron_fwhm_mm &&
            a.half_life_s == b.half_life_s && a.duration_s == b.duration_s;
  for (int k = 0; k < 3; ++k)
    eq = eq && a.pos_mm[k] == b.pos_mm[k] && a.beam_dir[k] == b.beam_dir[k] && a.dims[k] == b.dims[k] && a.voxel_mm[k] == b.voxel_mm[k] &&
         a.origin_mm[k] == b.origin_mm[k];
  return eq;
}
}
extern "C" int gpet_run_host(const gpet_geometry *g, const gpet_materials *m, const gpet_source *src, uint64_t n_pairs_total,
                             uint64_t first_history, uint64_t n_pairs, uint64_t seed, const gpet_digitizer *dig, double hits_per_pair,
                             gpet_host_outputs *out) {
  if (!g || !m || !src || !dig || !out) return fail(GPET_E_INVALID_ARG, "gpet_run_host: NULL argument");
  const uint32_t want = (out->hits.history ? GPET_WANT_HITS : 0u) | (out->singles.history ? GPET_WANT_SINGLES : 0u) | (out->hits.outcome_hash ? GPET_WANT_HASH : 0u);
  std::lock_guard<std::mutex> lk(g_host_lock);
  gpet_pipeline *p = g_host_pipe;
  const bool reuse = p && p->g == g && p->m == m && p->max_pairs == n_pairs && p->n_pairs_total == n_pairs_total && p->hits_per_pair == hits_per_pair &&
                     p->want == want && !p->phantom_dev && !(src->kind == 1 && src->phantom_material) &&
                     same_digitizer(p->dig, *dig) && same_source(p->src, *src);
  if (!reuse) {
    if (p) gpet_pipeline_destroy(p);
    g_host_pipe = nullptr;
    int rc = gpet_pipeline_create(g, m, src, dig, n_pairs_total, n_pairs, hits_per_pair, want, 1, &p); if (rc) return rc;
    g_host_pipe = p;
  }
  int rc = gpet_pipeline_submit(p, first_history, n_pairs, seed);
  if (!rc) rc = gpet_pipeline_collect(p, out);
  return rc;
}

extern "C" int gpet_shutdown(void) {
  { std::lock_guard<std::mutex> lk(g_host_lock); if (g_host_pipe) gpet_pipeline_destroy(g_host_pipe); g_host_pipe = nullptr; }
  work_ring_release();
  return GPET_OK;
}
