/* gpet_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded fp64 CPU implementation of the hot path of
 * "Extending gPET for Multi-Layer PET Simulation" (arxiv 2603.07327): source -> (phantom) ->
 * panel search -> in-panel Woodcock tracking with layer selection -> photoelectric / Klein-Nishina
 * Compton / Rayleigh -> hits -> adder -> energy blur -> window -> time sort -> coincidences.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this.  It shares no code, header, table or constant generator with the CUDA path under
 * paper_2603_07327_b200/csrc; the two only consume the same inputs and the same Philox words.
 *
 * The paper fixes the structure (PAPER.md:33 hierarchy, line-plane transfer, global->local;
 * PAPER.md:43 Woodcock tracking + layer selection from the local depth, run until exit or
 * cutoff; PAPER.md:37 crystal/layer/module/panel ids per interaction; PAPER.md:61 blur, window,
 * coincidence window).  It gives no physics detail; every reading of a silent passage is listed
 * in DESIGN.md ("Readings R1..R30") and cited below as [Rn].  BASELINE.json configs[0] fixes the
 * interaction model and the mu tables (inputs here).
 *
 * Parity pins: tests/test_oracle_pins.py (Philox vs cuRAND's header and published vectors,
 * exp(-mu L) transmission, interaction fractions, Klein-Nishina pdf, Thomson cdf, solid angle,
 * energy conservation, brute-force indexing, split-layer identity, time of flight, brute-force
 * adder/coincidences, blur width).  Unpinned: absolute agreement with gPET/GATE (not available).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_Q        1048576.0          /* [R7] lengths are quantised to 2^-20 mm            */
#define ORC_MEC2     510.99895          /* [R12] electron rest energy, keV                   */
#define ORC_C_MM_NS  299.792458         /* speed of light, mm/ns                             */
#define ORC_CUTOFF   10.0               /* [R12] cutoff energy = table floor, keV            */
#define ORC_FWHM     2.354820045030949  /* 2*sqrt(2 ln 2)                                    */
#define ORC_PI       3.14159265358979323846
#define ORC_KN_CAP   64                 /* [R22] Klein-Nishina trial cap                     */
#define ORC_NONE     0xFFFFFFFFu
#define ORC_MAX_LAYERS 4

/* ------------------------------------------------------------------ public structures */
typedef struct {
  int32_t n[2]; float pitch[2], reflector[2], offset[2]; float depth, gap_before;
  int32_t crystal_material, gap_material;
} orc_layer;

typedef struct {
  int32_t n_panels; const float *pose;           /* n_panels x 12: centre, u, v, w (fp32)   */
  int32_t n_modules[2]; float module_size[2], module_pitch[2];
  int32_t n_layers; const orc_layer *layers;
} orc_geometry;

typedef struct {
  int32_t n_materials, n_energies; float e_min, e_step;
  const float *mu_pe, *mu_c, *mu_r;              /* [n_materials][n_energies], 1/mm         */
} orc_materials;

typedef struct {
  int32_t kind; float pos[3]; float acol_fwhm_deg; double activity_bq; uint64_t pairs_per_slice;
  const float *activity; const uint8_t *phantom; int32_t phantom_majorant;
  int32_t dims[3]; float voxel[3]; float origin[3];
  float beam_dir[3];                             /* kind 2: pencil beam along beam_dir (photon A) */
  float positron_fwhm_mm;                        /* [R35] 0 = annihilation at the emission site */
  double half_life_s, duration_s;                /* [R34] half_life_s > 0: decay law over duration_s, activity_bq = initial activity */
  /* derived once by orc_source_prepare (active voxel list + integer CDF) [R13] */
  uint32_t *act_index; uint64_t *act_cdf; uint64_t n_active; uint64_t w_total;
} orc_source;

typedef struct {
  uint32_t *history, *ids; float *x, *y, *z, *e, *tof; uint64_t capacity, n;
} orc_hits;

typedef struct {             /* event counters (metrics; also feed the roofline model) */
  uint64_t pairs, searches, entries, steps, step_vacuum, virtuals, pe, compton, kn_trials,
           rayleigh, cutoffs, exits, escapes, hits, ph_steps, ph_compton, ph_absorbed, ph_cutoff, region_crossings;
} orc_counters;

typedef struct { float fwhm_frac, ref_keV, e_lo, e_hi; double window_ns; int32_t level; } orc_digitizer;

typedef struct { uint32_t *history, *ids; float *x, *y, *z, *e; double *t; uint64_t capacity, n; } orc_singles;
typedef struct { uint32_t *ids_a, *ids_b, *history_a, *history_b; float *e_a, *e_b, *dt_ns; double *t;
                 uint64_t capacity, n; } orc_coinc;

/* ------------------------------------------------------------------ [R1] Philox4x32-10 */
/* Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3" (SC'11). */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
  for (int r = 0; r < 10; ++r) {
    uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* [R1] key = seed; counter = (history lo, history hi, stream, block) */
typedef struct { uint32_t key[2], ctr[4]; uint32_t ndraw; uint32_t blk[4]; } rng_t;
enum { STREAM_SOURCE = 0, STREAM_A = 1, STREAM_B = 2, STREAM_DIGI = 3 };

static void rng_init(rng_t *r, uint64_t seed, uint64_t history, uint32_t stream) {
  r->key[0] = (uint32_t)seed; r->key[1] = (uint32_t)(seed >> 32);
  r->ctr[0] = (uint32_t)history; r->ctr[1] = (uint32_t)(history >> 32); r->ctr[2] = stream; r->ctr[3] = 0;
  r->ndraw = 0;
}
static uint32_t rng_word_at(rng_t *r, uint32_t j) {      /* random access (fixed slots, [R3]) */
  uint32_t b[4]; r->ctr[3] = j >> 2; orc_philox4x32_10(r->ctr, r->key, b); return b[j & 3];
}
/* [R4] transport streams are consumed one whole Philox block per event: u[0..3] of block number ndraw++ */
static void rng_next_block(rng_t *r, double u[4]) {
  r->ctr[3] = r->ndraw++; orc_philox4x32_10(r->ctr, r->key, r->blk);
  for (int k = 0; k < 4; ++k) u[k] = ((double)(r->blk[k] >> 9) + 0.5) * (1.0 / 8388608.0);
}
/* [R2] u = ((x >> 9) + 0.5) * 2^-23, in (0,1): 2k+1 < 2^24, so exactly representable in fp32 and fp64 */
double orc_uniform(uint32_t x) { return ((double)(x >> 9) + 0.5) * (1.0 / 8388608.0); }

/* ------------------------------------------------------------------ geometry (quantised) */
typedef struct { double o[3], u[3], v[3], w[3]; } panel_t;
typedef struct {
  int n_panels; panel_t *panel;
  int64_t Wq, Hq, Dq, hWq, hHq;                 /* panel box in Q units; tracking origin (hWq,hHq,0) */
  int nmod[2]; int64_t msq[2], mpq[2];
  int n_layers;
  struct { int n[2]; int64_t pitch[2], gap[2], off[2], c0, depth; int cmat, gmat; } layer[ORC_MAX_LAYERS];
  /* [R19] majorant regions: maximal runs of consecutive layers with the same crystal and gap material; region r spans
   * the depths [reg_c[r], reg_c[r+1]) (the gap in front of a region's first layer belongs to the region before it) */
  int n_regions; int64_t reg_c[ORC_MAX_LAYERS + 1]; uint32_t reg_mask[ORC_MAX_LAYERS];
} geom_t;

static int64_t quant(float x) { return llrint((double)x * ORC_Q); }   /* [R7] */

/* [R5] ring placement (repetition mode): writes n x 12 fp32 pose entries */
void orc_ring_poses(int n, double radius_mm, double first_angle_deg, float *pose) {
  for (int p = 0; p < n; ++p) {
    double phi = (first_angle_deg + 360.0 * (double)p / (double)n) * (ORC_PI / 180.0);
    double c = cos(phi), s = sin(phi);
    if (fabs(c) < 1e-12) c = 0.0;
    if (fabs(s) < 1e-12) s = 0.0;
    float *q = pose + 12 * p;
    q[0] = (float)(radius_mm * c); q[1] = (float)(radius_mm * s); q[2] = 0.0f;   /* front-face centre */
    q[3] = (float)(-s); q[4] = (float)c; q[5] = 0.0f;                            /* u tangential      */
    q[6] = 0.0f; q[7] = 0.0f; q[8] = 1.0f;                                       /* v axial           */
    q[9] = (float)c; q[10] = (float)s; q[11] = 0.0f;                             /* w depth, outward  */
  }
}

/* returns 0 or a negative code: -1 bad counts, -2 lattice overhangs module / negative length */
static int geom_build(const orc_geometry *d, geom_t *g) {
  memset(g, 0, sizeof *g);
  if (d->n_panels < 1 || d->n_panels > 63 || d->n_layers < 1 || d->n_layers > ORC_MAX_LAYERS) return -1;
  g->n_panels = d->n_panels;
  g->panel = (panel_t *)malloc(sizeof(panel_t) * (size_t)d->n_panels);
  for (int p = 0; p < d->n_panels; ++p)
    for (int k = 0; k < 3; ++k) {
      g->panel[p].o[k] = d->pose[12 * p + k];     g->panel[p].u[k] = d->pose[12 * p + 3 + k];
      g->panel[p].v[k] = d->pose[12 * p + 6 + k]; g->panel[p].w[k] = d->pose[12 * p + 9 + k];
    }
  for (int a = 0; a < 2; ++a) {
    g->nmod[a] = d->n_modules[a];
    g->msq[a] = quant(d->module_size[a]); g->mpq[a] = quant(d->module_pitch[a]);
    if (g->nmod[a] < 1 || g->msq[a] <= 0 || g->mpq[a] < g->msq[a]) return -2;
  }
  g->Wq = (g->nmod[0] - 1) * g->mpq[0] + g->msq[0];   /* [R5] panel = modules incl. inter-module gaps */
  g->Hq = (g->nmod[1] - 1) * g->mpq[1] + g->msq[1];
  g->hWq = g->Wq >> 1; g->hHq = g->Hq >> 1;
  g->n_layers = d->n_layers;
  int64_t c = 0;
  for (int l = 0; l < d->n_layers; ++l) {
    const orc_layer *s = &d->layers[l];
    int64_t gb = quant(s->gap_before), dp = quant(s->depth);
    if (gb < 0 || dp <= 0) return -2;
    c += gb; g->layer[l].c0 = c; g->layer[l].depth = dp; c += dp;
    g->layer[l].cmat = s->crystal_material; g->layer[l].gmat = s->gap_material;
    for (int a = 0; a < 2; ++a) {
      g->layer[l].n[a] = s->n[a]; g->layer[l].pitch[a] = quant(s->pitch[a]);
      g->layer[l].gap[a] = quant(s->reflector[a]); g->layer[l].off[a] = quant(s->offset[a]);
      if (s->n[a] < 1 || g->layer[l].pitch[a] <= 0 || g->layer[l].gap[a] < 0 ||
          g->layer[l].gap[a] >= g->layer[l].pitch[a] || g->layer[l].off[a] < 0 ||
          g->layer[l].off[a] + s->n[a] * g->layer[l].pitch[a] > g->msq[a]) return -2;
    }
    if (s->n[0] * s->n[1] > 8192) return -1;
  }
  g->Dq = c;
  g->n_regions = 0;
  for (int l = 0; l < g->n_layers; ++l) {
    if (l == 0 || g->layer[l].cmat != g->layer[l - 1].cmat || g->layer[l].gmat != g->layer[l - 1].gmat) {
      g->reg_c[g->n_regions] = l == 0 ? 0 : g->layer[l].c0; g->reg_mask[g->n_regions] = 0; g->n_regions++;
    }
    g->reg_mask[g->n_regions - 1] |= 1u << g->layer[l].cmat;
    if (g->layer[l].gmat >= 0) g->reg_mask[g->n_regions - 1] |= 1u << g->layer[l].gmat;
  }
  g->reg_c[g->n_regions] = g->Dq;
  return 0;
}
static void geom_free(geom_t *g) { free(g->panel); g->panel = NULL; }

/* [R9] packed ids: seq[0:4) photon[4] crystal[5:18) layer[18:20) module[20:26) panel[26:32) */
static uint32_t pack_ids(int panel, int module, int layer, int crystal) {
  return ((uint32_t)panel << 26) | ((uint32_t)module << 20) | ((uint32_t)layer << 18) | ((uint32_t)crystal << 5);
}

static int64_t floor_div(int64_t a, int64_t b) { int64_t q = a / b; return (a % b < 0) ? q - 1 : q; }

/* [R7] Lattice lookup in panel-local Q coordinates measured from the panel's low corner
 * (depth picks the layer, that layer's crystal parameters give material + index;
 * pitch = crystal + gap).  Returns the material index (-1 vacuum) and writes the ids
 * (ORC_NONE when the point is not inside a crystal).  All intervals half-open. */
static int lattice_lookup(const geom_t *g, int panel, int64_t qa, int64_t qb, int64_t qc, uint32_t *ids) {
  *ids = ORC_NONE;
  if (qa < 0 || qa >= g->Wq || qb < 0 || qb >= g->Hq || qc < 0 || qc >= g->Dq) return -1;
  int64_t m[2], r[2], q[2] = { qa, qb };
  for (int a = 0; a < 2; ++a) {
    m[a] = q[a] / g->mpq[a]; r[a] = q[a] - m[a] * g->mpq[a];
    if (m[a] >= g->nmod[a] || r[a] >= g->msq[a]) return -1;              /* inter-module gap: vacuum */
  }
  int l = -1;
  for (int k = 0; k < g->n_layers; ++k)
    if (qc >= g->layer[k].c0 && qc < g->layer[k].c0 + g->layer[k].depth) l = k;
  if (l < 0) return -1;                                                   /* inter-layer gap: vacuum  */
  int64_t ix[2]; int inside = 1;
  for (int a = 0; a < 2; ++a) {
    int64_t rel = r[a] - g->layer[l].off[a], p = g->layer[l].pitch[a], gp = g->layer[l].gap[a];
    ix[a] = floor_div(rel, p);
    int64_t fr = rel - ix[a] * p, glo = gp >> 1, ghi = gp - glo;
    if (ix[a] < 0 || ix[a] >= g->layer[l].n[a] || fr < glo || fr >= p - ghi) inside = 0;
  }
  if (!inside) return g->layer[l].gmat;                                   /* reflector / rim          */
  *ids = pack_ids(panel, (int)(m[0] + g->nmod[0] * m[1]), l, (int)(ix[0] + g->layer[l].n[0] * ix[1]));
  return g->layer[l].cmat;
}

static double dot3(const double a[3], const double b[3]) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

static void to_local(const panel_t *P, const double x[3], const double d[3], double xl[3], double dl[3]) {
  double r[3] = { x[0] - P->o[0], x[1] - P->o[1], x[2] - P->o[2] };       /* PAPER.md:33 global->local */
  xl[0] = dot3(r, P->u); xl[1] = dot3(r, P->v); xl[2] = dot3(r, P->w);
  if (d) { dl[0] = dot3(d, P->u); dl[1] = dot3(d, P->v); dl[2] = dot3(d, P->w); }
}
static void to_global(const panel_t *P, const double xl[3], const double dl[3], double x[3], double d[3]) {
  for (int k = 0; k < 3; ++k) {
    x[k] = P->o[k] + xl[0] * P->u[k] + xl[1] * P->v[k] + xl[2] * P->w[k];
    if (d) d[k] = dl[0] * P->u[k] + dl[1] * P->v[k] + dl[2] * P->w[k];
  }
}
static void box_bounds(const geom_t *g, double lo[3], double hi[3]) {
  lo[0] = -(double)g->hWq / ORC_Q; hi[0] = (double)(g->Wq - g->hWq) / ORC_Q;
  lo[1] = -(double)g->hHq / ORC_Q; hi[1] = (double)(g->Hq - g->hHq) / ORC_Q;
  lo[2] = 0.0;                     hi[2] = (double)g->Dq / ORC_Q;
}
/* [R6] slab test of a local ray against the panel box; returns 1 and (t_near, t_far) unless an
 * axis with zero direction lies outside its slab (never forms 0*inf). */
static int slab(const double lo[3], const double hi[3], const double x[3], const double d[3], double *tn, double *tf) {
  double a = -INFINITY, b = INFINITY;
  for (int k = 0; k < 3; ++k) {
    if (d[k] == 0.0) { if (x[k] < lo[k] || x[k] >= hi[k]) return 0; continue; }
    double t1 = (lo[k] - x[k]) / d[k], t2 = (hi[k] - x[k]) / d[k];
    if (t1 > t2) { double s = t1; t1 = t2; t2 = s; }
    if (t1 > a) a = t1;
    if (t2 < b) b = t2;
  }
  *tn = a; *tf = b; return 1;
}
/* Distance along the ray to the far face of each slab of a box the point is inside of, and their minimum; returns the
 * axis of the face met first (ties: the first of a, b, c).  A zero direction component never limits [R32]. */
static int slab_far(const double lo[3], const double hi[3], const double x[3], const double d[3], double tfar[3], double *tf) {
  int kx = 2; double best = INFINITY;
  for (int k = 0; k < 3; ++k) tfar[k] = d[k] == 0.0 ? INFINITY : ((d[k] > 0.0 ? hi[k] : lo[k]) - x[k]) / d[k];
  for (int k = 2; k >= 0; --k) if (tfar[k] <= best) { best = tfar[k]; kx = k; }
  *tf = best; return kx;
}
/* [R6] nearest-entry panel over all panels but `excl`; ties -> lowest index; -1 = escapes */
static int panel_search(const geom_t *g, const double x[3], const double d[3], int excl, double *t_enter) {
  double lo[3], hi[3], best = INFINITY; int bp = -1;
  box_bounds(g, lo, hi);
  for (int p = 0; p < g->n_panels; ++p) {
    if (p == excl) continue;
    double xl[3], dl[3], tn, tf;
    to_local(&g->panel[p], x, d, xl, dl);
    if (!slab(lo, hi, xl, dl, &tn, &tf)) continue;
    double te = tn > 0.0 ? tn : 0.0;
    if (tf > te && te < best) { best = te; bp = p; }
  }
  *t_enter = best; return bp;
}

/* point -> packed ids (ORC_NONE if not in a crystal): the plain definition used for the indexing test */
uint32_t orc_locate_point(const geom_t *g, const float xyz[3]) {
  double lo[3], hi[3]; box_bounds(g, lo, hi);
  for (int p = 0; p < g->n_panels; ++p) {                        /* lowest panel index containing it */
    double x[3] = { xyz[0], xyz[1], xyz[2] }, xl[3];
    to_local(&g->panel[p], x, NULL, xl, NULL);
    if (xl[0] < lo[0] || xl[0] >= hi[0] || xl[1] < lo[1] || xl[1] >= hi[1] || xl[2] < lo[2] || xl[2] >= hi[2]) continue;
    uint32_t ids;
    lattice_lookup(g, p, (int64_t)floor(xl[0] * ORC_Q) + g->hWq, (int64_t)floor(xl[1] * ORC_Q) + g->hHq,
                   (int64_t)floor(xl[2] * ORC_Q), &ids);
    return ids;
  }
  return ORC_NONE;
}
int orc_locate(const orc_geometry *d, int64_t n, const float *xyz, uint32_t *ids) {
  geom_t g; int rc = geom_build(d, &g); if (rc) { geom_free(&g); return rc; }
  for (int64_t i = 0; i < n; ++i) ids[i] = orc_locate_point(&g, xyz + 3 * i);
  geom_free(&g); return 0;
}
/* local-frame variant: (a,b,c) in the tracking frame of `panel` */
int orc_locate_local(const orc_geometry *d, int panel, int64_t n, const double *abc, uint32_t *ids, int32_t *material) {
  geom_t g; int rc = geom_build(d, &g); if (rc) { geom_free(&g); return rc; }
  for (int64_t i = 0; i < n; ++i)
    material[i] = lattice_lookup(&g, panel, (int64_t)floor(abc[3 * i] * ORC_Q) + g.hWq,
                                 (int64_t)floor(abc[3 * i + 1] * ORC_Q) + g.hHq, (int64_t)floor(abc[3 * i + 2] * ORC_Q), &ids[i]);
  geom_free(&g); return 0;
}

/* ------------------------------------------------------------------ [R11] mu tables */
typedef struct { double pe, c, r; } mu3_t;
static mu3_t mu_lookup(const orc_materials *M, int m, double E) {
  double x = (E - (double)M->e_min) / (double)M->e_step;
  int i = (int)floor(x); if (i > M->n_energies - 2) i = M->n_energies - 2; if (i < 0) i = 0;
  double f = x - (double)i;
  const float *pe = M->mu_pe + (size_t)m * M->n_energies, *c = M->mu_c + (size_t)m * M->n_energies,
              *r = M->mu_r + (size_t)m * M->n_energies;
  mu3_t o = { pe[i] + f * ((double)pe[i + 1] - pe[i]), c[i] + f * ((double)c[i + 1] - c[i]),
              r[i] + f * ((double)r[i + 1] - r[i]) };
  return o;
}
static double mu_total(const orc_materials *M, int m, double E) { mu3_t u = mu_lookup(M, m, E); return u.pe + u.c + u.r; }
/* [R19] majorant of a material set given as a bitmask: max over the set of the interpolated mu_tot(E).
 * (Interpolating each table and taking the max equals interpolating the pointwise-max table whenever
 * the ordering does not change inside a cell; the CUDA side tabulates the pointwise max.) */
static double mu_majorant(const orc_materials *M, uint32_t mask, double E) {
  double x = (E - (double)M->e_min) / (double)M->e_step;
  int i = (int)floor(x); if (i > M->n_energies - 2) i = M->n_energies - 2; if (i < 0) i = 0;
  double f = x - (double)i, lo = 0.0, hi = 0.0;
  for (int m = 0; m < M->n_materials; ++m) if (mask >> m & 1u) {
    size_t k = (size_t)m * M->n_energies + i;
    double a = (double)M->mu_pe[k] + (double)M->mu_c[k] + (double)M->mu_r[k];
    double b = (double)M->mu_pe[k + 1] + (double)M->mu_c[k + 1] + (double)M->mu_r[k + 1];
    if (a > lo) lo = a;
    if (b > hi) hi = b;
  }
  return lo + f * (hi - lo);
}

void orc_mu_lookup(const orc_materials *M, int m, double E, double out[3]) { mu3_t u = mu_lookup(M, m, E); out[0] = u.pe; out[1] = u.c; out[2] = u.r; }  /* test hook */
double orc_mu_majorant(const orc_materials *M, uint32_t mask, double E) { return mu_majorant(M, mask, E); }                                      /* test hook */

/* ------------------------------------------------------------------ sampling */
/* [R21] branchless orthonormal basis + rotation by polar (cos t, sin t) and azimuth (cos p, sin p) */
void orc_rotate(double d[3], double ct, double st, double cp, double sp) {
  double sg = copysign(1.0, d[2]), a = -1.0 / (sg + d[2]), b = d[0] * d[1] * a;
  double b1[3] = { 1.0 + sg * d[0] * d[0] * a, sg * b, -sg * d[0] };
  double b2[3] = { b, sg + d[1] * d[1] * a, -d[1] };
  double n[3], s = 0.0;
  for (int k = 0; k < 3; ++k) { n[k] = ct * d[k] + st * (cp * b1[k] + sp * b2[k]); s += n[k] * n[k]; }
  s = 1.0 / sqrt(s);
  for (int k = 0; k < 3; ++k) d[k] = n[k] * s;
}
static void azimuth(double u, double *c, double *s) { *c = cos(2.0 * ORC_PI * u); *s = sin(2.0 * ORC_PI * u); }

/* [R20] Klein-Nishina by composition-rejection (free electron).  Returns eps = E'/E, writes
 * cos(theta), sin^2(theta) and the number of trials.  3 draws per trial. */
/* where a trial's four uniforms come from: the photon's Philox stream, or (test hook below) a prepared list */
typedef struct { rng_t *r; const double *prepared; int n_prepared, i_prepared; } kn_draws_t;
static void kn_next_block(kn_draws_t *d, double u[4]) {
  if (d->r) { rng_next_block(d->r, u); return; }
  for (int k = 0; k < 4; ++k) u[k] = d->i_prepared < d->n_prepared ? d->prepared[4 * d->i_prepared + k] : 0.5;
  ++d->i_prepared;
}
static double kn_sample_draws(kn_draws_t *r, double E, double *cos_t, double *sin2_t, int *trials, double *u_azimuth) {
  double k = E / ORC_MEC2, e0 = 1.0 / (1.0 + 2.0 * k), a1 = -log(e0), a2 = 0.5 * (1.0 - e0 * e0);
  double eps = 1.0, t = 0.0;
  for (int n = 1; n <= ORC_KN_CAP; ++n) {
    double u[4]; kn_next_block(r, u);                              /* [R4] one block per trial: u_a, u_b, u_c, azimuth */
    double ua = u[0], ub = u[1], uc = u[2]; *u_azimuth = u[3];
    if (ua < a1 / (a1 + a2)) eps = exp(-a1 * ub);
    else eps = sqrt(e0 * e0 + (1.0 - e0 * e0) * ub);
    t = (1.0 - eps) / (k * eps);
    double g = 1.0 - eps * t * (2.0 - t) / (1.0 + eps * eps);
    *trials = n;
    if (g >= uc || n == ORC_KN_CAP) break;
  }
  *cos_t = 1.0 - t; *sin2_t = t * (2.0 - t); if (*sin2_t < 0.0) *sin2_t = 0.0;
  return eps;
}
static double kn_sample(rng_t *r, double E, double *cos_t, double *sin2_t, int *trials, double *u_azimuth) {
  kn_draws_t d = { r, NULL, 0, 0 }; return kn_sample_draws(&d, E, cos_t, sin2_t, trials, u_azimuth);
}
/* test hook: the same sampler on a PREPARED list of n_blocks x 4 uniforms {u_a, u_b, u_c, azimuth}, so a
 * test can make every trial fail and reach the trial cap, which honest draws never do (p < 1e-30) */
int orc_kn_sample_prepared(const double *u4, int n_blocks, double E, double *eps, double *cos_t, double *u_azimuth) {
  kn_draws_t d = { NULL, u4, n_blocks, 0 }; double s2; int n; *eps = kn_sample_draws(&d, E, cos_t, &s2, &n, u_azimuth); return n;
}
int orc_kn_sample(uint64_t seed, uint64_t history, double E, double *eps, double *cos_t) {  /* test hook */
  rng_t r; rng_init(&r, seed, history, STREAM_A); double s2, ua; int n; *eps = kn_sample(&r, E, cos_t, &s2, &n, &ua); return n;
}
/* [R20] Rayleigh with the Thomson pdf 3/8 (1 + cos^2), closed-form inversion of the cdf */
double orc_rayleigh_cos(double u) { double a = 4.0 * u - 2.0, q = sqrt(a * a + 1.0); return cbrt(a + q) - cbrt(q - a); }

/* ------------------------------------------------------------------ hash [R23] */
enum { EV_ENTER = 1, EV_STEP_VACUUM, EV_VIRTUAL, EV_PE, EV_COMPTON, EV_RAYLEIGH, EV_CUTOFF, EV_EXIT, EV_ESCAPE,
       EV_PH_COMPTON, EV_PH_RAYLEIGH, EV_PH_ABSORBED, EV_PH_CUTOFF, EV_PH_LEAVE, EV_REGION };
static void hash_ev(uint64_t *h, uint32_t type, uint32_t payload) {
  *h = (*h ^ (uint64_t)type) * 0x100000001B3ull;        /* FNV-1a over 32-bit words */
  *h = (*h ^ (uint64_t)payload) * 0x100000001B3ull;
}

/* ------------------------------------------------------------------ source [R13-R16] */
int orc_source_prepare(orc_source *s) {
  s->act_index = NULL; s->act_cdf = NULL; s->n_active = 0; s->w_total = 0;
  if (s->kind != 1) return 0;
  uint64_t nv = (uint64_t)s->dims[0] * s->dims[1] * s->dims[2], na = 0;
  for (uint64_t i = 0; i < nv; ++i) if (s->activity[i] > 0.0f) ++na;
  if (na == 0) return -1;
  s->act_index = (uint32_t *)malloc(sizeof(uint32_t) * na); s->act_cdf = (uint64_t *)malloc(sizeof(uint64_t) * na);
  /* integer weights: activity scaled so the largest voxel weighs 2^20, rounded to nearest, min 1 [R13] */
  float amax = 0.0f; for (uint64_t i = 0; i < nv; ++i) if (s->activity[i] > amax) amax = s->activity[i];
  uint64_t cum = 0, j = 0;
  for (uint64_t i = 0; i < nv; ++i) if (s->activity[i] > 0.0f) {
    uint64_t w = (uint64_t)llrint((double)s->activity[i] / (double)amax * 1048576.0); if (w < 1) w = 1;
    cum += w; s->act_index[j] = (uint32_t)i; s->act_cdf[j] = cum; ++j;
  }
  s->n_active = na; s->w_total = cum; return 0;
}
void orc_source_release(orc_source *s) { free(s->act_index); free(s->act_cdf); s->act_index = NULL; s->act_cdf = NULL; }

/* [R34] natural logarithm of z in (0, 1] from IEEE +, -, *, / only (no libm), so that the CUDA path, which restates
 * it with round-to-nearest intrinsics, gets bit-identical decay times: z = m 2^e with m in [sqrt(1/2), sqrt(2));
 * ln m = 2 atanh(s), s = (m-1)/(m+1), |s| <= 0.1716, odd series to s^25 (truncation < 1e-20). */
double orc_det_log(double z) {
  uint64_t bits; memcpy(&bits, &z, 8);
  int e = (int)((bits >> 52) & 0x7FF) - 1022;                       /* z = f 2^e, f in [0.5, 1) */
  bits = (bits & 0x000FFFFFFFFFFFFFull) | 0x3FE0000000000000ull;
  double m; memcpy(&m, &bits, 8);
  if (m < 0.70710678118654752440) { m = m * 2.0; e -= 1; }         /* m in [sqrt(1/2), sqrt(2)) */
  double s = (m - 1.0) / (m + 1.0), s2 = s * s, p = 1.0 / 25.0;
  for (int k = 23; k >= 1; k -= 2) p = p * s2 + 1.0 / (double)k;
  return (double)e * 0.69314718055994530942 + 2.0 * s * p;
}
/* ln(1 - y) for y in [0, 1): below 1/4 the series runs on s = -y / (2 - y) directly (1 - y is never formed, so short
 * acquisitions of long-lived sources keep full relative accuracy), above it is orc_det_log(1 - y) */
double orc_det_log1m(double y) {
  if (y < 0.25) {
    double s = -y / (2.0 - y), s2 = s * s, p = 1.0 / 25.0;
    for (int k = 23; k >= 1; k -= 2) p = p * s2 + 1.0 / (double)k;
    return 2.0 * s * p;
  }
  return orc_det_log(1.0 - y);
}
/* [R34] expected number of decays of a source of initial activity A0 (Bq) and half-life T_half over T seconds:
 * N = A0 / lambda (1 - exp(-lambda T)) (1.6e8 atoms of 18F, 1.70e-2 MBq, 120 s) */
uint64_t orc_decay_count(double activity_bq, double half_life_s, double duration_s) {
  if (!(half_life_s > 0.0)) return (uint64_t)llrint(activity_bq * duration_s);
  double lambda = 0.69314718055994530942 / half_life_s;
  return (uint64_t)llrint(activity_bq / lambda * -expm1(-lambda * duration_s));
}
/* [R16] decay time of history i, seconds (fp64): t0 = (floor(i/B) + u53) * (B/A).
 * [R34] with a half-life: the stratified quantile q = (k + u53 f_k) B / N of slice k = floor(i/B) goes through the
 * inverse cdf of the decay law truncated to the acquisition: t0 = -ln(1 - q P) / lambda, P = 1 - exp(-lambda T) (the
 * constant P comes from the C library's expm1 on the host, on both sides).  f_k = 1 for a full slice; the last slice of a
 * run whose N is not a multiple of B holds only N mod B histories and covers only [kB/N, 1): f_k = (N mod B) / B, so
 * that q stays in (0, 1] and t0 in (0, T] (stretching it to a full slice would run past the end of the acquisition). */
double orc_decay_time(const orc_source *s, uint64_t seed, uint64_t history, uint64_t n_pairs_total) {
  rng_t r; rng_init(&r, seed, history, STREAM_SOURCE);
  uint64_t w8 = rng_word_at(&r, 8), w9 = rng_word_at(&r, 9);
  double u53 = ((double)(((w8 << 32) | w9) >> 11) + 0.5) * (1.0 / 9007199254740992.0);
  uint64_t B = s->pairs_per_slice ? s->pairs_per_slice : n_pairs_total;
  if (s->half_life_s > 0.0) {
    double lambda = 0.69314718055994530942 / s->half_life_s, P = -expm1(-lambda * s->duration_s);
    uint64_t k = history / B;
    double f = (n_pairs_total % B != 0 && k == n_pairs_total / B) ? (double)(n_pairs_total % B) / (double)B : 1.0;
    double q = ((double)k + u53 * f) * ((double)B / (double)n_pairs_total);
    return -orc_det_log1m(q * P) / lambda;
  }
  return ((double)(history / B) + u53) * ((double)B / s->activity_bq);
}

/* ------------------------------------------------------------------ transport of one photon */
typedef struct {
  const geom_t *g; const orc_materials *M; const orc_source *S; uint32_t det_mask;
  orc_hits *hits; orc_counters *C; uint64_t *hash; double *e_escape;
} ctx_t;

static void record_hit(ctx_t *c, uint64_t history, uint32_t ids, int photon, int *seq, const panel_t *P,
                       const double xl[3], double e_dep, double path) {
  double x[3]; to_global(P, xl, NULL, x, NULL);                      /* [R22] hits carry global xyz */
  int s = *seq < 15 ? *seq : 15; ++*seq;                             /* [R9] 4-bit saturating       */
  orc_hits *h = c->hits; c->C->hits++;
  if (h->n < h->capacity) {
    uint64_t i = h->n;
    h->history[i] = (uint32_t)history; h->ids[i] = ids | ((uint32_t)photon << 4) | (uint32_t)s;
    h->x[i] = (float)x[0]; h->y[i] = (float)x[1]; h->z[i] = (float)x[2];
    h->e[i] = (float)e_dep; h->tof[i] = (float)(path / ORC_C_MM_NS);
  }
  h->n++;
}

/* Compton kinematics shared by phantom and detector: returns E' and rotates d */
static double compton(ctx_t *c, rng_t *r, double E, double d[3]) {
  double ct, s2, ua; int n; double eps = kn_sample(r, E, &ct, &s2, &n, &ua); c->C->kn_trials += (uint64_t)n;
  double cp, sp; azimuth(ua, &cp, &sp);
  orc_rotate(d, ct, sqrt(s2), cp, sp);
  return eps * E;
}

static void transport_photon(ctx_t *c, uint64_t seed, uint64_t history, int photon, double x[3], double d[3], int in_phantom) {
  rng_t r; rng_init(&r, seed, history, photon ? STREAM_B : STREAM_A);
  double E = 511.0, path = 0.0; int seq = 0; uint64_t *h = c->hash;
  const orc_source *S = c->S; const orc_materials *M = c->M; const geom_t *g = c->g;
  double e_left = E;                                                 /* for the energy-conservation pin */

  /* [R17] phantom: Woodcock tracking in the voxel grid */
  if (in_phantom) {
    for (;;) {
      double mu_maj = mu_total(M, S->phantom_majorant, E);
      double u[4]; rng_next_block(&r, u);                            /* [R4] free path, outcome, Rayleigh polar, azimuth */
      double s = -log(u[0]) / mu_maj; c->C->ph_steps++;
      /* [R17] tentative collision point; outside the grid: no collision happens before the grid face and vacuum
       * lies beyond it, so the photon leaves along its line of flight FROM ITS CURRENT POINT (the
       * escaping gamma is taken to its panel along that line) -- it is not moved by the overshooting step */
      double xt[3]; int v[3], out = 0;
      for (int k = 0; k < 3; ++k) {
        xt[k] = x[k] + s * d[k];
        v[k] = (int)floor((xt[k] - (double)S->origin[k]) / (double)S->voxel[k]); if (v[k] < 0 || v[k] >= S->dims[k]) out = 1;
      }
      if (out) { if (h) hash_ev(h, EV_PH_LEAVE, 0); break; }
      for (int k = 0; k < 3; ++k) x[k] = xt[k];
      path += s;
      int mat = (int)S->phantom[((size_t)v[2] * S->dims[1] + v[1]) * S->dims[0] + v[0]] - 1;
      if (mat < 0) continue;                                        /* vacuum voxel: virtual, no draw */
      mu3_t mu = mu_lookup(M, mat, E); double t = u[1] * mu_maj;
      if (t < mu.pe) { c->C->ph_absorbed++; if (h) hash_ev(h, EV_PH_ABSORBED, 0); e_left = 0.0; goto done; }
      else if (t < mu.pe + mu.c) {
        E = compton(c, &r, E, d); c->C->ph_compton++; if (h) hash_ev(h, EV_PH_COMPTON, 0);
        if (E < ORC_CUTOFF) { c->C->ph_cutoff++; if (h) hash_ev(h, EV_PH_CUTOFF, 0); e_left = 0.0; goto done; }  /* [R28] */
        e_left = E;
      } else if (t < mu.pe + mu.c + mu.r) {
        double ct = orc_rayleigh_cos(u[2]), cp, sp; azimuth(u[3], &cp, &sp);
        orc_rotate(d, ct, sqrt(fmax(0.0, 1.0 - ct * ct)), cp, sp); if (h) hash_ev(h, EV_PH_RAYLEIGH, 0);
      }
    }
  }

  /* detector: panel search -> in-panel Woodcock loop -> exit -> search again */
  int excl = -1;
  double blo[3], bhi[3]; box_bounds(g, blo, bhi);
  for (;;) {
    double te; c->C->searches++;
    int p = panel_search(g, x, d, excl, &te);
    if (p < 0) { c->C->escapes++; if (h) hash_ev(h, EV_ESCAPE, 0); break; }
    const panel_t *P = &g->panel[p]; c->C->entries++; if (h) hash_ev(h, EV_ENTER, (uint32_t)p);
    double xl[3], dl[3]; to_local(P, x, d, xl, dl);
    for (int k = 0; k < 3; ++k) xl[k] += te * dl[k];                 /* [R18] move to the entry point */
    path += te;
    int alive = 1;
    int reg = 0;                                                     /* [R19] region of the entry point (by its depth) */
    for (int k = 1; k < g->n_regions; ++k) if (xl[2] >= (double)g->reg_c[k] / ORC_Q) reg = k;
    for (;;) {                                                       /* [R19] Woodcock tracking, one majorant per region */
      double mu_maj = mu_majorant(M, g->reg_mask[reg], E);
      double u[4]; rng_next_block(&r, u);                            /* [R4] free path, outcome, Rayleigh polar, azimuth */
      double s = -log(u[0]) / mu_maj, tfar[3], tf; c->C->steps++;
      double rlo[3] = { blo[0], blo[1], (double)g->reg_c[reg] / ORC_Q }, rhi[3] = { bhi[0], bhi[1], (double)g->reg_c[reg + 1] / ORC_Q };
      int kx = slab_far(rlo, rhi, xl, dl, tfar, &tf);                /* distance to the face of the region's slab that is met first */
      if (s >= tf) {
        if (tf < 0.0) tf = 0.0;
        for (int k = 0; k < 3; ++k) xl[k] += tf * dl[k];
        path += tf;
        /* a depth face that is not a face of the panel box: the photon crosses into the next region, analytically, and
         * draws a fresh free path there */
        if (kx == 2 && ((dl[2] >= 0.0 && reg + 1 < g->n_regions) || (dl[2] < 0.0 && reg > 0))) {
          reg += dl[2] >= 0.0 ? 1 : -1; c->C->region_crossings++; if (h) hash_ev(h, EV_REGION, (uint32_t)reg); continue;
        }
        c->C->exits++; if (h) hash_ev(h, EV_EXIT, (uint32_t)p); break;
      }
      for (int k = 0; k < 3; ++k) xl[k] += s * dl[k];
      path += s;
      uint32_t ids;                                                  /* PAPER.md:43 layer selection   */
      int mat = lattice_lookup(g, p, (int64_t)floor(xl[0] * ORC_Q) + g->hWq, (int64_t)floor(xl[1] * ORC_Q) + g->hHq,
                               (int64_t)floor(xl[2] * ORC_Q), &ids);
      if (mat < 0) { c->C->step_vacuum++; if (h) hash_ev(h, EV_STEP_VACUUM, 0); continue; }
      mu3_t mu = mu_lookup(M, mat, E); double t = u[1] * mu_maj;     /* [R20] one draw picks the outcome */
      if (t < mu.pe) {
        c->C->pe++; if (h) hash_ev(h, EV_PE, ids);
        if (ids != ORC_NONE) record_hit(c, history, ids, photon, &seq, P, xl, E, path);
        e_left = 0.0; alive = 0; break;
      } else if (t < mu.pe + mu.c) {
        double E2 = compton(c, &r, E, dl); c->C->compton++; if (h) hash_ev(h, EV_COMPTON, ids);
        if (E2 < ORC_CUTOFF) {                                      /* [R12] below cutoff: deposit all */
          c->C->cutoffs++; if (h) hash_ev(h, EV_CUTOFF, ids);
          if (ids != ORC_NONE) record_hit(c, history, ids, photon, &seq, P, xl, E, path);
          e_left = 0.0; alive = 0; break;
        }
        if (ids != ORC_NONE) record_hit(c, history, ids, photon, &seq, P, xl, E - E2, path);
        E = E2; e_left = E;
      } else if (t < mu.pe + mu.c + mu.r) {
        double ct = orc_rayleigh_cos(u[2]), cp, sp; azimuth(u[3], &cp, &sp);
        orc_rotate(dl, ct, sqrt(fmax(0.0, 1.0 - ct * ct)), cp, sp);
        c->C->rayleigh++; if (h) hash_ev(h, EV_RAYLEIGH, ids);
      } else { c->C->virtuals++; if (h) hash_ev(h, EV_VIRTUAL, ids); }
    }
    if (!alive) break;
    to_global(P, xl, dl, x, d);                                      /* [R33] leave: exclude this panel */
    excl = p;
  }
done:
  if (c->e_escape) c->e_escape[photon] = e_left;
}

/* [R13] decay site: the given point, or a voxel from the integer CDF + a uniform point inside it */
static void decay_site(const orc_source *S, rng_t *rs, double x0[3]) {
  x0[0] = S->pos[0]; x0[1] = S->pos[1]; x0[2] = S->pos[2];
  if (S->kind == 1) {
    uint64_t target = (uint64_t)(((unsigned __int128)rng_word_at(rs, 0) * S->w_total) >> 32), lo = 0, hi = S->n_active - 1;
    while (lo < hi) { uint64_t mid = (lo + hi) >> 1; if (S->act_cdf[mid] > target) hi = mid; else lo = mid + 1; }
    uint32_t vi = S->act_index[lo]; int v[3] = { (int)(vi % (uint32_t)S->dims[0]), (int)((vi / (uint32_t)S->dims[0]) % (uint32_t)S->dims[1]),
                                                 (int)(vi / ((uint32_t)S->dims[0] * (uint32_t)S->dims[1])) };
    for (int k = 0; k < 3; ++k)
      x0[k] = (double)S->origin[k] + ((double)v[k] + orc_uniform(rng_word_at(rs, 1 + (uint32_t)k))) * (double)S->voxel[k];
  }
}
/* [R35] positron range (PAPER.md:61 switches it off; PAPER.md:145 quotes 0.102 mm FWHM for 18F): the annihilation point
 * is the emission site plus an isotropic Gaussian displacement of the given FWHM per axis -- three normal deviates by
 * Box-Muller from words 12-15 of the source stream [R3] */
static void positron_range(const orc_source *S, rng_t *rs, double x0[3]) {
  if (!(S->positron_fwhm_mm > 0.0f)) return;
  double sg = (double)S->positron_fwhm_mm / ORC_FWHM, c1, s1, c2, s2;
  double r1 = sqrt(-2.0 * log(orc_uniform(rng_word_at(rs, 12)))), r2 = sqrt(-2.0 * log(orc_uniform(rng_word_at(rs, 14))));
  azimuth(orc_uniform(rng_word_at(rs, 13)), &c1, &s1); azimuth(orc_uniform(rng_word_at(rs, 15)), &c2, &s2);
  x0[0] += sg * r1 * c1; x0[1] += sg * r1 * s1; x0[2] += sg * r2 * c2;
}
void orc_annihilation_sites(const orc_source *S, uint64_t seed, uint64_t first, uint64_t n, double *xyz) {   /* test hook */
  for (uint64_t i = 0; i < n; ++i) { rng_t rs; rng_init(&rs, seed, first + i, STREAM_SOURCE); decay_site(S, &rs, xyz + 3 * i); positron_range(S, &rs, xyz + 3 * i); }
}
void orc_decay_sites(const orc_source *S, uint64_t seed, uint64_t first, uint64_t n, double *xyz) {   /* test hook */
  for (uint64_t i = 0; i < n; ++i) { rng_t rs; rng_init(&rs, seed, first + i, STREAM_SOURCE); decay_site(S, &rs, xyz + 3 * i); }
}

/* ------------------------------------------------------------------ one history (pair) */
static void simulate_history(ctx_t *c, uint64_t seed, uint64_t history) {
  const orc_source *S = c->S; rng_t rs; rng_init(&rs, seed, history, STREAM_SOURCE);
  double x0[3]; decay_site(S, &rs, x0);
  positron_range(S, &rs, x0);
  /* [R14] isotropic direction */
  double ct = 1.0 - 2.0 * orc_uniform(rng_word_at(&rs, 4)), st = sqrt(fmax(0.0, 1.0 - ct * ct)), cp, sp;
  azimuth(orc_uniform(rng_word_at(&rs, 5)), &cp, &sp);
  double dA[3] = { st * cp, st * sp, ct };
  if (S->kind == 2) {                                                /* pencil beam (deterministic test rays) */
    double nb = sqrt((double)S->beam_dir[0] * S->beam_dir[0] + (double)S->beam_dir[1] * S->beam_dir[1] + (double)S->beam_dir[2] * S->beam_dir[2]);
    for (int k = 0; k < 3; ++k) dA[k] = (double)S->beam_dir[k] / nb;
  }
  double dB[3] = { -dA[0], -dA[1], -dA[2] };
  if (S->acol_fwhm_deg > 0.0f) {                                     /* [R15] 2-D Gaussian deviation of photon B */
    double sigma = (double)S->acol_fwhm_deg * (ORC_PI / 180.0) / ORC_FWHM;
    double rho = sigma * sqrt(-2.0 * log(orc_uniform(rng_word_at(&rs, 6)))), c2, s2;
    azimuth(orc_uniform(rng_word_at(&rs, 7)), &c2, &s2);
    orc_rotate(dB, cos(rho), sin(rho), c2, s2);
  }
  int in_ph = (S->kind == 1 && S->phantom != NULL);
  double xa[3] = { x0[0], x0[1], x0[2] }, xb[3] = { x0[0], x0[1], x0[2] };
  c->C->pairs++;
  uint64_t *hh = c->hash;                                            /* [R23] one hash per photon */
  if (hh) { hh[0] = hh[1] = 0xCBF29CE484222325ull; }
  transport_photon(c, seed, history, 0, xa, dA, in_ph);
  if (hh) c->hash = hh + 1;
  transport_photon(c, seed, history, 1, xb, dB, in_ph);
  c->hash = hh;
}

static uint32_t detector_mask(const geom_t *g) {
  uint32_t m = 0;
  for (int l = 0; l < g->n_layers; ++l) { m |= 1u << g->layer[l].cmat; if (g->layer[l].gmat >= 0) m |= 1u << g->layer[l].gmat; }
  return m;
}

/* Simulate histories [first, first + n).  hash_out (2n, optional: photon A, photon B) and e_escape (2n,
 * optional) are per photon.  Hits come out in canonical (history, photon, sequence) order. */
int orc_simulate(const orc_geometry *gd, const orc_materials *M, orc_source *S, uint64_t first, uint64_t n,
                 uint64_t seed, orc_hits *hits, uint64_t *hash_out, double *e_escape, orc_counters *counters) {
  geom_t g; int rc = geom_build(gd, &g); if (rc) { geom_free(&g); return rc; }
  orc_counters C; memset(&C, 0, sizeof C);
  ctx_t c = { &g, M, S, detector_mask(&g), hits, &C, NULL, NULL };
  hits->n = 0;
  for (uint64_t i = 0; i < n; ++i) {
    c.hash = hash_out ? hash_out + 2 * i : NULL; c.e_escape = e_escape ? e_escape + 2 * i : NULL;
    simulate_history(&c, seed, first + i);
  }
  if (counters) *counters = C;
  geom_free(&g); return 0;
}

/* ------------------------------------------------------------------ digitizer [R24-R27] */
static int level_shift(int level) { return level == 0 ? 5 : (level == 1 ? 20 : 26); }   /* crystal/module/panel */

typedef struct { uint32_t history, unit; uint64_t idx; } hkey_t;
static int cmp_hkey(const void *a, const void *b) {
  const hkey_t *p = (const hkey_t *)a, *q = (const hkey_t *)b;
  if (p->history != q->history) return p->history < q->history ? -1 : 1;
  if (p->unit != q->unit) return p->unit < q->unit ? -1 : 1;
  return p->idx < q->idx ? -1 : (p->idx > q->idx);
}
typedef struct { double t; uint32_t history, unit; uint64_t idx; } tkey_t;
static int cmp_tkey(const void *a, const void *b) {
  const tkey_t *p = (const tkey_t *)a, *q = (const tkey_t *)b;
  if (p->t != q->t) return p->t < q->t ? -1 : 1;
  if (p->history != q->history) return p->history < q->history ? -1 : 1;
  if (p->unit != q->unit) return p->unit < q->unit ? -1 : 1;
  return 0;
}

/* hits (any order) -> kept singles (time-sorted) -> coincidences.  n_pairs_total and the source give
 * the decay times [R16].  Returns 0; counts exceeding a capacity are reported in ->n (records dropped). */
int orc_digitize(const orc_source *S, uint64_t seed, uint64_t n_pairs_total, const orc_hits *hits, uint64_t n_hits,
                 const orc_digitizer *D, orc_singles *singles, orc_coinc *coinc, uint64_t *n_singles_all) {
  int sh = level_shift(D->level);
  hkey_t *hk = (hkey_t *)malloc(sizeof(hkey_t) * (n_hits ? n_hits : 1));
  for (uint64_t i = 0; i < n_hits; ++i) { hk[i].history = hits->history[i]; hk[i].unit = hits->ids[i] >> sh; hk[i].idx = i; }
  qsort(hk, n_hits, sizeof(hkey_t), cmp_hkey);
  tkey_t *tk = (tkey_t *)malloc(sizeof(tkey_t) * (n_hits ? n_hits : 1));
  /* per-single scratch, indexed like tk */
  uint32_t *sid = (uint32_t *)malloc(4 * (n_hits ? n_hits : 1)); float *sx = (float *)malloc(4 * 4 * (n_hits ? n_hits : 1));
  uint64_t nk = 0, nall = 0;
  for (uint64_t i = 0; i < n_hits;) {
    uint64_t j = i;                                                 /* [R24] adder over one (history, unit) group */
    double e_sum = 0.0, e_best = -1.0, tof_min = INFINITY; uint64_t best = 0; uint32_t best_ord = 0;
    while (j < n_hits && hk[j].history == hk[i].history && hk[j].unit == hk[i].unit) {
      uint64_t k = hk[j].idx; double e = hits->e[k]; uint32_t ord = hits->ids[k] & 31u;  /* (photon, seq) */
      e_sum += e;
      if (e > e_best || (e == e_best && ord < best_ord)) { e_best = e; best = k; best_ord = ord; }
      if (hits->tof[k] < tof_min) tof_min = hits->tof[k];
      ++j;
    }
    ++nall;
    /* [R25] blur: sigma = (R/2.3548) sqrt(E_ref E) (or R/2.3548 E when ref = 0); Box-Muller, stream 3, block = unit */
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) }, ctr[4] = { hk[i].history, 0, STREAM_DIGI, hk[i].unit }, w[4];
    orc_philox4x32_10(ctr, key, w);
    double nrm = sqrt(-2.0 * log(orc_uniform(w[0]))) * cos(2.0 * ORC_PI * orc_uniform(w[1]));
    double sigma = (double)D->fwhm_frac / ORC_FWHM * (D->ref_keV > 0.0f ? sqrt((double)D->ref_keV * e_sum) : e_sum);
    double e_b = e_sum + sigma * nrm;
    if (e_b >= (double)D->e_lo && e_b < (double)D->e_hi) {          /* [R26] window */
      double t = orc_decay_time(S, seed, hk[i].history, n_pairs_total) + tof_min * 1e-9;
      tk[nk].t = t; tk[nk].history = hk[i].history; tk[nk].unit = hk[i].unit; tk[nk].idx = nk;
      sid[nk] = hits->ids[best]; sx[4 * nk] = hits->x[best]; sx[4 * nk + 1] = hits->y[best]; sx[4 * nk + 2] = hits->z[best];
      sx[4 * nk + 3] = (float)e_b; ++nk;
    }
    i = j;
  }
  if (n_singles_all) *n_singles_all = nall;
  qsort(tk, nk, sizeof(tkey_t), cmp_tkey);                          /* [R27] sort by (t, history, unit) */
  singles->n = nk;
  for (uint64_t i = 0; i < nk && i < singles->capacity; ++i) {
    uint64_t k = tk[i].idx;
    singles->history[i] = tk[i].history; singles->ids[i] = sid[k]; singles->x[i] = sx[4 * k]; singles->y[i] = sx[4 * k + 1];
    singles->z[i] = sx[4 * k + 2]; singles->e[i] = sx[4 * k + 3]; singles->t[i] = tk[i].t;
  }
  /* [R27] coincidence windows: an unconsumed single opens a window; members are the following singles
   * with t - t_open < tau; all members are consumed; exactly two members on different panels -> one pair */
  double tau = D->window_ns * 1e-9; uint64_t nc = 0;
  for (uint64_t i = 0; i < nk;) {
    uint64_t j = i + 1; while (j < nk && tk[j].t - tk[i].t < tau) ++j;
    if (j - i == 2) {
      uint64_t a = tk[i].idx, b = tk[i + 1].idx;
      if ((sid[a] >> 26) != (sid[b] >> 26)) {
        if (nc < coinc->capacity) {
          coinc->ids_a[nc] = sid[a]; coinc->ids_b[nc] = sid[b]; coinc->history_a[nc] = tk[i].history; coinc->history_b[nc] = tk[i + 1].history;
          coinc->e_a[nc] = sx[4 * a + 3]; coinc->e_b[nc] = sx[4 * b + 3];
          coinc->dt_ns[nc] = (float)((tk[i + 1].t - tk[i].t) * 1e9); coinc->t[nc] = tk[i].t;
        }
        ++nc;
      }
    }
    i = j;
  }
  coinc->n = nc;
  free(hk); free(tk); free(sid); free(sx);
  return 0;
}

/* ------------------------------------------------------------------ small exported helpers for the pins */
int orc_panel_box(const orc_geometry *d, double lo[3], double hi[3]) {
  geom_t g; int rc = geom_build(d, &g); if (!rc) box_bounds(&g, lo, hi); geom_free(&g); return rc;
}
int orc_panel_search(const orc_geometry *d, const double x[3], const double dir[3], int excl, double *t_enter) {
  geom_t g; int rc = geom_build(d, &g); if (rc) { geom_free(&g); return -2; }
  int p = panel_search(&g, x, dir, excl, t_enter); geom_free(&g); return p;
}
