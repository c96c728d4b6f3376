/* gpet.h -- C ABI of libgpet: GPU Monte Carlo transport of 511 keV annihilation photon pairs through a
 * parameterised panel -> module -> layer -> crystal PET detector, plus the singles digitizer and
 * coincidence sorter.  Hot path of "Extending gPET for Multi-Layer PET Simulation" (arxiv 2603.07327),
 * written for NVIDIA B200 (sm_100a).  Citations are PAPER.md:<line>; "[Rn]" is a reading in DESIGN.md 2.
 *
 * Conventions
 *  - Every call returns GPET_OK (0) or a negative GPET_E_* code; gpet_last_error() gives the text.
 *  - Handles (geometry, materials, activity) are created and destroyed by the library and are immutable.
 *  - All bulk device memory (hit / singles / coincidence buffers, scratch, phantom map) is owned by the
 *    caller and passed as raw *device* pointers; pointers marked HOST are host memory.
 *  - gpet_simulate and gpet_digitize only enqueue work on `cuda_stream` (a cudaStream_t, NULL = default
 *    stream) and return; argument errors are reported synchronously.
 *  - Lengths are millimetres, energies keV, hit times ns, absolute times seconds.
 *  - There is no CPU fallback: without a CUDA device every compute call returns GPET_E_CUDA.
 */
#ifndef GPET_H
#define GPET_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define GPET_OK              0
#define GPET_E_INVALID_ARG  -1   /* NULL pointer, count out of range                                   */
#define GPET_E_GEOMETRY     -2   /* lattice overhangs its module, non-positive size, too many panels  */
#define GPET_E_TABLE        -3   /* negative or non-finite mu, fewer than 2 energies                  */
#define GPET_E_OVERFLOW     -4   /* scratch too small, hits dropped in a library-owned buffer          */
#define GPET_E_CUDA         -5   /* CUDA runtime error or no device                                   */

#define GPET_MAX_PANELS   63
#define GPET_MAX_LAYERS    4
#define GPET_MAX_MATERIALS 8
#define GPET_IDS_NONE 0xFFFFFFFFu /* packed ids of a point that is not inside a crystal */
#define GPET_HIT_CHUNK_PAIRS 512   /* pairs per chunk of the chunked hit layout (gpet_hits.chunk_fill) */

/* Packed ids [R9] (every interaction is labelled with crystal, layer, module, panel):
 *   bits 0-3 sequence (per-photon hit counter, saturating at 15), bit 4 photon (0 = A, 1 = B),
 *   bits 5-17 crystal (ix + nx*iy), bits 18-19 layer (0 = front), bits 20-25 module (mx + nmx*my),
 *   bits 26-31 panel. */
#define GPET_IDS_PANEL(ids)   ((ids) >> 26)
#define GPET_IDS_MODULE(ids)  (((ids) >> 20) & 63u)
#define GPET_IDS_LAYER(ids)   (((ids) >> 18) & 3u)
#define GPET_IDS_CRYSTAL(ids) (((ids) >> 5) & 8191u)
#define GPET_IDS_PHOTON(ids)  (((ids) >> 4) & 1u)
#define GPET_IDS_SEQ(ids)     ((ids) & 15u)

typedef struct gpet_geometry  gpet_geometry;
typedef struct gpet_materials gpet_materials;
typedef struct gpet_activity  gpet_activity;

/* ---------------------------------------------------------------- geometry (Fig. 1) */
typedef struct {                 /* one crystal layer, front (layer 0) to back        */
  int32_t n_crystals[2];         /* along local u (tangential) and v (axial)                           */
  float   pitch_mm[2];           /* crystal size + reflector gap                         */
  float   reflector_mm[2];       /* gap between neighbours; half on each side of a cell                */
  float   offset_mm[2];          /* lattice origin relative to the module's low corner                 */
  float   depth_mm;              /* radial thickness of the layer                                      */
  float   gap_before_mm;         /* inter-layer gap in front of this layer (vacuum)                    */
  int32_t crystal_material;      /* index into gpet_materials                                          */
  int32_t gap_material;          /* reflector / rim material, -1 = vacuum                              */
} gpet_layer_desc;

typedef struct {
  int32_t n_panels;              /* 1..GPET_MAX_PANELS                                                 */
  const float *panel_pose;       /* HOST. NULL = repetition mode: ring of n_panels about */
                                 /* z [R5]; else non-repetition mode: n_panels x 12 floats per panel:  */
                                 /* front-face centre xyz, then unit axes u (tangential), v (axial),   */
                                 /* w (depth, pointing into the detector), with u x v = w              */
  float   ring_inner_radius_mm;  /* repetition mode: distance of the front face from the z axis        */
  float   ring_first_angle_deg;  /* repetition mode: azimuth of panel 0                                */
  int32_t n_modules[2];          /* modules per panel along u, v (1..8 each, product <= 64)            */
  float   module_size_mm[2];
  float   module_pitch_mm[2];    /* size + spacing; inter-module gaps are vacuum                       */
  int32_t n_layers;              /* 1..GPET_MAX_LAYERS ("the number of layers")           */
  const gpet_layer_desc *layers; /* HOST, n_layers entries                                             */
} gpet_geometry_desc;

/* Builds the quantised descriptor [R7] and uploads it.  GPET_E_GEOMETRY if a lattice does not fit in
 * its module, a size is non-positive, or a count exceeds the packed-id ranges. */
int gpet_geometry_create(const gpet_geometry_desc *desc, gpet_geometry **out);
int gpet_geometry_destroy(gpet_geometry *g);
/* Copies the fp32 pose (12 floats, layout as panel_pose) of one panel to HOST memory. */
int gpet_geometry_panel_pose(const gpet_geometry *g, int32_t panel, float *pose12);
/* Faces of one panel box beyond which no other panel has a point (bit 2k + 1: the high face of local axis k, bit 2k:
 * the low face; k = 0 u, 1 v, 2 w).  A photon leaving through such a face escapes: gpet_simulate skips the panel search
 * for it, with the result the search would give.  Host-side query of what gpet_geometry_create derived. */
int gpet_geometry_open_faces(const gpet_geometry *g, int32_t panel, uint32_t *mask);
/* Bore radius of a planar detector (all panels share the axial range and have no axial tilt, e.g. any repetition-mode
 * ring): the smallest distance from the z axis to any panel box, minus 1 um; <= 0 when the detector is not planar or
 * the axis runs through a panel.  gpet_simulate drops, without a panel search, a photon inside the bore that passes an
 * axial end of the detector before it can reach this radius (the search would report that it escapes). */
int gpet_geometry_bore_radius(const gpet_geometry *g, float *radius_mm);
/* Point -> packed ids (GPET_IDS_NONE if the point is in no crystal) for n points; xyz_global and
 * packed_ids are HOST arrays (n x 3 floats, n words); runs on the device (synchronous).  The lowest-index
 * panel whose box contains the point decides.  Same lattice code as the transport kernel. */
int gpet_geometry_locate(const gpet_geometry *g, int64_t n, const float *xyz_global, uint32_t *packed_ids);

/* ---------------------------------------------------------------- materials (BASELINE.json configs[0]) */
/* mu_pe, mu_compton, mu_rayleigh: HOST [n_materials][n_energies] in 1/mm on the grid
 * e_min_keV + i*e_step_keV.  Staged on the device as interleaved fp32 {mu_pe, mu_pe+mu_C, mu_tot, 0}
 * per energy [R11]; photons never leave [e_min, e_min + (n_energies-1)*e_step]. */
int gpet_materials_load(int32_t n_materials, int32_t n_energies, float e_min_keV, float e_step_keV,
                        const float *mu_pe, const float *mu_compton, const float *mu_rayleigh,
                        gpet_materials **out);
int gpet_materials_destroy(gpet_materials *m);

/* ---------------------------------------------------------------- source */
/* Activity map -> active-voxel list with an integer cumulative weight [R13]. activity: HOST,
 * dims[0]*dims[1]*dims[2] floats, x fastest; voxels with activity > 0 are active. */
int gpet_activity_create(const float *activity, const int32_t dims[3], gpet_activity **out);
int gpet_activity_destroy(gpet_activity *a);

typedef struct {
  int32_t  kind;                  /* 0 point source, 1 activity map, 2 pencil beam (deterministic test rays) */
  float    pos_mm[3];             /* kinds 0, 2                                                         */
  float    beam_dir[3];           /* kind 2: direction of photon A (normalised by the library)          */
  float    acolinearity_fwhm_deg; /* 0 = exactly back to back [R15]                                     */
  double   activity_bq;           /* decay-time scale [R16]                                             */
  uint64_t pairs_per_time_slice;  /* 0 = all pairs in one slice [R16]                                   */
  const gpet_activity *activity_map;   /* kind 1                                                        */
  const uint8_t *phantom_material;/* DEVICE, kind 1, optional: dims voxels, 0 = vacuum, k = material k-1 */
  int32_t  phantom_majorant_material;  /* material whose mu_tot bounds every phantom voxel [R17]         */
  int32_t  dims[3];               /* nx, ny, nz of the activity / phantom grid                          */
  float    voxel_mm[3];
  float    origin_mm[3];          /* low corner of voxel (0,0,0)                                        */
  float    positron_fwhm_mm;      /* [R35] positron range: isotropic Gaussian displacement of the        */
                                  /* annihilation point, FWHM per axis; 0 = off, as in the paper         */
                                  /* (PAPER.md:145 quotes 0.102 mm for 18F)                 */
  double   half_life_s;           /* [R34] > 0: the source decays (18F, 1.6e8 atoms, 120 s): */
  double   duration_s;            /* activity_bq is the INITIAL activity, the run covers [0, duration_s] */
                                  /* and simulates n_pairs_total = gpet_decay_count(...) histories;      */
                                  /* 0 = constant activity [R16]                                         */
} gpet_source;

/* Expected number of decays of a source of initial activity activity_bq and half-life half_life_s over duration_s
 * seconds: A0 / lambda (1 - exp(-lambda T)), rounded to nearest (half_life_s = 0: A0 T).  This is the n_pairs_total of
 * a run with the decay law switched on [R34]. */
int gpet_decay_count(double activity_bq, double half_life_s, double duration_s, uint64_t *n_pairs);

/* ---------------------------------------------------------------- transport */
typedef struct {                  /* struct of arrays, DEVICE, caller-owned                             */
  uint32_t *history;              /* low 32 bits of the history id                                      */
  uint32_t *ids;                  /* packed ids                                                         */
  float    *x, *y, *z;            /* global position of the deposit                                     */
  float    *e_keV;                /* deposited energy                                                   */
  float    *tof_ns;               /* time of flight from the decay                                      */
  uint64_t  capacity;             /* entries in each array                                              */
  uint64_t *n_hits;               /* DEVICE counter; NOT reset by the library, so several calls append  */
  uint64_t *outcome_hash;         /* DEVICE, optional (NULL = off): 2*n_pairs words, [2*i + photon] =   */
                                  /* FNV-1a over that photon's ordered event codes [R23] (parity tool)  */
  uint32_t *chunk_fill;           /* DEVICE, optional (NULL = dense layout above).  CHUNKED layout: the  */
                                  /* batch's pairs are taken in chunks of GPET_HIT_CHUNK_PAIRS; with     */
                                  /* n_chunks = ceil(n_pairs / 512) and cap = capacity / n_chunks, the   */
                                  /* hits of chunk c occupy entries [c*cap, c*cap + min(fill[c], cap))   */
                                  /* of the seven arrays, in no particular order, and chunk_fill[c]      */
                                  /* counts them (n_chunks + 1 words, zeroed by the caller; the last     */
                                  /* word counts hits dropped because their chunk's region was full).    */
                                  /* Grouping the hits of nearby histories lets gpet_digitize sort each  */
                                  /* chunk in shared memory instead of scattering records through HBM.   */
                                  /* One gpet_simulate batch per buffer (no appending); cap <= 2048.     */
} gpet_hits;

/* Simulates histories [first_history, first_history + n_pairs): source -> (phantom) -> panel search ->
 * in-panel Woodcock tracking with layer selection -> PE / Compton / Rayleigh; every deposit inside a
 * crystal is appended to `hits`.  Hits past `capacity` are dropped but counted: *n_hits > capacity means
 * "re-run the same (seed, first_history, n_pairs) with a larger buffer" (bit-identical by construction:
 * every draw is a pure function of seed, history, stream and draw index [R1]).  Buffer order is
 * unspecified; (history, photon, sequence) is the canonical order.  n_pairs < 2^32. */
int gpet_simulate(const gpet_geometry *g, const gpet_materials *m, const gpet_source *src,
                  uint64_t first_history, uint64_t n_pairs, uint64_t seed, gpet_hits *hits, void *cuda_stream);

/* ---------------------------------------------------------------- digitizer */
typedef struct {
  float   blur_fwhm_frac;         /* energy resolution R (FWHM / E) at blur_ref_keV [R25]               */
  float   blur_ref_keV;           /* sigma = R/2.3548*sqrt(ref*E); 0 selects sigma = R/2.3548*E         */
  float   e_lo_keV, e_hi_keV;     /* keep lo <= E < hi [R26]                                            */
  double  window_ns;              /* coincidence window [R27]                                           */
  int32_t readout_level;          /* 0 crystal, 1 module, 2 panel                         */
} gpet_digitizer;

typedef struct {                  /* kept singles, time-sorted; DEVICE, caller-owned                    */
  uint32_t *history, *ids;        /* ids/xyz of the largest deposit of the group [R24]                  */
  float    *x, *y, *z;
  float    *e_keV;                /* blurred energy                                                     */
  double   *t_s;                  /* absolute time: decay time [R16] + earliest tof                     */
  uint64_t  capacity;
  uint64_t *n_singles;            /* DEVICE counter, written by the call                                */
} gpet_singles;

typedef struct {                  /* list-mode coincidences; DEVICE, caller-owned                       */
  uint32_t *ids_a, *ids_b;        /* a is the earlier single                                            */
  uint32_t *history_a, *history_b;/* different histories = random coincidence                           */
  float    *e_a, *e_b;
  float    *dt_ns;                /* t_b - t_a                                                          */
  double   *t_s;                  /* t_a                                                                */
  uint64_t  capacity;
  uint64_t *n_coinc;              /* DEVICE counter, written by the call                                */
} gpet_coincidences;

/* Bytes of device scratch gpet_digitize needs for a batch of n_pairs histories holding n_hits hits. */
size_t gpet_digitize_scratch_bytes(uint64_t n_pairs, uint64_t n_hits);

/* hits (any order) -> adder per (history, readout unit) -> blur -> window -> absolute time -> time sort
 * -> coincidence windows.  The hits must belong to histories [first_history, first_history + n_pairs)
 * (one gpet_simulate batch, or several appended ones).  n_hits <= 2^31 is a HOST-side upper bound on the
 * valid entries (it sizes the scratch; pass hits->capacity to avoid reading the counter back): the kernels
 * use min(*hits->n_hits, hits->capacity, n_hits), read on the device.  n_pairs_total (pairs of the whole run, all batches) and
 * src give the decay times [R16].  Output is deterministic: it does not depend on the order of `hits`.
 * Records past a capacity are dropped but counted.  singles_out may be NULL (coincidences only), or have
 * NULL arrays with a valid n_singles (count only).
 * Batches that lie inside one time slice or cover whole slices [R16] are time-sorted through fixed-size bucket regions
 * that assume decay times spread evenly over the batch's time range -- true for any batch gpet_simulate produced.  If a
 * region fills all the same (say, the hits of one slice presented as a batch of a hundred), the singles that found no room
 * are counted and the call sets BOTH *n_coinc and *n_singles to UINT64_MAX: the lists are incomplete, do not use them
 * (gpet_pipeline_collect returns GPET_E_OVERFLOW); digitize the histories that have hits as their own slice-aligned
 * batch, or a batch that ends inside a slice (it takes the counting path, which has no such limit). */
int gpet_digitize(const gpet_source *src, uint64_t seed, uint64_t n_pairs_total, uint64_t first_history,
                  uint64_t n_pairs, const gpet_hits *hits, uint64_t n_hits, const gpet_digitizer *dig,
                  void *scratch, size_t scratch_bytes, gpet_singles *singles_out,
                  gpet_coincidences *coinc_out, void *cuda_stream);

/* gpet_digitize for callers that cannot allocate device memory.
 * Who that is: a digitizer stage plugged into a host program that has already handed the whole GPU to its own memory
 * pool (a cudaMalloc for our scratch would fail, or steal from a budget the host fixed at start-up), and an acquisition
 * loop that digitizes time slice after time slice [R16] (PAPER.md:65 list-mode output) and cannot afford
 * cudaMalloc/cudaFree in the loop, because both may stall every stream of the device.  Such callers already own their
 * hit, singles and coincidence buffers; what they lack is the temporary workspace between them.
 * This call takes the same arguments as gpet_digitize minus the scratch pair and gives the same output; its workspace is
 * a fixed array of GPET_STATIC_SCRATCH_BYTES built into the library's device code.  The call itself runs no cudaMalloc,
 * cudaFree or other allocating routine.  What to know:
 *  - Limit: gpet_digitize_scratch_bytes(n_pairs, n_hits) must not exceed GPET_STATIC_SCRATCH_BYTES (about 128 B per hit
 *    + 8 B per pair: e.g. 3e5 pairs with room for 4.5e5 hits).  Larger batches are refused with GPET_E_OVERFLOW and a
 *    message that names both sizes, before any GPU work; split the run into smaller time slices or use gpet_digitize.
 *  - Cost: every GPU on which this process runs the digitizer kernels holds the array (64 MiB) until the process exits,
 *    used or not.
 *  - First call on each device: looks up the array's device address (and, like any first launch, makes CUDA load the
 *    kernels).  Make that first call during set-up, with the device current, before any stream capture begins.
 *  - One workspace per device, shared by every call and every stream: two calls whose GPU work overlaps (different
 *    streams, or different host threads without ordering between them) race on it and produce garbage.  Order them on
 *    one stream, or with events.
 *  - The array keeps what the previous call left in it; each call clears the parts that must start from zero itself
 *    (on cuda_stream, ahead of its kernels), so no clean-up between calls is needed. */
#define GPET_STATIC_SCRATCH_BYTES (64u << 20)
int gpet_digitize_static(const gpet_source *src, uint64_t seed, uint64_t n_pairs_total, uint64_t first_history,
                         uint64_t n_pairs, const gpet_hits *hits, uint64_t n_hits, const gpet_digitizer *dig,
                         gpet_singles *singles_out, gpet_coincidences *coinc_out, void *cuda_stream);

/* ---------------------------------------------------------------- end to end with HOST buffers */
typedef struct {                  /* HOST outputs (pinned memory recommended); any array may be NULL    */
  gpet_hits         hits;         /* n_hits / outcome_hash / counters here are HOST pointers            */
  gpet_singles      singles;
  gpet_coincidences coinc;
} gpet_host_outputs;

/* Whole path for one batch with host-side outputs: runs gpet_simulate + gpet_digitize on library-owned device
 * buffers sized hits_per_pair * n_pairs, copies the requested outputs to the HOST arrays (counts in *n_hits,
 * *n_singles, *n_coinc; capacities limit what is copied) and synchronises.  phantom_material inside src is a HOST
 * pointer here (copied to the device by the call).  The buffers are kept for the next call of the same shape
 * (gpet_shutdown frees them).  One batch at a time: for a stream of batches use the pipeline below. */
int gpet_run_host(const gpet_geometry *g, const gpet_materials *m, const gpet_source *src,
                  uint64_t n_pairs_total, uint64_t first_history, uint64_t n_pairs, uint64_t seed,
                  const gpet_digitizer *dig, double hits_per_pair, gpet_host_outputs *out);

/* ---------------------------------------------------------------- a stream of batches with HOST outputs */
/* The paper's runs are long acquisitions written out as list-mode coincidences ("list-mode output");
 * a run of N pairs is cut into batches (time slices [R16]) and each batch's list is copied to the host.  The pipeline
 * keeps TWO batches in flight: while the list-mode output of batch k crosses PCIe on a copy stream, batch k+1 is
 * transported and digitized on the compute stream, so the copy costs no time as long as it is shorter than a batch.
 *   gpet_pipeline_create(..., n_slots = 2, &p);
 *   gpet_pipeline_submit(p, first_0, n, seed);
 *   for k: gpet_pipeline_submit(p, first_{k+1}, n, seed);  gpet_pipeline_collect(p, &out_k);   // out_k = batch k
 *   gpet_pipeline_collect(p, &out_last);  gpet_pipeline_destroy(p);
 * Handles, geometry and materials must outlive the pipeline.  src->phantom_material is a HOST pointer (uploaded once by
 * create; voxel values above the number of loaded materials are rejected).  `want` says which outputs besides the
 * coincidences will be asked for (it sizes the device buffers): without GPET_WANT_HITS the hits stay on the device in
 * the chunked layout.  submit only enqueues work and returns; at most n_slots (1 or 2) batches may be in flight.
 * collect waits for the OLDEST batch in flight, copies its outputs to the HOST arrays of `out` (as gpet_run_host does;
 * pinned memory recommended) and returns its counts; GPET_E_OVERFLOW if the batch dropped hits (raise hits_per_pair). */
#define GPET_WANT_HITS    1u
#define GPET_WANT_SINGLES 2u
#define GPET_WANT_HASH    4u
typedef struct gpet_pipeline gpet_pipeline;
int gpet_pipeline_create(const gpet_geometry *g, const gpet_materials *m, const gpet_source *src, const gpet_digitizer *dig,
                         uint64_t n_pairs_total, uint64_t max_pairs_per_batch, double hits_per_pair, uint32_t want,
                         int32_t n_slots, gpet_pipeline **out);
int gpet_pipeline_submit(gpet_pipeline *p, uint64_t first_history, uint64_t n_pairs, uint64_t seed);
int gpet_pipeline_collect(gpet_pipeline *p, gpet_host_outputs *out);
int gpet_pipeline_destroy(gpet_pipeline *p);

/* Frees what the library keeps between calls (gpet_run_host's buffers, the work counters of gpet_simulate).  Handles
 * created by the caller stay valid; any later call re-creates what it needs. */
int gpet_shutdown(void);

/* Tuning: warps per transport CTA (one persistent CTA per SM), 1..20, 0 = default 20; returns the value in force.  Fewer
 * warps leave registers and thread slots on every SM for kernels of OTHER streams: with 16, gpet_digitize of batch k on
 * one stream runs beside gpet_simulate of batch k+1 on another (the transport kernel is bound by instruction issue, the
 * digitizer by HBM latency), which is how bench.py pipelines its steps.  Applies to later gpet_simulate calls. */
int gpet_set_transport_warps(int32_t warps);

/* Thread-local text of the last error on this thread; valid until the next call on this thread. */
const char *gpet_last_error(void);
/* Number of kernel launches this library has enqueued since load (for bench.py's gpu_launches). */
uint64_t gpet_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* GPET_H */
