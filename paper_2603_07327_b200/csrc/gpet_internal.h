// gpet_internal.h -- declarations shared by the library's translation units (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "gpet_device.cuh"

namespace gpet {

struct HitBuf {            // device view of gpet_hits
  uint32_t *history, *ids; float *x, *y, *z, *e, *tof;
  unsigned long long capacity; unsigned long long *n_hits;
  uint32_t *chunk_fill;      // chunked layout (gpet.h): hits of pairs [512 c, 512 (c+1)) of the batch at [c cap, c cap + fill[c])
  uint32_t chunk_cap, n_chunks;
};
constexpr uint32_t kActGuideBits = 16, kActGuide = 1u << kActGuideBits;
constexpr uint32_t kHitChunkPairs = 512, kHitChunkShift = 9, kHitChunkCapMax = 2048;

struct DevSource {
  int kind; float pos[3], beam[3]; float acol_sigma;            // radians
  float acol_sin_max, acol_cos_max;                              // sin / cos of the largest acolinearity deviation that can be drawn
  const uint32_t *act_index; const uint64_t *act_cdf; uint32_t n_active; uint64_t w_total;
  QDiv div_nx, div_nxy;                                          // voxel index -> (ix, iy, iz) without integer divisions
  const uint32_t *act_guide;                                     // [R13] kActGuide + 1 entries: where the cdf search of a voxel-pick word starts and ends
  const uint8_t *phantom; int ph_major; int dims[3]; float voxel[3], inv_voxel[3], origin[3];
  double activity_bq; uint64_t pairs_per_slice;
  float positron_sigma;                                          // [R35] mm per axis, 0 = off
  uint32_t pre_klo, pre_khi;                                     // point-source pre-test: pairs whose polar word >> 9 lies outside [pre_klo, pre_khi] miss with both photons (set per launch)
};

struct DigiParams {
  float sigma_scale;       // R / 2.3548
  float ref_keV, e_lo, e_hi; double window_s; int shift;         // ids >> shift = readout unit
  double activity_bq, slice_s; uint64_t pairs_per_slice; uint64_t seed;   // slice_s = pairs_per_slice / activity_bq
  double lambda, pfrac, q_scale;                                 // [R34] decay law: ln2 / half-life (0 = constant activity), 1 - exp(-lambda T), B / N
  uint64_t n_pairs_total;                                        // pairs of the whole run
  uint64_t cut_slice; double cut_frac;                           // [R34] the run's last slice when it is cut short (N mod B != 0; else ~0): it covers only cut_frac = (N mod B) / B of a slice
  PhiloxKeys keys;                                               // [R1] the ten round keys of `seed`
};

struct SinglesBuf { uint32_t *history, *ids; float *x, *y, *z, *e; double *t; unsigned long long capacity; unsigned long long *n; };
struct CoincBuf { uint32_t *ids_a, *ids_b, *history_a, *history_b; float *e_a, *e_b, *dt_ns; double *t;
                  unsigned long long capacity; unsigned long long *n; };

void count_launch(uint64_t n = 1);

void set_transport_warps(int warps);
int transport_warps();
int transport_warps_that_fit(const DevGeom &host_geom, const DevTables &T, const DevSource &src, bool hash, size_t smem_limit);
cudaError_t launch_transport(const DevGeom &host_geom, const DevGeom *geom, const DevTables &T, const DevSource &src,
                             uint64_t first_history, uint64_t n_pairs, uint64_t seed, const HitBuf &H, uint64_t *hash_out,
                             unsigned long long *work_counter, int sm_count, int warps, cudaStream_t stream);
cudaError_t launch_locate(const DevGeom *geom, int64_t n, const float *xyz_dev, uint32_t *ids_dev, cudaStream_t stream);

size_t digitize_scratch_bytes(uint64_t n_pairs, uint64_t n_hits);
cudaError_t launch_digitize(const DigiParams &P, const HitBuf &H, uint64_t first_history, uint64_t n_pairs, uint64_t n_hits,
                            void *scratch, size_t scratch_bytes, const SinglesBuf &S, const CoincBuf &C, cudaStream_t stream);
// Device address and size of the library's built-in digitizer scratch on the CURRENT device (allocates nothing).
cudaError_t static_digitize_scratch(void **ptr, size_t *bytes);

}  // namespace gpet
