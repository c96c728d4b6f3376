// Test shim: exposes the library's own qdiv_make (paper_2603_07327_b200/csrc/gpet_device.cuh, the multiply-high division of
// the lattice lookup [R7] and of the voxel index [R13]) to the CPU tests by INCLUDING the header -- nothing is copied.
// Built by tests/test_abi.py with nvcc (host code only is called; no GPU needed).
#include "gpet_device.cuh"

extern "C" void qdiv_make_batch(const uint32_t *d, int n, uint32_t *magic, uint32_t *shift) {
  for (int i = 0; i < n; ++i) { const gpet::QDiv q = gpet::qdiv_make(d[i]); magic[i] = q.magic; shift[i] = q.shift; }
}
