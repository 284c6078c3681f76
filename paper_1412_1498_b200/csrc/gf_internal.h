// gf_internal.h — what gf_api.cu needs to know about the kernels in gf_kernels.cu (host-side declarations only).
#pragma once
#include <cuda_runtime.h>

#include "gf_device.cuh"

namespace gf {

struct KernelArgs {
  void* links;     // internal-layout link field (device)
  void* partials;  // double2 per measure block (device)
  void* qpartials; // double per half-sweep block: theta terms left by a fused odd half-sweep (device)
  void* result;    // 2 doubles: F, theta (device)
  Geo geo;
  cudaStream_t stream;
  int prec;     // 0 = FP64, 1 = FP32
  int storage;  // 18 or 12
  int gauge;    // 0 = Landau, 1 = Coulomb
  int variant;  // half-sweep kernel variant (GF_OPT_SWEEP_VARIANT)
  int block_threads;
};

// canonical <-> internal for the lexicographic site range [lex_begin, lex_end).  If chunk_base is non-null the canonical
// data of that range starts at chunk_base (a staging buffer); otherwise `canon` is the full canonical array.
cudaError_t launch_reorder(const KernelArgs& a, bool in, void* canon, long long lex_begin, long long lex_end,
                           const void* chunk_base);
// fuse_theta: the launch also leaves the updated sites' theta terms in a.qpartials[0..*qblocks) (only kernels for which
// halfsweep_can_fuse_theta(a) holds; *qblocks = 0 otherwise)
cudaError_t launch_halfsweep(const KernelArgs& a, int parity, double omega, bool fuse_theta, int* qblocks);
bool halfsweep_can_fuse_theta(const KernelArgs& a);
int halfsweep_max_qblocks(const Geo& g);
// 2 kernel launches.  nq > 0: a.qpartials[0..nq) hold the odd sites' theta terms of the links as they stand, so only
// the even sites are visited (every link read once); nq = 0: all sites are visited.
cudaError_t launch_measure(const KernelArgs& a, int nq);
cudaError_t launch_reunit(const KernelArgs& a);
int measure_num_partials(const Geo& g);

}  // namespace gf
