// gf_internal.h — what gf_api.cu needs to know about the kernels in gf_kernels.cu (host-side declarations only).
#pragma once
#include <cuda_runtime.h>

#include "gf_device.cuh"

namespace gf {

struct KernelArgs {
  void* links;     // internal-layout link field (device)
  void* partials;  // double2 per measure block (device)
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
cudaError_t launch_halfsweep(const KernelArgs& a, int parity, double omega);
cudaError_t launch_measure(const KernelArgs& a);  // 2 kernel launches
cudaError_t launch_reunit(const KernelArgs& a);
int measure_num_partials(const Geo& g);

}  // namespace gf
