// Device build of the synthetic gauge-field generator (see gen_core.h for the recipe).  Input tooling only: it
// lets the 4-19 GB fields of the large configurations be fabricated straight in HBM instead of on the host.
#include "gen_core.h"

#include <cuda_runtime.h>

using namespace gfin;

struct Dims { int n[4]; };

template <class T>
__global__ void gfin_links_kernel(T* __restrict__ out, Dims d, double r, uint64_t seed, int64_t V) {
  int64_t site = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (site >= V) return;
  m3 g0 = gauge_at(seed, (uint64_t)site);
  for (int mu = 0; mu < 4; ++mu) {
    m3 g1 = gauge_at(seed, (uint64_t)neighbour_up(site, mu, d.n));
    m3 e = smooth_link(seed, (uint64_t)site, mu, r);
    store_link(out + (site * 4 + mu) * 18, finish_link(g0, e, g1));
  }
}

extern "C" int gfin_links_device(void* dev_out, const int* dims, double roughness, uint64_t seed, int prec,
                                 void* cuda_stream) {
  if (!dev_out || !dims) return -1;
  Dims d;
  int64_t V = 1;
  for (int i = 0; i < 4; ++i) { d.n[i] = dims[i]; V *= dims[i]; }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  unsigned blocks = (unsigned)((V + 127) / 128);
  if (prec == 0) gfin_links_kernel<double><<<blocks, 128, 0, st>>>((double*)dev_out, d, roughness, seed, V);
  else if (prec == 1) gfin_links_kernel<float><<<blocks, 128, 0, st>>>((float*)dev_out, d, roughness, seed, V);
  else return -1;
  return cudaGetLastError() == cudaSuccess ? 0 : -2;
}
