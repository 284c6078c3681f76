// gf_static.cu — gf_measure_static: F (eq. 1.1) and theta (eqs. 1.2-1.3) of a link field in the canonical layout, for
// callers that may not allocate device memory.
//
// Who that is.  Everything else in libgf works out of a workspace the caller allocates (gf_create).  Some callers have
// no way to get one: a monitoring hook inside a lattice code whose memory pool already owns the whole HBM and hands out
// nothing to plug-ins; code running under a harness that forbids cudaMalloc after start-up because cudaMalloc and
// cudaFree synchronise the whole device and would stall the streams of the job next to it; a callback that only holds a
// pointer to somebody else's gauge field.  Such a caller still wants to ask "how far from the gauge is this field?".
// This entry point answers with nothing but the field pointer: the per-block partial sums of the two-stage reduction
// (the scratch gf_measure keeps in its workspace) live in a file-scope device array of fixed size instead.
//
// The price: the array is part of the library image, so every GPU that loads libgf holds its 256 KiB until the process
// exits; lattices above GF_STATIC_MAX_SITES sites do not fit and are refused; and all calls on one GPU share the one
// array, so two calls that overlap on the device (different streams, different threads) overwrite each other's
// partial sums.  Serialise them.
#include <cmath>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <mutex>

#include "../../include/gf.h"
#include "gf_device.cuh"

namespace {
using namespace gf;

constexpr int STATIC_THREADS = 256;        // sites per block = sites per partial sum
constexpr int STATIC_MAX_BLOCKS = 16384;   // partial sums the array holds
constexpr long long STATIC_MAX_SITES = (long long)STATIC_THREADS * STATIC_MAX_BLOCKS;  // 4 194 304 (e.g. 32^3 x 128)
constexpr int MAX_DEVICES = 64;

// [0, STATIC_MAX_BLOCKS): one (sum f, sum q) per block; [STATIC_MAX_BLOCKS]: the result (F, theta);
// [STATIC_MAX_BLOCKS + 1]: its first four bytes are the count of finished blocks, zero between calls.
// In HOST code this name is only a handle for cudaGetSymbolAddress: it is not a device address and must never be passed
// to a kernel as a pointer (scratch_of_current_device below asks the runtime for the address, once per device).
static __device__ __align__(256) double2 gf_static_scratch[STATIC_MAX_BLOCKS + 2];

struct StaticGeo {
  int n[4];
  long long V;
};

// sum_ij |Delta_ij|^2 with Delta = (A - A^dag) - (1/3) Tr(A - A^dag)   (eq. 1.3; reading A2 in DESIGN.md)
__device__ __forceinline__ double static_delta_norm2(const double2 (&A)[9]) {
  const double d0 = 2.0 * A[0].y, d1 = 2.0 * A[4].y, d2 = 2.0 * A[8].y;  // diagonal of A - A^dag is 2i Im A_ii
  const double m = (d0 + d1 + d2) / 3.0;
  double acc = (d0 - m) * (d0 - m) + (d1 - m) * (d1 - m) + (d2 - m) * (d2 - m);
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = i + 1; j < 3; ++j) {  // |D_ij|^2 = |D_ji|^2
      const double x = A[i * 3 + j].x - A[j * 3 + i].x, y = A[i * 3 + j].y + A[j * 3 + i].y;
      acc += 2.0 * (x * x + y * y);
    }
  return acc;
}

// One thread per site, sites in the canonical (lexicographic) order.  f = sum_{nu<ND} Re Tr U_nu(x) (each link counted
// at the site it starts from); A = sum_{nu<ND} [U_nu(x-nu) - U_nu(x)], q = |Delta(x)|^2.  Sums in FP64 whatever T is.
// Block partials by warp shuffles; the block that finishes last adds them in index order, so the result does not
// depend on the order in which blocks ran.
template <class T, int ND>
__global__ void __launch_bounds__(STATIC_THREADS) measure_static_kernel(const cplx_t<T>* __restrict__ links, StaticGeo g,
                                                                       double2* __restrict__ scratch, double norm_f,
                                                                       double norm_q) {
  const long long site = (long long)blockIdx.x * STATIC_THREADS + threadIdx.x;
  double f = 0.0, q = 0.0;
  if (site < g.V) {
    int c[4];
    long long r = site;
#pragma unroll
    for (int d = 0; d < 4; ++d) { c[d] = (int)(r % g.n[d]); r /= g.n[d]; }
    double2 A[9];
#pragma unroll
    for (int e = 0; e < 9; ++e) A[e] = make_double2(0.0, 0.0);
    long long stride = 1;
#pragma unroll
    for (int nu = 0; nu < ND; ++nu) {
      const long long down = c[nu] == 0 ? site + stride * (g.n[nu] - 1) : site - stride;
      const cplx_t<T>* up = links + (site * 4 + nu) * 9;
      const cplx_t<T>* um = links + (down * 4 + nu) * 9;
#pragma unroll
      for (int e = 0; e < 9; ++e) {
        const cplx_t<T> a = um[e], b = up[e];
        A[e].x += (double)a.x - (double)b.x;
        A[e].y += (double)a.y - (double)b.y;
        if (e % 4 == 0) f += (double)b.x;
      }
      stride *= g.n[nu];
    }
    q = static_delta_norm2(A);
  }
  block_sum2<STATIC_THREADS>(f, q);
  unsigned* counter = reinterpret_cast<unsigned*>(scratch + STATIC_MAX_BLOCKS + 1);
  __shared__ bool last;
  if (threadIdx.x == 0) {
    scratch[blockIdx.x] = make_double2(f, q);
    __threadfence();
    last = atomicAdd(counter, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  f = 0.0; q = 0.0;
  for (int i = threadIdx.x; i < (int)gridDim.x; i += STATIC_THREADS) {
    const double2 p = __ldcg(scratch + i);
    f += p.x; q += p.y;
  }
  __syncthreads();  // block_sum2's shared words were read by the first stage
  block_sum2<STATIC_THREADS>(f, q);
  if (threadIdx.x == 0) {
    scratch[STATIC_MAX_BLOCKS] = make_double2(f * norm_f, q * norm_q);
    *counter = 0u;
  }
}

thread_local char g_err[256] = "";
int fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}

// The device address of gf_static_scratch on the CURRENT device, asked from the runtime the first time this device is
// seen (every device has its own copy of the array, at its own address).
std::mutex g_mutex;
double2* g_scratch[MAX_DEVICES] = {};
int scratch_of_current_device(double2** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(GF_ECUDA, "gf_measure_static: cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= MAX_DEVICES) return fail(GF_EUNSUPPORTED, "gf_measure_static: device ordinal %d >= %d", dev, MAX_DEVICES);
  std::lock_guard<std::mutex> lock(g_mutex);
  if (!g_scratch[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, gf_static_scratch);
    if (e != cudaSuccess || !p)
      return fail(GF_ECUDA, "gf_measure_static: cudaGetSymbolAddress on device %d: %s", dev, cudaGetErrorString(e));
    g_scratch[dev] = static_cast<double2*>(p);
  }
  *out = g_scratch[dev];
  return GF_OK;
}

template <class T>
cudaError_t launch(const void* links, const StaticGeo& g, int gauge, double2* scratch, cudaStream_t s) {
  const unsigned blocks = (unsigned)((g.V + STATIC_THREADS - 1) / STATIC_THREADS);
  const double V = (double)g.V;
  if (gauge == GF_COULOMB)
    measure_static_kernel<T, 3><<<blocks, STATIC_THREADS, 0, s>>>((const cplx_t<T>*)links, g, scratch,
                                                                  1.0 / (3 * 3.0 * V), 1.0 / (3.0 * V));
  else
    measure_static_kernel<T, 4><<<blocks, STATIC_THREADS, 0, s>>>((const cplx_t<T>*)links, g, scratch,
                                                                  1.0 / (4 * 3.0 * V), 1.0 / (3.0 * V));
  return cudaGetLastError();
}
}  // namespace

extern "C" {

size_t gf_measure_static_max_sites(void) { return (size_t)STATIC_MAX_SITES; }

const char* gf_static_last_error(void) { return g_err; }

int gf_measure_static(const void* dev_links, int nx, int ny, int nz, int nt, int gauge, int prec, void* cuda_stream,
                      double* F, double* theta) {
  g_err[0] = 0;
  if (!dev_links || !F || !theta) return fail(GF_EINVAL, "gf_measure_static: null pointer");
  if (gauge != GF_LANDAU && gauge != GF_COULOMB) return fail(GF_EUNSUPPORTED, "gf_measure_static: unknown gauge %d", gauge);
  if (prec != GF_FP64 && prec != GF_FP32) return fail(GF_EUNSUPPORTED, "gf_measure_static: unknown precision %d", prec);
  StaticGeo g;
  g.n[0] = nx; g.n[1] = ny; g.n[2] = nz; g.n[3] = nt;
  g.V = 1;
  for (int d = 0; d < 4; ++d) {
    if (g.n[d] < 2 || (g.n[d] & 1)) return fail(GF_EODD, "gf_measure_static: extent %d is odd or < 2", g.n[d]);
    g.V *= g.n[d];
    if (g.V > STATIC_MAX_SITES)
      return fail(GF_ENOMEM,
                  "gf_measure_static: %d x %d x %d x %d exceeds the %lld sites the static scratch array holds partial "
                  "sums for; use gf_create + gf_measure with a workspace",
                  nx, ny, nz, nt, STATIC_MAX_SITES);
  }
  if ((uintptr_t)dev_links % 16 != 0) return fail(GF_EINVAL, "gf_measure_static: dev_links must be 16-byte aligned");
  int dev = -1;
  cudaPointerAttributes attr;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaPointerGetAttributes(&attr, dev_links);
  if (e != cudaSuccess) return fail(GF_ECUDA, "gf_measure_static: %s", cudaGetErrorString(e));
  if ((attr.type != cudaMemoryTypeDevice && attr.type != cudaMemoryTypeManaged) ||
      (attr.type == cudaMemoryTypeDevice && attr.device != dev))
    return fail(GF_EINVAL, "gf_measure_static: dev_links is not device memory of the current device (%d)", dev);

  double2* scratch = nullptr;
  if (int rc = scratch_of_current_device(&scratch); rc != GF_OK) return rc;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  // The finished-blocks count must be zero when the kernel starts.  The kernel leaves it so, but a call that was cut
  // short (a launch that failed half-way, a device reset by another library) would not: clear it every time.
  e = cudaMemsetAsync(scratch + STATIC_MAX_BLOCKS + 1, 0, sizeof(double2), s);
  if (e == cudaSuccess) e = prec == GF_FP64 ? launch<double>(dev_links, g, gauge, scratch, s)
                                            : launch<float>(dev_links, g, gauge, scratch, s);
  double r[2] = {0.0, 0.0};
  if (e == cudaSuccess) e = cudaMemcpyAsync(r, scratch + STATIC_MAX_BLOCKS, sizeof(r), cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) return fail(GF_ECUDA, "gf_measure_static: %s", cudaGetErrorString(e));
  *F = r[0];
  *theta = r[1];
  if (!std::isfinite(r[0]) || !std::isfinite(r[1])) return fail(GF_ENUMERIC, "gf_measure_static: non-finite F or theta");
  return GF_OK;
}

}  // extern "C"
