// gf_kernels.cu — the CUDA kernels of libgf (sm_100a) and their launch wrappers.
//   reorder_in / reorder_out : canonical layout <-> internal AoSoA-32 layout          (gf_set_links / gf_get_links)
//   ovr_halfsweep            : one parity of the overrelaxation sweep                  (Algorithm 1 l.3-12)
//   measure_partial / _final : F and theta, two-stage deterministic reduction          (eqs. 1.1-1.3)
//   reunit                   : Gram-Schmidt reunitarisation of every link
#include "gf_device.cuh"
#include "gf_internal.h"

namespace gf {

// ======================================================================================================================
// canonical <-> internal
// ======================================================================================================================
// One thread per (site of one parity, mu).  Canonical link = 18 contiguous reals at ((lex*4+mu)*18).
template <class T, int NELEM, bool IN>
__global__ void __launch_bounds__(256) reorder_kernel(cplx_t<T>* __restrict__ internal, T* __restrict__ canon, Geo g,
                                                      long long lex_begin, long long lex_end,
                                                      const T* __restrict__ canon_chunk_base) {
  // thread -> (parity, cb, mu): mu fastest so that a thread group touches contiguous canonical memory
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int mu = (int)(tid & 3);
  const long long sid = tid >> 2;  // site number within the range, in canonical (lexicographic) order
  const long long lex = lex_begin + sid;
  if (lex >= lex_end) return;
  unsigned q = (unsigned)lex;
  const int x = q % (unsigned)g.n[0]; q /= (unsigned)g.n[0];
  const int y = q % (unsigned)g.n[1]; q /= (unsigned)g.n[1];
  const int z = q % (unsigned)g.n[2];
  const int t = q / (unsigned)g.n[2];
  const int parity = (x + y + z + t) & 1;
  const int cb = (int)(lex >> 1);
  cplx_t<T>* p = internal + link_offset<NELEM>(g, parity, cb, mu);
  // canonical pointer: either the full array (chunk_base == nullptr) or a staging chunk that starts at lex_begin
  T* c = canon_chunk_base ? const_cast<T*>(canon_chunk_base) + (sid * 4 + mu) * 18 : canon + (lex * 4 + mu) * 18;
  cplx_t<T> u[9];
  if (IN) {
    const cplx_t<T>* cc = reinterpret_cast<const cplx_t<T>*>(c);
#pragma unroll
    for (int e = 0; e < NELEM; ++e) u[e] = cc[e];
    store_link<NELEM>(p, u);
  } else {
    load_link<NELEM, true>(p, u);
    cplx_t<T>* cc = reinterpret_cast<cplx_t<T>*>(c);
#pragma unroll
    for (int e = 0; e < 9; ++e) cc[e] = u[e];
  }
}

template <class T, int NELEM>
static cudaError_t reorder_T(const KernelArgs& a, bool in, void* canon, long long lex_begin, long long lex_end,
                             const void* chunk_base) {
  const long long nthreads = (lex_end - lex_begin) * 4;
  if (nthreads <= 0) return cudaSuccess;
  const unsigned blocks = (unsigned)((nthreads + 255) / 256);
  if (in)
    reorder_kernel<T, NELEM, true><<<blocks, 256, 0, a.stream>>>((cplx_t<T>*)a.links, (T*)canon, a.geo, lex_begin,
                                                                 lex_end, (const T*)chunk_base);
  else
    reorder_kernel<T, NELEM, false><<<blocks, 256, 0, a.stream>>>((cplx_t<T>*)a.links, (T*)canon, a.geo, lex_begin,
                                                                  lex_end, (const T*)chunk_base);
  return cudaGetLastError();
}

cudaError_t launch_reorder(const KernelArgs& a, bool in, void* canon, long long lex_begin, long long lex_end,
                           const void* chunk_base) {
  if (a.prec == 0) return a.storage == 18 ? reorder_T<double, 9>(a, in, canon, lex_begin, lex_end, chunk_base)
                                          : reorder_T<double, 6>(a, in, canon, lex_begin, lex_end, chunk_base);
  return a.storage == 18 ? reorder_T<float, 9>(a, in, canon, lex_begin, lex_end, chunk_base)
                         : reorder_T<float, 6>(a, in, canon, lex_begin, lex_end, chunk_base);
}

// ======================================================================================================================
// overrelaxation half-sweep, variant 0: one thread per site, two passes over the site's eight links
// ======================================================================================================================
// Pass 1 streams the 2*ND links that enter K(x) (eq. 1.5) and sums them in registers; the three SU(2) steps give
// G(x); pass 2 re-reads each of the eight links (L1/L2 hit: same thread, same addresses, nothing written between),
// multiplies and stores in place.  Same-parity sites touch disjoint links, so there is no inter-thread hazard.
template <class T, int NELEM, int ND, int THREADS, int MINBLOCKS>
__global__ void __launch_bounds__(THREADS, MINBLOCKS)
ovr_halfsweep_kernel(cplx_t<T>* __restrict__ links, Geo g, int parity, T omega) {
  using C = cplx_t<T>;
  const int cb = blockIdx.x * THREADS + threadIdx.x;
  if (cb >= g.vh) return;
  const Site s = site_of(g, parity, cb);
  C* fwd = links + link_offset<NELEM>(g, parity, cb, 0);  // + mu*NELEM*32 for direction mu
  C* bwd[4];
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) bwd[mu] = links + link_offset<NELEM>(g, parity ^ 1, cb_down(g, s, cb, mu), mu);

  C K[9];
#pragma unroll
  for (int e = 0; e < 9; ++e) K[e] = mk<T>(T(0), T(0));
#pragma unroll
  for (int mu = 0; mu < ND; ++mu) {
    C u[9];
    load_link<NELEM, true>(fwd + mu * NELEM * 32, u);
#pragma unroll
    for (int e = 0; e < 9; ++e) { K[e].x += u[e].x; K[e].y += u[e].y; }
    load_link<NELEM, true>(bwd[mu], u);
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = 0; j < 3; ++j) { K[i * 3 + j].x += u[j * 3 + i].x; K[i * 3 + j].y -= u[j * 3 + i].y; }
  }

  C G[9];
  site_gauge_rotation<T>(K, G, omega);

#pragma unroll
  for (int mu = 0; mu < 4; ++mu) {
    C u[9], w[9];
    load_link<NELEM, true>(fwd + mu * NELEM * 32, u);
    mul_left<NELEM / 3>(G, u, w);                       // U_mu(x) <- G U_mu(x)
    store_link<NELEM>(fwd + mu * NELEM * 32, w);
    load_link<NELEM, false>(bwd[mu], u);
    mul_right_adj<NELEM / 3>(u, G, w);                  // U_mu(x-mu) <- U_mu(x-mu) G^dagger
    store_link<NELEM>(bwd[mu], w);
  }
}

template <class T, int NELEM, int ND>
static cudaError_t halfsweep_T(const KernelArgs& a, int parity, double omega) {
  constexpr int THREADS = 128;
  const unsigned blocks = (unsigned)((a.geo.vh + THREADS - 1) / THREADS);
  ovr_halfsweep_kernel<T, NELEM, ND, THREADS, 1><<<blocks, THREADS, 0, a.stream>>>((cplx_t<T>*)a.links, a.geo, parity,
                                                                                  (T)omega);
  return cudaGetLastError();
}

cudaError_t launch_halfsweep(const KernelArgs& a, int parity, double omega) {
  const bool coul = a.gauge == 1;
  if (a.prec == 0) {
    if (a.storage == 18) return coul ? halfsweep_T<double, 9, 3>(a, parity, omega) : halfsweep_T<double, 9, 4>(a, parity, omega);
    return coul ? halfsweep_T<double, 6, 3>(a, parity, omega) : halfsweep_T<double, 6, 4>(a, parity, omega);
  }
  if (a.storage == 18) return coul ? halfsweep_T<float, 9, 3>(a, parity, omega) : halfsweep_T<float, 9, 4>(a, parity, omega);
  return coul ? halfsweep_T<float, 6, 3>(a, parity, omega) : halfsweep_T<float, 6, 4>(a, parity, omega);
}

// ======================================================================================================================
// F and theta
// ======================================================================================================================
// One thread per site (both parities).  Per site: f = sum_{mu<ND} Re Tr U_mu(x);  A = sum_{nu<ND} [U_nu(x-nu) - U_nu(x)];
// Delta = (A - A^dag) - (1/3) Tr(A - A^dag);  q = sum_ij |Delta_ij|^2   (eqs. 1.1-1.3, readings A1, A2).
// Block partials by warp shuffles (FP64), one double2 per block; a single-block second stage adds them in index order.
constexpr int MEASURE_THREADS = 256;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

template <class T, int NELEM, int ND>
__global__ void __launch_bounds__(MEASURE_THREADS) measure_partial_kernel(const cplx_t<T>* __restrict__ links, Geo g,
                                                                          double2* __restrict__ partials) {
  using C = cplx_t<T>;
  const int blocks_per_parity = gridDim.x >> 1;
  const int parity = blockIdx.x >= blocks_per_parity;
  const int cb = (blockIdx.x - parity * blocks_per_parity) * MEASURE_THREADS + threadIdx.x;
  double f = 0.0, q = 0.0;
  if (cb < g.vh) {
    const Site s = site_of(g, parity, cb);
    const C* fwd = links + link_offset<NELEM>(g, parity, cb, 0);
    C A[9];
#pragma unroll
    for (int e = 0; e < 9; ++e) A[e] = mk<T>(T(0), T(0));
    T tr = T(0);
#pragma unroll
    for (int nu = 0; nu < ND; ++nu) {
      C u[9];
      load_link<NELEM, true>(links + link_offset<NELEM>(g, parity ^ 1, cb_down(g, s, cb, nu), nu), u);
#pragma unroll
      for (int e = 0; e < 9; ++e) { A[e].x += u[e].x; A[e].y += u[e].y; }
      load_link<NELEM, true>(fwd + nu * NELEM * 32, u);
#pragma unroll
      for (int e = 0; e < 9; ++e) { A[e].x -= u[e].x; A[e].y -= u[e].y; }
      tr += u[0].x + u[4].x + u[8].x;
    }
    f = (double)tr;
    // D = A - A^dag: D_ii = 2i Im A_ii; D_ij = A_ij - conj(A_ji);  traceless part: D_ii -= (1/3) sum_k D_kk
    const T d0 = T(2) * A[0].y, d1 = T(2) * A[4].y, d2 = T(2) * A[8].y;
    const T m = (d0 + d1 + d2) / T(3);
    T acc = (d0 - m) * (d0 - m) + (d1 - m) * (d1 - m) + (d2 - m) * (d2 - m);
    // off-diagonal: |D_ij|^2 = |D_ji|^2, so count each pair twice
    {
      const T ax = A[1].x - A[3].x, ay = A[1].y + A[3].y; acc += T(2) * (ax * ax + ay * ay);
      const T bx = A[2].x - A[6].x, by = A[2].y + A[6].y; acc += T(2) * (bx * bx + by * by);
      const T cx = A[5].x - A[7].x, cy = A[5].y + A[7].y; acc += T(2) * (cx * cx + cy * cy);
    }
    q = (double)acc;
  }
  __shared__ double sf[MEASURE_THREADS / 32], sq[MEASURE_THREADS / 32];
  f = warp_sum(f);
  q = warp_sum(q);
  if ((threadIdx.x & 31) == 0) { sf[threadIdx.x >> 5] = f; sq[threadIdx.x >> 5] = q; }
  __syncthreads();
  if (threadIdx.x < 32) {
    f = threadIdx.x < MEASURE_THREADS / 32 ? sf[threadIdx.x] : 0.0;
    q = threadIdx.x < MEASURE_THREADS / 32 ? sq[threadIdx.x] : 0.0;
    f = warp_sum(f);
    q = warp_sum(q);
    if (threadIdx.x == 0) partials[blockIdx.x] = make_double2(f, q);
  }
}

// second stage: one block of 1024 threads; thread i adds partials i, i+1024, ... in order; fixed tree afterwards
__global__ void __launch_bounds__(1024) measure_final_kernel(const double2* __restrict__ partials, int n, double norm_f,
                                                             double norm_q, double* __restrict__ result) {
  double f = 0.0, q = 0.0;
  for (int i = threadIdx.x; i < n; i += 1024) { f += partials[i].x; q += partials[i].y; }
  __shared__ double sf[32], sq[32];
  f = warp_sum(f);
  q = warp_sum(q);
  if ((threadIdx.x & 31) == 0) { sf[threadIdx.x >> 5] = f; sq[threadIdx.x >> 5] = q; }
  __syncthreads();
  if (threadIdx.x < 32) {
    f = warp_sum(sf[threadIdx.x]);
    q = warp_sum(sq[threadIdx.x]);
    if (threadIdx.x == 0) { result[0] = f * norm_f; result[1] = q * norm_q; }
  }
}

int measure_num_partials(const Geo& g) { return 2 * ((g.vh + MEASURE_THREADS - 1) / MEASURE_THREADS); }

template <class T, int NELEM, int ND>
static cudaError_t measure_T(const KernelArgs& a) {
  const int nblk = measure_num_partials(a.geo);
  measure_partial_kernel<T, NELEM, ND><<<nblk, MEASURE_THREADS, 0, a.stream>>>((const cplx_t<T>*)a.links, a.geo,
                                                                              (double2*)a.partials);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  const double V = 2.0 * (double)a.geo.vh;
  measure_final_kernel<<<1, 1024, 0, a.stream>>>((const double2*)a.partials, nblk, 1.0 / (ND * 3.0 * V),
                                                 1.0 / (3.0 * V), (double*)a.result);
  return cudaGetLastError();
}

cudaError_t launch_measure(const KernelArgs& a) {
  const bool coul = a.gauge == 1;
  if (a.prec == 0) {
    if (a.storage == 18) return coul ? measure_T<double, 9, 3>(a) : measure_T<double, 9, 4>(a);
    return coul ? measure_T<double, 6, 3>(a) : measure_T<double, 6, 4>(a);
  }
  if (a.storage == 18) return coul ? measure_T<float, 9, 3>(a) : measure_T<float, 9, 4>(a);
  return coul ? measure_T<float, 6, 3>(a) : measure_T<float, 6, 4>(a);
}

// ======================================================================================================================
// reunitarisation
// ======================================================================================================================
// One thread per stored link: the internal array is a sequence of (block, mu) tiles of NELEM*32 complex numbers.
template <class T, int NELEM>
__global__ void __launch_bounds__(256) reunit_kernel(cplx_t<T>* __restrict__ links, long long ntiles) {
  using C = cplx_t<T>;
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long tile = tid >> 5;
  if (tile >= ntiles) return;
  C* p = links + (size_t)tile * NELEM * 32 + (tid & 31);
  C u[9];
  load_link<NELEM, false>(p, u);
  // padding lanes of the last block hold zeros: leave them alone (0/0)
  if (u[0].x == T(0) && u[0].y == T(0) && u[1].x == T(0) && u[1].y == T(0) && u[2].x == T(0) && u[2].y == T(0)) return;
  reunitarize<T>(u);
  store_link<NELEM>(p, u);
}

template <class T, int NELEM>
static cudaError_t reunit_T(const KernelArgs& a) {
  const long long ntiles = 2LL * a.geo.nblk * 4;
  const unsigned blocks = (unsigned)((ntiles * 32 + 255) / 256);
  reunit_kernel<T, NELEM><<<blocks, 256, 0, a.stream>>>((cplx_t<T>*)a.links, ntiles);
  return cudaGetLastError();
}

cudaError_t launch_reunit(const KernelArgs& a) {
  if (a.prec == 0) return a.storage == 18 ? reunit_T<double, 9>(a) : reunit_T<double, 6>(a);
  return a.storage == 18 ? reunit_T<float, 9>(a) : reunit_T<float, 6>(a);
}

}  // namespace gf
