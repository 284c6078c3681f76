// gf_fftsd.cu — Algorithm 2 of arXiv:1412.1498: steepest descent with Fourier acceleration (eqs.
// 1.7-1.9; Algorithm 2).  Kernels, cuFFT plans and launch wrappers; the driver loop is in gf_api.cu.
//
//   sd_delta    : Delta(x) of eq. 1.3 for every site, packed, plus the F / theta block partials (Alg. 2 l.1, l.17)
//   cuFFT       : forward transform of the packed fields                                        (l.4)
//   sd_filter   : multiply by (alpha/2) (p^2_max / p^2) / N                                     (l.5, l.7, eq. 1.8)
//   cuFFT       : backward transform                                                            (l.6)
//   sd_rotate   : g(x) = reunitarise(1 + w(x)); U_mu(x) <- g(x) U_mu(x) g(x+mu)^dagger          (l.9-15)
//
// What differs from the paper (N x N x (4-D FFT + 4-D IFFT), 6 with the 12-real parametrisation):
// Delta(x) is anti-Hermitian and traceless, i.e. 8 real numbers per site, and the Fourier factor p^2_max/p^2 is real
// and even in p, so its x-space kernel is real: it filters the real and the imaginary part of a complex field
// independently and keeps the anti-Hermitian structure.  The three upper off-diagonal elements (complex) and the pair
// (Im Delta_00) + i (Im Delta_11) are therefore transformed as FOUR complex fields — 4 transform pairs per
// iteration instead of 9 (or 6); the rest of w(x) follows from w_ji = -conj(w_ij), Im w_22 = -(Im w_00 + Im w_11).
// The 4-D transform (cuFFT has no rank 4) is a batched 3-D transform of every time slice followed by
// a strided batched 1-D transform along t; in Coulomb gauge only the 3-D part runs (time slices are independent).
#include <cufft.h>

#include <cstdio>

#include "gf_device.cuh"
#include "gf_internal.h"

namespace gf {

// ---- small helpers ----------------------------------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum_d(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// lexicographic index of the site (parity, cb) and of its forward neighbours (periodic)
__device__ __forceinline__ int lex_of(const Geo& g, const Site& s) {
  return s.x + g.n[0] * (s.y + g.n[1] * (s.z + g.n[2] * s.t));
}
__device__ __forceinline__ int lex_up(const Geo& g, const Site& s, int lex, int mu) {
  switch (mu) {
    case 0: return s.x == g.n[0] - 1 ? lex - (g.n[0] - 1) : lex + 1;
    case 1: return s.y == g.n[1] - 1 ? lex - g.n[0] * (g.n[1] - 1) : lex + g.n[0];
    case 2: return s.z == g.n[2] - 1 ? lex - g.n[0] * g.n[1] * (g.n[2] - 1) : lex + g.n[0] * g.n[1];
    default: return s.t == g.n[3] - 1 ? lex - g.n[0] * g.n[1] * g.n[2] * (g.n[3] - 1) : lex + g.n[0] * g.n[1] * g.n[2];
  }
}

// ======================================================================================================================
// Delta(x), packed, + F / theta partials
// ======================================================================================================================
// One thread per checkerboard index cb: it handles the two sites (parity 0 and parity 1) that share cb.  They are
// neighbours in x (lex = 2 cb and 2 cb + 1), so the thread writes two consecutive entries of each packed field.
// A = sum_{nu<ND} [U_nu(x-nu) - U_nu(x)];  Delta = (A - A^dag) - (1/3) Tr(A - A^dag)       (eq. 1.3, readings A2, B1)
// packed fields: 0: Delta_01, 1: Delta_02, 2: Delta_12, 3: Im Delta_00 + i Im Delta_11.
// f = sum over the parity-0 sites of Re Tr [U_nu(x) + U_nu(x-nu)] (= every link once);  q = sum_ij |Delta_ij|^2.
constexpr int SD_THREADS = 128;

// Block order.  A site's t-neighbours are one time slice away in cb order (151 MB of links on 64^3 x 128: more than
// L2), so in launch order the temporal links would come from HBM twice.  When a time slice is a whole number of
// blocks, blocks are renumbered so that a chunk of 1/16 slice runs through all t before the next chunk starts: the
// reuse distance in t drops to two chunks (a few MB) and the second use hits L2.
struct BlockOrder {
  int per_slice;  // blocks per time slice (0: identity order)
  int chunk;      // blocks per chunk
  int nt;
};
__device__ __forceinline__ int ordered_block(const BlockOrder& o, int b) {
  if (o.per_slice == 0) return b;
  const int span = o.nt * o.chunk;
  const int c = b / span, r = b - c * span;
  const int t = r / o.chunk, k = r - t * o.chunk;
  return t * o.per_slice + c * o.chunk + k;
}
static BlockOrder make_block_order(const Geo& g) {
  BlockOrder o{0, 0, g.n[3]};
  const int slice_cb = g.vh / g.n[3];
  if (slice_cb % SD_THREADS) return o;
  o.per_slice = slice_cb / SD_THREADS;
  o.chunk = o.per_slice % 16 == 0 ? o.per_slice / 16 : o.per_slice;
  return o;
}

// The anti-Hermitian part of A is all Delta needs: 3 imaginary diagonal parts and 3 complex upper off-diagonals
// (9 reals per site instead of the 18 of A), plus Re Tr for F.
template <class T, class C>
struct AntiHerm {
  T d0, d1, d2, tr;
  C o01, o02, o12;
  __device__ __forceinline__ void clear() {
    d0 = d1 = d2 = tr = T(0);
    o01 = o02 = o12 = mk<T>(T(0), T(0));
  }
  // += sign * (u - u^dag) / (diagonal: Im u_ii; the factor 2 is applied at the end), tr += Re Tr u
  template <int SIGN>
  __device__ __forceinline__ void add(const C (&u)[9]) {
    const T s = T(SIGN);
    d0 += s * u[0].y; d1 += s * u[4].y; d2 += s * u[8].y;
    o01.x += s * (u[1].x - u[3].x); o01.y += s * (u[1].y + u[3].y);
    o02.x += s * (u[2].x - u[6].x); o02.y += s * (u[2].y + u[6].y);
    o12.x += s * (u[5].x - u[7].x); o12.y += s * (u[5].y + u[7].y);
    tr += u[0].x + u[4].x + u[8].x;
  }
  // packed Delta and sum_ij |Delta_ij|^2
  __device__ __forceinline__ T finish(C (&d)[4]) const {
    T a0 = T(2) * d0, a1 = T(2) * d1, a2 = T(2) * d2;
    const T m = (a0 + a1 + a2) / T(3);
    a0 -= m; a1 -= m; a2 -= m;
    d[0] = o01; d[1] = o02; d[2] = o12; d[3] = mk<T>(a0, a1);
    return a0 * a0 + a1 * a1 + a2 * a2 +
           T(2) * (o01.x * o01.x + o01.y * o01.y + o02.x * o02.x + o02.y * o02.y + o12.x * o12.x + o12.y * o12.y);
  }
};

// Both sites of a pair are advanced direction by direction, so that the two uses of a link (as U_nu(x) of one site
// and as U_nu(x'-nu) of its neighbour x' = x+nu) fall at the same point of the program in neighbouring threads and
// the second one finds the line in L2.
template <class T, int NELEM, int ND>
__global__ void __launch_bounds__(SD_THREADS) sd_delta_kernel(const cplx_t<T>* __restrict__ links, Geo g,
                                                              cplx_t<T>* __restrict__ w, double2* __restrict__ partials,
                                                              BlockOrder order) {
  using C = cplx_t<T>;
  const int blk = ordered_block(order, blockIdx.x);
  const int cb = blk * SD_THREADS + threadIdx.x;
  double f = 0.0, q = 0.0;
  if (cb < g.vh) {
    const size_t V = 2 * (size_t)g.vh;
    const Site s0 = site_of(g, 0, cb), s1 = site_of(g, 1, cb);
    const int first = s0.x & 1;  // parity-0 site sits at lex = 2 cb + first, the parity-1 site at the other one
    const C* fwd0 = links + link_offset<NELEM>(g, 0, cb, 0);
    const C* fwd1 = links + link_offset<NELEM>(g, 1, cb, 0);
    AntiHerm<T, C> a0, a1;
    a0.clear();
    a1.clear();
#pragma unroll
    for (int nu = 0; nu < ND; ++nu) {
      C u[9];
      load_link<NELEM, true>(fwd0 + nu * NELEM * 32, u);
      a0.template add<-1>(u);
      load_link<NELEM, true>(fwd1 + nu * NELEM * 32, u);
      a1.template add<-1>(u);
      load_link<NELEM, true>(links + link_offset<NELEM>(g, 1, cb_down(g, s0, cb, nu), nu), u);
      a0.template add<1>(u);
      load_link<NELEM, true>(links + link_offset<NELEM>(g, 0, cb_down(g, s1, cb, nu), nu), u);
      a1.template add<1>(u);
    }
    C de[4], dodd[4];
    const T q0 = a0.finish(de), q1 = a1.finish(dodd);
    f = (double)a0.tr;
    q = (double)q0 + (double)q1;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      C* p = w + k * V + 2 * (size_t)cb;
      p[first] = de[k];
      p[first ^ 1] = dodd[k];
    }
  }
  f = warp_sum_d(f);
  q = warp_sum_d(q);
  __shared__ double sf[SD_THREADS / 32], sq[SD_THREADS / 32];
  if ((threadIdx.x & 31) == 0) { sf[threadIdx.x >> 5] = f; sq[threadIdx.x >> 5] = q; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double F = 0.0, Q = 0.0;
#pragma unroll
    for (int i = 0; i < SD_THREADS / 32; ++i) { F += sf[i]; Q += sq[i]; }
    partials[blk] = make_double2(F, Q);
  }
}

// one block: partial sums in index order, then a fixed tree (deterministic)
__global__ void __launch_bounds__(1024) sd_final_kernel(const double2* __restrict__ partials, int n, double norm_f,
                                                        double norm_q, double* __restrict__ result) {
  double f = 0.0, q = 0.0;
  for (int i = threadIdx.x; i < n; i += 1024) { f += partials[i].x; q += partials[i].y; }
  f = warp_sum_d(f);
  q = warp_sum_d(q);
  __shared__ double sf[32], sq[32];
  if ((threadIdx.x & 31) == 0) { sf[threadIdx.x >> 5] = f; sq[threadIdx.x >> 5] = q; }
  __syncthreads();
  if (threadIdx.x < 32) {
    f = warp_sum_d(sf[threadIdx.x]);
    q = warp_sum_d(sq[threadIdx.x]);
    if (threadIdx.x == 0) { result[0] = f * norm_f; result[1] = q * norm_q; }
  }
}

// ======================================================================================================================
// Fourier factor
// ======================================================================================================================
// table[off_mu + k] = 4 sin^2(pi k / n_mu)  (reading B2), FP64 in both precisions
__global__ void sd_table_kernel(double* __restrict__ table, int nx, int ny, int nz, int nt) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  int k = i, n = nx;
  if (k >= nx) { k -= nx; n = ny; if (k >= ny) { k -= ny; n = nz; if (k >= nz) { k -= nz; n = nt; if (k >= nt) return; } } }
  const double s = sinpi((double)k / (double)n);
  table[i] = 4.0 * s * s;
}

// w~(p) *= scale * p2max / p^2(p), 0 at p = 0 (reading B3); scale = (alpha/2) / N (reading B4).  One thread per
// momentum, all four fields.
template <class T, int ND>
__global__ void __launch_bounds__(256) sd_filter_kernel(cplx_t<T>* __restrict__ w, Geo g, const double* __restrict__ table,
                                                        double scale_p2max) {
  const size_t V = 2 * (size_t)g.vh;
  const size_t i = (size_t)blockIdx.x * 256 + threadIdx.x;
  if (i >= V) return;
  unsigned q = (unsigned)i;
  const int kx = q % (unsigned)g.n[0]; q /= (unsigned)g.n[0];
  const int ky = q % (unsigned)g.n[1]; q /= (unsigned)g.n[1];
  const int kz = q % (unsigned)g.n[2];
  const int kt = q / (unsigned)g.n[2];
  double p2 = table[kx] + table[g.n[0] + ky] + table[g.n[0] + g.n[1] + kz];
  if (ND == 4) p2 += table[g.n[0] + g.n[1] + g.n[2] + kt];
  const T fac = p2 > 0.0 ? (T)(scale_p2max / p2) : T(0);
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    cplx_t<T> v = w[k * V + i];
    v.x *= fac; v.y *= fac;
    w[k * V + i] = v;
  }
}

// eq. 1.7 (no Fourier factor): w *= alpha/2
template <class T>
__global__ void __launch_bounds__(256) sd_scale_kernel(cplx_t<T>* __restrict__ w, size_t n, T fac) {
  const size_t i = (size_t)blockIdx.x * 256 + threadIdx.x;
  if (i >= n) return;
  cplx_t<T> v = w[i];
  v.x *= fac; v.y *= fac;
  w[i] = v;
}

// ======================================================================================================================
// t direction: forward transform, Fourier factor and inverse transform in ONE pass (Landau gauge, n_t a power of two)
// ======================================================================================================================
// The factor is diagonal in 4-D momentum space and the transforms along different axes commute, so after the 3-D
// transform of every time slice the remaining work per spatial momentum (kx,ky,kz) is: transform the n_t numbers along
// t, multiply by (alpha/2) p^2_max / p^2 / N, transform back.  A block takes TLINE_XB consecutive x of one field and
// keeps their t-lines in shared memory: one read and one write of the field instead of three of each (cuFFT's strided
// 1-D transform, sd_filter, cuFFT's inverse) and one launch instead of nine.
// Radix-2: decimation in time on a bit-reversed load (natural-order output for the factor), then decimation in
// frequency for the inverse (bit-reversed output, undone by the store).  Thread (j, b): x offset j, butterfly b < n_t/2.
constexpr int TLINE_THREADS = 512;

template <class C> __device__ __forceinline__ C cmul_conj(const C a, const C b) {  // a * conj(b)
  C z; z.x = a.x * b.x + a.y * b.y; z.y = a.y * b.x - a.x * b.y; return z;
}

// XB consecutive x per block (XB * sizeof(complex) = 256 B contiguous per t);
// thread (j, b0): x offset j = tid % XB, butterflies b = b0, b0 + TLINE_THREADS/XB, ... < n_t/2.
template <class T, int XB>
__global__ void __launch_bounds__(TLINE_THREADS) sd_tline_kernel(cplx_t<T>* __restrict__ w, Geo g, int logn,
                                                                 const double* __restrict__ table, double scale_p2max) {
  using C = cplx_t<T>;
  extern __shared__ __align__(16) unsigned char tline_smem[];
  constexpr int BT = TLINE_THREADS / XB;
  const int n = g.n[3], nh = n / 2;
  C* data = reinterpret_cast<C*>(tline_smem);   // [n][XB]
  C* tw = data + n * XB;                        // [n/2]: exp(-2 pi i k / n)
  const int j = threadIdx.x % XB, b0 = threadIdx.x / XB;
  const size_t V3 = (size_t)g.n[0] * g.n[1] * g.n[2], V = V3 * n;
  const size_t s = (size_t)blockIdx.x * XB + j;  // spatial momentum index kx + nx (ky + ny kz)
  C* base = w + (size_t)blockIdx.y * V + s;
  for (int k = threadIdx.x; k < nh; k += TLINE_THREADS) {
    double sn, cs;
    sincospi(-2.0 * (double)k / (double)n, &sn, &cs);
    tw[k] = mk<T>((T)cs, (T)sn);
  }
  // bit-reversed load straight into shared memory (cp.async: every row of the block in flight at once)
  for (int e = b0; e < n; e += BT) {
    const unsigned dst = (unsigned)__cvta_generic_to_shared(data + (int)(__brev((unsigned)e) >> (32 - logn)) * XB + j);
    if (sizeof(C) == 16)
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(base + (size_t)e * V3) : "memory");
    else
      asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(base + (size_t)e * V3) : "memory");
  }
  asm volatile("cp.async.wait_all;" ::: "memory");
  __syncthreads();
  for (int st = 0; st < logn; ++st) {  // forward, decimation in time
    const int half = 1 << st;
    for (int b = b0; b < nh; b += BT) {
      const int pos = b & (half - 1), i0 = ((b >> st) << (st + 1)) + pos, i1 = i0 + half;
      const C t = tw[pos << (logn - 1 - st)];
      const C a = data[i0 * XB + j], c = cmul(data[i1 * XB + j], t);
      data[i0 * XB + j] = mk<T>(a.x + c.x, a.y + c.y);
      data[i1 * XB + j] = mk<T>(a.x - c.x, a.y - c.y);
    }
    __syncthreads();
  }
  {  // factor (readings B2-B4), natural order: entry e is k_t = e
    unsigned q = (unsigned)s;
    const int kx = q % (unsigned)g.n[0]; q /= (unsigned)g.n[0];
    const int ky = q % (unsigned)g.n[1];
    const int kz = q / (unsigned)g.n[1];
    const double p3 = table[kx] + table[g.n[0] + ky] + table[g.n[0] + g.n[1] + kz];
    const double* tt = table + g.n[0] + g.n[1] + g.n[2];
    for (int e = b0; e < n; e += BT) {
      const double p2 = p3 + tt[e];
      const T f = p2 > 0.0 ? (T)(scale_p2max / p2) : T(0);
      C v = data[e * XB + j];
      v.x *= f; v.y *= f;
      data[e * XB + j] = v;
    }
  }
  __syncthreads();
  for (int st = logn - 1; st >= 0; --st) {  // inverse, decimation in frequency
    const int half = 1 << st;
    for (int b = b0; b < nh; b += BT) {
      const int pos = b & (half - 1), i0 = ((b >> st) << (st + 1)) + pos, i1 = i0 + half;
      const C t = tw[pos << (logn - 1 - st)];
      const C a = data[i0 * XB + j], c = data[i1 * XB + j];
      data[i0 * XB + j] = mk<T>(a.x + c.x, a.y + c.y);
      data[i1 * XB + j] = cmul_conj(mk<T>(a.x - c.x, a.y - c.y), t);
    }
    __syncthreads();
  }
#pragma unroll 8
  for (int e = b0; e < n; e += BT) base[(size_t)(__brev((unsigned)e) >> (32 - logn)) * V3] = data[e * XB + j];
}

// can the fused t pass be used on this lattice?  (Landau gauge is the caller's business)
static int tline_xb(const Geo& g, int prec) {
  const long long V3 = (long long)g.n[0] * g.n[1] * g.n[2];
  const int want = prec == 0 ? 16 : 32;  // 256 B per t; smaller tiles = more blocks per SM to overlap load / butterfly / store phases
  for (int xb = want; xb >= 8; xb /= 2)
    if (V3 % xb == 0) return xb;
  return 0;
}
bool sd_tline_supported(const Geo& g) {
  const int n = g.n[3];
  return n >= 2 && n <= 256 && (n & (n - 1)) == 0 && tline_xb(g, 0) != 0;
}

template <class T, int XB>
static cudaError_t sd_tline_T(const KernelArgs& a, void* w, const double* table, int logn, double scale_p2max) {
  using C = cplx_t<T>;
  const int n = a.geo.n[3];
  const size_t V3 = (size_t)a.geo.n[0] * a.geo.n[1] * a.geo.n[2];
  const size_t smem = ((size_t)n * XB + n / 2) * sizeof(C);
  auto kern = sd_tline_kernel<T, XB>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  kern<<<dim3((unsigned)(V3 / XB), 4), TLINE_THREADS, smem, a.stream>>>((C*)w, a.geo, logn, table, scale_p2max);
  return cudaGetLastError();
}

cudaError_t launch_sd_tline(const KernelArgs& a, void* w, const double* table, double alpha) {
  const int n = a.geo.n[3];
  int logn = 0;
  while ((1 << logn) < n) ++logn;
  const double V = 2.0 * (double)a.geo.vh;
  const double scale_p2max = 0.5 * alpha / V * 16.0;
  const int xb = tline_xb(a.geo, a.prec);
  if (a.prec == 0) {
    switch (xb) {
      case 16: return sd_tline_T<double, 16>(a, w, table, logn, scale_p2max);
      case 8: return sd_tline_T<double, 8>(a, w, table, logn, scale_p2max);
    }
  } else {
    switch (xb) {
      case 32: return sd_tline_T<float, 32>(a, w, table, logn, scale_p2max);
      case 16: return sd_tline_T<float, 16>(a, w, table, logn, scale_p2max);
      case 8: return sd_tline_T<float, 8>(a, w, table, logn, scale_p2max);
    }
  }
  return cudaErrorInvalidValue;
}

// ======================================================================================================================
// g(x) and the gauge rotation
// ======================================================================================================================
// g = reunitarise(1 + w), w rebuilt from its packed form (reading B5)
template <class T, class C>
__device__ __forceinline__ void rotation_from_packed(const C* __restrict__ w, size_t V, size_t lex, C (&gm)[9]) {
  const C w01 = w[lex], w02 = w[V + lex], w12 = w[2 * V + lex], dd = w[3 * V + lex];
  gm[0] = mk<T>(T(1), dd.x);
  gm[1] = w01;
  gm[2] = w02;
  gm[3] = mk<T>(-w01.x, w01.y);
  gm[4] = mk<T>(T(1), dd.y);
  gm[5] = w12;
  gm[6] = mk<T>(-w02.x, w02.y);
  gm[7] = mk<T>(-w12.x, w12.y);
  gm[8] = mk<T>(T(1), -(dd.x + dd.y));
  reunitarize<T>(gm);
}

// One thread per site: U_mu(x) <- g(x) U_mu(x) g(x+mu)^dagger, mu = 0..3 (Alg. 2 l.11-15, reading B6).  The first
// blocks_per_parity blocks take parity 0, the rest parity 1.
template <class T, int NELEM>
__global__ void __launch_bounds__(SD_THREADS) sd_rotate_kernel(cplx_t<T>* __restrict__ links, Geo g,
                                                               const cplx_t<T>* __restrict__ w, int blocks_per_parity,
                                                               BlockOrder order) {
  using C = cplx_t<T>;
  const int parity = blockIdx.x >= blocks_per_parity;
  const int cb = ordered_block(order, blockIdx.x - parity * blocks_per_parity) * SD_THREADS + threadIdx.x;
  if (cb >= g.vh) return;
  const size_t V = 2 * (size_t)g.vh;
  const Site s = site_of(g, parity, cb);
  const int lex = lex_of(g, s);
  // the site's four links travel global -> shared with cp.async (no registers held) while g(x) is rebuilt from the
  // packed field; a thread reads back only what it copied itself, so there is no barrier
  extern __shared__ __align__(16) unsigned char rot_smem[];
  C* sm = reinterpret_cast<C*>(rot_smem) + threadIdx.x;
  C* fwd = links + link_offset<NELEM>(g, parity, cb, 0);
#pragma unroll
  for (int i = 0; i < 4 * NELEM; ++i) {
    const unsigned dst = (unsigned)__cvta_generic_to_shared(sm + i * SD_THREADS);
    if (sizeof(C) == 16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(fwd + i * 32) : "memory");
    else asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(fwd + i * 32) : "memory");
  }
  C gx[9];
  rotation_from_packed<T>(w, V, lex, gx);
  asm volatile("cp.async.wait_all;" ::: "memory");
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) {
    C gup[9], u[9], v[9], o[9];
    rotation_from_packed<T>(w, V, lex_up(g, s, lex, mu), gup);
    load_link<NELEM, true, SD_THREADS>(sm + mu * NELEM * SD_THREADS, u);
    mul_left<LinkRows<NELEM>::value>(gx, u, v);
    mul_right_adj<LinkRows<NELEM>::value>(v, gup, o);
    store_link<NELEM>(fwd + mu * NELEM * 32, o);
  }
}

// ======================================================================================================================
// host side: plans and launch wrappers
// ======================================================================================================================
struct FftPlans {
  cufftHandle plan3 = 0, plan1 = 0;
  bool have3 = false, have1 = false;
  size_t work3 = 0, work1 = 0;
};

static const char* cufft_err(cufftResult r) {
  static thread_local char buf[48];
  snprintf(buf, sizeof(buf), "cuFFT error %d", (int)r);
  return buf;
}

void fft_plans_destroy(FftPlans* p) {
  if (!p) return;
  if (p->have3) cufftDestroy(p->plan3);
  if (p->have1) cufftDestroy(p->plan1);
  delete p;
}

// Creates the plans without letting cuFFT allocate; *work = bytes of work area they need (the larger of the two).
const char* fft_plans_create(FftPlans** out, const Geo& g, int prec, int gauge, cudaStream_t stream, size_t* work) {
  FftPlans* p = new FftPlans();
  *out = nullptr;
  const cufftType type = prec == 0 ? CUFFT_Z2Z : CUFFT_C2C;
  const int nx = g.n[0], ny = g.n[1], nz = g.n[2], nt = g.n[3];
  const int V3 = nx * ny * nz;
  cufftResult r = cufftCreate(&p->plan3);
  if (r == CUFFT_SUCCESS) {
    p->have3 = true;
    r = cufftSetAutoAllocation(p->plan3, 0);
  }
  if (r == CUFFT_SUCCESS) {
    int n3[3] = {nz, ny, nx};
    r = cufftMakePlanMany(p->plan3, 3, n3, nullptr, 1, V3, nullptr, 1, V3, type, 4 * nt, &p->work3);
  }
  if (r == CUFFT_SUCCESS) r = cufftSetStream(p->plan3, stream);
  if (r == CUFFT_SUCCESS && gauge == 0) {
    r = cufftCreate(&p->plan1);
    if (r == CUFFT_SUCCESS) {
      p->have1 = true;
      r = cufftSetAutoAllocation(p->plan1, 0);
    }
    if (r == CUFFT_SUCCESS) {
      int n1[1] = {nt};
      int embed[1] = {nt};
      r = cufftMakePlanMany(p->plan1, 1, n1, embed, V3, 1, embed, V3, 1, type, V3, &p->work1);
    }
    if (r == CUFFT_SUCCESS) r = cufftSetStream(p->plan1, stream);
  }
  if (r != CUFFT_SUCCESS) {
    fft_plans_destroy(p);
    return cufft_err(r);
  }
  *work = p->work3 > p->work1 ? p->work3 : p->work1;
  *out = p;
  return nullptr;
}

const char* fft_plans_set_work(FftPlans* p, void* work) {
  cufftResult r = cufftSetWorkArea(p->plan3, work);
  if (r == CUFFT_SUCCESS && p->have1) r = cufftSetWorkArea(p->plan1, work);
  return r == CUFFT_SUCCESS ? nullptr : cufft_err(r);
}

// in-place transform of the four packed fields; *launches += number of cuFFT executions
const char* fft_exec(FftPlans* p, const Geo& g, int prec, void* w, bool forward, bool with_t, int* launches) {
  const int dir = forward ? CUFFT_FORWARD : CUFFT_INVERSE;
  const size_t V = 2 * (size_t)g.vh;
  cufftResult r;
  if (prec == 0) {
    r = cufftExecZ2Z(p->plan3, (cufftDoubleComplex*)w, (cufftDoubleComplex*)w, dir);
    *launches += 1;
    for (int k = 0; k < 4 && r == CUFFT_SUCCESS && p->have1 && with_t; ++k) {
      cufftDoubleComplex* f = (cufftDoubleComplex*)w + k * V;
      r = cufftExecZ2Z(p->plan1, f, f, dir);
      *launches += 1;
    }
  } else {
    r = cufftExecC2C(p->plan3, (cufftComplex*)w, (cufftComplex*)w, dir);
    *launches += 1;
    for (int k = 0; k < 4 && r == CUFFT_SUCCESS && p->have1 && with_t; ++k) {
      cufftComplex* f = (cufftComplex*)w + k * V;
      r = cufftExecC2C(p->plan1, f, f, dir);
      *launches += 1;
    }
  }
  return r == CUFFT_SUCCESS ? nullptr : cufft_err(r);
}

size_t sd_table_entries(const Geo& g) { return (size_t)g.n[0] + g.n[1] + g.n[2] + g.n[3]; }
int sd_num_partials(const Geo& g) { return (g.vh + SD_THREADS - 1) / SD_THREADS; }

cudaError_t launch_sd_table(const KernelArgs& a, double* table) {
  const int n = (int)sd_table_entries(a.geo);
  sd_table_kernel<<<(n + 127) / 128, 128, 0, a.stream>>>(table, a.geo.n[0], a.geo.n[1], a.geo.n[2], a.geo.n[3]);
  return cudaGetLastError();
}

template <class T, int NELEM, int ND>
static cudaError_t sd_delta_T(const KernelArgs& a, void* w) {
  sd_delta_kernel<T, NELEM, ND><<<sd_num_partials(a.geo), SD_THREADS, 0, a.stream>>>(
      (const cplx_t<T>*)a.links, a.geo, (cplx_t<T>*)w, (double2*)a.partials, make_block_order(a.geo));
  return cudaGetLastError();
}

cudaError_t launch_sd_delta(const KernelArgs& a, void* w) {
  const bool coul = a.gauge == 1;
  if (a.prec == 0) {
    if (a.storage == 18) return coul ? sd_delta_T<double, 9, 3>(a, w) : sd_delta_T<double, 9, 4>(a, w);
    return coul ? sd_delta_T<double, 6, 3>(a, w) : sd_delta_T<double, 6, 4>(a, w);
  }
  if (a.storage == 18) return coul ? sd_delta_T<float, 9, 3>(a, w) : sd_delta_T<float, 9, 4>(a, w);
  return coul ? sd_delta_T<float, 6, 3>(a, w) : sd_delta_T<float, 6, 4>(a, w);
}

// F, theta from the partials the last sd_delta launch left
cudaError_t launch_sd_final(const KernelArgs& a) {
  const double V = 2.0 * (double)a.geo.vh;
  const int nd = a.gauge == 1 ? 3 : 4;
  sd_final_kernel<<<1, 1024, 0, a.stream>>>((const double2*)a.partials, sd_num_partials(a.geo), 1.0 / (nd * 3.0 * V),
                                            1.0 / (3.0 * V), (double*)a.result);
  return cudaGetLastError();
}

cudaError_t launch_sd_filter(const KernelArgs& a, void* w, const double* table, double alpha, bool accelerate) {
  const size_t V = 2 * (size_t)a.geo.vh;
  if (!accelerate) {
    const size_t n = 4 * V;
    const unsigned blocks = (unsigned)((n + 255) / 256);
    if (a.prec == 0) sd_scale_kernel<double><<<blocks, 256, 0, a.stream>>>((double2*)w, n, 0.5 * alpha);
    else sd_scale_kernel<float><<<blocks, 256, 0, a.stream>>>((float2*)w, n, (float)(0.5 * alpha));
    return cudaGetLastError();
  }
  const bool coul = a.gauge == 1;
  const double N = coul ? (double)a.geo.n[0] * a.geo.n[1] * a.geo.n[2] : (double)V;
  const double scale_p2max = 0.5 * alpha / N * (coul ? 12.0 : 16.0);
  const unsigned blocks = (unsigned)((V + 255) / 256);
  if (a.prec == 0) {
    if (coul) sd_filter_kernel<double, 3><<<blocks, 256, 0, a.stream>>>((double2*)w, a.geo, table, scale_p2max);
    else sd_filter_kernel<double, 4><<<blocks, 256, 0, a.stream>>>((double2*)w, a.geo, table, scale_p2max);
  } else {
    if (coul) sd_filter_kernel<float, 3><<<blocks, 256, 0, a.stream>>>((float2*)w, a.geo, table, scale_p2max);
    else sd_filter_kernel<float, 4><<<blocks, 256, 0, a.stream>>>((float2*)w, a.geo, table, scale_p2max);
  }
  return cudaGetLastError();
}

template <class T, int NELEM>
static cudaError_t sd_rotate_T(const KernelArgs& a, const void* w) {
  const int bpp = sd_num_partials(a.geo);
  constexpr size_t SMEM = (size_t)4 * NELEM * SD_THREADS * sizeof(cplx_t<T>);
  cudaError_t e = cudaFuncSetAttribute(sd_rotate_kernel<T, NELEM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM);
  if (e != cudaSuccess) return e;
  sd_rotate_kernel<T, NELEM><<<2 * bpp, SD_THREADS, SMEM, a.stream>>>((cplx_t<T>*)a.links, a.geo, (const cplx_t<T>*)w, bpp,
                                                                      make_block_order(a.geo));
  return cudaGetLastError();
}

cudaError_t launch_sd_rotate(const KernelArgs& a, const void* w) {
  if (a.prec == 0) return a.storage == 18 ? sd_rotate_T<double, 9>(a, w) : sd_rotate_T<double, 6>(a, w);
  return a.storage == 18 ? sd_rotate_T<float, 9>(a, w) : sd_rotate_T<float, 6>(a, w);
}

}  // namespace gf
