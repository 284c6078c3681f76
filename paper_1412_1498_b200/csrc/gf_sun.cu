// gf_sun.cu — the overrelaxation path for a general number of colours ("SU(N) with N>2", "its
// N(N-1)/2 SU(2) subgroups").  N = 3 is the specialised path of gf_kernels.cu; this file is
// instantiated for N = 2 and N = 4, full storage (N^2 complex numbers per link), FP64 and FP32, both gauges.
//   reorder_sun   : canonical links[site][mu][N][N][re,im] <-> internal AoSoA-32 layout with NELEM = N^2
//   halfsweep_sun : one parity of the sweep; the N(N-1)/2 subgroups in the order of reading A24 (pairs (i,j) by
//                   increasing j - i, then i; N = 3 would give (0,1),(1,2),(0,2) = reading A4)
//   measure_sun   : F (normalised by d N V) and theta (by N V), eqs. 1.1-1.3
//   reunit_sun    : Gram-Schmidt over the rows in order, last row times conj(det)  (reading A25)
// One thread per site as in the SU(3) kernels; K(x) and the subgroup steps in FP64 in both storage precisions.
#include "gf_device.cuh"
#include "gf_internal.h"

namespace gf {

namespace {

constexpr int SUN_THREADS = 128;

template <int NN, class C>
__device__ __forceinline__ void load_mat(const C* __restrict__ p, C (&u)[NN]) {
#pragma unroll
  for (int e = 0; e < NN; ++e) u[e] = p[e * 32];
}
template <int NN, class C>
__device__ __forceinline__ void store_mat(C* __restrict__ p, const C (&u)[NN]) {
#pragma unroll
  for (int e = 0; e < NN; ++e) p[e * 32] = u[e];
}

// One subgroup step on rows/cols (I,J) of the N x N matrices K (FP64) and G (storage precision): eqs. 1.4-1.6 on the
// SU(2)-proportional part of the block (reading A5), exact power (A6, A7).
template <int N, int I, int J, class CG>
__device__ __forceinline__ void sun_step(double2 (&K)[N * N], CG (&G)[N * N], double omega) {
  using TG = decltype(G[0].x);
  const double r0 = K[I * N + I].x + K[J * N + J].x;
  const double r1 = -(K[I * N + J].y + K[J * N + I].y);
  const double r2 = K[J * N + I].x - K[I * N + J].x;
  const double r3 = -(K[I * N + I].y - K[J * N + J].y);
  double c, q1, q2, q3;
  su2_overrelax<double>(r0, r1, r2, r3, omega, c, q1, q2, q3);
  const double2 g00 = mk<double>(c, q3), g01 = mk<double>(q2, q1), g10 = mk<double>(-q2, q1), g11 = mk<double>(c, -q3);
#pragma unroll
  for (int col = 0; col < N; ++col) {
    const double2 ki = K[I * N + col], kj = K[J * N + col];
    double2 a = cmul(g00, ki); cfma(a, g01, kj);
    double2 b = cmul(g10, ki); cfma(b, g11, kj);
    K[I * N + col] = a; K[J * N + col] = b;
  }
  const TG cg = (TG)c, p1 = (TG)q1, p2 = (TG)q2, p3 = (TG)q3;
  const CG h00 = mk<TG>(cg, p3), h01 = mk<TG>(p2, p1), h10 = mk<TG>(-p2, p1), h11 = mk<TG>(cg, -p3);
#pragma unroll
  for (int col = 0; col < N; ++col) {
    const CG gi = G[I * N + col], gj = G[J * N + col];
    CG a = cmul(h00, gi); cfma(a, h01, gj);
    CG b = cmul(h10, gi); cfma(b, h11, gj);
    G[I * N + col] = a; G[J * N + col] = b;
  }
}

// the pairs (I, I + D) for I = 0 .. N-D-1, then D + 1  (reading A24), unrolled at compile time
template <int N, int D, int I, class CG>
__device__ __forceinline__ void sun_steps(double2 (&K)[N * N], CG (&G)[N * N], double omega) {
  if constexpr (D < N) {
    if constexpr (I + D < N) {
      sun_step<N, I, I + D>(K, G, omega);
      sun_steps<N, D, I + 1>(K, G, omega);
    } else {
      sun_steps<N, D + 1, 0>(K, G, omega);
    }
  }
}

// p <- G u, element by element (no product matrix in registers: SU(4) in FP64 already holds K, G and u)
template <int N, class C>
__device__ __forceinline__ void sun_mul_left_store(const C (&G)[N * N], const C (&u)[N * N], C* __restrict__ p) {
#pragma unroll
  for (int i = 0; i < N; ++i)
#pragma unroll
    for (int j = 0; j < N; ++j) {
      C z = cmul(G[i * N], u[j]);
#pragma unroll
      for (int k = 1; k < N; ++k) cfma(z, G[i * N + k], u[k * N + j]);
      p[(i * N + j) * 32] = z;
    }
}
// p <- u G^dagger
template <int N, class C>
__device__ __forceinline__ void sun_mul_right_adj_store(const C (&u)[N * N], const C (&G)[N * N], C* __restrict__ p) {
  using T = decltype(p[0].x);
#pragma unroll
  for (int i = 0; i < N; ++i)
#pragma unroll
    for (int j = 0; j < N; ++j) {
      C z = mk<T>(T(0), T(0));
#pragma unroll
      for (int k = 0; k < N; ++k) cfma_cj(z, u[i * N + k], G[j * N + k]);
      p[(i * N + j) * 32] = z;
    }
}

template <class T, int N, bool IN>
__global__ void __launch_bounds__(256) reorder_sun_kernel(cplx_t<T>* __restrict__ internal, T* __restrict__ canon, Geo g,
                                                          long long lex_begin, long long lex_end,
                                                          const T* __restrict__ canon_chunk_base) {
  using C = cplx_t<T>;
  constexpr int NN = N * N;
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int mu = (int)(tid & 3);
  const long long sid = tid >> 2;
  const long long lex = lex_begin + sid;
  if (lex >= lex_end) return;
  unsigned q = (unsigned)lex;
  const int x = q % (unsigned)g.n[0]; q /= (unsigned)g.n[0];
  const int y = q % (unsigned)g.n[1]; q /= (unsigned)g.n[1];
  const int z = q % (unsigned)g.n[2];
  const int t = q / (unsigned)g.n[2];
  const int parity = (x + y + z + t) & 1;
  C* p = internal + link_offset<NN>(g, parity, (int)(lex >> 1), mu);
  T* c = canon_chunk_base ? const_cast<T*>(canon_chunk_base) + (sid * 4 + mu) * (2 * NN) : canon + (lex * 4 + mu) * (2 * NN);
  C* cc = reinterpret_cast<C*>(c);
  C u[NN];
  if (IN) {
#pragma unroll
    for (int e = 0; e < NN; ++e) u[e] = cc[e];
    store_mat<NN>(p, u);
  } else {
    load_mat<NN>(p, u);
#pragma unroll
    for (int e = 0; e < NN; ++e) cc[e] = u[e];
  }
}

template <class T, int N, int ND>
__global__ void __launch_bounds__(SUN_THREADS) halfsweep_sun_kernel(cplx_t<T>* __restrict__ links, Geo g, int parity,
                                                                    double omega) {
  using C = cplx_t<T>;
  constexpr int NN = N * N;
  // serpentine block order (see gf_kernels.cu): the odd half-sweep starts where the even one ended, in L2
  const int cb = ((parity & 1) ? gridDim.x - 1u - blockIdx.x : blockIdx.x) * SUN_THREADS + threadIdx.x;
  if (cb >= g.vh) return;
  const Site s = site_of(g, parity, cb);
  C* fwd = links + link_offset<NN>(g, parity, cb, 0);
  C* bwd[4];
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) bwd[mu] = links + link_offset<NN>(g, parity ^ 1, cb_down(g, s, cb, mu), mu);

  // K(x) = sum_{mu<ND} [U_mu(x) + U_mu(x-mu)^dagger]   (eq. 1.5, reading A3), summed in FP64
  double2 K[NN];
#pragma unroll
  for (int e = 0; e < NN; ++e) K[e] = make_double2(0.0, 0.0);
#pragma unroll
  for (int mu = 0; mu < ND; ++mu) {
    C u[NN];
    load_mat<NN>(fwd + mu * NN * 32, u);
#pragma unroll
    for (int e = 0; e < NN; ++e) { K[e].x += (double)u[e].x; K[e].y += (double)u[e].y; }
    asm volatile("" ::: "memory");
    load_mat<NN>(bwd[mu], u);
#pragma unroll
    for (int i = 0; i < N; ++i)
#pragma unroll
      for (int j = 0; j < N; ++j) { K[i * N + j].x += (double)u[j * N + i].x; K[i * N + j].y -= (double)u[j * N + i].y; }
    asm volatile("" ::: "memory");
  }
  C G[NN];
#pragma unroll
  for (int e = 0; e < NN; ++e) G[e] = mk<T>((e % (N + 1) == 0) ? T(1) : T(0), T(0));
  sun_steps<N, 1, 0>(K, G, omega);

  // second pass (L1/L2 hits): all four directions are transformed, also in Coulomb gauge (reading A9)
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) {
    C u[NN];
    load_mat<NN>(fwd + mu * NN * 32, u);
    sun_mul_left_store<N>(G, u, fwd + mu * NN * 32);
    asm volatile("" ::: "memory");  // one link in registers at a time (SU(4) in FP64: K, G and u are 192 registers)
    load_mat<NN>(bwd[mu], u);
    sun_mul_right_adj_store<N>(u, G, bwd[mu]);
    asm volatile("" ::: "memory");
  }
}

constexpr int SUN_MEASURE_THREADS = 256;

template <class T, int N, int ND>
__global__ void __launch_bounds__(SUN_MEASURE_THREADS) measure_sun_kernel(const cplx_t<T>* __restrict__ links, Geo g,
                                                                          int blocks_per_parity,
                                                                          double2* __restrict__ partials) {
  using C = cplx_t<T>;
  constexpr int NN = N * N;
  const int parity = blockIdx.x >= blocks_per_parity;
  const int cb = (blockIdx.x - parity * blocks_per_parity) * SUN_MEASURE_THREADS + threadIdx.x;
  double f = 0.0, q = 0.0;
  if (cb < g.vh) {
    const Site s = site_of(g, parity, cb);
    const C* fwd = links + link_offset<NN>(g, parity, cb, 0);
    C A[NN];
#pragma unroll
    for (int e = 0; e < NN; ++e) A[e] = mk<T>(T(0), T(0));
    T tr = T(0);
#pragma unroll
    for (int nu = 0; nu < ND; ++nu) {
      C u[NN];
      load_mat<NN>(links + link_offset<NN>(g, parity ^ 1, cb_down(g, s, cb, nu), nu), u);
#pragma unroll
      for (int e = 0; e < NN; ++e) { A[e].x += u[e].x; A[e].y += u[e].y; }
#pragma unroll
      for (int i = 0; i < N; ++i) tr += u[i * N + i].x;
      load_mat<NN>(fwd + nu * NN * 32, u);
#pragma unroll
      for (int e = 0; e < NN; ++e) { A[e].x -= u[e].x; A[e].y -= u[e].y; }
#pragma unroll
      for (int i = 0; i < N; ++i) tr += u[i * N + i].x;
    }
    f = (double)tr;
    // Delta = (A - A^dag) - (1/N) Tr(A - A^dag): diagonal 2i Im A_ii minus its mean, off-diagonal A_ij - conj(A_ji)
    T m = T(0);
#pragma unroll
    for (int i = 0; i < N; ++i) m += T(2) * A[i * N + i].y;
    m /= T(N);
    T acc = T(0);
#pragma unroll
    for (int i = 0; i < N; ++i) {
      const T d = T(2) * A[i * N + i].y - m;
      acc += d * d;
#pragma unroll
      for (int j = i + 1; j < N; ++j) {
        const T ax = A[i * N + j].x - A[j * N + i].x, ay = A[i * N + j].y + A[j * N + i].y;
        acc += T(2) * (ax * ax + ay * ay);
      }
    }
    q = (double)acc;
  }
  block_sum2<SUN_MEASURE_THREADS>(f, q);
  if (threadIdx.x == 0) partials[blockIdx.x] = make_double2(f, q);
}

template <int N, class C>
__device__ __forceinline__ C sun_det(const C (&u)[N * N]) {
  if constexpr (N == 2) {
    C z = cmul(u[0], u[3]);
    const C w = cmul(u[1], u[2]);
    z.x -= w.x; z.y -= w.y;
    return z;
  } else {  // N == 4: expansion along row 0 into 3x3 minors
    static_assert(N == 4, "determinant written for N = 2 and 4");
    using T = decltype(u[0].x);
    C det = mk<T>(T(0), T(0));
#pragma unroll
    for (int c0 = 0; c0 < 4; ++c0) {
      int cols[3], k = 0;
#pragma unroll
      for (int c = 0; c < 4; ++c)
        if (c != c0) cols[k++] = c;
      auto e = [&](int r, int c) { return u[r * 4 + cols[c]]; };
      auto sub2 = [&](C a, C b, C c, C d) { C z = cmul(a, d); const C w = cmul(b, c); z.x -= w.x; z.y -= w.y; return z; };
      const C m0 = sub2(e(2, 1), e(2, 2), e(3, 1), e(3, 2));
      const C m1 = sub2(e(2, 0), e(2, 2), e(3, 0), e(3, 2));
      const C m2 = sub2(e(2, 0), e(2, 1), e(3, 0), e(3, 1));
      C minor = cmul(e(1, 0), m0);
      const C t1 = cmul(e(1, 1), m1), t2 = cmul(e(1, 2), m2);
      minor.x += t2.x - t1.x; minor.y += t2.y - t1.y;
      const C term = cmul(u[c0], minor);
      if (c0 & 1) { det.x -= term.x; det.y -= term.y; }
      else { det.x += term.x; det.y += term.y; }
    }
    return det;
  }
}

template <class T, int N>
__global__ void __launch_bounds__(256) reunit_sun_kernel(cplx_t<T>* __restrict__ links, long long ntiles, Geo g) {
  using C = cplx_t<T>;
  constexpr int NN = N * N;
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long tile = tid >> 5;
  if (tile >= ntiles) return;
  // tile = (parity * nblk + blk) * 4 + mu; padding lanes of the last block of a parity hold no link
  const long long blk = (tile >> 2) % g.nblk;
  if (blk * 32 + (tid & 31) >= g.vh) return;
  C* p = links + (size_t)tile * NN * 32 + (tid & 31);
  C u[NN];
  load_mat<NN>(p, u);
#pragma unroll
  for (int r = 0; r < N; ++r) {
#pragma unroll
    for (int pr = 0; pr < r; ++pr) {  // row r minus its projection on the finished row pr
      C c = mk<T>(T(0), T(0));
#pragma unroll
      for (int k = 0; k < N; ++k) {  // c += conj(u[pr][k]) u[r][k]
        c.x = fma(u[pr * N + k].x, u[r * N + k].x, c.x); c.x = fma(u[pr * N + k].y, u[r * N + k].y, c.x);
        c.y = fma(u[pr * N + k].x, u[r * N + k].y, c.y); c.y = fma(-u[pr * N + k].y, u[r * N + k].x, c.y);
      }
#pragma unroll
      for (int k = 0; k < N; ++k) {
        u[r * N + k].x -= c.x * u[pr * N + k].x - c.y * u[pr * N + k].y;
        u[r * N + k].y -= c.x * u[pr * N + k].y + c.y * u[pr * N + k].x;
      }
    }
    T n2 = T(0);
#pragma unroll
    for (int k = 0; k < N; ++k) n2 += u[r * N + k].x * u[r * N + k].x + u[r * N + k].y * u[r * N + k].y;
    const T inv = T(1) / sqrt_(n2);
#pragma unroll
    for (int k = 0; k < N; ++k) { u[r * N + k].x *= inv; u[r * N + k].y *= inv; }
  }
  const C det = sun_det<N>(u);
#pragma unroll
  for (int k = 0; k < N; ++k) {  // last row times conj(det)
    const C v = u[(N - 1) * N + k];
    u[(N - 1) * N + k] = mk<T>(v.x * det.x + v.y * det.y, v.y * det.x - v.x * det.y);
  }
  store_mat<NN>(p, u);
}

template <class T, int N>
cudaError_t reorder_sun_T(const KernelArgs& a, bool in, void* canon, long long lex_begin, long long lex_end,
                          const void* chunk_base) {
  const long long nthreads = (lex_end - lex_begin) * 4;
  if (nthreads <= 0) return cudaSuccess;
  const unsigned blocks = (unsigned)((nthreads + 255) / 256);
  if (in)
    reorder_sun_kernel<T, N, true><<<blocks, 256, 0, a.stream>>>((cplx_t<T>*)a.links, (T*)canon, a.geo, lex_begin, lex_end,
                                                                 (const T*)chunk_base);
  else
    reorder_sun_kernel<T, N, false><<<blocks, 256, 0, a.stream>>>((cplx_t<T>*)a.links, (T*)canon, a.geo, lex_begin, lex_end,
                                                                  (const T*)chunk_base);
  return cudaGetLastError();
}

template <class T, int N>
cudaError_t halfsweep_sun_T(const KernelArgs& a, int parity, double omega) {
  const unsigned blocks = (unsigned)((a.geo.vh + SUN_THREADS - 1) / SUN_THREADS);
  if (a.gauge == 1) halfsweep_sun_kernel<T, N, 3><<<blocks, SUN_THREADS, 0, a.stream>>>((cplx_t<T>*)a.links, a.geo, parity, omega);
  else halfsweep_sun_kernel<T, N, 4><<<blocks, SUN_THREADS, 0, a.stream>>>((cplx_t<T>*)a.links, a.geo, parity, omega);
  return cudaGetLastError();
}

template <class T, int N>
cudaError_t measure_sun_T(const KernelArgs& a) {
  const int bpp = (a.geo.vh + SUN_MEASURE_THREADS - 1) / SUN_MEASURE_THREADS;
  if (a.gauge == 1)
    measure_sun_kernel<T, N, 3><<<2 * bpp, SUN_MEASURE_THREADS, 0, a.stream>>>((const cplx_t<T>*)a.links, a.geo, bpp, (double2*)a.partials);
  else
    measure_sun_kernel<T, N, 4><<<2 * bpp, SUN_MEASURE_THREADS, 0, a.stream>>>((const cplx_t<T>*)a.links, a.geo, bpp, (double2*)a.partials);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  const double V = 2.0 * (double)a.geo.vh;
  const int nd = a.gauge == 1 ? 3 : 4;
  // second stage: f over the parity-0 partials (every link once), q over all; fixed order
  return launch_measure_tail(a, 2 * bpp, bpp, 1.0 / (nd * (double)N * V), 1.0 / ((double)N * V));
}

template <class T, int N>
cudaError_t reunit_sun_T(const KernelArgs& a) {
  const long long ntiles = 2LL * a.geo.nblk * 4;
  reunit_sun_kernel<T, N><<<(unsigned)((ntiles * 32 + 255) / 256), 256, 0, a.stream>>>((cplx_t<T>*)a.links, ntiles, a.geo);
  return cudaGetLastError();
}

}  // namespace

#define GF_SUN_DISPATCH(FN, ...)                                                                 \
  do {                                                                                           \
    if (a.ncolors == 2) return a.prec == 0 ? FN<double, 2>(__VA_ARGS__) : FN<float, 2>(__VA_ARGS__); \
    if (a.ncolors == 4) return a.prec == 0 ? FN<double, 4>(__VA_ARGS__) : FN<float, 4>(__VA_ARGS__); \
    return cudaErrorNotSupported;                                                                \
  } while (0)

bool sun_supported(int ncolors) { return ncolors == 2 || ncolors == 4; }

cudaError_t launch_reorder_sun(const KernelArgs& a, bool in, void* canon, long long lex_begin, long long lex_end,
                               const void* chunk_base) {
  GF_SUN_DISPATCH(reorder_sun_T, a, in, canon, lex_begin, lex_end, chunk_base);
}
cudaError_t launch_halfsweep_sun(const KernelArgs& a, int parity, double omega) {
  GF_SUN_DISPATCH(halfsweep_sun_T, a, parity, omega);
}
cudaError_t launch_measure_sun(const KernelArgs& a) { GF_SUN_DISPATCH(measure_sun_T, a); }
cudaError_t launch_reunit_sun(const KernelArgs& a) { GF_SUN_DISPATCH(reunit_sun_T, a); }

}  // namespace gf
