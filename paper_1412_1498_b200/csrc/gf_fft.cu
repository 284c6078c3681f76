// gf_fft.cu — hand-written transforms for Algorithm 2 (PAPER.md:97-124 l.4-7; eq. 1.8): the four packed fields are taken
// to momentum space, multiplied by (alpha/2) (p^2_max / p^2) / N and taken back in FIVE passes over HBM (Landau) or
// THREE (Coulomb) instead of cuFFT's separate transforms and a factor kernel:
//
//   plane pass (x,y) forward -> line pass z forward -> line pass t: forward, factor, inverse -> z inverse -> (x,y) inverse
//   Coulomb:  plane pass (x,y) forward -> line pass z: forward, factor, inverse -> (x,y) inverse
//
// Each pass reads and writes every field entry once.  An extent n = R1 * R2 (R1, R2 in {1,2,3,4,6,8,12,16}, n <= 256) is
// transformed in two register-level steps (Cooley-Tukey, t = R2 t1 + t2, k = k1 + R1 k2):
//   outer step: for each t2 an R1-point transform over the stride-R2 elements, times the twiddle W_n^(t2 k1), written
//               back IN PLACE (position R2 k1 + t2);  inner step: for each k1 an R2-point transform over the R2
//               consecutive positions, again in place.
// Position R2 k1 + k2 then holds frequency k1 + R1 k2: momentum space is kept in this digit-swapped order — only the
// diagonal factor is applied there, from tables of 4 sin^2(pi k / n) stored in the same order — and the inverse runs
// the two steps backwards.  No step moves data between threads except through one shared-memory tile.
// cuFFT (gf_fftsd.cu) stays as the path for extents this scheme does not cover and as a cross-check (GF_OPT_FFT_OWN).
#include "gf_device.cuh"
#include "gf_internal.h"

namespace gf {

// ---- 48th roots of unity as compile-time constants: every W_R^k with R in {2,3,4,6,8,12,16} is one of them ---------------
template <int J> struct Root48 {
  static constexpr int j = ((J % 48) + 48) % 48;
  static constexpr double quarter(int i) {  // cos(2 pi i / 48), 0 <= i <= 12
    constexpr double c[13] = {1.0,
                              0.99144486137381041114,
                              0.96592582628906828675,
                              0.92387953251128675613,
                              0.86602540378443864676,
                              0.79335334029123516458,
                              0.7071067811865475244,
                              0.60876142900872063942,
                              0.5,
                              0.38268343236508977173,
                              0.25881904510252076235,
                              0.13052619222005159155,
                              0.0};
    return c[i];
  }
  static constexpr double cosv(int i) {  // cos(2 pi i / 48), 0 <= i < 48
    return i <= 12 ? quarter(i) : i <= 24 ? -quarter(24 - i) : i <= 36 ? -quarter(i - 24) : quarter(48 - i);
  }
  static constexpr double re = cosv(j);
  static constexpr double im = cosv((j + 36) % 48);  // sin(a) = cos(a - pi/2) = cos(a + 3 pi/2)
};

template <class C> __device__ __forceinline__ C cadd(const C a, const C b) { C z; z.x = a.x + b.x; z.y = a.y + b.y; return z; }
template <class C> __device__ __forceinline__ C csub(const C a, const C b) { C z; z.x = a.x - b.x; z.y = a.y - b.y; return z; }
// a * (wr + i wi) with compile-time wr, wi; INV: the conjugate root
template <class T, int J, bool INV, class C> __device__ __forceinline__ C cmul_root(const C a) {
  constexpr T wr = (T)Root48<J>::re, wi = (T)(INV ? Root48<J>::im : -Root48<J>::im);  // forward: exp(-i theta)
  C z;
  if (Root48<J>::j == 0) return a;
  if (Root48<J>::j == 12) { z.x = INV ? -a.y : a.y; z.y = INV ? a.x : -a.x; return z; }
  if (Root48<J>::j == 24) { z.x = -a.x; z.y = -a.y; return z; }
  if (Root48<J>::j == 36) { z.x = INV ? a.y : -a.y; z.y = INV ? -a.x : a.x; return z; }
  z.x = a.x * wr - a.y * wi;
  z.y = a.x * wi + a.y * wr;
  return z;
}

// R-point transform in registers, natural order in and out.  Forward: X_k = sum_t x_t exp(-2 pi i t k / R); INV: + sign.
template <class T, int R, bool INV> struct Dft;
template <class T, bool INV> struct Dft<T, 1, INV> {
  template <class C> static __device__ __forceinline__ void run(C (&)[1]) {}
};
template <class T, bool INV> struct Dft<T, 3, INV> {
  template <class C> static __device__ __forceinline__ void run(C (&v)[3]) {
    const C a = v[0], b = v[1], c = v[2];
    v[0] = cadd(a, cadd(b, c));
    v[1] = cadd(a, cadd(cmul_root<T, 16, INV>(b), cmul_root<T, 32, INV>(c)));
    v[2] = cadd(a, cadd(cmul_root<T, 32, INV>(b), cmul_root<T, 16, INV>(c)));
  }
};
template <class T, int R, bool INV> struct Dft {
  static_assert(R % 2 == 0 && 48 % R == 0, "R in {2,4,6,8,12,16}");
  template <int K, class C> static __device__ __forceinline__ void combine(C (&v)[R], const C (&e)[R / 2], const C (&o)[R / 2]) {
    if constexpr (K < R / 2) {
      const C t = cmul_root<T, K*(48 / R), INV>(o[K]);
      v[K] = cadd(e[K], t);
      v[K + R / 2] = csub(e[K], t);
      combine<K + 1>(v, e, o);
    }
  }
  template <class C> static __device__ __forceinline__ void run(C (&v)[R]) {
    C e[R / 2], o[R / 2];
#pragma unroll
    for (int k = 0; k < R / 2; ++k) { e[k] = v[2 * k]; o[k] = v[2 * k + 1]; }
    Dft<T, R / 2, INV>::run(e);
    Dft<T, R / 2, INV>::run(o);
    combine<0>(v, e, o);
  }
};

// ---- one register-level step: R elements at `sstride` from src, transform, optional twiddle, R elements to dst -----------
// twiddle (TW): output m is multiplied by tw[m * twstep] (forward) or its conjugate (INV); tw[j] = exp(-2 pi i j / n).
template <class T, int R, bool INV, bool TW, class C>
__device__ __forceinline__ void fft_step(const C* src, size_t sstride, C* dst, size_t dstride, const double2* __restrict__ tw,
                                         int twstep) {
  C v[R];
#pragma unroll
  for (int m = 0; m < R; ++m) v[m] = src[m * sstride];
  Dft<T, R, INV>::run(v);
  if (TW) {
#pragma unroll
    for (int m = 1; m < R; ++m) {
      const double2 w = __ldg(tw + m * twstep);
      const T wr = (T)w.x, wi = (T)(INV ? -w.y : w.y);
      const C a = v[m];
      v[m].x = a.x * wr - a.y * wi;
      v[m].y = a.x * wi + a.y * wr;
    }
  }
#pragma unroll
  for (int m = 0; m < R; ++m) dst[m * dstride] = v[m];
}

// scale / p2 for the Fourier factor: FP32 reciprocal seed + two Newton steps (full double accuracy, no FP64 division)
template <class T> __device__ __forceinline__ T factor_of(double scale_p2max, double p2) {
  if (!(p2 > 0.0)) return T(0);  // p = 0 (reading B3)
  if (sizeof(T) == 4) return (T)scale_p2max * __frcp_rn((float)p2);
  double r = (double)__frcp_rn((float)p2);
  r = r * (2.0 - p2 * r);
  r = r * (2.0 - p2 * r);
  return (T)(scale_p2max * r);
}

// MAXR (a constexpr int in scope): the largest radix the enclosing kernel instantiation is launched with; the cases
// above it compile to nothing, so a kernel for radices <= 8 does not carry the register budget of a 16-point transform.
#define GF_R_CASES(R, ...)                                                                      \
  switch (R) {                                                                                  \
    case 1: { constexpr int RR = 1; __VA_ARGS__; } break;                                       \
    case 2: { constexpr int RR = 2; __VA_ARGS__; } break;                                       \
    case 3: { constexpr int RR = 3; __VA_ARGS__; } break;                                       \
    case 4: { constexpr int RR = 4; __VA_ARGS__; } break;                                       \
    case 6: { constexpr int RR = 6; __VA_ARGS__; } break;                                       \
    case 8: { constexpr int RR = 8; __VA_ARGS__; } break;                                       \
    case 12: { constexpr int RR = MAXR >= 12 ? 12 : 1; if (MAXR >= 12) { __VA_ARGS__; } } break; \
    default: { constexpr int RR = MAXR >= 16 ? 16 : 1; if (MAXR >= 16) { __VA_ARGS__; } } break; \
  }

// ---- tables ----------------------------------------------------------------------------------------------------------------
// Per axis mu (offset axis_offset(mu) doubles): p2[n] = 4 sin^2(pi k(pos) / n) in position order, then tw[n] as double2.
struct AxisSplit { int n, r1, r2; };
struct FftShape { AxisSplit ax[4]; };

static bool split_extent(int n, AxisSplit* s) {
  static const int radices[8] = {1, 2, 3, 4, 6, 8, 12, 16};
  s->n = n; s->r1 = s->r2 = 0;
  if (n > 256) return false;
  for (int i = 0; i < 8; ++i) {      // single step when the extent is itself a radix
    if (radices[i] == n) { s->r1 = n; s->r2 = 1; return true; }
  }
  for (int i = 1; i < 8; ++i) {      // else the most balanced pair R1 >= R2 (smallest R1)
    const int r1 = radices[i];
    if (n % r1) continue;
    const int r2 = n / r1;
    if (r2 > r1) continue;
    for (int j = 1; j < 8; ++j)
      if (radices[j] == r2) { s->r1 = r1; s->r2 = r2; return true; }
  }
  return false;
}

static size_t axis_offset(const Geo& g, int mu) {
  size_t o = 0;
  for (int d = 0; d < mu; ++d) o += 3 * (size_t)g.n[d];
  return o;
}
size_t own_fft_table_entries(const Geo& g) { return axis_offset(g, 4); }

__global__ void own_fft_table_kernel(double* __restrict__ table, int n, int r1, int r2) {
  const int pos = blockIdx.x * blockDim.x + threadIdx.x;
  if (pos >= n) return;
  const int k = pos / r2 + r1 * (pos % r2);  // frequency held at this position
  const double s = sinpi((double)k / (double)n);
  table[pos] = 4.0 * s * s;
  double sn, cs;
  sincospi(-2.0 * (double)pos / (double)n, &sn, &cs);
  reinterpret_cast<double2*>(table + n)[pos] = make_double2(cs, sn);
}

// ---- line pass: transforms along one axis whose elements are `es` apart; lines are (outer, inner) with inner < es ----------
// A block takes XB consecutive inner indices of one outer index: tile [n][XB] in shared memory between the two steps.
// Thread (j, ty): j = threadIdx.x % XB, ty = threadIdx.x / XB < TY.
enum { LINE_FWD = 0, LINE_INV = 1, LINE_FUSED = 2 };

struct LineArgs {
  int n, r1, r2;
  size_t es;            // element stride along the axis = number of inner indices
  size_t outer_stride;  // es * n
  int xb, ty;
  const double* p2_axis;   // position-ordered p^2 of this axis (FUSED)
  const double2* tw;       // twiddles of this axis
  // FUSED: p^2 of the other transformed axes from the inner index i = i0 + n0 (i1 + n1 i2)
  const double* p2_0; const double* p2_1; const double* p2_2;
  int n0, n1;
  double scale_p2max;
};

// The fused pass with 16-point FP64 transforms wants 164 registers (3 blocks of 128 threads per SM); capped at 128
// (a 128-byte spill) a fourth block fits.
template <class T, int MODE, int MAXR>
__global__ void __launch_bounds__(256, (MODE == LINE_FUSED && MAXR == 16) ? 2 : 1) fft_line_kernel(cplx_t<T>* __restrict__ w, LineArgs a) {
  using C = cplx_t<T>;
  extern __shared__ __align__(16) unsigned char line_smem[];
  C* tile = reinterpret_cast<C*>(line_smem);
  const int j = threadIdx.x % a.xb, ty = threadIdx.x / a.xb;
  const size_t inner = (size_t)blockIdx.x * a.xb + j;
  C* g = w + (size_t)blockIdx.y * a.outer_stride + inner;
  const int R1 = a.r1, R2 = a.r2, XB = a.xb;
  double p2_other = 0.0;
  if (MODE == LINE_FUSED) {
    unsigned q = (unsigned)inner;
    const int i0 = q % (unsigned)a.n0; q /= (unsigned)a.n0;
    const int i1 = q % (unsigned)a.n1;
    const int i2 = q / (unsigned)a.n1;
    p2_other = a.p2_0[i0] + a.p2_1[i1] + (a.p2_2 ? a.p2_2[i2] : 0.0);
  }
  if (R2 == 1) {  // the extent is one radix: everything in registers
    GF_R_CASES(R1, {
      if (MODE == LINE_FWD) fft_step<T, RR, false, false>(g, a.es, g, a.es, a.tw, 0);
      else if (MODE == LINE_INV) fft_step<T, RR, true, false>(g, a.es, g, a.es, a.tw, 0);
      else {
        C v[RR];
_Pragma("unroll")
        for (int m = 0; m < RR; ++m) v[m] = g[m * a.es];
        Dft<T, RR, false>::run(v);
_Pragma("unroll")
        for (int m = 0; m < RR; ++m) {
          const T f = factor_of<T>(a.scale_p2max, p2_other + a.p2_axis[m]);
          v[m].x *= f; v[m].y *= f;
        }
        Dft<T, RR, true>::run(v);
_Pragma("unroll")
        for (int m = 0; m < RR; ++m) g[m * a.es] = v[m];
      }
    });
    return;
  }
  if (MODE != LINE_INV) {
    // outer step, global -> tile: thread t2 = ty (one R1-point transform per column and t2)
    for (int t2 = ty; t2 < R2; t2 += a.ty) {
      GF_R_CASES(R1, fft_step<T, RR, false, true>(g + (size_t)t2 * a.es, (size_t)R2 * a.es, tile + t2 * XB + j,
                                                  (size_t)R2 * XB, a.tw, t2));
    }
    __syncthreads();
    for (int k1 = ty; k1 < R1; k1 += a.ty) {
      C* col = tile + (size_t)R2 * k1 * XB + j;
      if (MODE == LINE_FWD) {
        GF_R_CASES(R2, fft_step<T, RR, false, false>(col, (size_t)XB, g + (size_t)R2 * k1 * a.es, a.es, a.tw, 0));
      } else {  // inner step, factor, inverse inner step, all in registers; back into the tile
        GF_R_CASES(R2, {
          C v[RR];
_Pragma("unroll")
          for (int m = 0; m < RR; ++m) v[m] = col[m * XB];
          Dft<T, RR, false>::run(v);
_Pragma("unroll")
          for (int m = 0; m < RR; ++m) {
            const T f = factor_of<T>(a.scale_p2max, p2_other + a.p2_axis[R2 * k1 + m]);
            v[m].x *= f; v[m].y *= f;
          }
          Dft<T, RR, true>::run(v);
_Pragma("unroll")
          for (int m = 0; m < RR; ++m) {
            if (m > 0) {
              const double2 t = __ldg(a.tw + m * k1);
              const T wr = (T)t.x, wi = (T)(-t.y);
              const C z = v[m];
              v[m].x = z.x * wr - z.y * wi;
              v[m].y = z.x * wi + z.y * wr;
            }
            col[m * XB] = v[m];
          }
        });
      }
    }
    if (MODE == LINE_FWD) return;
    __syncthreads();
  } else {
    // inverse inner step, global -> tile
    for (int k1 = ty; k1 < R1; k1 += a.ty) {
      GF_R_CASES(R2, fft_step<T, RR, true, true>(g + (size_t)R2 * k1 * a.es, a.es, tile + (size_t)R2 * k1 * XB + j,
                                                 (size_t)XB, a.tw, k1));
    }
    __syncthreads();
  }
  // inverse outer step, tile -> global
  for (int t2 = ty; t2 < R2; t2 += a.ty) {
    GF_R_CASES(R1, fft_step<T, RR, true, false>(tile + t2 * XB + j, (size_t)R2 * XB, g + (size_t)t2 * a.es,
                                                (size_t)R2 * a.es, a.tw, 0));
  }
}

// ---- plane pass: the (x,y) plane of one (z,t,field) in shared memory, x lines then y lines (forward) or back -----------------
struct PlaneArgs {
  int nx, ny;
  int rx1, rx2, ry1, ry2;
  int row;  // row stride of the tile in elements (>= nx)
  const double2* twx; const double2* twy;
};

template <bool V> struct DirTag { static constexpr bool value = V; };

// 128 threads per block: three blocks (three 66 KB tiles on a 64 x 64 FP64 plane) share an SM, so one block's load and
// store phases overlap the others' register steps.
constexpr int PLANE_THREADS = 128;

template <class T, bool INV, int MAXR>
__global__ void __launch_bounds__(MAXR <= 8 ? 2 * PLANE_THREADS : PLANE_THREADS, 3)
fft_plane_kernel(cplx_t<T>* __restrict__ w, PlaneArgs a) {
  using C = cplx_t<T>;
  extern __shared__ __align__(16) unsigned char plane_smem[];
  C* tile = reinterpret_cast<C*>(plane_smem);
  const int nx = a.nx, ny = a.ny, row = a.row;
  C* g = w + (size_t)blockIdx.x * nx * ny;
  const int nthreads = blockDim.x;
  // The y steps at the two ends of the pass work straight on global memory (a y step's lanes are consecutive in x:
  // 512-byte runs): the forward pass writes the results of its last step to the field, the inverse pass reads the
  // operands of its first step from it, so that end of the pass needs no tile copy and no barrier.  The x steps stay in
  // the tile on the load side: measured on the cfg4 lattice, an x step that READS global memory (8 lanes per 128-byte
  // line) costs more than the tile copy it saves (forward pass 1.04 ms against 0.99 ms), one that WRITES it does not
  // (inverse pass 0.95 ms against 1.03 ms with a tile copy at the end).  Forward 0.99 -> 0.91 ms, inverse 0.99 -> 0.95 ms.
  // x lines: line y, elements base[y*rs + pos].  In the tile the work item is (sub, y) with y fastest: neighbouring lanes
  // are one row apart, and the row stride is odd, so they fall on different banks whatever the stride along the line is.
  // Against global memory it is (sub, y) with sub fastest: the rx2 lanes of a row read / write rx2 consecutive elements
  // (whole 128-byte lines for rx2 = 8 in FP64); the tile side of that step is conflict-free because row = 1 mod 8.
  auto x_outer = [&](auto inv_tag, const C* src, int srs, C* dst, int drs, bool sub_fastest) {
    constexpr bool I = decltype(inv_tag)::value;
    for (int it = threadIdx.x; it < ny * a.rx2; it += nthreads) {
      int t2, y;
      if (sub_fastest) { y = it / a.rx2; t2 = it - y * a.rx2; }
      else { t2 = it / ny; y = it - t2 * ny; }
      GF_R_CASES(a.rx1, fft_step<T, RR, I, !I>(src + y * srs + t2, (size_t)a.rx2, dst + y * drs + t2, (size_t)a.rx2, a.twx, t2));
    }
  };
  auto x_inner = [&](auto inv_tag) {
    constexpr bool I = decltype(inv_tag)::value;
    for (int it = threadIdx.x; it < ny * a.rx1; it += nthreads) {
      const int k1 = it / ny, y = it - k1 * ny;
      C* p = tile + y * row + a.rx2 * k1;
      GF_R_CASES(a.rx2, fft_step<T, RR, I, I>(p, (size_t)1, p, (size_t)1, a.twx, k1));
    }
  };
  // y lines: line x, elements base[pos*rs + x]; work item -> (sub, x) with x fastest (contiguous in global memory too)
  auto y_outer = [&](auto inv_tag, const C* src, int srs, C* dst, int drs) {
    constexpr bool I = decltype(inv_tag)::value;
    for (int it = threadIdx.x; it < nx * a.ry2; it += nthreads) {
      const int t2 = it / nx, x = it - t2 * nx;
      GF_R_CASES(a.ry1, fft_step<T, RR, I, !I>(src + t2 * srs + x, (size_t)a.ry2 * srs, dst + t2 * drs + x, (size_t)a.ry2 * drs,
                                                a.twy, t2));
    }
  };
  auto y_inner = [&](auto inv_tag, const C* src, int srs, C* dst, int drs) {
    constexpr bool I = decltype(inv_tag)::value;
    for (int it = threadIdx.x; it < nx * a.ry1; it += nthreads) {
      const int k1 = it / nx, x = it - k1 * nx;
      GF_R_CASES(a.ry2, fft_step<T, RR, I, I>(src + a.ry2 * k1 * srs + x, (size_t)srs, dst + a.ry2 * k1 * drs + x, (size_t)drs,
                                               a.twy, k1));
    }
  };
  using Fwd = DirTag<false>;
  using Inv = DirTag<true>;
  auto load_tile = [&]() {  // global -> tile without a register round trip
    for (int i = threadIdx.x; i < nx * ny; i += nthreads) {
      const int y = i / nx, x = i - y * nx;
      const unsigned dst = (unsigned)__cvta_generic_to_shared(tile + y * row + x);
      if (sizeof(C) == 16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(g + i) : "memory");
      else asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(g + i) : "memory");
    }
    asm volatile("cp.async.wait_all;" ::: "memory");
    __syncthreads();
  };
  if (!INV) {
    load_tile();
    x_outer(Fwd{}, tile, row, tile, row, false); __syncthreads();
    if (a.rx2 > 1) { x_inner(Fwd{}); __syncthreads(); }
    if (a.ry2 > 1) {
      y_outer(Fwd{}, tile, row, tile, row); __syncthreads();
      y_inner(Fwd{}, tile, row, g, nx);
    } else {
      y_outer(Fwd{}, tile, row, g, nx);
    }
  } else {
    if (a.ry2 > 1) {
      y_inner(Inv{}, g, nx, tile, row); __syncthreads();
      y_outer(Inv{}, tile, row, tile, row); __syncthreads();
    } else {
      y_outer(Inv{}, g, nx, tile, row); __syncthreads();
    }
    if (a.rx2 > 1) { x_inner(Inv{}); __syncthreads(); }
    x_outer(Inv{}, tile, row, g, nx, true);
  }
}

// ---- host side -------------------------------------------------------------------------------------------------------------
constexpr size_t OWN_FFT_MAX_SMEM = 200 * 1024;

static bool make_shape(const Geo& g, int gauge, FftShape* s) {
  const int nd = gauge == 0 ? 4 : 3;
  for (int d = 0; d < nd; ++d)
    if (!split_extent(g.n[d], &s->ax[d])) return false;
  if (nd == 3) s->ax[3] = AxisSplit{g.n[3], 0, 0};
  return true;
}

static int plane_row(int nx) { return nx + 1; }  // odd row stride (extents are even): neighbouring rows on different banks

static int line_xb(size_t inner, int n, int r2, size_t csize) {
  // consecutive inner indices per block: rows of up to 256 B (two full lines per row), block <= 256 threads; small
  // tiles (32 KB at n = 128) so that several blocks share an SM and their load / step / store phases overlap
  int xb = 1;
  while (xb * 2 <= 256 / r2 && inner % (size_t)(xb * 2) == 0 && (size_t)(xb * 2) * csize <= 256) xb *= 2;
  return xb;
}

bool own_fft_supported(const Geo& g, int gauge, int prec) {
  FftShape s;
  if (!make_shape(g, gauge, &s)) return false;
  const size_t csize = prec == 0 ? 16 : 8;
  return (size_t)plane_row(g.n[0]) * g.n[1] * csize <= OWN_FFT_MAX_SMEM;
}

cudaError_t launch_own_fft_tables(const KernelArgs& a, double* table) {
  FftShape s;
  if (!make_shape(a.geo, a.gauge, &s)) return cudaErrorInvalidValue;
  const int nd = a.gauge == 0 ? 4 : 3;
  for (int d = 0; d < nd; ++d) {
    const int n = a.geo.n[d];
    own_fft_table_kernel<<<(n + 127) / 128, 128, 0, a.stream>>>(table + axis_offset(a.geo, d), n, s.ax[d].r1, s.ax[d].r2);
  }
  return cudaGetLastError();
}

template <class T>
static cudaError_t plane_pass(const KernelArgs& a, const FftShape& s, void* w, const double* table, bool inverse) {
  using C = cplx_t<T>;
  const Geo& g = a.geo;
  PlaneArgs p;
  p.nx = g.n[0]; p.ny = g.n[1];
  p.rx1 = s.ax[0].r1; p.rx2 = s.ax[0].r2; p.ry1 = s.ax[1].r1; p.ry2 = s.ax[1].r2;
  p.row = plane_row(g.n[0]);
  p.twx = reinterpret_cast<const double2*>(table + axis_offset(g, 0) + g.n[0]);
  p.twy = reinterpret_cast<const double2*>(table + axis_offset(g, 1) + g.n[1]);
  const size_t smem = (size_t)p.row * p.ny * sizeof(C);
  const unsigned planes = (unsigned)((size_t)g.n[2] * g.n[3] * 4);
  // work items per step: ny*rx2 ... nx*ry1; one block of up to 256 threads per plane
  int items = p.ny * p.rx2;
  if (p.nx * p.ry2 > items) items = p.nx * p.ry2;
  const bool small = p.rx1 <= 8 && p.ry1 <= 8;  // r1 >= r2: the largest radix of the plane
  int threads = 32;
  while (threads < items && threads < (small ? 2 * PLANE_THREADS : PLANE_THREADS)) threads *= 2;
  auto go = [&](auto k) {
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)OWN_FFT_MAX_SMEM);
    if (e != cudaSuccess) return e;
    k<<<planes, threads, smem, a.stream>>>((C*)w, p);
    return cudaGetLastError();
  };
  if (inverse) return small ? go(fft_plane_kernel<T, true, 8>) : go(fft_plane_kernel<T, true, 16>);
  return small ? go(fft_plane_kernel<T, false, 8>) : go(fft_plane_kernel<T, false, 16>);
}

template <class T>
static cudaError_t line_pass(const KernelArgs& a, const FftShape& s, void* w, const double* table, int axis, int mode,
                             double scale_p2max) {
  using C = cplx_t<T>;
  const Geo& g = a.geo;
  LineArgs l;
  l.n = g.n[axis]; l.r1 = s.ax[axis].r1; l.r2 = s.ax[axis].r2;
  l.es = axis == 2 ? (size_t)g.n[0] * g.n[1] : (size_t)g.n[0] * g.n[1] * g.n[2];
  l.outer_stride = l.es * l.n;
  const size_t outer = axis == 2 ? (size_t)g.n[3] * 4 : 4;
  l.xb = line_xb(l.es, l.n, l.r2, sizeof(C));
  l.ty = l.r2;
  if (l.r2 == 1) {  // register-only path: no tile; let a block take up to 128 lines
    l.ty = 1;
    while (l.xb * 2 <= 128 && l.es % (size_t)(l.xb * 2) == 0) l.xb *= 2;
  }
  l.p2_axis = table + axis_offset(g, axis);
  l.tw = reinterpret_cast<const double2*>(table + axis_offset(g, axis) + l.n);
  l.p2_0 = table + axis_offset(g, 0);
  l.p2_1 = table + axis_offset(g, 1);
  l.p2_2 = axis == 3 ? table + axis_offset(g, 2) : nullptr;
  l.n0 = g.n[0]; l.n1 = g.n[1];
  l.scale_p2max = scale_p2max;
  const size_t smem = l.r2 == 1 ? 0 : (size_t)l.n * l.xb * sizeof(C);
  const dim3 grid((unsigned)(l.es / l.xb), (unsigned)outer);
  const int threads = l.xb * l.ty;
  const bool small = l.r1 <= 8;
  auto go = [&](auto k) {
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    if (e != cudaSuccess) return e;
    k<<<grid, threads, smem, a.stream>>>((C*)w, l);
    return cudaGetLastError();
  };
  if (mode == LINE_FWD) return small ? go(fft_line_kernel<T, LINE_FWD, 8>) : go(fft_line_kernel<T, LINE_FWD, 16>);
  if (mode == LINE_INV) return small ? go(fft_line_kernel<T, LINE_INV, 8>) : go(fft_line_kernel<T, LINE_INV, 16>);
  return small ? go(fft_line_kernel<T, LINE_FUSED, 8>) : go(fft_line_kernel<T, LINE_FUSED, 16>);
}

template <class T>
static cudaError_t own_update_T(const KernelArgs& a, void* w, const double* table, double alpha, int* launches) {
  FftShape s;
  if (!make_shape(a.geo, a.gauge, &s)) return cudaErrorInvalidValue;
  const bool landau = a.gauge == 0;
  // (alpha/2) / N * p^2_max with N = the transform's size and p^2_max = 4 per transformed direction (readings B2-B4)
  const double N = (double)a.geo.n[0] * a.geo.n[1] * a.geo.n[2] * (landau ? a.geo.n[3] : 1);
  const double scale_p2max = 0.5 * alpha / N * (landau ? 16.0 : 12.0);
  cudaError_t e = plane_pass<T>(a, s, w, table, false);
  if (e != cudaSuccess) return e;
  if (landau) {
    e = line_pass<T>(a, s, w, table, 2, LINE_FWD, 0.0);
    if (e == cudaSuccess) e = line_pass<T>(a, s, w, table, 3, LINE_FUSED, scale_p2max);
    if (e == cudaSuccess) e = line_pass<T>(a, s, w, table, 2, LINE_INV, 0.0);
    *launches += 3;
  } else {
    e = line_pass<T>(a, s, w, table, 2, LINE_FUSED, scale_p2max);
    *launches += 1;
  }
  if (e != cudaSuccess) return e;
  e = plane_pass<T>(a, s, w, table, true);
  *launches += 2;
  return e;
}

cudaError_t launch_own_fft_update(const KernelArgs& a, void* w, const double* table, double alpha, int* launches) {
  return a.prec == 0 ? own_update_T<double>(a, w, table, alpha, launches) : own_update_T<float>(a, w, table, alpha, launches);
}

}  // namespace gf
