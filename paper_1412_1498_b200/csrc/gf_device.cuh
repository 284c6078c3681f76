// gf_device.cuh — device-side building blocks of libgf (sm_100a): complex 3x3 arithmetic in registers, the internal
// link layout, checkerboard indexing, the SU(2) subgroup / overrelaxation step and row reconstruction.
// Equation and line numbers refer to arXiv:1412.1498 as PAPER.md:<line>; readings A1-A20 are listed in DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

namespace gf {

// ---- scalar traits ------------------------------------------------------------------------------------------------------
template <class T> struct Cplx;
template <> struct Cplx<double> { using type = double2; };
template <> struct Cplx<float> { using type = float2; };
template <class T> using cplx_t = typename Cplx<T>::type;

template <class T> __device__ __forceinline__ cplx_t<T> mk(T a, T b) { cplx_t<T> z; z.x = a; z.y = b; return z; }

// z += a*b
template <class C> __device__ __forceinline__ void cfma(C& z, const C a, const C b) {
  z.x = fma(a.x, b.x, z.x); z.x = fma(-a.y, b.y, z.x);
  z.y = fma(a.x, b.y, z.y); z.y = fma(a.y, b.x, z.y);
}
// z += a*conj(b)
template <class C> __device__ __forceinline__ void cfma_cj(C& z, const C a, const C b) {
  z.x = fma(a.x, b.x, z.x); z.x = fma(a.y, b.y, z.x);
  z.y = fma(a.y, b.x, z.y); z.y = fma(-a.x, b.y, z.y);
}
// a*b
template <class C> __device__ __forceinline__ C cmul(const C a, const C b) {
  C z; z.x = a.x * b.x; z.x = fma(-a.y, b.y, z.x); z.y = a.x * b.y; z.y = fma(a.y, b.x, z.y); return z;
}
// conj(a*b - c*d)
template <class C> __device__ __forceinline__ C cross_cj(const C a, const C b, const C c, const C d) {
  C z;
  z.x = a.x * b.x; z.x = fma(-a.y, b.y, z.x); z.x = fma(-c.x, d.x, z.x); z.x = fma(c.y, d.y, z.x);
  z.y = c.x * d.y; z.y = fma(c.y, d.x, z.y); z.y = fma(-a.x, b.y, z.y); z.y = fma(-a.y, b.x, z.y);
  return z;
}
// row 2 = conj(row0 x row1): third row of an SU(3) matrix from the stored two (12-real storage, A13)
template <class C> __device__ __forceinline__ void rebuild_row2(C (&u)[9]) {
  u[6] = cross_cj(u[1], u[5], u[2], u[4]);
  u[7] = cross_cj(u[2], u[3], u[0], u[5]);
  u[8] = cross_cj(u[0], u[4], u[1], u[3]);
}

// ---- geometry and the internal layout ------------------------------------------------------------------------------------
// Internal layout ("AoSoA-32"): the V/2 sites of one parity are numbered by the checkerboard index
//   cb = (x + nx*(y + ny*(z + nz*t))) / 2                                   (even/odd kept separate)
// and grouped in blocks of 32 consecutive cb.  One block of one direction is NELEM*32 complex numbers, element-major:
//   links[parity][cb/32][mu][elem][cb%32]          elem = 3*row+col, NELEM = 9 (18 reals) or 6 (12 reals: rows 0,1)
// so a warp that owns 32 consecutive sites reads element e of link mu as one contiguous 32*sizeof(complex) run
// (512 B in FP64, full 32-byte sectors), and the four forward links of those sites are one contiguous
// 4*NELEM*32*sizeof(complex) chunk (18 KB for FP64/18).  The last block is padded when V/2 is not a multiple of 32.
struct Geo {
  int n[4];     // nx, ny, nz, nt
  int nh0;      // nx/2: sites of one parity per x-row
  int vh;       // V/2 sites per parity
  int nblk;     // ceil(vh/32)
  int s1, s2, s3;  // checkerboard strides of a step in y, z, t: nh0, nh0*ny, nh0*ny*nz
};

template <int NELEM>
__device__ __forceinline__ size_t link_offset(const Geo& g, int parity, int cb, int mu) {
  return ((((size_t)parity * g.nblk + (size_t)(cb >> 5)) * 4 + mu) * NELEM) * 32 + (cb & 31);
}

struct Site {
  int xh, y, z, t, x;
};
__device__ __forceinline__ Site site_of(const Geo& g, int parity, int cb) {
  Site s;
  unsigned q = (unsigned)cb;
  s.xh = q % (unsigned)g.nh0; q /= (unsigned)g.nh0;
  s.y = q % (unsigned)g.n[1]; q /= (unsigned)g.n[1];
  s.z = q % (unsigned)g.n[2];
  s.t = q / (unsigned)g.n[2];
  s.x = 2 * s.xh + ((s.y + s.z + s.t + parity) & 1);
  return s;
}
// checkerboard index (in the OTHER parity) of x - mu, periodic
__device__ __forceinline__ int cb_down(const Geo& g, const Site& s, int cb, int mu) {
  switch (mu) {
    case 0: {
      int xm = s.x == 0 ? g.n[0] - 1 : s.x - 1;
      return cb - s.xh + (xm >> 1);
    }
    case 1: return s.y == 0 ? cb + g.s1 * (g.n[1] - 1) : cb - g.s1;
    case 2: return s.z == 0 ? cb + g.s2 * (g.n[2] - 1) : cb - g.s2;
    default: return s.t == 0 ? cb + g.s3 * (g.n[3] - 1) : cb - g.s3;
  }
}

// ---- 8-real storage (NELEM = 4; "Elems = 4", 144, 174; reading A23) --------------------------------------------
// Stored: a2, a3, b1 and the two phases arg a1, arg c1 for the rows a, b, c of the link.  With N = |a2|^2 + |a3|^2:
//   |a1| = sqrt(1 - N), |c1| = sqrt(N - |b1|^2)  (row a and column 0 have unit norm);
//   (b2, b3) = alpha (a2, a3) + beta (-conj a3, conj a2), alpha = -conj(a1) b1 / N, beta = conj(c1) / N;  c = conj(a x b).
// A phase theta is kept as its stereographic coordinate t = tan(theta/2), a rational chart of the unit circle:
//   e^{i theta} = ((1 - t^2) + 2 i t) / (1 + t^2),      t = y / (|z| + x)  (x >= 0)  or  (|z| - x) / y  (x < 0),
// so that a load costs divisions instead of two sincos and a store a square root and a division instead of atan2
// (d theta = 2 dt / (1 + t^2): a relative rounding of t moves theta by at most one rounding, also for |t| >> 1).
// Undefined for N = 0 (block-diagonal links); rounding is amplified by 1/N near it: a store with N below
// Domain8<T>::n_min raises gf_domain_flag, which gf_measure / gf_get_links_host report as GF_ENUMERIC.
__device__ __forceinline__ double hypot2_(double x, double y) { return x * x + y * y; }
__device__ __forceinline__ float hypot2_(float x, float y) { return x * x + y * y; }
template <class T> struct Domain8;
template <> struct Domain8<double> { static constexpr double n_min = 1e-6, t_max = 1e75; };
template <> struct Domain8<float> { static constexpr float n_min = 1e-3f, t_max = 1e9f; };
static __device__ unsigned gf_domain_flag = 0;  // one per translation unit; only gf_kernels.cu stores 8-real links

// t = tan(arg(z) / 2) for z = x + i y (0 for z = 0)
template <class T>
__device__ __forceinline__ T phase_to_t(T x, T y) {
  const T m = sqrt(x * x + y * y);
  const bool right = x >= T(0);
  const T num = right ? y : m - x, den = right ? m + x : y;
  T t = den != T(0) ? num / den : (num != T(0) ? Domain8<T>::t_max : T(0));
  return fmin(fmax(t, -Domain8<T>::t_max), Domain8<T>::t_max);
}

template <class T, class C, bool ROW2 = true>
__device__ __forceinline__ void decode8(const C a2, const C a3, const C b1, const C phases, C (&u)[9]) {
  const T N = hypot2_(a2.x, a2.y) + hypot2_(a3.x, a3.y);
  const T ta = phases.x, tc = phases.y;
  const T da = T(1) + ta * ta, dc = T(1) + tc * tc;
  // one division for 1/da, 1/dc and 1/N
  const T inv = T(1) / (da * dc * N);
  const T inv_da = inv * dc * N, inv_dc = inv * da * N, invN = inv * da * dc;
  const T ra = sqrt(fmax(T(0), T(1) - N)) * inv_da;
  const C a1 = mk<T>(ra * (T(1) - ta * ta), ra * (ta + ta));
  const T rc = sqrt(fmax(T(0), N - hypot2_(b1.x, b1.y))) * inv_dc;
  const C c1 = mk<T>(rc * (T(1) - tc * tc), rc * (tc + tc));
  // alpha = -conj(a1) b1 / N, beta = conj(c1) / N
  const C alpha = mk<T>(-(a1.x * b1.x + a1.y * b1.y) * invN, -(a1.x * b1.y - a1.y * b1.x) * invN);
  const C beta = mk<T>(c1.x * invN, -c1.y * invN);
  u[0] = a1; u[1] = a2; u[2] = a3; u[3] = b1;
  // b2 = alpha a2 - beta conj(a3);  b3 = alpha a3 + beta conj(a2)
  u[4] = mk<T>(alpha.x * a2.x - alpha.y * a2.y - (beta.x * a3.x + beta.y * a3.y),
               alpha.x * a2.y + alpha.y * a2.x - (beta.y * a3.x - beta.x * a3.y));
  u[5] = mk<T>(alpha.x * a3.x - alpha.y * a3.y + (beta.x * a2.x + beta.y * a2.y),
               alpha.x * a3.y + alpha.y * a3.x + (beta.y * a2.x - beta.x * a2.y));
  if (ROW2) rebuild_row2(u);
}

// rows of a product that a store of this storage format needs: 18 reals 3, 12 reals 2, 8 reals 3 (it reads c1)
template <int NELEM> struct LinkRows { static constexpr int value = NELEM == 6 ? 2 : 3; };

// ---- link load / store in the internal layout ------------------------------------------------------------------------------
// STRIDE: distance between consecutive elements of one link (32 in the global layout; THREADS in the shared staging area)
template <int NELEM, bool FULL, int STRIDE = 32, class C>
__device__ __forceinline__ void load_link(const C* __restrict__ p, C (&u)[9]) {
  if constexpr (NELEM == 4) {
    using T = decltype(u[0].x);
    decode8<T>(p[0], p[STRIDE], p[2 * STRIDE], p[3 * STRIDE], u);
  } else {
#pragma unroll
    for (int e = 0; e < NELEM; ++e) u[e] = p[e * STRIDE];
    if (NELEM == 6 && FULL) rebuild_row2(u);
  }
}
template <int NELEM, class C>
__device__ __forceinline__ void store_link(C* __restrict__ p, const C (&u)[9]) {
  if constexpr (NELEM == 4) {
    using T = decltype(u[0].x);
    p[0] = u[1]; p[32] = u[2]; p[64] = u[3];
    p[96] = mk<T>(phase_to_t(u[0].x, u[0].y), phase_to_t(u[6].x, u[6].y));
    if (hypot2_(u[1].x, u[1].y) + hypot2_(u[2].x, u[2].y) < Domain8<T>::n_min) atomicOr(&gf_domain_flag, 1u);
  } else {
#pragma unroll
    for (int e = 0; e < NELEM; ++e) p[e * 32] = u[e];
  }
}

// ---- SU(2) subgroup step with overrelaxation -------------------------------------------------------------------------------
template <class T> __device__ __forceinline__ T tiny_of();
template <> __device__ __forceinline__ double tiny_of<double>() { return 2.2250738585072014e-308 * 1152921504606846976.0; }
template <> __device__ __forceinline__ float tiny_of<float>() { return 1.17549435e-38f * 1152921504606846976.0f; }

__device__ __forceinline__ void sincos_(double a, double* s, double* c) { sincos(a, s, c); }
__device__ __forceinline__ void sincos_(float a, float* s, float* c) { sincosf(a, s, c); }
__device__ __forceinline__ double atan2_(double y, double x) { return atan2(y, x); }
__device__ __forceinline__ float atan2_(float y, float x) { return atan2f(y, x); }
__device__ __forceinline__ double sqrt_(double x) { return sqrt(x); }
__device__ __forceinline__ float sqrt_(float x) { return sqrtf(x); }

// The quaternion (c; q1,q2,q3) of g^omega where g maximises Re Tr[g M] over SU(2) for the 2x2 block M of K
// (eqs. 1.4-1.6 on the SU(2)-proportional part r of the block, reading A5; exact power, principal branch, A6):
//   r0 = Re(M00+M11), r1 = -Im(M01+M10), r2 = Re(M10-M01), r3 = -Im(M00-M11);   a = r/|r|;
//   phi = atan2(|a_vec|, a0);  g^omega = (cos(omega phi); a_vec sin(omega phi)/|a_vec|).
// |r| cancels in both phi and the direction of a_vec, so it is never formed: phi = atan2(S, r0), S = |r_vec|.
#ifndef GF_SU2_INLINE
#define GF_SU2_INLINE __forceinline__
#endif
template <class T>
__device__ GF_SU2_INLINE void su2_overrelax(T r0, T r1, T r2, T r3, T omega, T& c, T& q1, T& q2, T& q3) {
  const T S2 = r1 * r1 + r2 * r2 + r3 * r3;
  const T S = sqrt_(S2);
  if (S <= tiny_of<T>() * fabs(r0)) {  // reading A7 (includes |r| = 0 and phi = pi: g = 1)
    if (r0 > T(0)) {
      const T phi = atan2_(S, r0);
      T sn;
      sincos_(omega * phi, &sn, &c);
      const T f = omega / r0;  // limit of sin(omega phi)/s, with a_k = r_k/|r|, |r| -> r0
      q1 = r1 * f; q2 = r2 * f; q3 = r3 * f;
    } else {
      c = T(1); q1 = q2 = q3 = T(0);
    }
    return;
  }
  const T phi = atan2_(S, r0);
  T sn;
  sincos_(omega * phi, &sn, &c);
  const T f = sn / S;
  q1 = r1 * f; q2 = r2 * f; q3 = r3 * f;
}

// Variant (GF_OPT_OVR_SERIES, reading A21; PAPER.md:50 cites Mandula & Ogilvie for g^omega, who truncate its binomial
// series): g^omega ~ sum_{n<=N} binom(omega,n) (g-1)^n, projected back to SU(2) by normalisation.  With a = r/|r| =
// (a0; a_vec), every power of g - 1 is P0 + i Pv (a_vec.sigma), and (P0, Pv)(g - 1) = (P0 (a0-1) - Pv |a_vec|^2,
// P0 + (a0-1) Pv); no division by |a_vec|, so the limit a_vec -> 0 needs no special case.
template <class T>
__device__ __forceinline__ void su2_overrelax_series(T r0, T r1, T r2, T r3, T omega, int order, T& c, T& q1, T& q2,
                                                     T& q3) {
  const T S2 = r1 * r1 + r2 * r2 + r3 * r3;
  const T n2 = r0 * r0 + S2;
  if (!(n2 > T(0))) { c = T(1); q1 = q2 = q3 = T(0); return; }  // reading A7
  const T inv = T(1) / sqrt_(n2);
  const T u0 = r0 * inv - T(1), s2 = S2 * inv * inv;
  T P0 = T(1), Pv = T(0), A0 = T(0), Av = T(0), b = T(1);
  for (int n = 0; n <= order; ++n) {
    A0 = fma(b, P0, A0); Av = fma(b, Pv, Av);
    const T t0 = P0 * u0 - Pv * s2, tv = P0 + u0 * Pv;
    P0 = t0; Pv = tv;
    b = b * (omega - T(n)) / T(n + 1);
  }
  const T norm2 = A0 * A0 + Av * Av * s2;
  if (!(norm2 > T(0))) { c = T(1); q1 = q2 = q3 = T(0); return; }
  const T f = T(1) / sqrt_(norm2);
  c = A0 * f;
  const T fv = Av * f * inv;  // a_k = r_k / |r|
  q1 = r1 * fv; q2 = r2 * fv; q3 = r3 * fv;
}

// One subgroup step on rows/cols (I,J): K <- gK, G <- gG with g = [[c+i q3, q2+i q1], [-q2+i q1, c-i q3]] embedded.
// K is in precision T; G may be kept in a lower precision TG (g is rounded once per step).
// TS: precision in which g^omega is evaluated from r.  r itself is always formed from K in precision T (the
// cancellation in the sum of eight links is what is ill-conditioned, not the map r -> g^omega, whose relative
// condition number is O(1) on the direction r/|r| and omega <= 2 on the angle); with FP32 links TS = float puts
// sqrt / atan2 / sincos / the division on the FP32 units while K(x) and K <- gK stay FP64.
// SERIES: g^omega by the truncated series of order `order` instead of the exact power.
// r2min (optional): receives min(*r2min, |r|^2) - the conditioning of this step (see FastPath in gf_kernels.cu).
template <int I, int J, bool UPDATE_K, bool SERIES = false, class TS = void, class T, class C, class CG>
__device__ __forceinline__ void su2_step(C (&K)[9], CG (&G)[9], T omega, int order = 0, T* r2min = nullptr) {
  using TG = decltype(G[0].x);
  using TE = typename std::conditional<std::is_void<TS>::value, T, TS>::type;
  const TE r0 = (TE)(K[I * 3 + I].x + K[J * 3 + J].x);
  const TE r1 = (TE)(-(K[I * 3 + J].y + K[J * 3 + I].y));
  const TE r2 = (TE)(K[J * 3 + I].x - K[I * 3 + J].x);
  const TE r3 = (TE)(-(K[I * 3 + I].y - K[J * 3 + J].y));
  if (r2min) *r2min = fmin(*r2min, (T)(r0 * r0 + r1 * r1 + r2 * r2 + r3 * r3));
  TE ce, e1, e2, e3;
  if (SERIES) su2_overrelax_series(r0, r1, r2, r3, (TE)omega, order, ce, e1, e2, e3);
  else su2_overrelax(r0, r1, r2, r3, (TE)omega, ce, e1, e2, e3);
  if (UPDATE_K) {
    const T c = (T)ce, q1 = (T)e1, q2 = (T)e2, q3 = (T)e3;
    const C g00 = mk<T>(c, q3), g01 = mk<T>(q2, q1), g10 = mk<T>(-q2, q1), g11 = mk<T>(c, -q3);
#pragma unroll
    for (int col = 0; col < 3; ++col) {
      const C ki = K[I * 3 + col], kj = K[J * 3 + col];
      C a = cmul(g00, ki); cfma(a, g01, kj);
      C b = cmul(g10, ki); cfma(b, g11, kj);
      K[I * 3 + col] = a; K[J * 3 + col] = b;
    }
  }
  const TG cg = (TG)ce, p1 = (TG)e1, p2 = (TG)e2, p3 = (TG)e3;
  const CG h00 = mk<TG>(cg, p3), h01 = mk<TG>(p2, p1), h10 = mk<TG>(-p2, p1), h11 = mk<TG>(cg, -p3);
#pragma unroll
  for (int col = 0; col < 3; ++col) {
    const CG gi = G[I * 3 + col], gj = G[J * 3 + col];
    CG a = cmul(h00, gi); cfma(a, h01, gj);
    CG b = cmul(h10, gi); cfma(b, h11, gj);
    G[I * 3 + col] = a; G[J * 3 + col] = b;
  }
}

// G = g3 g2 g1 for one site from its K (Algorithm 1 l.5-6; subgroup order (0,1),(1,2),(0,2), reading A4; A8)
// FINAL_K: also carry K through the last step, so that on return K = G K_in (= K(x) of the updated links).
template <class T, bool FINAL_K = false, bool SERIES = false, class TS = void, class C, class CG>
__device__ __forceinline__ void site_gauge_rotation(C (&K)[9], CG (&G)[9], T omega, int order = 0, T* r2min = nullptr) {
  using TG = decltype(G[0].x);
#pragma unroll
  for (int e = 0; e < 9; ++e) G[e] = mk<TG>((e % 4 == 0) ? TG(1) : TG(0), TG(0));
  su2_step<0, 1, true, SERIES, TS>(K, G, omega, order, r2min);
  su2_step<1, 2, true, SERIES, TS>(K, G, omega, order, r2min);
  su2_step<0, 2, FINAL_K, SERIES, TS>(K, G, omega, order, r2min);
}

// rows 0..NROW-1 of G.U
template <int NROW, class C>
__device__ __forceinline__ void mul_left(const C (&G)[9], const C (&u)[9], C (&out)[9]) {
#pragma unroll
  for (int i = 0; i < NROW; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      C z = cmul(G[i * 3], u[j]);
      cfma(z, G[i * 3 + 1], u[3 + j]);
      cfma(z, G[i * 3 + 2], u[6 + j]);
      out[i * 3 + j] = z;
    }
}
// rows 0..NROW-1 of U.G^dagger  (needs only rows 0..NROW-1 of U)
template <int NROW, class C>
__device__ __forceinline__ void mul_right_adj(const C (&u)[9], const C (&G)[9], C (&out)[9]) {
#pragma unroll
  for (int i = 0; i < NROW; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      C z;
      z.x = u[i * 3].x * G[j * 3].x; z.x = fma(u[i * 3].y, G[j * 3].y, z.x);
      z.y = u[i * 3].y * G[j * 3].x; z.y = fma(-u[i * 3].x, G[j * 3].y, z.y);
      cfma_cj(z, u[i * 3 + 1], G[j * 3 + 1]);
      cfma_cj(z, u[i * 3 + 2], G[j * 3 + 2]);
      out[i * 3 + j] = z;
    }
}

// Gram-Schmidt on rows 0,1; row 2 = conj(row0 x row1)  (reunitarisation, reading A12)
template <class T, class C>
__device__ __forceinline__ void reunitarize(C (&u)[9]) {
  T n0 = u[0].x * u[0].x + u[0].y * u[0].y + u[1].x * u[1].x + u[1].y * u[1].y + u[2].x * u[2].x + u[2].y * u[2].y;
  T i0 = T(1) / sqrt_(n0);
#pragma unroll
  for (int j = 0; j < 3; ++j) { u[j].x *= i0; u[j].y *= i0; }
  C p = mk<T>(T(0), T(0));
#pragma unroll
  for (int j = 0; j < 3; ++j) {  // p = sum conj(row0_j) row1_j
    p.x = fma(u[j].x, u[3 + j].x, p.x); p.x = fma(u[j].y, u[3 + j].y, p.x);
    p.y = fma(u[j].x, u[3 + j].y, p.y); p.y = fma(-u[j].y, u[3 + j].x, p.y);
  }
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    u[3 + j].x -= p.x * u[j].x - p.y * u[j].y;
    u[3 + j].y -= p.x * u[j].y + p.y * u[j].x;
  }
  T n1 = u[3].x * u[3].x + u[3].y * u[3].y + u[4].x * u[4].x + u[4].y * u[4].y + u[5].x * u[5].x + u[5].y * u[5].y;
  T i1 = T(1) / sqrt_(n1);
#pragma unroll
  for (int j = 0; j < 3; ++j) { u[3 + j].x *= i1; u[3 + j].y *= i1; }
  rebuild_row2(u);
}

// deterministic block sums (warp shuffles, then one shared-memory hop between warps; FP64 in both precisions)
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Sum of (f, q) over the THREADS threads of the block; valid in thread 0.  Every thread of the block must call it.
template <int THREADS>
__device__ __forceinline__ void block_sum2(double& f, double& q) {
  static_assert(THREADS % 32 == 0 && THREADS <= 1024, "whole warps");
  constexpr int NW = THREADS / 32;
  f = warp_sum(f);
  q = warp_sum(q);
  if (NW == 1) return;
  __shared__ double sf[NW], sq[NW];
  if ((threadIdx.x & 31) == 0) { sf[threadIdx.x >> 5] = f; sq[threadIdx.x >> 5] = q; }
  __syncthreads();
  if (threadIdx.x < 32) {
    f = threadIdx.x < NW ? sf[threadIdx.x] : 0.0;
    q = threadIdx.x < NW ? sq[threadIdx.x] : 0.0;
    f = warp_sum(f);
    q = warp_sum(q);
  }
}

}  // namespace gf
