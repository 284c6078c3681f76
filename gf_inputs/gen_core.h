// Seeded synthetic gauge-field generator — the recipe, shared by the host (g++) and device (nvcc) builds.
//
// This header is INPUT DATA tooling only.  It holds none of the gauge-fixing method's arithmetic (no K(x), no
// SU(2) subgroup step, no overrelaxation, no F/theta): it only fabricates the SU(3) link field the method is run
// on.  Neither oracle/ nor paper_1412_1498_b200/csrc/ includes it; both just receive the arrays it writes.
//
// Recipe (BASELINE.json "configs"; SURVEY.md §8(d) "Generator"; stands in for the MILC production configurations
// the paper measured on, which are not available):
//     U_mu(x) = G(x) . exp(i r H_mu(x)) . G(x+mu)^dagger            (periodic x+mu)
//   * H_mu(x) = sum_{a=1..8} c_a lambda_a,  c_a ~ N(0,1)  (Gell-Mann matrices, Tr l_a l_b = 2 d_ab),
//   * G(x)    = Haar-random SU(3): Gram-Schmidt of a 3x3 complex Gaussian matrix, then divided by det^(1/3),
//   * r       = "roughness".
// Random numbers are COUNTER based: every normal deviate is a pure function of (seed, stream, site, mu, k), so any
// link can be generated on its own, in any order, on any number of threads.
//
// Canonical layout written: links[site][mu][row][col][re,im], site = x + nx*(y + ny*(z + nz*t)), mu = 0..3 = x,y,z,t.
#pragma once
#include <math.h>
#include <stdint.h>

#if defined(__CUDACC__)
#define GFIN_HD __host__ __device__ inline
#else
#define GFIN_HD inline
#endif

namespace gfin {

struct cd { double re, im; };
GFIN_HD cd mk(double a, double b) { cd z; z.re = a; z.im = b; return z; }
GFIN_HD cd add(cd a, cd b) { return mk(a.re + b.re, a.im + b.im); }
GFIN_HD cd sub(cd a, cd b) { return mk(a.re - b.re, a.im - b.im); }
GFIN_HD cd mul(cd a, cd b) { return mk(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re); }
GFIN_HD cd cj(cd a) { return mk(a.re, -a.im); }
GFIN_HD cd scale(cd a, double s) { return mk(a.re * s, a.im * s); }

struct m3 { cd e[3][3]; };

GFIN_HD m3 matmul(const m3& a, const m3& b) {
  m3 c;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      cd s = mk(0.0, 0.0);
      for (int k = 0; k < 3; ++k) s = add(s, mul(a.e[i][k], b.e[k][j]));
      c.e[i][j] = s;
    }
  return c;
}
GFIN_HD m3 matmul_adj(const m3& a, const m3& b) {  // a . b^dagger
  m3 c;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      cd s = mk(0.0, 0.0);
      for (int k = 0; k < 3; ++k) s = add(s, mul(a.e[i][k], cj(b.e[j][k])));
      c.e[i][j] = s;
    }
  return c;
}

// ---- counter-based random numbers -------------------------------------------------------------------------------
GFIN_HD uint64_t mix64(uint64_t z) {  // SplitMix64 finaliser
  z += 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
GFIN_HD uint64_t key5(uint64_t seed, uint64_t stream, uint64_t site, uint64_t mu, uint64_t k) {
  uint64_t h = mix64(seed ^ 0x6A09E667F3BCC909ull);
  h = mix64(h + stream);
  h = mix64(h + site);
  h = mix64(h + mu);
  h = mix64(h + k);
  return h;
}
GFIN_HD double u01(uint64_t h) { return ((double)(h >> 11) + 0.5) * (1.0 / 9007199254740992.0); }  // (0,1)

// k-th pair of independent N(0,1) deviates of the (seed, stream, site, mu) counter (Box-Muller).
GFIN_HD void normal_pair(uint64_t seed, uint64_t stream, uint64_t site, uint64_t mu, uint64_t k, double* n0,
                         double* n1) {
  double u1 = u01(key5(seed, stream, site, mu, 2 * k));
  double u2 = u01(key5(seed, stream, site, mu, 2 * k + 1));
  double rad = sqrt(-2.0 * log(u1));
  double ang = 6.283185307179586476925286766559 * u2;
  *n0 = rad * cos(ang);
  *n1 = rad * sin(ang);
}

enum { STREAM_G = 1, STREAM_H = 2 };

// ---- projections ------------------------------------------------------------------------------------------------
GFIN_HD double row_norm2(const m3& a, int r) {
  double s = 0.0;
  for (int j = 0; j < 3; ++j) s += a.e[r][j].re * a.e[r][j].re + a.e[r][j].im * a.e[r][j].im;
  return s;
}
GFIN_HD cd row_dot(const m3& a, int r, int q) {  // <row r, row q> = sum_j conj(a_rj) a_qj
  cd s = mk(0.0, 0.0);
  for (int j = 0; j < 3; ++j) s = add(s, mul(cj(a.e[r][j]), a.e[q][j]));
  return s;
}
GFIN_HD void row_axpy(m3& a, int dst, cd c, int src) {  // row dst -= c * row src
  for (int j = 0; j < 3; ++j) a.e[dst][j] = sub(a.e[dst][j], mul(c, a.e[src][j]));
}
GFIN_HD void row_scale(m3& a, int r, double s) {
  for (int j = 0; j < 3; ++j) a.e[r][j] = scale(a.e[r][j], s);
}
GFIN_HD cd det3(const m3& a) {
  cd t0 = sub(mul(a.e[1][1], a.e[2][2]), mul(a.e[1][2], a.e[2][1]));
  cd t1 = sub(mul(a.e[1][0], a.e[2][2]), mul(a.e[1][2], a.e[2][0]));
  cd t2 = sub(mul(a.e[1][0], a.e[2][1]), mul(a.e[1][1], a.e[2][0]));
  return add(sub(mul(a.e[0][0], t0), mul(a.e[0][1], t1)), mul(a.e[0][2], t2));
}
// Gram-Schmidt on all three rows -> U(3)
GFIN_HD void gram_schmidt3(m3& a) {
  row_scale(a, 0, 1.0 / sqrt(row_norm2(a, 0)));
  row_axpy(a, 1, row_dot(a, 0, 1), 0);
  row_scale(a, 1, 1.0 / sqrt(row_norm2(a, 1)));
  row_axpy(a, 2, row_dot(a, 0, 2), 0);
  row_axpy(a, 2, row_dot(a, 1, 2), 1);
  row_scale(a, 2, 1.0 / sqrt(row_norm2(a, 2)));
}
// U(3) -> SU(3): divide by the principal cube root of the determinant (a pure phase).
GFIN_HD void fix_det(m3& a) {
  cd d = det3(a);
  double alpha = atan2(d.im, d.re) / 3.0;
  cd ph = mk(cos(alpha), -sin(alpha));
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) a.e[i][j] = mul(a.e[i][j], ph);
}

// ---- the fields ---------------------------------------------------------------------------------------------------
// Haar-random SU(3) gauge rotation G(x)
GFIN_HD m3 gauge_at(uint64_t seed, uint64_t site) {
  m3 z;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      double a, b;
      normal_pair(seed, STREAM_G, site, 0, (uint64_t)(3 * i + j), &a, &b);
      z.e[i][j] = mk(a, b);
    }
  gram_schmidt3(z);
  gram_schmidt3(z);  // second pass: classical Gram-Schmidt loses orthogonality on ill-conditioned Gaussian draws
  fix_det(z);
  return z;
}

// exp(i r H), H = sum_a c_a lambda_a: scaling (2^-4) and squaring of a 16-term Taylor series, then projected on SU(3)
GFIN_HD m3 smooth_link(uint64_t seed, uint64_t site, int mu, double r) {
  double c[8];
  for (int k = 0; k < 4; ++k) normal_pair(seed, STREAM_H, site, (uint64_t)mu, (uint64_t)k, &c[2 * k], &c[2 * k + 1]);
  const double is3 = 0.57735026918962576450914878050196;  // 1/sqrt(3)
  m3 h;
  h.e[0][0] = mk(c[2] + c[7] * is3, 0.0);
  h.e[1][1] = mk(-c[2] + c[7] * is3, 0.0);
  h.e[2][2] = mk(-2.0 * c[7] * is3, 0.0);
  h.e[0][1] = mk(c[0], -c[1]);
  h.e[1][0] = mk(c[0], c[1]);
  h.e[0][2] = mk(c[3], -c[4]);
  h.e[2][0] = mk(c[3], c[4]);
  h.e[1][2] = mk(c[5], -c[6]);
  h.e[2][1] = mk(c[5], c[6]);
  // A = i r H / 16
  m3 a;
  const double s = r / 16.0;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) a.e[i][j] = mk(-h.e[i][j].im * s, h.e[i][j].re * s);
  // Horner: E = 1 + A(1 + A/2(1 + A/3(... (1 + A/16))))
  m3 e;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) e.e[i][j] = mk(i == j ? 1.0 : 0.0, 0.0);
  for (int n = 16; n >= 1; --n) {
    m3 t = matmul(a, e);
    double inv = 1.0 / (double)n;
    for (int i = 0; i < 3; ++i)
      for (int j = 0; j < 3; ++j) e.e[i][j] = mk((i == j ? 1.0 : 0.0) + t.e[i][j].re * inv, t.e[i][j].im * inv);
  }
  for (int q = 0; q < 4; ++q) e = matmul(e, e);
  gram_schmidt3(e);
  fix_det(e);
  return e;
}

GFIN_HD int64_t neighbour_up(int64_t site, int mu, const int* n) {
  int64_t c[4];
  int64_t s = site;
  for (int d = 0; d < 4; ++d) { c[d] = s % n[d]; s /= n[d]; }
  c[mu] = (c[mu] + 1) % n[mu];
  return c[0] + (int64_t)n[0] * (c[1] + (int64_t)n[1] * (c[2] + (int64_t)n[2] * c[3]));
}

// G0 . E . G1^dagger, polished back onto SU(3) so that every link is unitary with det 1 to ~1e-15
GFIN_HD m3 finish_link(const m3& g0, const m3& e, const m3& g1) {
  m3 u = matmul_adj(matmul(g0, e), g1);
  gram_schmidt3(u);
  fix_det(u);
  return u;
}

// U_mu(x) = G(x) exp(i r H_mu(x)) G(x+mu)^dagger
GFIN_HD m3 link_at(uint64_t seed, int64_t site, int mu, double r, const int* n) {
  m3 g0 = gauge_at(seed, (uint64_t)site);
  m3 g1 = gauge_at(seed, (uint64_t)neighbour_up(site, mu, n));
  m3 e = smooth_link(seed, (uint64_t)site, mu, r);
  return finish_link(g0, e, g1);
}

template <class T>
GFIN_HD void store_link(T* out, const m3& u) {
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      out[(i * 3 + j) * 2 + 0] = (T)u.e[i][j].re;
      out[(i * 3 + j) * 2 + 1] = (T)u.e[i][j].im;
    }
}

}  // namespace gfin
