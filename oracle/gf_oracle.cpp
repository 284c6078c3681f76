// gf_oracle — TEST INFRASTRUCTURE, not product code.
//
// A plain, slow, obviously-correct CPU statement of the gauge-fixing hot path of arXiv:1412.1498 (N. Cardoso,
// "Coulomb and Landau Gauge Fixing in GPUs using CUDA and MILC"): eqs. 1.1-1.6 and Algorithm 1 (overrelaxation).
// It is written from the paper in the paper's order and notation, with std::complex, no
// blocking, no fusion, no reordering; where the paper is silent or garbled it follows the readings A1-A20 of
// SURVEY.md §8(c), every one of which is listed again in DESIGN.md.  It shares NO code with the CUDA path
// (paper_1412_1498_b200/csrc) and neither includes the other.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may call it.
//
// Pins (tests/test_oracle_pins.py, all "-m 'not gpu'"): F=1, theta=0 on unit and gauge-transformed pure-gauge
// fields; literal eq. 1.3 vs the K-based traceless form; brute-force maximisation of Re Tr[gK] over random SU(2) on
// a 2^4 lattice; eq. 1.6 closed form on SU(2)-embedded fields; g^omega group properties; gauge invariance of
// plaquettes, Wilson and Polyakov loops to 1e-12; unitarity/det to 1e-12; F monotone at omega=1 (per site update and
// per sweep); site-order independence; 2-site translation covariance; Coulomb slice independence; 12-real emulation;
// reunitarisation idempotence; for the two variants (readings A21, A22): the truncated series of g^omega against the
// binomial series of 2x2 numpy matrices, its terminating (omega = 1, 2) and order-1 closed forms, convergence to the
// exact power, gauge invariance of a series sweep; per-slice F_t / theta_t against the global values and against the
// slice copied into a two-slice lattice, masked half-sweeps (finished slices untouched, active ones as in the full
// sweep), per-slice sweep counts against each slice run alone.  The drivers' ORDER (tests/test_oracle_order_pins.py):
// sweeps() = even half-sweep then odd half-sweep against the two calls written out, against a numpy
// gauge transformation by G on the (x+y+z+t)-even sites first, and by stationarity of the parity visited last;
// reunitarisation after global sweep s iff s % k == 0 against the unrolled call sequence and the
// unitarity defect of an off-group input; fix() / fix_slices() histories and links against the same sequences.
// The whole trajectory on the five configs (sweep counts, final F) is "parity unpinned"
// by the paper, which prints no numbers (last row of the pin table).
//
// Canonical layout: links[site][mu][row][col][re,im], site = x + nx*(y + ny*(z + nz*t)) (x fastest),
// mu = 0..3 = (x,y,z,t), temporal direction mu = 3.  U_mu(x) is the link from x to x+mu.
#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

namespace {

template <class T>
using Cx = std::complex<T>;

template <class T>
struct Mat3 {
  Cx<T> m[3][3];
};

struct Geom {
  int n[4];
  int64_t V;
};

Geom make_geom(const int* dims) {
  Geom g;
  g.V = 1;
  for (int d = 0; d < 4; ++d) {
    g.n[d] = dims[d];
    g.V *= dims[d];
  }
  return g;
}

void site_coords(const Geom& g, int64_t s, int c[4]) {
  for (int d = 0; d < 4; ++d) {
    c[d] = (int)(s % g.n[d]);
    s /= g.n[d];
  }
}
int64_t site_index(const Geom& g, const int c[4]) {
  return c[0] + (int64_t)g.n[0] * (c[1] + (int64_t)g.n[1] * (c[2] + (int64_t)g.n[2] * c[3]));
}
int site_parity(const Geom& g, int64_t s) {  // even <=> (x+y+z+t)&1 == 0   (reading A10)
  int c[4];
  site_coords(g, s, c);
  return (c[0] + c[1] + c[2] + c[3]) & 1;
}
// x + dir*mu with periodic wrap, dir = +1 / -1
int64_t neighbour(const Geom& g, int64_t s, int mu, int dir) {
  int c[4];
  site_coords(g, s, c);
  c[mu] = (c[mu] + dir + g.n[mu]) % g.n[mu];
  return site_index(g, c);
}

template <class T>
Mat3<T> load_link(const T* U, int64_t s, int mu) {
  const T* p = U + (s * 4 + mu) * 18;
  Mat3<T> a;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) a.m[i][j] = Cx<T>(p[(i * 3 + j) * 2], p[(i * 3 + j) * 2 + 1]);
  return a;
}
template <class T>
void store_link(T* U, int64_t s, int mu, const Mat3<T>& a) {
  T* p = U + (s * 4 + mu) * 18;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      p[(i * 3 + j) * 2] = a.m[i][j].real();
      p[(i * 3 + j) * 2 + 1] = a.m[i][j].imag();
    }
}

template <class T>
Mat3<T> identity() {
  Mat3<T> a;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) a.m[i][j] = Cx<T>(i == j ? T(1) : T(0), T(0));
  return a;
}
template <class T>
Mat3<T> mul(const Mat3<T>& a, const Mat3<T>& b) {
  Mat3<T> c;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      Cx<T> s(0, 0);
      for (int k = 0; k < 3; ++k) s += a.m[i][k] * b.m[k][j];
      c.m[i][j] = s;
    }
  return c;
}
template <class T>
Mat3<T> dagger(const Mat3<T>& a) {
  Mat3<T> c;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) c.m[i][j] = std::conj(a.m[j][i]);
  return c;
}
template <class T>
Mat3<T> add(const Mat3<T>& a, const Mat3<T>& b) {
  Mat3<T> c;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) c.m[i][j] = a.m[i][j] + b.m[i][j];
  return c;
}
template <class T>
Mat3<T> sub(const Mat3<T>& a, const Mat3<T>& b) {
  Mat3<T> c;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) c.m[i][j] = a.m[i][j] - b.m[i][j];
  return c;
}
template <class T>
Cx<T> trace(const Mat3<T>& a) {
  return a.m[0][0] + a.m[1][1] + a.m[2][2];
}
template <class T>
Cx<T> det(const Mat3<T>& a) {
  return a.m[0][0] * (a.m[1][1] * a.m[2][2] - a.m[1][2] * a.m[2][1]) -
         a.m[0][1] * (a.m[1][0] * a.m[2][2] - a.m[1][2] * a.m[2][0]) +
         a.m[0][2] * (a.m[1][0] * a.m[2][1] - a.m[1][1] * a.m[2][0]);
}
// row 2 = conj(row 0 x row 1): the third row of an SU(3) matrix from the first two (12-real storage, reading A13)
template <class T>
void rebuild_row2(Mat3<T>& a) {
  a.m[2][0] = std::conj(a.m[0][1] * a.m[1][2] - a.m[0][2] * a.m[1][1]);
  a.m[2][1] = std::conj(a.m[0][2] * a.m[1][0] - a.m[0][0] * a.m[1][2]);
  a.m[2][2] = std::conj(a.m[0][0] * a.m[1][1] - a.m[0][1] * a.m[1][0]);
}

// 8-real storage ("Elems = 4", 144, 174; reading A23): a link is kept as a2, a3, b1 (row 0 columns 1,2;
// row 1 column 0) and the phases of a1 and c1 (rows a, b, c).  Everything else follows from unitarity and det = 1:
//   N = |a2|^2 + |a3|^2;  |a1| = sqrt(1 - N);  |c1| = sqrt(N - |b1|^2)      (row a and column 0 have unit norm)
//   (b2, b3) = alpha (a2, a3) + beta (-conj a3, conj a2),  alpha = -conj(a1) b1 / N  (row b orthogonal to row a),
//   beta = conj(c1) / N  (c1 = conj(a2 b3 - a3 b2));  row c = conj(a x b).
// Undefined for N = 0 (block-diagonal links) and ill-conditioned near it: rounding is amplified by 1/N.
template <class T>
void roundtrip8(Mat3<T>& u) {
  const Cx<T> a2 = u.m[0][1], a3 = u.m[0][2], b1 = u.m[1][0];
  const T th_a = std::arg(u.m[0][0]), th_c = std::arg(u.m[2][0]);
  const T N = std::norm(a2) + std::norm(a3);
  const Cx<T> a1 = std::polar(std::sqrt(std::max(T(0), T(1) - N)), th_a);
  const Cx<T> c1 = std::polar(std::sqrt(std::max(T(0), N - std::norm(b1))), th_c);
  const Cx<T> alpha = -std::conj(a1) * b1 / N, beta = std::conj(c1) / N;
  u.m[0][0] = a1;
  u.m[1][1] = alpha * a2 - beta * std::conj(a3);
  u.m[1][2] = alpha * a3 + beta * std::conj(a2);
  rebuild_row2(u);  // row c = conj(a x b); its first entry reproduces c1 up to rounding
}

int ndir(int gauge) { return gauge == 1 ? 3 : 4; }  // Landau mu=0..3, Coulomb mu=0..2

// ---- O1: F (eq. 1.1) and theta (eqs. 1.2-1.3), g == 1 because transformations are applied to the links in place -----
// F = 1/(d Nc V) sum_x sum_{mu<d} Re Tr U_mu(x)                         (eq. 1.1, normalised by d: reading A1)
// A(x) = sum_{nu<d} [U_nu(x-nu) - U_nu(x)];  Delta = (A - A^dag) - (1/Nc) Tr(A - A^dag) 1     (eq. 1.3, reading A2)
// theta = 1/(Nc V) sum_x Tr[Delta Delta^dag]                            (eq. 1.2)
template <class T>
Mat3<T> delta_at(const T* U, const Geom& g, int gauge, int64_t s) {
  const int d = ndir(gauge);
  Mat3<T> A;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) A.m[i][j] = Cx<T>(0, 0);
  for (int nu = 0; nu < d; ++nu) {
    A = add(A, load_link(U, neighbour(g, s, nu, -1), nu));
    A = sub(A, load_link(U, s, nu));
  }
  Mat3<T> D = sub(A, dagger(A));
  Cx<T> tr = trace(D) / T(3);
  for (int i = 0; i < 3; ++i) D.m[i][i] -= tr;
  return D;
}

template <class T>
void measure(const T* U, const Geom& g, int gauge, double* F, double* theta) {
  const int d = ndir(gauge);
  const int64_t slice = g.V / g.n[3];
  std::vector<long double> fpart(g.n[3]), tpart(g.n[3]);
#pragma omp parallel for schedule(static)
  for (int t = 0; t < g.n[3]; ++t) {
    long double fs = 0, ts = 0;
    for (int64_t s = t * slice; s < (t + 1) * slice; ++s) {  // fixed order: x fastest, then y, z
      for (int mu = 0; mu < d; ++mu) fs += (long double)trace(load_link(U, s, mu)).real();
      Mat3<T> D = delta_at(U, g, gauge, s);
      long double q = 0;
      for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) q += (long double)std::norm(D.m[i][j]);
      ts += q;
    }
    fpart[t] = fs;
    tpart[t] = ts;
  }
  long double fs = 0, ts = 0;
  for (int t = 0; t < g.n[3]; ++t) {
    fs += fpart[t];
    ts += tpart[t];
  }
  *F = (double)(fs / ((long double)d * 3.0L * (long double)g.V));
  *theta = (double)(ts / (3.0L * (long double)g.V));
}

// Per-time-slice values (Coulomb gauge: each slice is its own 3-D problem, BASELINE.json configs[1]; reading A22):
// F_t and theta_t are eqs. 1.1-1.2 with the sums restricted to the sites of slice t and V -> V/n_t.
template <class T>
void measure_slices(const T* U, const Geom& g, int gauge, double* F_t, double* theta_t) {
  const int d = ndir(gauge);
  const int64_t slice = g.V / g.n[3];
#pragma omp parallel for schedule(static)
  for (int t = 0; t < g.n[3]; ++t) {
    long double fs = 0, ts = 0;
    for (int64_t s = t * slice; s < (t + 1) * slice; ++s) {
      for (int mu = 0; mu < d; ++mu) fs += (long double)trace(load_link(U, s, mu)).real();
      Mat3<T> D = delta_at(U, g, gauge, s);
      for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) ts += (long double)std::norm(D.m[i][j]);
    }
    F_t[t] = (double)(fs / ((long double)d * 3.0L * (long double)slice));
    theta_t[t] = (double)(ts / (3.0L * (long double)slice));
  }
}

// ---- O2: one site update ---------------------------------------------------------------------------------------------
// K(x) = sum_{mu<d} [U_mu(x) + U_mu(x-mu)^dag]   (eq. 1.5 with the neighbours' g already absorbed: reading A3),
// summed in the order mu=0 fwd, mu=0 bwd, mu=1 fwd, ...
template <class T>
Mat3<T> build_K(const T* U, const Geom& g, int gauge, int64_t s) {
  const int d = ndir(gauge);
  Mat3<T> K;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) K.m[i][j] = Cx<T>(0, 0);
  for (int mu = 0; mu < d; ++mu) {
    K = add(K, load_link(U, s, mu));
    K = add(K, dagger(load_link(U, neighbour(g, s, mu, -1), mu)));
  }
  return K;
}

// g -> g^omega for a unit quaternion a = (a0; a1,a2,a3) <-> g = a0 + i a.sigma = exp(i phi n.sigma):
// exact power exp(i omega phi n.sigma), principal branch phi in [0,pi]  (readings A6, A7).
template <class T>
void su2_power(const T a[4], T omega, T out[4]) {
  const T s = std::sqrt(a[1] * a[1] + a[2] * a[2] + a[3] * a[3]);
  const T tiny = std::numeric_limits<T>::min() * T(1152921504606846976.0);  // smallest normal * 2^60
  if (s < tiny) {
    if (a[0] > T(0)) {  // limit of sin(omega phi)/s as s -> 0 is omega
      const T phi = std::atan2(s, a[0]);
      out[0] = std::cos(omega * phi);
      out[1] = omega * a[1];
      out[2] = omega * a[2];
      out[3] = omega * a[3];
    } else {  // phi = pi, axis undefined: leave g^omega = 1
      out[0] = T(1);
      out[1] = out[2] = out[3] = T(0);
    }
    return;
  }
  const T phi = std::atan2(s, a[0]);
  const T f = std::sin(omega * phi) / s;
  out[0] = std::cos(omega * phi);
  out[1] = a[1] * f;
  out[2] = a[2] * f;
  out[3] = a[3] * f;
}

// Variant (PAPER.md:50 cites ref. [1], Mandula & Ogilvie, for g -> g^omega; they evaluate it as a truncated binomial
// series followed by a projection back to the group; reading A21): g^omega ~ sum_{n=0}^{N} binom(omega, n) (g - 1)^n,
// binom(omega, n) = omega (omega-1) ... (omega-n+1) / n!, written out with quaternion products
// (p0 + i p.sigma)(q0 + i q.sigma) = (p0 q0 - p.q) + i (p0 q + q0 p - p x q).sigma, then normalised to a unit quaternion.
// order = 0 selects the exact power above; it is a process-wide switch of this test library (orc_set_series).
int g_series_order = 0;

template <class T>
void quat_mul(const T p[4], const T q[4], T out[4]) {
  out[0] = p[0] * q[0] - (p[1] * q[1] + p[2] * q[2] + p[3] * q[3]);
  out[1] = p[0] * q[1] + q[0] * p[1] - (p[2] * q[3] - p[3] * q[2]);
  out[2] = p[0] * q[2] + q[0] * p[2] - (p[3] * q[1] - p[1] * q[3]);
  out[3] = p[0] * q[3] + q[0] * p[3] - (p[1] * q[2] - p[2] * q[1]);
}

template <class T>
void su2_power_series(const T a[4], T omega, int order, T out[4]) {
  const T u[4] = {a[0] - T(1), a[1], a[2], a[3]};  // g - 1
  T P[4] = {T(1), T(0), T(0), T(0)};               // (g - 1)^n
  T acc[4] = {T(0), T(0), T(0), T(0)};
  T b = T(1);                                      // binom(omega, n)
  for (int n = 0; n <= order; ++n) {
    for (int k = 0; k < 4; ++k) acc[k] += b * P[k];
    T next[4];
    quat_mul(P, u, next);
    for (int k = 0; k < 4; ++k) P[k] = next[k];
    b = b * (omega - T(n)) / T(n + 1);
  }
  const T norm = std::sqrt(acc[0] * acc[0] + acc[1] * acc[1] + acc[2] * acc[2] + acc[3] * acc[3]);
  if (norm == T(0)) {
    out[0] = T(1);
    out[1] = out[2] = out[3] = T(0);
    return;
  }
  for (int k = 0; k < 4; ++k) out[k] = acc[k] / norm;
}

// One SU(2) subgroup step on rows/columns (i,j): maximise Re Tr[g K] over the embedded SU(2) (eq. 1.6 applied to the
// SU(2)-proportional part of the 2x2 block, reading A5), raise to omega, K <- gK, G <- gG.  a_out = quaternion of g^omega.
template <class T>
void su2_subgroup_step(Mat3<T>& K, Mat3<T>& G, int i, int j, T omega, T a_out[4]) {
  const Cx<T> M00 = K.m[i][i], M01 = K.m[i][j], M10 = K.m[j][i], M11 = K.m[j][j];
  T r[4];
  r[0] = (M00 + M11).real();
  r[1] = -(M01 + M10).imag();
  r[2] = (M10 - M01).real();
  r[3] = -(M00 - M11).imag();
  const T n = std::sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2] + r[3] * r[3]);
  if (n == T(0)) {  // reading A7: nothing to maximise, g = 1
    a_out[0] = T(1);
    a_out[1] = a_out[2] = a_out[3] = T(0);
    return;
  }
  T a[4] = {r[0] / n, r[1] / n, r[2] / n, r[3] / n};
  if (g_series_order > 0) su2_power_series(a, omega, g_series_order, a_out);
  else su2_power(a, omega, a_out);
  // g = [[a0 + i a3, a2 + i a1], [-a2 + i a1, a0 - i a3]] on rows/cols (i,j), 1 on the third
  const Cx<T> g00(a_out[0], a_out[3]), g01(a_out[2], a_out[1]), g10(-a_out[2], a_out[1]), g11(a_out[0], -a_out[3]);
  for (int c = 0; c < 3; ++c) {
    const Cx<T> ki = K.m[i][c], kj = K.m[j][c];
    K.m[i][c] = g00 * ki + g01 * kj;
    K.m[j][c] = g10 * ki + g11 * kj;
    const Cx<T> gi = G.m[i][c], gj = G.m[j][c];
    G.m[i][c] = g00 * gi + g01 * gj;
    G.m[j][c] = g10 * gi + g11 * gj;
  }
}

// Algorithm 1 lines 5-10 for one site (reading A8: accumulate G = g3 g2 g1, apply once; A4: subgroup order
// (0,1),(1,2),(0,2); A9: all four directions are transformed, also in Coulomb gauge).
template <class T>
void site_update(T* U, const Geom& g, int gauge, int64_t s, T omega, int storage) {
  Mat3<T> K = build_K(U, g, gauge, s);
  Mat3<T> G = identity<T>();
  T a[4];
  su2_subgroup_step(K, G, 0, 1, omega, a);
  su2_subgroup_step(K, G, 1, 2, omega, a);
  su2_subgroup_step(K, G, 0, 2, omega, a);
  const Mat3<T> Gd = dagger(G);
  for (int mu = 0; mu < 4; ++mu) {
    Mat3<T> f = mul(G, load_link(U, s, mu));  // U_mu(x) <- G U_mu(x)
    if (storage == 12) rebuild_row2(f);
    if (storage == 8) roundtrip8(f);
    store_link(U, s, mu, f);
    const int64_t sb = neighbour(g, s, mu, -1);
    Mat3<T> b = mul(load_link(U, sb, mu), Gd);  // U_mu(x-mu) <- U_mu(x-mu) G^dag
    if (storage == 12) rebuild_row2(b);
    if (storage == 8) roundtrip8(b);
    store_link(U, sb, mu, b);
  }
}

// Algorithm 1 lines 3-12 for one parity.  Same-parity sites touch disjoint links, so the visiting order is free.
template <class T>
void half_sweep(T* U, const Geom& g, int gauge, int parity, T omega, int storage) {
#pragma omp parallel for schedule(static)
  for (int64_t s = 0; s < g.V; ++s)
    if (site_parity(g, s) == parity) site_update(U, g, gauge, s, omega, storage);
}

// ---- O4: reunitarisation (reading A12): Gram-Schmidt on rows 0,1; row 2 = conj(row0 x row1) --------------------------
template <class T>
void reunitarize_link(Mat3<T>& a) {
  T n0 = 0;
  for (int j = 0; j < 3; ++j) n0 += std::norm(a.m[0][j]);
  n0 = std::sqrt(n0);
  for (int j = 0; j < 3; ++j) a.m[0][j] /= n0;
  Cx<T> p(0, 0);
  for (int j = 0; j < 3; ++j) p += std::conj(a.m[0][j]) * a.m[1][j];
  for (int j = 0; j < 3; ++j) a.m[1][j] -= p * a.m[0][j];
  T n1 = 0;
  for (int j = 0; j < 3; ++j) n1 += std::norm(a.m[1][j]);
  n1 = std::sqrt(n1);
  for (int j = 0; j < 3; ++j) a.m[1][j] /= n1;
  rebuild_row2(a);
}
template <class T>
void reunitarize(T* U, const Geom& g) {
#pragma omp parallel for schedule(static)
  for (int64_t s = 0; s < g.V; ++s)
    for (int mu = 0; mu < 4; ++mu) {
      Mat3<T> a = load_link(U, s, mu);
      reunitarize_link(a);
      store_link(U, s, mu, a);
    }
}
template <class T>
void project12(T* U, const Geom& g) {  // what gf_set_links does to the input when storage = 12 (reading A13)
#pragma omp parallel for schedule(static)
  for (int64_t s = 0; s < g.V; ++s)
    for (int mu = 0; mu < 4; ++mu) {
      Mat3<T> a = load_link(U, s, mu);
      rebuild_row2(a);
      store_link(U, s, mu, a);
    }
}

template <class T>
void project8(T* U, const Geom& g) {  // what gf_set_links does to the input when storage = 8 (reading A23)
#pragma omp parallel for schedule(static)
  for (int64_t s = 0; s < g.V; ++s)
    for (int mu = 0; mu < 4; ++mu) {
      Mat3<T> a = load_link(U, s, mu);
      roundtrip8(a);
      store_link(U, s, mu, a);
    }
}

// n sweeps = (even half-sweep, odd half-sweep) x n (reading A10), reunitarising after global sweep number s when
// reunit_every > 0 and s % reunit_every == 0.  first_sweep = number of sweeps already done before this call.
template <class T>
void sweeps(T* U, const Geom& g, int gauge, T omega, int storage, int n, int reunit_every, int first_sweep) {
  for (int k = 1; k <= n; ++k) {
    half_sweep(U, g, gauge, 0, omega, storage);
    half_sweep(U, g, gauge, 1, omega, storage);
    const int s = first_sweep + k;
    if (reunit_every > 0 && s % reunit_every == 0) reunitarize(U, g);
  }
}

// ---- O5: Algorithm 1 with a measurement cadence (reading A11) --------------------------------------------------------
template <class T>
int fix(T* U, const Geom& g, int gauge, T omega, double eps, int max_sweeps, int check_every, int reunit_every,
        int storage, int* sweeps_done, double* hist, int hist_cap, int* nhist) {
  double F, th;
  int done = 0, nh = 0;
  measure(U, g, gauge, &F, &th);
  auto record = [&]() {
    if (hist && nh < hist_cap) {
      hist[3 * nh] = (double)done;
      hist[3 * nh + 1] = F;
      hist[3 * nh + 2] = th;
    }
    ++nh;
  };
  record();
  while (!(th < eps) && done < max_sweeps) {
    const int n = std::min(check_every, max_sweeps - done);
    sweeps(U, g, gauge, omega, storage, n, reunit_every, done);
    done += n;
    measure(U, g, gauge, &F, &th);
    record();
  }
  *sweeps_done = done;
  if (nhist) *nhist = nh;
  return 0;
}

// ---- O5b: Coulomb gauge with a stop test per time slice (reading A22) ---------------------------------------------------
// K(x) of a Coulomb-gauge site holds links of its own time slice only, so the slices are independent problems
// (BASELINE.json configs[1]: "each of the 32 time slices is fixed independently").  Variant of Algorithm 1: theta_t per
// slice; a slice with theta_t < eps is finished and its sites are not visited any more; the run ends when every slice
// is finished or the sweep cap is reached.  slice_sweeps[t] = sweeps spent on slice t.
template <class T>
void half_sweep_masked(T* U, const Geom& g, int gauge, int parity, T omega, int storage, const uint8_t* active) {
  const int64_t slice = g.V / g.n[3];
#pragma omp parallel for schedule(static)
  for (int64_t s = 0; s < g.V; ++s)
    if (active[s / slice] && site_parity(g, s) == parity) site_update(U, g, gauge, s, omega, storage);
}

template <class T>
int fix_slices(T* U, const Geom& g, int gauge, T omega, double eps, int max_sweeps, int check_every, int reunit_every,
               int storage, int* sweeps_done, int* slice_sweeps, double* hist, int hist_cap, int* nhist) {
  const int nt = g.n[3];
  std::vector<double> Ft(nt), tht(nt);
  std::vector<uint8_t> active(nt);
  int done = 0, nh = 0;
  for (int t = 0; t < nt; ++t) slice_sweeps[t] = 0;
  auto look = [&]() {  // record (sweeps, mean F, max theta_t); returns the number of unfinished slices
    measure_slices(U, g, gauge, Ft.data(), tht.data());
    double F = 0, thmax = 0;
    int n_active = 0;
    for (int t = 0; t < nt; ++t) {
      F += Ft[t];
      thmax = std::max(thmax, tht[t]);
      active[t] = !(tht[t] < eps);
      n_active += active[t];
    }
    if (hist && nh < hist_cap) {
      hist[3 * nh] = (double)done;
      hist[3 * nh + 1] = F / nt;
      hist[3 * nh + 2] = thmax;
    }
    ++nh;
    return n_active;
  };
  int n_active = look();
  while (n_active > 0 && done < max_sweeps) {
    const int n = std::min(check_every, max_sweeps - done);
    for (int k = 1; k <= n; ++k) {
      half_sweep_masked(U, g, gauge, 0, omega, storage, active.data());
      half_sweep_masked(U, g, gauge, 1, omega, storage, active.data());
      if (reunit_every > 0 && (done + k) % reunit_every == 0) reunitarize(U, g);
    }
    for (int t = 0; t < nt; ++t) slice_sweeps[t] += active[t] ? n : 0;
    done += n;
    n_active = look();
  }
  *sweeps_done = done;
  if (nhist) *nhist = nh;
  return 0;
}

// ---- O6: gauge-invariant observables for the invariance pins ---------------------------------------------------------
// product of links along a rectangular a x b loop in the (mu,nu) plane starting at s
template <class T>
Cx<T> wilson_loop_trace(const T* U, const Geom& g, int64_t s, int mu, int nu, int a, int b) {
  Mat3<T> P = identity<T>();
  int64_t x = s;
  for (int k = 0; k < a; ++k) { P = mul(P, load_link(U, x, mu)); x = neighbour(g, x, mu, +1); }
  for (int k = 0; k < b; ++k) { P = mul(P, load_link(U, x, nu)); x = neighbour(g, x, nu, +1); }
  for (int k = 0; k < a; ++k) { x = neighbour(g, x, mu, -1); P = mul(P, dagger(load_link(U, x, mu))); }
  for (int k = 0; k < b; ++k) { x = neighbour(g, x, nu, -1); P = mul(P, dagger(load_link(U, x, nu))); }
  return trace(P);
}
template <class T>
void wilson_traces(const T* U, const Geom& g, int mu, int nu, int a, int b, double* out) {
#pragma omp parallel for schedule(static)
  for (int64_t s = 0; s < g.V; ++s) {
    Cx<T> t = wilson_loop_trace(U, g, s, mu, nu, a, b);
    out[2 * s] = (double)t.real();
    out[2 * s + 1] = (double)t.imag();
  }
}
// Tr of the product of all n_mu links of the closed line through s in direction mu (every s: V values)
template <class T>
void polyakov_traces(const T* U, const Geom& g, int mu, double* out) {
#pragma omp parallel for schedule(static)
  for (int64_t s = 0; s < g.V; ++s) {
    Mat3<T> P = identity<T>();
    int64_t x = s;
    for (int k = 0; k < g.n[mu]; ++k) { P = mul(P, load_link(U, x, mu)); x = neighbour(g, x, mu, +1); }
    Cx<T> t = trace(P);
    out[2 * s] = (double)t.real();
    out[2 * s + 1] = (double)t.imag();
  }
}
template <class T>
void unitarity_defects(const T* U, const Geom& g, double* max_uudag, double* max_det) {
  double mu_ = 0, md_ = 0;
#pragma omp parallel for schedule(static) reduction(max : mu_, md_)
  for (int64_t s = 0; s < g.V; ++s)
    for (int mu = 0; mu < 4; ++mu) {
      Mat3<T> a = load_link(U, s, mu);
      Mat3<T> p = sub(mul(a, dagger(a)), identity<T>());
      for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) mu_ = std::max(mu_, (double)std::abs(p.m[i][j]));
      md_ = std::max(md_, (double)std::abs(det(a) - Cx<T>(1, 0)));
    }
  *max_uudag = mu_;
  *max_det = md_;
}

template <class T>
void mat_from(const T* p, Mat3<T>& a) {
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) a.m[i][j] = Cx<T>(p[(i * 3 + j) * 2], p[(i * 3 + j) * 2 + 1]);
}
template <class T>
void mat_to(T* p, const Mat3<T>& a) {
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      p[(i * 3 + j) * 2] = a.m[i][j].real();
      p[(i * 3 + j) * 2 + 1] = a.m[i][j].imag();
    }
}

}  // namespace

// ---- C ABI for the ctypes wrapper (oracle/__init__.py) --------------------------------------------------------------
#define ORC_API(SUF, T)                                                                                               \
  extern "C" {                                                                                                        \
  void orc_measure_##SUF(const T* U, const int* dims, int gauge, double* F, double* theta) {                          \
    measure<T>(U, make_geom(dims), gauge, F, theta);                                                                  \
  }                                                                                                                   \
  void orc_half_sweep_##SUF(T* U, const int* dims, int gauge, int parity, double omega, int storage) {                \
    half_sweep<T>(U, make_geom(dims), gauge, parity, (T)omega, storage);                                              \
  }                                                                                                                   \
  void orc_sweeps_##SUF(T* U, const int* dims, int gauge, double omega, int storage, int n, int reunit_every,         \
                        int first_sweep) {                                                                            \
    sweeps<T>(U, make_geom(dims), gauge, (T)omega, storage, n, reunit_every, first_sweep);                            \
  }                                                                                                                   \
  void orc_site_update_##SUF(T* U, const int* dims, int gauge, int64_t site, double omega, int storage) {             \
    site_update<T>(U, make_geom(dims), gauge, site, (T)omega, storage);                                               \
  }                                                                                                                   \
  void orc_reunitarize_##SUF(T* U, const int* dims) { reunitarize<T>(U, make_geom(dims)); }                           \
  void orc_project12_##SUF(T* U, const int* dims) { project12<T>(U, make_geom(dims)); }                               \
  void orc_project8_##SUF(T* U, const int* dims) { project8<T>(U, make_geom(dims)); }                                 \
  int orc_fix_##SUF(T* U, const int* dims, int gauge, double omega, double eps, int max_sweeps, int check_every,      \
                    int reunit_every, int storage, int* sweeps_done, double* hist, int hist_cap, int* nhist) {        \
    return fix<T>(U, make_geom(dims), gauge, (T)omega, eps, max_sweeps, check_every, reunit_every, storage,           \
                  sweeps_done, hist, hist_cap, nhist);                                                                \
  }                                                                                                                   \
  void orc_measure_slices_##SUF(const T* U, const int* dims, int gauge, double* F_t, double* theta_t) {               \
    measure_slices<T>(U, make_geom(dims), gauge, F_t, theta_t);                                                       \
  }                                                                                                                   \
  void orc_half_sweep_masked_##SUF(T* U, const int* dims, int gauge, int parity, double omega, int storage,           \
                                   const uint8_t* active) {                                                           \
    half_sweep_masked<T>(U, make_geom(dims), gauge, parity, (T)omega, storage, active);                               \
  }                                                                                                                   \
  int orc_fix_slices_##SUF(T* U, const int* dims, int gauge, double omega, double eps, int max_sweeps,                \
                           int check_every, int reunit_every, int storage, int* sweeps_done, int* slice_sweeps,       \
                           double* hist, int hist_cap, int* nhist) {                                                  \
    return fix_slices<T>(U, make_geom(dims), gauge, (T)omega, eps, max_sweeps, check_every, reunit_every, storage,    \
                         sweeps_done, slice_sweeps, hist, hist_cap, nhist);                                           \
  }                                                                                                                   \
  void orc_site_K_##SUF(const T* U, const int* dims, int gauge, int64_t site, T* K18) {                               \
    mat_to<T>(K18, build_K<T>(U, make_geom(dims), gauge, site));                                                      \
  }                                                                                                                   \
  void orc_site_delta_##SUF(const T* U, const int* dims, int gauge, int64_t site, T* D18) {                           \
    mat_to<T>(D18, delta_at<T>(U, make_geom(dims), gauge, site));                                                     \
  }                                                                                                                   \
  void orc_su2_step_##SUF(T* K18, T* G18, int i, int j, double omega, T* a4) {                                        \
    Mat3<T> K, G;                                                                                                     \
    mat_from<T>(K18, K);                                                                                              \
    mat_from<T>(G18, G);                                                                                              \
    su2_subgroup_step<T>(K, G, i, j, (T)omega, a4);                                                                   \
    mat_to<T>(K18, K);                                                                                                \
    mat_to<T>(G18, G);                                                                                                \
  }                                                                                                                   \
  void orc_su2_power_##SUF(const T* a4, double omega, T* out4) { su2_power<T>(a4, (T)omega, out4); }                  \
  void orc_su2_power_series_##SUF(const T* a4, double omega, int order, T* out4) {                                    \
    su2_power_series<T>(a4, (T)omega, order, out4);                                                                   \
  }                                                                                                                   \
  void orc_wilson_traces_##SUF(const T* U, const int* dims, int mu, int nu, int a, int b, double* out) {              \
    wilson_traces<T>(U, make_geom(dims), mu, nu, a, b, out);                                                          \
  }                                                                                                                   \
  void orc_polyakov_traces_##SUF(const T* U, const int* dims, int mu, double* out) {                                  \
    polyakov_traces<T>(U, make_geom(dims), mu, out);                                                                  \
  }                                                                                                                   \
  void orc_unitarity_##SUF(const T* U, const int* dims, double* max_uudag, double* max_det) {                         \
    unitarity_defects<T>(U, make_geom(dims), max_uudag, max_det);                                                     \
  }                                                                                                                   \
  }

ORC_API(f64, double)
ORC_API(f32, float)

// 0: g^omega is the exact power (default); N > 0: the truncated binomial series of order N (su2_power_series)
extern "C" void orc_set_series(int order) { g_series_order = order < 0 ? 0 : order; }
extern "C" int orc_get_series() { return g_series_order; }
