// gf_kernels.cu — the CUDA kernels of libgf (sm_100a) and their launch wrappers.
//   reorder_in / reorder_out : canonical layout <-> internal AoSoA-32 layout          (gf_set_links / gf_get_links)
//   ovr_halfsweep            : one parity of the overrelaxation sweep                  (Algorithm 1 l.3-12)
//   measure_partial / _final : F and theta, two-stage deterministic reduction          (eqs. 1.1-1.3)
//   reunit                   : Gram-Schmidt reunitarisation of every link
#include <atomic>

#include "gf_device.cuh"
#include "gf_internal.h"

namespace gf {

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device attribute: a process that drives contexts on several
// GPUs must opt in once on each of them.  One flag per (kernel instantiation, device); racing host threads at worst
// set the attribute twice.
struct PerDeviceOnce {
  std::atomic<unsigned long long> done[2];
  template <class F>
  cudaError_t run(F&& f) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 128) return f();
    std::atomic<unsigned long long>& w = done[dev >> 6];
    const unsigned long long bit = 1ull << (dev & 63);
    if (w.load(std::memory_order_acquire) & bit) return cudaSuccess;
    e = f();
    if (e == cudaSuccess) w.fetch_or(bit, std::memory_order_release);
    return e;
  }
};
template <class K>
static cudaError_t opt_in_smem(PerDeviceOnce& once, K kern, size_t bytes) {
  return once.run([&] { return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes); });
}

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
    for (int e = 0; e < (NELEM == 4 ? 9 : NELEM); ++e) u[e] = cc[e];  // the 8-real form needs a1 and c1 too
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
  if (a.storage == 8)
    return a.prec == 0 ? reorder_T<double, 4>(a, in, canon, lex_begin, lex_end, chunk_base)
                       : reorder_T<float, 4>(a, in, canon, lex_begin, lex_end, chunk_base);
  if (a.prec == 0) return a.storage == 18 ? reorder_T<double, 9>(a, in, canon, lex_begin, lex_end, chunk_base)
                                          : reorder_T<double, 6>(a, in, canon, lex_begin, lex_end, chunk_base);
  return a.storage == 18 ? reorder_T<float, 9>(a, in, canon, lex_begin, lex_end, chunk_base)
                         : reorder_T<float, 6>(a, in, canon, lex_begin, lex_end, chunk_base);
}

// sum_ij |Delta_ij|^2 for Delta = (A - A^dag) - (1/3) Tr(A - A^dag)  (eqs. 1.2-1.3, reading A2).  The sign of A drops
// out, so A may be sum_nu [U_nu(x-nu) - U_nu(x)] or K(x) of eq. 1.5 (A - A^dag = -(K - K^dag)).
template <class T, class C>
__device__ __forceinline__ T delta_norm2(const C (&A)[9]) {
  // D = A - A^dag: D_ii = 2i Im A_ii; D_ij = A_ij - conj(A_ji);  traceless part: D_ii -= (1/3) sum_k D_kk
  const T d0 = T(2) * A[0].y, d1 = T(2) * A[4].y, d2 = T(2) * A[8].y;
  const T m = (d0 + d1 + d2) / T(3);
  T acc = (d0 - m) * (d0 - m) + (d1 - m) * (d1 - m) + (d2 - m) * (d2 - m);
  // off-diagonal: |D_ij|^2 = |D_ji|^2, so count each pair twice
  const T ax = A[1].x - A[3].x, ay = A[1].y + A[3].y; acc += T(2) * (ax * ax + ay * ay);
  const T bx = A[2].x - A[6].x, by = A[2].y + A[6].y; acc += T(2) * (bx * bx + by * by);
  const T cx = A[5].x - A[7].x, cy = A[5].y + A[7].y; acc += T(2) * (cx * cx + cy * cy);
  return acc;
}

// ======================================================================================================================
// overrelaxation half-sweep
// ======================================================================================================================
// One thread per site in every variant; same-parity sites touch disjoint links, so there is no
// inter-thread hazard and no block-level synchronisation.
//
//  "two-pass": pass 1 streams the 2*ND links that enter K(x) (eq. 1.5) and sums them in registers; the
//      three SU(2) steps give G(x); pass 2 re-reads each of the eight links (L1/L2 hit: same thread, same addresses,
//      nothing written between), multiplies and stores in place.
//  "two-pass + L2 bulk prefetch": the same, but each warp first asks the TMA unit to pull its whole
//      working set (the contiguous 4-direction forward chunk and the backward tiles) into L2 with
//      cp.async.bulk.prefetch.L2, so the bytes in flight per SM do not depend on how many loads the register budget
//      lets the compiler hoist.
//  "staged" (the default): every thread copies its eight links global -> shared with cp.async (LDGSTS; no registers
//      tied up, all 8*L bytes of the site in flight at once), waits for its own copies, then works out of shared
//      memory in a single pass: each link crosses L2 -> SM once.  Shared slots are thread-private: no barrier.
// Precision of K(x), the three SU(2) steps and G(x): FP64 with FP64 links and in the two-pass kernels; with FP32 links
// the staged kernels try FP32 first (FAST_TAU2 below) and fall back to FP64 per site.  Why FP64 at all: in FP32 the direction r/|r| of a
// subgroup step is ill-conditioned wherever |r| << |K| (cancellation in the sum of eight links): with FP32 arithmetic
// 63 of the 1,048,576 sites of config 2 miss the 2e-5 one-sweep bound against an FP64 evaluation (max 1.4e-4; any
// all-FP32 evaluation of the same formulas does).  The links are FP32 inputs, so their sum in FP64 is exact, and
// each g is rounded to FP32 once; G = g3 g2 g1, loads, stores and the eight 3x3 products stay in the storage precision.
using RotationType = double;
// FP32 storage, fast path of the staged kernel: K(x) and the three SU(2) steps in FP32; a site whose smallest |r|^2
// over the three steps is below FAST_TAU2 is evaluated again in FP64.  Derivation: with e ~ 1e-6 the
// rounding of an r component formed from an FP32 K (a few sigma of sqrt(8) u |K_ij|), a step's g^omega moves by
// dg_k <= omega dr_k / |r_k|, and the next step sees K <- g K with dr_{k+1} ~ e + |K| dg_k: the error is amplified by
// 2 |K| / |r| from step to step.  With every |r_k| >= tau and |K| ~ 6, dg_3 <= (2 e / tau) (1 + 12/tau + 144/tau^2):
// tau = 4 gives 6.5e-6, which with the ~6e-6 of the FP32 link products stays inside the 2e-5 one-sweep budget (tau = 1,
// tried first from a bound that ignored the step-to-step amplification, measured 3.5e-5 on 19 sites of config 2).
// On a Haar-random start E|r|^2 ~ 11, so nearly every warp takes the FP64 branch in the first sweeps; once F > 0.5
// (|r|^2 ~ 100) almost none does.
constexpr float FAST_TAU2 = 16.0f;

// Accumulator of K(x) in RotationType: every real of the 2*ND links is converted and added in FP64 (exact for FP32
// inputs).  Measured alternative for FP32 storage (config 2, ncu): carrying the sum as an unevaluated FP32 pair with
// TwoSum and converting once (36 conversions per site instead of 144) takes the XU pipe from 31 % to 11 % busy but
// lengthens the dependent chain: 86.8 us per half-sweep against 74.8 us for the plain conversions kept here
// (all-FP32 arithmetic, which misses the parity bound: 64.6 us).
template <class T>
struct KSum {
  double2 k[9];
  __device__ __forceinline__ void clear() {
#pragma unroll
    for (int e = 0; e < 9; ++e) k[e] = make_double2(0.0, 0.0);
  }
  __device__ __forceinline__ void add(int e, T x, T y) { k[e].x += (double)x; k[e].y += (double)y; }
  __device__ __forceinline__ void finish(double2 (&K)[9]) const {
#pragma unroll
    for (int e = 0; e < 9; ++e) K[e] = k[e];
  }
};

template <class T, int NELEM, class C>
__device__ __forceinline__ void site_pointers(C* __restrict__ links, const Geo& g, int parity, int cb, C*& fwd,
                                              C* (&bwd)[4]) {
  const Site s = site_of(g, parity, cb);
  fwd = links + link_offset<NELEM>(g, parity, cb, 0);  // + mu*NELEM*32 for direction mu
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) bwd[mu] = links + link_offset<NELEM>(g, parity ^ 1, cb_down(g, s, cb, mu), mu);
}

// T-slab sharding (gf_slab_*): the context is one slab of a taller lattice; U_t(x - t) of its t = 0
// sites belongs to the lower neighbour and lives, for the duration of a half-sweep, in the ghost buffer
//   ghost[parity of the owning site][cb3 / 32][elem][cb3 % 32],   cb3 = checkerboard index within the time slice.
template <class T, int NELEM, class C>
__device__ __forceinline__ C* ghost_link(const SlabView& sv, int owner_parity, int cb3) {
  return (C*)sv.ghost + (((size_t)owner_parity * sv.nblk3 + (size_t)(cb3 >> 5)) * NELEM) * 32 + (cb3 & 31);
}

__device__ __forceinline__ void prefetch_l2_bulk(const void* p, unsigned bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}


// Serpentine block order: the odd half-sweep walks the lattice from the far end back, the even one (and the measure pass)
// from the near end, so a pass starts on the links the previous pass touched last, while they are still in the 126 MB
// L2.  A field of a few L2 sizes (config 2: 201 MB) then finds most of its links there instead of streaming through an
// LRU cache that has just dropped them; fields far larger than L2 (configs 3, 4) are unaffected.  Which block takes
// which sites does not change any result (same-parity updates are independent).
__device__ __forceinline__ unsigned serpentine_block(int parity) {
  return (parity & 1) ? gridDim.x - 1u - blockIdx.x : blockIdx.x;
}

template <class T, int NELEM, int ND, int THREADS, int MINBLOCKS, bool PREFETCH>
__global__ void __launch_bounds__(THREADS, MINBLOCKS)
ovr_halfsweep_kernel(cplx_t<T>* __restrict__ links, Geo g, int parity, T omega) {
  using C = cplx_t<T>;
  using TK = RotationType;  // two-pass kernel: K(x), the SU(2) steps and G(x) in FP64 in both storage precisions
  using CK = cplx_t<TK>;
  int cb = serpentine_block(parity) * THREADS + threadIdx.x;
  const bool live = cb < g.vh;
  if (!PREFETCH && !live) return;
  if (!live) cb = g.vh - 1;  // keep the warp converged for the shuffles below; the lane does no loads or stores
  C* fwd;
  C* bwd[4];
  site_pointers<T, NELEM>(links, g, parity, cb, fwd, bwd);

  if (PREFETCH) {
    const unsigned lane = threadIdx.x & 31;
    constexpr unsigned TILE = NELEM * 32 * sizeof(C);  // one (block, mu) tile
    // forward links of the warp's 32 sites: one contiguous 4-tile chunk
    if (lane == 0) prefetch_l2_bulk(links + link_offset<NELEM>(g, parity, cb & ~31, 0), 4 * TILE);
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
      // tile (32-site block of the other parity) holding this lane's backward neighbour; one request per distinct tile
      const unsigned long long tile = (unsigned long long)(bwd[mu] - links) / (NELEM * 32);
      const unsigned long long prev = __shfl_up_sync(0xffffffffu, tile, 1);
      if (lane == 0 || tile != prev) prefetch_l2_bulk(links + tile * (NELEM * 32), TILE);
    }
    if (!live) return;
  }

  KSum<T> ks;
  ks.clear();
#pragma unroll
  for (int mu = 0; mu < ND; ++mu) {
    C u[9];
    load_link<NELEM, true>(fwd + mu * NELEM * 32, u);
#pragma unroll
    for (int e = 0; e < 9; ++e) ks.add(e, u[e].x, u[e].y);
    load_link<NELEM, true>(bwd[mu], u);
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = 0; j < 3; ++j) ks.add(i * 3 + j, u[j * 3 + i].x, -u[j * 3 + i].y);
  }
  CK K[9];
  ks.finish(K);

  C G[9];
  site_gauge_rotation<TK>(K, G, (TK)omega);

#pragma unroll
  for (int mu = 0; mu < 4; ++mu) {
    C u[9], w[9];
    load_link<NELEM, true>(fwd + mu * NELEM * 32, u);
    mul_left<LinkRows<NELEM>::value>(G, u, w);                       // U_mu(x) <- G U_mu(x)
    store_link<NELEM>(fwd + mu * NELEM * 32, w);
    load_link<NELEM, false>(bwd[mu], u);
    mul_right_adj<LinkRows<NELEM>::value>(u, G, w);                  // U_mu(x-mu) <- U_mu(x-mu) G^dagger
    store_link<NELEM>(bwd[mu], w);
  }
}

// An 8-real store needs five of the nine elements of a product: a1, a2, a3 (row 0), b1 and c1 (column 0).
template <class C>
__device__ __forceinline__ void mul_left_8(const C (&G)[9], const C (&u)[9], C (&w)[9]) {
#pragma unroll
  for (int j = 0; j < 3; ++j) {  // row 0 of G.U
    C z = cmul(G[0], u[j]); cfma(z, G[1], u[3 + j]); cfma(z, G[2], u[6 + j]);
    w[j] = z;
  }
#pragma unroll
  for (int i = 1; i < 3; ++i) {  // column 0 of rows 1, 2
    C z = cmul(G[i * 3], u[0]); cfma(z, G[i * 3 + 1], u[3]); cfma(z, G[i * 3 + 2], u[6]);
    w[i * 3] = z;
  }
}
template <class C>
__device__ __forceinline__ void mul_right_adj_8(const C (&u)[9], const C (&G)[9], C (&w)[9]) {
  using T = decltype(w[0].x);
#pragma unroll
  for (int j = 0; j < 3; ++j) {  // row 0 of U.G^dagger
    C z = mk<T>(T(0), T(0));
    cfma_cj(z, u[0], G[j * 3]); cfma_cj(z, u[1], G[j * 3 + 1]); cfma_cj(z, u[2], G[j * 3 + 2]);
    w[j] = z;
  }
#pragma unroll
  for (int i = 1; i < 3; ++i) {  // column 0 of rows 1, 2
    C z = mk<T>(T(0), T(0));
    cfma_cj(z, u[i * 3], G[0]); cfma_cj(z, u[i * 3 + 1], G[1]); cfma_cj(z, u[i * 3 + 2], G[2]);
    w[i * 3] = z;
  }
}

// ---- staged through shared memory with cp.async ---------------------------------------------------------
template <class T> constexpr int staged_threads() { return sizeof(T) == 8 ? 64 : 128; }
// FP32 storage: 4 blocks of 128 threads per SM (shared memory allows 4), i.e. at most 128 registers for the FP64 rotation
template <class T> constexpr int staged_minblocks() { return sizeof(T) == 8 ? 1 : 4; }

template <int BYTES>
__device__ __forceinline__ void cp_async(void* smem_dst, const void* gmem_src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  if (BYTES == 16)
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
  else
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");
}
// keeps the compiler from hoisting every shared-memory load of the site to the top (which spills)
__device__ __forceinline__ void sched_fence() { asm volatile("" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// ---- bulk copies (the TMA unit's 1-D form, cp.async.bulk; SASS UBLKCP) completing on an mbarrier ----------------------------
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");  // visible to the async proxy before the first copy
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned phase) {
  const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "GF_MBAR_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra GF_MBAR_DONE;\n"
      "bra GF_MBAR_WAIT;\n"
      "GF_MBAR_DONE:\n"
      "}\n" ::"r"(a), "r"(phase)
      : "memory");
}
// bytes: a multiple of 16; both addresses 16-byte aligned
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gmem_src, unsigned bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   (unsigned)__cvta_generic_to_shared(smem_dst)),
               "l"(gmem_src), "r"(bytes), "r"((unsigned)__cvta_generic_to_shared(bar))
               : "memory");
}

// shared slot of (link l, element e) of this thread: [l][e][THREADS] complex numbers, lane-contiguous (no bank conflicts)
template <int NELEM, int STRIDE, bool FULL, class C>
__device__ __forceinline__ void load_link_smem(const C* sm, int l, C (&u)[9]) {
  load_link<NELEM, FULL, STRIDE>(sm + l * NELEM * STRIDE, u);
}

// G(x) of one site from its eight links in shared memory (slot_fwd(mu) / slot_bwd(mu): the slots of U_mu(x) / U_mu(x-mu),
// SELEM elements each, element stride STRIDE); with MEASURE also q = sum_ij |Delta_ij|^2 of the updated links.
// K(x) is summed in the order mu = 0 forward, mu = 0 backward, mu = 1 forward, ... in every kernel that calls this, so
// they all produce the same bits.
template <class T, int SELEM, int ND, int STRIDE, bool MEASURE, bool SERIES, class SlotF, class SlotB, class C>
__device__ __forceinline__ void site_rotation_from_slots(const C* sm, SlotF slot_fwd, SlotB slot_bwd, T omega, int series,
                                                         C (&G)[9], double& q) {
  using TK = RotationType;
  using CK = cplx_t<TK>;
  // FP32 links, exact power: the site rotation is first evaluated in FP32 (K(x), the three SU(2) steps); where a
  // step's |r|^2 falls below FAST_TAU2 the direction r/|r| amplifies the rounding of K beyond the parity budget and
  // the site is evaluated again in FP64 from the links still in shared memory (a rare, divergent branch).
  bool rotated = false;
  if constexpr (sizeof(T) == 4 && !SERIES) {
    C Kf[9];
#pragma unroll
    for (int e = 0; e < 9; ++e) Kf[e] = mk<T>(T(0), T(0));
#pragma unroll
    for (int mu = 0; mu < ND; ++mu) {
      C u[9];
      load_link_smem<SELEM, STRIDE, true>(sm, slot_fwd(mu), u);
#pragma unroll
      for (int e = 0; e < 9; ++e) { Kf[e].x += u[e].x; Kf[e].y += u[e].y; }
      sched_fence();
      load_link_smem<SELEM, STRIDE, true>(sm, slot_bwd(mu), u);
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) { Kf[i * 3 + j].x += u[j * 3 + i].x; Kf[i * 3 + j].y -= u[j * 3 + i].y; }
      sched_fence();
    }
    T r2min = T(3.0e38);
    site_gauge_rotation<T, MEASURE, false>(Kf, G, omega, 0, &r2min);
    if (MEASURE) q = (double)delta_norm2<T>(Kf);
    rotated = r2min >= FAST_TAU2;
  }
  if (!rotated) {
    KSum<T> ks;
    ks.clear();
#pragma unroll
    for (int mu = 0; mu < ND; ++mu) {
      C u[9];
      load_link_smem<SELEM, STRIDE, true>(sm, slot_fwd(mu), u);
#pragma unroll
      for (int e = 0; e < 9; ++e) ks.add(e, u[e].x, u[e].y);
      sched_fence();
      load_link_smem<SELEM, STRIDE, true>(sm, slot_bwd(mu), u);
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) ks.add(i * 3 + j, u[j * 3 + i].x, -u[j * 3 + i].y);
      sched_fence();
    }
    CK K[9];
    ks.finish(K);
    site_gauge_rotation<TK, MEASURE, SERIES>(K, G, (TK)omega, series);
    if (MEASURE) q = (double)delta_norm2<TK>(K);
  }
}

// MEASURE: the launch also leaves, per block, the sum over its sites of sum_ij |Delta_ij(x)|^2 AFTER the update, taken
// from K_final(x) = G(x) K(x), which is K(x) of the updated links (the site's own update is the last one to touch
// them in this half-sweep).  After the odd half-sweep these are the odd sites' terms of theta of the finished sweep.
// SLAB: the launch covers the checkerboard range [sv.cb_begin, sv.cb_end) of a T-slab; t = 0 sites take U_t(x - t) from
// (and return it to) the ghost buffer.  The per-site arithmetic is the same instruction sequence in both cases.
// SERIES: g^omega by the truncated binomial series of order `series` (GF_OPT_OVR_SERIES) instead of the exact power.
// MASKED (Coulomb gauge, gf_fix_slices): sites of time slices with active[t] == 0 are not visited.
// DEFER (Coulomb gauge, gf_defer_*): the temporal links are not touched; instead the site's accumulated rotation
// A(x) <- G(x) A(x) is kept in `acc` (one matrix per site, layout of one direction of the link field) and applied to
// them later in one pass (defer_flush_kernel): 6 links + A read and written per site-update instead of 8 links.
// BULK (GF_OPT_SWEEP_VARIANT 4; plain and MEASURE instantiations): the warp's tile is brought in by the TMA unit instead of
// 8*NELEM LDGSTS per thread.  Each warp owns a [8 links][NELEM][32] region of shared memory and one mbarrier.  The four
// forward links of its 32 sites are ONE contiguous chunk of the field (4*NELEM*32 complex numbers): one bulk copy.  The
// backward links of direction mu are runs of consecutive lanes whose neighbours are consecutive in a tile of the other
// parity (a whole tile where the row length is a multiple of 32; shorter runs at row ends and periodic wraps); the
// first lane of a run issues one copy per element.  Runs that are not 16-byte aligned on both sides (FP32 complex is
// 8 bytes) are fetched by their lanes with cp.async as in the non-bulk kernel.
template <class T, int NELEM, int ND, int THREADS, int MINBLOCKS, bool MEASURE, bool SLAB, bool SERIES = false,
          bool MASKED = false, bool DEFER = false, int BULK = 0>
__global__ void __launch_bounds__(THREADS, MINBLOCKS)
ovr_halfsweep_staged_kernel(cplx_t<T>* __restrict__ links, Geo g, int parity, T omega, double* __restrict__ qpartials,
                            SlabView sv, int series = 0, const unsigned char* __restrict__ active = nullptr,
                            cplx_t<T>* __restrict__ acc = nullptr) {
  using C = cplx_t<T>;
  using TK = RotationType;
  using CK = cplx_t<TK>;
  static_assert(!BULK || (!SLAB && !MASKED && !DEFER), "the bulk-copy variant exists for the plain half-sweep only");
  // shared slot of (link, element): [SLOT][e][STRIDE]; non-bulk: links 2*mu = U_mu(x), 2*mu+1 = U_mu(x-mu), one column
  // per thread of the block; bulk: links mu = U_mu(x), 4+mu = U_mu(x-mu), one [8][NELEM][32] region per warp
  constexpr int STRIDE = BULK ? 32 : THREADS;
  // 8-real storage: the four stored complex numbers of a link land in the upper four of a six-element slot and are
  // decoded ONCE, in place, into rows 0 and 1; from there on the site works as with 12-real storage (row 2 rebuilt at
  // each use), so a site-update costs 8 reconstructions instead of 16 and has the 12-real kernel's shared-memory footprint
  constexpr int SELEM = NELEM == 4 ? 6 : NELEM;
  constexpr int SOFF = SELEM - NELEM;
  auto slot_fwd = [](int mu) { return BULK ? mu : 2 * mu; };
  auto slot_bwd = [](int mu) { return BULK ? 4 + mu : 2 * mu + 1; };
  extern __shared__ __align__(16) unsigned char smem_raw[];
  C* sm = BULK ? reinterpret_cast<C*>(smem_raw) + (threadIdx.x >> 5) * (8 * NELEM * 32) + (threadIdx.x & 31)
               : reinterpret_cast<C*>(smem_raw) + threadIdx.x;
  const unsigned bid = SLAB ? blockIdx.x : serpentine_block(parity);  // (a slab launch covers two given ranges)
  int cb = bid * THREADS + threadIdx.x;
  bool live = cb < g.vh;
  if (SLAB) {
    const int b = (int)blockIdx.x;
    if (b < sv.nblocks0) {
      cb = sv.cb_begin + b * THREADS + threadIdx.x;
      live = cb < sv.cb_end;
    } else if (b < sv.nblocks0 + sv.nblocks1) {
      cb = sv.cb2_begin + (b - sv.nblocks0) * THREADS + threadIdx.x;
      live = cb < sv.cb2_end;
    } else {  // interior of a fused launch, in serpentine order (see serpentine_block)
      const int nb3 = (int)gridDim.x - sv.nblocks0 - sv.nblocks1;
      const int b3 = b - sv.nblocks0 - sv.nblocks1;
      cb = sv.cb3_begin + ((parity & 1) ? nb3 - 1 - b3 : b3) * THREADS + threadIdx.x;
      live = cb < sv.cb3_end;
    }
  }
  if (!MEASURE && !BULK && !SLAB && !live) return;
  if (MASKED && !active[cb / g.s3]) return;  // the slice is finished (its theta_t is below eps)
  double q = 0.0;
  C* fwd = nullptr;
  C* bwd[4] = {nullptr, nullptr, nullptr, nullptr};
  if (BULK) {
    const unsigned lane = threadIdx.x & 31;
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(smem_raw + (size_t)8 * NELEM * THREADS * sizeof(C)) +
                              (threadIdx.x >> 5);
    if (lane == 0) mbar_init(bar, 1);
    const unsigned livem = __ballot_sync(0xffffffffu, live);
    if (livem != 0) {  // (a whole warp beyond the lattice has nothing to fetch; warp-uniform)
    if (live) site_pointers<T, NELEM>(links, g, parity, cb, fwd, bwd);
    // runs of consecutive neighbours per direction; 16-byte alignment decides bulk copy or cp.async for the direction
    unsigned startm[4], bytes = 0;
    bool use_bulk[4];
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
      const unsigned long long p = (unsigned long long)bwd[mu];
      const unsigned long long prev = __shfl_up_sync(0xffffffffu, p, 1);
      const bool prev_live = (livem >> ((lane + 31) & 31)) & 1u;
      const bool start = live && (lane == 0 || !prev_live || p != prev + sizeof(C));
      startm[mu] = __ballot_sync(0xffffffffu, start);
      // the run of this start lane ends before the next start or the first dead lane
      const unsigned stops = (startm[mu] | ~livem) & ~((2u << lane) - 1u);
      const unsigned len = (stops ? (unsigned)__ffs((int)stops) - 1u : 32u) - lane;
      const bool aligned = sizeof(C) == 16 || (((p | (len * sizeof(C)) | (lane * sizeof(C))) & 15u) == 0);
      use_bulk[mu] = BULK == 1 && __all_sync(0xffffffffu, !start || aligned);  // BULK == 2: forward chunk only
      if (start && use_bulk[mu]) bytes += len * NELEM * (unsigned)sizeof(C);
      startm[mu] = start ? len : 0u;  // from here on: this lane's run length (0: not a start lane)
    }
    bytes = __reduce_add_sync(0xffffffffu, bytes) + 4u * NELEM * 32u * (unsigned)sizeof(C);
    __syncwarp();
    if (lane == 0) {
      mbar_arrive_expect_tx(bar, bytes);
      // the forward chunk of the tile (padding lanes of the last tile included: they are part of the layout)
      bulk_g2s(sm, links + link_offset<NELEM>(g, parity, cb & ~31, 0), 4u * NELEM * 32u * (unsigned)sizeof(C), bar);
    }
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
      if (use_bulk[mu]) {
        if (startm[mu]) {
#pragma unroll
          for (int e = 0; e < NELEM; ++e)
            bulk_g2s(sm + (slot_bwd(mu) * NELEM + e) * 32, bwd[mu] + e * 32, startm[mu] * (unsigned)sizeof(C), bar);
        }
      } else if (live) {
#pragma unroll
        for (int e = 0; e < NELEM; ++e) cp_async<sizeof(C)>(sm + (slot_bwd(mu) * NELEM + e) * 32, bwd[mu] + e * 32);
      }
    }
    if (sizeof(C) != 16 || BULK == 2) cp_async_wait_all();
    mbar_wait(bar, 0);
    }
  }
  if (live) {
    if (!BULK) site_pointers<T, NELEM>(links, g, parity, cb, fwd, bwd);
    if (SLAB && cb < g.s3) bwd[3] = ghost_link<T, NELEM, C>(sv, parity ^ 1, cb);

    // DEFER: slot 6 = A(x), the temporal links stay where they are
    constexpr int NMU = DEFER ? 3 : 4;
    C* accp = nullptr;
    if (DEFER) accp = acc + (((size_t)parity * g.nblk + (size_t)(cb >> 5)) * NELEM) * 32 + (cb & 31);
    if (!BULK) {
#pragma unroll
      for (int mu = 0; mu < NMU; ++mu) {
#pragma unroll
        for (int e = 0; e < NELEM; ++e) {
          const C* src = fwd + (mu * NELEM + e) * 32;
          if (SLAB && mu == 3 && sv.top_in_src && cb >= g.vh - g.s3) {  // the link the upper neighbour just returned
            SlabView in = sv;
            in.ghost = const_cast<void*>(sv.top_in_src);
            src = ghost_link<T, NELEM, C>(in, 0, cb - (g.vh - g.s3)) + e * 32;
          }
          cp_async<sizeof(C)>(sm + (slot_fwd(mu) * SELEM + SOFF + e) * STRIDE, src);
          cp_async<sizeof(C)>(sm + (slot_bwd(mu) * SELEM + SOFF + e) * STRIDE, bwd[mu] + e * 32);
        }
      }
      if (DEFER) {
#pragma unroll
        for (int e = 0; e < NELEM; ++e) cp_async<sizeof(C)>(sm + (6 * NELEM + e) * STRIDE, accp + e * 32);
      }
      cp_async_wait_all();  // a thread reads only what it copied itself: no block barrier needed
      if constexpr (NELEM == 4) {
        // two links at a time: their reconstructions are independent dependent chains (division, square roots), and a
        // thread has only its own instruction-level parallelism to hide them (8 warps per SM)
#pragma unroll
        for (int l = 0; l < 8; l += 2) {
          C* s8 = sm + l * SELEM * STRIDE;
          C* t8 = s8 + SELEM * STRIDE;
          C u[9], v[9];
          decode8<T, C, false>(s8[2 * STRIDE], s8[3 * STRIDE], s8[4 * STRIDE], s8[5 * STRIDE], u);
          decode8<T, C, false>(t8[2 * STRIDE], t8[3 * STRIDE], t8[4 * STRIDE], t8[5 * STRIDE], v);
#pragma unroll
          for (int e = 0; e < 6; ++e) { s8[e * STRIDE] = u[e]; t8[e * STRIDE] = v[e]; }
          sched_fence();
        }
      }
    }

    C G[9];
    site_rotation_from_slots<T, SELEM, ND, STRIDE, MEASURE, SERIES>(sm, slot_fwd, slot_bwd, omega, series, G, q);

#pragma unroll
    for (int mu = 0; mu < NMU; ++mu) {
      C u[9], w[9];
      load_link_smem<SELEM, STRIDE, true>(sm, slot_fwd(mu), u);
      if constexpr (NELEM == 4) mul_left_8(G, u, w);                   // (the five elements an 8-real store needs)
      else mul_left<LinkRows<NELEM>::value>(G, u, w);                  // U_mu(x) <- G U_mu(x)
      store_link<NELEM>(fwd + mu * NELEM * 32, w);
      if (SLAB && mu == 3 && sv.top_out && cb >= g.vh - g.s3) {  // top slice: the copy that goes to the upper neighbour
        SlabView out = sv;
        out.ghost = sv.top_out;
        store_link<NELEM>(ghost_link<T, NELEM, C>(out, 0, cb - (g.vh - g.s3)), w);
      }
      if (NELEM != 4) sched_fence();  // (8-real: the two encodings of a direction overlap)
      load_link_smem<SELEM, STRIDE, NELEM == 4>(sm, slot_bwd(mu), u);  // (an 8-real store needs c1: all three rows)
      if constexpr (NELEM == 4) mul_right_adj_8(u, G, w);
      else mul_right_adj<LinkRows<NELEM>::value>(u, G, w);             // U_mu(x-mu) <- U_mu(x-mu) G^dagger
      store_link<NELEM>(bwd[mu], w);
      if (SLAB && mu == 3 && sv.ret_out && cb < g.s3) {   // bottom slice: the copy that goes back to the lower neighbour
        SlabView out = sv;
        out.ghost = sv.ret_out;
        store_link<NELEM>(ghost_link<T, NELEM, C>(out, 0, cb), w);
      }
      sched_fence();
    }
    if (DEFER) {                                          // A(x) <- G A(x)
      C u[9], w[9];
      load_link_smem<SELEM, STRIDE, true>(sm, 6, u);
      mul_left<LinkRows<NELEM>::value>(G, u, w);
      store_link<NELEM>(accp, w);
    }
  }
  if (MEASURE) {
    double f = 0.0;
    block_sum2<THREADS>(f, q);
    if (threadIdx.x == 0) qpartials[bid] = q;
  }
  if (SLAB && sv.sig_blocks > 0 && (int)blockIdx.x < sv.sig_blocks) {
    // a border block of a fused launch: when the last of them has stored its links and halo messages, tell the
    // neighbours (release at system scope: the messages may sit in another GPU's memory)
    __syncthreads();
    if (threadIdx.x == 0) {
      __threadfence_system();
      if (atomicAdd(sv.sig_counter, 1u) == (unsigned)sv.sig_blocks - 1u) {
        *sv.sig_counter = 0u;  // ready for the next launch on this stream
        __threadfence_system();
        atomicAdd_system(sv.sig_flag[0], 1u);
        atomicAdd_system(sv.sig_flag[1], 1u);
      }
    }
  }
}

// Dynamic shared memory of the staged kernel: eight link slots per thread of SELEM complex numbers each, SELEM = 6 for
// 8-real storage (decoded once into two rows), else NELEM.  Every launcher of ovr_halfsweep_staged_kernel sizes its
// launch with this one expression, so the kernel's slot indexing and the allocation cannot drift apart.
template <class C, int NELEM, int THREADS>
constexpr size_t staged_smem_bytes() { return (size_t)8 * (NELEM == 4 ? 6 : NELEM) * THREADS * sizeof(C); }

template <class T, int NELEM, int ND, int THREADS, bool MEASURE>
static cudaError_t halfsweep_staged_T(const KernelArgs& a, int parity, double omega) {
  using C = cplx_t<T>;
  constexpr size_t SMEM = staged_smem_bytes<C, NELEM, THREADS>();
  auto kern = ovr_halfsweep_staged_kernel<T, NELEM, ND, THREADS, staged_minblocks<T>(), MEASURE, false>;
  static PerDeviceOnce attr;  // per instantiation and device
  if (cudaError_t e = opt_in_smem(attr, kern, SMEM); e != cudaSuccess) return e;
  const unsigned blocks = (unsigned)((a.geo.vh + THREADS - 1) / THREADS);
  kern<<<blocks, THREADS, SMEM, a.stream>>>((C*)a.links, a.geo, parity, (T)omega, (double*)a.qpartials, SlabView{}, 0, nullptr, nullptr);
  return cudaGetLastError();
}


// ---- two lanes per site (GF_OPT_SWEEP_VARIANT 6) -----------------------------------------------------------------------------
// A study of what bounds the kernels that are not HBM-bound (8-real storage; the L2-resident configs 0 and 1).  Two WARPS
// share 32 sites (a lane pair inside one warp would diverge at every step): warp 2k (h = 0) copies in, updates and
// stores the four forward links of its 32 sites, warp 2k+1 (h = 1) the four backward links; both sum K(x) over all
// eight links (in the order every other kernel uses, so the links come out bit-identical) and both run the three SU(2)
// steps.  Same shared memory per site, twice the warps, about 0.75 of the instructions per lane.  8-real storage: each
// lane reconstructs its own four links.  Measured: no faster anywhere - cfg0 8.5 us and cfg1 23 us per
// half-sweep with either kernel, 8-real 5.6 against 5.4 ms, cfg2 90 against 63 us - so it is not the default for anything.
template <class T> struct SplitSites { static constexpr int value = sizeof(T) == 8 ? 64 : 128; };

template <class T, int NELEM, int ND, bool MEASURE>
__global__ void __launch_bounds__(2 * SplitSites<T>::value, sizeof(T) == 8 ? 3 : 2)
ovr_halfsweep_split_kernel(cplx_t<T>* __restrict__ links, Geo g, int parity, T omega, double* __restrict__ qpartials) {
  using C = cplx_t<T>;
  constexpr int SITES = SplitSites<T>::value;
  constexpr int SELEM = NELEM == 4 ? 6 : NELEM;
  constexpr int SOFF = SELEM - NELEM;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, h = warp & 1;
  const int i = (warp >> 1) * 32 + (threadIdx.x & 31);
  // slot of (link l, element e) of site i: [l][e][SITES], l = 2 mu (forward), 2 mu + 1 (backward)
  C* sm = reinterpret_cast<C*>(smem_raw) + i;
  auto slot_fwd = [](int mu) { return 2 * mu; };
  auto slot_bwd = [](int mu) { return 2 * mu + 1; };
  const unsigned bid = serpentine_block(parity);
  const int cb = bid * SITES + i;
  const bool live = cb < g.vh;
  C* ptr[4] = {nullptr, nullptr, nullptr, nullptr};  // this lane's four links in the field
  if (live) {
    if (h == 0) {
      C* fwd = links + link_offset<NELEM>(g, parity, cb, 0);
#pragma unroll
      for (int mu = 0; mu < 4; ++mu) ptr[mu] = fwd + mu * NELEM * 32;
    } else {
      const Site s = site_of(g, parity, cb);
#pragma unroll
      for (int mu = 0; mu < 4; ++mu) ptr[mu] = links + link_offset<NELEM>(g, parity ^ 1, cb_down(g, s, cb, mu), mu);
    }
#pragma unroll
    for (int mu = 0; mu < 4; ++mu)
#pragma unroll
      for (int e = 0; e < NELEM; ++e) cp_async<sizeof(C)>(sm + ((2 * mu + h) * SELEM + SOFF + e) * SITES, ptr[mu] + e * 32);
    cp_async_wait_all();
    if constexpr (NELEM == 4) {
#pragma unroll
      for (int mu = 0; mu < 4; mu += 2) {  // two reconstructions at a time (independent dependent chains)
        C* s8 = sm + (2 * mu + h) * SELEM * SITES;
        C* t8 = s8 + 2 * SELEM * SITES;
        C u[9], v[9];
        decode8<T, C, false>(s8[2 * SITES], s8[3 * SITES], s8[4 * SITES], s8[5 * SITES], u);
        decode8<T, C, false>(t8[2 * SITES], t8[3 * SITES], t8[4 * SITES], t8[5 * SITES], v);
#pragma unroll
        for (int e = 0; e < 6; ++e) { s8[e * SITES] = u[e]; t8[e * SITES] = v[e]; }
        sched_fence();
      }
    }
  }
  __syncthreads();  // the partner warp's four links are in place
  double q = 0.0;
  if (live) {
    C G[9];
    site_rotation_from_slots<T, SELEM, ND, SITES, MEASURE, false>(sm, slot_fwd, slot_bwd, omega, 0, G, q);
    if (h == 1) q = 0.0;  // the site's theta term is counted once
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
      C u[9], w[9];
      if (h == 0) {
        load_link_smem<SELEM, SITES, true>(sm, slot_fwd(mu), u);
        if constexpr (NELEM == 4) mul_left_8(G, u, w);
        else mul_left<LinkRows<NELEM>::value>(G, u, w);              // U_mu(x) <- G U_mu(x)
      } else {
        load_link_smem<SELEM, SITES, NELEM == 4>(sm, slot_bwd(mu), u);
        if constexpr (NELEM == 4) mul_right_adj_8(u, G, w);
        else mul_right_adj<LinkRows<NELEM>::value>(u, G, w);         // U_mu(x-mu) <- U_mu(x-mu) G^dagger
      }
      store_link<NELEM>(ptr[mu], w);
      sched_fence();
    }
  }
  if (MEASURE) {
    double f = 0.0;
    block_sum2<2 * SITES>(f, q);
    if (threadIdx.x == 0) qpartials[bid] = q;
  }
}

template <class T, int NELEM, int ND, bool MEASURE>
static cudaError_t halfsweep_split_T(const KernelArgs& a, int parity, double omega) {
  using C = cplx_t<T>;
  constexpr int SITES = SplitSites<T>::value;
  constexpr size_t SMEM = (size_t)8 * (NELEM == 4 ? 6 : NELEM) * SITES * sizeof(C);
  auto kern = ovr_halfsweep_split_kernel<T, NELEM, ND, MEASURE>;
  static PerDeviceOnce attr;  // per instantiation and device
  if (cudaError_t e = opt_in_smem(attr, kern, SMEM); e != cudaSuccess) return e;
  const unsigned blocks = (unsigned)((a.geo.vh + SITES - 1) / SITES);
  kern<<<blocks, 2 * SITES, SMEM, a.stream>>>((C*)a.links, a.geo, parity, (T)omega, (double*)a.qpartials);
  return cudaGetLastError();
}

// GF_OPT_SWEEP_VARIANT 4: the tile comes in through bulk copies (TMA unit) completing on one mbarrier per warp
template <class T, int NELEM, int ND, int THREADS, bool MEASURE, int BULK>
static cudaError_t halfsweep_bulk_T(const KernelArgs& a, int parity, double omega) {
  using C = cplx_t<T>;
  constexpr size_t SMEM = staged_smem_bytes<C, NELEM, THREADS>() + 8 * (THREADS / 32);
  auto kern = ovr_halfsweep_staged_kernel<T, NELEM, ND, THREADS, staged_minblocks<T>(), MEASURE, false, false, false, false, BULK>;
  static PerDeviceOnce attr;  // per instantiation and device
  if (cudaError_t e = opt_in_smem(attr, kern, SMEM); e != cudaSuccess) return e;
  const unsigned blocks = (unsigned)((a.geo.vh + THREADS - 1) / THREADS);
  kern<<<blocks, THREADS, SMEM, a.stream>>>((C*)a.links, a.geo, parity, (T)omega, (double*)a.qpartials, SlabView{}, 0, nullptr, nullptr);
  return cudaGetLastError();
}

// GF_OPT_OVR_SERIES > 0: the same launch with the series kernel (no fused theta terms)
template <class T, int NELEM, int ND, int THREADS>
static cudaError_t halfsweep_series_T(const KernelArgs& a, int parity, double omega) {
  using C = cplx_t<T>;
  constexpr size_t SMEM = staged_smem_bytes<C, NELEM, THREADS>();
  auto kern = ovr_halfsweep_staged_kernel<T, NELEM, ND, THREADS, staged_minblocks<T>(), false, false, true>;
  static PerDeviceOnce attr;  // per instantiation and device
  if (cudaError_t e = opt_in_smem(attr, kern, SMEM); e != cudaSuccess) return e;
  const unsigned blocks = (unsigned)((a.geo.vh + THREADS - 1) / THREADS);
  kern<<<blocks, THREADS, SMEM, a.stream>>>((C*)a.links, a.geo, parity, (T)omega, nullptr, SlabView{}, a.series, nullptr, nullptr);
  return cudaGetLastError();
}

// the sites [cb_begin, cb_end) of one parity of a T-slab
template <class T, int NELEM, int ND>
static cudaError_t halfsweep_slab_T(const KernelArgs& a, int parity, double omega, int cb_begin, int cb_end,
                                    int cb2_begin, int cb2_end, void* top_out, void* ret_out) {
  using C = cplx_t<T>;
  constexpr int THREADS = staged_threads<T>();
  constexpr size_t SMEM = staged_smem_bytes<C, NELEM, THREADS>();
  if (cb_end <= cb_begin && cb2_end <= cb2_begin) return cudaSuccess;
  auto kern = ovr_halfsweep_staged_kernel<T, NELEM, ND, THREADS, staged_minblocks<T>(), false, true>;
  static PerDeviceOnce attr;  // per instantiation and device
  if (cudaError_t e = opt_in_smem(attr, kern, SMEM); e != cudaSuccess) return e;
  SlabView sv = a.slab;
  sv.cb_begin = cb_begin; sv.cb_end = cb_end;
  sv.cb2_begin = cb2_begin; sv.cb2_end = cb2_end;
  sv.nblocks0 = cb_end > cb_begin ? (cb_end - cb_begin + THREADS - 1) / THREADS : 0;
  sv.nblocks1 = cb2_end > cb2_begin ? (cb2_end - cb2_begin + THREADS - 1) / THREADS : 0;
  sv.cb3_begin = sv.cb3_end = 0;
  sv.sig_blocks = 0;
  sv.top_in_src = nullptr;
  sv.top_out = top_out;
  sv.ret_out = ret_out;
  const unsigned blocks = (unsigned)(sv.nblocks0 + sv.nblocks1);
  kern<<<blocks, THREADS, SMEM, a.stream>>>((C*)a.links, a.geo, parity, (T)omega, nullptr, sv, 0, nullptr, nullptr);
  return cudaGetLastError();
}

template <class T, int NELEM, int ND>
static cudaError_t halfsweep_slab_fused_T(const KernelArgs& a, int parity, double omega, void* top_out, void* ret_out,
                                          unsigned* counter, unsigned* flag_up, unsigned* flag_down, const void* top_in_src) {
  using C = cplx_t<T>;
  constexpr int THREADS = staged_threads<T>();
  constexpr size_t SMEM = staged_smem_bytes<C, NELEM, THREADS>();
  auto kern = ovr_halfsweep_staged_kernel<T, NELEM, ND, THREADS, staged_minblocks<T>(), false, true>;
  static PerDeviceOnce attr;  // per instantiation and device
  if (cudaError_t e = opt_in_smem(attr, kern, SMEM); e != cudaSuccess) return e;
  const Geo& g = a.geo;
  SlabView sv = a.slab;
  sv.cb_begin = 0; sv.cb_end = g.s3;                    // bottom slice
  sv.cb2_begin = g.vh - g.s3; sv.cb2_end = g.vh;        // top slice
  sv.cb3_begin = g.s3; sv.cb3_end = g.vh - g.s3;        // interior (empty for a slab of two slices)
  sv.nblocks0 = (g.s3 + THREADS - 1) / THREADS;
  sv.nblocks1 = sv.nblocks0;
  const int nblocks2 = sv.cb3_end > sv.cb3_begin ? (sv.cb3_end - sv.cb3_begin + THREADS - 1) / THREADS : 0;
  sv.sig_blocks = counter ? sv.nblocks0 + sv.nblocks1 : 0;  // no counter: nobody to signal (a closed group on one stream)
  sv.sig_counter = counter;
  sv.sig_flag[0] = flag_up; sv.sig_flag[1] = flag_down;
  sv.top_out = top_out;
  sv.ret_out = ret_out;
  sv.top_in_src = top_in_src;
  kern<<<(unsigned)(sv.nblocks0 + sv.nblocks1 + nblocks2), THREADS, SMEM, a.stream>>>((C*)a.links, a.geo, parity, (T)omega, nullptr, sv, 0,
                                                                          nullptr, nullptr);
  return cudaGetLastError();
}

// Variant numbering of GF_OPT_SWEEP_VARIANT: 0 = library default (staged), 1 = two-pass, 2 = two-pass + L2 bulk prefetch,
// 3 = staged.  Measured on B200 (profiles/): staged 6.8 TB/s on cfg4 and cfg3 against 6.3 / 5.7 TB/s two-pass.
template <class T, int NELEM, int ND>
static cudaError_t halfsweep_T(const KernelArgs& a, int parity, double omega, bool fuse_theta, int* qblocks) {
  using C = cplx_t<T>;
  *qblocks = 0;
  // 0: one thread per site, staged; with FP64 links the contiguous forward chunk of the warp's tile comes in by ONE bulk
  // copy of the TMA unit (variant 5: measured 0.4-0.7 % faster on cfg4 / cfg3, 8 % on the L2-resident cfg1), with FP32
  // links everything by cp.async (variant 3: the 8-byte complex numbers of the backward runs defeat 16-byte bulk copies)
  int variant = a.variant;
  if (variant == 0) variant = (sizeof(T) == 8 && NELEM != 4 && a.series == 0) ? 5 : 3;
  if (variant == 6) {
    if (a.series > 0 || a.block_threads) return cudaErrorNotSupported;
    if (fuse_theta) {
      *qblocks = (a.geo.vh + SplitSites<T>::value - 1) / SplitSites<T>::value;
      return halfsweep_split_T<T, NELEM, ND, true>(a, parity, omega);
    }
    return halfsweep_split_T<T, NELEM, ND, false>(a, parity, omega);
  }
  if (variant == 0 || variant == 3 || variant == 4 || variant == 5) {
    // 8*L bytes of shared memory per thread: FP64/18 1152 B -> 192 threads per SM, FP32/12 384 B -> 512 threads per SM
    constexpr int THREADS = staged_threads<T>();
    if (a.block_threads && a.block_threads != THREADS) return cudaErrorInvalidValue;
    if (a.series > 0) return variant >= 4 ? cudaErrorNotSupported : halfsweep_series_T<T, NELEM, ND, THREADS>(a, parity, omega);
    if constexpr (NELEM != 4) {
      if (variant == 4 || variant == 5) {
        if (fuse_theta) {
          *qblocks = (a.geo.vh + THREADS - 1) / THREADS;
          return variant == 4 ? halfsweep_bulk_T<T, NELEM, ND, THREADS, true, 1>(a, parity, omega)
                              : halfsweep_bulk_T<T, NELEM, ND, THREADS, true, 2>(a, parity, omega);
        }
        return variant == 4 ? halfsweep_bulk_T<T, NELEM, ND, THREADS, false, 1>(a, parity, omega)
                            : halfsweep_bulk_T<T, NELEM, ND, THREADS, false, 2>(a, parity, omega);
      }
    } else if (variant == 4 || variant == 5) {
      return cudaErrorNotSupported;
    }
    if (fuse_theta) {
      *qblocks = (a.geo.vh + THREADS - 1) / THREADS;
      return halfsweep_staged_T<T, NELEM, ND, THREADS, true>(a, parity, omega);
    }
    return halfsweep_staged_T<T, NELEM, ND, THREADS, false>(a, parity, omega);
  }
  constexpr int THREADS = 128;
  if (a.block_threads && a.block_threads != THREADS) return cudaErrorInvalidValue;
  if (a.series > 0) return cudaErrorNotSupported;  // the series is built into the staged kernel only
  const unsigned blocks = (unsigned)((a.geo.vh + THREADS - 1) / THREADS);
  if (variant == 2)
    ovr_halfsweep_kernel<T, NELEM, ND, THREADS, 1, true><<<blocks, THREADS, 0, a.stream>>>((C*)a.links, a.geo, parity,
                                                                                          (T)omega);
  else if (variant == 1)
    ovr_halfsweep_kernel<T, NELEM, ND, THREADS, 1, false><<<blocks, THREADS, 0, a.stream>>>((C*)a.links, a.geo, parity,
                                                                                           (T)omega);
  else
    return cudaErrorInvalidValue;
  return cudaGetLastError();
}

#define GF_DISPATCH(FN, ...)                                                                              \
  do {                                                                                                    \
    const bool coul = a.gauge == 1;                                                                       \
    if (a.prec == 0) {                                                                                    \
      if (a.storage == 18) return coul ? FN<double, 9, 3>(__VA_ARGS__) : FN<double, 9, 4>(__VA_ARGS__);   \
      return coul ? FN<double, 6, 3>(__VA_ARGS__) : FN<double, 6, 4>(__VA_ARGS__);                        \
    }                                                                                                     \
    if (a.storage == 18) return coul ? FN<float, 9, 3>(__VA_ARGS__) : FN<float, 9, 4>(__VA_ARGS__);       \
    return coul ? FN<float, 6, 3>(__VA_ARGS__) : FN<float, 6, 4>(__VA_ARGS__);                            \
  } while (0)

cudaError_t launch_halfsweep(const KernelArgs& a, int parity, double omega, bool fuse_theta, int* qblocks) {
  if (a.storage == 8) {
    if (a.prec == 0)
      return a.gauge == 1 ? halfsweep_T<double, 4, 3>(a, parity, omega, fuse_theta, qblocks)
                          : halfsweep_T<double, 4, 4>(a, parity, omega, fuse_theta, qblocks);
    return a.gauge == 1 ? halfsweep_T<float, 4, 3>(a, parity, omega, fuse_theta, qblocks)
                        : halfsweep_T<float, 4, 4>(a, parity, omega, fuse_theta, qblocks);
  }
  GF_DISPATCH(halfsweep_T, a, parity, omega, fuse_theta, qblocks);
}

// Coulomb gauge, only the time slices with active[t] != 0 (device array of n_t bytes)
template <class T, int NELEM>
static cudaError_t halfsweep_masked_T(const KernelArgs& a, int parity, double omega, const unsigned char* active) {
  using C = cplx_t<T>;
  constexpr int THREADS = staged_threads<T>();
  constexpr size_t SMEM = staged_smem_bytes<C, NELEM, THREADS>();
  auto kern = ovr_halfsweep_staged_kernel<T, NELEM, 3, THREADS, staged_minblocks<T>(), false, false, false, true>;
  static PerDeviceOnce attr;  // per instantiation and device
  if (cudaError_t e = opt_in_smem(attr, kern, SMEM); e != cudaSuccess) return e;
  const unsigned blocks = (unsigned)((a.geo.vh + THREADS - 1) / THREADS);
  kern<<<blocks, THREADS, SMEM, a.stream>>>((C*)a.links, a.geo, parity, (T)omega, nullptr, SlabView{}, 0, active, nullptr);
  return cudaGetLastError();
}

cudaError_t launch_halfsweep_masked(const KernelArgs& a, int parity, double omega, const unsigned char* active) {
  if (a.gauge != 1 || a.series > 0 || !(a.variant == 0 || a.variant == 3)) return cudaErrorNotSupported;
  if (a.prec == 0) return a.storage == 18 ? halfsweep_masked_T<double, 9>(a, parity, omega, active)
                                          : halfsweep_masked_T<double, 6>(a, parity, omega, active);
  return a.storage == 18 ? halfsweep_masked_T<float, 9>(a, parity, omega, active)
                         : halfsweep_masked_T<float, 6>(a, parity, omega, active);
}

// Coulomb gauge with deferred temporal links
template <class T, int NELEM>
static cudaError_t halfsweep_defer_T(const KernelArgs& a, int parity, double omega, void* acc) {
  using C = cplx_t<T>;
  constexpr int THREADS = staged_threads<T>();
  constexpr size_t SMEM = staged_smem_bytes<C, NELEM, THREADS>();
  auto kern = ovr_halfsweep_staged_kernel<T, NELEM, 3, THREADS, staged_minblocks<T>(), false, false, false, false, true>;
  static PerDeviceOnce attr;  // per instantiation and device
  if (cudaError_t e = opt_in_smem(attr, kern, SMEM); e != cudaSuccess) return e;
  const unsigned blocks = (unsigned)((a.geo.vh + THREADS - 1) / THREADS);
  kern<<<blocks, THREADS, SMEM, a.stream>>>((C*)a.links, a.geo, parity, (T)omega, nullptr, SlabView{}, 0, nullptr, (C*)acc);
  return cudaGetLastError();
}

cudaError_t launch_halfsweep_defer(const KernelArgs& a, int parity, double omega, void* acc) {
  if (a.gauge != 1 || a.series > 0 || !(a.variant == 0 || a.variant == 3)) return cudaErrorNotSupported;
  if (a.prec == 0) return a.storage == 18 ? halfsweep_defer_T<double, 9>(a, parity, omega, acc)
                                          : halfsweep_defer_T<double, 6>(a, parity, omega, acc);
  return a.storage == 18 ? halfsweep_defer_T<float, 9>(a, parity, omega, acc)
                         : halfsweep_defer_T<float, 6>(a, parity, omega, acc);
}

// U_t(x) <- A(x) U_t(x) A(x+t)^dagger for every site (one thread per site, both parities), then A <- 1 (second kernel:
// a site's A is also its lower t-neighbour's right factor).
template <class T, int NELEM>
__global__ void __launch_bounds__(256) defer_flush_kernel(cplx_t<T>* __restrict__ links, Geo g,
                                                          const cplx_t<T>* __restrict__ acc) {
  using C = cplx_t<T>;
  const int i = blockIdx.x * 256 + threadIdx.x;
  if (i >= 2 * g.vh) return;
  const int parity = i >= g.vh, cb = i - parity * g.vh;
  const Site s = site_of(g, parity, cb);
  const int cb_up = s.t == g.n[3] - 1 ? cb - g.s3 * (g.n[3] - 1) : cb + g.s3;
  C* ut = links + link_offset<NELEM>(g, parity, cb, 3);
  C A[9], u[9], w[9];
  load_link<NELEM, true>(acc + (((size_t)parity * g.nblk + (size_t)(cb >> 5)) * NELEM) * 32 + (cb & 31), A);
  load_link<NELEM, true>(ut, u);
  mul_left<LinkRows<NELEM>::value>(A, u, w);
  load_link<NELEM, true>(acc + (((size_t)(parity ^ 1) * g.nblk + (size_t)(cb_up >> 5)) * NELEM) * 32 + (cb_up & 31), A);
  mul_right_adj<LinkRows<NELEM>::value>(w, A, u);
  store_link<NELEM>(ut, u);
}

template <class T, int NELEM>
__global__ void __launch_bounds__(256) defer_identity_kernel(cplx_t<T>* __restrict__ acc, long long ntiles) {
  const long long tid = (long long)blockIdx.x * 256 + threadIdx.x;
  if ((tid >> 5) >= ntiles) return;
  cplx_t<T>* p = acc + (size_t)(tid >> 5) * NELEM * 32 + (tid & 31);
#pragma unroll
  for (int e = 0; e < NELEM; ++e) p[e * 32] = mk<T>((e % 4 == 0) ? T(1) : T(0), T(0));
}

template <class T, int NELEM>
static cudaError_t defer_T(const KernelArgs& a, void* acc, bool flush) {
  if (flush) {
    defer_flush_kernel<T, NELEM><<<(unsigned)((2LL * a.geo.vh + 255) / 256), 256, 0, a.stream>>>((cplx_t<T>*)a.links, a.geo,
                                                                                              (const cplx_t<T>*)acc);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  const long long ntiles = 2LL * a.geo.nblk;
  defer_identity_kernel<T, NELEM><<<(unsigned)((ntiles * 32 + 255) / 256), 256, 0, a.stream>>>((cplx_t<T>*)acc, ntiles);
  return cudaGetLastError();
}

// flush = true: apply the accumulated rotations to the temporal links; then (always) A <- 1
cudaError_t launch_defer(const KernelArgs& a, void* acc, bool flush) {
  if (a.prec == 0) return a.storage == 18 ? defer_T<double, 9>(a, acc, flush) : defer_T<double, 6>(a, acc, flush);
  return a.storage == 18 ? defer_T<float, 9>(a, acc, flush) : defer_T<float, 6>(a, acc, flush);
}

cudaError_t launch_halfsweep_slab(const KernelArgs& a, int parity, double omega, int cb_begin, int cb_end,
                                  int cb2_begin, int cb2_end, void* top_out, void* ret_out) {
  GF_DISPATCH(halfsweep_slab_T, a, parity, omega, cb_begin, cb_end, cb2_begin, cb2_end, top_out, ret_out);
}

cudaError_t launch_halfsweep_slab_fused(const KernelArgs& a, int parity, double omega, void* top_out, void* ret_out,
                                        unsigned* counter, unsigned* flag_up, unsigned* flag_down, const void* top_in_src) {
  GF_DISPATCH(halfsweep_slab_fused_T, a, parity, omega, top_out, ret_out, counter, flag_up, flag_down, top_in_src);
}

// ---- top time slice of a slab <-> message buffer (ghost layout of one parity) ------------------------------------------
// One thread per site of the slice: U_t(x) of the `parity` sites of slice n_t - 1, element by element (both sides are
// 32-lane runs of one element, so reads and writes are full sectors).
template <class T, int NELEM, bool PACK>
__global__ void __launch_bounds__(256) slab_top_kernel(cplx_t<T>* __restrict__ links, Geo g, int parity,
                                                       cplx_t<T>* __restrict__ buf) {
  using C = cplx_t<T>;
  const int cb3 = blockIdx.x * 256 + threadIdx.x;
  if (cb3 >= g.s3) return;
  C* l = links + link_offset<NELEM>(g, parity, g.s3 * (g.n[3] - 1) + cb3, 3);
  C* b = buf + ((size_t)(cb3 >> 5) * NELEM) * 32 + (cb3 & 31);
#pragma unroll
  for (int e = 0; e < NELEM; ++e) {
    if (PACK) b[e * 32] = l[e * 32];
    else l[e * 32] = b[e * 32];
  }
}

template <class T, int NELEM>
static cudaError_t slab_top_T(const KernelArgs& a, int parity, void* buf, bool pack) {
  const unsigned blocks = (unsigned)((a.geo.s3 + 255) / 256);
  if (pack) slab_top_kernel<T, NELEM, true><<<blocks, 256, 0, a.stream>>>((cplx_t<T>*)a.links, a.geo, parity, (cplx_t<T>*)buf);
  else slab_top_kernel<T, NELEM, false><<<blocks, 256, 0, a.stream>>>((cplx_t<T>*)a.links, a.geo, parity, (cplx_t<T>*)buf);
  return cudaGetLastError();
}

cudaError_t launch_slab_top(const KernelArgs& a, int parity, void* buf, bool pack) {
  if (a.prec == 0) return a.storage == 18 ? slab_top_T<double, 9>(a, parity, buf, pack) : slab_top_T<double, 6>(a, parity, buf, pack);
  return a.storage == 18 ? slab_top_T<float, 9>(a, parity, buf, pack) : slab_top_T<float, 6>(a, parity, buf, pack);
}

bool halfsweep_can_fuse_theta(const KernelArgs& a) {
  return (a.variant == 0 || a.variant == 3 || a.variant == 4 || a.variant == 5 || a.variant == 6) && a.series == 0;
}
int halfsweep_max_qblocks(const Geo& g) { return (g.vh + 31) / 32; }

// ======================================================================================================================
// F and theta
// ======================================================================================================================
// One thread per site.  Per site: f = sum_{nu<ND} Re Tr [U_nu(x) + U_nu(x-nu)] (= Re Tr K(x));
// A = sum_{nu<ND} [U_nu(x-nu) - U_nu(x)];  Delta = (A - A^dag) - (1/3) Tr(A - A^dag);  q = sum_ij |Delta_ij|^2
// (eqs. 1.1-1.3, readings A1, A2).  Every link touches exactly one site of each parity, so the sum of f over the sites
// of ONE parity is the sum of Re Tr U over all links: F needs the even sites only, and a pass over the sites of one
// parity reads every link exactly once.
// Grid: blocks_per_parity * nparity blocks; the first blocks_per_parity blocks take parity `parity0`, the rest the other.
// Block partials by warp shuffles (FP64), one double2 per block; a single-block second stage adds them in index order.
constexpr int MEASURE_THREADS = 256;
constexpr int MEASURE_SINGLE_LAUNCH_MAX_BLOCKS = 4096;

// what the last block of measure_partial_kernel needs to finish the reduction
struct MeasureTail {
  unsigned* counter;        // zero before the launch; left at zero
  int nf;                   // f is summed over the first nf partials only (the even sites: every link once)
  const double* qpartials;  // nq theta terms left by the last odd half-sweep (may be 0)
  int nq;
  double norm_f, norm_q;
  double* result;           // F, theta
};

// thread i adds partials i, i+THREADS, ... in order; fixed tree afterwards (deterministic).  One block of THREADS.
template <int THREADS>
__device__ __forceinline__ void measure_tail(const double2* __restrict__ partials, int n, const MeasureTail& tail) {
  double f = 0.0, q = 0.0;
  for (int i = threadIdx.x; i < n; i += THREADS) {
    const double2 p = __ldcg(partials + i);
    if (i < tail.nf) f += p.x;
    q += p.y;
  }
  for (int i = threadIdx.x; i < tail.nq; i += THREADS) q += __ldcg(tail.qpartials + i);
  __syncthreads();  // block_sum2's shared scratch may still be in use by the caller's first stage
  block_sum2<THREADS>(f, q);
  if (threadIdx.x == 0) {
    tail.result[0] = f * tail.norm_f;
    tail.result[1] = q * tail.norm_q;
  }
}

// the two per-site terms: f = Re Tr sum_nu [U_nu(x) + U_nu(x-nu)], q = sum_ij |Delta_ij(x)|^2
template <class T, int NELEM, int ND, bool SLAB>
__device__ __forceinline__ void site_f_q(const cplx_t<T>* __restrict__ links, const Geo& g, int parity, int cb,
                                         const SlabView& sv, double& f, double& q) {
  using C = cplx_t<T>;
  const Site s = site_of(g, parity, cb);
  const C* fwd = links + link_offset<NELEM>(g, parity, cb, 0);
  C A[9];
#pragma unroll
  for (int e = 0; e < 9; ++e) A[e] = mk<T>(T(0), T(0));
  T tr = T(0);
#pragma unroll
  for (int nu = 0; nu < ND; ++nu) {
    C u[9];
    const C* down = links + link_offset<NELEM>(g, parity ^ 1, cb_down(g, s, cb, nu), nu);
    if (SLAB && nu == 3 && cb < g.s3) down = ghost_link<T, NELEM, C>(sv, parity ^ 1, cb);
    load_link<NELEM, true>(down, u);
#pragma unroll
    for (int e = 0; e < 9; ++e) { A[e].x += u[e].x; A[e].y += u[e].y; }
    tr += u[0].x + u[4].x + u[8].x;
    load_link<NELEM, true>(fwd + nu * NELEM * 32, u);
#pragma unroll
    for (int e = 0; e < 9; ++e) { A[e].x -= u[e].x; A[e].y -= u[e].y; }
    tr += u[0].x + u[4].x + u[8].x;
  }
  f = (double)tr;
  q = (double)delta_norm2<T>(A);
}

template <class T, int NELEM, int ND, bool SLAB>
__global__ void __launch_bounds__(MEASURE_THREADS) measure_partial_kernel(const cplx_t<T>* __restrict__ links, Geo g,
                                                                          int blocks_per_parity,
                                                                          double2* __restrict__ partials, MeasureTail tail,
                                                                          SlabView sv) {
  const int parity = blockIdx.x >= blocks_per_parity;
  const int cb = (blockIdx.x - parity * blocks_per_parity) * MEASURE_THREADS + threadIdx.x;
  double f = 0.0, q = 0.0;
  if (cb < g.vh) site_f_q<T, NELEM, ND, SLAB>(links, g, parity, cb, sv, f, q);
  block_sum2<MEASURE_THREADS>(f, q);
  if (tail.counter == nullptr) {  // large grids: the second stage is its own small launch (see measure_T)
    if (threadIdx.x == 0) partials[blockIdx.x] = make_double2(f, q);
    return;
  }
  // Second stage in the same launch: the block that finishes last adds the partials in index order, so the result
  // does not depend on which block that is.
  __shared__ bool last;
  if (threadIdx.x == 0) {
    partials[blockIdx.x] = make_double2(f, q);
    __threadfence();
    last = atomicAdd(tail.counter, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  measure_tail<MEASURE_THREADS>(partials, (int)gridDim.x, tail);
  if (threadIdx.x == 0) *tail.counter = 0u;  // ready for the next launch on this stream
}

__global__ void __launch_bounds__(1024) measure_tail_kernel(const double2* __restrict__ partials, int n, MeasureTail tail) {
  measure_tail<1024>(partials, n, tail);
}

int measure_launches(const Geo& g, int nq) {
  const int bpp = ((g.vh + MEASURE_THREADS - 1) / MEASURE_THREADS);
  return (nq > 0 ? bpp : 2 * bpp) <= MEASURE_SINGLE_LAUNCH_MAX_BLOCKS ? 1 : 2;
}
int measure_num_partials(const Geo& g) { return 2 * ((g.vh + MEASURE_THREADS - 1) / MEASURE_THREADS); }

// nq > 0: the odd sites' theta terms are already in a.qpartials[0..nq): visit the even sites only.
template <class T, int NELEM, int ND>
static cudaError_t measure_T(const KernelArgs& a, int nq) {
  const int bpp = measure_num_partials(a.geo) / 2;
  const int nblk = nq > 0 ? bpp : 2 * bpp;
  const double V = 2.0 * (double)a.geo.vh;
  // Small lattices are latency bound: one launch, the last block to finish does the second stage.  On large grids
  // 65536 blocks queueing on one completion counter cost more (cfg4: +0.13 ms) than a second small launch.
  const bool single = nblk <= MEASURE_SINGLE_LAUNCH_MAX_BLOCKS;
  const MeasureTail tail{single ? (unsigned*)a.counter : nullptr, bpp, (const double*)a.qpartials, nq,
                         1.0 / (ND * 3.0 * V), 1.0 / (3.0 * V), (double*)a.result};
  if (a.slab.ghost)
    measure_partial_kernel<T, NELEM, ND, true><<<nblk, MEASURE_THREADS, 0, a.stream>>>(
        (const cplx_t<T>*)a.links, a.geo, bpp, (double2*)a.partials, tail, a.slab);
  else
    measure_partial_kernel<T, NELEM, ND, false><<<nblk, MEASURE_THREADS, 0, a.stream>>>(
        (const cplx_t<T>*)a.links, a.geo, bpp, (double2*)a.partials, tail, SlabView{});
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess || single) return e;
  measure_tail_kernel<<<1, 1024, 0, a.stream>>>((const double2*)a.partials, nblk, tail);
  return cudaGetLastError();
}

// second stage alone: F = norm_f * sum of the first nf partials' f, theta = norm_q * sum of all n partials' q -> a.result
cudaError_t launch_measure_tail(const KernelArgs& a, int n, int nf, double norm_f, double norm_q) {
  const MeasureTail tail{nullptr, nf, nullptr, 0, norm_f, norm_q, (double*)a.result};
  measure_tail_kernel<<<1, 1024, 0, a.stream>>>((const double2*)a.partials, n, tail);
  return cudaGetLastError();
}

cudaError_t launch_measure(const KernelArgs& a, int nq) {
  if (a.storage == 8) {
    if (a.prec == 0) return a.gauge == 1 ? measure_T<double, 4, 3>(a, nq) : measure_T<double, 4, 4>(a, nq);
    return a.gauge == 1 ? measure_T<float, 4, 3>(a, nq) : measure_T<float, 4, 4>(a, nq);
  }
  GF_DISPATCH(measure_T, a, nq);
}

// ---- per-time-slice F_t, theta_t (Coulomb gauge, gf_measure_slices / gf_fix_slices; reading A22) -------------------------
// Block (chunk, 2 t + parity): 256 consecutive checkerboard sites of one parity of slice t.  In Coulomb gauge the even
// sites of a slice see every spatial link of the slice once, so F_t needs the parity-0 blocks only.
template <class T, int NELEM>
__global__ void __launch_bounds__(MEASURE_THREADS) measure_slices_kernel(const cplx_t<T>* __restrict__ links, Geo g,
                                                                         double2* __restrict__ partials) {
  const int t = blockIdx.y >> 1, parity = blockIdx.y & 1;
  const int i = blockIdx.x * MEASURE_THREADS + threadIdx.x;
  double f = 0.0, q = 0.0;
  if (i < g.s3) site_f_q<T, NELEM, 3, false>(links, g, parity, t * g.s3 + i, SlabView{}, f, q);
  block_sum2<MEASURE_THREADS>(f, q);
  if (threadIdx.x == 0) partials[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = make_double2(f, q);
}

// one block per slice: its 2 * nchunk partials added in index order -> out[t] = F_t, out[nt + t] = theta_t
__global__ void __launch_bounds__(MEASURE_THREADS) measure_slices_tail_kernel(const double2* __restrict__ partials,
                                                                              int nchunk, int nt, double norm_f,
                                                                              double norm_q, double* __restrict__ out) {
  const int t = blockIdx.x;
  double f = 0.0, q = 0.0;
  for (int i = threadIdx.x; i < 2 * nchunk; i += MEASURE_THREADS) {
    const double2 p = partials[(size_t)t * 2 * nchunk + i];
    if (i < nchunk) f += p.x;  // parity 0
    q += p.y;
  }
  block_sum2<MEASURE_THREADS>(f, q);
  if (threadIdx.x == 0) { out[t] = f * norm_f; out[nt + t] = q * norm_q; }
}

int measure_slices_num_partials(const Geo& g) { return 2 * g.n[3] * ((g.s3 + MEASURE_THREADS - 1) / MEASURE_THREADS); }

template <class T, int NELEM>
static cudaError_t measure_slices_T(const KernelArgs& a, double* out) {
  const Geo& g = a.geo;
  const int nchunk = (g.s3 + MEASURE_THREADS - 1) / MEASURE_THREADS;
  measure_slices_kernel<T, NELEM><<<dim3(nchunk, 2 * g.n[3]), MEASURE_THREADS, 0, a.stream>>>(
      (const cplx_t<T>*)a.links, g, (double2*)a.partials);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  const double V3 = 2.0 * (double)g.s3;
  measure_slices_tail_kernel<<<g.n[3], MEASURE_THREADS, 0, a.stream>>>((const double2*)a.partials, nchunk, g.n[3],
                                                                      1.0 / (3.0 * 3.0 * V3), 1.0 / (3.0 * V3), out);
  return cudaGetLastError();
}

cudaError_t launch_measure_slices(const KernelArgs& a, double* out) {
  if (a.prec == 0) return a.storage == 18 ? measure_slices_T<double, 9>(a, out) : measure_slices_T<double, 6>(a, out);
  return a.storage == 18 ? measure_slices_T<float, 9>(a, out) : measure_slices_T<float, 6>(a, out);
}

// ======================================================================================================================
// reunitarisation
// ======================================================================================================================
// One thread per stored link: the internal array is a sequence of (block, mu) tiles of NELEM*32 complex numbers.
template <class T, int NELEM>
__global__ void __launch_bounds__(256) reunit_kernel(cplx_t<T>* __restrict__ links, long long ntiles, int nblk, int vh) {
  using C = cplx_t<T>;
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long tile = tid >> 5;  // (parity * nblk + blk) * 4 + mu
  if (tile >= ntiles) return;
  if (((tile >> 2) % nblk) * 32 + (tid & 31) >= vh) return;  // padding lanes of a parity's last block hold no link
  C* p = links + (size_t)tile * NELEM * 32 + (tid & 31);
  C u[9];
  load_link<NELEM, false>(p, u);
  reunitarize<T>(u);
  store_link<NELEM>(p, u);
}

template <class T, int NELEM>
static cudaError_t reunit_T(const KernelArgs& a) {
  const long long ntiles = 2LL * a.geo.nblk * 4;
  const unsigned blocks = (unsigned)((ntiles * 32 + 255) / 256);
  reunit_kernel<T, NELEM><<<blocks, 256, 0, a.stream>>>((cplx_t<T>*)a.links, ntiles, a.geo.nblk, a.geo.vh);
  return cudaGetLastError();
}

// 8-real storage: has any store since the last call seen a link outside the validity domain (N < Domain8::n_min)?
// Reads and clears the flag of the current device; the caller has synchronised the stream.
cudaError_t take_domain_flag(unsigned* out) {
  cudaError_t e = cudaMemcpyFromSymbol(out, gf_domain_flag, sizeof(unsigned));
  if (e == cudaSuccess && *out) {
    const unsigned zero = 0;
    e = cudaMemcpyToSymbol(gf_domain_flag, &zero, sizeof(unsigned));
  }
  return e;
}

// Forget, in stream order, what earlier stores reported: a new field is about to be loaded (gf_set_links[_host]).
cudaError_t clear_domain_flag(cudaStream_t stream) {
  void* p = nullptr;
  cudaError_t e = cudaGetSymbolAddress(&p, gf_domain_flag);
  return e == cudaSuccess ? cudaMemsetAsync(p, 0, sizeof(unsigned), stream) : e;
}

cudaError_t launch_reunit(const KernelArgs& a) {
  if (a.storage == 8) return a.prec == 0 ? reunit_T<double, 4>(a) : reunit_T<float, 4>(a);
  if (a.prec == 0) return a.storage == 18 ? reunit_T<double, 9>(a) : reunit_T<double, 6>(a);
  return a.storage == 18 ? reunit_T<float, 9>(a) : reunit_T<float, 6>(a);
}

}  // namespace gf
