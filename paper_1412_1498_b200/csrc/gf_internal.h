// gf_internal.h — what gf_api.cu needs to know about the kernels in gf_kernels.cu (host-side declarations only).
#pragma once
#include <cuda_runtime.h>

#include "gf_device.cuh"

namespace gf {

// A context that is one T-slab of a taller lattice (gf_slab_*): see ghost_link in gf_kernels.cu for the buffer layout.
struct SlabView {
  void* ghost;           // two parities of nblk3 tiles; nullptr: the lattice is periodic in t (not a slab)
  int nblk3;             // ceil(s3 / 32): tiles per parity of one time slice
  int cb_begin, cb_end;  // checkerboard range of a half-sweep launch ...
  int nblocks0;          // ... covered by the first nblocks0 blocks; the remaining blocks cover
  int cb2_begin, cb2_end;  //     a second range (border launch: bottom and top slice in one grid)
  void* top_out;         // non-null: top-slice sites also leave their updated U_t(x) here (message layout)
  void* ret_out;         // non-null: t = 0 sites also leave their updated U_t(x - t) here (message layout, one parity)
  // fused launch (border and interior in one grid): a third range behind the two border ranges, and the signal the last
  // of the first sig_blocks blocks (the border) raises in both neighbours' flag words once all of them have stored
  int nblocks1;            // blocks of the second range
  int cb3_begin, cb3_end;  // third range (the interior); empty if cb3_end <= cb3_begin
  int sig_blocks;          // 0: no signal
  unsigned* sig_counter;   // zero between launches
  unsigned* sig_flag[2];   // the neighbours' arrival counters: each gets +1 (system-scope atomic)
  // non-null: the top-slice sites take U_t(x) from this message buffer (what the upper neighbour's last half-sweep
  // returned) instead of from the field - the unpack kernel between two half-sweeps is then not needed
  const void* top_in_src;
};

struct KernelArgs {
  void* links;     // internal-layout link field (device)
  void* partials;  // double2 per measure block (device)
  void* qpartials; // double per half-sweep block: theta terms left by a fused odd half-sweep (device)
  void* result;    // 2 doubles: F, theta (device pointer of mapped pinned host memory)
  void* counter;   // one unsigned, zero between launches: block-completion count of the measure kernel (device)
  Geo geo;
  cudaStream_t stream;
  int prec;     // 0 = FP64, 1 = FP32
  int storage;  // 18 or 12
  int gauge;    // 0 = Landau, 1 = Coulomb
  int variant;  // half-sweep kernel variant (GF_OPT_SWEEP_VARIANT)
  int block_threads;
  int series;   // GF_OPT_OVR_SERIES: 0 = exact g^omega, N > 0 = truncated binomial series of order N
  int ncolors;  // 3 (everything above), or 2 / 4: the general SU(N) kernels of gf_sun.cu, N^2 complex numbers per link
  SlabView slab;
};

// canonical <-> internal for the lexicographic site range [lex_begin, lex_end).  If chunk_base is non-null the canonical
// data of that range starts at chunk_base (a staging buffer); otherwise `canon` is the full canonical array.
cudaError_t launch_reorder(const KernelArgs& a, bool in, void* canon, long long lex_begin, long long lex_end,
                           const void* chunk_base);
// fuse_theta: the launch also leaves the updated sites' theta terms in a.qpartials[0..*qblocks) (only kernels for which
// halfsweep_can_fuse_theta(a) holds; *qblocks = 0 otherwise)
cudaError_t launch_halfsweep(const KernelArgs& a, int parity, double omega, bool fuse_theta, int* qblocks);
bool halfsweep_can_fuse_theta(const KernelArgs& a);
// T-slab: the sites [cb_begin, cb_end) and [cb2_begin, cb2_end) of `parity` in one launch (staged kernel; t = 0 sites
// use a.slab.ghost; with top_out the top-slice sites also write their updated U_t(x) there)
cudaError_t launch_halfsweep_slab(const KernelArgs& a, int parity, double omega, int cb_begin, int cb_end,
                                  int cb2_begin, int cb2_end, void* top_out, void* ret_out);
// The whole half-sweep of a slab in ONE launch: bottom slice, top slice (both deliver their halo messages to top_out /
// ret_out), then the interior; the border blocks come first in the grid, and the last of them to finish adds 1 to the
// two neighbours' arrival counters (system-scope atomics), so the neighbours can go on while the interior is still being updated.
cudaError_t launch_halfsweep_slab_fused(const KernelArgs& a, int parity, double omega, void* top_out, void* ret_out,
                                        unsigned* counter, unsigned* flag_up, unsigned* flag_down, const void* top_in_src);
// U_t of the `parity` sites of the top time slice -> buf (pack) or buf -> those links (unpack); buf: one parity, ghost layout
cudaError_t launch_slab_top(const KernelArgs& a, int parity, void* buf, bool pack);
int halfsweep_max_qblocks(const Geo& g);
// 1 kernel launch on small grids (the last block to finish does the second stage), else 2.  nq > 0: a.qpartials[0..nq) hold the odd sites' theta terms of the links as they stand, so only
// the even sites are visited (every link read once); nq = 0: all sites are visited.
cudaError_t launch_measure(const KernelArgs& a, int nq);
cudaError_t launch_reunit(const KernelArgs& a);
cudaError_t take_domain_flag(unsigned* out);  // 8-real storage: a stored link had N below the validity threshold
cudaError_t clear_domain_flag(cudaStream_t stream);  // before a new field is loaded: reports concern the current field only
int measure_num_partials(const Geo& g);
// Coulomb gauge with a stop test per time slice (gf_measure_slices / gf_fix_slices)
int measure_slices_num_partials(const Geo& g);  // double2 entries launch_measure_slices needs in a.partials
cudaError_t launch_measure_slices(const KernelArgs& a, double* out);  // out[t] = F_t, out[nt + t] = theta_t (device-visible)
cudaError_t launch_halfsweep_masked(const KernelArgs& a, int parity, double omega, const unsigned char* active);
// Coulomb gauge with deferred temporal links (gf_defer_*): acc = one matrix per site, layout of one link direction
cudaError_t launch_halfsweep_defer(const KernelArgs& a, int parity, double omega, void* acc);
cudaError_t launch_defer(const KernelArgs& a, void* acc, bool flush);  // flush: U_t <- A U_t A(x+t)^dag; then A <- 1
int measure_launches(const Geo& g, int nq);  // kernels launch_measure issues: 1 (small grids) or 2
cudaError_t launch_measure_tail(const KernelArgs& a, int n, int nf, double norm_f, double norm_q);

// ---- general SU(N) (gf_sun.cu): N = 2, 4, full storage ---------------------------------------------------
bool sun_supported(int ncolors);
cudaError_t launch_reorder_sun(const KernelArgs& a, bool in, void* canon, long long lex_begin, long long lex_end,
                               const void* chunk_base);
cudaError_t launch_halfsweep_sun(const KernelArgs& a, int parity, double omega);
cudaError_t launch_measure_sun(const KernelArgs& a);  // 2 launches
cudaError_t launch_reunit_sun(const KernelArgs& a);

// ---- Algorithm 2 (gf_fftsd.cu): steepest descent with Fourier acceleration ------------------------------------------------
struct FftPlans;  // the cuFFT plans of one context
// Plans are created with cuFFT's own allocation switched off; *work = bytes of work area they need.  These return
// nullptr on success or a static error text.
const char* fft_plans_create(FftPlans** out, const Geo& g, int prec, int gauge, cudaStream_t stream, size_t* work);
const char* fft_plans_set_work(FftPlans* p, void* work);
void fft_plans_destroy(FftPlans* p);
// in-place forward / backward (unnormalised) transform of the four packed fields at w; *launches += cuFFT executions
// with_t = false: only the 3-D transform of every time slice (the t direction is done by launch_sd_tline)
const char* fft_exec(FftPlans* p, const Geo& g, int prec, void* w, bool forward, bool with_t, int* launches);
bool sd_tline_supported(const Geo& g);
// forward transform along t, Fourier factor, inverse transform along t in one pass (Landau, n_t a power of two)
cudaError_t launch_sd_tline(const KernelArgs& a, void* w, const double* table, double alpha);
// hand-written transforms (gf_fft.cu): forward, Fourier factor, inverse in 5 (Landau) / 3 (Coulomb) passes
bool own_fft_supported(const Geo& g, int gauge, int prec);
size_t own_fft_table_entries(const Geo& g);  // doubles: per axis the position-ordered p^2 and the twiddles
cudaError_t launch_own_fft_tables(const KernelArgs& a, double* table);
cudaError_t launch_own_fft_update(const KernelArgs& a, void* w, const double* table, double alpha, int* launches);
size_t sd_table_entries(const Geo& g);  // doubles in the 4 sin^2(pi k/n) table
int sd_num_partials(const Geo& g);      // <= measure_num_partials(g): a.partials is shared
cudaError_t launch_sd_table(const KernelArgs& a, double* table);
cudaError_t launch_sd_delta(const KernelArgs& a, void* w);  // packed Delta(x) -> w, F/theta block partials -> a.partials
cudaError_t launch_sd_final(const KernelArgs& a);           // a.partials -> a.result (F, theta)
cudaError_t launch_sd_filter(const KernelArgs& a, void* w, const double* table, double alpha, bool accelerate);
cudaError_t launch_sd_rotate(const KernelArgs& a, const void* w);

}  // namespace gf
