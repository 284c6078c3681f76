// gf_api.cu — the C ABI of include/gf.h: context, argument checking, the Algorithm 1 driver loop.
// Every step of the hot path runs in the kernels of gf_kernels.cu; this file only sequences launches.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/gf.h"
#include "gf_internal.h"

using namespace gf;

namespace {
constexpr size_t ALIGN = 256;
constexpr size_t STAGING_BYTES = 64u << 20;  // each of the two staging buffers used by the *_host calls
size_t align_up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

struct Sizes {
  size_t links, partials, qpartials, result, staging, total;
};

bool valid_lattice(int nx, int ny, int nz, int nt, int* err) {
  const int n[4] = {nx, ny, nz, nt};
  long long V = 1;
  for (int d = 0; d < 4; ++d) {
    if (n[d] < 2 || (n[d] & 1)) { *err = GF_EODD; return false; }
    V *= n[d];
    if (V >= (1LL << 31)) { *err = GF_EUNSUPPORTED; return false; }
  }
  return true;
}

Geo make_geo(int nx, int ny, int nz, int nt) {
  Geo g;
  g.n[0] = nx; g.n[1] = ny; g.n[2] = nz; g.n[3] = nt;
  g.nh0 = nx / 2;
  g.vh = (int)((long long)nx * ny * nz * nt / 2);
  g.nblk = (g.vh + 31) / 32;
  g.s1 = g.nh0; g.s2 = g.nh0 * ny; g.s3 = g.nh0 * ny * nz;
  return g;
}

// storage = reals per stored link: 18 / 12 / 8 for SU(3), 2 N^2 for the general SU(N) kernels
Sizes sizes_of(const Geo& g, int prec, int storage) {
  Sizes s;
  const size_t csize = prec == GF_FP64 ? 16 : 8;
  s.links = align_up((size_t)2 * g.nblk * 4 * (storage / 2) * 32 * csize);
  const int np = measure_num_partials(g) > measure_slices_num_partials(g) ? measure_num_partials(g) : measure_slices_num_partials(g);
  s.partials = align_up((size_t)np * sizeof(double2));
  s.qpartials = align_up((size_t)halfsweep_max_qblocks(g) * sizeof(double));
  s.result = align_up(2 * sizeof(double));
  s.staging = align_up(STAGING_BYTES);
  s.total = s.links + s.partials + s.qpartials + s.result + 2 * s.staging;
  return s;
}
}  // namespace

struct gf_ctx {
  KernelArgs k;
  Sizes sz;
  int device;                 // the CUDA device that was current at gf_create: every entry point runs on it
  char* staging[2];
  cudaStream_t copy_stream;   // host <-> staging copies of the *_host calls, beside the reorder kernels on k.stream
  cudaEvent_t staging_free[2];  // staging[b] may be overwritten (its last reader has finished)
  cudaEvent_t staging_full[2];  // staging[b] holds a chunk (its last writer has finished)
  double* host_result;  // pinned and mapped, 2 doubles: the reduction kernels write F, theta straight into it
  char* defer_acc;      // gf_defer_attach: the accumulated rotation A(x) of every site, or null
  bool defer_dirty;     // sweeps have run since the last flush
  double* host_slices;  // pinned and mapped, 2 n_t doubles (F_t, theta_t), allocated by the first gf_measure_slices
  double* dev_slices;   // its device pointer
  int reunit_every;
  int fuse_measure;  // GF_OPT_FUSE_MEASURE
  int domain8_check;  // GF_OPT_DOMAIN8_CHECK
  int slab_force_flags;  // GF_OPT_SLAB_FORCE_FLAGS
  int qblocks;       // > 0: k.qpartials[0..qblocks) hold the odd sites' theta terms of the links as they stand
  long long sweeps_total;  // sweeps since the last gf_set_links (reunitarisation cadence)
  long long launches;
  std::vector<double> history;
  long long history_n;
  // Algorithm 2 (gf_fft_*): plans, and the caller's second workspace once attached
  FftPlans* fft;
  size_t fft_w_bytes, fft_table_bytes, fft_work_bytes;
  char* fft_w;        // four packed complex fields of V entries
  double* fft_table;  // 4 sin^2(pi k/n) per direction
  int fft_accelerate; // GF_OPT_FFT_ACCELERATE
  int fft_fused_t;    // GF_OPT_FFT_FUSED_T
  int fft_own;        // GF_OPT_FFT_OWN
  double* own_table;  // tables of the hand-written transforms (behind fft_table in the same workspace slot)
  // T-slab sharding (gf_slab_*): the caller's halo workspace once attached
  size_t halo_bytes;  // one message: U_t of one parity of one time slice
  char* top_out;      // packed top-slice links on their way to the upper neighbour's ghost buffer
  char* top_in;       // ghost links coming back from the upper neighbour
  char* fwd_target[2];  // gf_slab_set_targets: the upper neighbour's ghost[0], ghost[1] (peer-mapped), or null
  char* ret_target;     //                      the lower neighbour's top_in, or null
  char* ret_target_odd; // gf_slab_set_peer_targets: where the odd half-sweep's "ret" message goes (even: ret_target)
  bool alt_top_in;      // gf_slab_set_peer_targets: unpack_top(1-p) reads top_in (p = 0) or the top_out slot (p = 1)
  // gf_slab_set_peer_flags: stream-ordered synchronisation with the two neighbours (no host wait, no collective)
  unsigned* own_flags;     // [0] written by the upper neighbour, [1] by the lower one (device memory of this slab)
  unsigned* upper_flag;    // the upper neighbour's own_flags[1] (this process's or a CUDA-IPC mapping)
  unsigned* lower_flag;    // the lower neighbour's own_flags[0]
  unsigned epoch;          // last epoch signalled by stream memory operations (entry / refresh synchronisation)
  unsigned arrivals;       // the fused launches so far: what own_flags[3] (upper neighbour) and own_flags[4] (lower) must reach
  char err[256];
};

namespace {
// Makes the context's device current for the duration of an entry point (a caller may drive contexts on several GPUs
// from one thread) and puts the caller's device back afterwards.
struct DeviceGuard {
  int prev = -1;
  explicit DeviceGuard(const gf_ctx* c) {
    int cur = -1;
    if (c && cudaGetDevice(&cur) == cudaSuccess && cur != c->device && cudaSetDevice(c->device) == cudaSuccess) prev = cur;
  }
  ~DeviceGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};
#define GF_ENTER(c)              \
  if (!(c)) return GF_EINVAL;    \
  DeviceGuard gf_device_guard_(c)

int fail_cuda(gf_ctx* c, cudaError_t e, const char* where) {
  snprintf(c->err, sizeof(c->err), "%s: %s", where, cudaGetErrorString(e));
  return GF_ECUDA;
}
int fail(gf_ctx* c, int code, const char* msg) {
  if (c) snprintf(c->err, sizeof(c->err), "%s", msg);
  return code;
}
size_t elem_size(const gf_ctx* c) { return c->k.prec == GF_FP64 ? sizeof(double) : sizeof(float); }
bool is_sun(const gf_ctx* c) { return c->k.ncolors != 3; }  // the general SU(N) kernels (gf_sun.cu)
cudaError_t reorder(const gf_ctx* c, bool in, void* canon, long long lex_begin, long long lex_end, const void* chunk_base) {
  return is_sun(c) ? launch_reorder_sun(c->k, in, canon, lex_begin, lex_end, chunk_base)
                   : launch_reorder(c->k, in, canon, lex_begin, lex_end, chunk_base);
}
long long volume(const gf_ctx* c) { return 2LL * c->k.geo.vh; }
}  // namespace

extern "C" {

size_t gf_workspace_bytes(int nx, int ny, int nz, int nt, int prec, int storage) {
  int err;
  if (!valid_lattice(nx, ny, nz, nt, &err)) return 0;
  if ((prec != GF_FP64 && prec != GF_FP32) || (storage != 18 && storage != 12 && storage != 8)) return 0;
  return sizes_of(make_geo(nx, ny, nz, nt), prec, storage).total;
}

size_t gf_workspace_bytes_sun(int ncolors, int nx, int ny, int nz, int nt, int prec) {
  if (ncolors == 3) return gf_workspace_bytes(nx, ny, nz, nt, prec, 18);
  int err;
  if (!sun_supported(ncolors) || !valid_lattice(nx, ny, nz, nt, &err) || (prec != GF_FP64 && prec != GF_FP32)) return 0;
  return sizes_of(make_geo(nx, ny, nz, nt), prec, 2 * ncolors * ncolors).total;
}

static int create_ctx(gf_ctx** out, int ncolors, int nx, int ny, int nz, int nt, int gauge, int prec, int storage,
                      void* dev_workspace, size_t workspace_bytes, void* cuda_stream);

int gf_create(gf_ctx** out, int nx, int ny, int nz, int nt, int gauge, int prec, int storage, void* dev_workspace,
              size_t workspace_bytes, void* cuda_stream) {
  if (!out) return GF_EINVAL;
  *out = nullptr;
  if (storage != 18 && storage != 12 && storage != 8) return GF_EUNSUPPORTED;
  return create_ctx(out, 3, nx, ny, nz, nt, gauge, prec, storage, dev_workspace, workspace_bytes, cuda_stream);
}

int gf_create_sun(gf_ctx** out, int ncolors, int nx, int ny, int nz, int nt, int gauge, int prec, void* dev_workspace,
                  size_t workspace_bytes, void* cuda_stream) {
  if (!out) return GF_EINVAL;
  *out = nullptr;
  if (ncolors == 3) return create_ctx(out, 3, nx, ny, nz, nt, gauge, prec, 18, dev_workspace, workspace_bytes, cuda_stream);
  if (!sun_supported(ncolors)) return GF_EUNSUPPORTED;
  return create_ctx(out, ncolors, nx, ny, nz, nt, gauge, prec, 2 * ncolors * ncolors, dev_workspace, workspace_bytes,
                    cuda_stream);
}

static int create_ctx(gf_ctx** out, int ncolors, int nx, int ny, int nz, int nt, int gauge, int prec, int storage,
                      void* dev_workspace, size_t workspace_bytes, void* cuda_stream) {
  int err;
  if (!valid_lattice(nx, ny, nz, nt, &err)) return err;
  if (gauge != GF_LANDAU && gauge != GF_COULOMB) return GF_EUNSUPPORTED;
  if (prec != GF_FP64 && prec != GF_FP32) return GF_EUNSUPPORTED;
  if (!dev_workspace) return GF_EINVAL;
  const Geo g = make_geo(nx, ny, nz, nt);
  const Sizes sz = sizes_of(g, prec, storage);
  if (workspace_bytes < sz.total || ((uintptr_t)dev_workspace % ALIGN) != 0) return GF_ENOMEM;

  gf_ctx* c = new (std::nothrow) gf_ctx();
  if (!c) return GF_ENOMEM;
  c->k.geo = g;
  c->k.stream = (cudaStream_t)cuda_stream;
  c->k.prec = prec; c->k.storage = storage; c->k.gauge = gauge;
  c->k.variant = 0; c->k.block_threads = 0; c->k.series = 0;
  c->k.ncolors = ncolors;
  c->sz = sz;
  char* base = (char*)dev_workspace;
  c->k.links = base;
  c->k.partials = base + sz.links;
  c->k.qpartials = base + sz.links + sz.partials;
  c->k.result = base + sz.links + sz.partials + sz.qpartials;  // replaced by the mapped host pointer below
  c->k.counter = base + sz.links + sz.partials + sz.qpartials;  // the workspace's result slot holds the counter
  c->staging[0] = base + sz.links + sz.partials + sz.qpartials + sz.result;
  c->staging[1] = c->staging[0] + sz.staging;
  c->fuse_measure = 1; c->qblocks = 0; c->domain8_check = 1; c->slab_force_flags = 0;
  c->reunit_every = 0; c->sweeps_total = 0; c->launches = 0; c->history_n = 0;
  c->err[0] = 0;
  c->fft = nullptr; c->fft_w = nullptr; c->fft_table = nullptr; c->fft_accelerate = 1; c->fft_fused_t = 0; c->fft_own = 1; c->own_table = nullptr;
  c->fft_w_bytes = c->fft_table_bytes = c->fft_work_bytes = 0;
  c->k.slab = SlabView{};
  c->k.slab.nblk3 = (g.s3 + 31) / 32;
  c->halo_bytes = align_up((size_t)c->k.slab.nblk3 * (storage / 2) * 32 * (prec == GF_FP64 ? 16 : 8));
  c->top_out = c->top_in = nullptr;
  c->fwd_target[0] = c->fwd_target[1] = c->ret_target = c->ret_target_odd = nullptr;
  c->alt_top_in = false;
  c->own_flags = c->upper_flag = c->lower_flag = nullptr;
  c->epoch = 0;
  c->arrivals = 0;
  c->host_result = nullptr;
  c->host_slices = c->dev_slices = nullptr;
  c->defer_acc = nullptr; c->defer_dirty = false;
  c->staging_free[0] = c->staging_free[1] = c->staging_full[0] = c->staging_full[1] = nullptr;
  c->copy_stream = nullptr;
  cudaError_t e = cudaGetDevice(&c->device);
  if (e == cudaSuccess) e = cudaHostAlloc((void**)&c->host_result, 2 * sizeof(double), cudaHostAllocMapped);
  if (e == cudaSuccess) {  // zero-copy result: saves a 16-byte D2H copy per measurement (latency on small lattices)
    void* dev = nullptr;
    e = cudaHostGetDevicePointer(&dev, c->host_result, 0);
    if (e == cudaSuccess) c->k.result = dev;
  }
  for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
    e = cudaEventCreateWithFlags(&c->staging_free[i], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->staging_full[i], cudaEventDisableTiming);
  }
  if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking);
  // padding lanes of the last 32-site block must read as zeros
  if (e == cudaSuccess) e = cudaMemsetAsync(c->k.links, 0, sz.links, c->k.stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(c->k.counter, 0, sz.result, c->k.stream);
  if (e != cudaSuccess) {
    gf_destroy(c);
    return GF_ECUDA;
  }
  *out = c;
  return GF_OK;
}

void gf_destroy(gf_ctx* c) {
  if (!c) return;
  {
    DeviceGuard guard(c);
    if (c->host_result) cudaFreeHost(c->host_result);
    if (c->host_slices) cudaFreeHost(c->host_slices);
    fft_plans_destroy(c->fft);
    for (int i = 0; i < 2; ++i) {
      if (c->staging_free[i]) cudaEventDestroy(c->staging_free[i]);
      if (c->staging_full[i]) cudaEventDestroy(c->staging_full[i]);
    }
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
  }
  delete c;
}

// ---- Coulomb gauge, deferred temporal links (SURVEY.md A9 "cheaper alternative") ---------------------------------------
static size_t defer_bytes(const gf_ctx* c) {
  return align_up((size_t)2 * c->k.geo.nblk * (c->k.storage / 2) * 32 * (c->k.prec == GF_FP64 ? 16 : 8));
}
static int defer_flush(gf_ctx* c) {
  if (!c->defer_acc || !c->defer_dirty) return GF_OK;
  cudaError_t e = launch_defer(c->k, c->defer_acc, true);
  if (e != cudaSuccess) return fail_cuda(c, e, "gf_defer_flush");
  c->launches += 2;
  c->defer_dirty = false;
  return GF_OK;
}

size_t gf_defer_bytes(const gf_ctx* c) { return c ? defer_bytes(c) : 0; }

int gf_defer_attach(gf_ctx* c, void* dev_acc, size_t bytes) {
  GF_ENTER(c);
  if (c->k.gauge != GF_COULOMB || c->k.slab.ghost || c->k.storage == 8 || is_sun(c))
    return fail(c, GF_EUNSUPPORTED, "gf_defer_attach: Coulomb gauge on a whole lattice only, 18- or 12-real storage");
  if (!dev_acc) {  // detach: bring the temporal links up to date first
    int rc = defer_flush(c);
    if (rc == GF_OK) c->defer_acc = nullptr;
    return rc;
  }
  if (bytes < defer_bytes(c) || ((uintptr_t)dev_acc % ALIGN)) return fail(c, GF_ENOMEM, "gf_defer_attach: buffer too small or misaligned");
  int rc = defer_flush(c);
  if (rc != GF_OK) return rc;
  c->defer_acc = (char*)dev_acc;
  cudaError_t e = launch_defer(c->k, c->defer_acc, false);  // A = 1
  if (e != cudaSuccess) { c->defer_acc = nullptr; return fail_cuda(c, e, "gf_defer_attach"); }
  c->launches += 1;
  c->defer_dirty = false;
  return GF_OK;
}

int gf_defer_flush(gf_ctx* c) {
  GF_ENTER(c);
  return defer_flush(c);
}

int gf_set_links(gf_ctx* c, const void* dev_links) {
  GF_ENTER(c);
  if (!dev_links) return fail(c, GF_EINVAL, "gf_set_links: null links");
  // 8-real storage: what the field that is being replaced left in the validity-domain flag says nothing about this one
  cudaError_t e = c->k.storage == 8 && c->k.ncolors == 3 ? clear_domain_flag(c->k.stream) : cudaSuccess;
  if (e == cudaSuccess) e = reorder(c, true, const_cast<void*>(dev_links), 0, volume(c), nullptr);
  if (e == cudaSuccess && c->defer_acc && c->defer_dirty) e = launch_defer(c->k, c->defer_acc, false);  // A = 1
  if (e != cudaSuccess) return fail_cuda(c, e, "gf_set_links");
  c->launches += 1;
  c->sweeps_total = 0;
  c->qblocks = 0;
  c->defer_dirty = false;
  return GF_OK;
}

int gf_get_links(gf_ctx* c, void* dev_links_out) {
  GF_ENTER(c);
  if (!dev_links_out) return fail(c, GF_EINVAL, "gf_get_links: null output");
  int rc = defer_flush(c);
  if (rc != GF_OK) return rc;
  cudaError_t e = reorder(c, false, dev_links_out, 0, volume(c), nullptr);
  if (e != cudaSuccess) return fail_cuda(c, e, "gf_get_links");
  c->launches += 1;
  return GF_OK;
}

// Host <-> device through the two staging buffers: chunk i uses buffer i & 1.  The copies run on the context's own copy
// stream, the reorder kernels on the context's stream, ordered by events per buffer, so that (with pinned host
// memory) the copy of chunk i+1 runs beside the reorder kernel of chunk i.
// 8-real storage: a link stored since the last check had N = |a2|^2 + |a3|^2 below the validity threshold (reading A23)
static int domain8_check(gf_ctx* c, const char* who) {
  if (c->k.storage != 8 || c->k.ncolors != 3 || !c->domain8_check) return GF_OK;
  unsigned flag = 0;
  cudaError_t e = take_domain_flag(&flag);
  if (e != cudaSuccess) return fail_cuda(c, e, who);
  if (flag) {
    snprintf(c->err, sizeof(c->err), "%s: 8-real storage met a link with |a2|^2+|a3|^2 below %g: outside the domain of "
             "the parametrisation (nearly block-diagonal link); use storage 12 or 18", who, c->k.prec == GF_FP64 ? 1e-6 : 1e-3);
    return GF_ENUMERIC;
  }
  return GF_OK;
}

static int links_host(gf_ctx* c, void* host, bool in) {
  const size_t link_bytes = 2 * (size_t)c->k.ncolors * c->k.ncolors * elem_size(c);
  const long long sites_per_chunk = (long long)(STAGING_BYTES / (4 * link_bytes));
  const long long V = volume(c);
  cudaStream_t main = c->k.stream, copy = c->copy_stream;
  // everything enqueued on the context's stream so far (an earlier get/set, the sweeps) comes first
  cudaError_t e = cudaEventRecord(c->staging_free[0], main);
  if (e == cudaSuccess) e = cudaEventRecord(c->staging_free[1], main);
  int i = 0;
  for (long long s0 = 0; s0 < V && e == cudaSuccess; s0 += sites_per_chunk, ++i) {
    const long long s1 = s0 + sites_per_chunk < V ? s0 + sites_per_chunk : V;
    const size_t bytes = (size_t)(s1 - s0) * 4 * link_bytes;
    char* h = (char*)host + (size_t)s0 * 4 * link_bytes;
    const int b = i & 1;
    char* st = c->staging[b];
    if (in) {
      e = cudaStreamWaitEvent(copy, c->staging_free[b], 0);  // the reorder kernel of chunk i-2 has read it
      if (e == cudaSuccess) e = cudaMemcpyAsync(st, h, bytes, cudaMemcpyHostToDevice, copy);
      if (e == cudaSuccess) e = cudaEventRecord(c->staging_full[b], copy);
      if (e == cudaSuccess) e = cudaStreamWaitEvent(main, c->staging_full[b], 0);
      if (e == cudaSuccess) e = reorder(c, true, nullptr, s0, s1, st);
      if (e == cudaSuccess) e = cudaEventRecord(c->staging_free[b], main);
    } else {
      if (i >= 2) e = cudaStreamWaitEvent(main, c->staging_free[b], 0);  // the copy of chunk i-2 has left it
      if (e == cudaSuccess) e = reorder(c, false, nullptr, s0, s1, st);
      if (e == cudaSuccess) e = cudaEventRecord(c->staging_full[b], main);
      if (e == cudaSuccess) e = cudaStreamWaitEvent(copy, c->staging_full[b], 0);
      if (e == cudaSuccess) e = cudaMemcpyAsync(h, st, bytes, cudaMemcpyDeviceToHost, copy);
      if (e == cudaSuccess) e = cudaEventRecord(c->staging_free[b], copy);
    }
    c->launches += 1;
  }
  if (e == cudaSuccess) e = cudaStreamSynchronize(copy);
  if (e == cudaSuccess) e = cudaStreamSynchronize(main);
  if (e != cudaSuccess) return fail_cuda(c, e, in ? "gf_set_links_host" : "gf_get_links_host");
  return domain8_check(c, in ? "gf_set_links_host" : "gf_get_links_host");
}

int gf_set_links_host(gf_ctx* c, const void* host_links) {
  GF_ENTER(c);
  if (!host_links) return fail(c, GF_EINVAL, "gf_set_links_host: null links");
  if (c->k.storage == 8 && c->k.ncolors == 3) {
    cudaError_t e = clear_domain_flag(c->k.stream);
    if (e != cudaSuccess) return fail_cuda(c, e, "gf_set_links_host");
  }
  if (c->defer_acc && c->defer_dirty) {
    cudaError_t e = launch_defer(c->k, c->defer_acc, false);  // A = 1
    if (e != cudaSuccess) return fail_cuda(c, e, "gf_set_links_host");
    c->defer_dirty = false;
  }
  c->sweeps_total = 0;
  c->qblocks = 0;
  return links_host(c, const_cast<void*>(host_links), true);
}

int gf_get_links_host(gf_ctx* c, void* host_links_out) {
  GF_ENTER(c);
  if (!host_links_out) return fail(c, GF_EINVAL, "gf_get_links_host: null output");
  int rc = defer_flush(c);
  if (rc != GF_OK) return rc;
  return links_host(c, host_links_out, false);
}

int gf_reunitarize(gf_ctx* c) {
  GF_ENTER(c);
  int rc = defer_flush(c);  // every link is projected as it would stand after an in-place update
  if (rc != GF_OK) return rc;
  c->qblocks = 0;
  cudaError_t e = is_sun(c) ? launch_reunit_sun(c->k) : launch_reunit(c->k);
  if (e != cudaSuccess) return fail_cuda(c, e, "gf_reunitarize");
  c->launches += 1;
  return GF_OK;
}

int gf_set_reunit_every(gf_ctx* c, int k) {
  GF_ENTER(c);
  if (k < 0) return fail(c, GF_EINVAL, "gf_set_reunit_every: k < 0");
  c->reunit_every = k;
  return GF_OK;
}

int gf_set_option(gf_ctx* c, int key, int value) {
  GF_ENTER(c);
  if (is_sun(c)) return fail(c, GF_EUNSUPPORTED, "gf_set_option: no options on an SU(N != 3) context");
  switch (key) {
    case GF_OPT_SWEEP_VARIANT:
      if (value < 0 || value > 6) return fail(c, GF_EINVAL, "gf_set_option: bad variant");
      c->k.variant = value;
      return GF_OK;
    case GF_OPT_FUSE_MEASURE:
      c->fuse_measure = value != 0;
      if (!c->fuse_measure) c->qblocks = 0;
      return GF_OK;
    case GF_OPT_FFT_ACCELERATE:
      c->fft_accelerate = value != 0;
      return GF_OK;
    case GF_OPT_FFT_FUSED_T:
      c->fft_fused_t = value != 0;
      return GF_OK;
    case GF_OPT_FFT_OWN:
      c->fft_own = value != 0;
      return GF_OK;
    case GF_OPT_OVR_SERIES:
      if (value < 0 || value > 16) return fail(c, GF_EINVAL, "gf_set_option: series order outside 0..16");
      if (value > 0 && (c->k.slab.ghost || c->k.storage == 8))
        return fail(c, GF_EUNSUPPORTED, "gf_set_option: no series variant on a slab context or with 8-real storage");
      c->k.series = value;
      c->qblocks = 0;
      return GF_OK;
    case GF_OPT_DOMAIN8_CHECK:
      c->domain8_check = value != 0;
      return GF_OK;
    case GF_OPT_SLAB_FORCE_FLAGS:
      c->slab_force_flags = value != 0;
      return GF_OK;
    case GF_OPT_BLOCK_THREADS:
      if (value < 0 || value % 32 || value > 1024) return fail(c, GF_EINVAL, "gf_set_option: bad block size");
      c->k.block_threads = value;
      return GF_OK;
    default:
      return fail(c, GF_EINVAL, "gf_set_option: unknown key");
  }
}

int gf_ovr_sweep(gf_ctx* c, int n, double omega) {
  GF_ENTER(c);
  if (n < 0) return fail(c, GF_EINVAL, "gf_ovr_sweep: n < 0");
  if (!(omega >= 1.0 && omega < 2.0)) return fail(c, GF_EINVAL, "gf_ovr_sweep: omega outside [1,2)");
  if (c->k.slab.ghost) return fail(c, GF_EINVAL, "gf_ovr_sweep: the context is a slab, use gf_slab_halfsweep_*");
  if (n > 0) c->qblocks = 0;
  if (is_sun(c)) {  // general SU(N): the N(N-1)/2 subgroups per site, no fused theta terms
    for (int i = 0; i < n; ++i) {
      for (int parity = 0; parity < 2; ++parity) {  // even first
        cudaError_t e = launch_halfsweep_sun(c->k, parity, omega);
        if (e != cudaSuccess) return fail_cuda(c, e, "gf_ovr_sweep (SU(N))");
        c->launches += 1;
      }
      c->sweeps_total += 1;
      if (c->reunit_every > 0 && c->sweeps_total % c->reunit_every == 0) {
        int rc = gf_reunitarize(c);
        if (rc != GF_OK) return rc;
      }
    }
    return GF_OK;
  }
  if (c->defer_acc) {  // Coulomb gauge, temporal links deferred: 6 links + A(x) per site-update
    for (int i = 0; i < n; ++i) {
      for (int parity = 0; parity < 2; ++parity) {
        cudaError_t e = launch_halfsweep_defer(c->k, parity, omega, c->defer_acc);
        if (e != cudaSuccess) return fail_cuda(c, e, "gf_ovr_sweep (deferred temporal links)");
        c->launches += 1;
      }
      c->defer_dirty = true;
      c->sweeps_total += 1;
      if (c->reunit_every > 0 && c->sweeps_total % c->reunit_every == 0) {
        int rc = gf_reunitarize(c);
        if (rc != GF_OK) return rc;
      }
    }
    return GF_OK;
  }
  for (int i = 0; i < n; ++i) {
    for (int parity = 0; parity < 2; ++parity) {  // even first
      // the last odd half-sweep of the call also leaves the odd sites' theta terms for a gf_measure that may follow
      const bool fuse = c->fuse_measure && parity == 1 && i == n - 1 && halfsweep_can_fuse_theta(c->k);
      int qblocks = 0;
      cudaError_t e = launch_halfsweep(c->k, parity, omega, fuse, &qblocks);
      if (e != cudaSuccess) return fail_cuda(c, e, "gf_ovr_sweep");
      c->launches += 1;
      c->qblocks = qblocks;
    }
    c->sweeps_total += 1;
    if (c->reunit_every > 0 && c->sweeps_total % c->reunit_every == 0) {
      int rc = gf_reunitarize(c);
      if (rc != GF_OK) return rc;
    }
  }
  return GF_OK;
}

int gf_measure(gf_ctx* c, double* F, double* theta) {
  GF_ENTER(c);
  if (!F || !theta) return fail(c, GF_EINVAL, "gf_measure: null out-param");
  cudaError_t e = is_sun(c) ? launch_measure_sun(c->k) : launch_measure(c->k, c->qblocks);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->k.stream);
  if (e != cudaSuccess) return fail_cuda(c, e, "gf_measure");
  c->launches += is_sun(c) ? 2 : measure_launches(c->k.geo, c->qblocks);
  *F = c->host_result[0];
  *theta = c->host_result[1];
  if (int rc = domain8_check(c, "gf_measure"); rc != GF_OK) return rc;
  if (!std::isfinite(*F) || !std::isfinite(*theta)) return fail(c, GF_ENUMERIC, "gf_measure: non-finite F or theta");
  return GF_OK;
}

int gf_fix(gf_ctx* c, double omega, double eps, int max_sweeps, int check_every, int* sweeps_done) {
  GF_ENTER(c);
  if (!sweeps_done) return fail(c, GF_EINVAL, "gf_fix: null sweeps_done");
  if (check_every < 1 || max_sweeps < 0 || !(eps >= 0.0))
    return fail(c, GF_EINVAL, "gf_fix: need check_every >= 1, max_sweeps >= 0, eps >= 0");
  if (!(omega >= 1.0 && omega < 2.0)) return fail(c, GF_EINVAL, "gf_fix: omega outside [1,2)");
  if (c->k.slab.ghost) return fail(c, GF_EINVAL, "gf_fix: the context is a slab, the driver loop belongs to the caller");
  c->history.clear();
  c->history_n = 0;
  *sweeps_done = 0;
  int done = 0;
  double F, th;
  int rc = gf_measure(c, &F, &th);  // Algorithm 1 l.1
  auto record = [&]() {
    c->history.push_back((double)done);
    c->history.push_back(F);
    c->history.push_back(th);
    c->history_n += 1;
  };
  if (rc != GF_OK) return rc;
  record();
  while (!(th < eps) && done < max_sweeps) {  // Algorithm 1 l.2
    const int n = check_every < max_sweeps - done ? check_every : max_sweeps - done;
    rc = gf_ovr_sweep(c, n, omega);
    if (rc != GF_OK) return rc;
    done += n;
    *sweeps_done = done;
    rc = gf_measure(c, &F, &th);  // Algorithm 1 l.13
    if (rc != GF_OK) return rc;
    record();
  }
  return GF_OK;
}

// ---- Coulomb gauge, every time slice its own stop test (reading A22) -------------------------------------------------------
static int slices_check(gf_ctx* c, const char* who) {
  if (c->k.gauge != GF_COULOMB || c->k.slab.ghost || c->k.storage == 8 || is_sun(c)) return fail(c, GF_EUNSUPPORTED, who);
  if (!c->host_slices) {
    cudaError_t e = cudaHostAlloc((void**)&c->host_slices, 2 * sizeof(double) * c->k.geo.n[3], cudaHostAllocMapped);
    if (e == cudaSuccess) e = cudaHostGetDevicePointer((void**)&c->dev_slices, c->host_slices, 0);
    if (e != cudaSuccess) return fail_cuda(c, e, who);
  }
  return GF_OK;
}

int gf_measure_slices(gf_ctx* c, double* F_t, double* theta_t) {
  GF_ENTER(c);
  if (!F_t || !theta_t) return fail(c, GF_EINVAL, "gf_measure_slices: null out-param");
  int rc = slices_check(c, "gf_measure_slices: Coulomb gauge on a whole lattice only");
  if (rc != GF_OK) return rc;
  cudaError_t e = launch_measure_slices(c->k, c->dev_slices);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->k.stream);
  if (e != cudaSuccess) return fail_cuda(c, e, "gf_measure_slices");
  c->launches += 2;
  const int nt = c->k.geo.n[3];
  bool finite = true;
  for (int t = 0; t < nt; ++t) {
    F_t[t] = c->host_slices[t];
    theta_t[t] = c->host_slices[nt + t];
    finite = finite && std::isfinite(F_t[t]) && std::isfinite(theta_t[t]);
  }
  return finite ? GF_OK : fail(c, GF_ENUMERIC, "gf_measure_slices: non-finite F_t or theta_t");
}

int gf_fix_slices(gf_ctx* c, double omega, double eps, int max_sweeps, int check_every, int* sweeps_done,
                  int* slice_sweeps) {
  GF_ENTER(c);
  if (!sweeps_done) return fail(c, GF_EINVAL, "gf_fix_slices: null sweeps_done");
  if (check_every < 1 || max_sweeps < 0 || !(eps >= 0.0))
    return fail(c, GF_EINVAL, "gf_fix_slices: need check_every >= 1, max_sweeps >= 0, eps >= 0");
  if (!(omega >= 1.0 && omega < 2.0)) return fail(c, GF_EINVAL, "gf_fix_slices: omega outside [1,2)");
  int rc = slices_check(c, "gf_fix_slices: Coulomb gauge on a whole lattice only");
  if (rc != GF_OK) return rc;
  if (c->k.series > 0 || !(c->k.variant == 0 || c->k.variant == 3) || c->defer_acc)
    return fail(c, GF_EUNSUPPORTED, "gf_fix_slices: default sweep variant, exact power, no deferred temporal links");
  const int nt = c->k.geo.n[3];
  std::vector<double> Ft(nt), tht(nt);
  std::vector<unsigned char> active(nt);
  unsigned char* dev_active = (unsigned char*)c->k.qpartials;  // unused while no theta terms are fused
  c->history.clear();
  c->history_n = 0;
  c->qblocks = 0;
  *sweeps_done = 0;
  int done = 0;
  if (slice_sweeps)
    for (int t = 0; t < nt; ++t) slice_sweeps[t] = 0;
  auto look = [&](int* n_active) -> int {  // record (sweeps, mean F, max theta_t)
    int r = gf_measure_slices(c, Ft.data(), tht.data());
    if (r != GF_OK) return r;
    double F = 0.0, thmax = 0.0;
    *n_active = 0;
    for (int t = 0; t < nt; ++t) {
      F += Ft[t];
      thmax = tht[t] > thmax ? tht[t] : thmax;
      active[t] = !(tht[t] < eps);
      *n_active += active[t];
    }
    c->history.push_back((double)done);
    c->history.push_back(F / nt);
    c->history.push_back(thmax);
    c->history_n += 1;
    return GF_OK;
  };
  int n_active = 0;
  rc = look(&n_active);
  if (rc != GF_OK) return rc;
  while (n_active > 0 && done < max_sweeps) {
    const int n = check_every < max_sweeps - done ? check_every : max_sweeps - done;
    // pageable source: the copy is staged before the call returns, so `active` may change afterwards
    cudaError_t e = cudaMemcpyAsync(dev_active, active.data(), nt, cudaMemcpyHostToDevice, c->k.stream);
    for (int i = 0; i < n && e == cudaSuccess; ++i) {
      for (int parity = 0; parity < 2 && e == cudaSuccess; ++parity) {
        e = launch_halfsweep_masked(c->k, parity, omega, dev_active);
        c->launches += 1;
      }
      c->sweeps_total += 1;
      if (e == cudaSuccess && c->reunit_every > 0 && c->sweeps_total % c->reunit_every == 0) {
        rc = gf_reunitarize(c);
        if (rc != GF_OK) return rc;
      }
    }
    if (e != cudaSuccess) return fail_cuda(c, e, "gf_fix_slices");
    if (slice_sweeps)
      for (int t = 0; t < nt; ++t) slice_sweeps[t] += active[t] ? n : 0;
    done += n;
    *sweeps_done = done;
    rc = look(&n_active);
    if (rc != GF_OK) return rc;
  }
  return GF_OK;
}

int gf_get_history(gf_ctx* c, double* hist, int cap, int* n) {
  GF_ENTER(c);
  if (!n || (cap > 0 && !hist) || cap < 0) return fail(c, GF_EINVAL, "gf_get_history: bad arguments");
  *n = (int)c->history_n;
  const long long m = c->history_n < cap ? c->history_n : cap;
  if (m > 0) memcpy(hist, c->history.data(), (size_t)m * 3 * sizeof(double));
  return GF_OK;
}

// ---- Algorithm 2: steepest descent with Fourier acceleration -------------------------------------
static int fft_plan(gf_ctx* c) {
  if (c->k.storage == 8 && !is_sun(c)) return fail(c, GF_EUNSUPPORTED, "Algorithm 2 is not built for 8-real storage");
  if (is_sun(c)) return fail(c, GF_EUNSUPPORTED, "Algorithm 2 is built for SU(3) only");
  if (c->k.slab.ghost)  // no multi-GPU steepest descent (no distributed 4-D transform)
    return fail(c, GF_EUNSUPPORTED, "Algorithm 2 is not available on a slab context");
  if (c->fft) return GF_OK;
  size_t work = 0;
  const char* msg = fft_plans_create(&c->fft, c->k.geo, c->k.prec, c->k.gauge, c->k.stream, &work);
  if (msg) return fail(c, GF_ECUDA, msg);
  const size_t csize = c->k.prec == GF_FP64 ? 16 : 8;
  c->fft_w_bytes = align_up((size_t)4 * volume(c) * csize);
  c->fft_table_bytes = align_up(sd_table_entries(c->k.geo) * sizeof(double)) +
                       align_up(own_fft_table_entries(c->k.geo) * sizeof(double));
  c->fft_work_bytes = align_up(work);
  return GF_OK;
}

int gf_fft_workspace_bytes(gf_ctx* c, size_t* bytes) {
  GF_ENTER(c);
  if (!bytes) return fail(c, GF_EINVAL, "gf_fft_workspace_bytes: null out-param");
  int rc = fft_plan(c);
  if (rc != GF_OK) return rc;
  *bytes = c->fft_w_bytes + c->fft_table_bytes + c->fft_work_bytes;
  return GF_OK;
}

int gf_fft_attach(gf_ctx* c, void* dev_workspace, size_t workspace_bytes) {
  GF_ENTER(c);
  if (!dev_workspace) return fail(c, GF_EINVAL, "gf_fft_attach: null workspace");
  int rc = fft_plan(c);
  if (rc != GF_OK) return rc;
  if (workspace_bytes < c->fft_w_bytes + c->fft_table_bytes + c->fft_work_bytes || ((uintptr_t)dev_workspace % ALIGN))
    return fail(c, GF_ENOMEM, "gf_fft_attach: workspace too small or misaligned");
  c->fft_w = (char*)dev_workspace;
  c->fft_table = (double*)(c->fft_w + c->fft_w_bytes);
  const char* msg = fft_plans_set_work(c->fft, c->fft_w + c->fft_w_bytes + c->fft_table_bytes);
  if (msg) { c->fft_w = nullptr; return fail(c, GF_ECUDA, msg); }
  c->own_table = (double*)((char*)c->fft_table + align_up(sd_table_entries(c->k.geo) * sizeof(double)));
  cudaError_t e = launch_sd_table(c->k, c->fft_table);
  if (e == cudaSuccess && own_fft_supported(c->k.geo, c->k.gauge, c->k.prec)) e = launch_own_fft_tables(c->k, c->own_table);
  if (e != cudaSuccess) { c->fft_w = nullptr; return fail_cuda(c, e, "gf_fft_attach"); }
  c->launches += 1;
  return GF_OK;
}

// Alg. 2 l.3-16 given Delta(x) already in fft_w: transform, factor, transform back, rotate the links.
static int fft_update(gf_ctx* c, double alpha) {
  int n = 0;
  const char* msg = nullptr;
  cudaError_t e;
  if (c->fft_accelerate && c->fft_own && own_fft_supported(c->k.geo, c->k.gauge, c->k.prec)) {
    // hand-written passes: transform, factor and inverse transform without cuFFT (gf_fft.cu)
    e = launch_own_fft_update(c->k, c->fft_w, c->own_table, alpha, &n);
    if (e != cudaSuccess) return fail_cuda(c, e, "gf_fft_step (transforms)");
    e = launch_sd_rotate(c->k, c->fft_w);
    if (e != cudaSuccess) return fail_cuda(c, e, "gf_fft_step (rotate)");
    c->launches += n + 1;
    c->qblocks = 0;
    c->sweeps_total += 1;
    if (c->reunit_every > 0 && c->sweeps_total % c->reunit_every == 0) return gf_reunitarize(c);
    return GF_OK;
  }
  // Landau gauge, n_t a power of two: the t direction (transform, factor, inverse transform) is one fused pass
  const bool fused_t = c->fft_accelerate && c->fft_fused_t && c->k.gauge == GF_LANDAU && sd_tline_supported(c->k.geo);
  if (c->fft_accelerate) msg = fft_exec(c->fft, c->k.geo, c->k.prec, c->fft_w, true, !fused_t, &n);
  if (msg) return fail(c, GF_ECUDA, msg);
  if (fused_t) e = launch_sd_tline(c->k, c->fft_w, c->fft_table, alpha);
  else e = launch_sd_filter(c->k, c->fft_w, c->fft_table, alpha, c->fft_accelerate != 0);
  if (e != cudaSuccess) return fail_cuda(c, e, "gf_fft_step (factor)");
  if (c->fft_accelerate) msg = fft_exec(c->fft, c->k.geo, c->k.prec, c->fft_w, false, !fused_t, &n);
  if (msg) return fail(c, GF_ECUDA, msg);
  e = launch_sd_rotate(c->k, c->fft_w);
  if (e != cudaSuccess) return fail_cuda(c, e, "gf_fft_step (rotate)");
  c->launches += n + 2;
  c->qblocks = 0;
  c->sweeps_total += 1;
  if (c->reunit_every > 0 && c->sweeps_total % c->reunit_every == 0) return gf_reunitarize(c);
  return GF_OK;
}

static int fft_delta(gf_ctx* c) {
  int rc = defer_flush(c);  // the rotation of Algorithm 2 works on all four directions in place
  if (rc != GF_OK) return rc;
  cudaError_t e = launch_sd_delta(c->k, c->fft_w);
  if (e != cudaSuccess) return fail_cuda(c, e, "gf_fft_step (Delta)");
  c->launches += 1;
  return GF_OK;
}

// F, theta from the partials of the last fft_delta; synchronises
static int fft_read_result(gf_ctx* c, double* F, double* theta) {
  cudaError_t e = launch_sd_final(c->k);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->k.stream);
  if (e != cudaSuccess) return fail_cuda(c, e, "gf_fix_fft (F, theta)");
  c->launches += 1;
  *F = c->host_result[0];
  *theta = c->host_result[1];
  if (!std::isfinite(*F) || !std::isfinite(*theta)) return fail(c, GF_ENUMERIC, "gf_fix_fft: non-finite F or theta");
  return GF_OK;
}

int gf_fft_step(gf_ctx* c, int n, double alpha) {
  GF_ENTER(c);
  if (n < 0) return fail(c, GF_EINVAL, "gf_fft_step: n < 0");
  if (!(alpha > 0.0) || !std::isfinite(alpha)) return fail(c, GF_EINVAL, "gf_fft_step: alpha must be positive");
  if (!c->fft_w) return fail(c, GF_EINVAL, "gf_fft_step: no workspace attached (gf_fft_attach)");
  for (int i = 0; i < n; ++i) {
    int rc = fft_delta(c);
    if (rc == GF_OK) rc = fft_update(c, alpha);
    if (rc != GF_OK) return rc;
  }
  return GF_OK;
}

int gf_fix_fft(gf_ctx* c, double alpha, double eps, int max_iters, int check_every, int* iters_done) {
  GF_ENTER(c);
  if (!iters_done) return fail(c, GF_EINVAL, "gf_fix_fft: null iters_done");
  if (check_every < 1 || max_iters < 0 || !(eps >= 0.0))
    return fail(c, GF_EINVAL, "gf_fix_fft: need check_every >= 1, max_iters >= 0, eps >= 0");
  if (!(alpha > 0.0) || !std::isfinite(alpha)) return fail(c, GF_EINVAL, "gf_fix_fft: alpha must be positive");
  if (!c->fft_w) return fail(c, GF_EINVAL, "gf_fix_fft: no workspace attached (gf_fft_attach)");
  c->history.clear();
  c->history_n = 0;
  *iters_done = 0;
  int done = 0;
  double F, th;
  // Alg. 2 l.1: Delta(x), F and theta in one pass; the same Delta(x) feeds the first iteration
  int rc = fft_delta(c);
  if (rc == GF_OK) rc = fft_read_result(c, &F, &th);
  if (rc != GF_OK) return rc;
  auto record = [&]() {
    c->history.push_back((double)done);
    c->history.push_back(F);
    c->history.push_back(th);
    c->history_n += 1;
  };
  record();
  while (!(th < eps) && done < max_iters) {  // l.2
    const int n = check_every < max_iters - done ? check_every : max_iters - done;
    for (int i = 0; i < n; ++i) {
      rc = fft_update(c, alpha);              // l.3-16
      if (rc == GF_OK) rc = fft_delta(c);     // l.17 (its F, theta are read back only at the cadence)
      if (rc != GF_OK) return rc;
    }
    done += n;
    *iters_done = done;
    rc = fft_read_result(c, &F, &th);
    if (rc != GF_OK) return rc;
    record();
  }
  return GF_OK;
}

// ---- T-slab sharding --------------------------------------------------------------------------------
size_t gf_slab_halo_bytes(const gf_ctx* c) { return c ? c->halo_bytes : 0; }

int gf_slab_attach(gf_ctx* c, void* dev_halo, size_t bytes) {
  GF_ENTER(c);
  if (!dev_halo) return fail(c, GF_EINVAL, "gf_slab_attach: null workspace");
  if (c->k.storage == 8 || is_sun(c)) return fail(c, GF_EUNSUPPORTED, "gf_slab_attach: SU(3) with 18- or 12-real storage only");
  if (bytes < 4 * c->halo_bytes || ((uintptr_t)dev_halo % ALIGN))
    return fail(c, GF_ENOMEM, "gf_slab_attach: workspace too small or misaligned");
  if (c->fft_w) return fail(c, GF_EUNSUPPORTED, "gf_slab_attach: Algorithm 2 is attached to this context");
  if (c->k.series > 0) return fail(c, GF_EUNSUPPORTED, "gf_slab_attach: no series variant (GF_OPT_OVR_SERIES) on a slab");
  if (c->defer_acc) return fail(c, GF_EUNSUPPORTED, "gf_slab_attach: temporal links are deferred on this context");
  char* base = (char*)dev_halo;
  c->k.slab.ghost = base;  // ghost[0], ghost[1]
  c->top_out = base + 2 * c->halo_bytes;
  c->top_in = base + 3 * c->halo_bytes;
  c->qblocks = 0;
  return GF_OK;
}

int gf_slab_set_targets(gf_ctx* c, void* upper_ghost0, void* upper_ghost1, void* lower_top_in) {
  GF_ENTER(c);
  if (!c->k.slab.ghost) return fail(c, GF_EINVAL, "gf_slab_set_targets: no halo workspace attached (gf_slab_attach)");
  if ((upper_ghost0 == nullptr) != (upper_ghost1 == nullptr) || (upper_ghost0 == nullptr) != (lower_top_in == nullptr))
    return fail(c, GF_EINVAL, "gf_slab_set_targets: give all three targets or none");
  c->fwd_target[0] = (char*)upper_ghost0;
  c->fwd_target[1] = (char*)upper_ghost1;
  c->ret_target = c->ret_target_odd = (char*)lower_top_in;
  c->alt_top_in = false;
  return GF_OK;
}

int gf_slab_set_peer_targets(gf_ctx* c, void* upper_ghost0, void* upper_ghost1, void* lower_top_in_even,
                             void* lower_top_in_odd) {
  GF_ENTER(c);
  if (!c->k.slab.ghost) return fail(c, GF_EINVAL, "gf_slab_set_peer_targets: no halo workspace attached (gf_slab_attach)");
  if (!upper_ghost0 || !upper_ghost1 || !lower_top_in_even || !lower_top_in_odd)
    return fail(c, GF_EINVAL, "gf_slab_set_peer_targets: null target");
  c->fwd_target[0] = (char*)upper_ghost0;
  c->fwd_target[1] = (char*)upper_ghost1;
  c->ret_target = (char*)lower_top_in_even;
  c->ret_target_odd = (char*)lower_top_in_odd;
  c->alt_top_in = true;
  return GF_OK;
}

// ---- stream-ordered neighbour synchronisation and the whole sharded sweep behind one call -----------------------------------
namespace {
typedef int (*stream_memop_fn)(cudaStream_t, unsigned long long, unsigned, unsigned);
// cuStreamWriteValue32 / cuStreamWaitValue32, looked up at run time (no link dependency on libcuda)
stream_memop_fn driver_memop(const char* name) {
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult q;
  if (cudaGetDriverEntryPoint(name, &fn, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) return nullptr;
  return (stream_memop_fn)fn;
}
// "everything this slab queued so far is done": written into both neighbours' flag slots, in stream order
int slab_signal(gf_ctx* c, unsigned epoch) {
  static stream_memop_fn write32 = driver_memop("cuStreamWriteValue32");
  if (!write32) return fail(c, GF_ECUDA, "cuStreamWriteValue32 is not available");
  DeviceGuard guard(c);
  if (write32(c->k.stream, (unsigned long long)(uintptr_t)c->upper_flag, epoch, 0) != 0 ||
      write32(c->k.stream, (unsigned long long)(uintptr_t)c->lower_flag, epoch, 0) != 0)
    return fail(c, GF_ECUDA, "cuStreamWriteValue32 failed");
  c->epoch = epoch;
  return GF_OK;
}
// the slab's stream goes on once both neighbours have signalled `epoch` (wrap-safe >= comparison)
int slab_wait(gf_ctx* c, unsigned epoch) {
  static stream_memop_fn wait32 = driver_memop("cuStreamWaitValue32");
  if (!wait32) return fail(c, GF_ECUDA, "cuStreamWaitValue32 is not available");
  DeviceGuard guard(c);
  if (wait32(c->k.stream, (unsigned long long)(uintptr_t)&c->own_flags[0], epoch, 0 /* GEQ */) != 0 ||
      wait32(c->k.stream, (unsigned long long)(uintptr_t)&c->own_flags[1], epoch, 0) != 0)
    return fail(c, GF_ECUDA, "cuStreamWaitValue32 failed");
  return GF_OK;
}
// A group is closed if every neighbour of every slab is itself a slab of the group and all of them run on one stream
// of one device (the whole lattice in one process): stream order already is the order the flags would enforce.
bool group_is_closed(gf_ctx* const* slabs, int n) {
  for (int s = 0; s < n; ++s) {
    if (slabs[s]->k.stream != slabs[0]->k.stream || slabs[s]->device != slabs[0]->device || slabs[s]->slab_force_flags)
      return false;
    bool up = false, lo = false;
    for (int r = 0; r < n; ++r) {
      up = up || slabs[s]->upper_flag == slabs[r]->own_flags + 1;
      lo = lo || slabs[s]->lower_flag == slabs[r]->own_flags;
    }
    if (!up || !lo) return false;
  }
  return true;
}
// the slab's stream goes on once both neighbours' border blocks of the current fused launch have stored: from inside its
// kernel (system-scope atomic) the upper neighbour adds 1 to own_flags[3], the lower one to own_flags[4].  One word per
// neighbour, one wait per word: a single summed counter cannot tell "both at launch n" from "one at n+1, the other at
// n-1", a state a ring of four or more slabs on different streams or ranks does reach (a slab's launch n+1 needs only ITS
// neighbours at n), and the slab between the two would read a ghost buffer its late neighbour has not written yet.
int slab_wait_arrivals(gf_ctx* c) {
  static stream_memop_fn wait32 = driver_memop("cuStreamWaitValue32");
  if (!wait32) return fail(c, GF_ECUDA, "cuStreamWaitValue32 is not available");
  DeviceGuard guard(c);
  if (wait32(c->k.stream, (unsigned long long)(uintptr_t)&c->own_flags[3], c->arrivals, 0 /* GEQ */) != 0 ||
      wait32(c->k.stream, (unsigned long long)(uintptr_t)&c->own_flags[4], c->arrivals, 0) != 0)
    return fail(c, GF_ECUDA, "cuStreamWaitValue32 failed");
  return GF_OK;
}
// one ordering point of the group with its neighbours (local or remote): every slab signals, then every slab waits
int group_sync(gf_ctx* const* slabs, int n) {
  if (group_is_closed(slabs, n)) return GF_OK;
  for (int s = 0; s < n; ++s)
    if (int rc = slab_signal(slabs[s], slabs[s]->epoch + 1); rc != GF_OK) return rc;
  for (int s = 0; s < n; ++s)
    if (int rc = slab_wait(slabs[s], slabs[s]->epoch); rc != GF_OK) return rc;
  return GF_OK;
}
int group_check(gf_ctx* const* slabs, int n, const char* who) {
  if (!slabs || n < 1) return GF_EINVAL;
  for (int s = 0; s < n; ++s) {
    gf_ctx* c = slabs[s];
    if (!c) return GF_EINVAL;
    if (!c->k.slab.ghost || !c->alt_top_in || !c->own_flags) return fail(c, GF_EINVAL, who);
    if (c->epoch != slabs[0]->epoch || c->arrivals != slabs[0]->arrivals)
      return fail(c, GF_EINVAL, "the slabs of a group must have been driven together");
  }
  return GF_OK;
}
// both ghost buffers of every neighbour from this group's top slices (after set_links, reunitarize)
int group_refresh(gf_ctx* const* slabs, int n) {
  int rc = group_sync(slabs, n);  // nobody still reads the ghost buffers that are about to be overwritten
  for (int q = 0; q < 2 && rc == GF_OK; ++q)
    for (int s = 0; s < n && rc == GF_OK; ++s) rc = gf_slab_pack_top(slabs[s], q);
  if (rc == GF_OK) rc = group_sync(slabs, n);
  return rc;
}
}  // namespace

int gf_slab_set_peer_flags(gf_ctx* c, void* own_flags, void* upper_flag, void* lower_flag) {
  GF_ENTER(c);
  if (!c->k.slab.ghost) return fail(c, GF_EINVAL, "gf_slab_set_peer_flags: no halo workspace attached (gf_slab_attach)");
  if (!own_flags || !upper_flag || !lower_flag || ((uintptr_t)own_flags % 32))
    return fail(c, GF_EINVAL, "gf_slab_set_peer_flags: null or misaligned flag address");
  c->own_flags = (unsigned*)own_flags;
  c->upper_flag = (unsigned*)upper_flag;
  c->lower_flag = (unsigned*)lower_flag;
  c->epoch = 0;
  c->arrivals = 0;
  // two epoch words, the border-block counter, two arrival counters (3 words of padding)
  cudaError_t e = cudaMemsetAsync(own_flags, 0, 8 * sizeof(unsigned), c->k.stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->k.stream);  // zero before any neighbour can signal
  if (e != cudaSuccess) return fail_cuda(c, e, "gf_slab_set_peer_flags");
  return GF_OK;
}

int gf_slab_group_refresh(gf_ctx* const* slabs, int n_slabs) {
  int rc = group_check(slabs, n_slabs, "gf_slab_group_refresh: every slab needs gf_slab_set_peer_targets and gf_slab_set_peer_flags");
  return rc == GF_OK ? group_refresh(slabs, n_slabs) : rc;
}

int gf_slab_group_sweep(gf_ctx* const* slabs, int n_slabs, int n_sweeps, double omega, int reunit_every, long long sweeps_before) {
  int rc = group_check(slabs, n_slabs, "gf_slab_group_sweep: every slab needs gf_slab_set_peer_targets and gf_slab_set_peer_flags");
  if (rc != GF_OK) return rc;
  if (n_sweeps < 0 || reunit_every < 0 || sweeps_before < 0) return fail(slabs[0], GF_EINVAL, "gf_slab_group_sweep: negative argument");
  if (!(omega >= 1.0 && omega < 2.0)) return fail(slabs[0], GF_EINVAL, "gf_slab_group_sweep: omega outside [1,2)");
  if (n_sweeps == 0) return GF_OK;
  // entry: whatever the neighbours still run on the buffers of the last call (a measurement reads the ghost links) is done
  rc = group_sync(slabs, n_slabs);
  // The links the upper neighbour returns during half-sweep p (into top_in, double-buffered by p) belong to the top-slice
  // sites of parity 1-p, which are visited next: the next launch reads them straight from that buffer, and only the
  // last half-sweep of the call (or one before a reunitarisation) is followed by gf_slab_unpack_top.
  bool pending = false;  // top-slice U_t of parity 0 still sits in the buffer the odd half-sweep filled
  const bool closed = group_is_closed(slabs, n_slabs);  // no flags needed: one stream orders everything
  for (int i = 0; i < n_sweeps && rc == GF_OK; ++i) {
    for (int p = 0; p < 2 && rc == GF_OK; ++p) {  // even first
      // ONE kernel per slab and half-sweep: its border blocks come first, store both halo messages at their destination
      // (gf_slab_set_peer_targets) and the last of them raises the neighbours' flags, while the rest of the grid
      // updates the interior ("overlap ... with the update of the remaining gauge links")
      for (int s = 0; s < n_slabs && rc == GF_OK; ++s) {
        gf_ctx* c = slabs[s];
        DeviceGuard guard(c);
        const void* returned = nullptr;  // what half-sweep 1-p left for this one
        if (p == 1) returned = c->top_in;
        else if (pending) returned = c->top_out;
        cudaError_t e = launch_halfsweep_slab_fused(c->k, p, omega, c->fwd_target[p], p ? c->ret_target_odd : c->ret_target,
                                                    closed ? nullptr : c->own_flags + 2,
                                                    c->upper_flag + 3 /* its own_flags[4]: from below */,
                                                    c->lower_flag + 3 /* its own_flags[3]: from above */, returned);
        if (e != cudaSuccess) { rc = fail_cuda(c, e, "gf_slab_group_sweep"); break; }
        c->arrivals += 1;
        c->launches += 1;
        c->qblocks = 0;
      }
      for (int s = 0; s < n_slabs && rc == GF_OK && !closed; ++s) rc = slab_wait_arrivals(slabs[s]);
    }
    pending = true;
    const bool last = i == n_sweeps - 1;
    const bool reunit = reunit_every > 0 && (sweeps_before + i + 1) % reunit_every == 0;
    if (rc == GF_OK && (last || reunit)) {
      for (int s = 0; s < n_slabs && rc == GF_OK; ++s) rc = gf_slab_unpack_top(slabs[s], 0);
      pending = false;
    }
    if (rc == GF_OK && reunit) {
      for (int s = 0; s < n_slabs && rc == GF_OK; ++s) rc = gf_reunitarize(slabs[s]);
      if (rc == GF_OK) rc = group_refresh(slabs, n_slabs);
    }
  }
  return rc;
}

// ---- device memory of another process (CUDA IPC), for gf_slab_set_peer_targets between ranks --------------------------------
int gf_ipc_export(const void* dev_ptr, unsigned char* handle64, size_t* offset) {
  if (!dev_ptr || !handle64 || !offset) return GF_EINVAL;
  // the handle names the whole allocation dev_ptr lies in (torch hands out pieces of larger cudaMalloc segments):
  // find its base through the driver's cuMemGetAddressRange, looked up at run time (no link dependency on libcuda)
  typedef int (*range_fn)(unsigned long long*, size_t*, unsigned long long);
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult q;
  if (cudaGetDriverEntryPoint("cuMemGetAddressRange", &fn, cudaEnableDefault, &q) != cudaSuccess || !fn ||
      q != cudaDriverEntryPointSuccess)
    return GF_ECUDA;
  unsigned long long base = 0;
  size_t size = 0;
  if (((range_fn)fn)(&base, &size, (unsigned long long)(uintptr_t)dev_ptr) != 0) return GF_ECUDA;
  cudaIpcMemHandle_t h;
  static_assert(sizeof(h) == 64, "cudaIpcMemHandle_t is 64 bytes");
  if (cudaIpcGetMemHandle(&h, (void*)(uintptr_t)base) != cudaSuccess) { cudaGetLastError(); return GF_ECUDA; }
  memcpy(handle64, &h, 64);
  *offset = (size_t)((uintptr_t)dev_ptr - (uintptr_t)base);
  return GF_OK;
}

int gf_ipc_open(const unsigned char* handle64, size_t offset, void** dev_ptr) {
  if (!handle64 || !dev_ptr) return GF_EINVAL;
  cudaIpcMemHandle_t h;
  memcpy(&h, handle64, 64);
  void* base = nullptr;
  if (cudaIpcOpenMemHandle(&base, h, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess) { cudaGetLastError(); return GF_ECUDA; }
  *dev_ptr = (char*)base + offset;
  return GF_OK;
}

int gf_ipc_close(void* dev_ptr, size_t offset) {
  if (!dev_ptr) return GF_EINVAL;
  if (cudaIpcCloseMemHandle((char*)dev_ptr - offset) != cudaSuccess) { cudaGetLastError(); return GF_ECUDA; }
  return GF_OK;
}

// ---- the driver's decisions, for callers that run Algorithm 1 over several contexts (slabs) -------------------------------
int gf_combine_slabs(const double* F_slab, const double* theta_slab, int n_slabs, double* F, double* theta) {
  if (!F_slab || !theta_slab || !F || !theta || n_slabs < 1) return GF_EINVAL;
  double f = 0.0, t = 0.0;
  for (int s = 0; s < n_slabs; ++s) {  // slab order: every rank adds the same numbers in the same order
    f += F_slab[s];
    t += theta_slab[s];
  }
  *F = f / n_slabs;  // slabs have equal volumes: the global normalisation d Nc V is n_slabs times a slab's
  *theta = t / n_slabs;
  return (std::isfinite(*F) && std::isfinite(*theta)) ? GF_OK : GF_ENUMERIC;
}

int gf_fix_plan(double omega, double eps, int max_sweeps, int check_every, int sweeps_done, double theta, int* n_next) {
  if (!n_next) return GF_EINVAL;
  *n_next = 0;
  if (check_every < 1 || max_sweeps < 0 || sweeps_done < 0 || !(eps >= 0.0)) return GF_EINVAL;
  if (!(omega >= 1.0 && omega < 2.0)) return GF_EINVAL;
  if (theta < eps || sweeps_done >= max_sweeps) return GF_OK;  // Algorithm 1 l.2: stop
  *n_next = check_every < max_sweeps - sweeps_done ? check_every : max_sweeps - sweeps_done;
  return GF_OK;
}

static int slab_check(gf_ctx* c, int parity, const char* who) {
  if (!c) return GF_EINVAL;
  if (!c->k.slab.ghost) return fail(c, GF_EINVAL, "gf_slab_*: no halo workspace attached (gf_slab_attach)");
  if (parity != 0 && parity != 1) return fail(c, GF_EINVAL, who);
  return GF_OK;
}

int gf_slab_pack_top(gf_ctx* c, int parity) {
  DeviceGuard gf_device_guard_(c);
  int rc = slab_check(c, parity, "gf_slab_pack_top: parity must be 0 or 1");
  if (rc != GF_OK) return rc;
  cudaError_t e = launch_slab_top(c->k, parity, c->fwd_target[parity] ? c->fwd_target[parity] : c->top_out, true);
  if (e != cudaSuccess) return fail_cuda(c, e, "gf_slab_pack_top");
  c->launches += 1;
  return GF_OK;
}

int gf_slab_unpack_top(gf_ctx* c, int parity) {
  DeviceGuard gf_device_guard_(c);
  int rc = slab_check(c, parity, "gf_slab_unpack_top: parity must be 0 or 1");
  if (rc != GF_OK) return rc;
  // with peer targets the odd half-sweep's "ret" message arrived in the top_out slot (top_in is double-buffered, so that
  // one cross-rank synchronisation per half-sweep is enough); unpack_top(1 - p) follows half-sweep p
  cudaError_t e = launch_slab_top(c->k, parity, (c->alt_top_in && parity == 0) ? c->top_out : c->top_in, false);
  if (e != cudaSuccess) return fail_cuda(c, e, "gf_slab_unpack_top");
  c->launches += 1;
  c->qblocks = 0;
  return GF_OK;
}

int gf_slab_halfsweep_border(gf_ctx* c, int parity, double omega) {
  DeviceGuard gf_device_guard_(c);
  int rc = slab_check(c, parity, "gf_slab_halfsweep_border: parity must be 0 or 1");
  if (rc != GF_OK) return rc;
  if (!(omega >= 1.0 && omega < 2.0)) return fail(c, GF_EINVAL, "gf_slab_halfsweep_border: omega outside [1,2)");
  const Geo& g = c->k.geo;
  // one launch: bottom slice, top slice; the top-slice sites also write their updated U_t(x) into top_out
  cudaError_t e = launch_halfsweep_slab(c->k, parity, omega, 0, g.s3, g.vh - g.s3, g.vh,
                                        c->fwd_target[parity] ? c->fwd_target[parity] : c->top_out,
                                        parity ? c->ret_target_odd : c->ret_target);
  if (e != cudaSuccess) return fail_cuda(c, e, "gf_slab_halfsweep_border");
  c->launches += 1;
  c->qblocks = 0;
  return GF_OK;
}

int gf_slab_halfsweep_interior(gf_ctx* c, int parity, double omega) {
  DeviceGuard gf_device_guard_(c);
  int rc = slab_check(c, parity, "gf_slab_halfsweep_interior: parity must be 0 or 1");
  if (rc != GF_OK) return rc;
  if (!(omega >= 1.0 && omega < 2.0)) return fail(c, GF_EINVAL, "gf_slab_halfsweep_interior: omega outside [1,2)");
  const Geo& g = c->k.geo;
  if (g.n[3] == 2) return GF_OK;
  cudaError_t e = launch_halfsweep_slab(c->k, parity, omega, g.s3, g.vh - g.s3, 0, 0, nullptr, nullptr);
  if (e != cudaSuccess) return fail_cuda(c, e, "gf_slab_halfsweep_interior");
  c->launches += 1;
  c->qblocks = 0;
  return GF_OK;
}

long long gf_kernel_launches(const gf_ctx* c) { return c ? c->launches : 0; }

const char* gf_strerror(int code) {
  switch (code) {
    case GF_OK: return "ok";
    case GF_EINVAL: return "invalid argument";
    case GF_EODD: return "lattice extents must be even and >= 2";
    case GF_EUNSUPPORTED: return "unsupported gauge / precision / storage / volume";
    case GF_ENOMEM: return "workspace too small or misaligned";
    case GF_ECUDA: return "CUDA error";
    case GF_ENUMERIC: return "non-finite F or theta";
    default: return "unknown error";
  }
}

const char* gf_last_error(const gf_ctx* c) { return c ? c->err : ""; }

}  // extern "C"
