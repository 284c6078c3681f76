/* gf.h — C ABI of libgf: the data-parallel hot path of lattice Landau/Coulomb gauge fixing by overrelaxation on one
 * NVIDIA B200 (sm_100a), after N. Cardoso, "Coulomb and Landau Gauge Fixing in GPUs using CUDA and MILC",
 * arXiv:1412.1498 (cited below as PAPER.md:<line>, the text under /root/reference).
 *
 * What the library computes (eqs. 1.1-1.6; Algorithm 1):
 *   - the checkerboarded SU(3) overrelaxation sweep: for every site x of one parity, K(x) = sum_mu [U_mu(x) +
 *     U_mu(x-mu)^dagger] (eq. 1.5; mu = 0..3 Landau, mu = 0..2 Coulomb), local maximisation of
 *     Re Tr[g K] (eq. 1.4) over the three SU(2) subgroups (eq. 1.6), each raised to the overrelaxation
 *     power omega, then g(x) applied to U_mu(x) and U_mu(x-mu) for all four mu (Alg. 1 l.7-8);
 *   - the reduction that gives F (eq. 1.1) and theta (eqs. 1.2-1.3);
 *   - link reunitarisation every k sweeps;
 *   - the driver loop of Algorithm 1 with a measurement cadence;
 * and, to the same parity bar (sections further down): Algorithm 2, steepest descent with Fourier acceleration
 * (gf_fft_*); the paper's multi-GPU decomposition of the sweep into T-slabs (gf_slab_*); two variants of Algorithm 1
 * (g^omega as a truncated series, GF_OPT_OVR_SERIES; Coulomb gauge with a stop test per time slice, gf_fix_slices).
 * Readings taken where the paper is silent or ambiguous are listed in DESIGN.md (A1-A22, B1-B6).
 *
 * Conventions
 *   - Every function returns 0 (GF_OK) or a negative GF_E* code; nothing throws, nothing aborts.
 *   - "dev" pointers are CUDA device pointers, "host" pointers are ordinary host pointers.  The caller owns all device
 *     memory: the library never allocates or frees device memory and keeps no pointer to a links buffer after the
 *     call that received it returns (copies are ordered on the context's stream).  gf_ctx itself (plus a few bytes of
 *     pinned host memory for the two result scalars) is host memory owned by the library until gf_destroy.
 *   - All work is enqueued on the cuda_stream given to gf_create (a cudaStream_t passed as void*; NULL = default
 *     stream).  Calls documented "async" return without waiting for the device.
 *   - Canonical (external) link layout, used by every set/get call regardless of the internal storage:
 *         links[site][mu][row][col][re,im],  site = x + nx*(y + ny*(z + nz*t))   (x fastest),
 *     mu = 0..3 = (x,y,z,t) with mu = 3 temporal; 18 reals per link, element type double (GF_FP64) or
 *     float (GF_FP32).  U_mu(x) is the link from x to x+mu.  Total 72*V elements, V = nx*ny*nz*nt.
 *   - Site parity is (x+y+z+t)&1 in both gauges; a sweep updates parity 0 ("even") first, then parity 1
 *     (PAPER.md:134).
 */
#ifndef GF_H
#define GF_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gf_ctx gf_ctx; /* opaque */

enum { GF_LANDAU = 0, GF_COULOMB = 1 };
enum { GF_FP64 = 0, GF_FP32 = 1 };      /* PAPER.md:140 (SP/DP) */
/* storage: 18 (full 3x3), 12 (rows 0,1 stored; row 2 = conj(row0 x row1) rebuilt at every load) or 8 reals per link,
 * PAPER.md:128, 144, 174.  8 (reading A23 in DESIGN.md): a2, a3, b1 and the phases of a1 and c1 (each as tan(phase/2))
 * are kept, the rest follows from unitarity and det = 1 with a division by N = |a2|^2 + |a3|^2.
 * VALIDITY DOMAIN of storage = 8: undefined for block-diagonal links (N = 0: the unit field, a cold start) and
 * rounding is amplified by 1/N.  Whenever a link with N < 1e-6 (GF_FP64; error ~1e-10) or N < 1e-3 (GF_FP32; error
 * ~6e-5) is stored - by gf_set_links or by a sweep - a flag is raised and the next gf_measure, gf_fix or
 * gf_*_links_host returns GF_ENUMERIC with the reason in gf_last_error (the flag is then cleared; gf_set_links[_host]
 * clear it too before they load the new field, so a report always concerns the field the context holds.  It is kept
 * per device, not per context: two storage = 8 contexts working on one GPU at the same time see, and clear, each
 * other's reports - run such contexts one after the other).  Smooth fields close to Landau gauge have N ~ |U - 1|^2 and leave the domain: use 12 or
 * 18 there.  With storage = 8 the library offers gf_set/get_links[_host], gf_ovr_sweep, gf_measure, gf_fix,
 * gf_reunitarize; the gf_fft_*, gf_slab_*, gf_defer_*, gf_*_slices calls and GF_OPT_OVR_SERIES return
 * GF_EUNSUPPORTED. */

enum {
  GF_OK = 0,
  GF_EINVAL = -1,       /* null pointer, n < 0, check_every < 1, omega outside [1,2), bad option */
  GF_EODD = -2,         /* an extent is odd or < 2 (all lattice dimensions must be even) */
  GF_EUNSUPPORTED = -3, /* storage not in {8,12,18} (8: FP64 only), unknown gauge / precision, V >= 2^31 */
  GF_ENOMEM = -4,       /* workspace too small or misaligned (256-byte alignment required) */
  GF_ECUDA = -5,        /* a CUDA call failed; text via gf_last_error */
  GF_ENUMERIC = -6      /* F or theta came back NaN/Inf */
};

/* Bytes of device workspace gf_create needs for this lattice: the internal-layout link field, the partial-sum
 * scratch of the F/theta reduction, the result scalars and two staging buffers for the *_host calls.
 * Returns 0 if the arguments are invalid. */
size_t gf_workspace_bytes(int nx, int ny, int nz, int nt, int prec, int storage);

/* Create a context.  dev_workspace: caller-owned device memory of at least gf_workspace_bytes(...) bytes, 256-byte
 * aligned, which must stay valid until gf_destroy.  cuda_stream: the stream all work of this context runs on.
 * The link field is undefined until gf_set_links[_host].  Errors: GF_EINVAL, GF_EODD, GF_EUNSUPPORTED, GF_ENOMEM,
 * GF_ECUDA. */
int gf_create(gf_ctx** out, int nx, int ny, int nz, int nt, int gauge, int prec, int storage, void* dev_workspace,
              size_t workspace_bytes, void* cuda_stream);

/* General number of colours ("SU(N) with N>2": "iterating over its N(N-1)/2 SU(2)
 * subgroups"; readings A24, A25 in DESIGN.md).  ncolors = 3 is gf_create with storage = 18; ncolors = 2 and 4 run the
 * general kernels: all N^2 complex entries of a link are stored, the canonical layout is
 * links[site][mu][row][col][re,im] with N x N matrices (8 N^2 V elements), the subgroups (i,j), i < j, are visited by
 * increasing j - i, then i, F is normalised by d N V and theta by N V, and reunitarisation is Gram-Schmidt over the rows
 * followed by the last row times conj(det).  On such a context gf_set/get_links[_host], gf_ovr_sweep, gf_measure,
 * gf_fix, gf_get_history, gf_reunitarize and gf_set_reunit_every work as described here; every other call
 * (gf_set_option, gf_fft_*, gf_slab_*, gf_defer_*, gf_*_slices) returns GF_EUNSUPPORTED.  Other ncolors:
 * GF_EUNSUPPORTED (gf_workspace_bytes_sun: 0). */
size_t gf_workspace_bytes_sun(int ncolors, int nx, int ny, int nz, int nt, int prec);
int gf_create_sun(gf_ctx** out, int ncolors, int nx, int ny, int nz, int nt, int gauge, int prec, void* dev_workspace,
                  size_t workspace_bytes, void* cuda_stream);

/* Canonical layout (device) -> internal layout.  With storage = 12 only rows 0 and 1 are kept.  Resets the sweep
 * counter used by the reunitarisation cadence.  Async. */
int gf_set_links(gf_ctx* ctx, const void* dev_links);
/* Internal layout -> canonical layout (device), 18 reals per link always (row 2 rebuilt if storage = 12).  Async. */
int gf_get_links(gf_ctx* ctx, void* dev_links_out);
/* Same, from / to HOST memory (pinned memory makes the copies asynchronous and faster, pageable works): the field is
 * streamed through the workspace's staging buffers in chunks, copy and reorder overlapped.  gf_get_links_host
 * synchronises the stream before returning; gf_set_links_host returns once the host buffer has been consumed. */
int gf_set_links_host(gf_ctx* ctx, const void* host_links);
int gf_get_links_host(gf_ctx* ctx, void* host_links_out);

/* n overrelaxation sweeps (Algorithm 1 l.3-12): each sweep is the parity-0 half-sweep then the
 * parity-1 half-sweep with overrelaxation parameter omega in [1,2); after global sweep number s the links are
 * reunitarised if reunit_every > 0 and s % reunit_every == 0.  n = 0 is a no-op.  Async. */
int gf_ovr_sweep(gf_ctx* ctx, int n, double omega);

/* F (eq. 1.1, normalised by the d directions summed) and theta (eqs. 1.2-1.3) of the links as they stand, written to
 * host out-params.  FP64 accumulation in both precisions, deterministic summation order.  Synchronises the stream.
 * GF_ENUMERIC if either value is not finite (the values are still written). */
int gf_measure(gf_ctx* ctx, double* F, double* theta);

/* Algorithm 1 with a measurement cadence: measure; while theta >= eps and sweeps < max_sweeps: do
 * min(check_every, remaining) sweeps, measure.  *sweeps_done = sweeps performed (0 if already converged).  eps = 0
 * gives a fixed-sweep run.  The (sweep, F, theta) triple of every measurement is kept and can be read with
 * gf_get_history.  Synchronises the stream at every measurement. */
int gf_fix(gf_ctx* ctx, double omega, double eps, int max_sweeps, int check_every, int* sweeps_done);
/* Copies up to cap triples {sweep, F, theta} (3 doubles each) of the last gf_fix into hist (host); *n = number of
 * measurements the run made (may exceed cap). */
int gf_get_history(gf_ctx* ctx, double* hist, int cap, int* n);

/* Coulomb gauge with a stop test per time slice (BASELINE.json configs[1]: "each of the 32 time slices is fixed
 * independently"; K(x) of a Coulomb-gauge site holds links of its own slice only; reading A22 in DESIGN.md).
 * gf_measure_slices: F_t and theta_t, eqs. 1.1-1.2 with the sums restricted to time slice t (V -> nx ny nz), into two
 *   host arrays of n_t doubles.  Synchronises the stream.
 * gf_fix_slices: as gf_fix, but a slice with theta_t < eps is finished and its sites are no longer visited; the run ends
 *   when every slice is finished or after max_sweeps.  History triples are {sweep, mean_t F_t, max_t theta_t}.
 *   slice_sweeps (host, n_t ints, may be NULL) receives the sweeps spent on each slice.
 * Errors: GF_EUNSUPPORTED unless the context is Coulomb gauge on a whole lattice with the default sweep variant and
 * the exact power; GF_EINVAL, GF_ECUDA, GF_ENUMERIC as gf_fix. */
int gf_measure_slices(gf_ctx* ctx, double* F_t, double* theta_t);
int gf_fix_slices(gf_ctx* ctx, double omega, double eps, int max_sweeps, int check_every, int* sweeps_done,
                  int* slice_sweeps);

/* Coulomb gauge with deferred temporal links (SURVEY.md reading A9, "cheaper alternative").  K(x) and
 * theta never read a temporal link in Coulomb gauge, so U_t need not be rewritten by every site update: once a buffer
 * is attached, gf_ovr_sweep / gf_fix update the six spatial links of a site and multiply its accumulated rotation
 * A(x) <- G(x) A(x) (one matrix per site): 6 links + A read and written per site-update instead of 8 links.
 * U_t(x) <- A(x) U_t(x) A(x+t)^dagger is applied - and A reset to 1 - by gf_defer_flush, and automatically before
 * gf_get_links[_host], gf_reunitarize, gf_fft_* and on detach; gf_set_links[_host] reset A.  Same result as the in-place
 * update up to rounding (the products are associated differently).
 * gf_defer_bytes: size of the buffer (one direction of the link field).  gf_defer_attach(ctx, dev, bytes): caller-owned,
 *   256-byte aligned, valid until detached with gf_defer_attach(ctx, NULL, 0) or gf_destroy.  Async.
 * Errors: GF_EUNSUPPORTED unless Coulomb gauge on a whole lattice (gf_fix_slices and gf_slab_attach refuse a context
 * with deferred links); GF_ENOMEM; GF_ECUDA (also from gf_ovr_sweep with a non-default sweep variant or series). */
size_t gf_defer_bytes(const gf_ctx* ctx);
int gf_defer_attach(gf_ctx* ctx, void* dev_acc, size_t bytes);
int gf_defer_flush(gf_ctx* ctx);

/* Project every link back onto SU(3): Gram-Schmidt on rows 0,1, row 2 = conj(row0 x row1).  Async. */
int gf_reunitarize(gf_ctx* ctx);
/* k = 0 (default): never; k > 0: reunitarise after every k-th sweep inside gf_ovr_sweep / gf_fix. */
int gf_set_reunit_every(gf_ctx* ctx, int k);

/* Tuning knobs for benchmarking kernel variants; the defaults are the fastest measured.  GF_EINVAL on unknown keys. */
enum {
  GF_OPT_SWEEP_VARIANT = 1, /* half-sweep kernel: 0 = default (5 with FP64 links, 3 with FP32 links or 8-real storage); 1 = two-pass; 2 = two-pass + L2
                               bulk prefetch; 3 = staged through shared memory with cp.async; 4 = staged, the tile
                               fetched by bulk copies of the TMA unit (cp.async.bulk on an mbarrier); 5 = staged, only
                               the contiguous forward chunk by bulk copy; 6 = two warps per 32 sites (forward / backward links; a study, never
                               the default); see DESIGN.md.  {3,4,5} give bit-identical
                               links, so do {1,2}; in FP64 all five do. */
  GF_OPT_BLOCK_THREADS = 2, /* threads per block of the half-sweep kernel (0 = default; a value the chosen variant
                               has no instantiation for makes the next sweep fail with GF_ECUDA) */
  GF_OPT_FUSE_MEASURE = 3,  /* 1 (default): the last odd half-sweep of every gf_ovr_sweep call also leaves the odd
                               sites' terms of theta, so a gf_measure that follows directly visits the even sites only
                               and reads every link once; 0: gf_measure always visits all sites */
  GF_OPT_FFT_ACCELERATE = 4, /* 1 (default): gf_fft_step / gf_fix_fft use the Fourier factor of eq. 1.8; 0: the naive
                               steepest descent of eq. 1.7 (no transforms) */
  GF_OPT_FFT_FUSED_T = 5,   /* 1: in Landau gauge with n_t a power of two (<= 256) the transform along t, the Fourier
                               factor and the inverse transform along t are one hand-written pass through shared
                               memory; 0 (default): cuFFT's strided 1-D transforms and a separate factor kernel */
  GF_OPT_FFT_OWN = 6,       /* 1 (default): when every transformed extent is a product of two of {1,2,3,4,6,8,12,16}
                               (<= 256) and an (x,y) plane fits shared memory, the transforms, the Fourier factor and
                               the inverse transforms run as hand-written passes (5 over the fields in Landau gauge,
                               3 in Coulomb gauge), without cuFFT; other lattices, or 0: the cuFFT path */
  GF_OPT_OVR_SERIES = 7,    /* 0 (default): g^omega of every SU(2) subgroup step is the exact power (reading A6);
                               N = 1..16: the binomial series sum_{n<=N} binom(omega,n) (g-1)^n, normalised back to
                               SU(2) - the way ref. [1] of the paper evaluates g^omega (reading A21).
                               Default sweep variant only; GF_EUNSUPPORTED on a slab context. */
  GF_OPT_DOMAIN8_CHECK = 8, /* 1 (default): storage = 8 reports links outside its validity domain (above); 0: the
                               flag is ignored (kernel studies on rough fields only) */
  GF_OPT_SLAB_FORCE_FLAGS = 9 /* 1: gf_slab_group_sweep signals and waits even where one stream already orders a closed
                               group (to time, in one process, what a rank of a multi-rank run executes) */
};
int gf_set_option(gf_ctx* ctx, int key, int value);

/* ---- Algorithm 2: steepest descent with Fourier acceleration (eqs. 1.7-1.9) ----------
 * One iteration: Delta(x) of eq. 1.3 at every site; each of its independent components is Fourier transformed over
 * the d gauge-fixing directions (4-D for Landau; the 3-D transform of every time slice for Coulomb), multiplied by
 * (alpha/2) p^2_max/p^2 with p^2 = sum_mu 4 sin^2(pi k_mu/n_mu) (0 at p = 0) and transformed back (normalised);
 * g(x) = reunitarise(1 + w(x)) (first-order exponential; Gram-Schmidt as gf_reunitarize);
 * U_mu(x) <- g(x) U_mu(x) g(x+mu)^dagger for all four mu.  Readings B1-B6 in DESIGN.md.  The transforms are the
 * library's own passes (GF_OPT_FFT_OWN) where the lattice extents allow it, else cuFFT calls; cuFFT's own allocation
 * is switched off, its work area lives in the caller's workspace.
 *
 * gf_fft_workspace_bytes: *bytes = size of the SECOND device workspace these calls need (the packed Delta/w fields,
 *   4 complex numbers per site; the momentum table; cuFFT's work area).  Creates the cuFFT plans (needs a device).
 * gf_fft_attach: hands that workspace over (caller-owned, 256-byte aligned, valid until gf_destroy).  Async.
 * gf_fft_step: n iterations with step size alpha > 0 (the paper's value is 0.08).  The reunitarisation cadence of
 *   gf_set_reunit_every counts iterations like sweeps.  Async.
 * gf_fix_fft: Algorithm 2 with a measurement cadence: Delta, F, theta; while theta >= eps and iterations <
 *   max_iters: min(check_every, remaining) iterations (each ends with the Delta/F/theta pass that feeds the next),
 *   read F, theta.  History as for gf_fix (gf_get_history).  Synchronises at every read.
 * Errors: GF_EINVAL (null pointer, n < 0, alpha <= 0, no workspace attached), GF_ENOMEM, GF_ECUDA (CUDA or cuFFT
 * failure, text via gf_last_error), GF_ENUMERIC. */
int gf_fft_workspace_bytes(gf_ctx* ctx, size_t* bytes);
int gf_fft_attach(gf_ctx* ctx, void* dev_workspace, size_t workspace_bytes);
int gf_fft_step(gf_ctx* ctx, int n, double alpha);
int gf_fix_fft(gf_ctx* ctx, double alpha, double eps, int max_iters, int check_every, int* iters_done);

/* ---- T-slab sharding of the overrelaxation sweep (PAPER.md:132-134 border / interior split and the exchange of the
 * top links "and back"; PAPER.md:146 partition T first) ------------------------------------------------------------------
 * A lattice nx*ny*nz*(R*lt) is cut into R slabs of lt time slices (lt even, so local and global site parity agree).
 * Each slab is an ordinary context created with gf_create(nx, ny, nz, lt, ...) that becomes a slab once a halo
 * workspace is attached.  The only links a slab's sites touch that it does not own are U_t(x - t) of its t = 0 sites:
 * the lower neighbour's top-slice temporal links.  They are kept in a ghost buffer that the half-sweep kernels read
 * and update in place; the caller (one process per GPU) moves the four messages below between neighbours with its
 * own transport (device-to-device copies, NCCL send/recv), all device memory, no host staging.
 *
 * Halo workspace (caller-owned device memory, 256-byte aligned, valid until gf_destroy), B = gf_slab_halo_bytes:
 *   [0, B)    ghost[0]: U_t(x) of the parity-0 sites of the lower neighbour's top slice     (kernels read + write)
 *   [B, 2B)   ghost[1]: the same for its parity-1 sites
 *   [2B, 3B)  top_out : U_t(x) of one parity of this slab's top slice, packed by gf_slab_pack_top /
 *                       gf_slab_halfsweep_border, to be delivered into the UPPER neighbour's ghost[parity]
 *   [3B, 4B)  top_in  : a ghost buffer coming back from the upper neighbour, scattered by gf_slab_unpack_top
 * Message layout = the internal layout of one parity of one time slice, direction t only:
 *   [cb3 / 32][element][cb3 % 32] complex numbers, cb3 = (x + nx (y + ny z)) / 2, 9 or 6 elements per link.
 *
 * One half-sweep of parity p on every slab (even first, then odd, as gf_ovr_sweep):
 *   1. gf_slab_halfsweep_border(p, omega): the parity-p sites of slices 0 and lt-1; the t = 0 sites update ghost[1-p];
 *      then top_out <- U_t of the parity-p sites of the top slice (just updated).
 *   2. gf_slab_halfsweep_interior(p, omega): slices 1 .. lt-2; touches no link of step 3, so the transport may run
 *      beside it on another stream.
 *   3. transport: ghost[1-p] -> lower neighbour's top_in;  top_out -> upper neighbour's ghost[p].
 *   4. gf_slab_unpack_top(1-p): top_in -> U_t of the parity-(1-p) sites of the top slice.
 * Before the first half-sweep (after gf_set_links, gf_reunitarize): for q = 0, 1: gf_slab_pack_top(q), transport
 * top_out -> upper neighbour's ghost[q].
 * On a slab context gf_measure returns the slab's own F and theta (the global values are the means over the R
 * equal slabs); gf_ovr_sweep and gf_fix return GF_EINVAL, the gf_fft_* calls GF_EUNSUPPORTED (the paper has no
 * multi-GPU Algorithm 2 either).  With R = 1 (the slab is its own neighbour) the calls reproduce
 * gf_ovr_sweep bit for bit.  All Async.  Errors: GF_EINVAL (no halo attached, parity not 0/1, omega), GF_ENOMEM,
 * GF_ECUDA.
 *
 * Direct delivery (gf_slab_set_targets): where the neighbours' halo workspaces are addressable from this device (slabs
 * of the same process; peer-mapped memory of another GPU over NVLink), the border kernel itself stores the two
 * messages at their destination — the top-slice sites write their new U_t(x) into the upper neighbour's ghost[p]
 * (instead of top_out), the t = 0 sites write the updated ghost links into the lower neighbour's top_in as well as
 * into ghost[1-p] — and step 3 disappears; the caller only orders the kernels: a neighbour's border kernel of this
 * half-sweep must have finished before gf_slab_unpack_top(1-p) and before the next half-sweep's border kernel, and a
 * slab's unpack before a neighbour's next border kernel.  Pass the three pointers of the neighbours' workspaces (upper:
 * offset 0 and B, lower: offset 3B), or three nulls to go back to top_out.  gf_slab_pack_top then writes to the upper
 * neighbour's ghost[parity] too. */
/* Between PROCESSES (one per GPU) the neighbours' workspaces are mapped with CUDA IPC and handed to
 * gf_slab_set_peer_targets: as gf_slab_set_targets, but the "ret" message of the even half-sweep goes to
 * lower_top_in_even (the lower neighbour's workspace + 3B) and that of the odd half-sweep to lower_top_in_odd (its
 * workspace + 2B, the top_out slot, unused when messages are delivered directly), and gf_slab_unpack_top(1-p) reads the
 * buffer half-sweep p filled.  With top_in double-buffered ONE synchronisation of neighbouring ranks per half-sweep is
 * enough: between the border kernels (all messages stored) and gf_slab_unpack_top; a rank's next border kernel only
 * writes buffers whose last readers ran before that point.
 *   gf_ipc_export: a 64-byte CUDA IPC handle of the allocation dev_ptr lies in, and dev_ptr's offset in it (host out).
 *   gf_ipc_open:   maps that allocation in this process; *dev_ptr = its base + offset.  gf_ipc_close unmaps it.
 * Errors: GF_EINVAL (null), GF_ECUDA (not a cudaMalloc allocation, same process, no peer access). */
int gf_slab_set_peer_targets(gf_ctx* ctx, void* upper_ghost0, void* upper_ghost1, void* lower_top_in_even,
                             void* lower_top_in_odd);
int gf_ipc_export(const void* dev_ptr, unsigned char* handle64, size_t* offset);
int gf_ipc_open(const unsigned char* handle64, size_t offset, void** dev_ptr);
int gf_ipc_close(void* dev_ptr, size_t offset);

/* The whole sharded sweep behind one call, synchronised with the neighbours by flags instead of host waits or
 * collectives.  gf_slab_set_peer_flags: own_flags = 32 bytes (32-byte aligned) of this slab's device memory (inside the allocation that is
 * exported with gf_ipc_export, e.g. behind the 4B bytes of the halo workspace); upper_flag = the address of the UPPER
 * neighbour's own_flags + 4 (its "written by my lower neighbour" word), lower_flag = the LOWER neighbour's own_flags + 0;
 * addresses of this process or CUDA-IPC mappings.  A slab signals by a stream-ordered 32-bit write of an epoch counter
 * into both neighbours' words (cuStreamWriteValue32, after the kernels queued before it) and waits by a stream-ordered
 * compare (cuStreamWaitValue32, >=) on its own two words: no kernel spins, no host thread waits.  The call zeroes own_flags
 * and synchronises the stream; every slab of a lattice must have made it before any of them is swept.
 * gf_slab_group_sweep(slabs, n, n_sweeps, omega, reunit_every, sweeps_before): n_sweeps sweeps of the n local slabs (all
 * with peer targets and flags set; neighbours inside or outside the group): per half-sweep p ONE kernel per slab - its
 * border blocks come first, store both halo messages at their destination, and the last of them adds 1 to the arrival
 * counter each neighbour keeps for it (the upper neighbour's own_flags + 16 "from below", the lower one's own_flags + 12
 * "from above"; system-scope atomics) while the rest of the grid updates the interior -, then two stream-ordered waits
 * of the slab, one on each of its own two counters (one counter per neighbour: a sum of the two could be reached by one
 * neighbour running a launch ahead while the other has not arrived), and gf_slab_unpack_top(1-p); after global sweep number s =
 * sweeps_before + i with reunit_every > 0 and s % reunit_every == 0 every link is reunitarised and the ghost buffers are
 * refreshed.  Asynchronous.  EVERY rank of the lattice must make the same call (same n_sweeps, reunit
 * cadence), else the waits never complete.  gf_slab_group_refresh: fills the neighbours' ghost buffers from the group's top
 * slices (after gf_set_links on the slabs).  Errors: GF_EINVAL (slab without peer targets / flags, slabs at different
 * epochs, bad omega), GF_ECUDA (stream memory operations unavailable). */
int gf_slab_set_peer_flags(gf_ctx* ctx, void* own_flags, void* upper_flag, void* lower_flag);
int gf_slab_group_sweep(gf_ctx* const* slabs, int n_slabs, int n_sweeps, double omega, int reunit_every,
                        long long sweeps_before);
int gf_slab_group_refresh(gf_ctx* const* slabs, int n_slabs);

/* The driver's decisions of Algorithm 1 for callers that run it over several contexts:
 *   gf_combine_slabs: global F and theta from the gf_measure values of n_slabs equal slabs (host arrays, slab order):
 *     their means, added in slab order so that every rank gets the same bits.  GF_ENUMERIC if not finite.
 *   gf_fix_plan: *n_next = the number of sweeps to do before the next measurement - 0 when theta < eps or
 *     sweeps_done >= max_sweeps (stop), else min(check_every, max_sweeps - sweeps_done); validates omega in [1,2),
 *     check_every >= 1, max_sweeps >= 0, eps >= 0 as gf_fix does (GF_EINVAL). */
int gf_combine_slabs(const double* F_slab, const double* theta_slab, int n_slabs, double* F, double* theta);
int gf_fix_plan(double omega, double eps, int max_sweeps, int check_every, int sweeps_done, double theta, int* n_next);

size_t gf_slab_halo_bytes(const gf_ctx* ctx);
int gf_slab_set_targets(gf_ctx* ctx, void* upper_ghost0, void* upper_ghost1, void* lower_top_in);
int gf_slab_attach(gf_ctx* ctx, void* dev_halo, size_t halo_workspace_bytes);
int gf_slab_pack_top(gf_ctx* ctx, int parity);
int gf_slab_unpack_top(gf_ctx* ctx, int parity);
int gf_slab_halfsweep_border(gf_ctx* ctx, int parity, double omega);
int gf_slab_halfsweep_interior(gf_ctx* ctx, int parity, double omega);

/* Number of kernels this context has launched since gf_create (for benchmark bookkeeping). */
long long gf_kernel_launches(const gf_ctx* ctx);

/* Measurement aid, not a step of the method (the flops leg of the roofline needs a MEASURED FP64 / FP32
 * CUDA-core peak): runs a register-only FMA-chain kernel (16 independent chains per thread, 2048 threads per SM asked
 * for) on the current device for about seconds_target seconds (0 < seconds_target <= 10) and writes the achieved
 * TFLOP/s (FMA = 2 flop) of precision prec (GF_FP64: DFMA, GF_FP32: FFMA) to *tflops (host).  dev_scratch: at least 8
 * bytes of device memory (never written in practice).  Synchronises cuda_stream.  Errors: GF_EINVAL, GF_ECUDA. */
int gf_peak_fma(int prec, double seconds_target, void* dev_scratch, void* cuda_stream, double* tflops);

/* ---- F and theta for callers that cannot allocate device memory -----------------------------------------------------------
 * Every call above works out of a workspace that the caller allocated for gf_create.  A caller with no means to get
 * device memory - a hook inside an application whose own pool has taken the whole GPU, code that runs under a rule of
 * "no cudaMalloc / cudaFree after start-up" because those calls synchronise the device and stall its other streams, a
 * callback that is only lent a pointer to somebody else's field - cannot create a context at all.  gf_measure_static
 * gives that caller the convergence monitor of Algorithm 1 (eqs. 1.1-1.3; Alg. 1 l.1, l.13): F and theta
 * of a field in the CANONICAL layout (top of this file), read where it lies, with no context and no workspace.  The
 * scratch of the reduction (one pair of partial sums per 256 sites, the result, a block counter) is a fixed array
 * inside the library image, 256 KiB on every GPU that loads libgf, held until the process exits.
 *
 *   dev_links    device memory of the CURRENT device, canonical layout, 72 V elements of double (GF_FP64) or float
 *                (GF_FP32), 16-byte aligned; only read.
 *   gauge        GF_LANDAU (nu = 0..3) or GF_COULOMB (nu = 0..2), as gf_create.
 *   cuda_stream  the stream the work is queued on (NULL = default stream); the call synchronises it before returning.
 *   F, theta     host out-params, FP64 sums in both precisions, deterministic summation order (not gf_measure's order:
 *                the two agree to rounding, not bit for bit).
 * Limits and rules:
 *   - V <= gf_measure_static_max_sites() = 4 194 304 sites (32^3 x 128 just fits, 48^3 x 96 does not); a larger lattice is refused with
 *     GF_ENOMEM and a message that says so: use gf_create + gf_measure there.
 *   - The call allocates nothing: no cudaMalloc, cudaMallocHost, cudaFree, no library routine that does.
 *   - The first call on each device looks up the array's device address (cudaGetSymbolAddress, which may make the
 *     runtime load the library's kernels onto that device); later calls reuse it.  Make that first call at start-up,
 *     before any stream capture is begun.
 *   - All calls on one device share the array, and it keeps what the last call left in it (the counter is cleared at the
 *     start of every call).  Two calls that overlap on the GPU - from two threads, or on two streams - race on it and
 *     both results are garbage: serialise them.  Calls on different devices are independent.
 * Errors (text of the last failure of the calling thread: gf_static_last_error): GF_EINVAL (null or misaligned
 * pointer, memory that is not the current device's), GF_EODD, GF_EUNSUPPORTED (gauge, precision), GF_ENOMEM (lattice
 * above the limit), GF_ECUDA, GF_ENUMERIC (F or theta not finite; the values are still written). */
size_t gf_measure_static_max_sites(void);
int gf_measure_static(const void* dev_links, int nx, int ny, int nz, int nt, int gauge, int prec, void* cuda_stream,
                      double* F, double* theta);
const char* gf_static_last_error(void);

void gf_destroy(gf_ctx* ctx);
const char* gf_strerror(int code);
/* Text of the last failure on this context (CUDA error string for GF_ECUDA); valid until the next call. */
const char* gf_last_error(const gf_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* GF_H */
