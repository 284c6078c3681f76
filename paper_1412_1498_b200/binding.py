"""Thin ctypes binding of libgf (include/gf.h).  Argument marshalling only: every step of the hot path runs in the
CUDA kernels behind the C ABI.  PyTorch is used for device memory and streams, nothing else.

The module-level functions carry the C names (gf_create, gf_set_links, gf_ovr_sweep, gf_measure, gf_fix,
gf_get_links, ...) and take raw pointers / ints; `GaugeFixer` is a small convenience owner of a context plus the torch
workspace tensor it lives in.  There is no CPU fallback: if libgf.so cannot be built or loaded, importing fails.
"""
from __future__ import annotations

import ctypes
from ctypes import POINTER, byref, c_char_p, c_double, c_int, c_longlong, c_size_t, c_void_p

from . import build as _build

GF_LANDAU, GF_COULOMB = 0, 1
GF_FP64, GF_FP32 = 0, 1
GF_OK, GF_EINVAL, GF_EODD, GF_EUNSUPPORTED, GF_ENOMEM, GF_ECUDA, GF_ENUMERIC = 0, -1, -2, -3, -4, -5, -6
GF_OPT_SWEEP_VARIANT, GF_OPT_BLOCK_THREADS, GF_OPT_FUSE_MEASURE, GF_OPT_FFT_ACCELERATE, GF_OPT_FFT_FUSED_T = 1, 2, 3, 4, 5
GF_OPT_FFT_OWN, GF_OPT_OVR_SERIES, GF_OPT_DOMAIN8_CHECK, GF_OPT_SLAB_FORCE_FLAGS = 6, 7, 8, 9

SYMBOLS = ["gf_workspace_bytes", "gf_create", "gf_set_links", "gf_get_links", "gf_set_links_host",
           "gf_get_links_host", "gf_ovr_sweep", "gf_measure", "gf_fix", "gf_get_history", "gf_reunitarize",
           "gf_set_reunit_every", "gf_set_option", "gf_kernel_launches", "gf_destroy", "gf_strerror", "gf_last_error",
           "gf_fft_workspace_bytes", "gf_fft_attach", "gf_fft_step", "gf_fix_fft",
           "gf_measure_slices", "gf_fix_slices", "gf_defer_bytes", "gf_defer_attach", "gf_defer_flush",
           "gf_slab_halo_bytes", "gf_slab_attach", "gf_slab_set_targets", "gf_slab_pack_top", "gf_slab_unpack_top",
           "gf_slab_halfsweep_border", "gf_slab_halfsweep_interior", "gf_peak_fma", "gf_workspace_bytes_sun",
           "gf_create_sun", "gf_slab_set_peer_targets", "gf_ipc_export", "gf_ipc_open", "gf_ipc_close", "gf_combine_slabs",
           "gf_fix_plan", "gf_slab_set_peer_flags", "gf_slab_group_sweep", "gf_slab_group_refresh",
           "gf_measure_static", "gf_measure_static_max_sites", "gf_static_last_error"]


def _load() -> ctypes.CDLL:
    lib = ctypes.CDLL(_build.build())
    lib.gf_workspace_bytes.restype = c_size_t
    lib.gf_workspace_bytes.argtypes = [c_int] * 6
    lib.gf_create.restype = c_int
    lib.gf_create.argtypes = [POINTER(c_void_p)] + [c_int] * 7 + [c_void_p, c_size_t, c_void_p]
    lib.gf_workspace_bytes_sun.restype = c_size_t
    lib.gf_workspace_bytes_sun.argtypes = [c_int] * 6
    lib.gf_create_sun.restype = c_int
    lib.gf_create_sun.argtypes = [POINTER(c_void_p)] + [c_int] * 7 + [c_void_p, c_size_t, c_void_p]
    for name in ("gf_set_links", "gf_get_links", "gf_set_links_host", "gf_get_links_host"):
        getattr(lib, name).restype = c_int
        getattr(lib, name).argtypes = [c_void_p, c_void_p]
    lib.gf_ovr_sweep.restype = c_int
    lib.gf_ovr_sweep.argtypes = [c_void_p, c_int, c_double]
    lib.gf_measure.restype = c_int
    lib.gf_measure.argtypes = [c_void_p, POINTER(c_double), POINTER(c_double)]
    lib.gf_fix.restype = c_int
    lib.gf_fix.argtypes = [c_void_p, c_double, c_double, c_int, c_int, POINTER(c_int)]
    lib.gf_get_history.restype = c_int
    lib.gf_get_history.argtypes = [c_void_p, POINTER(c_double), c_int, POINTER(c_int)]
    lib.gf_reunitarize.restype = c_int
    lib.gf_reunitarize.argtypes = [c_void_p]
    lib.gf_set_reunit_every.restype = c_int
    lib.gf_set_reunit_every.argtypes = [c_void_p, c_int]
    lib.gf_set_option.restype = c_int
    lib.gf_set_option.argtypes = [c_void_p, c_int, c_int]
    lib.gf_fft_workspace_bytes.restype = c_int
    lib.gf_fft_workspace_bytes.argtypes = [c_void_p, POINTER(c_size_t)]
    lib.gf_fft_attach.restype = c_int
    lib.gf_fft_attach.argtypes = [c_void_p, c_void_p, c_size_t]
    lib.gf_fft_step.restype = c_int
    lib.gf_fft_step.argtypes = [c_void_p, c_int, c_double]
    lib.gf_fix_fft.restype = c_int
    lib.gf_fix_fft.argtypes = [c_void_p, c_double, c_double, c_int, c_int, POINTER(c_int)]
    lib.gf_measure_slices.restype = c_int
    lib.gf_measure_slices.argtypes = [c_void_p, POINTER(c_double), POINTER(c_double)]
    lib.gf_fix_slices.restype = c_int
    lib.gf_fix_slices.argtypes = [c_void_p, c_double, c_double, c_int, c_int, POINTER(c_int), POINTER(c_int)]
    lib.gf_defer_bytes.restype = c_size_t
    lib.gf_defer_bytes.argtypes = [c_void_p]
    lib.gf_defer_attach.restype = c_int
    lib.gf_defer_attach.argtypes = [c_void_p, c_void_p, c_size_t]
    lib.gf_defer_flush.restype = c_int
    lib.gf_defer_flush.argtypes = [c_void_p]
    lib.gf_slab_halo_bytes.restype = c_size_t
    lib.gf_slab_halo_bytes.argtypes = [c_void_p]
    lib.gf_slab_attach.restype = c_int
    lib.gf_slab_attach.argtypes = [c_void_p, c_void_p, c_size_t]
    lib.gf_slab_set_targets.restype = c_int
    lib.gf_slab_set_targets.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p]
    for name in ("gf_slab_pack_top", "gf_slab_unpack_top"):
        getattr(lib, name).restype = c_int
        getattr(lib, name).argtypes = [c_void_p, c_int]
    for name in ("gf_slab_halfsweep_border", "gf_slab_halfsweep_interior"):
        getattr(lib, name).restype = c_int
        getattr(lib, name).argtypes = [c_void_p, c_int, c_double]
    lib.gf_slab_set_peer_targets.restype = c_int
    lib.gf_slab_set_peer_targets.argtypes = [c_void_p] * 5
    lib.gf_slab_set_peer_flags.restype = c_int
    lib.gf_slab_set_peer_flags.argtypes = [c_void_p] * 4
    lib.gf_slab_group_sweep.restype = c_int
    lib.gf_slab_group_sweep.argtypes = [POINTER(c_void_p), c_int, c_int, c_double, c_int, c_longlong]
    lib.gf_slab_group_refresh.restype = c_int
    lib.gf_slab_group_refresh.argtypes = [POINTER(c_void_p), c_int]
    lib.gf_ipc_export.restype = c_int
    lib.gf_ipc_export.argtypes = [c_void_p, c_char_p, POINTER(c_size_t)]
    lib.gf_ipc_open.restype = c_int
    lib.gf_ipc_open.argtypes = [c_char_p, c_size_t, POINTER(c_void_p)]
    lib.gf_ipc_close.restype = c_int
    lib.gf_ipc_close.argtypes = [c_void_p, c_size_t]
    lib.gf_combine_slabs.restype = c_int
    lib.gf_combine_slabs.argtypes = [POINTER(c_double), POINTER(c_double), c_int, POINTER(c_double), POINTER(c_double)]
    lib.gf_fix_plan.restype = c_int
    lib.gf_fix_plan.argtypes = [c_double, c_double, c_int, c_int, c_int, c_double, POINTER(c_int)]
    lib.gf_peak_fma.restype = c_int
    lib.gf_peak_fma.argtypes = [c_int, c_double, c_void_p, c_void_p, POINTER(c_double)]
    lib.gf_measure_static.restype = c_int
    lib.gf_measure_static.argtypes = [c_void_p] + [c_int] * 6 + [c_void_p, POINTER(c_double), POINTER(c_double)]
    lib.gf_measure_static_max_sites.restype = c_size_t
    lib.gf_measure_static_max_sites.argtypes = []
    lib.gf_static_last_error.restype = c_char_p
    lib.gf_static_last_error.argtypes = []
    lib.gf_kernel_launches.restype = c_longlong
    lib.gf_kernel_launches.argtypes = [c_void_p]
    lib.gf_destroy.restype = None
    lib.gf_destroy.argtypes = [c_void_p]
    lib.gf_strerror.restype = c_char_p
    lib.gf_strerror.argtypes = [c_int]
    lib.gf_last_error.restype = c_char_p
    lib.gf_last_error.argtypes = [c_void_p]
    return lib


lib = _load()


class GFError(RuntimeError):
    def __init__(self, code: int, detail: str = ""):
        self.code = code
        msg = lib.gf_strerror(code).decode()
        super().__init__(f"libgf error {code} ({msg})" + (f": {detail}" if detail else ""))


# ---- the C ABI, same names, raw arguments (return codes are returned, not raised) -------------------------------------
def gf_workspace_bytes(nx, ny, nz, nt, prec, storage) -> int:
    return int(lib.gf_workspace_bytes(nx, ny, nz, nt, prec, storage))


def gf_create(nx, ny, nz, nt, gauge, prec, storage, dev_workspace: int, workspace_bytes: int, cuda_stream: int):
    """Returns (rc, ctx_handle)."""
    h = c_void_p()
    rc = lib.gf_create(byref(h), nx, ny, nz, nt, gauge, prec, storage, c_void_p(dev_workspace), workspace_bytes,
                       c_void_p(cuda_stream))
    return rc, h


def gf_workspace_bytes_sun(ncolors, nx, ny, nz, nt, prec) -> int:
    return int(lib.gf_workspace_bytes_sun(ncolors, nx, ny, nz, nt, prec))


def gf_create_sun(ncolors, nx, ny, nz, nt, gauge, prec, dev_workspace: int, workspace_bytes: int, cuda_stream: int):
    """Returns (rc, ctx_handle)."""
    h = c_void_p()
    rc = lib.gf_create_sun(byref(h), ncolors, nx, ny, nz, nt, gauge, prec, c_void_p(dev_workspace), workspace_bytes,
                           c_void_p(cuda_stream))
    return rc, h


def gf_set_links(ctx, dev_links: int) -> int:
    return lib.gf_set_links(ctx, c_void_p(dev_links))


def gf_get_links(ctx, dev_links_out: int) -> int:
    return lib.gf_get_links(ctx, c_void_p(dev_links_out))


def gf_set_links_host(ctx, host_links: int) -> int:
    return lib.gf_set_links_host(ctx, c_void_p(host_links))


def gf_get_links_host(ctx, host_links_out: int) -> int:
    return lib.gf_get_links_host(ctx, c_void_p(host_links_out))


def gf_ovr_sweep(ctx, n: int, omega: float) -> int:
    return lib.gf_ovr_sweep(ctx, n, omega)


def gf_measure(ctx):
    """Returns (rc, F, theta)."""
    F, th = c_double(), c_double()
    rc = lib.gf_measure(ctx, byref(F), byref(th))
    return rc, F.value, th.value


def gf_fix(ctx, omega: float, eps: float, max_sweeps: int, check_every: int):
    """Returns (rc, sweeps_done)."""
    done = c_int()
    rc = lib.gf_fix(ctx, omega, eps, max_sweeps, check_every, byref(done))
    return rc, done.value


def gf_get_history(ctx, cap: int = 100000):
    """Returns (rc, [(sweep, F, theta), ...])."""
    buf = (c_double * (3 * cap))()
    n = c_int()
    rc = lib.gf_get_history(ctx, buf, cap, byref(n))
    m = min(n.value, cap)
    return rc, [(int(buf[3 * i]), buf[3 * i + 1], buf[3 * i + 2]) for i in range(m)]


def gf_reunitarize(ctx) -> int:
    return lib.gf_reunitarize(ctx)


def gf_set_reunit_every(ctx, k: int) -> int:
    return lib.gf_set_reunit_every(ctx, k)


def gf_set_option(ctx, key: int, value: int) -> int:
    return lib.gf_set_option(ctx, key, value)


def gf_fft_workspace_bytes(ctx):
    """Returns (rc, bytes)."""
    n = c_size_t()
    rc = lib.gf_fft_workspace_bytes(ctx, byref(n))
    return rc, int(n.value)


def gf_fft_attach(ctx, dev_workspace: int, workspace_bytes: int) -> int:
    return lib.gf_fft_attach(ctx, c_void_p(dev_workspace), workspace_bytes)


def gf_fft_step(ctx, n: int, alpha: float) -> int:
    return lib.gf_fft_step(ctx, n, alpha)


def gf_fix_fft(ctx, alpha: float, eps: float, max_iters: int, check_every: int):
    """Returns (rc, iterations_done)."""
    done = c_int()
    rc = lib.gf_fix_fft(ctx, alpha, eps, max_iters, check_every, byref(done))
    return rc, done.value


def gf_measure_slices(ctx, nt: int):
    """Returns (rc, [F_t], [theta_t])."""
    F, th = (c_double * nt)(), (c_double * nt)()
    rc = lib.gf_measure_slices(ctx, F, th)
    return rc, list(F), list(th)


def gf_fix_slices(ctx, omega: float, eps: float, max_sweeps: int, check_every: int, nt: int):
    """Returns (rc, sweeps_done, [sweeps spent on slice t])."""
    done = c_int()
    per = (c_int * nt)()
    rc = lib.gf_fix_slices(ctx, omega, eps, max_sweeps, check_every, byref(done), per)
    return rc, done.value, list(per)


def gf_defer_bytes(ctx) -> int:
    return int(lib.gf_defer_bytes(ctx))


def gf_defer_attach(ctx, dev_acc: int, nbytes: int) -> int:
    return lib.gf_defer_attach(ctx, c_void_p(dev_acc or None), nbytes)


def gf_defer_flush(ctx) -> int:
    return lib.gf_defer_flush(ctx)


def gf_slab_halo_bytes(ctx) -> int:
    return int(lib.gf_slab_halo_bytes(ctx))


def gf_slab_attach(ctx, dev_halo: int, halo_workspace_bytes: int) -> int:
    return lib.gf_slab_attach(ctx, c_void_p(dev_halo), halo_workspace_bytes)


def gf_slab_set_targets(ctx, upper_ghost0: int, upper_ghost1: int, lower_top_in: int) -> int:
    return lib.gf_slab_set_targets(ctx, c_void_p(upper_ghost0 or None), c_void_p(upper_ghost1 or None),
                                   c_void_p(lower_top_in or None))


def gf_slab_set_peer_targets(ctx, upper_ghost0: int, upper_ghost1: int, lower_top_in_even: int, lower_top_in_odd: int) -> int:
    return lib.gf_slab_set_peer_targets(ctx, c_void_p(upper_ghost0), c_void_p(upper_ghost1), c_void_p(lower_top_in_even),
                                        c_void_p(lower_top_in_odd))


def gf_slab_set_peer_flags(ctx, own_flags: int, upper_flag: int, lower_flag: int) -> int:
    return lib.gf_slab_set_peer_flags(ctx, c_void_p(own_flags), c_void_p(upper_flag), c_void_p(lower_flag))


def _ctx_array(ctxs):
    return (c_void_p * len(ctxs))(*[c.value if isinstance(c, c_void_p) else c for c in ctxs])


def gf_slab_group_sweep(ctxs, n_sweeps: int, omega: float, reunit_every: int = 0, sweeps_before: int = 0) -> int:
    return lib.gf_slab_group_sweep(_ctx_array(ctxs), len(ctxs), n_sweeps, omega, reunit_every, sweeps_before)


def gf_slab_group_refresh(ctxs) -> int:
    return lib.gf_slab_group_refresh(_ctx_array(ctxs), len(ctxs))


def gf_ipc_export(dev_ptr: int):
    """Returns (rc, 64-byte handle, offset)."""
    buf = ctypes.create_string_buffer(64)
    off = c_size_t()
    rc = lib.gf_ipc_export(c_void_p(dev_ptr), buf, byref(off))
    return rc, buf.raw, off.value


def gf_ipc_open(handle: bytes, offset: int):
    """Returns (rc, device pointer)."""
    p = c_void_p()
    rc = lib.gf_ipc_open(handle, offset, byref(p))
    return rc, (p.value or 0)


def gf_ipc_close(dev_ptr: int, offset: int) -> int:
    return lib.gf_ipc_close(c_void_p(dev_ptr), offset)


def gf_combine_slabs(F_slab, theta_slab):
    """Returns (rc, F, theta)."""
    n = len(F_slab)
    Fa, ta = (c_double * n)(*F_slab), (c_double * n)(*theta_slab)
    F, th = c_double(), c_double()
    rc = lib.gf_combine_slabs(Fa, ta, n, byref(F), byref(th))
    return rc, F.value, th.value


def gf_fix_plan(omega, eps, max_sweeps, check_every, sweeps_done, theta):
    """Returns (rc, n_next)."""
    n = c_int()
    rc = lib.gf_fix_plan(omega, eps, max_sweeps, check_every, sweeps_done, theta, byref(n))
    return rc, n.value


def gf_slab_pack_top(ctx, parity: int) -> int:
    return lib.gf_slab_pack_top(ctx, parity)


def gf_slab_unpack_top(ctx, parity: int) -> int:
    return lib.gf_slab_unpack_top(ctx, parity)


def gf_slab_halfsweep_border(ctx, parity: int, omega: float) -> int:
    return lib.gf_slab_halfsweep_border(ctx, parity, omega)


def gf_slab_halfsweep_interior(ctx, parity: int, omega: float) -> int:
    return lib.gf_slab_halfsweep_interior(ctx, parity, omega)


def gf_peak_fma(prec: int, seconds_target: float, dev_scratch: int, stream: int = 0):
    """Returns (rc, TFLOP/s) of the FMA-chain micro-kernel on the current device."""
    t = c_double()
    rc = lib.gf_peak_fma(prec, seconds_target, c_void_p(dev_scratch), c_void_p(stream or None), byref(t))
    return rc, t.value


def gf_measure_static(dev_links: int, nx, ny, nz, nt, gauge: int, prec: int, stream: int = 0):
    """Returns (rc, F, theta) of a canonical-layout device field; no context, no workspace, no allocation."""
    F, th = c_double(), c_double()
    rc = lib.gf_measure_static(c_void_p(dev_links or None), nx, ny, nz, nt, gauge, prec, c_void_p(stream or None),
                               byref(F), byref(th))
    return rc, F.value, th.value


def gf_measure_static_max_sites() -> int:
    return int(lib.gf_measure_static_max_sites())


def gf_static_last_error() -> str:
    return lib.gf_static_last_error().decode()


def gf_kernel_launches(ctx) -> int:
    return int(lib.gf_kernel_launches(ctx))


def gf_destroy(ctx) -> None:
    lib.gf_destroy(ctx)


def gf_strerror(code: int) -> str:
    return lib.gf_strerror(code).decode()


def gf_last_error(ctx) -> str:
    return lib.gf_last_error(ctx).decode()


# ---- convenience owner ---------------------------------------------------------------------------------------------------
_GAUGE = {"landau": GF_LANDAU, "coulomb": GF_COULOMB}
_PREC = {"f64": GF_FP64, "f32": GF_FP32}


def measure_static(links, dims, gauge="landau", stream=None):
    """F and theta of a torch CUDA tensor in the canonical layout (V,4,3,3,2), float64 or float32, through
    gf_measure_static: for callers that hold a field but may not allocate device memory.  Nothing is allocated here
    either (no context, no workspace tensor); lattices above gf_measure_static_max_sites() sites raise GFError."""
    import torch

    assert links.is_cuda and links.is_contiguous() and links.dtype in (torch.float64, torch.float32)
    prec = GF_FP64 if links.dtype == torch.float64 else GF_FP32
    with torch.cuda.device(links.device):
        s = stream if stream is not None else torch.cuda.current_stream(links.device)
        rc, F, th = gf_measure_static(links.data_ptr(), *[int(d) for d in dims], _GAUGE[gauge], prec, s.cuda_stream)
    if rc != GF_OK:
        raise GFError(rc, gf_static_last_error())
    return F, th


class GaugeFixer:
    """Owns a gf_ctx and the torch workspace tensor behind it.  All methods marshal arguments and check return codes."""

    def __init__(self, dims, gauge="landau", prec="f64", storage=18, device="cuda:0", stream=None, ncolors=3):
        import torch

        self.torch = torch
        self.dims = tuple(int(d) for d in dims)
        self.gauge, self.prec, self.storage = gauge, prec, int(storage)
        self.ncolors = int(ncolors)  # 3: gf_create; 2 or 4: gf_create_sun (all N^2 entries stored)
        self.device = torch.device(device)
        self.dtype = torch.float64 if prec == "f64" else torch.float32
        self.volume = 1
        for d in self.dims:
            self.volume *= d
        if self.ncolors == 3:
            nbytes = gf_workspace_bytes(*self.dims, _PREC[prec], self.storage)
        else:
            nbytes = gf_workspace_bytes_sun(self.ncolors, *self.dims, _PREC[prec])
        if nbytes == 0:
            # let gf_create produce the precise error code
            nbytes = 256
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self.workspace = self._alloc(nbytes)
            if self.ncolors == 3:
                rc, self.ctx = gf_create(*self.dims, _GAUGE[gauge], _PREC[prec], self.storage, self.workspace.data_ptr(),
                                         nbytes, self.stream.cuda_stream)
            else:
                rc, self.ctx = gf_create_sun(self.ncolors, *self.dims, _GAUGE[gauge], _PREC[prec],
                                             self.workspace.data_ptr(), nbytes, self.stream.cuda_stream)
        if rc != GF_OK:
            self.ctx = None
            raise GFError(rc)

    def _alloc(self, nbytes):
        """Device bytes the library will use on self.stream: allocated under that stream, so that the caching
        allocator ties the block to it (a block freed later is not handed to another stream while kernels of this
        one may still be running on it)."""
        torch = self.torch
        with torch.cuda.device(self.device), torch.cuda.stream(self.stream):
            return torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=self.device)

    def _check(self, rc):
        if rc != GF_OK:
            raise GFError(rc, gf_last_error(self.ctx))

    def new_links_buffer(self):
        """An uninitialised device tensor in the canonical layout (V,4,N,N,2)."""
        return self.torch.empty((self.volume, 4, self.ncolors, self.ncolors, 2), dtype=self.dtype, device=self.device)

    def set_links(self, links):
        assert links.is_cuda and links.is_contiguous() and links.dtype == self.dtype and links.numel() == self.volume * 8 * self.ncolors ** 2
        self._check(gf_set_links(self.ctx, links.data_ptr()))

    def get_links(self, out=None):
        if out is None:
            out = self.new_links_buffer()
        assert out.is_cuda and out.is_contiguous() and out.dtype == self.dtype and out.numel() == self.volume * 8 * self.ncolors ** 2
        self._check(gf_get_links(self.ctx, out.data_ptr()))
        return out

    def set_links_host(self, links):
        """links: CPU torch tensor or numpy array (pinned memory recommended), canonical layout."""
        ptr = links.data_ptr() if hasattr(links, "data_ptr") else links.ctypes.data
        self._check(gf_set_links_host(self.ctx, ptr))

    def get_links_host(self, out):
        ptr = out.data_ptr() if hasattr(out, "data_ptr") else out.ctypes.data
        self._check(gf_get_links_host(self.ctx, ptr))
        return out

    def ovr_sweep(self, n, omega):
        self._check(gf_ovr_sweep(self.ctx, int(n), float(omega)))

    def measure(self):
        rc, F, th = gf_measure(self.ctx)
        self._check(rc)
        return F, th

    def fix(self, omega, eps, max_sweeps, check_every):
        rc, done = gf_fix(self.ctx, float(omega), float(eps), int(max_sweeps), int(check_every))
        self._check(rc)
        return done

    def defer_temporal_links(self, on=True):
        """Coulomb gauge: keep the sites' accumulated rotations instead of rewriting the temporal links every update."""
        if on:
            n = gf_defer_bytes(self.ctx)
            self.defer_buffer = self._alloc(n)
            self._check(gf_defer_attach(self.ctx, self.defer_buffer.data_ptr(), n))
        else:
            self._check(gf_defer_attach(self.ctx, 0, 0))
            self.defer_buffer = None

    def defer_flush(self):
        self._check(gf_defer_flush(self.ctx))

    def measure_slices(self):
        rc, F, th = gf_measure_slices(self.ctx, self.dims[3])
        self._check(rc)
        return F, th

    def fix_slices(self, omega, eps, max_sweeps, check_every):
        """Coulomb gauge, a stop test per time slice.  Returns (sweeps_done, sweeps spent on each slice)."""
        rc, done, per = gf_fix_slices(self.ctx, float(omega), float(eps), int(max_sweeps), int(check_every), self.dims[3])
        self._check(rc)
        return done, per

    def history(self):
        rc, h = gf_get_history(self.ctx)
        self._check(rc)
        return h

    def reunitarize(self):
        self._check(gf_reunitarize(self.ctx))

    def set_reunit_every(self, k):
        self._check(gf_set_reunit_every(self.ctx, int(k)))

    def set_option(self, key, value):
        self._check(gf_set_option(self.ctx, int(key), int(value)))

    def fft_attach(self):
        """Allocate (torch) and hand over the second workspace Algorithm 2 needs.  Idempotent."""
        if getattr(self, "fft_workspace", None) is not None:
            return
        rc, nbytes = gf_fft_workspace_bytes(self.ctx)
        self._check(rc)
        self.fft_workspace = self._alloc(nbytes)
        self._check(gf_fft_attach(self.ctx, self.fft_workspace.data_ptr(), nbytes))

    def fft_step(self, n, alpha):
        self.fft_attach()
        self._check(gf_fft_step(self.ctx, int(n), float(alpha)))

    def fix_fft(self, alpha, eps, max_iters, check_every=1):
        self.fft_attach()
        rc, done = gf_fix_fft(self.ctx, float(alpha), float(eps), int(max_iters), int(check_every))
        self._check(rc)
        return done

    def kernel_launches(self):
        return gf_kernel_launches(self.ctx)

    def close(self):
        if getattr(self, "ctx", None):
            self.stream.synchronize()  # nothing of this context is in flight when its memory goes back to torch
            gf_destroy(self.ctx)
            self.ctx = None
            self.workspace = None
            self.fft_workspace = None
            self.defer_buffer = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
