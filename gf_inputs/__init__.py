"""Seeded synthetic SU(3) gauge fields — the ONLY module shared by the oracle-side and the CUDA-side tests.

It holds none of the gauge-fixing method's arithmetic; it only fabricates inputs (recipe: gen_core.h, after
BASELINE.json "configs" and SURVEY.md §8(d)).  The fields stand in for the MILC production configurations the paper
measured on, which are not available.

    U_mu(x) = G(x) exp(i r H_mu(x)) G(x+mu)^dagger,   H Gaussian in the Gell-Mann basis, G Haar SU(3).

Canonical layout everywhere: links[site][mu][row][col][re,im], site = x + nx*(y + ny*(z + nz*t)), mu=0..3=(x,y,z,t).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_CPU_SO = os.path.join(_HERE, "libgfinputs_cpu.so")
_CUDA_SO = os.path.join(_HERE, "libgfinputs_cuda.so")
_cpu = None
_cuda = None

# The five workloads of BASELINE.json "configs" (lattice, gauge, precision, storage, generator and run parameters).
CONFIGS = [
    dict(name="cfg0", dims=(8, 8, 8, 8), gauge="landau", prec="f64", storage=18, roughness=0.3, seed=1, omega=1.70,
         eps=1e-12, max_sweeps=2000, check_every=10, reunit_every=0),
    dict(name="cfg1", dims=(16, 16, 16, 32), gauge="coulomb", prec="f64", storage=18, roughness=0.5, seed=2,
         omega=1.70, eps=1e-12, max_sweeps=3000, check_every=10, reunit_every=0),
    dict(name="cfg2", dims=(32, 32, 32, 32), gauge="landau", prec="f32", storage=12, roughness=0.4, seed=3,
         omega=1.75, eps=1e-7, max_sweeps=3000, check_every=10, reunit_every=50),
    dict(name="cfg3", dims=(48, 48, 48, 96), gauge="landau", prec="f64", storage=12, roughness=0.5, seed=4,
         omega=1.80, eps=0.0, max_sweeps=500, check_every=25, reunit_every=0),
    dict(name="cfg4", dims=(64, 64, 64, 128), gauge="landau", prec="f64", storage=18, roughness=0.6, seed=5,
         omega=1.80, eps=0.0, max_sweeps=200, check_every=20, reunit_every=0),
]


def _stale(so: str, srcs) -> bool:
    if not os.path.exists(so):
        return True
    t = os.path.getmtime(so)
    return any(os.path.getmtime(os.path.join(_HERE, s)) > t for s in srcs)


def build(cuda: bool = True, force: bool = False) -> None:
    """Compile the host generator (g++) and, if asked, the device generator (nvcc, sm_100a)."""
    if force or _stale(_CPU_SO, ["gen_cpu.cpp", "gen_core.h"]):
        subprocess.check_call(["g++", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c++17", "-o", _CPU_SO,
                               os.path.join(_HERE, "gen_cpu.cpp")])
    if cuda and (force or _stale(_CUDA_SO, ["gen_cuda.cu", "gen_core.h"])):
        subprocess.check_call(["nvcc", "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
                               "-shared", "-Xcompiler", "-fPIC", "-o", _CUDA_SO, os.path.join(_HERE, "gen_cuda.cu")])


def _lib_cpu():
    global _cpu
    if _cpu is None:
        build(cuda=False)
        _cpu = ctypes.CDLL(_CPU_SO)
        _cpu.gfin_links_host.restype = ctypes.c_int
        _cpu.gfin_links_host.argtypes = [ctypes.c_void_p, ctypes.POINTER(ctypes.c_int), ctypes.c_double,
                                         ctypes.c_uint64, ctypes.c_void_p, ctypes.c_int64, ctypes.c_int]
        _cpu.gfin_gauge_host.restype = ctypes.c_int
        _cpu.gfin_gauge_host.argtypes = [ctypes.c_void_p, ctypes.POINTER(ctypes.c_int), ctypes.c_uint64,
                                         ctypes.c_void_p, ctypes.c_int64]
    return _cpu


def _lib_cuda():
    global _cuda
    if _cuda is None:
        build(cuda=True)
        _cuda = ctypes.CDLL(_CUDA_SO)
        _cuda.gfin_links_device.restype = ctypes.c_int
        _cuda.gfin_links_device.argtypes = [ctypes.c_void_p, ctypes.POINTER(ctypes.c_int), ctypes.c_double,
                                            ctypes.c_uint64, ctypes.c_int, ctypes.c_void_p]
    return _cuda


def _dims(dims):
    d = (ctypes.c_int * 4)(*[int(v) for v in dims])
    vol = int(np.prod([int(v) for v in dims], dtype=np.int64))
    return d, vol


def volume(dims) -> int:
    return _dims(dims)[1]


def make_links(dims, roughness: float, seed: int, dtype=np.float64, sites=None, out=None) -> np.ndarray:
    """Links of the whole lattice, shape (V,4,3,3,2), or of the listed lexicographic sites, shape (n,4,3,3,2)."""
    d, vol = _dims(dims)
    dtype = np.dtype(dtype)
    prec = {np.dtype(np.float64): 0, np.dtype(np.float32): 1}[dtype]
    if sites is None:
        n, sp = vol, None
    else:
        sites = np.ascontiguousarray(sites, dtype=np.int64)
        n, sp = int(sites.size), sites.ctypes.data
    if out is None:
        out = np.empty((n, 4, 3, 3, 2), dtype=dtype)
    assert out.dtype == dtype and out.size == n * 72 and out.flags.c_contiguous
    rc = _lib_cpu().gfin_links_host(out.ctypes.data, d, float(roughness), int(seed), sp, n, prec)
    if rc != 0:
        raise RuntimeError(f"gfin_links_host failed ({rc})")
    return out


def make_gauge(dims, seed: int, sites=None) -> np.ndarray:
    """The hidden Haar-random rotation G(x) of the recipe as complex128, shape (V,3,3) (or (n,3,3))."""
    d, vol = _dims(dims)
    if sites is None:
        n, sp = vol, None
    else:
        sites = np.ascontiguousarray(sites, dtype=np.int64)
        n, sp = int(sites.size), sites.ctypes.data
    out = np.empty((n, 3, 3, 2), dtype=np.float64)
    rc = _lib_cpu().gfin_gauge_host(out.ctypes.data, d, int(seed), sp, n)
    if rc != 0:
        raise RuntimeError(f"gfin_gauge_host failed ({rc})")
    return out.view(np.complex128)[..., 0]


def make_links_device(dev_ptr: int, dims, roughness: float, seed: int, prec: str, stream: int = 0) -> None:
    """Fill a caller-owned DEVICE buffer of V*72 elements (f64 or f32) with the field; asynchronous on `stream`."""
    d, _ = _dims(dims)
    rc = _lib_cuda().gfin_links_device(ctypes.c_void_p(dev_ptr), d, float(roughness), int(seed),
                                       {"f64": 0, "f32": 1}[prec], ctypes.c_void_p(stream))
    if rc != 0:
        raise RuntimeError(f"gfin_links_device failed ({rc})")


def as_complex(links: np.ndarray) -> np.ndarray:
    """(…,3,3,2) real view -> (…,3,3) complex view (no copy)."""
    ct = np.complex128 if links.dtype == np.float64 else np.complex64
    return links.view(ct)[..., 0]


# ---- SU(N) fields (general number of colours, host only) ---------------------------------------------------------------
# The same recipe with N x N matrices, in numpy: U_mu(x) = G(x) exp(i r H_mu(x)) G(x+mu)^dagger, H = sum_a c_a lambda_a
# over the N^2 - 1 generalised Gell-Mann matrices (Tr lambda_a lambda_b = 2 delta_ab), c_a ~ N(0,1); G(x) Haar SU(N).
# Random numbers: numpy's PCG64 seeded by (seed, N); drawn in one fixed order, so a field is reproducible as a whole.
def _gellmann_hermitian(rng, n, N):
    """n random traceless Hermitian N x N matrices sum_a c_a lambda_a with unit-variance coefficients."""
    H = np.zeros((n, N, N), dtype=np.complex128)
    for i in range(N):
        for j in range(i + 1, N):
            cs, ca = rng.normal(size=n), rng.normal(size=n)  # symmetric and antisymmetric generator of the pair
            H[:, i, j] = cs - 1j * ca
            H[:, j, i] = cs + 1j * ca
    for k in range(1, N):  # diagonal generators sqrt(2/(k(k+1))) diag(1,..,1,-k,0,..)
        c = rng.normal(size=n) * np.sqrt(2.0 / (k * (k + 1)))
        for i in range(k):
            H[:, i, i] += c
        H[:, k, k] -= k * c
    return H


def _haar_sun(rng, n, N):
    z = rng.normal(size=(n, N, N)) + 1j * rng.normal(size=(n, N, N))
    q, r = np.linalg.qr(z)
    d = np.diagonal(r, axis1=-2, axis2=-1)
    q = q * (d / np.abs(d))[:, None, :]
    det = np.linalg.det(q)
    return q * np.exp(-1j * np.angle(det) / N)[:, None, None]


def make_gauge_sun(dims, ncolors: int, seed: int) -> np.ndarray:
    """The hidden Haar-random rotation G(x), complex128 (V,N,N)."""
    _, vol = _dims(dims)
    return _haar_sun(np.random.default_rng([int(seed), int(ncolors), 1]), vol, int(ncolors))


def make_links_sun(dims, ncolors: int, roughness: float, seed: int, dtype=np.float64) -> np.ndarray:
    """SU(N) links of the whole lattice in the canonical layout, shape (V,4,N,N,2)."""
    N = int(ncolors)
    nx, ny, nz, nt = (int(v) for v in dims)
    _, vol = _dims(dims)
    G = make_gauge_sun(dims, N, seed).reshape(nt, nz, ny, nx, N, N)
    rng = np.random.default_rng([int(seed), N, 2])
    out = np.empty((vol, 4, N, N), dtype=np.complex128)
    for mu in range(4):
        H = _gellmann_hermitian(rng, vol, N)
        w, v = np.linalg.eigh(H)
        E = (v * np.exp(1j * roughness * w)[:, None, :]) @ np.conj(np.swapaxes(v, -1, -2))  # exp(i r H), det = 1
        Gup = np.roll(G, -1, axis=3 - mu).reshape(vol, N, N)  # G(x + mu)
        out[:, mu] = G.reshape(vol, N, N) @ E @ np.conj(np.swapaxes(Gup, -1, -2))
    res = np.empty((vol, 4, N, N, 2), dtype=np.dtype(dtype))
    res[..., 0] = out.real
    res[..., 1] = out.imag
    return np.ascontiguousarray(res)
