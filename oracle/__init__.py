"""ctypes front end of the CPU oracle (oracle/gf_oracle.cpp).  TEST INFRASTRUCTURE, not product code.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this package.
It never imports paper_1412_1498_b200 and shares no code with it.  All arrays are host numpy arrays in the canonical
layout links[site][mu][row][col][re,im] (shape (V,4,3,3,2)), float64 or float32; updates are IN PLACE.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gf_oracle.cpp")
_SO = os.path.join(_HERE, "libgf_oracle.so")
_lib = None

LANDAU, COULOMB = 0, 1
_GAUGE = {"landau": LANDAU, "coulomb": COULOMB, LANDAU: LANDAU, COULOMB: COULOMB}


def build(force: bool = False) -> None:
    """Compile the oracle with g++ (plain -O2, no FMA contraction, OpenMP over the sites of one parity)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-fcx-limited-range",
                               "-shared", "-fPIC", "-o", _SO, _SRC])


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_SO)
    return _lib


def _suf(U: np.ndarray) -> str:
    assert U.flags.c_contiguous and U.flags.writeable is not None
    if U.dtype == np.float64:
        return "f64"
    if U.dtype == np.float32:
        return "f32"
    raise TypeError(f"links must be float64 or float32, not {U.dtype}")


def _dims(dims):
    return (ctypes.c_int * 4)(*[int(v) for v in dims])


def _p(a: np.ndarray):
    return ctypes.c_void_p(a.ctypes.data)


def _fn(name: str, U: np.ndarray):
    return getattr(_load(), f"{name}_{_suf(U)}")


def num_threads() -> int:
    return int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))


def measure(U, dims, gauge):
    """(F, theta) of eqs. 1.1-1.3 on the links as they stand."""
    F, th = ctypes.c_double(), ctypes.c_double()
    _fn("orc_measure", U)(_p(U), _dims(dims), _GAUGE[gauge], ctypes.byref(F), ctypes.byref(th))
    return F.value, th.value


def half_sweep(U, dims, gauge, parity, omega, storage=18):
    """Algorithm 1 lines 3-12 for one parity, in place."""
    _fn("orc_half_sweep", U)(_p(U), _dims(dims), _GAUGE[gauge], int(parity), ctypes.c_double(omega), int(storage))


def sweeps(U, dims, gauge, omega, n=1, storage=18, reunit_every=0, first_sweep=0):
    """n full sweeps, even then odd, reunitarising every `reunit_every` sweeps."""
    _fn("orc_sweeps", U)(_p(U), _dims(dims), _GAUGE[gauge], ctypes.c_double(omega), int(storage), int(n),
                         int(reunit_every), int(first_sweep))


def site_update(U, dims, gauge, site, omega, storage=18):
    _fn("orc_site_update", U)(_p(U), _dims(dims), _GAUGE[gauge], ctypes.c_int64(int(site)), ctypes.c_double(omega),
                              int(storage))


def reunitarize(U, dims):
    _fn("orc_reunitarize", U)(_p(U), _dims(dims))


def project12(U, dims):
    """Overwrite row 2 of every link with conj(row0 x row1): what 12-real storage does to its input."""
    _fn("orc_project12", U)(_p(U), _dims(dims))


def project8(U, dims):
    """Send every link through the 8-real parametrisation and back: what 8-real storage does to its input (A23)."""
    _fn("orc_project8", U)(_p(U), _dims(dims))


def fix(U, dims, gauge, omega, eps, max_sweeps, check_every, reunit_every=0, storage=18):
    """Algorithm 1 with a measurement cadence.  Returns (sweeps_done, history[(sweep, F, theta), ...])."""
    cap = max_sweeps // max(check_every, 1) + 3
    hist = np.zeros((cap, 3), dtype=np.float64)
    done, nh = ctypes.c_int(), ctypes.c_int()
    _fn("orc_fix", U)(_p(U), _dims(dims), _GAUGE[gauge], ctypes.c_double(omega), ctypes.c_double(eps),
                      int(max_sweeps), int(check_every), int(reunit_every), int(storage), ctypes.byref(done),
                      _p(hist), cap, ctypes.byref(nh))
    return done.value, hist[: min(nh.value, cap)].copy()


def measure_slices(U, dims, gauge):
    """(F_t, theta_t): eqs. 1.1-1.2 restricted to each time slice (reading A22)."""
    nt = int(dims[3])
    Ft, tht = np.zeros(nt), np.zeros(nt)
    _fn("orc_measure_slices", U)(_p(U), _dims(dims), _GAUGE[gauge], _p(Ft), _p(tht))
    return Ft, tht


def half_sweep_masked(U, dims, gauge, parity, omega, active, storage=18):
    """One parity of the sweep over the time slices with active[t] != 0 only."""
    m = np.ascontiguousarray(active, dtype=np.uint8)
    _fn("orc_half_sweep_masked", U)(_p(U), _dims(dims), _GAUGE[gauge], int(parity), ctypes.c_double(omega), int(storage),
                                    _p(m))


def fix_slices(U, dims, gauge, omega, eps, max_sweeps, check_every, reunit_every=0, storage=18):
    """Algorithm 1 with a stop test per time slice (reading A22).
    Returns (sweeps_done, slice_sweeps[nt], history[(sweep, mean F, max theta_t), ...])."""
    cap = max_sweeps // max(check_every, 1) + 3
    hist = np.zeros((cap, 3), dtype=np.float64)
    per = np.zeros(int(dims[3]), dtype=np.int32)
    done, nh = ctypes.c_int(), ctypes.c_int()
    _fn("orc_fix_slices", U)(_p(U), _dims(dims), _GAUGE[gauge], ctypes.c_double(omega), ctypes.c_double(eps),
                             int(max_sweeps), int(check_every), int(reunit_every), int(storage), ctypes.byref(done),
                             _p(per), _p(hist), cap, ctypes.byref(nh))
    return done.value, per, hist[: min(nh.value, cap)].copy()


def site_K(U, dims, gauge, site):
    """K(x) of eq. 1.5 as a complex 3x3."""
    K = np.zeros(18, dtype=U.dtype)
    _fn("orc_site_K", U)(_p(U), _dims(dims), _GAUGE[gauge], ctypes.c_int64(int(site)), _p(K))
    return K.reshape(3, 3, 2)[..., 0] + 1j * K.reshape(3, 3, 2)[..., 1]


def site_delta(U, dims, gauge, site):
    """Delta(x) of eq. 1.3 as a complex 3x3."""
    D = np.zeros(18, dtype=U.dtype)
    _fn("orc_site_delta", U)(_p(U), _dims(dims), _GAUGE[gauge], ctypes.c_int64(int(site)), _p(D))
    return D.reshape(3, 3, 2)[..., 0] + 1j * D.reshape(3, 3, 2)[..., 1]


def _pack(M, dtype):
    out = np.empty((3, 3, 2), dtype=dtype)
    out[..., 0] = M.real
    out[..., 1] = M.imag
    return np.ascontiguousarray(out)


def su2_step(K, G, i, j, omega, dtype=np.float64):
    """One SU(2) subgroup step on complex 3x3 K, G.  Returns (K', G', a) with a the quaternion of g^omega."""
    Kr, Gr = _pack(np.asarray(K), dtype), _pack(np.asarray(G), dtype)
    a = np.zeros(4, dtype=dtype)
    _fn("orc_su2_step", Kr)(_p(Kr), _p(Gr), int(i), int(j), ctypes.c_double(omega), _p(a))
    return Kr[..., 0] + 1j * Kr[..., 1], Gr[..., 0] + 1j * Gr[..., 1], a


def su2_power(a, omega, dtype=np.float64):
    a = np.ascontiguousarray(a, dtype=dtype)
    out = np.zeros(4, dtype=dtype)
    _fn("orc_su2_power", a)(_p(a), ctypes.c_double(omega), _p(out))
    return out


def su2_power_series(a, omega, order, dtype=np.float64):
    """Truncated binomial series of g^omega (order terms beyond 1), renormalised (reading A21)."""
    a = np.ascontiguousarray(a, dtype=dtype)
    out = np.zeros(4, dtype=dtype)
    _fn("orc_su2_power_series", a)(_p(a), ctypes.c_double(omega), int(order), _p(out))
    return out


def set_series(order: int) -> None:
    """Process-wide switch: 0 = every update uses the exact power g^omega (default), N > 0 = the order-N series."""
    _load().orc_set_series(int(order))


def get_series() -> int:
    return int(_load().orc_get_series())


def wilson_traces(U, dims, mu, nu, a, b):
    """Tr of the a x b Wilson loop in the (mu,nu) plane at every site, complex array of length V."""
    V = int(np.prod(dims))
    out = np.zeros((V, 2), dtype=np.float64)
    _fn("orc_wilson_traces", U)(_p(U), _dims(dims), int(mu), int(nu), int(a), int(b), _p(out))
    return out[:, 0] + 1j * out[:, 1]


def polyakov_traces(U, dims, mu):
    V = int(np.prod(dims))
    out = np.zeros((V, 2), dtype=np.float64)
    _fn("orc_polyakov_traces", U)(_p(U), _dims(dims), int(mu), _p(out))
    return out[:, 0] + 1j * out[:, 1]


def unitarity(U, dims):
    """(max |U U^dag - 1|_ij, max |det U - 1|) over all links."""
    a, b = ctypes.c_double(), ctypes.c_double()
    _fn("orc_unitarity", U)(_p(U), _dims(dims), ctypes.byref(a), ctypes.byref(b))
    return a.value, b.value
