"""CPU oracle of Algorithm 2 — steepest descent with Fourier acceleration (eqs. 1.7-1.9, 97-124 Alg. 2).

TEST INFRASTRUCTURE, not product code: plain numpy in FP64 (complex128), one statement per step of the paper's
listing, numpy.fft as the library FFT.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may
import it; it shares nothing with paper_1412_1498_b200.

Links: host array in the canonical layout links[site][mu][row][col][re,im], shape (V,4,3,3,2), float64,
site = x + nx*(y + ny*(z + nz*t)); updated IN PLACE.  Internally viewed as W[t,z,y,x,mu,row,col] complex128.

Readings (B1-B6; A-numbers are those of Algorithm 1 and carry over):
  B1  The bracket of eqs. 1.7/1.8, sum_nu Delta_{-nu}[U_nu(x) - U_nu(x)^dag] - trace with eq. 1.9, is Delta(x) of
      eq. 1.3 (reading A2): A = sum_{nu<d}[U_nu(x-nu) - U_nu(x)], Delta = (A - A^dag) - (1/3)Tr(A - A^dag).
  B2  p^2 = eigenvalues of (-d^2) on the periodic lattice: p^2(k) = sum_{mu<d} 4 sin^2(pi k_mu / n_mu), a = 1;
      p^2_max = 4d (all extents even).  d = 4 Landau; d = 3 Coulomb, where the FFT is the 3-D transform of each time
      slice (only mu = 0,1,2 enter), so slices stay decoupled (A9).
  B3  The zero mode: sum_x Delta(x) = 0 identically (periodic telescoping sum), so the p = 0 factor multiplies
      rounding noise only; it is set to 0.
  B4  "normalize" (Alg. 2 l.7) = the 1/N of the inverse discrete transform, N = number of sites transformed.
  B5  "expand to first order the exponential, followed by a reunitarization": g = 1 + w,
      w = F^-1 (alpha/2)(p^2_max/p^2) F Delta, then the Gram-Schmidt of reading A12 (rows 0,1; row 2 = conj(r0 x r1)).
  B6  U_mu(x) <- g(x) U_mu(x) g(x+mu)^dag for all four mu, also in Coulomb gauge (A9); with 12-real storage
      emulation row 2 of every link is rebuilt after the write (A13).
`accelerate=False` replaces the Fourier factor by 1: the naive steepest descent of eq. 1.7 (first order).

Parity unpinned: whole-trajectory values (iteration counts, final F) — the paper prints none.  Everything else is
pinned in tests/test_fftsd_oracle_pins.py (p^2 against the lattice Laplacian, dF/dalpha against the closed form
theta/(4d) and its momentum-space generalisation, gauge invariance, unitarity, convergence to F = 1 on a pure gauge);
fix()'s iteration / reunitarisation order in tests/test_oracle_order_pins.py (against step + reunitarize_links unrolled).
"""
from __future__ import annotations

import numpy as np

_AXIS = {0: 3, 1: 2, 2: 1, 3: 0}  # mu -> axis of W[t,z,y,x,...]


def _view(U, dims):
    nx, ny, nz, nt = (int(v) for v in dims)
    assert U.dtype == np.float64 and U.flags.c_contiguous and U.size == nx * ny * nz * nt * 72
    return U.view(np.complex128).reshape(nt, nz, ny, nx, 4, 3, 3)


def _nd(gauge):
    return 3 if gauge in ("coulomb", 1) else 4


def delta_field(U, dims, gauge):
    """Delta(x) of eq. 1.3 (B1), array [t,z,y,x,3,3]."""
    W = _view(U, dims)
    A = np.zeros(W.shape[:4] + (3, 3), dtype=np.complex128)
    for nu in range(_nd(gauge)):
        Unu = W[..., nu, :, :]
        A += np.roll(Unu, 1, axis=_AXIS[nu]) - Unu  # U_nu(x - nu) - U_nu(x)      (eq. 1.9)
    D = A - np.conj(np.swapaxes(A, -1, -2))
    tr = np.trace(D, axis1=-2, axis2=-1) / 3.0
    for i in range(3):
        D[..., i, i] -= tr
    return D


def measure(U, dims, gauge):
    """(F, theta) of eqs. 1.1-1.2 (readings A1, A2)."""
    W = _view(U, dims)
    d = _nd(gauge)
    V = W.shape[0] * W.shape[1] * W.shape[2] * W.shape[3]
    F = sum(np.trace(W[..., mu, :, :], axis1=-2, axis2=-1).real.sum() for mu in range(d)) / (d * 3.0 * V)
    D = delta_field(U, dims, gauge)
    theta = (np.abs(D) ** 2).sum() / (3.0 * V)
    return float(F), float(theta)


def p2_table(dims, gauge):
    """p^2(k) on the transformed axes (B2), array broadcastable to [t,z,y,x]; and p^2_max."""
    nx, ny, nz, nt = (int(v) for v in dims)
    d = _nd(gauge)
    n = {0: nx, 1: ny, 2: nz, 3: nt}
    p2 = np.zeros((nt if d == 4 else 1, nz, ny, nx))
    for mu in range(d):
        s = 4.0 * np.sin(np.pi * np.arange(n[mu]) / n[mu]) ** 2
        shape = [1, 1, 1, 1]
        shape[_AXIS[mu]] = n[mu]
        p2 = p2 + s.reshape(shape)
    return p2, 4.0 * d


def fourier_accelerate(D, dims, gauge, alpha, accelerate=True):
    """w = F^-1 (alpha/2)(p^2_max/p^2) F Delta, per matrix element (Alg. 2 l.3-8; eq. 1.8; B2-B4)."""
    if not accelerate:
        return 0.5 * alpha * D  # eq. 1.7
    d = _nd(gauge)
    axes = (0, 1, 2, 3) if d == 4 else (1, 2, 3)
    p2, p2max = p2_table(dims, gauge)
    with np.errstate(divide="ignore"):
        fac = np.where(p2 > 0.0, p2max / p2, 0.0)  # B3
    w = np.empty_like(D)
    for i in range(3):
        for j in range(3):
            Dh = np.fft.fftn(D[..., i, j], axes=axes)       # apply FFT forward
            Dh = Dh * fac                                   # apply p^2_max / p^2
            w[..., i, j] = np.fft.ifftn(Dh, axes=axes)      # apply FFT backward, normalize
    return 0.5 * alpha * w


def reunitarize_rows(g):
    """Gram-Schmidt on rows 0,1; row 2 = conj(row0 x row1) (reading A12), on an array [...,3,3]."""
    r0 = g[..., 0, :]
    r0 = r0 / np.sqrt((np.abs(r0) ** 2).sum(-1, keepdims=True))
    r1 = g[..., 1, :]
    r1 = r1 - (np.conj(r0) * r1).sum(-1, keepdims=True) * r0
    r1 = r1 / np.sqrt((np.abs(r1) ** 2).sum(-1, keepdims=True))
    r2 = np.conj(np.cross(r0, r1))
    return np.stack([r0, r1, r2], axis=-2)


def gauge_rotation(w):
    """g(x) = reunitarize(1 + w(x))  (Alg. 2 l.10; B5)."""
    g = w.copy()
    for i in range(3):
        g[..., i, i] += 1.0
    return reunitarize_rows(g)


def apply_rotation(U, dims, g, storage=18):
    """U_mu(x) <- g(x) U_mu(x) g(x+mu)^dag, all four mu (Alg. 2 l.11-15; B6), in place."""
    W = _view(U, dims)
    for mu in range(4):
        gup = np.roll(g, -1, axis=_AXIS[mu])  # g(x + mu)
        new = np.einsum("...ij,...jk,...lk->...il", g, W[..., mu, :, :], np.conj(gup))
        if storage == 12:
            new[..., 2, :] = np.conj(np.cross(new[..., 0, :], new[..., 1, :]))  # A13
        W[..., mu, :, :] = new


def step(U, dims, gauge, alpha, storage=18, accelerate=True):
    """One iteration of Algorithm 2 (l.3-16), in place."""
    D = delta_field(U, dims, gauge)
    w = fourier_accelerate(D, dims, gauge, alpha, accelerate)
    g = gauge_rotation(w)
    apply_rotation(U, dims, g, storage)


def reunitarize_links(U, dims):
    """Project every link back onto SU(3) (reading A12), in place."""
    W = _view(U, dims)
    W[...] = reunitarize_rows(W)


def fix(U, dims, gauge, alpha, eps, max_iters, check_every=1, storage=18, accelerate=True, reunit_every=0):
    """Algorithm 2 with a measurement cadence: measure; while theta >= eps: `check_every` iterations; measure.
    After iteration s the links are reunitarised if reunit_every > 0 and s % reunit_every == 0.
    Returns (iterations_done, history[(iteration, F, theta), ...])."""
    done = 0
    F, th = measure(U, dims, gauge)
    hist = [(0, F, th)]
    while not (th < eps) and done < max_iters:
        n = min(check_every, max_iters - done)
        for i in range(n):
            step(U, dims, gauge, alpha, storage, accelerate)
            if reunit_every > 0 and (done + i + 1) % reunit_every == 0:
                reunitarize_links(U, dims)
        done += n
        F, th = measure(U, dims, gauge)
        hist.append((done, F, th))
    return done, hist
