"""CPU oracle of the overrelaxation sweep for general SU(N) — TEST INFRASTRUCTURE, not product code.

The paper states the method for "SU(N) with N>2" and says how: "we update the link variables by
iterating over its N(N-1)/2 SU(2) subgroups".  This file is eqs. 1.1-1.6 and Algorithm 1
 for an N x N link, step by step, in plain numpy (complex128); all sites of one parity are
updated in one vectorised statement, which Algorithm 1 allows because same-parity updates touch disjoint links
(PAPER.md:74-75, 134).  It shares no code with gf_oracle.cpp (the SU(3) oracle) nor with paper_1412_1498_b200; only
tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import it.

Links: host array links[site][mu][row][col][re,im], shape (V,4,N,N,2), float64, site = x + nx*(y + ny*(z + nz*t)),
updated IN PLACE.  Internally W[t,z,y,x,mu,row,col] complex128.

Readings (A1-A20 carry over with Nc = N):
  A1   F = 1/(d N V) sum_x sum_{mu<d} Re Tr U_mu(x), d = 4 Landau / 3 Coulomb.
  A2   Delta = (A - A^dag) - (1/N) Tr(A - A^dag), A = sum_{nu<d}[U_nu(x-nu) - U_nu(x)]; theta = 1/(N V) sum Tr Delta Delta^dag.
  A3   K(x) = sum_{mu<d}[U_mu(x) + U_mu(x-mu)^dag].
  A5-7 the subgroup step is the SU(3) one: r from the 2x2 block on rows/cols (i,j), a = r/|r|, exact power g^omega.
  A24  order of the N(N-1)/2 subgroups (the paper gives none): pairs (i,j), i<j, by increasing distance j-i, then by
       increasing i.  N=2: (0,1).  N=3: (0,1),(1,2),(0,2) - reading A4.  N=4: (0,1),(1,2),(2,3),(0,2),(1,3),(0,3).
  A25  reunitarisation for N x N: Gram-Schmidt over the rows in order (each row minus its projections on
       the finished rows, one after the other, then normalised), then the last row times conj(det) so that det = 1.
  Storage: all N^2 complex entries (no 12-/8-real forms: they are SU(3) constructions).

Pins (tests/test_sun_oracle_pins.py): N = 3 against the SU(3) C++ oracle (links after sweeps, F, theta, reunitarisation
up to rounding); N = 2: one omega = 1 update equals eq. 1.6's closed form g = K^dag / sqrt(det K^dag) literally; brute
force over random SU(2) per subgroup (N = 2, 4); gauge invariance of plaquettes, unitarity and det = 1 after sweeps;
F = 1, theta = 0 on a gauge-transformed unit field; F non-decreasing at omega = 1; the subgroup list; even-before-odd
and the reunitarisation cadence.  Parity unpinned: whole-trajectory values (the paper prints none).
"""
from __future__ import annotations

import numpy as np

_AXIS = {0: 3, 1: 2, 2: 1, 3: 0}  # mu -> axis of W[t,z,y,x,...]
_TINY = np.finfo(np.float64).tiny * 2.0 ** 60  # reading A7


def _view(U, dims, N):
    nx, ny, nz, nt = (int(v) for v in dims)
    assert U.dtype == np.float64 and U.flags.c_contiguous and U.size == nx * ny * nz * nt * 4 * N * N * 2
    return U.view(np.complex128).reshape(nt, nz, ny, nx, 4, N, N)


def _nd(gauge):
    return 3 if gauge in ("coulomb", 1) else 4


def _dag(M):
    return np.conj(np.swapaxes(M, -1, -2))


def subgroups(N):
    """The N(N-1)/2 index pairs in the order of reading A24."""
    return [(i, i + d) for d in range(1, N) for i in range(N - d)]


def parity_mask(dims):
    """mask[t,z,y,x] = (x+y+z+t) & 1   (reading A10: even <=> 0)."""
    nx, ny, nz, nt = (int(v) for v in dims)
    t, z, y, x = np.meshgrid(np.arange(nt), np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    return (x + y + z + t) & 1


def measure(U, dims, gauge, N):
    """(F, theta), eqs. 1.1-1.3 (readings A1, A2)."""
    W = _view(U, dims, N)
    d = _nd(gauge)
    V = W.shape[0] * W.shape[1] * W.shape[2] * W.shape[3]
    F = sum(np.trace(W[..., mu, :, :], axis1=-2, axis2=-1).real.sum() for mu in range(d)) / (d * N * V)
    A = np.zeros(W.shape[:4] + (N, N), dtype=np.complex128)
    for nu in range(d):
        Unu = W[..., nu, :, :]
        A += np.roll(Unu, 1, axis=_AXIS[nu]) - Unu  # U_nu(x - nu) - U_nu(x)
    D = A - _dag(A)
    tr = np.trace(D, axis1=-2, axis2=-1) / N
    for i in range(N):
        D[..., i, i] -= tr
    theta = (np.abs(D) ** 2).sum() / (N * V)
    return float(F), float(theta)


def build_K(U, dims, gauge, N):
    """K(x) of eq. 1.5 at every site (reading A3), array [t,z,y,x,N,N]."""
    W = _view(U, dims, N)
    K = np.zeros(W.shape[:4] + (N, N), dtype=np.complex128)
    for mu in range(_nd(gauge)):
        Umu = W[..., mu, :, :]
        K += Umu
        K += _dag(np.roll(Umu, 1, axis=_AXIS[mu]))  # U_mu(x - mu)^dag
    return K


def su2_power(a, omega):
    """a: (...,4) unit quaternions (a0; a1,a2,a3) <-> g = a0 + i a.sigma.  Exact power g^omega, principal branch
    (readings A6, A7)."""
    a0, av = a[..., 0], a[..., 1:]
    s = np.sqrt((av ** 2).sum(axis=-1))
    phi = np.arctan2(s, a0)
    out = np.empty_like(a)
    small = s < _TINY
    safe = np.where(small, 1.0, s)
    f = np.where(small, omega, np.sin(omega * phi) / safe)
    out[..., 0] = np.cos(omega * phi)
    out[..., 1:] = av * f[..., None]
    flip = small & ~(a0 > 0)  # phi = pi, axis undefined: g^omega = 1
    out[flip] = np.array([1.0, 0.0, 0.0, 0.0])
    return out


def subgroup_step(K, G, i, j, omega):
    """One SU(2) subgroup step on rows/cols (i,j) of K, G (arrays [...,N,N], updated in place): the maximiser of
    Re Tr[g K] over the embedded SU(2) (eq. 1.6 on the SU(2)-proportional part of the block, reading A5), raised to
    omega; K <- gK, G <- gG.  Returns the quaternion of g^omega."""
    M00, M01, M10, M11 = K[..., i, i], K[..., i, j], K[..., j, i], K[..., j, j]
    r = np.stack([(M00 + M11).real, -(M01 + M10).imag, (M10 - M01).real, -(M00 - M11).imag], axis=-1)
    n = np.sqrt((r ** 2).sum(axis=-1))
    zero = n == 0.0
    a = r / np.where(zero, 1.0, n)[..., None]
    a[zero] = np.array([1.0, 0.0, 0.0, 0.0])  # reading A7: nothing to maximise, g = 1
    q = su2_power(a, omega)
    q[zero] = np.array([1.0, 0.0, 0.0, 0.0])
    g00 = q[..., 0] + 1j * q[..., 3]
    g01 = q[..., 2] + 1j * q[..., 1]
    g10 = -q[..., 2] + 1j * q[..., 1]
    g11 = q[..., 0] - 1j * q[..., 3]
    for M in (K, G):
        ri, rj = M[..., i, :].copy(), M[..., j, :].copy()
        M[..., i, :] = g00[..., None] * ri + g01[..., None] * rj
        M[..., j, :] = g10[..., None] * ri + g11[..., None] * rj
    return q


def site_rotations(U, dims, gauge, N, omega):
    """G(x) = product of the subgroup rotations of Algorithm 1 l.5-6 at EVERY site, from the links as they stand
    (reading A8: accumulate, apply once).  Array [t,z,y,x,N,N]."""
    K = build_K(U, dims, gauge, N)
    G = np.zeros_like(K)
    for i in range(N):
        G[..., i, i] = 1.0
    for i, j in subgroups(N):
        subgroup_step(K, G, i, j, omega)
    return G


def half_sweep(U, dims, gauge, N, parity, omega):
    """Algorithm 1 l.3-12 for one parity: U_mu(x) <- G(x) U_mu(x), U_mu(x-mu) <- U_mu(x-mu) G(x)^dag for the sites x of
    that parity, all four mu (reading A9).  The other parity's sites get G = 1."""
    W = _view(U, dims, N)
    G = site_rotations(U, dims, gauge, N, omega)
    other = parity_mask(dims) != parity
    G[other] = np.eye(N)
    for mu in range(4):
        Gup = np.roll(G, -1, axis=_AXIS[mu])  # G(x + mu): the link U_mu(x) is the backward link of x + mu
        W[..., mu, :, :] = G @ W[..., mu, :, :] @ _dag(Gup)


def reunitarize(U, dims, N):
    """Reading A25 on every link."""
    W = _view(U, dims, N)
    M = W.reshape(-1, N, N)
    for r in range(N):
        for p in range(r):
            c = (np.conj(M[:, p, :]) * M[:, r, :]).sum(axis=-1)
            M[:, r, :] -= c[:, None] * M[:, p, :]
        M[:, r, :] /= np.sqrt((np.abs(M[:, r, :]) ** 2).sum(axis=-1))[:, None]
    M[:, N - 1, :] *= np.conj(np.linalg.det(M))[:, None]


def sweeps(U, dims, gauge, N, omega, n=1, reunit_every=0, first_sweep=0):
    """n sweeps, even half-sweep first, reunitarising after global sweep s iff s % k == 0."""
    for k in range(1, n + 1):
        half_sweep(U, dims, gauge, N, 0, omega)
        half_sweep(U, dims, gauge, N, 1, omega)
        s = first_sweep + k
        if reunit_every > 0 and s % reunit_every == 0:
            reunitarize(U, dims, N)


def fix(U, dims, gauge, N, omega, eps, max_sweeps, check_every, reunit_every=0):
    """Algorithm 1 with a measurement cadence (reading A11).  Returns (sweeps_done, [(sweep, F, theta), ...])."""
    done = 0
    F, th = measure(U, dims, gauge, N)
    hist = [(0, F, th)]
    while not (th < eps) and done < max_sweeps:
        n = min(check_every, max_sweeps - done)
        sweeps(U, dims, gauge, N, omega, n=n, reunit_every=reunit_every, first_sweep=done)
        done += n
        F, th = measure(U, dims, gauge, N)
        hist.append((done, F, th))
    return done, hist


def unitarity(U, dims, N):
    """(max |U U^dag - 1|_ij, max |det U - 1|) over all links."""
    M = _view(U, dims, N).reshape(-1, N, N)
    return float(np.abs(M @ _dag(M) - np.eye(N)).max()), float(np.abs(np.linalg.det(M) - 1.0).max())
