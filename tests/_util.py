"""numpy helpers for the tests: independent (vectorised, np.roll based) restatements used to pin the oracle."""
import numpy as np


def lex_coords(dims):
    nx, ny, nz, nt = dims
    s = np.arange(nx * ny * nz * nt)
    return np.stack([s % nx, (s // nx) % ny, (s // (nx * ny)) % nz, s // (nx * ny * nz)], axis=1)


def parity(dims):
    return lex_coords(dims).sum(axis=1) & 1


def to_c(U):
    """(V,4,3,3,2) real -> (V,4,3,3) complex copy in the grid shape (nt,nz,ny,nx,4,3,3)."""
    return (U[..., 0] + 1j * U[..., 1])


def from_c(Uc, dtype=np.float64):
    out = np.empty(Uc.shape + (2,), dtype=dtype)
    out[..., 0] = Uc.real
    out[..., 1] = Uc.imag
    return np.ascontiguousarray(out)


def grid(a, dims):
    nx, ny, nz, nt = dims
    return a.reshape((nt, nz, ny, nx) + a.shape[1:])


def flat(a):
    return a.reshape((-1,) + a.shape[4:])


AX = {0: 3, 1: 2, 2: 1, 3: 0}  # direction mu -> numpy axis of the (nt,nz,ny,nx,...) grid


def shift(a, dims, mu, step):
    """field value at x + step*mu (periodic): result[x] = a[x + step mu]; `a` is flat (V,...)"""
    g = grid(a, dims)
    return flat(np.roll(g, -step, axis=AX[mu]))


def dag(M):
    return np.conj(np.swapaxes(M, -1, -2))


def gauge_transform(Uc, g, dims):
    """U_mu(x) -> g(x) U_mu(x) g(x+mu)^dagger  (eq. 1.1); Uc (V,4,3,3), g (V,3,3)."""
    out = np.empty_like(Uc)
    for mu in range(4):
        out[:, mu] = g @ Uc[:, mu] @ dag(shift(g, dims, mu, +1))
    return out


def plaquettes(Uc, dims):
    """mean Re Tr P_{mu nu} / 3 for the six planes."""
    res = {}
    for mu in range(4):
        for nu in range(mu + 1, 4):
            P = Uc[:, mu] @ shift(Uc[:, nu], dims, mu, 1) @ dag(shift(Uc[:, mu], dims, nu, 1)) @ dag(Uc[:, nu])
            res[(mu, nu)] = np.trace(P, axis1=-2, axis2=-1)
    return res


def random_su3(rng, n):
    z = rng.normal(size=(n, 3, 3)) + 1j * rng.normal(size=(n, 3, 3))
    q, r = np.linalg.qr(z)
    d = np.diagonal(r, axis1=-2, axis2=-1)
    q = q * (d / np.abs(d))[:, None, :]
    det = np.linalg.det(q)
    return q / (det ** (1.0 / 3.0))[:, None, None]


def random_unit_quaternions(rng, n):
    a = rng.normal(size=(n, 4))
    return a / np.linalg.norm(a, axis=1, keepdims=True)


def su2_matrix(a):
    """quaternion(s) a=(a0,a1,a2,a3) -> [[a0+i a3, a2+i a1],[-a2+i a1, a0-i a3]]"""
    a = np.asarray(a)
    g = np.empty(a.shape[:-1] + (2, 2), dtype=complex)
    g[..., 0, 0] = a[..., 0] + 1j * a[..., 3]
    g[..., 0, 1] = a[..., 2] + 1j * a[..., 1]
    g[..., 1, 0] = -a[..., 2] + 1j * a[..., 1]
    g[..., 1, 1] = a[..., 0] - 1j * a[..., 3]
    return g


def embed_su2(g2, i, j):
    g2 = np.asarray(g2)
    out = np.zeros(g2.shape[:-2] + (3, 3), dtype=complex)
    out[...] = np.eye(3)
    out[..., i, i] = g2[..., 0, 0]
    out[..., i, j] = g2[..., 0, 1]
    out[..., j, i] = g2[..., 1, 0]
    out[..., j, j] = g2[..., 1, 1]
    return out
