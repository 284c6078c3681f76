"""Pins of oracle/sun.py (the SU(N) overrelaxation oracle) against what the paper and the
mathematics fix: the SU(3) C++ oracle at N = 3 (an independent implementation, itself pinned), eq. 1.6's closed form at
N = 2, hand-computed F / theta of a one-link defect, brute force over random SU(2) elements, gauge invariance, and
the drivers' order.  CPU only."""
import numpy as np
import pytest

import gf_inputs as gi
import oracle
from oracle import sun

DIMS = (4, 4, 2, 6)


def cview(U, N):
    return U.view(np.complex128).reshape(-1, 4, N, N)


def dag(M):
    return np.conj(np.swapaxes(M, -1, -2))


def grid(a, dims):
    nx, ny, nz, nt = dims
    return a.reshape((nt, nz, ny, nx) + a.shape[1:])


def shift(a, dims, mu, step):
    """a[x + step*mu] for a flat (V,...) field"""
    g = grid(a, dims)
    return np.roll(g, -step, axis=3 - mu).reshape(a.shape)


def plaquette_traces(U, dims, N):
    W = cview(U, N)
    out = []
    for mu in range(4):
        for nu in range(mu + 1, 4):
            P = W[:, mu] @ shift(W[:, nu], dims, mu, 1) @ dag(shift(W[:, mu], dims, nu, 1)) @ dag(W[:, nu])
            out.append(np.trace(P, axis1=-2, axis2=-1))
    return np.stack(out)


def pack(Wc):
    out = np.empty(Wc.shape + (2,))
    out[..., 0], out[..., 1] = Wc.real, Wc.imag
    return np.ascontiguousarray(out)


def test_subgroup_list_reading_A24():
    assert sun.subgroups(2) == [(0, 1)]
    assert sun.subgroups(3) == [(0, 1), (1, 2), (0, 2)]  # reading A4 of the SU(3) path
    assert sun.subgroups(4) == [(0, 1), (1, 2), (2, 3), (0, 2), (1, 3), (0, 3)]
    for N in (5, 6):
        s = sun.subgroups(N)
        assert len(s) == N * (N - 1) // 2 == len(set(s)) and all(i < j for i, j in s)  # N(N-1)/2 subgroups


@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
def test_n3_is_the_su3_cpp_oracle(gauge):
    """The same algorithm written twice (std::complex loops per site vs vectorised numpy): N = 3 must reproduce the
    pinned SU(3) oracle up to summation order."""
    U = gi.make_links(DIMS, 0.5, 11)
    A, B = U.copy(), U.copy()
    Fa, ta = oracle.measure(A, DIMS, gauge)
    Fb, tb = sun.measure(B, DIMS, gauge, 3)
    assert abs(Fa - Fb) <= 1e-14 and abs(ta - tb) <= 1e-13 * ta
    for omega in (1.0, 1.7):
        oracle.sweeps(A, DIMS, gauge, omega, n=2)
        sun.sweeps(B, DIMS, gauge, 3, omega, n=2)
        assert np.abs(A - B).max() <= 1e-12
    Fa, ta = oracle.measure(A, DIMS, gauge)
    Fb, tb = sun.measure(B, DIMS, gauge, 3)
    assert abs(Fa - Fb) <= 1e-13 and abs(ta - tb) <= 1e-11 * ta
    # one half-sweep of each parity separately (the parity convention, reading A10)
    for parity in (0, 1):
        A, B = U.copy(), U.copy()
        oracle.half_sweep(A, DIMS, gauge, parity, 1.5)
        sun.half_sweep(B, DIMS, gauge, 3, parity, 1.5)
        assert np.abs(A - B).max() <= 1e-13
        assert np.abs(A - U).max() > 0.1


def test_n3_reunitarisation_agrees_with_the_su3_reading():
    """A25 (Gram-Schmidt over all rows, last row times conj(det)) and A12 (rows 0,1, row 2 = conj(row0 x row1)) describe
    the same projection for N = 3."""
    rng = np.random.default_rng(3)
    U = gi.make_links(DIMS, 0.5, 12)
    U += 1e-3 * rng.normal(size=U.shape)
    A, B = U.copy(), U.copy()
    oracle.reunitarize(A, DIMS)
    sun.reunitarize(B, DIMS, 3)
    assert np.abs(A - B).max() <= 1e-12
    a, b = sun.unitarity(B, DIMS, 3)
    assert max(a, b) <= 1e-14


@pytest.mark.parametrize("N", [2, 4, 5])
def test_reunitarisation_properties(N):
    rng = np.random.default_rng(N)
    U = gi.make_links_sun(DIMS, N, 0.5, 21)
    exact = U.copy()
    sun.reunitarize(exact, DIMS, N)
    assert np.abs(exact - U).max() <= 1e-14  # identity on SU(N)
    U += 1e-3 * rng.normal(size=U.shape)
    sun.reunitarize(U, DIMS, N)
    a, b = sun.unitarity(U, DIMS, N)
    assert max(a, b) <= 1e-14
    again = U.copy()
    sun.reunitarize(again, DIMS, N)
    assert np.abs(again - U).max() <= 1e-14  # idempotent
    # against a library QR: Gram-Schmidt on the rows of M is the QR factorisation of M^T (columns of Q = the
    # orthonormalised rows, up to a unit phase each)
    M = cview(gi.make_links_sun(DIMS, N, 0.5, 22), N)[:50, 0] + 0.01
    q, _ = np.linalg.qr(M.transpose(0, 2, 1))
    X = pack(np.broadcast_to(M[:, None], (50, 4, N, N)).copy())
    sun.reunitarize(X, (50, 1, 1, 1), N)
    R = cview(X, N)[:, 0]
    overlap = np.abs(np.einsum("nrk,nkr->nr", R.conj(), q))
    assert np.abs(overlap - 1.0).max() <= 1e-12
    assert np.abs(np.linalg.det(R) - 1.0).max() <= 1e-13


def test_su2_closed_form_eq_1_6():
    """N = 2: K(x) is proportional to an SU(2) matrix and the exact local maximiser is g = K^dag / sqrt(det K^dag)
    (eq. 1.6).  The subgroup step at omega = 1 must give exactly that."""
    U = gi.make_links_sun(DIMS, 2, 0.6, 31)
    for gauge in ("landau", "coulomb"):
        K = sun.build_K(U, DIMS, gauge, 2)
        G = sun.site_rotations(U, DIMS, gauge, 2, 1.0)
        Kd = dag(K)
        g = Kd / np.sqrt(np.linalg.det(Kd))[..., None, None]
        # det K^dag is real and positive for a sum of SU(2) matrices, so the root has no branch ambiguity
        assert np.abs(np.linalg.det(Kd).imag).max() <= 1e-12 and np.linalg.det(Kd).real.min() > 0
        assert np.abs(G - g).max() <= 1e-13
        # and g K is then Hermitian positive: (gK) = |k| 1
        gK = G @ K
        assert np.abs(gK - dag(gK)).max() <= 1e-12


@pytest.mark.parametrize("N", [2, 4])
def test_brute_force_maximum_per_subgroup(N):
    """Re Tr[g K] at the step's g (omega = 1) is not beaten by any of 4000 random embedded SU(2) elements, and the best
    of them comes close from below - for every subgroup in turn, on a 2^4 lattice (north_star's brute-force check)."""
    dims = (2, 2, 2, 2)
    rng = np.random.default_rng(17)
    U = gi.make_links_sun(dims, N, 0.7, 41)
    K = sun.build_K(U, dims, "landau", N).reshape(-1, N, N)
    G = np.broadcast_to(np.eye(N, dtype=complex), K.shape).copy()
    for i, j in sun.subgroups(N):
        before = K.copy()
        sun.subgroup_step(K, G, i, j, 1.0)
        best = np.trace(K, axis1=-2, axis2=-1).real
        a = rng.normal(size=(4000, 4))
        a /= np.linalg.norm(a, axis=1, keepdims=True)
        # Re Tr[g' K] = const + a . r with r the 4-vector of the block: evaluate the full matrix product instead
        trial = np.empty((4000, K.shape[0]))
        for n in range(0, 4000, 500):
            g = np.broadcast_to(np.eye(N, dtype=complex), (500, N, N)).copy()
            q = a[n:n + 500]
            g[:, i, i] = q[:, 0] + 1j * q[:, 3]
            g[:, i, j] = q[:, 2] + 1j * q[:, 1]
            g[:, j, i] = -q[:, 2] + 1j * q[:, 1]
            g[:, j, j] = q[:, 0] - 1j * q[:, 3]
            trial[n:n + 500] = np.einsum("nab,sba->ns", g, before).real
        assert (trial.max(axis=0) <= best + 1e-12).all()
        assert (best - trial.max(axis=0) <= 0.15 * np.abs(best) + 0.3).all()
        # stationarity: a second application finds nothing to gain
        K2, G2 = K.copy(), G.copy()
        q = sun.subgroup_step(K2, G2, i, j, 1.0)
        assert np.abs(q - np.array([1.0, 0, 0, 0])).max() <= 1e-14


def test_su2_power_group_properties():
    rng = np.random.default_rng(5)
    a = rng.normal(size=(200, 4))
    a /= np.linalg.norm(a, axis=1, keepdims=True)
    assert np.abs(sun.su2_power(a, 1.0) - a).max() <= 1e-15

    def qmul(p, q):
        return np.stack([p[:, 0] * q[:, 0] - (p[:, 1:] * q[:, 1:]).sum(1),
                         p[:, 0] * q[:, 1] + q[:, 0] * p[:, 1] - (p[:, 2] * q[:, 3] - p[:, 3] * q[:, 2]),
                         p[:, 0] * q[:, 2] + q[:, 0] * p[:, 2] - (p[:, 3] * q[:, 1] - p[:, 1] * q[:, 3]),
                         p[:, 0] * q[:, 3] + q[:, 0] * p[:, 3] - (p[:, 1] * q[:, 2] - p[:, 2] * q[:, 1])], axis=1)

    assert np.abs(sun.su2_power(a, 2.0) - qmul(a, a)).max() <= 1e-14
    assert np.abs(qmul(sun.su2_power(a, 0.7), sun.su2_power(a, 1.1)) - sun.su2_power(a, 1.8)).max() <= 1e-14
    assert np.abs(np.linalg.norm(sun.su2_power(a, 1.7), axis=1) - 1).max() <= 1e-15
    # the SU(3) oracle's scalar routine, element by element
    for k in range(20):
        assert np.abs(sun.su2_power(a[k:k + 1], 1.7)[0] - oracle.su2_power(a[k], 1.7)).max() <= 1e-15
    # degenerate inputs (reading A7)
    e = np.array([[1.0, 0, 0, 0], [-1.0, 0, 0, 0], [1.0, 1e-300, 0, 0]])
    out = sun.su2_power(e, 1.7)
    assert np.array_equal(out[0], [1, 0, 0, 0]) and np.array_equal(out[1], [1, 0, 0, 0])
    assert out[2, 0] == 1.0 and abs(out[2, 1] - 1.7e-300) <= 1e-315


@pytest.mark.parametrize("N", [2, 4])
def test_one_link_defect_closed_forms(N):
    """Unit field with U_0(x0) = diag(e^{ia}, e^{-ia}, 1, ...): by hand, A(x0) = 1 - D, A(x0 + 0) = D - 1, the two
    Delta are -+2i diag(sin a, -sin a, 0, ...) (already traceless), so theta = 16 sin^2 a / (N V) and
    F = 1 - (2 - 2 cos a) / (d N V)  (eqs. 1.1-1.3 with readings A1, A2)."""
    dims = (4, 2, 2, 2)
    V, alpha = 32, 0.37
    W = np.broadcast_to(np.eye(N, dtype=complex), (V, 4, N, N)).copy()
    W[5, 0, 0, 0] = np.exp(1j * alpha)
    W[5, 0, 1, 1] = np.exp(-1j * alpha)
    U = pack(W)
    for gauge, d in (("landau", 4), ("coulomb", 3)):
        F, th = sun.measure(U, dims, gauge, N)
        assert abs(F - (1 - (2 - 2 * np.cos(alpha)) / (d * N * V))) <= 1e-15
        assert abs(th - 16 * np.sin(alpha) ** 2 / (N * V)) <= 1e-15
    # a temporal defect is invisible to the Coulomb functional
    W[5, 0] = np.eye(N)
    W[5, 3, 0, 0], W[5, 3, 1, 1] = np.exp(1j * alpha), np.exp(-1j * alpha)
    F, th = sun.measure(pack(W), dims, "coulomb", N)
    assert F == 1.0 and th == 0.0


@pytest.mark.parametrize("N", [2, 4])
@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
def test_sweeps_are_gauge_transformations_and_raise_F(N, gauge):
    U = gi.make_links_sun(DIMS, N, 0.5, 51)
    P0 = plaquette_traces(U, DIMS, N)
    F0, _ = sun.measure(U, DIMS, gauge, N)
    Fs = [F0]
    for _ in range(3):  # omega = 1: relaxation, F must not decrease after any half-sweep
        for parity in (0, 1):
            sun.half_sweep(U, DIMS, gauge, N, parity, 1.0)
            Fs.append(sun.measure(U, DIMS, gauge, N)[0])
    assert all(b >= a - 1e-14 for a, b in zip(Fs, Fs[1:])) and Fs[-1] > Fs[0] + 0.2
    sun.sweeps(U, DIMS, gauge, N, 1.8, n=3)
    assert np.abs(plaquette_traces(U, DIMS, N) - P0).max() <= 1e-12
    a, b = sun.unitarity(U, DIMS, N)
    assert max(a, b) <= 1e-12


@pytest.mark.parametrize("N", [2, 4])
def test_pure_gauge_F1_theta0_and_convergence(N):
    dims = (4, 4, 4, 4)
    G = gi.make_gauge_sun(dims, N, 61)
    W = np.stack([G @ dag(shift(G, dims, mu, 1)) for mu in range(4)], axis=1)
    U = pack(W)
    # transformed back by g = G^dag the field is the unit field: F = 1, theta = 0 in both gauges
    back = np.stack([dag(G) @ W[:, mu] @ shift(G, dims, mu, 1) for mu in range(4)], axis=1)
    for gauge in ("landau", "coulomb"):
        F, th = sun.measure(pack(back), dims, gauge, N)
        assert abs(F - 1) <= 1e-14 and th <= 1e-26
    done, hist = sun.fix(U, dims, "landau", N, 1.7, 1e-20, 400, 10)
    assert hist[-1][2] < 1e-20 and abs(hist[-1][1] - 1.0) <= 1e-12 and done < 400


def test_order_even_first_and_reunit_cadence():
    """sweeps() = even half-sweep, then odd; reunitarisation after global sweep s iff s % k == 0
    (PAPER.md:144); fix() measures first and then every check_every sweeps."""
    N, gauge, omega = 4, "landau", 1.7
    rng = np.random.default_rng(9)
    U0 = gi.make_links_sun(DIMS, N, 0.5, 71)
    A, B, C = U0.copy(), U0.copy(), U0.copy()
    sun.sweeps(A, DIMS, gauge, N, omega, n=1)
    sun.half_sweep(B, DIMS, gauge, N, 0, omega)
    sun.half_sweep(B, DIMS, gauge, N, 1, omega)
    sun.half_sweep(C, DIMS, gauge, N, 1, omega)
    sun.half_sweep(C, DIMS, gauge, N, 0, omega)
    assert np.array_equal(A, B) and np.abs(A - C).max() > 1e-3
    # even sites are (x+y+z+t) even: after an even half-sweep at omega = 1 every even site is stationary
    # (N = 2: one subgroup, so a visited site sits exactly at its local maximum afterwards)
    D = gi.make_links_sun(DIMS, 2, 0.5, 72)
    sun.half_sweep(D, DIMS, gauge, 2, 0, 1.0)
    G = sun.site_rotations(D, DIMS, gauge, 2, 1.0)
    even = sun.parity_mask(DIMS) == 0
    assert np.abs(G[even] - np.eye(2)).max() <= 1e-12 and np.abs(G[~even] - np.eye(2)).max() > 1e-2
    # cadence
    off = U0 + 1e-4 * rng.normal(size=U0.shape)
    A, B = off.copy(), off.copy()
    sun.sweeps(A, DIMS, gauge, N, omega, n=5, reunit_every=2, first_sweep=1)  # global sweeps 2..6: after 2, 4, 6
    for s in range(2, 7):
        sun.half_sweep(B, DIMS, gauge, N, 0, omega)
        sun.half_sweep(B, DIMS, gauge, N, 1, omega)
        if s in (2, 4, 6):
            sun.reunitarize(B, DIMS, N)
    assert np.array_equal(A, B)
    assert max(sun.unitarity(A, DIMS, N)) <= 1e-13
    Cc, Dd = off.copy(), off.copy()
    sun.sweeps(Cc, DIMS, gauge, N, omega, n=1, reunit_every=2, first_sweep=0)  # global sweep 1: no projection
    assert max(sun.unitarity(Cc, DIMS, N)) > 1e-5
    sun.sweeps(Dd, DIMS, gauge, N, omega, n=1, reunit_every=2, first_sweep=1)  # global sweep 2: projected
    assert max(sun.unitarity(Dd, DIMS, N)) <= 1e-13
    # fix(): history checkpoints and the same link sequence
    A, B = U0.copy(), U0.copy()
    done, hist = sun.fix(A, DIMS, gauge, N, omega, 0.0, 25, 10, reunit_every=3)
    assert done == 25 and [h[0] for h in hist] == [0, 10, 20, 25]
    assert hist[0][1:] == sun.measure(U0, DIMS, gauge, N)
    sun.sweeps(B, DIMS, gauge, N, omega, n=10, reunit_every=3, first_sweep=0)
    sun.sweeps(B, DIMS, gauge, N, omega, n=10, reunit_every=3, first_sweep=10)
    sun.sweeps(B, DIMS, gauge, N, omega, n=5, reunit_every=3, first_sweep=20)
    assert np.array_equal(A, B)
