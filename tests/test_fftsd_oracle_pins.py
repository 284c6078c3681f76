"""Pins for the Algorithm 2 oracle (oracle/fftsd.py: steepest descent with Fourier acceleration, PAPER.md:52-68,
97-124) against what the paper and the mathematics fix.  The paper prints no numbers for it, so every pin is a closed
form, an invariant or an independent restatement; none of these tests touches the CUDA path.
"""
import numpy as np
import pytest

import gf_inputs as gi
import oracle
from oracle import fftsd
from _util import dag, flat, from_c, gauge_transform, grid, lex_coords, plaquettes, shift, to_c

D = {"landau": 4, "coulomb": 3}


def rough(dims, r=0.4, seed=21):
    return gi.make_links(dims, r, seed)


# ---------------------------------------------------------------------------------------------------------------------
# Delta, F, theta: the numpy statement against the C++ oracle of Algorithm 1 (an independent implementation, itself
# pinned in test_oracle_pins.py) and against closed forms
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
def test_measure_agrees_with_alg1_oracle(gauge):
    dims = (4, 6, 4, 8)
    U = rough(dims)
    F, th = fftsd.measure(U, dims, gauge)
    Fo, tho = oracle.measure(U, dims, gauge)
    assert abs(F - Fo) < 1e-13 and abs(th - tho) < 1e-12 * tho
    Dn = fftsd.delta_field(U, dims, gauge).reshape(-1, 3, 3)
    for site in (0, 5, 191, 700):
        assert np.abs(Dn[site] - oracle.site_delta(U, dims, gauge, site)).max() < 1e-14


@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
def test_delta_is_antihermitian_traceless_and_sums_to_zero(gauge):
    dims = (4, 4, 6, 4)
    Dn = fftsd.delta_field(rough(dims), dims, gauge)
    assert np.abs(Dn + dag(Dn)).max() < 1e-15
    assert np.abs(np.trace(Dn, axis1=-2, axis2=-1)).max() < 1e-14
    # reading B3: the zero mode of Delta vanishes identically (per time slice in Coulomb gauge)
    axes = (0, 1, 2, 3) if gauge == "landau" else (1, 2, 3)
    assert np.abs(Dn.sum(axis=axes)).max() < 1e-12


# ---------------------------------------------------------------------------------------------------------------------
# p^2: eigenvalues of the lattice (-d^2)  (reading B2)
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
def test_p2_is_the_eigenvalue_of_minus_laplacian_on_plane_waves(gauge):
    dims = (4, 6, 8, 4)
    d = D[gauge]
    p2, p2max = fftsd.p2_table(dims, gauge)
    p2 = np.broadcast_to(p2, (dims[3] if d == 4 else 1, dims[2], dims[1], dims[0]))
    c = lex_coords(dims)
    rng = np.random.default_rng(3)
    for _ in range(6):
        k = [int(rng.integers(0, n)) for n in dims]
        if d == 3:
            k[3] = 0
        phi = np.exp(2j * np.pi * sum(k[m] * c[:, m] / dims[m] for m in range(4)))
        lap = sum(2 * phi - shift(phi, dims, m, 1) - shift(phi, dims, m, -1) for m in range(d))  # (-d^2) phi
        assert np.abs(lap - p2[k[3], k[2], k[1], k[0]] * phi).max() < 1e-12
    assert p2max == 4 * d and abs(p2.max() - p2max) < 1e-12  # attained at k = n/2 (all extents even)


@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
def test_fourier_factor_on_a_single_mode(gauge):
    # F^-1 f(p) F applied to a plane wave of momentum k returns f(k) times the wave: pins the transform pair, its
    # normalisation (B4), the axes transformed (B2) and the zero-mode rule (B3)
    dims = (4, 6, 4, 8)
    d = D[gauge]
    c = lex_coords(dims)
    p2, p2max = fftsd.p2_table(dims, gauge)
    M = np.array([[0, 1 + 2j, 0.5], [-1 + 2j, 0, -1j], [-0.5, -1j, 0]])
    for k in ([1, 2, 3, 5], [0, 0, 0, 0], [2, 3, 2, 4]):
        if d == 3:
            k = k[:3] + [0]
        phi = np.exp(2j * np.pi * sum(k[m] * c[:, m] / dims[m] for m in range(4)))
        field = grid(phi[:, None, None] * M, dims)
        w = fftsd.fourier_accelerate(field, dims, gauge, alpha=0.08)
        pk = sum(4 * np.sin(np.pi * k[m] / dims[m]) ** 2 for m in range(d))
        want = 0.0 if pk == 0 else 0.04 * p2max / pk
        assert np.abs(w - want * field).max() < 1e-13
    # and with the factor switched off: eq. 1.7
    assert np.abs(fftsd.fourier_accelerate(field, dims, gauge, 0.08, accelerate=False) - 0.04 * field).max() == 0


# ---------------------------------------------------------------------------------------------------------------------
# the direction: dF/dalpha at alpha = 0 (closed forms)
# ---------------------------------------------------------------------------------------------------------------------
def _F_after(U, dims, gauge, alpha, accelerate):
    V = U.copy()
    fftsd.step(V, dims, gauge, alpha, accelerate=accelerate)
    return fftsd.measure(V, dims, gauge)[0]


@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
def test_plain_steepest_descent_slope_is_theta_over_4d(gauge):
    # g = 1 + (alpha/2) Delta + O(alpha^2):  dF/dalpha|0 = (1/(d 3 V)) (1/4) sum_x Tr Delta Delta^dag = theta / (4 d).
    # A wrong sign of Delta, of the step, or a swapped g / g^dag makes the slope negative or different.
    dims = (4, 4, 4, 6)
    U = rough(dims, 0.5)
    _, th = fftsd.measure(U, dims, gauge)
    h = 1e-5
    slope = (_F_after(U, dims, gauge, h, False) - _F_after(U, dims, gauge, -h, False)) / (2 * h)
    assert abs(slope - th / (4 * D[gauge])) < 1e-7 * th


@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
def test_accelerated_slope_in_momentum_space(gauge):
    # with the Fourier factor f(p): dF/dalpha|0 = (1/(4 d 3 V)) sum_p f(p) sum_ij |Delta_ij(p)|^2 / N  (Parseval),
    # N = sites per transform.  Computed here from numpy.fft directly, not through the oracle's filter.
    dims = (4, 6, 4, 4)
    d = D[gauge]
    U = rough(dims, 0.5)
    Dn = fftsd.delta_field(U, dims, gauge)
    axes = (0, 1, 2, 3) if d == 4 else (1, 2, 3)
    N = np.prod([Dn.shape[a] for a in axes])
    k = [np.arange(n) for n in dims]
    s = [4 * np.sin(np.pi * k[m] / dims[m]) ** 2 for m in range(4)]
    p2 = s[0][None, None, None, :] + s[1][None, None, :, None] + s[2][None, :, None, None]
    if d == 4:
        p2 = p2 + s[3][:, None, None, None]
    f = np.zeros_like(p2)
    f[p2 > 0] = 4 * d / p2[p2 > 0]
    Dh = np.fft.fftn(Dn, axes=axes)
    want = (f[..., None, None] * np.abs(Dh) ** 2).sum() / N / (4 * d * 3 * np.prod(dims))
    h = 1e-6
    slope = (_F_after(U, dims, gauge, h, True) - _F_after(U, dims, gauge, -h, True)) / (2 * h)
    assert abs(slope - want) < 1e-6 * want


def test_first_order_plus_reunitarisation_is_exp_to_second_order():
    # g = reunit(1 + w) stands for exp(w); they differ at O(|w|^2)
    from scipy.linalg import expm
    rng = np.random.default_rng(9)
    for scale in (1e-2, 1e-3):
        a = rng.normal(size=(3, 3)) + 1j * rng.normal(size=(3, 3))
        w = a - a.conj().T
        w -= np.trace(w) / 3 * np.eye(3)
        w *= scale / np.abs(w).max()
        g = fftsd.gauge_rotation(w[None])[0]
        assert np.abs(g - expm(w)).max() < 3 * scale ** 2
        assert np.abs(g @ g.conj().T - np.eye(3)).max() < 1e-15 and abs(np.linalg.det(g) - 1) < 1e-15


# ---------------------------------------------------------------------------------------------------------------------
# the step is a gauge transformation; the iteration converges
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gauge,storage", [("landau", 18), ("coulomb", 18), ("landau", 12)])
def test_step_is_a_gauge_transformation(gauge, storage):
    dims = (4, 4, 6, 4)
    U = rough(dims, 0.5)
    if storage == 12:
        oracle.project12(U, dims)
    before = plaquettes(to_c(U), dims)
    wl = oracle.wilson_traces(U, dims, 0, 3, 1, 2)
    pl = oracle.polyakov_traces(U, dims, 3)
    for _ in range(3):
        fftsd.step(U, dims, gauge, 0.08, storage=storage)
    after = plaquettes(to_c(U), dims)
    for key in before:
        assert np.abs(before[key] - after[key]).max() < 1e-12
    assert np.abs(wl - oracle.wilson_traces(U, dims, 0, 3, 1, 2)).max() < 1e-12
    assert np.abs(pl - oracle.polyakov_traces(U, dims, 3)).max() < 1e-12
    a, b = oracle.unitarity(U, dims)
    assert max(a, b) < 1e-13


@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
def test_F_increases_every_iteration_at_alpha_008(gauge):
    dims = (4, 4, 4, 8)
    U = rough(dims, 0.3)
    _, hist = fftsd.fix(U, dims, gauge, 0.08, 0.0, 40, 1)
    F = np.array([h[1] for h in hist])
    th = np.array([h[2] for h in hist])
    rising = th[:-1] > 1e-12  # once theta is at the rounding floor F only moves in its last bits
    assert rising.sum() >= 10 and (np.diff(F)[rising] > 0).all() and (np.diff(F) > -1e-14).all()
    assert hist[-1][2] < 1e-3 * hist[0][2]


@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
def test_converges_to_F1_on_a_hidden_pure_gauge(gauge):
    dims = (4, 4, 4, 4)
    U = gi.make_links(dims, 0.0, 4)  # r = 0: G(x) G(x+mu)^dag exactly
    F0, th0 = fftsd.measure(U, dims, gauge)
    assert F0 < 0.3 and th0 > 1
    done, hist = fftsd.fix(U, dims, gauge, 0.08, 1e-13, 5000, 50)
    assert hist[-1][2] < 1e-13
    if hist[-1][1] < 1 - 1e-6:  # a lattice Gribov copy / local maximum is legitimate; the global one has F = 1
        pytest.skip("converged to a local maximum of F")
    assert abs(hist[-1][1] - 1.0) < 1e-10


def test_fourier_acceleration_needs_fewer_iterations_than_plain_descent():
    # Fourier acceleration attenuates critical slowing down (alpha = 0.08 in both)
    dims = (8, 8, 8, 8)
    U = rough(dims, 0.3, seed=1)
    n_acc, h_acc = fftsd.fix(U.copy(), dims, "landau", 0.08, 1e-8, 2000, 10, accelerate=True)
    n_plain, h_plain = fftsd.fix(U.copy(), dims, "landau", 0.08, 1e-8, 2000, 10, accelerate=False)
    assert h_acc[-1][2] < 1e-8
    assert n_acc < n_plain


def test_coulomb_time_slices_decouple():
    dims = (4, 4, 4, 6)
    U = rough(dims, 0.5)
    V = U.copy()
    t_pert = 2
    sl = grid(V, dims)[t_pert]
    sl[..., :3, :, :, :] = grid(gi.make_links(dims, 0.5, 99), dims)[t_pert][..., :3, :, :, :]  # other spatial links on slice 2
    fftsd.step(U, dims, "coulomb", 0.08)
    fftsd.step(V, dims, "coulomb", 0.08)
    gU, gV = grid(U, dims), grid(V, dims)
    for t in range(dims[3]):
        same = np.array_equal(gU[t][..., :3, :, :, :], gV[t][..., :3, :, :, :])
        assert same == (t != t_pert)
