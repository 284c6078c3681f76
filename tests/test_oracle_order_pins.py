"""Pins for the ORDER in which the oracle's drivers apply their steps: which parity goes first inside a sweep
(§2 "first ... in the even lattice sites and then in the odd sites"; reading A10: even <=> (x+y+z+t)&1 == 0)
and after which sweeps / iterations the links are reunitarised (§3 "reunitarization at each 20 steps":
after global sweep s when s % k == 0, counted from the start of the run, not from the start of a call).

`half_sweep`, `reunitarize`, `measure` and `fftsd.step` are pinned on their own (test_oracle_pins.py,
test_fftsd_oracle_pins.py); here `sweeps`, `fix`, `fix_slices` and `fftsd.fix` are held to the sequence of those calls
the paper states, written out by hand, and to a numpy statement of "even sites, then odd sites" that uses its own parity
and neighbour arithmetic (_util.parity, _util.gauge_transform).  A driver that visits odd sites first, or that
reunitarises one sweep early or late, fails every test of this file.  None of these tests touches the CUDA path.
"""
import numpy as np
import pytest

import gf_inputs as gi
import oracle
from oracle import fftsd
from _util import gauge_transform, parity, to_c

SUBGROUPS = [(0, 1), (1, 2), (0, 2)]


def rough(dims, r=0.45, seed=31):
    return gi.make_links(dims, r, seed)


def off_group(U, eps=2e-3, seed=3):
    """Links pushed off SU(3) by a relative eps, so that a reunitarisation is visible far above rounding.
    A gauge transformation keeps U U^dag, so the defect survives any number of sweeps until a projection removes it."""
    rng = np.random.default_rng(seed)
    return np.ascontiguousarray(U * (1.0 + eps * rng.standard_normal(U.shape)))


def defect(U, dims):
    return oracle.unitarity(U, dims)[0]


def _site_rotations(U, dims, gauge, par, omega):
    """g(x) = G(x) on the sites of parity `par` (from K(x) of the field as it stands), 1 elsewhere."""
    V = U.shape[0]
    g = np.broadcast_to(np.eye(3, dtype=complex), (V, 3, 3)).copy()
    for s in np.nonzero(parity(dims) == par)[0]:
        K = oracle.site_K(U, dims, gauge, s)
        G = np.eye(3, dtype=complex)
        for (i, j) in SUBGROUPS:
            K, G, _ = oracle.su2_step(K, G, i, j, omega)
        g[s] = G
    return g


def _np_half_sweep(U, dims, gauge, par, omega):
    out = np.empty_like(U)
    c = gauge_transform(to_c(U), _site_rotations(U, dims, gauge, par, omega), dims)
    out[..., 0], out[..., 1] = c.real, c.imag
    return out


# ---------------------------------------------------------------------------------------------------------------------
# sweeps: even half-sweep first (A10)
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
def test_one_sweep_is_even_sites_then_odd_sites(gauge):
    dims = (4, 2, 4, 6)
    U = rough(dims)
    omega = 1.7
    W = U.copy()
    oracle.sweeps(W, dims, gauge, omega, n=1)
    # bit-equal to the two half-sweeps in the paper's order, and not to the other order
    E = U.copy()
    oracle.half_sweep(E, dims, gauge, 0, omega)
    oracle.half_sweep(E, dims, gauge, 1, omega)
    assert np.array_equal(W, E)
    O = U.copy()
    oracle.half_sweep(O, dims, gauge, 1, omega)
    oracle.half_sweep(O, dims, gauge, 0, omega)
    assert np.abs(W - O).max() > 1e-2
    # the same from numpy: transform by G on the sites with (x+y+z+t) even, rebuild K, then on the odd ones
    ref = _np_half_sweep(_np_half_sweep(U, dims, gauge, 0, omega), dims, gauge, 1, omega)
    assert np.abs(W - ref).max() < 1e-14
    rev = _np_half_sweep(_np_half_sweep(U, dims, gauge, 1, omega), dims, gauge, 0, omega)
    assert np.abs(W - rev).max() > 1e-2


def test_last_parity_visited_is_the_odd_one():
    # omega = 1: the last subgroup step of a site update, (0,2), leaves K(x) at its maximum over that subgroup, so a
    # second (0,2) step on the same K returns g = 1 to rounding ("stationarity").  After sweeps(n=1)
    # this holds on the parity visited LAST and no longer on the one visited first (its eight neighbours moved since):
    # the last one must be the odd one.
    dims = (4, 4, 2, 4)
    W = rough(dims, 0.5, 5)
    oracle.sweeps(W, dims, "landau", 1.0, n=1)
    p = parity(dims)
    dev = [[], []]
    for s in range(W.shape[0]):
        _, _, a = oracle.su2_step(oracle.site_K(W, dims, "landau", s), np.eye(3), 0, 2, 1.0)
        dev[p[s]].append(np.abs(a[1:]).max())
    assert max(dev[1]) < 1e-14 and min(dev[0]) > 1e-6


# ---------------------------------------------------------------------------------------------------------------------
# sweeps: reunitarisation after global sweep s iff s % k == 0
# ---------------------------------------------------------------------------------------------------------------------
def _unrolled(U, dims, gauge, omega, n, k, first, storage=18):
    """The sequence the paper states, call by call; returns the global sweep numbers after which it projected."""
    hit = []
    for i in range(1, n + 1):
        oracle.half_sweep(U, dims, gauge, 0, omega, storage)
        oracle.half_sweep(U, dims, gauge, 1, omega, storage)
        if k > 0 and (first + i) % k == 0:
            oracle.reunitarize(U, dims)
            hit.append(first + i)
    return hit


@pytest.mark.parametrize("n,k,first,expect", [(5, 2, 1, [2, 4, 6]), (6, 3, 0, [3, 6]), (4, 5, 3, [5]), (3, 4, 4, []),
                                              (3, 1, 7, [8, 9, 10]), (4, 0, 0, [])])
def test_sweeps_reunitarise_after_multiples_of_k_of_the_global_count(n, k, first, expect):
    dims = (4, 4, 2, 2)
    U0 = off_group(rough(dims))
    W = U0.copy()
    oracle.sweeps(W, dims, "landau", 1.6, n=n, reunit_every=k, first_sweep=first)
    R = U0.copy()
    assert _unrolled(R, dims, "landau", 1.6, n, k, first) == expect
    assert np.array_equal(W, R)
    if expect:
        # shifting the projections by one sweep either way gives a different field, far above rounding
        for shift in (-1, +1):
            S = U0.copy()
            for i in range(1, n + 1):
                oracle.half_sweep(S, dims, "landau", 0, 1.6)
                oracle.half_sweep(S, dims, "landau", 1, 1.6)
                if (first + i + shift) % k == 0:
                    oracle.reunitarize(S, dims)
            if k > 1:
                assert np.abs(W - S).max() > 1e-5


def test_unitarity_defect_vanishes_exactly_at_the_cadence():
    # one sweep at a time with the running count handed over in first_sweep: the defect of the off-group input is
    # untouched by sweeps (gauge transformations keep U U^dag) and is removed after sweeps 3, 6, 9 only.
    dims = (4, 2, 2, 4)
    W = off_group(rough(dims), 2e-3)
    d0 = defect(W, dims)
    assert d0 > 1e-3
    rng = np.random.default_rng(9)
    for s in range(1, 10):
        oracle.sweeps(W, dims, "coulomb", 1.5, n=1, reunit_every=3, first_sweep=s - 1)
        d = defect(W, dims)
        if s % 3 == 0:
            assert d < 1e-14
            W *= 1.0 + 2e-3 * rng.standard_normal(W.shape)  # push it off again for the next period
        else:
            assert d > 1e-3


# ---------------------------------------------------------------------------------------------------------------------
# fix / fix_slices: the same order and cadence inside Algorithm 1's loop, seen through the history and the links
# ---------------------------------------------------------------------------------------------------------------------
def test_fix_history_and_links_follow_the_unrolled_sequence():
    dims = (4, 4, 2, 2)
    U0 = off_group(rough(dims, 0.4, 41))
    W = U0.copy()
    done, hist = oracle.fix(W, dims, "landau", 1.7, 0.0, 7, 3, reunit_every=2)
    assert done == 7 and list(hist[:, 0]) == [0, 3, 6, 7]
    R = U0.copy()
    rows = [(0,) + oracle.measure(R, dims, "landau")]
    sweeps_done = 0
    for n in (3, 3, 1):
        _unrolled(R, dims, "landau", 1.7, n, 2, sweeps_done)
        sweeps_done += n
        rows.append((sweeps_done,) + oracle.measure(R, dims, "landau"))
    assert np.array_equal(W, R)
    assert np.array_equal(hist, np.array(rows))
    # sweep 6 was followed by a projection (measured on the group), sweep 7 was not
    assert defect(R, dims) < 1e-13
    # a reversed parity order or a cadence off by one changes F at the first read-back far above rounding
    for (first_par, off) in [(1, 0), (0, 1)]:
        S = U0.copy()
        for i in range(1, 4):
            oracle.half_sweep(S, dims, "landau", first_par, 1.7)
            oracle.half_sweep(S, dims, "landau", 1 - first_par, 1.7)
            if (i + off) % 2 == 0:
                oracle.reunitarize(S, dims)
        assert abs(oracle.measure(S, dims, "landau")[0] - hist[1, 1]) > 1e-7


def test_fix_slices_follows_the_unrolled_sequence():
    dims = (4, 4, 2, 4)
    U0 = off_group(rough(dims, 0.4, 43))
    W = U0.copy()
    done, per, hist = oracle.fix_slices(W, dims, "coulomb", 1.7, 0.0, 5, 2, reunit_every=2)
    assert done == 5 and list(per) == [5] * 4 and list(hist[:, 0]) == [0, 2, 4, 5]
    R = U0.copy()
    _unrolled(R, dims, "coulomb", 1.7, 5, 2, 0)  # eps = 0: every slice stays active, so the mask is all ones
    assert np.array_equal(W, R)


# ---------------------------------------------------------------------------------------------------------------------
# fftsd.fix: iterations and the reunitarisation cadence of PAPER.md:144 inside Algorithm 2's loop
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
def test_fftsd_fix_follows_the_unrolled_sequence(gauge):
    dims = (4, 4, 2, 4)
    U0 = off_group(rough(dims, 0.3, 47), 1e-3)
    W = U0.copy()
    done, hist = fftsd.fix(W, dims, gauge, 0.08, 0.0, 7, check_every=3, reunit_every=2)
    assert done == 7 and [h[0] for h in hist] == [0, 3, 6, 7]
    R = U0.copy()
    rows = [(0,) + fftsd.measure(R, dims, gauge)]
    hits = []
    for it in range(1, 8):
        fftsd.step(R, dims, gauge, 0.08)
        if it % 2 == 0:
            fftsd.reunitarize_links(R, dims)
            hits.append(it)
        if it in (3, 6, 7):
            rows.append((it,) + fftsd.measure(R, dims, gauge))
    assert hits == [2, 4, 6]
    assert np.array_equal(W, R)
    assert np.array_equal(np.array(hist), np.array(rows))
    # off by one: a different field
    S = U0.copy()
    for it in range(1, 8):
        fftsd.step(S, dims, gauge, 0.08)
        if it % 2 == 1:
            fftsd.reunitarize_links(S, dims)
    assert np.abs(W - S).max() > 1e-6
