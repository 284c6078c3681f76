"""GPU parity: the CUDA path (through the C ABI, via the thin binding) against the CPU oracle, element by element on the
same seeded inputs.  Tolerances are BASELINE.json north_star's: after one sweep max |dU_ij| <= 1e-12 (FP64) / 2e-5
(FP32); F relative 1e-10 / 1e-5; theta within a factor 1.5; sweeps-to-convergence within +-2 %.

FP32 runs are compared with the FP64 oracle fed the FP32-rounded input (reading A18); 12-real storage is emulated in
the oracle by rebuilding row 2 after every link write (reading A13).
"""
import json
import os

import numpy as np
import pytest

import gf_inputs as gi
import oracle

pytestmark = pytest.mark.gpu

HERE = os.path.dirname(os.path.abspath(__file__))

# lattices: several 32-site blocks, a ragged tail (V/2 not a multiple of 32), minimal extents, unequal extents
SHAPES = [(8, 8, 8, 8), (6, 4, 2, 2), (2, 2, 2, 2), (4, 6, 10, 2), (10, 6, 4, 4), (16, 4, 4, 6)]
TOL_LINK = {"f64": 1e-12, "f32": 2e-5}
TOL_F = {"f64": 1e-10, "f32": 1e-5}


@pytest.fixture(scope="module")
def gf():
    import paper_1412_1498_b200 as m
    return m


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available()
    return t


def host_input(dims, roughness, seed, prec, storage):
    """(what the GPU gets, what the FP64 oracle gets) for one field."""
    dt = np.float32 if prec == "f32" else np.float64
    U = gi.make_links(dims, roughness, seed, dtype=dt)
    Uo = np.ascontiguousarray(U.astype(np.float64))
    if storage == 12:
        oracle.project12(Uo, dims)
    return U, Uo


def gpu_fixer(gf, torch, dims, gauge, prec, storage, U):
    fx = gf.GaugeFixer(dims, gauge=gauge, prec=prec, storage=storage)
    fx.set_links(torch.from_numpy(U).cuda())
    return fx


@pytest.mark.parametrize("dims", SHAPES)
@pytest.mark.parametrize("prec,storage", [("f64", 18), ("f64", 12), ("f32", 18), ("f32", 12)])
def test_set_get_roundtrip(gf, torch, dims, prec, storage):
    U, Uo = host_input(dims, 0.5, 11, prec, storage)
    fx = gpu_fixer(gf, torch, dims, "landau", prec, storage, U)
    back = fx.get_links().cpu().numpy()
    if storage == 18:
        assert np.array_equal(back, U)  # bit-identical
    else:
        assert np.array_equal(back[:, :, :2], U[:, :, :2])  # stored rows bit-identical
        tol = 1e-15 if prec == "f64" else 5e-7
        assert np.abs(back.astype(np.float64) - Uo).max() <= tol  # row 2 = conj(row0 x row1)
    fx.close()


@pytest.mark.parametrize("dims", SHAPES)
@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
@pytest.mark.parametrize("prec,storage", [("f64", 18), ("f64", 12), ("f32", 18), ("f32", 12)])
def test_measure_matches_oracle(gf, torch, dims, gauge, prec, storage):
    U, Uo = host_input(dims, 0.5, 12, prec, storage)
    fx = gpu_fixer(gf, torch, dims, gauge, prec, storage, U)
    F, th = fx.measure()
    Fo, tho = oracle.measure(Uo, dims, gauge)
    # F is O(1e-2) on a random gauge copy while the summands are O(1): compare on the scale of the summands
    atol = 1e-13 if prec == "f64" else 2e-7
    assert abs(F - Fo) <= atol
    assert abs(th - tho) <= (1e-12 if prec == "f64" else 2e-6) * tho
    fx.close()


@pytest.mark.parametrize("dims", SHAPES)
@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
@pytest.mark.parametrize("prec,storage", [("f64", 18), ("f64", 12), ("f32", 18), ("f32", 12)])
def test_one_sweep_links_match_oracle(gf, torch, dims, gauge, prec, storage):
    omega = 1.7
    U, Uo = host_input(dims, 0.5, 13, prec, storage)
    fx = gpu_fixer(gf, torch, dims, gauge, prec, storage, U)
    fx.ovr_sweep(1, omega)
    got = fx.get_links().cpu().numpy().astype(np.float64)
    oracle.sweeps(Uo, dims, gauge, omega, n=1, storage=storage)
    assert np.abs(got - Uo).max() <= TOL_LINK[prec]
    F, th = fx.measure()
    Fo, tho = oracle.measure(Uo, dims, gauge)
    assert abs(F - Fo) <= TOL_F[prec] * abs(Fo)
    assert tho / 1.5 <= th <= tho * 1.5
    fx.close()


# The one-sweep bar is 1e-12.  Over several sweeps on a still-random field the map itself amplifies rounding: where a
# subgroup's g is close to -1 (phi near pi) the rotation axis a_vec/|a_vec| is ill-conditioned (error x 1/|a_vec|), and
# the closer omega is to 2 the less the sweep contracts.  The bounds below are 5 sweeps x that amplification.
@pytest.mark.parametrize("omega,tol", [(1.0, 5e-12), (1.5, 5e-12), (1.99, 2e-9)])
def test_several_sweeps_and_omegas(gf, torch, omega, tol):
    dims = (6, 6, 4, 8)
    U, Uo = host_input(dims, 0.3, 14, "f64", 18)
    fx = gpu_fixer(gf, torch, dims, "landau", "f64", 18, U)
    fx.ovr_sweep(5, omega)
    got = fx.get_links().cpu().numpy()
    oracle.sweeps(Uo, dims, "landau", omega, n=5)
    assert np.abs(got - Uo).max() <= tol
    fx.close()


def test_degenerate_inputs_unit_and_converged(gf, torch):
    # unit links: every r_vec = 0 exactly (reading A7 branch), F = 1, theta = 0, and the sweep is the identity
    dims = (4, 4, 4, 4)
    V = gi.volume(dims)
    U = np.zeros((V, 4, 3, 3, 2))
    for i in range(3):
        U[:, :, i, i, 0] = 1.0
    for prec, storage in [("f64", 18), ("f32", 12)]:
        Ui = U.astype(np.float32 if prec == "f32" else np.float64)
        fx = gpu_fixer(gf, torch, dims, "landau", prec, storage, Ui)
        assert fx.measure() == (1.0, 0.0)
        fx.ovr_sweep(2, 1.8)
        assert np.array_equal(fx.get_links().cpu().numpy(), Ui)
        assert fx.measure() == (1.0, 0.0)
        fx.close()
    # all links = -1 on the (0,1) block: a0 < 0 with s = 0 (phi = pi, axis undefined -> g = 1 on both sides)
    Um = U.copy()
    Um[:, :, 0, 0, 0] = -1.0
    Um[:, :, 1, 1, 0] = -1.0
    Uo = Um.copy()
    fx = gpu_fixer(gf, torch, dims, "landau", "f64", 18, Um)
    fx.ovr_sweep(1, 1.5)
    oracle.sweeps(Uo, dims, "landau", 1.5, n=1)
    got = fx.get_links().cpu().numpy()
    assert np.isfinite(got).all() and np.abs(got - Uo).max() <= 1e-12
    fx.close()


@pytest.mark.parametrize("prec,storage", [("f64", 18), ("f64", 12), ("f32", 18), ("f32", 12)])
def test_reunitarize_matches_oracle(gf, torch, prec, storage):
    dims = (6, 4, 2, 2)
    U, _ = host_input(dims, 0.5, 15, prec, storage)
    rng = np.random.default_rng(3)
    U = (U * (1 + 1e-3 * rng.standard_normal(U.shape))).astype(U.dtype)  # knock the links off SU(3)
    Uo = np.ascontiguousarray(U.astype(np.float64))
    if storage == 12:
        oracle.project12(Uo, dims)
    fx = gpu_fixer(gf, torch, dims, "landau", prec, storage, U)
    fx.reunitarize()
    got = fx.get_links().cpu().numpy().astype(np.float64)
    oracle.reunitarize(Uo, dims)
    assert np.abs(got - Uo).max() <= (1e-14 if prec == "f64" else 1e-6)
    a, b = oracle.unitarity(np.ascontiguousarray(got), dims)
    assert max(a, b) <= (1e-14 if prec == "f64" else 1e-6)
    fx.close()


def test_reunit_cadence_inside_sweeps(gf, torch):
    dims = (4, 4, 4, 4)
    U, Uo = host_input(dims, 0.4, 16, "f32", 12)
    fx = gpu_fixer(gf, torch, dims, "landau", "f32", 12, U)
    fx.set_reunit_every(3)
    fx.ovr_sweep(4, 1.75)
    fx.ovr_sweep(4, 1.75)  # global sweeps 3 and 6 reunitarise, across the two calls
    n_launch = fx.kernel_launches()
    got = fx.get_links().cpu().numpy().astype(np.float64)
    oracle.sweeps(Uo, dims, "landau", 1.75, n=8, storage=12, reunit_every=3)
    assert np.abs(got - Uo).max() <= 8 * 2e-5
    assert n_launch == 1 + 16 + 2  # set_links + 16 half-sweeps + 2 reunitarisations
    fx.close()


def test_host_set_get(gf, torch):
    dims = (8, 8, 8, 8)
    U, _ = host_input(dims, 0.5, 17, "f64", 18)
    fx = gf.GaugeFixer(dims)
    pinned = torch.from_numpy(U).pin_memory()
    fx.set_links_host(pinned)
    out = torch.empty_like(pinned).pin_memory()
    fx.get_links_host(out)
    assert np.array_equal(out.numpy(), U)
    fx.set_links_host(U)  # pageable numpy works too
    assert np.array_equal(fx.get_links().cpu().numpy(), U)
    fx.close()


def test_argument_errors(gf, torch):
    fx = gf.GaugeFixer((4, 4, 4, 4))
    assert gf.gf_ovr_sweep(fx.ctx, 1, 2.0) == gf.GF_EINVAL      # omega in [1,2[
    assert gf.gf_ovr_sweep(fx.ctx, 1, 0.99) == gf.GF_EINVAL
    assert gf.gf_ovr_sweep(fx.ctx, -1, 1.5) == gf.GF_EINVAL
    assert gf.gf_ovr_sweep(fx.ctx, 0, 1.5) == gf.GF_OK
    assert gf.gf_fix(fx.ctx, 1.5, 1e-10, 10, 0)[0] == gf.GF_EINVAL
    assert gf.gf_fix(fx.ctx, 1.5, -1.0, 10, 1)[0] == gf.GF_EINVAL
    assert gf.gf_set_links(fx.ctx, 0) == gf.GF_EINVAL
    assert gf.gf_set_reunit_every(fx.ctx, -1) == gf.GF_EINVAL
    assert gf.gf_set_option(fx.ctx, 99, 0) == gf.GF_EINVAL
    assert gf.gf_set_option(fx.ctx, gf.GF_OPT_SWEEP_VARIANT, 7) == gf.GF_EINVAL
    assert "omega" in gf.gf_last_error(fx.ctx) or gf.gf_last_error(fx.ctx)
    # NaN links -> GF_ENUMERIC from measure
    U = np.full((256, 4, 3, 3, 2), np.nan)
    fx.set_links(torch.from_numpy(U).cuda())
    assert gf.gf_measure(fx.ctx)[0] == gf.GF_ENUMERIC
    fx.close()
    with pytest.raises(gf.GFError):
        gf.GaugeFixer((4, 4, 3, 4))


# ---- kernel variants and the fused theta terms ---------------------------------------------------------------------------
@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (6, 4, 2, 2), (10, 6, 4, 4), (2, 2, 2, 2)])
@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
@pytest.mark.parametrize("prec,storage", [("f64", 18), ("f64", 12), ("f32", 18), ("f32", 12)])
def test_halfsweep_variants_agree_bit_for_bit_and_match_oracle(gf, torch, dims, gauge, prec, storage):
    """GF_OPT_SWEEP_VARIANT 1 (two-pass), 2 (two-pass + L2 bulk prefetch), 3 (staged, the default), 4 (staged, the tile
    fetched by bulk copies of the TMA unit), 5 (staged, only the forward chunk by bulk copy), 6 (two lanes per site).  Within a family the
    arithmetic per site is the same in the same order, so the links must be bit-identical: {0, 3, 4, 5, 6} (staged) and
    {1, 2} (two-pass); in FP64 the two families coincide too (with FP32 links the staged kernels evaluate
    well-conditioned sites in FP32, the two-pass kernels every site in FP64).  Each variant is also held to the
    one-sweep oracle bar."""
    omega = 1.7
    U, Uo = host_input(dims, 0.5, 13, prec, storage)  # the input of test_one_sweep_links_match_oracle
    oracle.sweeps(Uo, dims, gauge, omega, n=1, storage=storage)
    ref = {}
    for variant in (0, 1, 2, 3, 4, 5, 6):
        fx = gpu_fixer(gf, torch, dims, gauge, prec, storage, U)
        fx.set_option(gf.GF_OPT_SWEEP_VARIANT, variant)
        fx.ovr_sweep(1, omega)
        got = fx.get_links().cpu().numpy()
        assert np.abs(got.astype(np.float64) - Uo).max() <= TOL_LINK[prec]
        fx.ovr_sweep(2, omega)
        got = fx.get_links().cpu().numpy()
        family = "all" if prec == "f64" else ("two-pass" if variant in (1, 2) else "staged")
        assert np.array_equal(got, ref.setdefault(family, got)), f"variant {variant} differs from its family ({family})"
        fx.close()


@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (6, 4, 2, 2), (10, 6, 4, 4)])
@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
@pytest.mark.parametrize("prec,storage", [("f64", 18), ("f64", 12), ("f32", 18), ("f32", 12)])
def test_fused_theta_terms_match_full_measure_and_oracle(gf, torch, dims, gauge, prec, storage):
    """After gf_ovr_sweep the odd sites' theta terms come from K_final = G K inside the odd half-sweep and gf_measure
    visits the even sites only; with GF_OPT_FUSE_MEASURE = 0 it visits all sites.  Both against the oracle."""
    omega = 1.7
    U, Uo = host_input(dims, 0.4, 22, prec, storage)
    oracle.sweeps(Uo, dims, gauge, omega, n=3, storage=storage)
    Fo, tho = oracle.measure(Uo, dims, gauge)
    res = {}
    for fuse in (1, 0):
        fx = gpu_fixer(gf, torch, dims, gauge, prec, storage, U)
        fx.set_option(gf.GF_OPT_FUSE_MEASURE, fuse)
        fx.ovr_sweep(3, omega)
        n0 = fx.kernel_launches()
        res[fuse] = fx.measure()
        assert fx.kernel_launches() - n0 == 1  # one launch: the last block to finish does the second stage
        again = fx.measure()  # the fused terms stay valid until the links change
        assert again == res[fuse]
        fx.reunitarize()  # changes the links: the next measure must visit all sites again
        F2, th2 = fx.measure()
        fx.close()
    rtol_th = 1e-9 if prec == "f64" else 2e-4
    assert res[1][0] == res[0][0]  # F is summed over the even sites in both modes
    assert abs(res[1][1] - res[0][1]) <= rtol_th * res[0][1]
    for F, th in res.values():
        assert abs(F - Fo) <= TOL_F[prec] * abs(Fo)
        assert abs(th - tho) <= (1e-8 if prec == "f64" else 1e-3) * tho


def test_fused_theta_terms_near_convergence(gf, torch):
    """theta ~ 1e-13: the fused terms are differences of O(1) entries of G K; they must still track the oracle."""
    dims = (4, 4, 4, 4)
    U, Uo = host_input(dims, 0.2, 23, "f64", 18)
    fx = gpu_fixer(gf, torch, dims, "landau", "f64", 18, U)
    done = fx.fix(1.6, 1e-13, 2000, 10)
    hist = fx.history()
    do, ho = oracle.fix(Uo, dims, "landau", 1.6, 1e-13, 2000, 10)
    assert done == do and len(hist) == len(ho)
    for (s, F, th), (so, Fo, tho) in zip(hist, ho):
        assert s == so and abs(F - Fo) <= 1e-10 * abs(Fo)
        assert tho / 1.5 <= th <= tho * 1.5 or max(th, tho) < 1e-25
    fx.close()


def test_two_contexts_on_their_own_streams(gf, torch):
    """Work is ordered on the stream handed to gf_create (include/gf.h): two contexts on two non-default streams,
    launched interleaved, each reproduce the oracle; Algorithm 1 on one, Algorithm 2 on the other."""
    from oracle import fftsd

    dims = (8, 6, 4, 6)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    U1, O1 = host_input(dims, 0.4, 41, "f64", 18)
    U2, O2 = host_input(dims, 0.5, 42, "f64", 12)
    d1, d2 = torch.from_numpy(U1).cuda(), torch.from_numpy(U2).cuda()
    torch.cuda.synchronize()
    with torch.cuda.stream(s1):
        f1 = gf.GaugeFixer(dims, gauge="landau", prec="f64", storage=18, stream=s1)
        f1.set_links(d1)
    with torch.cuda.stream(s2):
        f2 = gf.GaugeFixer(dims, gauge="coulomb", prec="f64", storage=12, stream=s2)
        f2.set_links(d2)
        f2.fft_attach()
    for _ in range(3):
        f1.ovr_sweep(1, 1.6)
        f2.fft_step(1, 0.08)
    with torch.cuda.stream(s1):
        g1 = f1.get_links()
    with torch.cuda.stream(s2):
        g2 = f2.get_links()
    s1.synchronize()
    s2.synchronize()
    oracle.sweeps(O1, dims, "landau", 1.6, n=3)
    for _ in range(3):
        fftsd.step(O2, dims, "coulomb", 0.08, storage=12)
    assert np.abs(g1.cpu().numpy() - O1).max() <= 3e-12
    assert np.abs(g2.cpu().numpy() - O2).max() <= 3e-12
    f1.close()
    f2.close()


@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (6, 4, 2, 2), (10, 6, 4, 4)])
@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
@pytest.mark.parametrize("prec,storage", [("f64", 18), ("f64", 12), ("f32", 18), ("f32", 12)])
@pytest.mark.parametrize("order", [1, 4])
def test_series_variant_of_the_overrelaxation_power(gf, torch, dims, gauge, prec, storage, order):
    """GF_OPT_OVR_SERIES: g^omega as the truncated binomial series (reading A21), against the oracle in the same mode."""
    omega = 1.7
    U, Uo = host_input(dims, 0.5, 19, prec, storage)
    fx = gpu_fixer(gf, torch, dims, gauge, prec, storage, U)
    fx.set_option(gf.GF_OPT_OVR_SERIES, order)
    fx.ovr_sweep(1, omega)
    got = fx.get_links().cpu().numpy().astype(np.float64)
    F, th = fx.measure()
    # back to the exact power on the same context
    fx.set_option(gf.GF_OPT_OVR_SERIES, 0)
    fx.set_links(torch.from_numpy(U).cuda())
    fx.ovr_sweep(1, omega)
    exact = fx.get_links().cpu().numpy().astype(np.float64)
    fx.close()
    try:
        oracle.set_series(order)
        oracle.sweeps(Uo, dims, gauge, omega, n=1, storage=storage)
    finally:
        oracle.set_series(0)
    Fo, tho = oracle.measure(Uo, dims, gauge)
    assert np.abs(got - Uo).max() <= TOL_LINK[prec]  # north_star's one-sweep bound
    assert abs(F - Fo) <= TOL_F[prec] * abs(Fo) and tho / 1.5 <= th <= tho * 1.5
    assert np.abs(got - exact).max() > 1e-3  # the option is live: a visibly different update


def test_series_option_errors(gf, torch):
    fx = gf.GaugeFixer((4, 4, 4, 4))
    assert gf.gf_set_option(fx.ctx, gf.GF_OPT_OVR_SERIES, -1) == gf.GF_EINVAL
    assert gf.gf_set_option(fx.ctx, gf.GF_OPT_OVR_SERIES, 17) == gf.GF_EINVAL
    assert gf.gf_set_option(fx.ctx, gf.GF_OPT_OVR_SERIES, 3) == gf.GF_OK
    assert gf.gf_set_option(fx.ctx, gf.GF_OPT_SWEEP_VARIANT, 1) == gf.GF_OK
    U = gi.make_links((4, 4, 4, 4), 0.3, 1)
    fx.set_links(torch.from_numpy(U).cuda())
    assert gf.gf_ovr_sweep(fx.ctx, 1, 1.7) == gf.GF_ECUDA  # the two-pass kernels have no series form
    B = gf.gf_slab_halo_bytes(fx.ctx)
    halo = torch.zeros(4 * B, dtype=torch.uint8, device="cuda")
    assert gf.gf_slab_attach(fx.ctx, halo.data_ptr(), 4 * B) == gf.GF_EUNSUPPORTED
    fx.close()


# ---- Coulomb gauge with a stop test per time slice (gf_measure_slices / gf_fix_slices; reading A22) --------------------
@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (6, 4, 2, 6), (16, 16, 4, 4), (2, 2, 2, 4)])
@pytest.mark.parametrize("prec,storage", [("f64", 18), ("f64", 12), ("f32", 18), ("f32", 12)])
def test_measure_slices_matches_oracle(gf, torch, dims, prec, storage):
    U, Uo = host_input(dims, 0.5, 61, prec, storage)
    fx = gpu_fixer(gf, torch, dims, "coulomb", prec, storage, U)
    Ft, tht = fx.measure_slices()
    F, th = fx.measure()
    fx.close()
    Fo, tho = oracle.measure_slices(Uo, dims, "coulomb")
    atol = 1e-13 if prec == "f64" else 2e-7
    assert np.abs(np.array(Ft) - Fo).max() <= atol
    assert np.abs(np.array(tht) / tho - 1).max() <= (1e-12 if prec == "f64" else 1e-5)
    assert abs(np.mean(Ft) - F) <= atol and abs(np.mean(tht) / th - 1) <= 1e-6


@pytest.mark.parametrize("prec,storage,eps", [("f64", 18, 1e-10), ("f64", 12, 1e-10), ("f32", 12, 1e-6)])
def test_fix_slices_against_oracle(gf, torch, prec, storage, eps):
    dims, omega, cap, every = (8, 8, 8, 8), 1.7, 1500, 5
    U, Uo = host_input(dims, 0.4, 62, prec, storage)
    fx = gpu_fixer(gf, torch, dims, "coulomb", prec, storage, U)
    done, per = fx.fix_slices(omega, eps, cap, every)
    hist = fx.history()
    Ft, tht = fx.measure_slices()
    got = fx.get_links().cpu().numpy().astype(np.float64)
    fx.close()
    do, pero, histo = oracle.fix_slices(Uo, dims, "coulomb", omega, eps, cap, every, storage=storage)
    assert done < cap and max(tht) < eps
    # north_star: sweeps to convergence within +-2 % (one cadence step at least), per slice and overall
    assert abs(done - do) <= max(every, 0.02 * do)
    assert all(abs(a - b) <= max(every, 0.02 * b) for a, b in zip(per, pero))
    assert min(per) < max(per)  # the slices did finish at different times on this input
    assert abs(hist[-1][1] - histo[-1][1]) <= TOL_F[prec] * abs(histo[-1][1])
    if list(per) == list(pero):  # same stop decisions: the same sequence of updates
        assert np.abs(got - Uo).max() <= (1e-9 if prec == "f64" else 5e-3)


def test_slices_abi_errors(gf, torch):
    fx = gf.GaugeFixer((4, 4, 4, 4), gauge="landau")
    assert gf.gf_measure_slices(fx.ctx, 4)[0] == gf.GF_EUNSUPPORTED
    assert gf.gf_fix_slices(fx.ctx, 1.7, 1e-9, 10, 1, 4)[0] == gf.GF_EUNSUPPORTED
    fx.close()
    fx = gf.GaugeFixer((4, 4, 4, 4), gauge="coulomb")
    fx.set_links(torch.from_numpy(gi.make_links((4, 4, 4, 4), 0.3, 1)).cuda())
    assert gf.gf_fix_slices(fx.ctx, 2.0, 1e-9, 10, 1, 4)[0] == gf.GF_EINVAL
    assert gf.gf_fix_slices(fx.ctx, 1.7, 1e-9, 10, 0, 4)[0] == gf.GF_EINVAL
    assert gf.gf_set_option(fx.ctx, gf.GF_OPT_OVR_SERIES, 2) == gf.GF_OK
    assert gf.gf_fix_slices(fx.ctx, 1.7, 1e-9, 10, 1, 4)[0] == gf.GF_EUNSUPPORTED
    assert gf.gf_set_option(fx.ctx, gf.GF_OPT_OVR_SERIES, 0) == gf.GF_OK
    rc, done, per = gf.gf_fix_slices(fx.ctx, 1.7, 0.0, 4, 3, 4)  # eps = 0: fixed sweep count, every slice active
    assert rc == gf.GF_OK and done == 4 and per == [4, 4, 4, 4]
    assert gf.gf_measure_slices(None, 4)[0] == gf.GF_EINVAL
    fx.close()


# ---- Coulomb gauge with deferred temporal links (gf_defer_*) -------------------------------------------------------------
@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (6, 4, 2, 2), (10, 6, 4, 4), (2, 2, 2, 2), (16, 4, 4, 6)])
@pytest.mark.parametrize("prec,storage", [("f64", 18), ("f64", 12), ("f32", 18), ("f32", 12)])
@pytest.mark.parametrize("sweeps", [1, 3])
def test_deferred_temporal_links_against_oracle_and_in_place(gf, torch, dims, prec, storage, sweeps):
    omega = 1.7
    U, Uo = host_input(dims, 0.5, 71, prec, storage)
    fx = gpu_fixer(gf, torch, dims, "coulomb", prec, storage, U)
    fx.defer_temporal_links()
    l0 = fx.kernel_launches()
    fx.ovr_sweep(sweeps, omega)
    assert fx.kernel_launches() - l0 == 2 * sweeps
    F, th = fx.measure()                      # Coulomb F and theta do not read temporal links: valid before the flush
    got = fx.get_links().cpu().numpy().astype(np.float64)   # flushes
    again = fx.get_links().cpu().numpy().astype(np.float64)  # nothing left to flush
    fx.defer_flush()
    fx.defer_temporal_links(False)
    fx.set_links(torch.from_numpy(U).cuda())
    fx.ovr_sweep(sweeps, omega)
    inplace = fx.get_links().cpu().numpy().astype(np.float64)
    Fi, thi = fx.measure()
    fx.close()
    oracle.sweeps(Uo, dims, "coulomb", omega, n=sweeps, storage=storage)
    Fo, tho = oracle.measure(Uo, dims, "coulomb")
    assert np.array_equal(got, again)
    assert np.abs(got - Uo).max() <= sweeps * TOL_LINK[prec]
    assert np.array_equal(got[:, :3], inplace[:, :3])          # spatial links: the same instruction sequence
    assert np.abs(got[:, 3] - inplace[:, 3]).max() <= sweeps * (1e-14 if prec == "f64" else 5e-6)
    assert abs(F - Fo) <= TOL_F[prec] * abs(Fo) and tho / 1.5 <= th <= tho * 1.5
    assert abs(F - Fi) <= 1e-6 * abs(Fi)


def test_deferred_links_whole_run_with_reunitarisation_and_errors(gf, torch):
    dims, omega, eps, cap, every = (8, 8, 8, 8), 1.7, 1e-9, 600, 10
    U, Uo = host_input(dims, 0.3, 72, "f64", 18)
    fx = gpu_fixer(gf, torch, dims, "coulomb", "f64", 18, U)
    fx.set_reunit_every(20)
    fx.defer_temporal_links()
    done = fx.fix(omega, eps, cap, every)
    hist = fx.history()
    got = fx.get_links().cpu().numpy()
    assert gf.gf_fix_slices(fx.ctx, omega, eps, cap, every, dims[3])[0] == gf.GF_EUNSUPPORTED
    fx.close()
    do, histo = oracle.fix(Uo, dims, "coulomb", omega, eps, cap, every, reunit_every=20)
    assert abs(done - do) <= max(every, 0.02 * do) and done < cap
    assert abs(hist[-1][1] - histo[-1][1]) <= 1e-10 * abs(histo[-1][1])
    if done == do:
        assert np.abs(got - Uo).max() <= 1e-9
    a, b = oracle.unitarity(np.ascontiguousarray(got), dims)
    assert a < 1e-12 and b < 1e-12
    # gauge invariance of the flushed field: temporal plaquettes as in the input
    for mu in (0, 2):
        assert np.abs(oracle.wilson_traces(np.ascontiguousarray(got), dims, mu, 3, 1, 1)
                      - oracle.wilson_traces(np.ascontiguousarray(U), dims, mu, 3, 1, 1)).max() < 1e-11
    fx = gf.GaugeFixer((4, 4, 4, 4), gauge="landau")
    assert gf.gf_defer_attach(fx.ctx, 256, 1 << 20) == gf.GF_EUNSUPPORTED
    fx.close()
    fx = gf.GaugeFixer((4, 4, 4, 4), gauge="coulomb")
    n = gf.gf_defer_bytes(fx.ctx)
    buf = torch.empty(n, dtype=torch.uint8, device="cuda")
    assert n >= 4 ** 4 * 9 * 16 and gf.gf_defer_bytes(None) == 0
    assert gf.gf_defer_attach(fx.ctx, buf.data_ptr(), n - 1) == gf.GF_ENOMEM
    assert gf.gf_defer_attach(fx.ctx, buf.data_ptr(), n) == gf.GF_OK
    B = gf.gf_slab_halo_bytes(fx.ctx)
    halo = torch.zeros(4 * B, dtype=torch.uint8, device="cuda")
    assert gf.gf_slab_attach(fx.ctx, halo.data_ptr(), 4 * B) == gf.GF_EUNSUPPORTED
    assert gf.gf_defer_attach(fx.ctx, 0, 0) == gf.GF_OK and gf.gf_defer_flush(fx.ctx) == gf.GF_OK
    assert gf.gf_defer_flush(None) == gf.GF_EINVAL
    fx.close()


# ---- 8-real storage (reading A23); tolerance scaled by the conditioning 1/N of the reconstruction ---------------------------
@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (6, 4, 2, 2), (10, 6, 4, 4), (2, 2, 2, 2)])
@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_8_real_storage_against_oracle(gf, torch, dims, gauge, prec):
    omega = 1.7
    f64 = prec == "f64"
    u = 1.1e-16 if f64 else 6e-8
    U = gi.make_links(dims, 0.5, 84, dtype=np.float64 if f64 else np.float32)
    Uo = np.ascontiguousarray(U.astype(np.float64))  # reading A18: the FP64 oracle on the rounded input
    oracle.project8(Uo, dims)
    fx = gf.GaugeFixer(dims, gauge=gauge, prec=prec, storage=8)
    fx.set_links(torch.from_numpy(U).cuda())
    back = fx.get_links().cpu().numpy().astype(np.float64)
    F0, th0 = fx.measure()
    Fo0, tho0 = oracle.measure(Uo, dims, gauge)
    Uc = U[..., 0].astype(np.float64) + 1j * U[..., 1]
    Nmin = (np.abs(Uc[:, :, 0, 1]) ** 2 + np.abs(Uc[:, :, 0, 2]) ** 2).min()
    assert np.abs(back - Uo).max() <= 100 * u / Nmin           # storing and reading back = the oracle's round trip
    assert abs(F0 - Fo0) <= (1e-12 if f64 else 1e-5) and abs(th0 / tho0 - 1) <= (1e-10 if f64 else 1e-4)
    fx.ovr_sweep(1, omega)
    got = fx.get_links().cpu().numpy().astype(np.float64)
    F, th = fx.measure()
    fx.reunitarize()
    after = fx.get_links().cpu().numpy().astype(np.float64)
    fx.close()
    oracle.sweeps(Uo, dims, gauge, omega, n=1, storage=8)
    Fo, tho = oracle.measure(Uo, dims, gauge)
    # the one-sweep bound, widened where 1/N demands it (1000 u / N: 1e-13 / N in FP64, 6e-5 / N ... in FP32)
    assert np.abs(got - Uo).max() <= max(1e-12 if f64 else 2e-5, 1000 * u / Nmin)
    assert abs(F - Fo) <= (1e-10 if f64 else 1e-5) * abs(Fo) and tho / 1.5 <= th <= tho * 1.5
    assert np.abs(after - got).max() <= 1e4 * u / Nmin         # the links were unitary: reunitarisation changes nothing
    assert gf.gf_workspace_bytes(*dims, int(not f64), 8) < gf.gf_workspace_bytes(*dims, int(not f64), 12)


def test_8_real_storage_reports_links_outside_its_domain(gf, torch):
    """A cold start (unit links: N = 0), a pure gauge and a nearly fixed smooth field are where 8-real storage is
    undefined or inaccurate: the store raises a flag and the next synchronising call says GF_ENUMERIC
    instead of returning garbage."""
    dims = (4, 4, 4, 4)
    V = 256
    unit = np.zeros((V, 4, 3, 3, 2))
    unit[:, :, 0, 0, 0] = unit[:, :, 1, 1, 0] = unit[:, :, 2, 2, 0] = 1.0
    fx = gf.GaugeFixer(dims, prec="f64", storage=8)
    fx.set_links(torch.from_numpy(unit).cuda())
    rc, F, th = gf.gf_measure(fx.ctx)
    assert rc == gf.GF_ENUMERIC and "8-real" in gf.gf_last_error(fx.ctx)
    # a rough field is inside the domain: the flag was cleared by the report
    U = gi.make_links(dims, 0.5, 3)
    fx.set_links(torch.from_numpy(U).cuda())
    rc, F, th = gf.gf_measure(fx.ctx)
    assert rc == gf.GF_OK and np.isfinite(F) and np.isfinite(th)
    # a report concerns the field the context holds: the unit field loaded and replaced WITHOUT a report in between
    # must not make the valid field fail, here or in a context created afterwards
    fx.set_links(torch.from_numpy(unit).cuda())
    fx.set_links(torch.from_numpy(U).cuda())
    assert gf.gf_measure(fx.ctx)[0] == gf.GF_OK
    fx.set_links(torch.from_numpy(unit).cuda())
    fx2 = gf.GaugeFixer(dims, prec="f64", storage=8)
    fx2.set_links(torch.from_numpy(U).cuda())
    assert gf.gf_measure(fx2.ctx)[0] == gf.GF_OK
    fx2.close()
    # a smooth field driven towards Landau gauge from a cold-ish start: links near 1, N ~ roughness^2
    Us = gi.make_links(dims, 1e-4, 4)
    G = gi.make_gauge(dims, 4)  # undo the hidden rotation: the field is then exp(i r H), r = 1e-4
    Uc = Us[..., 0] + 1j * Us[..., 1]
    nx, ny, nz, nt = dims
    Gg = G.reshape(nt, nz, ny, nx, 3, 3)
    for mu in range(4):
        Gup = np.roll(Gg, -1, axis=3 - mu).reshape(V, 3, 3)
        Uc[:, mu] = np.conj(np.swapaxes(G, -1, -2)) @ Uc[:, mu] @ Gup
    Us = np.ascontiguousarray(np.stack([Uc.real, Uc.imag], axis=-1))
    fx.set_links(torch.from_numpy(Us).cuda())
    rc, F, th = gf.gf_measure(fx.ctx)
    assert rc == gf.GF_ENUMERIC
    fx.close()


def test_8_real_storage_fix_and_unsupported_calls(gf, torch):
    dims = (8, 8, 8, 8)
    U = gi.make_links(dims, 0.3, 85)
    Uo = U.copy()
    oracle.project8(Uo, dims)
    fx = gf.GaugeFixer(dims, gauge="landau", prec="f64", storage=8)
    fx.set_links(torch.from_numpy(U).cuda())
    done = fx.fix(1.7, 1e-10, 600, 10)
    hist = fx.history()
    do, histo = oracle.fix(Uo, dims, "landau", 1.7, 1e-10, 600, 10, storage=8)
    assert abs(done - do) <= max(10, 0.02 * do) and done < 600
    assert abs(hist[-1][1] - histo[-1][1]) <= 1e-10 * abs(histo[-1][1])
    assert gf.gf_fft_workspace_bytes(fx.ctx)[0] == gf.GF_EUNSUPPORTED
    assert gf.gf_set_option(fx.ctx, gf.GF_OPT_OVR_SERIES, 2) == gf.GF_EUNSUPPORTED
    B = gf.gf_slab_halo_bytes(fx.ctx)
    halo = torch.zeros(4 * B, dtype=torch.uint8, device="cuda")
    assert gf.gf_slab_attach(fx.ctx, halo.data_ptr(), 4 * B) == gf.GF_EUNSUPPORTED
    fx.close()
    assert gf.gf_workspace_bytes(8, 8, 8, 8, gf.GF_FP32, 8) > 0


@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
@pytest.mark.parametrize("storage", [18, 12])
def test_fp32_fast_path_on_a_smoothed_field(gf, torch, gauge, storage):
    """With FP32 links the staged kernel evaluates a site in FP32 unless a subgroup's |r|^2 < 16.  On a
    random start nearly every site takes the FP64 branch, so the one-sweep bound is checked here where the FP32 branch
    does the work: the state after 30 sweeps (F ~ 0.7, |r|^2 ~ 100) is handed to the oracle and both take one more sweep."""
    dims, omega = (16, 16, 16, 8), 1.75
    U, _ = host_input(dims, 0.4, 77, "f32", storage)
    fx = gpu_fixer(gf, torch, dims, gauge, "f32", storage, U)
    fx.ovr_sweep(30, omega)
    start = fx.get_links().cpu().numpy()
    F, _ = fx.measure()
    assert F > 0.6
    fx.ovr_sweep(1, omega)
    got = fx.get_links().cpu().numpy().astype(np.float64)
    fx.close()
    Uo = np.ascontiguousarray(start.astype(np.float64))
    if storage == 12:
        oracle.project12(Uo, dims)
    oracle.sweeps(Uo, dims, gauge, omega, n=1, storage=storage)
    assert np.abs(got - Uo).max() <= TOL_LINK["f32"]
