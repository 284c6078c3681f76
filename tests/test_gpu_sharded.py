"""GPU parity of the T-slab sharded overrelaxation path (include/gf.h "T-slab sharding") through the
C ABI: n_slabs slab contexts in ONE process on one GPU (halo messages are device-to-device copies; across processes the
same buffers go through torch.distributed, covered on CPU ranks by tests/test_sharded_gloo.py).

* against the oracle's sweep of the whole lattice: north_star tolerances (1e-12 / 2e-5 per link after one sweep, F rel
  1e-10 / 1e-5, theta within a factor 1.5);
* against libgf's own single-context path on the whole lattice: bit-identical links (same per-site instruction
  sequence, only the addresses differ)."""
import numpy as np
import pytest

import gf_inputs as gi
import oracle

pytestmark = pytest.mark.gpu

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
    dt = np.float32 if prec == "f32" else np.float64
    U = gi.make_links(dims, roughness, seed, dtype=dt)
    Uo = np.ascontiguousarray(U.astype(np.float64))
    if storage == 12:
        oracle.project12(Uo, dims)
    return U, Uo


def assembled(sh, torch):
    links = sh.get_links()
    return torch.cat([links[s].reshape(-1) for s in range(sh.n_slabs)]).cpu().numpy()


# (global lattice, slabs): lt = 8, 4, 2 (border only), ragged tails, slices that are not whole 32-site blocks
LATTICES = [((8, 8, 8, 8), 1), ((8, 8, 8, 8), 2), ((8, 8, 8, 8), 4), ((6, 4, 2, 12), 3), ((4, 6, 10, 4), 2),
            ((2, 2, 2, 4), 2), ((16, 4, 4, 12), 2), ((10, 6, 4, 8), 1)]


@pytest.mark.parametrize("mode", ["flags", "events", "transport"])
@pytest.mark.parametrize("dims,n_slabs", LATTICES)
@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
@pytest.mark.parametrize("prec,storage", [("f64", 18), ("f64", 12), ("f32", 18), ("f32", 12)])
def test_sharded_sweeps_against_oracle_and_single_context(gf, torch, dims, n_slabs, gauge, prec, storage, mode):
    """flags: the border kernels store the halo messages into the neighbours' buffers (gf_slab_set_peer_targets), the
    neighbours are ordered by stream-ordered flags and the sweep is one libgf call (gf_slab_group_sweep);
    events: the same delivery (gf_slab_set_targets), kernels ordered by CUDA events from Python;
    transport: the messages stay in top_out / ghost and the plumbing copies them."""
    omega, sweeps = 1.7, 2
    direct = mode != "transport"
    U, Uo = host_input(dims, 0.5, 31, prec, storage)
    sh = gf.ShardedGaugeFixer(dims, n_slabs, gauge=gauge, prec=prec, storage=storage, group=False, mode=mode)
    assert sh.mode == mode
    sh.set_links_global(torch.from_numpy(U).cuda())
    F0, th0 = sh.measure()
    sh.ovr_sweep(sweeps, omega)
    got = assembled(sh, torch)
    F, th = sh.measure()
    n_launch = sh.kernel_launches()
    sh.close()

    # the single-context path on the whole lattice
    fx = gf.GaugeFixer(dims, gauge=gauge, prec=prec, storage=storage)
    fx.set_links(torch.from_numpy(U).cuda())
    F0s, th0s = fx.measure()
    fx.ovr_sweep(sweeps, omega)
    single = fx.get_links().cpu().numpy().reshape(-1)
    Fs, ths = fx.measure()
    fx.close()
    assert np.array_equal(got, single), f"max diff {np.abs(got - single).max()}"
    # same terms, different summation tree; in FP32 the single context takes the odd sites' theta terms from the FP64
    # K(x) of the last half-sweep, a slab evaluates Delta(x) of every site in FP32
    rel, relth = (1e-13, 1e-9) if prec == "f64" else (1e-6, 1e-6)
    assert abs(F - Fs) <= rel * abs(Fs) + 1e-15 and abs(th - ths) <= relth * ths + 1e-30
    assert abs(F0 - F0s) <= rel * abs(F0s) + 1e-15 and abs(th0 - th0s) <= relth * th0s + 1e-30

    # the oracle
    oracle.sweeps(Uo, dims, gauge, omega, n=sweeps, storage=storage)
    Fo, tho = oracle.measure(Uo, dims, gauge)
    assert np.abs(got.astype(np.float64) - Uo.reshape(-1)).max() <= sweeps * TOL_LINK[prec]
    assert abs(F - Fo) <= TOL_F[prec] * abs(Fo)
    assert tho / 1.5 <= th <= tho * 1.5
    assert n_launch > 0
    assert (sh.copies == 0) == direct


@pytest.mark.parametrize("gauge,prec,storage,n_slabs", [("landau", "f64", 18, 2), ("coulomb", "f64", 12, 4),
                                                        ("landau", "f32", 12, 2)])
@pytest.mark.parametrize("mode", ["flags", "events", "transport"])
def test_sharded_fix_matches_single_context_trajectory(gf, torch, gauge, prec, storage, n_slabs, mode):
    """The whole driver loop (measurement cadence, stop test, reunitarisation + ghost refresh) on slabs against gf_fix."""
    dims, omega, eps, cap, every, reunit = (8, 8, 8, 8), 1.7, 1e-9 if prec == "f64" else 1e-6, 300, 10, 20
    U, _ = host_input(dims, 0.3, 32, prec, storage)
    sh = gf.ShardedGaugeFixer(dims, n_slabs, gauge=gauge, prec=prec, storage=storage, group=False, mode=mode)
    sh.set_reunit_every(reunit)
    sh.set_links_global(torch.from_numpy(U).cuda())
    done, hist = sh.fix(omega, eps, cap, every)
    got = assembled(sh, torch)
    sh.close()
    fx = gf.GaugeFixer(dims, gauge=gauge, prec=prec, storage=storage)
    fx.set_reunit_every(reunit)
    fx.set_links(torch.from_numpy(U).cuda())
    done_s = fx.fix(omega, eps, cap, every)
    hist_s = fx.history()
    single = fx.get_links().cpu().numpy().reshape(-1)
    fx.close()
    assert done == done_s and len(hist) == len(hist_s)
    assert np.array_equal(got, single)
    for (n, F, th), (ns, Fs, ths) in zip(hist, hist_s):
        assert n == ns and abs(F - Fs) <= 1e-6 * abs(Fs) and abs(th - ths) <= 1e-3 * ths + 1e-30


def test_slab_abi_errors(gf, torch):
    fx = gf.GaugeFixer((4, 4, 4, 4), gauge="landau", prec="f64", storage=18)
    B = gf.gf_slab_halo_bytes(fx.ctx)
    assert B >= 4 * 4 * 4 // 2 * 9 * 16 and B % 256 == 0
    assert gf.gf_slab_halo_bytes(None) == 0
    # no halo attached yet
    assert gf.gf_slab_halfsweep_border(fx.ctx, 0, 1.7) == gf.GF_EINVAL
    assert gf.gf_slab_pack_top(fx.ctx, 0) == gf.GF_EINVAL
    assert gf.gf_slab_set_targets(fx.ctx, 0, 0, 0) == gf.GF_EINVAL
    halo = torch.zeros(4 * B, dtype=torch.uint8, device="cuda")
    assert gf.gf_slab_attach(fx.ctx, 0, 4 * B) == gf.GF_EINVAL
    assert gf.gf_slab_attach(fx.ctx, halo.data_ptr(), 4 * B - 1) == gf.GF_ENOMEM
    assert gf.gf_slab_attach(fx.ctx, halo.data_ptr() + 8, 4 * B) == gf.GF_ENOMEM
    assert gf.gf_slab_attach(fx.ctx, halo.data_ptr(), 4 * B) == gf.GF_OK
    assert gf.gf_slab_set_targets(fx.ctx, halo.data_ptr(), 0, 0) == gf.GF_EINVAL  # all three or none
    assert gf.gf_slab_set_targets(fx.ctx, 0, 0, 0) == gf.GF_OK
    assert gf.gf_slab_halfsweep_border(fx.ctx, 2, 1.7) == gf.GF_EINVAL
    assert gf.gf_slab_halfsweep_interior(fx.ctx, -1, 1.7) == gf.GF_EINVAL
    assert gf.gf_slab_halfsweep_border(fx.ctx, 0, 2.0) == gf.GF_EINVAL
    assert gf.gf_slab_unpack_top(fx.ctx, 5) == gf.GF_EINVAL
    # a slab is not a periodic lattice: the whole-lattice drivers refuse it
    assert gf.gf_ovr_sweep(fx.ctx, 1, 1.7) == gf.GF_EINVAL
    assert gf.gf_fix(fx.ctx, 1.7, 1e-9, 10, 1)[0] == gf.GF_EINVAL
    assert gf.gf_fft_workspace_bytes(fx.ctx)[0] == gf.GF_EUNSUPPORTED
    for f in (gf.gf_slab_pack_top, gf.gf_slab_unpack_top):
        assert f(None, 0) == gf.GF_EINVAL
    fx.close()
