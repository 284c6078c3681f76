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


# ---- the multi-rank schedule under real concurrency, on one GPU ------------------------------------------------------------
# Every slab of ONE process on a CUDA stream of its own (slab_streams="own"): the fused kernels of neighbouring slabs
# overlap on the device, group_is_closed() is false, and every ordering between neighbours goes through the arrival
# counters and cuStreamWaitValue32 - what the ranks of a multi-GPU run execute.
# late: the slab whose stream is held back by a sleep kernel before every call, far longer than the whole call takes, so
# that the other slabs run as far ahead as the protocol lets them.  This is the state a single summed arrival counter
# (round 2) gets wrong: (R0: n-1, R1: n, R2: n+1, R3: n) satisfies R1's "sum >= 2n" although R0 has not delivered.  The
# late slab's two neighbours are stopped by the entry signal of the call, so the slabs that run ahead are those at
# distance >= 2 on both sides: it takes five or more slabs for a stream sleep to produce the state (the cases with 5, 6
# and 8 slabs fail on the summed counter, measured on the round-2 library).  (lattice, slabs, gauge, prec, storage, late)
OWN_STREAM_CASES = [
    ((8, 8, 8, 8), 4, "landau", "f64", 18, 0),       # lt = 2: every slice is a border slice
    ((8, 8, 8, 8), 4, "coulomb", "f32", 12, 2),
    ((8, 8, 8, 8), 2, "landau", "f64", 12, 1),
    ((6, 4, 2, 12), 3, "coulomb", "f64", 18, 0),     # ragged x-rows, lt = 4
    ((10, 6, 4, 16), 4, "landau", "f32", 18, 3),     # slices that are not whole 32-site blocks
    ((8, 8, 8, 16), 4, "landau", "f64", 18, None),   # nobody held back: whatever skew the device produces
    ((16, 4, 4, 24), 6, "coulomb", "f64", 12, 0),
    ((8, 8, 8, 20), 5, "landau", "f64", 18, 2),
    ((4, 4, 4, 16), 8, "landau", "f32", 12, 3),
]
SLEEP_CYCLES = 100_000_000  # ~50 ms at 1.9 GHz; 37 sweeps of these lattices take about 2 ms


def run_single_context(gf, torch, U, dims, gauge, prec, storage, calls, omega, reunit):
    fx = gf.GaugeFixer(dims, gauge=gauge, prec=prec, storage=storage)
    fx.set_reunit_every(reunit)
    fx.set_links(U)
    for n in calls:
        fx.ovr_sweep(n, omega)
    links = fx.get_links().reshape(-1)
    F, th = fx.measure()
    fx.close()
    return links, F, th


def run_slabs(gf, torch, U, dims, n_slabs, gauge, prec, storage, calls, omega, reunit, late, own=True, force=False):
    sh = gf.ShardedGaugeFixer(dims, n_slabs, gauge=gauge, prec=prec, storage=storage, group=False, mode="flags",
                              slab_streams="own" if own else None)
    assert sh.mode == "flags"
    if own:
        assert len({sh.engines[s].stream.cuda_stream for s in sh.slabs}) == n_slabs
    if force:
        for s in sh.slabs:
            sh.engines[s].fx.set_option(gf.GF_OPT_SLAB_FORCE_FLAGS, 1)
    sh.set_reunit_every(reunit)
    sh.set_links_global(U)
    for n in calls:
        if late is not None:
            with torch.cuda.stream(sh.engines[late].stream):
                torch.cuda._sleep(SLEEP_CYCLES)
        sh.ovr_sweep(n, omega)
    links = sh.get_links()
    links = torch.cat([links[s].reshape(-1) for s in range(n_slabs)])
    F, th = sh.measure()
    sh.close()
    return links, F, th


@pytest.mark.parametrize("dims,n_slabs,gauge,prec,storage,late", OWN_STREAM_CASES)
def test_slabs_on_their_own_streams_bit_identical_to_the_single_context(gf, torch, dims, n_slabs, gauge, prec, storage,
                                                                         late):
    """100 sweeps in three calls (37 + 37 + 26) with a reunitarisation every 7 sweeps - a cadence that divides none of
    the call lengths, so reunitarisations (and the ghost refresh behind them) fall inside and across calls."""
    omega, calls, reunit = 1.7, (37, 37, 26), 7
    U = torch.from_numpy(host_input(dims, 0.5, 33, prec, storage)[0]).cuda()
    want, Fs, ths = run_single_context(gf, torch, U, dims, gauge, prec, storage, calls, omega, reunit)
    got, F, th = run_slabs(gf, torch, U, dims, n_slabs, gauge, prec, storage, calls, omega, reunit, late)
    assert torch.equal(got, want), f"max diff {(got - want).abs().max().item()}"
    rel, relth = (1e-13, 1e-9) if prec == "f64" else (1e-6, 1e-6)
    assert abs(F - Fs) <= rel * abs(Fs) + 1e-15 and abs(th - ths) <= relth * ths + 1e-30


@pytest.mark.parametrize("n_slabs", [2, 4])
def test_flags_forced_on_one_stream(gf, torch, n_slabs):
    """GF_OPT_SLAB_FORCE_FLAGS: all slabs on one stream, yet every signal and wait of the multi-rank schedule is issued
    (the launches of a half-sweep are queued for all slabs before their waits, so one stream cannot deadlock)."""
    dims, gauge, prec, storage, omega, calls, reunit = (8, 8, 8, 8), "landau", "f64", 18, 1.7, (37, 37, 26), 7
    U = torch.from_numpy(host_input(dims, 0.5, 34, prec, storage)[0]).cuda()
    want, _, _ = run_single_context(gf, torch, U, dims, gauge, prec, storage, calls, omega, reunit)
    got, _, _ = run_slabs(gf, torch, U, dims, n_slabs, gauge, prec, storage, calls, omega, reunit, None, own=False,
                          force=True)
    assert torch.equal(got, want)


def test_cfg2_sized_slab_stack_on_four_streams(gf, torch):
    """32^4 in FP32 with 12-real storage (BASELINE.json configs[2]) as four 32^3 x 8 slabs - the paper's weak-scaling
    local volume - on four streams, slab 0 held back; 100 sweeps, reunitarisation every 50 as the
    config says and once more at a cadence that falls inside a call."""
    dims, n_slabs, gauge, prec, storage, omega = (32, 32, 32, 32), 4, "landau", "f32", 12, 1.75
    U = torch.empty((gi.volume(dims), 4, 3, 3, 2), dtype=torch.float32, device="cuda")
    gi.make_links_device(U.data_ptr(), dims, 0.4, 3, "f32", torch.cuda.current_stream().cuda_stream)
    for calls, reunit in [((37, 37, 26), 50), ((60, 40), 7)]:
        want, Fs, ths = run_single_context(gf, torch, U, dims, gauge, prec, storage, calls, omega, reunit)
        got, F, th = run_slabs(gf, torch, U, dims, n_slabs, gauge, prec, storage, calls, omega, reunit, late=0)
        assert torch.equal(got, want), f"max diff {(got - want).abs().max().item()}"
        assert abs(F - Fs) <= 1e-6 * abs(Fs) and abs(th - ths) <= 1e-6 * ths + 1e-30


def test_own_streams_fix_history_equals_single_context(gf, torch):
    """The driver loop (measure, plan, sweep) over slabs on their own streams: same sweep count, same history."""
    dims, gauge, prec, storage, n_slabs = (8, 8, 8, 16), "landau", "f64", 18, 4
    omega, eps, cap, every, reunit = 1.7, 1e-9, 300, 10, 20
    U = torch.from_numpy(host_input(dims, 0.3, 35, prec, storage)[0]).cuda()
    sh = gf.ShardedGaugeFixer(dims, n_slabs, gauge=gauge, prec=prec, storage=storage, group=False, slab_streams="own")
    sh.set_reunit_every(reunit)
    sh.set_links_global(U)
    done, hist = sh.fix(omega, eps, cap, every)
    links = sh.get_links()
    got = torch.cat([links[s].reshape(-1) for s in range(n_slabs)])
    sh.close()
    fx = gf.GaugeFixer(dims, gauge=gauge, prec=prec, storage=storage)
    fx.set_reunit_every(reunit)
    fx.set_links(U)
    done_s = fx.fix(omega, eps, cap, every)
    hist_s = fx.history()
    want = fx.get_links().reshape(-1)
    fx.close()
    assert done == done_s and len(hist) == len(hist_s) and torch.equal(got, want)
    for (n, F, th), (ns, Fs, ths) in zip(hist, hist_s):
        assert n == ns and abs(F - Fs) <= 1e-12 * abs(Fs) and abs(th - ths) <= 1e-8 * ths + 1e-30
