"""GPU parity of the general SU(N) path (gf_create_sun) against oracle/sun.py,
through the C ABI: links after sweeps element by element, F, theta, reunitarisation, whole gf_fix runs, error codes.
Bars as for SU(3): one sweep <= 1e-12 (FP64) / 2e-5 (FP32 against the FP64 oracle on the rounded input, reading A18),
F relative 1e-10 / 1e-5, theta within x1.5, sweeps +-2 %."""
import numpy as np
import pytest

import gf_inputs as gi
from oracle import sun

pytestmark = pytest.mark.gpu

TOL_LINK = {"f64": 1e-12, "f32": 2e-5}
LATTICES = [(8, 8, 8, 8), (6, 4, 2, 2), (10, 6, 4, 4), (2, 2, 2, 2), (16, 4, 6, 2)]  # tiles, ragged tails, 2^4, wraps


@pytest.fixture(scope="module")
def gf():
    import paper_1412_1498_b200 as gf

    return gf


def fixer(gf, dims, N, gauge, prec, U):
    import torch

    fx = gf.GaugeFixer(dims, gauge=gauge, prec=prec, ncolors=N)
    fx.set_links(torch.from_numpy(U).cuda())
    return fx


def host_input(dims, N, roughness, seed, prec):
    U = gi.make_links_sun(dims, N, roughness, seed, dtype=np.float32 if prec == "f32" else np.float64)
    return U, np.ascontiguousarray(U.astype(np.float64))


@pytest.mark.parametrize("dims", LATTICES)
@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N", [2, 4])
def test_sun_one_sweep_links_F_theta(gf, N, prec, gauge, dims):
    U, Uo = host_input(dims, N, 0.5, 100 + N, prec)
    fx = fixer(gf, dims, N, gauge, prec, U)
    got = fx.get_links().cpu().numpy()
    assert np.array_equal(got, U)  # set/get round trip is exact (index work only)
    F, th = fx.measure()
    Fo, tho = sun.measure(Uo, dims, gauge, N)
    assert abs(F - Fo) <= (1e-13 if prec == "f64" else 2e-6) and abs(th - tho) <= (1e-12 if prec == "f64" else 1e-5) * tho
    for omega in (1.0, 1.7):
        fx.ovr_sweep(1, omega)
        sun.sweeps(Uo, dims, gauge, N, omega, n=1)
        got = fx.get_links().cpu().numpy().astype(np.float64)
        assert np.abs(got - Uo).max() <= TOL_LINK[prec]
        if prec == "f32":  # next sweep from the same (rounded) state on both sides
            Uo = np.ascontiguousarray(got)
    F, th = fx.measure()
    Fo, tho = sun.measure(Uo, dims, gauge, N)
    assert abs(F - Fo) <= (1e-10 if prec == "f64" else 1e-5) * abs(Fo) and tho / 1.5 <= th <= tho * 1.5
    fx.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N", [2, 4])
def test_sun_reunitarize_matches_oracle(gf, N, prec):
    dims = (6, 4, 4, 2)
    rng = np.random.default_rng(N)
    U, _ = host_input(dims, N, 0.5, 7, prec)
    U = np.ascontiguousarray(U + (1e-3 * rng.normal(size=U.shape)).astype(U.dtype))
    Uo = np.ascontiguousarray(U.astype(np.float64))
    fx = fixer(gf, dims, N, "landau", prec, U)
    fx.reunitarize()
    got = fx.get_links().cpu().numpy().astype(np.float64)
    fx.close()
    sun.reunitarize(Uo, dims, N)
    assert np.abs(got - Uo).max() <= (1e-13 if prec == "f64" else 5e-6)
    a, b = sun.unitarity(np.ascontiguousarray(got), dims, N)
    assert max(a, b) <= (1e-13 if prec == "f64" else 5e-6)


@pytest.mark.parametrize("N,gauge,prec,reunit", [(2, "landau", "f64", 0), (4, "landau", "f64", 0), (4, "coulomb", "f64", 7),
                                               (2, "coulomb", "f32", 20), (4, "landau", "f32", 20)])
def test_sun_fix_trajectory(gf, N, gauge, prec, reunit):
    dims = (8, 8, 8, 8) if gauge == "landau" else (8, 8, 8, 4)
    omega, eps, cap, every = 1.7, (1e-12 if prec == "f64" else 1e-7), 400, 10
    U, Uo = host_input(dims, N, 0.4, 55, prec)
    fx = fixer(gf, dims, N, gauge, prec, U)
    fx.set_reunit_every(reunit)
    done = fx.fix(omega, eps, cap, every)
    hist = fx.history()
    links = fx.get_links().cpu().numpy().astype(np.float64)
    fx.close()
    odone, ohist = sun.fix(Uo, dims, gauge, N, omega, eps, cap, every, reunit_every=reunit)
    assert abs(done - odone) <= 0.02 * odone
    tolF = 1e-10 if prec == "f64" else 1e-5
    floor = 1e-28 if prec == "f64" else 1e-11
    for (s, F, th), (so, Fo, tho) in zip(hist, ohist):
        assert s == so and abs(F - Fo) <= tolF * abs(Fo)
        if tho > floor:
            assert tho / 1.5 <= th <= tho * 1.5, (s, th, tho)
    a, b = sun.unitarity(np.ascontiguousarray(links), dims, N)
    assert max(a, b) <= (1e-12 if prec == "f64" else 1e-4)
    if prec == "f64" and ohist[-1][2] < eps:
        assert hist[-1][2] < eps


def test_sun_ncolors3_is_the_su3_path_and_error_codes(gf):
    import torch

    dims = (4, 4, 4, 4)
    assert gf.gf_workspace_bytes_sun(3, *dims, gf.GF_FP64) == gf.gf_workspace_bytes(*dims, gf.GF_FP64, 18)
    assert gf.gf_workspace_bytes_sun(5, *dims, gf.GF_FP64) == 0 and gf.gf_workspace_bytes_sun(1, *dims, gf.GF_FP64) == 0
    assert gf.gf_workspace_bytes_sun(2, 4, 4, 3, 4, gf.GF_FP64) == 0
    ws = torch.empty(gf.gf_workspace_bytes_sun(4, *dims, gf.GF_FP64), dtype=torch.uint8, device="cuda")
    rc, _ = gf.gf_create_sun(5, *dims, gf.GF_LANDAU, gf.GF_FP64, ws.data_ptr(), ws.numel(), 0)
    assert rc == gf.GF_EUNSUPPORTED
    rc, _ = gf.gf_create_sun(4, 4, 4, 4, 5, gf.GF_LANDAU, gf.GF_FP64, ws.data_ptr(), ws.numel(), 0)
    assert rc == gf.GF_EODD
    rc, _ = gf.gf_create_sun(4, *dims, gf.GF_LANDAU, gf.GF_FP64, ws.data_ptr(), 1024, 0)
    assert rc == gf.GF_ENOMEM
    # ncolors = 3 through gf_create_sun: bit-identical to gf_create(storage = 18)
    U = gi.make_links(dims, 0.5, 3)
    a = gf.GaugeFixer(dims, ncolors=3)
    a.set_links(torch.from_numpy(U).cuda())
    a.ovr_sweep(2, 1.7)
    rc, h = gf.gf_create_sun(3, *dims, gf.GF_LANDAU, gf.GF_FP64, ws.data_ptr(), ws.numel(), 0)
    assert rc == gf.GF_OK
    dev = torch.from_numpy(U).cuda()
    assert gf.gf_set_links(h, dev.data_ptr()) == gf.GF_OK and gf.gf_ovr_sweep(h, 2, 1.7) == gf.GF_OK
    assert gf.gf_get_links(h, dev.data_ptr()) == gf.GF_OK
    torch.cuda.synchronize()
    assert torch.equal(dev, a.get_links())
    gf.gf_destroy(h)
    a.close()
    # what an SU(N != 3) context refuses
    fx = gf.GaugeFixer(dims, gauge="coulomb", ncolors=4)
    for call in (lambda: fx.set_option(gf.GF_OPT_SWEEP_VARIANT, 1), fx.fft_attach, fx.measure_slices,
                 fx.defer_temporal_links):
        with pytest.raises(gf.GFError) as e:
            call()
        assert e.value.code == gf.GF_EUNSUPPORTED
    fx.close()
