"""gf_measure_static: the one entry point of libgf that allocates nothing.

Who needs it: a caller that holds a gauge field on the GPU but has no way to obtain more device memory - a plug-in
inside an application whose pool already owns the card, or code that must not call cudaMalloc / cudaFree once the job
is running because those calls synchronise the whole device.  Such a caller cannot even create a gf context (gf_create
wants a workspace), so it gets F and theta from a kernel whose reduction scratch is a fixed 256 KiB array inside the
library, good for lattices of up to gf_measure_static_max_sites() sites.

What is checked: the new entry point against the existing path (GaugeFixer.set_links + measure, which the parity tests
hold to the CPU reference), to the tolerances tests/test_gpu_parity.py::test_measure_matches_oracle uses, on two calls
in a row - the second on a DIFFERENT field and lattice shape, so that anything the first call left behind in the shared
array (stale partial sums beyond the new block count, a counter that was not put back to zero) would show.  The file
sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the parity tests.  It
holds no state of its own, so it passes alone in a fresh process (the very first call then does the per-device set-up)
as well as after the whole suite.
"""
import numpy as np
import pytest

import gf_inputs as gi

pytestmark = pytest.mark.gpu

# as test_measure_matches_oracle: F is compared on the scale of its O(1) summands, theta relative to itself
ATOL_F = {"f64": 1e-13, "f32": 2e-7}
RTOL_THETA = {"f64": 1e-12, "f32": 2e-6}


@pytest.fixture(scope="module")
def gf():
    import paper_1412_1498_b200 as m
    return m


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available()
    return t


def existing_path(gf, torch, links, dims, gauge, prec):
    fx = gf.GaugeFixer(dims, gauge=gauge, prec=prec, storage=18)
    fx.set_links(links)
    F, th = fx.measure()
    fx.close()
    return F, th


@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_two_calls_in_a_row_match_the_existing_measure(gf, torch, gauge, prec):
    dt = np.float64 if prec == "f64" else np.float32
    # first a lattice of 40 blocks, then a ragged one of 3 blocks (960 / 256 = 3.75): the second call reuses the array
    # the first one filled
    cases = [((16, 8, 8, 10), 0.5, 21), ((10, 6, 4, 4), 0.3, 22)]
    fields = [torch.from_numpy(gi.make_links(dims, rough, seed, dtype=dt)).cuda() for dims, rough, seed in cases]
    got = [gf.measure_static(U, dims, gauge=gauge) for U, (dims, _, _) in zip(fields, cases)]
    again = gf.measure_static(fields[0], cases[0][0], gauge=gauge)
    assert again == got[0]  # deterministic summation order: the same field gives the same bits, whatever ran between
    for U, (dims, _, _), (F, th) in zip(fields, cases, got):
        Fe, the = existing_path(gf, torch, U, dims, gauge, prec)
        assert abs(F - Fe) <= ATOL_F[prec], (dims, F, Fe)
        assert abs(th - the) <= RTOL_THETA[prec] * the, (dims, th, the)


def test_allocates_nothing_and_refuses_what_does_not_fit(gf, torch):
    dims = (8, 8, 8, 8)
    U = torch.from_numpy(gi.make_links(dims, 0.4, 23)).cuda()
    gf.measure_static(U, dims)  # per-device set-up done
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    reserved_before = torch.cuda.memory_reserved()
    F, th = gf.measure_static(U, dims)
    torch.cuda.synchronize()
    # free device memory did not go down (nothing else runs on the test box) and torch's pool was not asked either
    assert torch.cuda.mem_get_info()[0] >= free_before and torch.cuda.memory_reserved() == reserved_before
    assert 0.0 < F < 1.0 and th > 0.0

    limit = gf.gf_measure_static_max_sites()
    assert limit == 256 * 16384
    # 32^3 x 128 is exactly the limit (test_the_largest_lattice_that_fits runs it); the next even extent up is refused
    # by the size check, before the pointer is looked at
    rc, _, _ = gf.gf_measure_static(U.data_ptr(), 32, 32, 32, 130, gf.GF_LANDAU, gf.GF_FP64)
    assert rc == gf.GF_ENOMEM
    msg = gf.gf_static_last_error()
    assert "4194304" in msg and "gf_create" in msg
    with pytest.raises(gf.GFError) as ei:
        gf.measure_static(U, (48, 48, 48, 96))
    assert ei.value.code == gf.GF_ENOMEM
    # the other documented refusals, none of which reaches a kernel
    assert gf.gf_measure_static(0, *dims, gf.GF_LANDAU, gf.GF_FP64)[0] == gf.GF_EINVAL
    assert gf.gf_measure_static(U.data_ptr(), 7, 8, 8, 8, gf.GF_LANDAU, gf.GF_FP64)[0] == gf.GF_EODD
    assert gf.gf_measure_static(U.data_ptr(), *dims, 2, gf.GF_FP64)[0] == gf.GF_EUNSUPPORTED
    assert gf.gf_measure_static(U.data_ptr(), *dims, gf.GF_LANDAU, 2)[0] == gf.GF_EUNSUPPORTED
    assert gf.gf_measure_static(U.data_ptr() + 8, *dims, gf.GF_LANDAU, gf.GF_FP64)[0] == gf.GF_EINVAL
    host = np.zeros(72 * 4096)
    assert gf.gf_measure_static(host.ctypes.data & ~15, *dims, gf.GF_LANDAU, gf.GF_FP64)[0] == gf.GF_EINVAL
    # and the entry point still works after the refusals
    assert gf.measure_static(U, dims) == (F, th)


def test_the_largest_lattice_that_fits(gf, torch):
    """32^3 x 128 = the stated limit, FP32 (2.4 GB of links): every slot of the array is in use."""
    dims = (32, 32, 32, 128)
    U = torch.empty((gi.volume(dims), 4, 3, 3, 2), dtype=torch.float32, device="cuda")
    gi.make_links_device(U.data_ptr(), dims, 0.4, 24, "f32", torch.cuda.current_stream().cuda_stream)
    F, th = gf.measure_static(U, dims)
    Fe, the = existing_path(gf, torch, U, dims, "landau", "f32")
    assert abs(F - Fe) <= ATOL_F["f32"] and abs(th - the) <= RTOL_THETA["f32"] * the, (F, Fe, th, the)
