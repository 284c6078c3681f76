"""CPU-side checks of the C-ABI library: it builds, loads, exports every symbol include/gf.h declares, and rejects bad
arguments with the documented codes before touching the device (no compute calls here)."""
import ctypes
import os
import re

import paper_1412_1498_b200 as gf

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "gf.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(gf_[a-z_0-9]+)\s*\(", header))
    assert declared == set(gf.SYMBOLS), declared ^ set(gf.SYMBOLS)
    lib = ctypes.CDLL(os.path.join(ROOT, "paper_1412_1498_b200", "libgf.so"))
    for name in declared:
        assert hasattr(lib, name), name


def test_workspace_bytes():
    # links 4V*L + partials + result + 2 staging buffers of 64 MiB
    for dims, prec, storage, L in [((8, 8, 8, 8), gf.GF_FP64, 18, 144), ((8, 8, 8, 8), gf.GF_FP32, 12, 48),
                                   ((64, 64, 64, 128), gf.GF_FP64, 18, 144), ((48, 48, 48, 96), gf.GF_FP64, 12, 96)]:
        V = dims[0] * dims[1] * dims[2] * dims[3]
        n = gf.gf_workspace_bytes(*dims, prec, storage)
        assert 4 * V * L + (128 << 20) <= n <= 4 * V * L + (128 << 20) + (8 << 20)
    assert gf.gf_workspace_bytes(7, 8, 8, 8, 0, 18) == 0
    assert gf.gf_workspace_bytes(8, 8, 8, 8, 0, 10) == 0
    assert 0 < gf.gf_workspace_bytes(8, 8, 8, 8, 1, 8) < gf.gf_workspace_bytes(8, 8, 8, 8, 1, 12)  # 8-real, FP32
    assert 0 < gf.gf_workspace_bytes(8, 8, 8, 8, 0, 8) < gf.gf_workspace_bytes(8, 8, 8, 8, 0, 12)
    assert gf.gf_workspace_bytes(8, 8, 8, 8, 2, 18) == 0


def test_create_rejects_bad_arguments_before_touching_the_device():
    big = 1 << 40
    assert gf.gf_create(7, 8, 8, 8, 0, 0, 18, 256, big, 0)[0] == gf.GF_EODD
    assert gf.gf_create(8, 8, 0, 8, 0, 0, 18, 256, big, 0)[0] == gf.GF_EODD
    assert gf.gf_create(8, 8, 8, 8, 2, 0, 18, 256, big, 0)[0] == gf.GF_EUNSUPPORTED
    assert gf.gf_create(8, 8, 8, 8, 0, 3, 18, 256, big, 0)[0] == gf.GF_EUNSUPPORTED
    assert gf.gf_create(8, 8, 8, 8, 0, 0, 10, 256, big, 0)[0] == gf.GF_EUNSUPPORTED  # storage must be 18, 12 or 8
    assert gf.gf_create(8, 8, 8, 8, 0, 1, 9, 256, big, 0)[0] == gf.GF_EUNSUPPORTED   # storage must be 18, 12 or 8
    assert gf.gf_create(8, 8, 8, 8, 0, 0, 18, 0, big, 0)[0] == gf.GF_EINVAL
    assert gf.gf_create(8, 8, 8, 8, 0, 0, 18, 256, 1024, 0)[0] == gf.GF_ENOMEM
    assert gf.gf_create(8, 8, 8, 8, 0, 0, 18, 264, big, 0)[0] == gf.GF_ENOMEM        # misaligned
    assert gf.gf_create(2048, 2048, 2048, 2, 0, 0, 18, 256, big, 0)[0] == gf.GF_EUNSUPPORTED  # V >= 2^31


def test_null_context_is_einval():
    assert gf.gf_ovr_sweep(None, 1, 1.5) == gf.GF_EINVAL
    assert gf.gf_measure(None)[0] == gf.GF_EINVAL
    assert gf.gf_fix(None, 1.5, 1e-10, 10, 1)[0] == gf.GF_EINVAL
    assert gf.gf_set_links(None, 256) == gf.GF_EINVAL
    assert gf.gf_get_links(None, 256) == gf.GF_EINVAL
    assert gf.gf_reunitarize(None) == gf.GF_EINVAL
    assert gf.gf_kernel_launches(None) == 0
    gf.gf_destroy(None)
    for code in range(0, -7, -1):
        assert gf.gf_strerror(code) not in ("", "unknown error")


def test_product_does_not_import_oracle():
    # the product path must never route through the oracle (or any CPU fallback)
    pkg = os.path.join(ROOT, "paper_1412_1498_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no oracle", ""), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            assert "paper_1412_1498_b200 import" not in open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1412_1498_b200" not in open(os.path.join(ROOT, "oracle", f)).read()


def test_header_compiles_as_c99_and_links_from_c(tmp_path):
    """include/gf.h is advertised as a C ABI: a C99 translation unit includes it, links libgf.so and walks the error
    paths that return before any device work."""
    import subprocess

    libdir = os.path.join(ROOT, "paper_1412_1498_b200")
    exe = str(tmp_path / "cabi_consumer")
    subprocess.check_call(["gcc", "-std=c99", "-pedantic", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"),
                           os.path.join(ROOT, "tests", "cabi_consumer.c"), "-o", exe, "-L", libdir, "-lgf",
                           f"-Wl,-rpath,{libdir}"])
    r = subprocess.run([exe], capture_output=True, text=True, timeout=120)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "cabi_consumer: ok" in r.stdout


def test_driver_decisions_behind_the_abi():
    """gf_fix_plan / gf_combine_slabs: the stop test, cadence and the slabs' means that callers driving several contexts
    take from the library (Algorithm 1 l.2); no device work."""
    # (omega, eps, max_sweeps, check_every, sweeps_done, theta) -> sweeps to the next measurement
    assert gf.gf_fix_plan(1.7, 1e-12, 2000, 10, 0, 5.0) == (gf.GF_OK, 10)
    assert gf.gf_fix_plan(1.7, 1e-12, 2000, 10, 1995, 5.0) == (gf.GF_OK, 5)      # capped by max_sweeps
    assert gf.gf_fix_plan(1.7, 1e-12, 2000, 10, 2000, 5.0) == (gf.GF_OK, 0)      # cap reached
    assert gf.gf_fix_plan(1.7, 1e-12, 2000, 10, 40, 9e-13) == (gf.GF_OK, 0)      # theta < eps: stop
    assert gf.gf_fix_plan(1.7, 1e-12, 2000, 10, 40, 1e-12) == (gf.GF_OK, 10)     # theta == eps: not yet
    assert gf.gf_fix_plan(1.7, 0.0, 200, 20, 180, 0.0) == (gf.GF_OK, 20)         # eps = 0: fixed-sweep run
    for bad in [(2.0, 1e-12, 10, 1, 0, 1.0), (0.99, 1e-12, 10, 1, 0, 1.0), (1.7, -1.0, 10, 1, 0, 1.0),
                (1.7, 1e-12, -1, 1, 0, 1.0), (1.7, 1e-12, 10, 0, 0, 1.0), (1.7, 1e-12, 10, 1, -1, 1.0)]:
        assert gf.gf_fix_plan(*bad)[0] == gf.GF_EINVAL
    rc, F, th = gf.gf_combine_slabs([0.25, 0.5, 0.75, 1.0], [4.0, 3.0, 2.0, 1.0])
    assert (rc, F, th) == (gf.GF_OK, 0.625, 2.5)
    # slab order: the sum is taken left to right, so every rank gets the same bits
    xs = [0.1, 0.2, 0.3]
    assert gf.gf_combine_slabs(xs, xs)[1] == ((0.1 + 0.2) + 0.3) / 3
    assert gf.gf_combine_slabs([float("nan")], [1.0])[0] == gf.GF_ENUMERIC
    # the group calls refuse contexts that are not slabs with peer targets and flags, before any device work
    assert gf.gf_slab_group_sweep([], 1, 1.7) == gf.GF_EINVAL
    assert gf.gf_slab_group_refresh([]) == gf.GF_EINVAL
    assert gf.gf_ipc_export(0)[0] == gf.GF_EINVAL and gf.gf_ipc_open(b"\0" * 64, 0)[0] in (gf.GF_ECUDA, gf.GF_EINVAL)
