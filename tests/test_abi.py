"""The C-ABI library builds, loads without a GPU and exports every symbol include/hydro.h
declares; argument errors that need no device are reported through the status code."""
import ctypes as C
import os
import re

import pytest

from paper_1812_07977_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libs():
    build.build()
    return binding.load_library(False), binding.load_library(True)


def test_header_symbols_all_exported(libs):
    header = open(os.path.join(ROOT, "include", "hydro.h")).read()
    declared = set(re.findall(r"\b(hydro_[a-z_]+)\s*\(", header))
    assert declared == set(binding.SYMBOLS), declared ^ set(binding.SYMBOLS)
    for L in libs:
        for name in declared:
            assert hasattr(L, name), name


def test_build_flavours(libs):
    prod, ver = libs
    assert prod.hydro_is_verification_build() == 0
    assert ver.hydro_is_verification_build() == 1


def test_argument_errors_without_device(libs):
    L = libs[0]
    h = C.c_void_p()
    ok = (C.c_int * 6)(0, 0, 0, 0, 0, 0)
    assert L.hydro_create(1, 4, 4, 1.4, 0.1, ok, C.byref(h)) == 1          # HYDRO_ERR_ARG
    assert L.hydro_create(4, 4, 4, 1.0, 0.1, ok, C.byref(h)) == 1
    assert L.hydro_create(4, 4, 4, 1.4, -1.0, ok, C.byref(h)) == 1
    bad = (C.c_int * 6)(2, 0, 0, 0, 0, 0)
    assert L.hydro_create(4, 4, 4, 1.4, 0.1, bad, C.byref(h)) == 1
    assert b"periodic" in L.hydro_last_error()
    assert L.hydro_step(None, 0.1) == 1
    assert L.hydro_launch_count() == 0


def test_no_cpu_fallback_without_device(libs):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    L = libs[0]
    h = C.c_void_p()
    ok = (C.c_int * 6)(0, 0, 0, 0, 0, 0)
    assert L.hydro_create(4, 4, 4, 1.4, 0.1, ok, C.byref(h)) == 3          # HYDRO_ERR_CUDA
    assert not h.value
    with pytest.raises(RuntimeError):
        binding.Hydro(4, 4, 4, 1.4, 0.1, (0,) * 6)


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1812_07977_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "liboracle" not in text, f


def test_tiling_partition_covers_every_plane_once(libs):
    """Host logic of the fused kernel's launch geometry (hydro_tiling_partition, no device): whatever the
    grid, the tile height, the requested chunk length and the plane range, the layers tile [kb, ke)
    exactly, in order, without empty layers -- the same arithmetic the kernel uses to find its chunk."""
    import random
    rnd = random.Random(7)
    cases = [(256, 256, 256, 16, 0, 148, 0, 256), (128, 128, 128, 16, 0, 148, 0, 128), (32, 32, 32, 8, 0, 148, 0, 32),
             (512, 512, 512, 16, 0, 148, 0, 512), (160, 160, 160, 16, 0, 148, 0, 160), (33, 257, 65, 16, 0, 148, 0, 65),
             (64, 64, 2048, 16, 0, 148, 16, 2032), (2, 2, 2, 8, 0, 148, 0, 2), (100, 70, 45, 8, 7, 148, 0, 45)]
    for _ in range(300):
        nx, ny, nz = (rnd.randint(2, 600), rnd.randint(2, 600), rnd.randint(2, 700))
        kb = rnd.choice([0, 0, rnd.randint(0, nz - 1)])
        ke = rnd.choice([nz, nz, rnd.randint(kb + 1, nz)])
        cases.append((nx, ny, nz, rnd.choice([8, 16]), rnd.choice([0, 0, 0, rnd.randint(1, nz)]),
                      rnd.choice([148, 148, 132, 1, 7]), kb, ke))
    for nx, ny, nz, ty, lzreq, sms, kb, ke in cases:
        layers, (lz, km, nprim, lzr, nlayer) = binding.tiling_partition(nx, ny, nz, ty, lzreq, sms, kb, ke)
        assert len(layers) == nlayer >= 1 and lz >= 1 and lzr >= 1 and kb < km <= ke, (nx, ny, nz, ty, lzreq, sms)
        assert layers[0][0] == kb and layers[-1][1] == ke
        for (a0, a1), (b0, b1) in zip(layers, layers[1:]):
            assert a1 == b0
        assert all(k1 > k0 for k0, k1 in layers), (layers, nx, ny, nz, ty, lzreq, sms, kb, ke)
        if lzreq:
            assert km == ke and lz == min(lzreq, ke - kb)


def test_tiling_partition_balances_the_paper_sizes(libs):
    """256^3 per GPU is the paper's benchmark size and 128^3 its production size: on 148
    SMs with 32 x 16 tiles the balanced layers put one thick chunk of every tile on its own SM and hand
    the thin remainder to the SMs left over, instead of 6.9 / 0.86 waves of uniform 32-plane chunks."""
    for n, tiles in ((256, 128), (128, 32)):
        layers, (lz, km, nprim, lzr, nlayer) = binding.tiling_partition(n, n, n, 16)
        q = 148 // tiles
        assert nprim == q and km < n and tiles * nprim <= 148
        left = 148 - tiles * nprim
        rest = nlayer - nprim
        rounds = -(-tiles * rest // left)
        primary = lz + 1.25
        remainder = rounds * (lzr + 1.25)
        assert abs(primary - remainder) <= 0.15 * primary          # the two sides finish together
        assert primary < 1.06 * (n * tiles / 148 + 1.25)            # within 6 % of a perfect split


def test_committed_ncu_capture_is_of_the_committed_sources():
    """bench.py's roofline.traffic comes from profiles/traffic.txt, which names the sources (hash of
    csrc/) its ncu capture was taken from; bench.py refuses a capture of other sources.  The committed
    pair must match, so that the bench line carries a measured traffic figure."""
    import sys
    sys.path.insert(0, ROOT)
    import bench
    p = os.path.join(ROOT, "profiles", "traffic.txt")
    if not os.path.exists(p):
        pytest.skip("no committed capture")
    kv = dict(ln.split() for ln in open(p) if len(ln.split()) == 2 and not ln.startswith("#"))
    assert kv["csrc_sha256"] == bench.csrc_sha256(), "re-capture profiles/ after changing csrc/"
    t = bench.load_traffic(3)
    assert t["dram"] and abs(t["dram"] / (200.0 * 256 ** 3) - 1.0) < 0.1      # within 10 % of the algorithmic bytes
