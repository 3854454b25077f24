"""Pins for the oracle's RNG and trigonometry (CPU only)."""
import ctypes as C
import math
import os
import shutil
import subprocess

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def curand_kat(tmp_path_factory):
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available")
    exe = str(tmp_path_factory.mktemp("kat") / "kat")
    subprocess.run([nvcc, "-Wno-deprecated-gpu-targets", "-o", exe, os.path.join(HERE, "curand_philox_kat.cu")], check=True,
                   capture_output=True)
    return exe


def test_philox_matches_curand_header(oracle, curand_kat):
    """cuRAND's own block function (toolkit header, compiled for the host) on 64 counter/key sets."""
    rng = np.random.default_rng(7)
    cases = [(0, 0, 0, 0, 0, 0), (1, 2, 3, 4, 5, 6), (0xFFFFFFFF,) * 6] + [tuple(int(x) for x in rng.integers(0, 2**32, 6)) for _ in range(61)]
    args = [str(v) for c in cases for v in c]
    out = subprocess.run([curand_kat, *args], check=True, capture_output=True, text=True).stdout.split("\n")
    for c, line in zip(cases, out):
        assert oracle.philox(*c) == tuple(int(x) for x in line.split())


def test_philox_matches_libcurand_host_generator(oracle):
    """libcurand's HOST Philox4_32_10 generator: output word 4*i+j == philox(counter=(0,0,i,0), key=seed)[j]
    (the host generator hands block i to cuRAND subsequence i, which is counter word 2)."""
    try:
        lib = C.CDLL("libcurand.so.10")
    except OSError:
        pytest.skip("libcurand not loadable")
    gen = C.c_void_p()
    if lib.curandCreateGeneratorHost(C.byref(gen), 161) != 0:   # CURAND_RNG_PSEUDO_PHILOX4_32_10
        pytest.skip("host generator unavailable")
    seed = 0x0123456789ABCDEF
    assert lib.curandSetPseudoRandomGeneratorSeed(gen, C.c_ulonglong(seed)) == 0
    buf = (C.c_uint32 * 64)()
    assert lib.curandGenerate(gen, buf, C.c_size_t(64)) == 0
    lib.curandDestroyGenerator(gen)
    got = list(buf)
    exp = []
    for i in range(16):
        exp += list(oracle.philox(0, 0, i, 0, seed & 0xFFFFFFFF, seed >> 32))
    assert got == exp


def test_u01_range_and_exactness(oracle):
    assert oracle.u01(0) == 0.0
    assert oracle.u01(0xFFFFFFFF) == (2**24 - 1) / 2**24 < 1.0
    assert oracle.u01(0x80000000) == 0.5
    assert oracle.u01(0x000000FF) == 0.0           # low 8 bits dropped


def test_sincos2pi_against_libm(oracle):
    us = np.concatenate([np.linspace(0, 1, 4001, endpoint=False), np.random.default_rng(0).random(4000),
                         [0.125, 0.25, 0.375, 0.5, 0.625, 0.75, 0.875, 1 - 2**-24]]).astype(np.float32)
    worst = 0.0
    for u in us:
        s, c = oracle.sincos2pi(float(u))
        worst = max(worst, abs(s - math.sin(2 * math.pi * float(u))), abs(c - math.cos(2 * math.pi * float(u))))
        assert abs(s * s + c * c - 1) < 5e-7
    assert worst < 4e-7, worst
    assert oracle.sincos2pi(0.0) == (0.0, 1.0)
    assert oracle.sincos2pi(0.25)[0] == 1.0 and oracle.sincos2pi(0.5)[1] == -1.0
