"""Pins for the oracle's random numbers (BASELINE north_star: counter-based hash of (min(i,j), max(i,j), step, seed),
Philox-4x32-10; replaces PAPER.md:142).  The third implementation is cuRAND's own curand_Philox4x32_10 from the
CUDA toolkit header, compiled for the HOST by nvcc (tests/helpers/curand_philox_host.cu)."""
import os
import shutil
import subprocess

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def curand_host(tmp_path_factory):
    if shutil.which("nvcc") is None:
        pytest.skip("nvcc not available")
    d = tmp_path_factory.mktemp("curand")
    exe = str(d / "curand_philox_host")
    subprocess.check_call(["nvcc", "-O2", "-Wno-deprecated-gpu-targets", "-o", exe,
                           os.path.join(HERE, "helpers", "curand_philox_host.cu")])
    return exe, d


def test_philox_words_match_curand_bit_exact(orc, curand_host):
    exe, d = curand_host
    rng = np.random.Generator(np.random.PCG64(5))
    n = 1_000_000
    ctr = rng.integers(0, 2 ** 32, size=(n, 4), dtype=np.uint64).astype(np.uint32)
    # structured counters too: small ids, consecutive steps, the tags the method uses
    m = 4096
    ctr[:m, 0] = np.arange(m) % 64
    ctr[:m, 1] = ctr[:m, 0] + 1 + (np.arange(m) // 64)
    ctr[:m, 2] = np.arange(m) % 7
    ctr[:m, 3] = np.arange(m) % 5
    ctr[m] = 0
    ctr[m + 1] = 0xFFFFFFFF
    for key in ([0, 0], [20161119, 0], [0xDEADBEEF, 0x12345678]):
        fin, fout = str(d / "in.bin"), str(d / "out.bin")
        ctr.tofile(fin)
        subprocess.check_call([exe, fin, fout, str(key[0]), str(key[1])])
        ref = np.fromfile(fout, np.uint32).reshape(-1, 4)
        got = orc.philox_batch(ctr, key)
        assert np.array_equal(got, ref)


def test_gaussians_moments(orc):
    n = 2_500_000                                  # x4 Gaussians = 1e7 draws
    i = np.arange(n, dtype=np.int64)
    g = orc.gauss_batch(i, i + 1 + (i % 1000), 3, 0, 20161119).ravel()
    assert abs(g.mean()) < 1e-3
    assert abs(g.var() - 1.0) < 1e-3
    assert abs((g ** 4).mean() / g.var() ** 2 - 3.0) < 1e-2
    g4 = g.reshape(-1, 4)
    c = np.corrcoef(g4.T)
    assert np.abs(c - np.eye(4)).max() < 2e-3      # the four outputs are uncorrelated
    assert np.isfinite(g).all() and np.abs(g).max() < 5.7   # |g| <= sqrt(-2 ln 2^-24)


def test_uniform_mapping_and_box_muller_definition(orc):
    """u = ((x>>9)+1/2) 2^-23, (g0,g1) = sqrt(-2 ln u0) (cos, sin)(2 pi u1) on the raw Philox words."""
    ids = (np.arange(1000, dtype=np.int64), np.arange(1000, dtype=np.int64) * 3 + 7)
    seed = (0x12345678 << 32) | 0xDEADBEEF
    g = orc.gauss_batch(ids[0], ids[1], 11, 2, seed)
    lo, hi = np.minimum(*ids), np.maximum(*ids)
    ctr = np.stack([lo, hi, np.full(1000, 11), np.full(1000, 2)], 1).astype(np.uint32)
    x = orc.philox_batch(ctr, [0xDEADBEEF, 0x12345678]).astype(np.float64)
    u = (np.floor(x / 512.0) + 0.5) / 2 ** 23
    assert (u > 0).all() and (u < 1).all()
    assert np.array_equal(u.astype(np.float32).astype(np.float64), u)       # exactly representable in fp32
    for a, b, k in ((0, 1, 0), (2, 3, 2)):
        R = np.sqrt(-2 * np.log(u[:, a]))
        assert np.allclose(g[:, k], R * np.cos(2 * np.pi * u[:, b]), rtol=0, atol=1e-12)
        assert np.allclose(g[:, k + 1], R * np.sin(2 * np.pi * u[:, b]), rtol=0, atol=1e-12)


def test_pair_symmetry_of_the_stream(orc):
    """xi_ij = xi_ji ("symmetric"): the counter uses (min, max)."""
    a = orc.gauss4(17, 4000, 5, 0, 99)
    b = orc.gauss4(4000, 17, 5, 0, 99)
    assert np.array_equal(a, b)
    assert not np.array_equal(a, orc.gauss4(17, 4000, 6, 0, 99))     # step word matters
    assert not np.array_equal(a, orc.gauss4(17, 4000, 5, 1, 99))     # tag matters
    assert not np.array_equal(a, orc.gauss4(17, 4000, 5, 0, 100))    # seed matters
