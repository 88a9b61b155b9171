"""Pins for G1: the oracle's Philox4x32-10 and its uniform construction.

External pin: cuRAND's *host* generator CURAND_RNG_PSEUDO_PHILOX4_32_10 (runs without a GPU).  Observed
mapping (probed, not assumed): with seed s and default ordering, output words 4j..4j+3 (j < 8192) are
Philox4x32-10(counter = (0, 0, j, 0), key = (s_lo, s_hi)).  The Random123 known-answer file is not in this
container and is not written out from memory."""
import ctypes
import glob

import numpy as np
import pytest

import oracle


def _curand():
    cands = ["/usr/local/cuda/lib64/libcurand.so.10"] + glob.glob(
        "/opt/prime-rl/.venv/lib/python3*/site-packages/nvidia/curand/lib/libcurand.so.10")
    for c in cands:
        try:
            return ctypes.CDLL(c)
        except OSError:
            continue
    return None


def _curand_words(lib, seed, n):
    gen = ctypes.c_void_p()
    assert lib.curandCreateGeneratorHost(ctypes.byref(gen), 161) == 0  # PHILOX4_32_10
    assert lib.curandSetPseudoRandomGeneratorSeed(gen, ctypes.c_ulonglong(seed)) == 0
    out = np.zeros(n, dtype=np.uint32)
    assert lib.curandGenerate(gen, out.ctypes.data_as(ctypes.c_void_p), ctypes.c_size_t(n)) == 0
    lib.curandDestroyGenerator(gen)
    return out


@pytest.mark.parametrize("seed", [0, 42, 0x0123456789ABCDEF, 0xFFFFFFFFFFFFFFFF])
def test_philox_matches_curand_host(seed):
    lib = _curand()
    if lib is None:
        pytest.skip("libcurand not found")
    nq = 2048
    words = _curand_words(lib, seed, 4 * nq)
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for j in range(nq):
        assert oracle.philox4x32_10([0, 0, j, 0], key) == [int(v) for v in words[4 * j:4 * j + 4]]


def test_uniform_pair_is_53_bit_of_words():
    # u = ((w0 * 2^32 + w1) >> 11) * 2^-53: exact integer reconstruction, u in [0, 1)
    for idx, blk, strm in [(0, 0, 0), (7, 3, 2), ((1 << 40) + 5, 4, 1)]:
        w = oracle.philox4x32_10([idx & 0xFFFFFFFF, idx >> 32, blk, strm], [42, 0])
        u = oracle.uniform_pair(42, idx, blk, strm)
        assert u[0] == (((w[0] << 32) | w[1]) >> 11) / float(1 << 53)
        assert u[1] == (((w[2] << 32) | w[3]) >> 11) / float(1 << 53)
        assert 0.0 <= u[0] < 1.0 and 0.0 <= u[1] < 1.0


def test_counter_words_all_matter():
    base = oracle.philox4x32_10([1, 2, 3, 4], [5, 6])
    for pos in range(4):
        c = [1, 2, 3, 4]
        c[pos] += 1
        assert oracle.philox4x32_10(c, [5, 6]) != base
    assert oracle.philox4x32_10([1, 2, 3, 4], [6, 6]) != base
    assert oracle.philox4x32_10([1, 2, 3, 4], [5, 7]) != base


def test_uniform_moments():
    n = 200_000
    u = np.array([oracle.uniform_pair(42, i, 0, 0) for i in range(0, n, 40)]).ravel()
    m = len(u)
    assert abs(u.mean() - 0.5) < 5 / np.sqrt(12 * m)
    assert abs((u ** 2).mean() - 1 / 3) < 5 * np.sqrt(4 / 45 / m)
    a, b = u[0::2], u[1::2]
    assert abs(np.corrcoef(a, b)[0, 1]) < 5 / np.sqrt(len(a))
