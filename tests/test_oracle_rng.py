"""Pins for the oracle's Philox-4x32-10 and its uniform map.

The published known-answer vectors are not in this container and are not typed from memory; the
pin is the CUDA toolkit's own cuRAND *host* generator (CURAND_RNG_PSEUDO_PHILOX4_32_10), a library
implementation that runs on the CPU.  Its default ordering emits 4-word group G (G = offset/4 + position)
as the block Philox(counter=(c0, c1, G mod 65536, 0), key=seed) with c0 + 2^32 c1 = G div 65536 --
found by experiment, asserted below.
"""
import ctypes

import numpy as np
import pytest

import oracle


def _curand():
    try:
        return ctypes.CDLL("libcurand.so.10")
    except OSError:
        try:
            return ctypes.CDLL("/usr/local/cuda/lib64/libcurand.so.10")
        except OSError:
            pytest.skip("libcurand not loadable")


def _curand_words(seed, offset, n_words):
    lib = _curand()
    gen = ctypes.c_void_p()
    assert lib.curandCreateGeneratorHost(ctypes.byref(gen), 161) == 0   # PHILOX4_32_10
    lib.curandSetPseudoRandomGeneratorSeed.argtypes = [ctypes.c_void_p, ctypes.c_ulonglong]
    lib.curandSetGeneratorOffset.argtypes = [ctypes.c_void_p, ctypes.c_ulonglong]
    lib.curandGenerate.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t]
    assert lib.curandSetPseudoRandomGeneratorSeed(gen, seed) == 0
    assert lib.curandSetGeneratorOffset(gen, offset) == 0
    out = np.zeros(n_words, dtype=np.uint32)
    assert lib.curandGenerate(gen, out.ctypes.data_as(ctypes.c_void_p), n_words) == 0
    lib.curandDestroyGenerator.argtypes = [ctypes.c_void_p]
    lib.curandDestroyGenerator(gen)
    return out


@pytest.mark.parametrize("seed", [0, 1, 3, 0x0123456789ABCDEF, 0xFFFFFFFFFFFFFFFF])
def test_philox_matches_curand_host_subsequences(seed):
    words = _curand_words(seed, 0, 4 * 512).reshape(-1, 4)
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for g in range(512):
        assert oracle.philox4x32_10([0, 0, g, 0], key) == [int(v) for v in words[g]], g


@pytest.mark.parametrize("c0,c1", [(1, 0), (12345, 0), (0xFFFFFFFF, 0), (0, 1), (0xDEADBEEF, 0x7), (0xFFFFFFFE, 0x3FF)])
def test_philox_matches_curand_host_offsets(c0, c1):
    seed = 0x9E3779B97F4A7C15
    c2_start = 65530                      # crosses the 65536-subsequence wrap into c0 + 1
    offset = 4 * (c2_start + 65536 * (c0 + (c1 << 32)))
    words = _curand_words(seed, offset, 4 * 12).reshape(-1, 4)
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for g in range(12):
        G = c2_start + g
        hi = c0 + (c1 << 32) + G // 65536
        ctr = [hi & 0xFFFFFFFF, (hi >> 32) & 0xFFFFFFFF, G % 65536, 0]
        assert oracle.philox4x32_10(ctr, key) == [int(v) for v in words[g]]


def test_philox_is_sensitive_to_every_input_word():
    base_c, base_k = [5, 6, 7, 3], [11, 13]
    ref = oracle.philox4x32_10(base_c, base_k)
    for w in range(4):
        c = list(base_c)
        c[w] ^= 1
        out = oracle.philox4x32_10(c, base_k)
        flipped = sum(bin(a ^ b).count("1") for a, b in zip(ref, out))
        assert 40 <= flipped <= 88, (w, flipped)   # ~64 of 128 bits
    for w in range(2):
        k = list(base_k)
        k[w] ^= 1
        out = oracle.philox4x32_10(base_c, k)
        flipped = sum(bin(a ^ b).count("1") for a, b in zip(ref, out))
        assert 40 <= flipped <= 88, (w, flipped)


def test_counter_layout_and_uniform_map():
    seed, idx, k, tag = 0xABCDEF0123456789, (7 << 32) | 99, 17, oracle.TAG_E
    r = oracle.philox4x32_10([99, 7, 17, tag], [seed & 0xFFFFFFFF, seed >> 32])
    ua, ub = oracle.uniforms(seed, idx, k, tag)
    from fractions import Fraction
    assert Fraction(ua) == Fraction(2 * ((r[0] << 20) | (r[1] >> 12)) + 1, 1 << 53)
    assert Fraction(ub) == Fraction(2 * ((r[2] << 20) | (r[3] >> 12)) + 1, 1 << 53)


def test_uniforms_open_interval_exact_complement_and_moments():
    from fractions import Fraction
    us = np.array([oracle.uniforms(3, i, 1, oracle.TAG_Z)[0] for i in range(20000)])
    assert us.min() > 0.0 and us.max() < 1.0
    for u in us[:200]:
        assert Fraction(1.0 - u) == 1 - Fraction(u)     # 1-u exact in fp64
    n = us.size
    assert abs(us.mean() - 0.5) < 4 * np.sqrt(1 / 12 / n)
    assert abs(us.var() - 1 / 12) < 4 * np.sqrt(1 / 180 / n)
    # different tags / sweeps give unrelated streams
    vs = np.array([oracle.uniforms(3, i, 2, oracle.TAG_Z)[0] for i in range(20000)])
    assert abs(np.corrcoef(us, vs)[0, 1]) < 0.03
