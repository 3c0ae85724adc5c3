"""Pin of the Philox counter layout against the CUDA toolkit's cuRAND DEVICE generator.

tests/test_oracle_rng.py pins the oracle's Philox-4x32-10 against cuRAND's HOST generator, which reaches counter words
c0, c1 and the key but never c2 / c3 (sweep, tag).  The device API addresses all four:
`curand_init(seed, subsequence, offset)` puts `subsequence` into (c2, c3) and `offset / 4` into (c0, c1).  A test-only
kernel (tests/cuda/curand_philox_probe.cu, compiled here with nvcc, not part of libhsp.so) draws one block per
(idx, k, tag) and the words are compared with `oracle.philox_many` -- something other than the builder's two
implementations agreeing with each other."""
import ctypes as C
import os
import shutil
import subprocess

import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def probe(tmp_path_factory):
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available to build the cuRAND probe")
    out = str(tmp_path_factory.mktemp("curand") / "libcurand_probe.so")
    subprocess.run([nvcc, "-O2", "-gencode", "arch=compute_100a,code=sm_100a", "-Xcompiler", "-fPIC", "-shared", "-o", out,
                    os.path.join(HERE, "cuda", "curand_philox_probe.cu")], check=True)
    L = C.CDLL(out)
    L.curand_philox_probe.argtypes = [C.c_ulonglong, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
    return L


@pytest.mark.parametrize("seed", [0, 3, 0xC0FFEE1234567890])
def test_counter_words_c2_c3_match_curand_device_philox(probe, seed):
    idx = np.array([0, 1, 2, 999_999, 2 ** 32 - 1, 2 ** 32, 2 ** 40 + 17, 2 ** 61 + 5], dtype=np.uint64)
    cases = [(i, k, tag) for i in idx for k in (1, 2, 77, 2 ** 32 - 1) for tag in range(7)]
    ii = np.array([c[0] for c in cases], dtype=np.uint64)
    kk = np.array([c[1] for c in cases], dtype=np.uint64)
    tt = np.array([c[2] for c in cases], dtype=np.uint64)
    subseq = (tt << np.uint64(32)) | kk
    offset = ii * np.uint64(4)
    out = np.zeros((len(cases), 4), dtype=np.uint32)
    rc = probe.curand_philox_probe(seed, subseq.ctypes.data, offset.ctypes.data, out.ctypes.data, len(cases))
    assert rc == 0
    ctr = np.stack([ii & np.uint64(0xFFFFFFFF), ii >> np.uint64(32), kk, tt], axis=1).astype(np.uint32)
    key = np.tile(np.array([seed & 0xFFFFFFFF, seed >> 32], dtype=np.uint32), (len(cases), 1))
    ref = oracle.philox_many(ctr, key)
    assert np.array_equal(out, ref)
    # the tag really moves the stream: blocks of different tags differ
    assert len({tuple(r) for r in out[:7]}) == 7
    # and the oracle's variate addressing (seed; idx, sweep, tag) IS that counter: U_A from words (r0, r1), U_B from (r2, r3)
    for q in range(0, len(cases), 5):
        i, k, tag = cases[q]
        ua, ub = oracle.uniforms(seed, int(i), int(k), int(tag))
        r = [int(v) for v in out[q]]
        assert ua == (float((r[0] << 20) | (r[1] >> 12)) + 0.5) * 2.0 ** -52
        assert ub == (float((r[2] << 20) | (r[3] >> 12)) + 0.5) * 2.0 ** -52
