"""GPU device-function parity: Philox words and uniforms bit-exact, variate maps within fp64
tolerance of the oracle's long-double evaluation."""
import numpy as np
import pytest
import torch

import oracle
import paper_1608_04329_b200 as hsp

pytestmark = pytest.mark.gpu


def test_philox_words_bit_exact():
    rng = np.random.default_rng(0)
    n = 300000
    ctr = rng.integers(0, 2 ** 32, size=(n, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2 ** 32, size=(n, 2), dtype=np.uint64).astype(np.uint32)
    ctr[:8] = [[0, 0, 0, 0], [1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 0], [0, 0, 0, 1], [0xFFFFFFFF] * 4, [5, 0, 1, 3], [7, 7, 7, 7]]
    got = hsp.dbg_philox(torch.from_numpy(ctr.view(np.int32)).cuda(), torch.from_numpy(key.view(np.int32)).cuda())
    got = got.cpu().numpy().view(np.uint32)
    assert np.array_equal(got, oracle.philox_many(ctr, key))


@pytest.mark.parametrize("tag", [0, 1, 2, 3, 4, 5])
def test_uniform_addressing_bit_exact(tag):
    seed = 0xC0FFEE1234567890
    idx = np.concatenate([np.arange(5000, dtype=np.uint64), np.array([2 ** 32 - 1, 2 ** 32, 2 ** 40 + 17, 2 ** 63], dtype=np.uint64)])
    ua, ub = hsp.dbg_uniform(seed, torch.from_numpy(idx.view(np.int64)).cuda(), 77, tag)
    oa, ob = oracle.uniforms_many(seed, idx, 77, tag)
    assert np.array_equal(ua.cpu().numpy(), oa) and np.array_equal(ub.cpu().numpy(), ob)


def test_tnpos_matches_oracle():
    rng = np.random.default_rng(1)
    m = np.concatenate([rng.uniform(-45, 45, 200000), rng.normal(0, 3, 200000), np.repeat([-100.0, -37.4, -30.0, -29.999, 0.0, 0.47, 8.0, 37.0], 64)])
    u = np.array(oracle.uniforms_many(5, np.arange(m.size), 1, 0)[0])
    u[-512::8] = 2.0 ** -53
    u[-511::8] = 1 - 2.0 ** -53
    w = hsp.dbg_tnpos(torch.from_numpy(m).cuda(), torch.from_numpy(u).cuda()).cpu().numpy()
    ref = oracle.tnpos_many(m, u)
    assert np.all(w > 0) and np.all(np.isfinite(w))
    t = ref - m
    err = np.abs(w - ref) / np.maximum(1.0, np.abs(t))
    print("tnpos max scaled err", err.max(), "at m,u", m[err.argmax()], u[err.argmax()])
    assert err.max() < 2e-13
    rel = np.abs(w - ref) / ref
    print("tnpos rel err: median", np.median(rel), "p99.9", np.quantile(rel, 0.999))


def test_norm_inv_matches_oracle():
    u = np.concatenate([oracle.uniforms_many(6, np.arange(200000), 1, 3)[0], [2.0 ** -53, 1 - 2.0 ** -53, 0.5]])
    x = hsp.dbg_norm_inv(torch.from_numpy(u).cuda()).cpu().numpy()
    ref = oracle.norm_inv_many(u)
    assert np.max(np.abs(x - ref) / np.maximum(1.0, np.abs(ref))) < 1e-14


@pytest.mark.parametrize("alpha", [1.5, 5.5, 50.5, 500.5, 2000.5])
def test_cheng_gamma_matches_oracle(alpha):
    n = 2000
    x = hsp.dbg_cheng(alpha, 99, 1, n).cpu().numpy()
    ref = np.array([oracle.cheng_gamma(alpha, 99, k)[0] for k in range(1, n + 1)])
    assert np.max(np.abs(x - ref) / ref) < 1e-13
