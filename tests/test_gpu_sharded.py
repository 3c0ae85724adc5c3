"""Row-sharded chains (include/hsp.h) on ONE GPU: the ranks are emulated as two chains in
one process whose X^T z and Gram buffers are summed with torch between hsp_sweep_begin and hsp_sweep_end (no
kernel waits on another).  The multi-process loop itself (multi.sharded_sweeps + all-reduce) is covered on CPU by
tests/test_multi_gloo.py."""
import numpy as np
import pytest
import torch

import hsp_synth
import oracle
import paper_1608_04329_b200 as hsp
from paper_1608_04329_b200 import multi
from conftest import mixed_err

pytestmark = pytest.mark.gpu


def test_single_shard_equals_plain_chain_bitwise():
    wl = hsp_synth.make("C3", "cuda", n_rows=9001)
    g = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed)
    g.sweep(6)
    b0, l0, t0 = g.get_draws()
    g.close()
    s = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed, row_offset=0)
    with pytest.raises(RuntimeError):
        multi.sharded_sweeps(s, 1)                      # no explicit stream: the collective could not be ordered
    s.close()
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        s = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed, stream=stream, row_offset=0)
        multi.sharded_init(s)
        multi.sharded_sweeps(s, 6)
    with pytest.raises(RuntimeError):
        multi.sharded_sweeps(s, 1)                      # called outside the chain's stream
    b, l, t = s.get_draws()
    assert np.array_equal(b, b0) and np.array_equal(l, l0) and np.array_equal(t, t0)
    with pytest.raises(hsp.HspError):
        s.sweep_end()                                   # out of order
    s.close()


@pytest.mark.parametrize("name,n_rows,p,tol", [("C2", 20011, 100, 1e-9), ("C3", 20003, 1000, 1e-4), ("C1", 1000, 10, 1e-9)])
def test_two_shards_match_the_oracle_on_the_whole_data(name, n_rows, p, tol):
    wl = hsp_synth.make(name, "cuda", n_rows=n_rows, p=p)
    Xh, yh = wl.host()
    X64 = wl.X.double()
    o = oracle.OracleChain(Xh, yh, wl.seed, gram=(X64.T @ X64).cpu().numpy())
    cuts = [multi.shard_rows(wl.N, r, 2) for r in range(2)]
    assert cuts[0][0] == 0 and cuts[0][1] == cuts[1][0] and cuts[1][1] == wl.N
    chains = []
    for r0, r1 in cuts:
        c = hsp.HorseshoeProbit(wl.X[r0:r1], wl.y[r0:r1], wl.seed, row_offset=r0)
        c.set_flags(hsp.HSP_STORE_Z)
        chains.append(c)
    G = sum(c.gram_tensor() for c in chains)
    for c in chains:
        c.gram_tensor().copy_(G)
    n = 8
    for c in chains:
        c.sweep_prepare(n)
    for k in range(n):
        for c in chains:
            c.sweep_begin()
        g = sum(c.xtz_tensor() for c in chains)           # the all-reduce, emulated
        for c in chains:
            c.xtz_tensor().copy_(g)
        for c in chains:
            c.sweep_end()
    o.sweep(n)
    bo, lo, to = o.get_draws()
    zo, so = o.get_latent()
    draws = [c.get_draws() for c in chains]
    for a, b in zip(draws[0], draws[1]):
        assert np.array_equal(a, b)                       # every rank holds the same chain, bit for bit
    bg, lg, tg = draws[0]
    worst = dict(beta=max(mixed_err(bg[k], bo[k]) for k in range(n)), lam=max(mixed_err(np.log(lg[k]), np.log(lo[k])) for k in range(n)),
                 tau=float(np.max(np.abs(tg / to - 1))))
    zs = np.concatenate([c.get_latent()[0] for c in chains])
    worst["z"] = mixed_err(zs, zo)
    print(name, "two shards vs oracle:", worst)
    assert all(v <= tol for v in worst.values()), worst
    for c in chains:
        c.close()
