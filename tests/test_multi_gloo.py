"""N > 1 path on CPU: world_size-2 gloo.  The multi-GPU design is one independent chain per rank (seed + rank,
no data-path collective); what crosses ranks is the timing reduction and the gather of
draws for cross-chain diagnostics.  The chains here are oracle chains (test infrastructure) standing in for the
CUDA chains, which need a GPU."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import hsp_synth
import oracle
from paper_1608_04329_b200 import multi


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, ws, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(ws))
    dist.init_process_group("gloo", rank=rank, world_size=ws)
    try:
        assert multi.world() == (rank, ws)
        wl = hsp_synth.make("C1", "cpu")
        Xh, yh = wl.host()
        seed = multi.chain_seed(wl.seed, rank)
        ch = oracle.OracleChain(Xh, yh, seed)
        ch.sweep(600)
        beta = torch.from_numpy(ch.get_draws()[0][200:].copy())
        allb = multi.gather_draws(beta)
        assert allb.shape == (ws, 400, wl.p)
        assert torch.equal(allb[rank], beta)
        ms = multi.max_over_ranks(10.0 * (rank + 1))
        assert ms == 10.0 * ws
        rate = multi.whole_job_rate(400, ms)
        assert abs(rate - ws * 400 / (ms * 1e-3)) < 1e-9
        rhat = multi.split_rhat(allb)
        torch.save({"allb": allb, "rhat": rhat, "seed": seed}, os.path.join(out_dir, f"r{rank}.pt"))
    finally:
        dist.destroy_process_group()


def test_two_ranks_independent_chains_gather_and_timing(tmp_path):
    ws, port = 2, _free_port()
    mp.spawn(_worker, args=(ws, port, str(tmp_path)), nprocs=ws, join=True)
    r0 = torch.load(tmp_path / "r0.pt")
    r1 = torch.load(tmp_path / "r1.pt")
    assert r0["seed"] + 1 == r1["seed"]
    assert torch.equal(r0["allb"], r1["allb"])                      # every rank sees every chain
    assert not torch.equal(r0["allb"][0], r0["allb"][1])            # the chains differ (different Philox keys)
    # both chains sample the same posterior: split-R-hat near 1 on the planted coordinates
    assert torch.all(r0["rhat"][:3] < 1.2), r0["rhat"]
    m = r0["allb"].mean(dim=(0, 1)).numpy()
    assert np.all(np.abs(m[3:]) < 0.15) and np.all(np.abs(m[:3]) > 0.4)


def test_split_rhat_detects_disagreeing_chains():
    g = torch.Generator().manual_seed(0)
    a = torch.randn((2, 500, 3), generator=g, dtype=torch.float64)
    assert torch.all(multi.split_rhat(a) < 1.05)
    a[1, :, 0] += 3.0
    r = multi.split_rhat(a)
    assert r[0] > 1.5 and torch.all(r[1:] < 1.05)


def test_single_process_defaults():
    assert multi.world() == (0, 1)
    assert multi.max_over_ranks(3.5) == 3.5
    assert multi.gather_draws(torch.zeros(4, 2)).shape == (1, 4, 2)
    assert multi.chain_seed(2 ** 64 - 1, 1) == 0


# ---- row-sharded chain: the driver loop of multi.py over gloo, with an oracle-backed stand-in for the CUDA chain
class _OracleShard:
    """Same interface as HorseshoeProbit(row_offset=...) for multi.sharded_init / sharded_sweeps, built from the
    oracle's per-element functions on this rank's rows (global row index in the Philox counter)."""

    def __init__(self, X, y, seed, row_offset):
        self.X, self.y, self.seed, self.r0 = X, y, seed, row_offset
        self.N, self.p = X.shape
        self.G = torch.from_numpy(X.T @ X)
        self.g = torch.zeros(self.p, dtype=torch.float64)
        self.scales = oracle.OracleChain(np.zeros((4, self.p)), np.zeros(4, dtype=np.uint8), seed, gram=np.zeros((self.p, self.p)))
        self.scales.set_flags(oracle.FREEZE_Z | oracle.FREEZE_BETA)
        self.beta = np.zeros(self.p)
        self.k = 0
        self.hist = []

    def gram_tensor(self):
        return self.G

    def xtz_tensor(self):
        return self.g

    def sweep_prepare(self, n):
        self.hist = []

    def sweep_begin(self):
        self.k += 1
        side = 2.0 * self.y - 1.0
        idx = np.arange(self.r0, self.r0 + self.N, dtype=np.uint64)
        u = np.asarray(oracle.uniforms_many(self.seed, idx, self.k, 0)[0])
        z = side * np.asarray(oracle.tnpos_many(side * (self.X @ self.beta), u))
        self.g.copy_(torch.from_numpy(self.X.T @ z))
        self.scales.set_state(beta=self.beta, sweep=self.k - 1)
        self.scales.sweep(1)

    def sweep_end(self):
        st = self.scales.get_state()
        rc, L = oracle.cholesky_lower(self.G.numpy() + np.diag(st["tau_inv2"] * st["lam_inv2"]))
        assert rc == 0
        e = np.asarray(oracle.norm_inv_many(np.asarray(oracle.uniforms_many(self.seed, np.arange(self.p, dtype=np.uint64), self.k, 3)[0])))
        self.beta = oracle.solve_lower(L, oracle.solve_lower(L, self.g.numpy()) + e, transpose=True)
        self.hist.append(self.beta.copy())


def _shard_worker(rank, ws, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(ws))
    dist.init_process_group("gloo", rank=rank, world_size=ws)
    try:
        wl = hsp_synth.make("C2", "cpu", n_rows=3001, p=12)
        Xh, yh = wl.host()
        r0, r1 = multi.shard_rows(wl.N, rank, ws)
        ch = _OracleShard(Xh[r0:r1], yh[r0:r1].astype(np.float64), wl.seed, r0)
        multi.sharded_init(ch)
        multi.sharded_sweeps(ch, 5)
        torch.save({"beta": np.array(ch.hist), "rows": (r0, r1)}, os.path.join(out_dir, f"s{rank}.pt"))
    finally:
        dist.destroy_process_group()


def test_row_sharded_chain_over_gloo_matches_the_whole_data_oracle(tmp_path):
    ws, port = 2, _free_port()
    mp.spawn(_shard_worker, args=(ws, port, str(tmp_path)), nprocs=ws, join=True)
    s0 = torch.load(tmp_path / "s0.pt", weights_only=False)
    s1 = torch.load(tmp_path / "s1.pt", weights_only=False)
    assert s0["rows"][1] == s1["rows"][0] and s0["rows"][0] == 0 and s1["rows"][1] == 3001
    assert np.array_equal(s0["beta"], s1["beta"])           # every rank draws the same beta
    wl = hsp_synth.make("C2", "cpu", n_rows=3001, p=12)
    Xh, yh = wl.host()
    o = oracle.OracleChain(Xh, yh, wl.seed)
    o.sweep(5)
    assert np.max(np.abs(s0["beta"] - o.get_draws()[0])) < 1e-10   # = the chain on the whole data (summation order only)


def test_shard_rows_partition():
    for N, ws in [(10, 3), (7, 7), (1000001, 8), (5, 8)]:
        cuts = [multi.shard_rows(N, r, ws) for r in range(ws)]
        assert cuts[0][0] == 0 and cuts[-1][1] == N
        assert all(a[1] == b[0] for a, b in zip(cuts, cuts[1:]))
        sizes = [b - a for a, b in cuts]
        assert max(sizes) - min(sizes) <= 1
