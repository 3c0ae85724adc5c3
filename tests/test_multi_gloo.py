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
