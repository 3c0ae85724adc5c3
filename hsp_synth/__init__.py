"""Seeded synthetic inputs shaped like the paper's workloads (eq. 13) and the five
BASELINE.json configs.  This module serves BOTH the CUDA path's tests/bench and the oracle's
tests; it holds none of the method's arithmetic (no sampler, no Philox, no Cholesky): it only
draws a design matrix, a planted sparse beta and probit responses with torch's own generators.

The same arrays are handed to both paths, so data generation is outside the parity contract.
Data seed = sampler seed + 1000.
"""
from dataclasses import dataclass

import numpy as np
import torch

_CHUNK = 65536  # rows generated per generator call: fixes the stream for a given device


@dataclass
class Workload:
    name: str
    X: torch.Tensor          # N x p, row-major, float32 or float64, on `device`
    y: torch.Tensor          # N, uint8 in {0,1}, on `device`
    beta_true: np.ndarray    # p, float64
    seed: int                # sampler (Philox) seed
    n_sweeps: int            # sweeps BASELINE.json quotes for this config
    positive_rate: float

    @property
    def N(self):
        return self.X.shape[0]

    @property
    def p(self):
        return self.X.shape[1]

    def host(self):
        """(X, y) as contiguous numpy arrays (what the oracle consumes)."""
        return self.X.cpu().numpy(), self.y.cpu().numpy()


CONFIGS = {
    # name: N, p, dtype, sampler seed, sweeps
    "C1": dict(N=1_000, p=10, dtype=torch.float64, seed=1, sweeps=2000),
    "C2": dict(N=100_000, p=100, dtype=torch.float64, seed=2, sweeps=1000),
    "C3": dict(N=1_000_000, p=1000, dtype=torch.float32, seed=3, sweeps=1000),
    "C4": dict(N=250_000, p=4000, dtype=torch.float32, seed=4, sweeps=500),
    "C5": dict(N=2_000_000, p=2000, dtype=torch.float32, seed=5, sweeps=300),
    "C5b": dict(N=2_000_000, p=2000, dtype=torch.float32, seed=5, sweeps=300),
    # stand-in for the SHAPE of the paper's real-data run (N = 1,295,848, p = 141, ybar = 0.0048;
    # the clinical data itself is not available): iid N(0,1) columns + intercept, rare positives
    "R1": dict(N=1_295_848, p=141, dtype=torch.float32, seed=6, sweeps=1000),
}


def _planted_beta(name, p, rng):
    beta = np.zeros(p)
    if name == "C1":
        beta[:3] = [2.0, -1.5, 1.0]
        return beta
    nnz, lo, hi, first = {"C2": (10, 0.5, 2.0, 0), "C3": (20, 0.5, 2.0, 0), "C4": (40, 0.25, 1.5, 1),
                          "C5": (50, 0.5, 2.0, 1), "C5b": (50, 0.5, 2.0, 1), "R1": (10, 0.2, 0.6, 1)}[name]
    nnz = min(nnz, p - first)
    idx = first + rng.choice(p - first, size=nnz, replace=False)
    beta[idx] = rng.uniform(lo, hi, size=nnz) * rng.choice([-1.0, 1.0], size=nnz)
    if name == "C5":
        beta[0] = -2.0           # literal BASELINE.json reading (R15)
    if name == "R1":
        beta[0] = -2.59 * np.sqrt(1.0 + float(np.sum(beta ** 2)))    # Phi(-2.59) = 0.0048
    if name == "C5b":
        beta[0] = -1.645 * np.sqrt(1.0 + float(np.sum(beta ** 2)))   # gives ~5 % positives
    return beta


def make(name, device="cpu", n_rows=None, p=None):
    """Generate config `name` (optionally with fewer rows / columns, same recipe) on `device`."""
    cfg = CONFIGS[name]
    N = int(n_rows) if n_rows is not None else cfg["N"]
    p = int(p) if p is not None else cfg["p"]
    dtype = cfg["dtype"]
    data_seed = cfg["seed"] + 1000
    rng = np.random.default_rng(data_seed)
    beta_true = _planted_beta(name, p, rng)
    dev = torch.device(device)
    gen = torch.Generator(device=dev)
    gen.manual_seed(data_seed)
    X = torch.empty((N, p), dtype=dtype, device=dev)
    y = torch.empty(N, dtype=torch.uint8, device=dev)
    bt = torch.from_numpy(beta_true).to(dev)
    chunk = max(1, min(_CHUNK, (1 << 28) // max(p, 1)))
    for r0 in range(0, N, chunk):
        r1 = min(N, r0 + chunk)
        blk = torch.randn((r1 - r0, p), dtype=dtype, device=dev, generator=gen)
        if name == "C4":
            # column 0 = intercept of ones; columns 1.. are AR(1): Sigma_jk = 0.5^|j-k|
            e = blk
            blk = torch.empty_like(e)
            blk[:, 0] = 1.0
            if p > 1:
                blk[:, 1] = e[:, 1]
            s = 0.75 ** 0.5
            for j in range(2, p):
                blk[:, j] = 0.5 * blk[:, j - 1] + s * e[:, j]
        elif name in ("C5", "C5b", "R1"):
            blk[:, 0] = 1.0
        X[r0:r1] = blk
        eps = torch.randn(r1 - r0, dtype=torch.float64, device=dev, generator=gen)
        y[r0:r1] = ((blk.double() @ bt + eps) > 0).to(torch.uint8)
    rate = float(y.double().mean().item())
    return Workload(name=name, X=X, y=y, beta_true=beta_true, seed=cfg["seed"], n_sweeps=cfg["sweeps"],
                    positive_rate=rate)
