"""Parity at BASELINE.json's FULL sizes (C3, C4, C5) in the launch configuration bench.py times (direct
launches on two streams; the only difference is HSP_STORE_Z so that z can be read back).

One whole sweep is checked against the oracle's definitions evaluated at full size:
  a1  eta = X beta               fp64 library matrix-vector product on the host (chunked)
  a2  z_i = s_i TNpos(s_i eta_i, U_A(i, k, Z))   oracle.uniforms_many / oracle.tnpos_many, every row
  a3+b g = X^T z                 fp64 library product on the host from the ORACLE's z
  e1-e3 scale conditionals       the oracle chain itself (its scale step does not touch X)
  c0 G = X^T X                   fp64 library product (the tensor-core Gram is within 1e-6 of it)
  c, d1, d2  Q = G + diag, L, beta   oracle.cholesky_lower / solve_lower (numpy.linalg.cholesky for p = 4000)
No expected value comes from the CUDA path: the oracle side starts from the chain state read BEFORE the sweep.
Tolerances: north_star's 1e-4 for fp32 X in the mixed metric of DESIGN.md R12 (observed values are printed);
the truncation side is bit-exact for every row.
"""
import numpy as np
import pytest
import torch

import hsp_synth
import oracle
import paper_1608_04329_b200 as hsp
from conftest import mixed_err

pytestmark = pytest.mark.gpu

CHUNK = 1 << 16


def host_matvec(X, b):
    """eta = X b in fp64, X a (possibly fp32) CUDA tensor, evaluated on the host in row chunks."""
    out = np.empty(X.shape[0])
    for r in range(0, X.shape[0], CHUNK):
        out[r:r + CHUNK] = X[r:r + CHUNK].cpu().numpy().astype(np.float64) @ b
    return out


def host_rmatvec(X, z):
    g = np.zeros(X.shape[1])
    for r in range(0, X.shape[0], CHUNK):
        g += X[r:r + CHUNK].cpu().numpy().astype(np.float64).T @ z[r:r + CHUNK]
    return g


def gram_fp64(X):
    G = torch.zeros((X.shape[1], X.shape[1]), dtype=torch.float64, device=X.device)
    for r in range(0, X.shape[0], 4 * CHUNK):
        Xc = X[r:r + 4 * CHUNK].double()
        G += Xc.T @ Xc
    return G.cpu().numpy()


@pytest.mark.parametrize("name,warm", [("C3", 3), ("C4", 2), ("C5", 2), ("R1", 12)])
def test_full_size_sweep_against_oracle(name, warm):
    wl = hsp_synth.make(name, "cuda")
    N, p, seed = wl.N, wl.p, wl.seed
    g = hsp.HorseshoeProbit(wl.X, wl.y, seed)
    g.set_flags(hsp.HSP_NO_GRAPH | hsp.HSP_STORE_Z)
    g.sweep(warm)
    st0 = g.get_state()
    k = st0["sweep"] + 1
    g.sweep(1)
    zg, sg = g.get_latent()
    bg, lg, tg = g.get_draws()
    st1 = g.get_state()
    xtz_g = g.get_xtz()
    plan = g.plan()
    variant = g.fused_variant()
    Gg = g.get_gram()
    g.close()
    assert variant == ("tma-narrow" if name == "R1" else "tma")

    # ---- a1, a2: every row
    y = wl.y.cpu().numpy()
    side = (2 * y.astype(np.int8) - 1).astype(np.int8)
    assert np.array_equal(sg, side)                                     # bit-exact
    assert np.all(np.isfinite(zg)) and np.all(zg * side > 0)
    eta = host_matvec(wl.X, st0["beta"])
    u = np.asarray(oracle.uniforms_many(seed, np.arange(N, dtype=np.uint64), k, 0)[0])
    z_ref = side * np.asarray(oracle.tnpos_many(side * eta, u))
    ez = mixed_err(zg, z_ref)
    # ---- a3 + b
    g_ref = host_rmatvec(wl.X, z_ref)
    eg = mixed_err(xtz_g, g_ref)

    # ---- e1, e2, e3: the oracle chain's own scale step (X is not involved: a 4-row stand-in design)
    o = oracle.OracleChain(np.zeros((4, p)), np.zeros(4, dtype=np.uint8), seed, gram=np.zeros((p, p)))
    o.set_flags(oracle.FREEZE_Z | oracle.FREEZE_BETA)
    o.set_state(beta=st0["beta"], lam_inv2=st0["lam_inv2"], nu_inv=st0["nu_inv"], tau_inv2=st0["tau_inv2"],
                xi_inv=st0["xi_inv"], sweep=st0["sweep"])
    o.sweep(1)
    so = o.get_state()
    e_lam = float(np.max(np.abs(st1["lam_inv2"] / so["lam_inv2"] - 1)))
    e_nu = float(np.max(np.abs(st1["nu_inv"] / so["nu_inv"] - 1)))
    e_tau = abs(st1["tau_inv2"] / so["tau_inv2"] - 1)
    e_xi = abs(st1["xi_inv"] / so["xi_inv"] - 1)
    assert np.allclose(lg[0], so["lam_inv2"] ** -0.5, rtol=1e-12) and np.isclose(tg[0], so["tau_inv2"] ** -0.5, rtol=1e-12)

    # ---- c0, c, d1, d2
    G_ref = gram_fp64(wl.X)
    e_gram = float(np.max(np.abs(np.tril(Gg) - np.tril(G_ref))) / np.max(np.abs(G_ref)))
    Q = G_ref + np.diag(so["tau_inv2"] * so["lam_inv2"])
    if p > 2000:
        L = np.linalg.cholesky(Q)
    else:
        rc, L = oracle.cholesky_lower(Q)
        assert rc == 0
    e = np.asarray(oracle.norm_inv_many(np.asarray(oracle.uniforms_many(seed, np.arange(p, dtype=np.uint64), k, 3)[0])))
    if p > 2000:
        import scipy.linalg as sl
        v = sl.solve_triangular(L, g_ref, lower=True) + e
        beta_ref = sl.solve_triangular(L.T, v, lower=False)
    else:
        v = oracle.solve_lower(L, g_ref) + e
        beta_ref = oracle.solve_lower(L, v, transpose=True)
    eb = mixed_err(bg[0], beta_ref)
    assert np.array_equal(bg[0], st1["beta"])

    print(f"{name} full size N={N} p={p} sweep {k} plan {plan}: z {ez:.3e}  X^Tz {eg:.3e}  beta {eb:.3e}  gram {e_gram:.3e}  "
          f"lam {e_lam:.3e} nu {e_nu:.3e} tau {e_tau:.3e} xi {e_xi:.3e}")
    assert ez <= 1e-4 and eg <= 1e-4 and eb <= 1e-4
    # C3-C5 are above the size where create uses the tensor-core Gram (fp32 X, N p^2 >= 2e10): split-bf16 products with
    # a truncating fp32 TMEM accumulation over <= 128 rows -> relative bias ~2e-7; exact DFMA path: 1e-13
    assert e_gram <= 1e-6
    assert max(e_lam, e_nu, e_tau, e_xi) <= 1e-9
