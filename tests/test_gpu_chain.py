"""Chain-level behaviour of the CUDA path: determinism, execution modes, checkpoint/resume,
conditional laws and long-run agreement with the oracle."""
import numpy as np
import pytest
import torch

import hsp_synth
import oracle
import paper_1608_04329_b200 as hsp

pytestmark = pytest.mark.gpu


def batch_means_se(x, n_batches=40):
    n = (len(x) // n_batches) * n_batches
    b = np.asarray(x[:n]).reshape(n_batches, -1).mean(axis=1)
    return b.std(ddof=1) / np.sqrt(n_batches)


def _draws(wl, n, flags=0):
    g = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed)
    g.set_flags(flags)
    g.sweep(n)
    out = g.get_draws()
    k = g.launch_count()
    g.close()
    return out, k


def test_bitwise_reproducible_and_mode_independent():
    """Same seed, same inputs: graph replay, direct launches and the single-stream schedule give
    bit-identical draws (static tile->CTA map, fixed-order reductions, counter-based RNG)."""
    for wl in (hsp_synth.make("C1", "cuda"), hsp_synth.make("C3", "cuda", n_rows=9001)):
        (b0, l0, t0), k0 = _draws(wl, 12)
        for flags in (0, hsp.HSP_NO_GRAPH, hsp.HSP_SERIAL, hsp.HSP_NO_GRAPH | hsp.HSP_SERIAL):
            (b, l, t), k = _draws(wl, 12, flags)
            assert np.array_equal(b, b0) and np.array_equal(l, l0) and np.array_equal(t, t0), flags
            assert k == k0 and k > 12 * 5


def test_checkpoint_resume_is_exact():
    wl = hsp_synth.make("C2", "cuda", n_rows=5000)
    (b_ref, l_ref, t_ref), _ = _draws(wl, 20)
    g = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed)
    g.sweep(8)
    st = g.get_state()
    g.close()
    h = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed)
    h.set_state(**st)
    h.sweep(12)
    b, l, t = h.get_draws()
    assert np.array_equal(b, b_ref[8:]) and np.array_equal(l, l_ref[8:]) and np.array_equal(t, t_ref[8:])


def test_beta_conditional_law_on_gpu():
    """PAPER.md:180 with z, lambda, tau frozen: mean Q^-1 X^T z, covariance Q^-1 (reading R5)."""
    rng = np.random.default_rng(5)
    N, p, n = 64, 5, 40000
    e = rng.standard_normal((N, p)); Xn = np.empty_like(e); Xn[:, 0] = e[:, 0]
    for j in range(1, p):
        Xn[:, j] = 0.8 * Xn[:, j - 1] + 0.6 * e[:, j]
    X = torch.from_numpy(Xn).cuda(); y = torch.from_numpy((rng.random(N) < 0.5).astype(np.uint8)).cuda()
    g = hsp.HorseshoeProbit(X, y, 31)
    g.set_flags(hsp.HSP_STORE_Z)
    g.sweep(1)
    z, _ = g.get_latent()
    st = g.get_state()
    g.set_flags(hsp.HSP_STORE_Z | hsp.HSP_FREEZE_Z | hsp.HSP_FREEZE_SCALES)
    g.sweep(n)
    b, lam, tau = g.get_draws()
    assert np.allclose(lam, st["lam_inv2"] ** -0.5) and np.allclose(tau, st["tau_inv2"] ** -0.5)
    Q = Xn.T @ Xn + np.diag(st["tau_inv2"] * st["lam_inv2"])
    Sigma = np.linalg.inv(Q); mu = Sigma @ Xn.T @ z
    assert np.all(np.abs(b.mean(axis=0) - mu) < 4.5 * np.sqrt(np.diag(Sigma) / n))
    seC = np.sqrt((np.outer(np.diag(Sigma), np.diag(Sigma)) + Sigma ** 2) / n)
    assert np.all(np.abs(np.cov(b.T) - Sigma) < 4.5 * seC)


def test_long_run_posterior_matches_oracle_c1():
    """north_star: long-run posterior means and variances agree within 3 Monte-Carlo standard errors
    (the GPU chain uses a different seed here, so this is a test of the law, not of the coupling)."""
    wl = hsp_synth.make("C1", "cuda")
    Xh, yh = wl.host()
    o = oracle.OracleChain(Xh, yh, wl.seed); o.sweep(wl.n_sweeps)
    bo = o.get_draws()[0][500:]
    g = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed + 100); g.sweep(4 * wl.n_sweeps)
    bg = g.get_draws()[0][500:]
    for j in range(wl.p):
        se = np.hypot(batch_means_se(bo[:, j]), batch_means_se(bg[:, j]))
        assert abs(bo[:, j].mean() - bg[:, j].mean()) < 3.5 * se + 1e-3, j
        vo, vg = (bo[:, j] - bo[:, j].mean()) ** 2, (bg[:, j] - bg[:, j].mean()) ** 2
        assert abs(vo.mean() - vg.mean()) < 3.5 * np.hypot(batch_means_se(vo), batch_means_se(vg)) + 1e-4, j
    # planted truth recovered
    m = bg.mean(axis=0)
    assert np.all(np.abs(m[:3] - wl.beta_true[:3]) < 0.6) and np.all(np.abs(m[3:]) < 0.12)


def test_host_buffer_entry_point_matches_device_entry():
    wl = hsp_synth.make("C2", "cuda", n_rows=3000)
    (b0, l0, t0), _ = _draws(wl, 5)
    Xh = wl.X.cpu().pin_memory(); yh = wl.y.cpu().pin_memory()
    g = hsp.HorseshoeProbit(Xh, yh, wl.seed, host=True)
    g.sweep(5)
    b, l, t = g.get_draws()
    assert np.array_equal(b, b0) and np.array_equal(t, t0)
    out = (torch.empty((5, wl.p), dtype=torch.float64, device="cuda"), None, torch.empty(5, dtype=torch.float64, device="cuda"))
    g.get_draws(out)
    assert np.array_equal(out[0].cpu().numpy(), b0) and np.array_equal(out[2].cpu().numpy(), t0)


def test_non_finite_state_is_reported_not_crashed():
    """SURVEY.md 5 (failure detection): a non-finite chain state surfaces as HSP_ENUMERIC at the next synchronising call."""
    wl = hsp_synth.make("C2", "cuda", n_rows=3000)
    g = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed)
    g.sweep(2)
    g.get_draws()
    beta = np.zeros(wl.p); beta[3] = np.nan
    g.set_state(beta=beta)
    g.sweep(1)
    with pytest.raises(hsp.HspError) as ei:
        g.get_draws()
    assert ei.value.code == -5
    g.close()


def test_host_entry_with_chunked_upload_matches_device_entry():
    """hsp_create_host uploads X in row chunks on a copy stream while the Gram of the previous chunk runs (here 3
    chunks, tensor-core Gram): the chain must be bit-identical to the device-pointer entry."""
    wl = hsp_synth.make("C3", "cuda", n_rows=250_000, p=400)          # 400 MB of fp32 X
    (b0, l0, t0), _ = _draws(wl, 4)
    Xh = wl.X.cpu().pin_memory(); yh = wl.y.cpu().pin_memory()
    g = hsp.HorseshoeProbit(Xh, yh, wl.seed, host=True)
    g.sweep(4)
    b, l, t = g.get_draws()
    g.close()
    assert np.array_equal(b, b0) and np.array_equal(l, l0) and np.array_equal(t, t0)
    # pageable host memory takes the same path
    g = hsp.HorseshoeProbit(wl.X.cpu(), wl.y.cpu(), wl.seed, host=True)
    g.sweep(4)
    assert np.array_equal(g.get_draws()[0], b0)
    g.close()
