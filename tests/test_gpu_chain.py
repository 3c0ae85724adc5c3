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
    """north_star: long-run posterior means and variances agree within 3 Monte-Carlo standard errors (batch means,
    50 batches; the GPU chain uses a different seed, so this is a test of the law, not of the coupling).  The chains
    are longer than C1's 2000 sweeps so that the standard errors themselves are well estimated: the second moments of
    the shrunk null coefficients are heavy-tailed."""
    wl = hsp_synth.make("C1", "cuda")
    Xh, yh = wl.host()
    burn = 1000
    o = oracle.OracleChain(Xh, yh, wl.seed); o.sweep(3 * wl.n_sweeps + burn)
    bo = o.get_draws()[0][burn:]
    g = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed + 100); g.sweep(30 * wl.n_sweeps + burn)
    bg = g.get_draws()[0][burn:]
    worst = 0.0
    for j in range(wl.p):
        se = np.hypot(batch_means_se(bo[:, j], 50), batch_means_se(bg[:, j], 50))
        dm = abs(bo[:, j].mean() - bg[:, j].mean()) / se
        vo, vg = (bo[:, j] - bo[:, j].mean()) ** 2, (bg[:, j] - bg[:, j].mean()) ** 2
        dv = abs(vo.mean() - vg.mean()) / np.hypot(batch_means_se(vo, 50), batch_means_se(vg, 50))
        worst = max(worst, dm, dv)
        assert dm < 3.0 and dv < 3.0, (j, dm, dv)
    print("long run C1: worst |difference| / MCSE over", 2 * wl.p, "statistics:", worst)
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


@pytest.mark.parametrize("name,n_rows,p,flags", [("C3", 9001, 1000, 0), ("C3", 9001, 1000, hsp.HSP_NO_GRAPH), ("C1", 1000, 10, 0),
                                                 ("C2", 20011, 100, hsp.HSP_SERIAL)])
def test_async_output_ring_matches_synchronous_draws(name, n_rows, p, flags):
    """hsp_set_output (the Monte Carlo output is downloaded while the next updates are computed): the
    draws that land in the pinned host ring are bit-identical to hsp_get_draws of a chain run synchronously."""
    wl = hsp_synth.make(name, "cuda", n_rows=n_rows, p=p)
    n1, n2 = 10, 13
    (b_ref, l_ref, t_ref), _ = _draws(wl, n1 + n2, flags)
    g = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed)
    g.set_flags(flags)
    n = n1 + n2
    hb = torch.zeros((n, p), dtype=torch.float64).pin_memory()
    hl = torch.zeros((n, p), dtype=torch.float64).pin_memory()
    ht = torch.zeros(n, dtype=torch.float64).pin_memory()
    g.set_output(hb, hl, ht, n)
    g.sweep(n1)
    g.sweep(n2)                                        # the second call may not overtake the download of the first
    r0 = g.output_ready()
    assert 0 <= r0 <= n
    assert g.output_wait() == n and g.output_ready() == n
    assert np.array_equal(hb.numpy(), b_ref) and np.array_equal(hl.numpy(), l_ref) and np.array_equal(ht.numpy(), t_ref)
    # hsp_get_draws still returns the draws of the last call
    b2, _, t2 = g.get_draws()
    assert np.array_equal(b2, b_ref[n1:]) and np.array_equal(t2, t_ref[n1:])
    # a ring smaller than the run keeps the most recent `cap` sweeps at row (r mod cap); beta only
    cap = 8
    rb = torch.zeros((cap, p), dtype=torch.float64).pin_memory()
    g.set_output(rb, None, None, cap)
    g.sweep(21)
    assert g.output_wait() == 21
    b3 = g.get_draws()[0]
    for r in range(21 - cap, 21):
        assert np.array_equal(rb.numpy()[r % cap], b3[r]), r
    # switched off: nothing more is written
    g.set_output(None, None, None, 0)
    keep = rb.clone()
    g.sweep(3)
    g.sync()
    assert g.output_wait() == 0 and torch.equal(rb, keep)
    g.close()


def test_async_output_with_sharded_begin_end():
    wl = hsp_synth.make("C3", "cuda", n_rows=9001)
    (b_ref, l_ref, t_ref), _ = _draws(wl, 7)
    g = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed, row_offset=0)
    hb = torch.zeros((7, wl.p), dtype=torch.float64).pin_memory()
    ht = torch.zeros(7, dtype=torch.float64).pin_memory()
    g.set_output(hb, None, ht, 7)
    g.sweep_prepare(7)
    for _ in range(7):
        g.sweep_begin(); g.sweep_end()
    assert g.output_wait() == 7
    assert np.array_equal(hb.numpy(), b_ref) and np.array_equal(ht.numpy(), t_ref)
    g.close()


def test_options_are_plan_time_and_process_wide(hsp_options):
    """hsp_set_option: no environment variables; plan-time keys are refused on an existing chain."""
    wl = hsp_synth.make("C3", "cuda", n_rows=9001)
    (b_ref, _, _), _ = _draws(wl, 4)
    hsp_options("fused_variant", 0)
    assert hsp.get_option("fused_variant") == 0
    g = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed)
    assert g.fused_variant() == "generic"
    with pytest.raises(hsp.HspError):
        g.set_option("fused_variant", 1)
    with pytest.raises(hsp.HspError):
        hsp.set_option("no_such_key", 1)
    g.set_option("no_pdl", 1)                          # launch mode: allowed, rebuilds the graph
    g.sweep(4)
    b = g.get_draws()[0]
    g.close()
    hsp.reset_options()
    assert hsp.get_option("fused_variant") == -1
    # generic kernel (exact fp64 eta) vs the TMA kernel (fp32 chains): same chain within the fp32-X tolerance
    assert np.max(np.abs(b - b_ref)) < 1e-4 * max(1.0, np.max(np.abs(b_ref)))


def test_reserve_history_changes_nothing_but_the_allocation_time():
    """hsp_reserve_history: the same draws with and without it; a later, longer call still grows the history."""
    wl = hsp_synth.make("C2", "cuda", n_rows=4000)
    (b_ref, l_ref, t_ref), _ = _draws(wl, 9)
    g = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed)
    g.reserve_history(64)
    g.sweep(4)
    g.reserve_history(8)                      # smaller than the capacity: nothing happens, the draws stay
    b, l, t = g.get_draws()
    assert np.array_equal(b, b_ref[:4]) and np.array_equal(t, t_ref[:4])
    g.sweep(5)
    b, l, t = g.get_draws()
    assert np.array_equal(b, b_ref[4:]) and np.array_equal(l, l_ref[4:]) and np.array_equal(t, t_ref[4:])
    g.sweep(100)                              # beyond the reservation: grows on demand
    assert g.get_draws()[0].shape == (100, wl.p)
    with pytest.raises(hsp.HspError):
        g.reserve_history(-1)
    g.close()
