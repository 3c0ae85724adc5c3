"""Pins for the oracle's sweep as a whole: indexing, schedule, and the conditionals as a system,
against what PAPER.md and the mathematics fix (no value here comes from the CUDA path)."""
import numpy as np
import pytest
from scipy import stats

import hsp_synth
import oracle


def batch_means_se(x, n_batches=40):
    x = np.asarray(x, dtype=np.float64)
    n = (len(x) // n_batches) * n_batches
    b = x[:n].reshape(n_batches, -1).mean(axis=1)
    return b.std(ddof=1) / np.sqrt(n_batches)


def ar1_design(N, p, rho, rng):
    e = rng.standard_normal((N, p))
    X = np.empty_like(e)
    X[:, 0] = e[:, 0]
    for j in range(1, p):
        X[:, j] = rho * X[:, j - 1] + np.sqrt(1 - rho * rho) * e[:, j]
    return X


def test_cold_start_and_first_sweep_schedule():
    """PAPER.md:289 cold start; PAPER.md:188-189 order: lam^-2 and tau^-2 are drawn from the OLD
    beta (=0), nu^-1 and xi^-1 from the NEW lam^-2, tau^-2."""
    rng = np.random.default_rng(3)
    N, p, seed = 40, 5, 123
    X = rng.standard_normal((N, p))
    y = (rng.random(N) < 0.5).astype(np.uint8)
    ch = oracle.OracleChain(X, y, seed)
    st = ch.get_state()
    assert np.all(st["beta"] == 0) and np.all(st["lam_inv2"] == 1) and np.all(st["nu_inv"] == 1)
    assert st["tau_inv2"] == 1 and st["xi_inv"] == 1 and st["sweep"] == 0
    ch.sweep(1)
    st = ch.get_state()
    z, side = ch.get_latent()
    assert np.array_equal(side, 2 * y.astype(np.int8) - 1)
    assert np.all(z * side > 0)
    # eta = 0 on the first sweep: z_i = s_i * TNpos(0, u_i), TNpos(0,u) = Q^-1(u/2)
    for i in range(N):
        u = oracle.uniforms(seed, i, 1, oracle.TAG_Z)[0]
        assert abs(z[i] - side[i] * stats.norm.isf(u / 2)) < 1e-12
    for j in range(p):
        u = oracle.uniforms(seed, j, 1, oracle.TAG_LAMBDA)[0]
        assert np.isclose(st["lam_inv2"][j], -np.log(u) / 1.0, rtol=1e-14)          # nu=1, beta=0
        un = oracle.uniforms(seed, j, 1, oracle.TAG_NU)[0]
        assert np.isclose(st["nu_inv"][j], -np.log(un) / (1 + st["lam_inv2"][j]), rtol=1e-14)
    gam, _ = oracle.cheng_gamma((p + 1) / 2, seed, 1)
    assert np.isclose(st["tau_inv2"], gam / 1.0, rtol=1e-14)                         # xi=1, S=0
    ux = oracle.uniforms(seed, 0, 1, oracle.TAG_XI)[0]
    assert np.isclose(st["xi_inv"], -np.log(ux) / (1 + st["tau_inv2"]), rtol=1e-14)
    # beta = Q^-1 g + L^-T e with the NEW scales
    g = X.T @ z
    assert np.allclose(ch.get_xtz(), g, rtol=1e-13, atol=1e-13)
    Q = X.T @ X + np.diag(st["tau_inv2"] * st["lam_inv2"])
    L = np.linalg.cholesky(Q)
    e = np.array([stats.norm.ppf(oracle.uniforms(seed, j, 1, oracle.TAG_E)[0]) for j in range(p)])
    beta = np.linalg.solve(Q, g) + np.linalg.solve(L.T, e)
    assert np.allclose(st["beta"], beta, rtol=1e-10, atol=1e-12)
    b, lam, tau = ch.get_draws()
    assert np.array_equal(b[0], st["beta"])
    assert np.allclose(lam[0], st["lam_inv2"] ** -0.5) and np.isclose(tau[0], st["tau_inv2"] ** -0.5)


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_eta_and_xtz_indexing_against_numpy(dtype):
    rng = np.random.default_rng(4)
    N, p = 57, 6
    X = rng.standard_normal((N, p)).astype(dtype)
    y = (rng.random(N) < 0.4).astype(np.uint8)
    ch = oracle.OracleChain(X, y, 9)
    assert np.allclose(np.tril(ch.get_gram()), np.tril(X.astype(np.float64).T @ X.astype(np.float64)), rtol=1e-13)
    beta = rng.standard_normal(p)
    ch.set_state(beta=beta)
    ch.sweep(1)
    eta = X.astype(np.float64) @ beta
    assert np.allclose(ch.get_eta(), eta, rtol=1e-13, atol=1e-13)
    z, side = ch.get_latent()
    u = np.array([oracle.uniforms(9, i, 1, oracle.TAG_Z)[0] for i in range(N)])
    assert np.allclose(z, side * oracle.tnpos_many(side * eta, u), rtol=1e-13)
    assert np.allclose(ch.get_xtz(), X.astype(np.float64).T @ z, rtol=1e-12, atol=1e-12)


def test_beta_conditional_mean_and_covariance():
    """north_star check 2 / PAPER.md:180: with z, lambda, tau held fixed, beta ~ N(Q^-1 X^T z, Q^-1).
    An AR(1) design makes Q^-1 = L^-T L^-1 differ from (L^T L)^-1, so the transpose reading R5
     is detectable."""
    rng = np.random.default_rng(5)
    N, p, n = 30, 4, 100000
    X = ar1_design(N, p, 0.8, rng)
    y = (rng.random(N) < 0.5).astype(np.uint8)
    ch = oracle.OracleChain(X, y, 31)
    z = rng.standard_normal(N) * 2
    lam_inv2 = np.array([0.3, 2.0, 5.0, 0.7]); tau_inv2 = 1.7
    ch.set_state(lam_inv2=lam_inv2, tau_inv2=tau_inv2)
    ch.set_latent(z)
    ch.set_flags(oracle.FREEZE_Z | oracle.FREEZE_SCALES)
    ch.sweep(n)
    b, _, _ = ch.get_draws()
    Q = X.T @ X + np.diag(tau_inv2 * lam_inv2)
    Sigma = np.linalg.inv(Q)
    mu = Sigma @ X.T @ z
    se = np.sqrt(np.diag(Sigma) / n)
    assert np.all(np.abs(b.mean(axis=0) - mu) < 4.5 * se)
    C = np.cov(b.T)
    # standard error of a sample covariance entry of a Gaussian: sqrt((S_ii S_jj + S_ij^2)/n)
    seC = np.sqrt((np.outer(np.diag(Sigma), np.diag(Sigma)) + Sigma ** 2) / n)
    assert np.all(np.abs(C - Sigma) < 4.5 * seC)
    L = np.linalg.cholesky(Q)
    wrong = np.linalg.inv(L.T @ L)                     # covariance of the literal L^-1 s reading
    assert np.max(np.abs(wrong - Sigma) / seC) > 20    # the test can tell them apart


def _theta_grid(n):
    t = (np.arange(n) + 0.5) / n * (np.pi / 2)         # scale = tan(theta): C+(0,1) is uniform in theta
    return np.tan(t)


def test_scale_conditionals_match_quadrature_p1_and_p2():
    """north_star check 3: (lam^-2, nu^-1, tau^-2, xi^-1 | beta) must target
    prod_j N(beta_j; 0, lam_j^2 tau^2) C+(lam_j) C+(tau).  Exposes reading R1 (Gamma vs IG)."""
    for beta in (np.array([0.8]), np.array([1.5, -0.1])):
        p = beta.size
        rng = np.random.default_rng(6)
        X = rng.standard_normal((5, p)); y = np.array([0, 1, 0, 1, 1], dtype=np.uint8)
        ch = oracle.OracleChain(X, y, 41 + p)
        ch.set_state(beta=beta)
        ch.set_flags(oracle.FREEZE_Z | oracle.FREEZE_BETA)
        n = 200000
        ch.sweep(n)
        _, lam, tau = ch.get_draws()
        lam, tau = lam[2000:], tau[2000:]
        f_tau = 1 / (1 + tau ** 2)
        f_l0 = 1 / (1 + lam[:, 0] ** 2)
        # brute force over (lam_1..lam_p, tau) on a tan-grid
        G = 300 if p == 1 else 140
        s = _theta_grid(G)
        if p == 1:
            L0, T = np.meshgrid(s, s, indexing="ij")
            dens = stats.norm.pdf(beta[0], scale=L0 * T)
        else:
            L0, L1, T = np.meshgrid(s, s, s, indexing="ij")
            dens = stats.norm.pdf(beta[0], scale=L0 * T) * stats.norm.pdf(beta[1], scale=L1 * T)
        Zc = dens.sum()
        q_tau = (dens / (1 + T ** 2)).sum() / Zc
        q_l0 = (dens / (1 + L0 ** 2)).sum() / Zc
        assert abs(f_tau.mean() - q_tau) < 4 * batch_means_se(f_tau) + 2e-3, (p, f_tau.mean(), q_tau)
        assert abs(f_l0.mean() - q_l0) < 4 * batch_means_se(f_l0) + 2e-3, (p, f_l0.mean(), q_l0)


def test_whole_chain_p1_matches_3d_quadrature():
    """p=1, N=20: posterior mean/variance of beta from
    prod_i Phi(s_i x_i beta) N(beta; 0, lam^2 tau^2) C+(lam) C+(tau)  (eq. 9-10)."""
    rng = np.random.default_rng(7)
    N = 20
    X = rng.standard_normal((N, 1))
    y = ((X[:, 0] * 0.9 + rng.standard_normal(N)) > 0).astype(np.uint8)
    ch = oracle.OracleChain(X, y, 51)
    n = 60000
    ch.sweep(n)
    b, _, _ = ch.get_draws()
    b = b[1000:, 0]
    bg = np.linspace(-3, 6, 1801)
    s = _theta_grid(200)
    loglik = np.sum(stats.norm.logcdf((2.0 * y - 1)[:, None] * X[:, 0][:, None] * bg[None, :]), axis=0)
    sc = (s[:, None] * s[None, :]).ravel()                       # lam*tau over the tan grid
    prior = stats.norm.pdf(bg[:, None], scale=sc[None, :]).mean(axis=1)
    post = np.exp(loglik) * prior
    post /= post.sum()
    qm = float((bg * post).sum()); qv = float((bg ** 2 * post).sum() - qm ** 2)
    assert abs(b.mean() - qm) < 4 * batch_means_se(b) + 5e-3, (b.mean(), qm)
    assert abs(b.var() - qv) < 4 * batch_means_se((b - b.mean()) ** 2) + 1e-2, (b.var(), qv)


def test_planted_beta_recovered_config_c1():
    """north_star check 4 / PAPER.md:289: nonzeros identified, irrelevant coefficients shrunk to 0."""
    wl = hsp_synth.make("C1")
    X, y = wl.host()
    ch = oracle.OracleChain(X, y, wl.seed)
    ch.sweep(wl.n_sweeps)
    b, lam, tau = ch.get_draws()
    m, sd = b[500:].mean(axis=0), b[500:].std(axis=0)
    assert np.all(np.abs(m[:3] - wl.beta_true[:3]) < 4 * sd[:3] + 0.1)
    assert np.all(np.sign(m[:3]) == np.sign(wl.beta_true[:3])) and np.all(np.abs(m[:3]) > 0.5)
    assert np.all(np.abs(m[3:]) < 0.12)
    assert np.all(np.isfinite(lam)) and np.all(tau > 0)


def test_inverse_cdf_and_paper_rejection_give_same_posterior():
    """O8: swapping the paper's rejection samplers for the inverse-CDF map keeps
    the target: posterior means/variances of beta agree within Monte-Carlo error."""
    rng = np.random.default_rng(8)
    N, p, n = 60, 3, 20000
    X = rng.standard_normal((N, p))
    y = ((X @ np.array([1.0, -0.5, 0.0]) + rng.standard_normal(N)) > 0).astype(np.uint8)
    a = oracle.OracleChain(X, y, 61)
    a.sweep(n)
    c = oracle.OracleChain(X, y, 62)
    c.set_flags(oracle.STORE_Z | oracle.LITERAL_Z)
    c.sweep(n)
    assert c.literal_trials() > N * n                      # the rejection loops really ran
    ba, bc = a.get_draws()[0][1000:], c.get_draws()[0][1000:]
    for j in range(p):
        se = np.hypot(batch_means_se(ba[:, j]), batch_means_se(bc[:, j]))
        assert abs(ba[:, j].mean() - bc[:, j].mean()) < 4 * se + 2e-3
        va, vc = (ba[:, j] - ba[:, j].mean()) ** 2, (bc[:, j] - bc[:, j].mean()) ** 2
        assert abs(va.mean() - vc.mean()) < 4 * np.hypot(batch_means_se(va), batch_means_se(vc)) + 1e-3


def test_row_chunk_mode_matches_default():
    """The timing-only ROW_CHUNKS mode of the oracle (steps 1-3 over fixed 4096-row chunks on all cores, partials of
    X^T z added in chunk order; SURVEY.md 8(d) oracle timing (ii)) is the same chain as the default path up to the
    summation order of g, and does not depend on the number of threads."""
    import ctypes
    gomp = ctypes.CDLL("libgomp.so.1")
    wl = hsp_synth.make("C2", "cpu", n_rows=9001, p=40)
    Xh, yh = wl.host()
    ref = oracle.OracleChain(Xh, yh, wl.seed); ref.sweep(6)
    b0, l0, t0 = ref.get_draws()
    z0, s0 = ref.get_latent()
    outs = []
    n_max = oracle.max_threads()
    for threads in (1, 3, n_max):
        gomp.omp_set_num_threads(threads)
        assert oracle.max_threads() == threads
        ch = oracle.OracleChain(Xh, yh, wl.seed)
        ch.set_flags(oracle.STORE_Z | oracle.ROW_CHUNKS)
        ch.sweep(6)
        outs.append((ch.get_draws(), ch.get_latent(), ch.get_xtz()))
    for (b, l, t), (z, s), g in outs:
        assert np.array_equal(s, s0)
        assert np.max(np.abs(b - b0)) < 1e-11 and np.max(np.abs(np.log(l / l0))) < 1e-10 and np.max(np.abs(t / t0 - 1)) < 1e-11
        assert np.max(np.abs(z - z0)) < 1e-10
    # chunk-ordered reduction: identical whatever the schedule
    for o in outs[1:]:
        assert np.array_equal(o[0][0], outs[0][0][0]) and np.array_equal(o[2], outs[0][2])
    assert oracle.max_threads() >= 1
