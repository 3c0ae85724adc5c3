"""Pins for the exponential inversion and the Cheng (1977) gamma sampler
 as the oracle implements them."""
import os

import numpy as np
import pytest
from scipy import stats

import oracle

GOLD = {}
for line in open(os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")):
    line = line.split("#")[0].split()
    if len(line) == 2:
        GOLD[line[0]] = float(line[1])


@pytest.mark.parametrize("alpha", [1.5, 5.5, 50.5, 500.5, 2000.5])
def test_cheng_gamma_law(alpha):
    n = 20000
    draws, trials = zip(*[oracle.cheng_gamma(alpha, 77, k) for k in range(1, n + 1)])
    x = np.array(draws)
    assert stats.kstest(x, stats.gamma(alpha).cdf).pvalue > 1e-3
    assert abs(x.mean() - alpha) < 4.5 * np.sqrt(alpha / n)
    assert abs(x.var() / alpha - 1) < 4.5 * np.sqrt((2 + 6 / alpha) / n)     # var of sample variance
    acc = n / (np.sum(trials) + n)                                           # trials are 0-based
    if alpha >= 50:
        # "each thread accepts with probability approximately 0.88"
        assert abs(acc - GOLD["cheng_lane_acceptance"]) < 0.015, acc
    else:
        assert 0.70 < acc < 0.90
    # all 32 lanes rejecting has probability ~3.4e-30 = (1-0.88)^32
    assert abs(np.log10((1 - GOLD["cheng_lane_acceptance"]) ** 32) - np.log10(GOLD["cheng_all32_reject"])) < 0.05


def test_cheng_first_accepted_trial_semantics():
    """The result is the proposal of the smallest accepted trial index: recompute it here."""
    alpha, seed = 7.5, 5
    a, b = 1 / np.sqrt(2 * alpha - 1), alpha - np.log(4)
    c = alpha + 1 / a
    for k in range(1, 200):
        x, t_acc = oracle.cheng_gamma(alpha, seed, k)
        for t in range(t_acc + 1):
            u1, u2 = oracle.uniforms(seed, t, k, oracle.TAG_TAU)
            V = a * np.log(u1 / (1 - u1))
            X = alpha * np.exp(V)
            ok = b + c * V - X >= np.log(u1 * u1 * u2)
            assert ok == (t == t_acc)
        assert abs(X - x) <= 1e-14 * x


def test_exponential_inversion_law():
    """lam^-2, nu^-1, xi^-1 are -ln(u)/rate: KS against Exp(rate) through the chain."""
    rng = np.random.default_rng(1)
    N, p = 8, 3
    X = rng.standard_normal((N, p))
    y = (rng.random(N) < 0.5).astype(np.uint8)
    ch = oracle.OracleChain(X, y, seed=11)
    ch.set_flags(oracle.FREEZE_Z | oracle.FREEZE_BETA)
    beta = np.array([0.7, -0.2, 0.0])
    lam, nu, tau, xi = [], [], [], []
    n = 4000
    for it in range(n):
        ch.set_state(beta=beta, lam_inv2=[1.0, 2.0, 3.0], nu_inv=[0.5, 1.0, 2.0], tau_inv2=1.5, xi_inv=0.8)
        ch.sweep(1)
        st = ch.get_state()
        lam.append(st["lam_inv2"].copy()); nu.append(st["nu_inv"].copy())
        tau.append(st["tau_inv2"]); xi.append(st["xi_inv"])
    lam, nu, tau, xi = map(np.array, (lam, nu, tau, xi))
    for j in range(p):
        rate = [0.5, 1.0, 2.0][j] + 1.5 * beta[j] ** 2 / 2          # eq. (12)
        assert stats.kstest(lam[:, j], stats.expon(scale=1 / rate).cdf).pvalue > 1e-3
        # nu | new lambda: -ln u * (1 + lam) ~ Exp(1)
        assert stats.kstest(nu[:, j] * (1 + lam[:, j]), stats.expon().cdf).pvalue > 1e-3
    # tau^-2 | new lambda ~ Gamma((p+1)/2, rate xi^-1 + S)  (PAPER.md:182 with reading R1)
    S = 0.5 * np.sum(lam * beta ** 2, axis=1)
    assert stats.kstest(tau * (0.8 + S), stats.gamma((p + 1) / 2).cdf).pvalue > 1e-3
    assert stats.kstest(xi * (1 + tau), stats.expon().cdf).pvalue > 1e-3
