"""Pins for the oracle's normal-tail inverse, Phi^-1 and TNpos (the truncated-normal map that
replaces the paper's rejection samplers; the target law is PAPER.md:174, 186)."""
import os

import mpmath as mp
import numpy as np
import pytest
from scipy import special, stats

import oracle

mp.mp.dps = 50
GOLD = {}
for line in open(os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")):
    line = line.split("#")[0].split()
    if len(line) == 2:
        GOLD[line[0]] = float(line[1])


def Qmp(x):
    return mp.erfc(mp.mpf(x) / mp.sqrt(2)) / 2


def test_norm_inv_matches_scipy_ndtri():
    u = np.concatenate([np.linspace(1e-6, 1 - 1e-6, 4001), 10.0 ** -np.arange(7, 300, 7.0)])
    got = np.array([oracle.norm_inv(v) for v in u])
    ref = special.ndtri(u)
    assert np.max(np.abs(got - ref) / np.maximum(1.0, np.abs(ref))) < 5e-14


@pytest.mark.parametrize("q", [0.5, 0.49, 0.3, 1e-3, 1e-10, 1e-100, 1e-300, 0.7, 0.999999, 1 - 2.0 ** -40])
def test_qinv_round_trip_mpmath(q):
    x = oracle.qinv(q)
    # dq/q = -(phi/Q) dx : a half-ulp error in x moves log Q by at most (phi/Q)*ulp(x)/2
    hazard = mp.npdf(x) / Qmp(x)
    tol = float(hazard) * np.spacing(abs(x) + 1e-300) + 1e-17
    assert abs(float(Qmp(x) / mp.mpf(q) - 1)) <= tol


@pytest.mark.parametrize("m", [-100.0, -30.0, -8.0, -2.0, -0.3, 0.0, 0.47, 1.0, 3.0, 8.0, 10.0, 30.0])
def test_tnpos_round_trip_mpmath(m):
    """The contract: w = m + t with Q(t) = u Q(-m).  Checked in 50-digit arithmetic."""
    us = [2.0 ** -53, 1e-9, 0.01, 0.3, 0.5, 0.9, 0.999, 1 - 1e-9, 1 - 2.0 ** -53]
    for u in us:
        w = oracle.tnpos(m, u)
        assert w > 0.0
        a = -mp.mpf(m)
        # exact w in high precision: solve Q(t) = u Q(a) by mp.findroot on log Q
        target = mp.log(mp.mpf(u)) + mp.log(Qmp(a))
        t0 = mp.mpf(w) - mp.mpf(m)
        t_exact = mp.findroot(lambda t: mp.log(Qmp(t)) - target, t0, tol=mp.mpf(10) ** -40, maxsteps=200)
        w_exact = mp.mpf(m) + t_exact
        if w_exact < mp.mpf(np.finfo(float).tiny):
            assert w == np.finfo(float).tiny
            continue
        err = abs(mp.mpf(w) - w_exact)
        # w is the fp64 rounding of a long-double evaluation of m + t
        bound = mp.mpf(np.spacing(w)) * mp.mpf("0.51") + (1 + abs(t_exact)) * mp.mpf(2) ** -60
        assert err <= bound, (m, u, float(err), float(bound))


def test_tnpos_matches_scipy_truncnorm():
    for m in [-6.0, -1.0, 0.0, 0.47, 2.0, 5.0]:
        u = np.linspace(0.001, 0.999, 999)
        got = oracle.tnpos_many(np.full_like(u, m), u)
        ref = stats.truncnorm.isf(u, a=-m, b=np.inf, loc=m, scale=1.0)
        assert np.max(np.abs(got - ref) / np.maximum(got, 1e-3)) < 1e-8     # scipy's own accuracy


def test_tnpos_sign_invariant_and_clamp():
    rng = np.random.default_rng(0)
    m = rng.uniform(-40, 40, 20000)
    u = np.array([oracle.uniforms(9, i, 1, 0)[0] for i in range(m.size)])
    w = oracle.tnpos_many(m, u)
    assert np.all(w > 0) and np.all(np.isfinite(w))
    # u -> 1 with large m: exact w ~ 1e-16-ish or smaller; must stay strictly positive
    assert oracle.tnpos(37.0, 1 - 2.0 ** -53) > 0.0
    assert oracle.tnpos(-100.0, 0.5) > 0.0
    # monotone decreasing in u (inverse survival function)
    uu = np.linspace(0.001, 0.999, 500)
    for mm in (-5.0, 0.0, 5.0):
        ww = oracle.tnpos_many(np.full_like(uu, mm), uu)
        assert np.all(np.diff(ww) < 0)


@pytest.mark.parametrize("m", [-30.0, -8.0, -2.0, 0.0, 0.47, 3.0, 10.0])
def test_tnpos_closed_form_moments(m):
    """E w = m + h, Var w = 1 - m h - h^2, h = phi(m)/Phi(m) (textbook truncated-normal moments)."""
    K = 400000
    u = (np.arange(K) + 0.5) / K                       # stratified: midpoint rule over u
    w = oracle.tnpos_many(np.full(K, m), u)
    h = float(mp.npdf(m) / mp.ncdf(m))
    mean, var = m + h, 1 - m * h - h * h
    assert abs(w.mean() - mean) < 2e-5 * max(1.0, abs(mean))
    assert abs(w.var() - var) < 2e-4 * max(var, 1e-6) + 1e-9


@pytest.mark.parametrize("m", [-3.0, 0.0, 0.4699, 0.4701, 2.5])
def test_tnpos_same_law_as_paper_rejection_samplers(m):
    """PAPER.md:210-216 with DESIGN.md reading R6: both samplers target TN(m,1) on (0,inf)."""
    n = 20000
    ours = oracle.tnpos_many(np.full(n, m), np.array([oracle.uniforms(21, i, 1, 0)[0] for i in range(n)]))
    theirs = np.array([oracle.tnpos_rejection(m, 22, i)[0] for i in range(n)])
    cdf = lambda w: 1.0 - stats.norm.sf(w - m) / stats.norm.sf(-m)
    assert stats.kstest(ours, cdf).pvalue > 1e-3
    assert stats.kstest(theirs, cdf).pvalue > 1e-3
    assert stats.ks_2samp(ours, theirs).pvalue > 1e-3


def test_rejection_acceptance_matches_paper_near_switch():
    """worst-case acceptance ~2/3 around mu* = 0.47, near 1 elsewhere; the two
    samplers cross at the switch point PAPER.md:210 prints."""
    sw = GOLD["tn_switch"]
    n = 40000
    for m, lo, hi in [(sw - 1e-6, 0.64, 0.72), (sw + 1e-6, 0.64, 0.72), (4.0, 0.999, 1.0), (-4.0, 0.85, 1.0)]:
        trials = sum(oracle.tnpos_rejection(m, 5, i)[1] for i in range(n))
        acc = n / trials
        assert lo <= acc <= hi, (m, acc)
    # closed forms: Gaussian sampler accepts with Phi(m); Robert's with
    # theta*exp(theta^2/2 + theta*m)*sqrt(2 pi)*Phi(m)... evaluated by quadrature instead
    theta = 0.5 * (-sw + np.sqrt(sw * sw + 4))
    acc_exp = float(mp.quad(lambda w: theta * mp.e ** (-theta * w) * mp.e ** (-(w - sw - theta) ** 2 / 2), [0, mp.inf]))
    acc_gau = float(mp.ncdf(sw))
    assert abs(acc_exp - acc_gau) < 2e-3                 # they cross at 0.47
    assert abs(acc_gau - GOLD["tn_worst_acceptance"]) < 0.02
