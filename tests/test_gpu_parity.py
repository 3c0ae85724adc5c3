"""GPU-vs-oracle parity of the whole sweep through the C-ABI (north_star acceptance):
z, beta, lambda, tau per iteration within 1e-9 (fp64 X) / 1e-4 (fp32 X) in the mixed metric of
DESIGN.md reading R12; the truncation side bit-exact."""
import numpy as np
import pytest
import torch

import hsp_synth
import oracle
import paper_1608_04329_b200 as hsp
from conftest import mixed_err

pytestmark = pytest.mark.gpu

TOL = {torch.float64: 1e-9, torch.float32: 1e-4}


def run_parity(wl, n_sweeps, gram=None, flags=0, check_every=1):
    Xh, yh = wl.host()
    tol = TOL[wl.X.dtype]
    g = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed)
    g.set_flags(hsp.HSP_STORE_Z | flags)
    o = oracle.OracleChain(Xh, yh, wl.seed, gram=gram)
    worst = dict(z=0.0, beta=0.0, lam=0.0, tau=0.0)
    for k in range(n_sweeps):
        g.sweep(1)
        o.sweep(1)
        if k % check_every and k != n_sweeps - 1:
            continue
        zg, sg = g.get_latent()
        zo, so = o.get_latent()
        assert np.array_equal(sg, so)                      # truncation side: bit-exact
        assert np.all(zg * sg > 0)
        bg, lg, tg = g.get_draws()
        bo, lo, to = o.get_draws()
        e = dict(z=mixed_err(zg, zo), beta=mixed_err(bg[0], bo[0]), lam=mixed_err(np.log(lg[0]), np.log(lo[0])),
                 tau=abs(tg[0] / to[0] - 1))
        for name, v in e.items():
            worst[name] = max(worst[name], v)
            assert v <= tol, (wl.name, k + 1, name, v)
    print(wl.name, g.fused_variant(), "N,p=", wl.N, wl.p, "worst mixed errors over", n_sweeps, "sweeps:", worst)
    g.close()
    return worst


def test_c1_full_50_sweeps():
    run_parity(hsp_synth.make("C1", "cuda"), 50)


def test_c2_reduced_50_sweeps():
    run_parity(hsp_synth.make("C2", "cuda", n_rows=20011), 50, check_every=5)


def test_c2_full_10_sweeps():
    run_parity(hsp_synth.make("C2", "cuda"), 10, check_every=3)


def test_c3_shape_tma_f32_ragged_50_sweeps():
    wl = hsp_synth.make("C3", "cuda", n_rows=20003)        # 148 CTAs x several tiles of 8 rows + ragged tail
    X64 = wl.X.double()
    gram = (X64.T @ X64).cpu().numpy()                      # library matmul as the oracle's step 6 input
    w = run_parity(wl, 50, gram=gram, check_every=7)
    assert w["beta"] < 1e-4


def test_c5_shape_tma_f32_p2000_5_sweeps():
    wl = hsp_synth.make("C5", "cuda", n_rows=6001)
    X64 = wl.X.double()
    run_parity(wl, 5, gram=(X64.T @ X64).cpu().numpy(), check_every=2)


@pytest.mark.parametrize("name,n_rows,p", [("C4", 3001, 4000), ("C4", 777, 3100), ("C5", 1501, 6000), ("C5", 901, 9000),
                                           ("C3", 4099, 640), ("C5", 300, 16000)])
@pytest.mark.parametrize("eta_mode,z_tol", [(2, 2e-6), (0, 1e-9)])
def test_fused_pass_only_wide_f32(name, n_rows, p, eta_mode, z_tol, hsp_options):
    """a1-a3 + b alone (scales and beta frozen at a planted state): z and X^T z against the oracle, in the
    two arithmetic modes of the eta phase (fp32 chains of 4 -> ~2e-7 in z; exact -> ~1e-13)."""
    hsp_options("fused_eta", eta_mode)
    wl = hsp_synth.make(name, "cuda", n_rows=n_rows, p=p)
    Xh, yh = wl.host()
    beta = wl.beta_true * 0.7
    g = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed)
    g.set_flags(hsp.HSP_STORE_Z | hsp.HSP_FREEZE_SCALES | hsp.HSP_FREEZE_BETA)
    g.set_state(beta=beta, sweep=41)
    o = oracle.OracleChain(Xh, yh, wl.seed, gram=np.zeros((p, p)))
    o.set_flags(oracle.STORE_Z | oracle.FREEZE_SCALES | oracle.FREEZE_BETA)
    o.set_state(beta=beta, sweep=41)
    g.sweep(1); o.sweep(1)
    zg, sg = g.get_latent(); zo, so = o.get_latent()
    assert np.array_equal(sg, so)
    ez, eg = mixed_err(zg, zo), mixed_err(g.get_xtz(), o.get_xtz())
    print(name, n_rows, p, g.fused_variant(), "eta mode", eta_mode, "z", ez, "xtz", eg)
    assert g.fused_variant() == "tma"
    assert ez < z_tol and eg < 1e-5


@pytest.mark.parametrize("n_rows,p", [(4099, 256), (3001, 600), (1000, 1500), (513, 3000)])
def test_fused_pass_only_f64_tma(n_rows, p):
    wl = hsp_synth.make("C2", "cuda", n_rows=n_rows, p=p)
    Xh, yh = wl.host()
    beta = wl.beta_true * 0.5
    g = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed)
    g.set_flags(hsp.HSP_STORE_Z | hsp.HSP_FREEZE_SCALES | hsp.HSP_FREEZE_BETA)
    g.set_state(beta=beta, sweep=3)
    o = oracle.OracleChain(Xh, yh, wl.seed, gram=np.zeros((p, p)))
    o.set_flags(oracle.STORE_Z | oracle.FREEZE_SCALES | oracle.FREEZE_BETA)
    o.set_state(beta=beta, sweep=3)
    g.sweep(1); o.sweep(1)
    zg, _ = g.get_latent(); zo, _ = o.get_latent()
    assert g.fused_variant() == "tma"
    assert mixed_err(zg, zo) < 1e-11 and mixed_err(g.get_xtz(), o.get_xtz()) < 1e-11


@pytest.mark.parametrize("N,p,dtype", [(2, 1, torch.float64), (3, 1, torch.float32), (257, 3, torch.float32), (1000, 7, torch.float64),
                                       (513, 129, torch.float32), (300, 1001, torch.float32), (64, 4099, torch.float32)])
def test_edge_shapes_generic_kernel(N, p, dtype):
    """Degenerate and unaligned shapes (rows not a multiple of 16 bytes) go through the generic kernel."""
    gen = torch.Generator(device="cuda").manual_seed(N * 1000 + p)
    X = torch.randn((N, p), dtype=dtype, device="cuda", generator=gen)
    y = (torch.rand(N, device="cuda", generator=gen) < 0.5).to(torch.uint8)
    wl = hsp_synth.Workload("edge", X, y, np.zeros(p), 17, 0, 0.5)
    w = run_parity(wl, 6)
    assert w["z"] < 1e-9 if dtype == torch.float64 else True


@pytest.mark.parametrize("fill", [0, 1])
def test_degenerate_all_same_response(fill):
    gen = torch.Generator(device="cuda").manual_seed(5)
    X = torch.randn((500, 4), dtype=torch.float64, device="cuda", generator=gen)
    y = torch.full((500,), fill, dtype=torch.uint8, device="cuda")
    run_parity(hsp_synth.Workload("same", X, y, np.zeros(4), 23, 0, float(fill)), 12)


def test_extreme_linear_predictor_uses_tail_form():
    """|eta| up to ~60 on the wrong side of the truncation: the exponential-tail branch of TNpos."""
    gen = torch.Generator(device="cuda").manual_seed(6)
    X = torch.randn((4000, 8), dtype=torch.float64, device="cuda", generator=gen)
    y = (torch.rand(4000, device="cuda", generator=gen) < 0.5).to(torch.uint8)
    beta = np.array([25.0, -18.0, 9.0, 0, 0, 0, 0, 3.0])
    g = hsp.HorseshoeProbit(X, y, 29)
    g.set_flags(hsp.HSP_STORE_Z | hsp.HSP_FREEZE_SCALES | hsp.HSP_FREEZE_BETA)
    g.set_state(beta=beta)
    o = oracle.OracleChain(X.cpu().numpy(), y.cpu().numpy(), 29)
    o.set_flags(oracle.STORE_Z | oracle.FREEZE_SCALES | oracle.FREEZE_BETA)
    o.set_state(beta=beta)
    g.sweep(1); o.sweep(1)
    zg, sg = g.get_latent(); zo, so = o.get_latent()
    eta = o.get_eta()
    assert np.max(-so * eta) > 35          # the test does reach the tail
    assert np.all(zg * sg > 0) and np.all(np.isfinite(zg))
    assert mixed_err(zg, zo) < 1e-12
    assert mixed_err(g.get_xtz(), o.get_xtz()) < 1e-11


def test_gram_matches_oracle():
    for name, n, p in [("C1", 1000, 10), ("C2", 5003, 100), ("C3", 3001, 333)]:
        wl = hsp_synth.make(name, "cuda", n_rows=n, p=p)
        Xh, yh = wl.host()
        g = hsp.HorseshoeProbit(wl.X, wl.y, 1)
        o = oracle.OracleChain(Xh, yh, 1)
        Gg, Go = np.tril(g.get_gram()), np.tril(o.get_gram())
        assert np.max(np.abs(Gg - Go)) <= 1e-12 * np.max(np.abs(Go))
        g.close()


def test_cholesky_factor_and_breakdown_status():
    wl = hsp_synth.make("C3", "cuda", n_rows=3000, p=333)
    g = hsp.HorseshoeProbit(wl.X, wl.y, 1)
    g.sweep(1)
    st = g.get_state()
    L = g.get_chol()
    Q = np.tril(g.get_gram()); Q = Q + np.tril(Q, -1).T + np.diag(st["tau_inv2"] * st["lam_inv2"])
    assert np.linalg.norm(L @ L.T - Q) <= 1e-13 * np.linalg.norm(Q)
    # a hugely negative prior precision makes Q indefinite: reported, not crashed
    g.set_flags(hsp.HSP_FREEZE_SCALES | hsp.HSP_FREEZE_Z)
    g.set_state(lam_inv2=np.full(333, -1e9))
    g.sweep(1)
    with pytest.raises(hsp.HspError) as ei:
        g.get_draws()
    assert ei.value.code == -4
    g.close()


def test_invalid_y_rejected():
    X = torch.randn((10, 2), dtype=torch.float64, device="cuda")
    y = torch.tensor([0, 1, 2, 0, 1, 0, 1, 0, 1, 0], dtype=torch.uint8, device="cuda")
    with pytest.raises(hsp.HspError) as ei:
        hsp.HorseshoeProbit(X, y, 1)
    assert ei.value.code == -1


@pytest.mark.parametrize("sb,p,n_rows", [(2, 333, 3001), (1, 200, 2003), (3, 1000, 4001), (8, 2000, 6001)])
def test_block_diagonal_inverse_and_block_substitution(sb, p, n_rows, hsp_options):
    """d2 by block forward/backward substitution with a block-diagonal inverse (the p > 1280 path), forced at
    small p through the option "chol_sb": the whole sweep against the oracle."""
    hsp_options("chol_sb", sb)
    wl = hsp_synth.make("C3", "cuda", n_rows=n_rows, p=p)
    X64 = wl.X.double()
    w = run_parity(wl, 6, gram=(X64.T @ X64).cpu().numpy())
    assert w["beta"] < 1e-5


@pytest.mark.parametrize("name,n,p", [("C3", 5003, 333), ("C3", 3001, 1000), ("C4", 7001, 520), ("C3", 257, 128), ("C5", 2100, 2000)])
def test_tensor_core_gram_matches_fp64_definition(name, n, p, hsp_options):
    """Row c0 on tcgen05 (split-bf16 products, fp32 TMEM accumulation over <= 128 rows, fp64 flush), forced at
    small sizes: against the fp64 definition G = X^T X (library matmul).  The TMEM accumulation truncates: the
    error is a relative bias of about -2e-7; bound 1e-6 of max|G|."""
    hsp_options("gram_tc", 1)
    wl = hsp_synth.make(name, "cuda", n_rows=n, p=p)
    X64 = wl.X.double()
    Go = (X64.T @ X64).cpu().numpy()
    g = hsp.HorseshoeProbit(wl.X, wl.y, 1)
    Gg = g.get_gram()
    g.close()
    assert np.array_equal(Gg, Gg.T)
    err = np.max(np.abs(Gg - Go)) / np.max(np.abs(Go))
    print(name, n, p, "tensor-core Gram: max|dG|/max|G| =", err)
    assert err <= 1e-6
    # and the whole chain on top of it stays inside the fp32-X tolerance
    run_parity(hsp_synth.make(name, "cuda", n_rows=n, p=p), 4, gram=Go)


# ---- fused_pass_narrow: every instantiation the default dispatch can reach (fused_pass.cu narrow_plan): the row is
# read in units of U = 4, 8 or 16 bytes (the largest power of two dividing the row), and rows of an even number q of
# 16-byte units are read with a per-lane start offset (skew shift 2, 1, 0 for gcd(q, 8) = 2, 4, 8); fp32 chains and exact
# fp64.  Whole sweeps against the oracle.
NARROW_CASES = [
    # config (dtype), rows, p, U, skew shift (3 = none)
    ("C3", 9001, 141, 4, 3),      # fp32, 564-byte rows: the shape of the paper's real-data run
    ("C3", 5003, 511, 4, 3),      # fp32, the widest row the narrow kernel takes
    ("C3", 9001, 250, 8, 3),      # fp32, 1000-byte rows
    ("C3", 20011, 100, 16, 3),    # fp32, q = 25
    ("C3", 9001, 180, 16, 3),     # fp32, q = 45
    ("C3", 12001, 200, 16, 2),    # fp32, q = 50: gcd 2
    ("C3", 6007, 400, 16, 1),     # fp32, q = 100: gcd 4
    ("C3", 24001, 96, 16, 0),     # fp32, q = 24: gcd 8
    ("C3", 32003, 17, 4, 3),      # fp32, very narrow rows (30 row groups in the x*z phase)
    ("C2", 6007, 150, 16, 3),     # fp64, q = 75
    ("C2", 5003, 101, 8, 3),      # fp64, 808-byte rows
    ("C2", 5003, 190, 16, 3),     # fp64, q = 95
    ("C2", 4001, 250, 16, 3),     # fp64, q = 125
    ("C2", 6007, 100, 16, 2),     # fp64, q = 50 (C2's own row width)
    ("C2", 5003, 252, 16, 2),     # fp64, q = 126: gcd 2, the widest fp64 rows just below the wide kernel
    ("C2", 8009, 64, 16, 0),      # fp64, q = 32: gcd 8
]


def _check_narrow_case(wl, U, shift):
    rb = wl.p * wl.X.element_size()
    assert rb % U == 0 and (U == 16 or rb % (2 * U) != 0)
    if U == 16:
        q, g = rb // 16, 1
        while g < 8 and q % (2 * g) == 0:
            g *= 2
        assert shift == {1: 3, 2: 2, 4: 1, 8: 0}[g]


@pytest.mark.parametrize("name,n_rows,p,U,shift", NARROW_CASES)
def test_narrow_kernel_every_instantiation_whole_sweeps(name, n_rows, p, U, shift):
    wl = hsp_synth.make(name, "cuda", n_rows=n_rows, p=p)
    _check_narrow_case(wl, U, shift)
    X64 = wl.X.double()
    probe = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed)
    assert probe.fused_variant() == "tma-narrow"
    probe.close()
    w = run_parity(wl, 8, gram=(X64.T @ X64).cpu().numpy())
    assert w["z"] < (2e-6 if wl.X.dtype == torch.float32 else 1e-9)


@pytest.mark.parametrize("eta_mode", [2, 0])
@pytest.mark.parametrize("name,n_rows,p,U,shift", NARROW_CASES)
def test_narrow_kernel_fused_pass_only(name, n_rows, p, U, shift, eta_mode, hsp_options):
    """a1-a3 + b alone at a planted beta (scales and beta frozen): z and X^T z against the oracle, in both arithmetic
    modes of the eta phase for fp32 X (fp32 chains / exact fp64)."""
    if name == "C2" and eta_mode == 0:
        pytest.skip("fp64 X has one eta mode")
    hsp_options("fused_eta", eta_mode)
    wl = hsp_synth.make(name, "cuda", n_rows=n_rows + 13, p=p)
    Xh, yh = wl.host()
    beta = wl.beta_true * 0.6
    g = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed)
    assert g.fused_variant() == "tma-narrow"
    g.set_flags(hsp.HSP_STORE_Z | hsp.HSP_FREEZE_SCALES | hsp.HSP_FREEZE_BETA)
    g.set_state(beta=beta, sweep=11)
    o = oracle.OracleChain(Xh, yh, wl.seed, gram=np.zeros((p, p)))
    o.set_flags(oracle.STORE_Z | oracle.FREEZE_SCALES | oracle.FREEZE_BETA)
    o.set_state(beta=beta, sweep=11)
    g.sweep(1); o.sweep(1)
    zg, sg = g.get_latent(); zo, so = o.get_latent()
    assert np.array_equal(sg, so)
    ez, eg = mixed_err(zg, zo), mixed_err(g.get_xtz(), o.get_xtz())
    print(name, n_rows, p, "U", U, "shift", shift, "eta mode", eta_mode, "narrow fused pass only: z", ez, "xtz", eg)
    f32 = wl.X.dtype == torch.float32
    assert ez < ((2e-6 if eta_mode else 1e-9) if f32 else 1e-11) and eg < (1e-5 if f32 else 1e-11)
    g.close()


def test_cholesky_does_not_depend_on_the_number_of_ctas(hsp_options):
    """every tile is accumulated in ascending k by a fixed sequence of products, whatever the schedule --
    one CTA (prefix + finish tasks), a chain CTA plus a few or many others: L and the draws are bit-identical.  (The grid
    of the fused pass is pinned: the per-CTA partials of X^T z are fp32 chains, whose grouping follows the grid.)"""
    wl = hsp_synth.make("C3", "cuda", n_rows=3001, p=640)         # nt = 10 tile rows
    ref = None
    hsp_options("fused_grid", 64)
    for K in (1, 2, 3, 7, 20):
        hsp_options("chol_ctas", K)
        g = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed)
        assert g.plan()["chol_ctas"] == K
        g.sweep(3)
        out = (g.get_chol(), *g.get_draws())
        g.close()
        if ref is None:
            ref = out
        else:
            for a, b in zip(out, ref):
                assert np.array_equal(a, b), K


def test_cholesky_very_large_p_round_robin_schedule():
    """p > 6144 (nt > 96): round-robin schedule without a chain CTA, block-diagonal inverse.  The oracle's O(p^3) sweep is not
    affordable here: the factor is checked against its definition, L L^T = G + diag(tau^-2 lambda^-2), and
    the beta draw against the solve with numpy's triangular routines on the same L."""
    p = 6200
    wl = hsp_synth.make("C3", "cuda", n_rows=1500, p=p)
    g = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed)
    G = g.get_gram()
    g.sweep(1)
    st = g.get_state()
    L = g.get_chol()
    b = g.get_draws()[0][-1]
    g.close()
    assert np.all(np.isfinite(L)) and np.all(np.isfinite(b))
    # the scales in `st` are the ones drawn in this sweep, i.e. the ones that entered Q
    Q = G + np.diag(st["tau_inv2"] * st["lam_inv2"])
    assert np.abs(np.triu(L, 1)).max() == 0.0
    err = np.abs(L @ L.T - Q).max() / np.abs(Q).max()
    print("p = 6200: |L L^T - Q| / max|Q| =", err)
    assert err < 1e-13
