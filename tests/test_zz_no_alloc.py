"""hsp_xtz_noalloc (include/hsp.h): rows a1-a3 + b through the entry point that allocates nothing (scratch in a static
device array) against the existing path (a chain created with hsp_create, one hsp_sweep), on two calls in a row that
share the static scratch: a wide fp32 problem first, then a smaller fp64 one, then the first again.  Collected last
(file name), passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest
import torch

import hsp_synth
import paper_1608_04329_b200 as hsp
from conftest import mixed_err

pytestmark = pytest.mark.gpu


def _existing_path(wl, n_sweeps):
    """g = X^T z and z of sweep n_sweeps of a chain, and the beta that sweep started from."""
    g = hsp.HorseshoeProbit(wl.X, wl.y, wl.seed)
    g.set_flags(hsp.HSP_STORE_Z)
    if n_sweeps > 1:
        g.sweep(n_sweeps - 1)
    beta_in = g.get_state()["beta"].copy()
    g.sweep(1)
    xtz = g.get_xtz()
    z, _ = g.get_latent()
    g.close()
    return beta_in, xtz, z


def _no_alloc(wl, k, beta_in, g_out, z_out):
    beta = torch.from_numpy(beta_in).cuda()
    hsp.xtz_noalloc(wl.X, wl.y, wl.seed, k, beta, g_out, z_out)
    torch.cuda.synchronize()
    return g_out.cpu().numpy().copy(), z_out.cpu().numpy().copy()


def test_no_alloc_entry_matches_the_chain_on_consecutive_calls():
    cases = [(hsp_synth.make("C3", "cuda", n_rows=4003, p=640), 3, 1e-4),      # fp32 X, wide TMA kernel, sweep 3 (beta != 0)
             (hsp_synth.make("C2", "cuda", n_rows=30011), 2, 1e-9),             # fp64 X, narrow kernel, fewer partials
             (hsp_synth.make("C1", "cuda"), 1, 1e-9)]                           # generic kernel, cold start (beta = 0)
    ref = [_existing_path(wl, k) for wl, k, _ in cases]
    outs = [(torch.empty(wl.p, dtype=torch.float64, device="cuda"), torch.empty(wl.N, dtype=torch.float64, device="cuda"))
            for wl, _, _ in cases]
    mem0 = torch.cuda.memory_allocated()
    # two (and more) calls in a row on the shared scratch, sizes going down and up again
    for idx in (0, 1, 2, 0, 1):
        wl, k, tol = cases[idx]
        beta_in, xtz_ref, z_ref = ref[idx]
        g_out, z_out = outs[idx]
        g_out.fill_(float("nan")); z_out.fill_(float("nan"))
        xtz, z = _no_alloc(wl, k, beta_in, g_out, z_out)
        assert np.all(np.isfinite(xtz)) and np.all(np.isfinite(z))
        assert np.array_equal(np.sign(z), 2.0 * wl.y.cpu().numpy() - 1.0)       # the truncation side is exact
        ez, eg = mixed_err(z, z_ref), mixed_err(xtz, xtz_ref)
        print(f"no-alloc call on {wl.N} x {wl.p} {wl.X.dtype}, sweep {k}: z {ez:.2e}, X^T z {eg:.2e} (tolerance {tol:g})")
        assert ez <= tol and eg <= tol
    assert hsp.noalloc_scratch_bytes() == 8 * (2 ** 20 + 32)
    assert torch.cuda.memory_allocated() >= mem0                                # (torch sees only its own allocations)


def test_no_alloc_entry_rejects_what_does_not_fit():
    L = hsp.lib()
    # wide TMA kernel, one CTA per SM, one row group: 148 x 8192 doubles of partials do not fit 2^20
    p = 8192
    X = torch.zeros((3000, p), dtype=torch.float32, device="cuda")
    y = torch.zeros(3000, dtype=torch.uint8, device="cuda")
    beta = torch.zeros(p, dtype=torch.float64, device="cuda")
    g_out = torch.zeros(p, dtype=torch.float64, device="cuda")
    with pytest.raises(hsp.HspError) as ei:
        hsp.xtz_noalloc(X, y, 1, 1, beta, g_out)
    assert ei.value.code == -1 and "too large for the static scratch" in str(ei.value)
    with pytest.raises(hsp.HspError):
        hsp.xtz_noalloc(X, y, 1, 0, beta, g_out)                                 # sweep numbers start at 1
    assert L.hsp_xtz_noalloc(None, hsp.HSP_F32, None, 10, 2, 1, 1, None, None, None, None) == -1
