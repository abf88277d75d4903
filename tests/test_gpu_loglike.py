"""GPU parity: likelihood kernels (K1 relative binning, K2 full grid) vs the oracle, through the C ABI.

Tolerance (north_star): |GPU - oracle| <= 1e-6 + 1e-9 |oracle|, fp64.
"""
import math

import numpy as np
import pytest

from paper_2509_24949_b200 import inputs

pytestmark = pytest.mark.gpu


def _close(got, ref):
    got, ref = np.asarray(got), np.asarray(ref)
    fin = np.isfinite(ref)
    assert np.array_equal(np.isfinite(got), fin)
    assert np.array_equal(got[~fin], ref[~fin])
    err = np.abs(got[fin] - ref[fin])
    tol = 1e-6 + 1e-9 * np.abs(ref[fin])
    assert np.all(err <= tol), f"max err {err.max():.3e} at logL {ref[fin][err.argmax()]:.6e}"
    return err.max() if err.size else 0.0


@pytest.fixture(scope="module")
def nssmod():
    from paper_2509_24949_b200 import build, nss
    build.build()
    return nss


def _near(w, p, n, seed):
    th0 = w.theta_fid[w.param_index]
    scale = 0.01 * (w.hi - w.lo)
    return inputs.draw_near(w, n, seed, scale)


@pytest.mark.parametrize("cfg,B,N", [("config1", 32, 10000), ("config2", 128, 10000), ("config2", 64, 6000),
                                      ("config2", 256, 6000), ("config2", 1024, 2500), ("config2", 7, 1500),
                                      ("config1", 1968, 800)])
def test_k1_relative_binning_matches_oracle(nssmod, oracle, cfg, B, N):
    w = inputs.make_data(getattr(inputs, cfg)(n_bins=B), oracle.waveform)
    p = oracle.Problem(w)
    g = nssmod.Nss(w)
    # setup tables: bin edges bit-exact, summary data to rounding
    idx, summ, dd = g.nss_get_tables()
    oidx, _ = p.edges()
    assert np.array_equal(idx, oidx)
    osum = p.summary()
    scale = np.abs(osum).max(axis=1, keepdims=True)
    assert np.max(np.abs(summ - osum) / scale) < 1e-9
    assert dd == pytest.approx(p.DD, rel=1e-13)
    X = np.concatenate([inputs.draw_prior(w, N, 5), _near(w, p, N // 10, 6), w.theta_fid[w.param_index][None, :]])
    ref = p.loglike_batch(X)
    for variant in (1, 2):
        g.set_loglike_variant(variant)
        got = g.nss_loglike_batch(X).cpu().numpy()
        _close(got, ref)
    g.close()


@pytest.mark.parametrize("n", [0, 1, 31, 33, 257, 4097])
def test_k1_ragged_batch_sizes_and_domain(nssmod, oracle, wl2, n):
    p = oracle.Problem(wl2)
    g = nssmod.Nss(wl2)
    X = inputs.draw_prior(wl2, max(n, 1), 9)[:n]
    if n >= 31:
        X[3, 0] = -5.0            # Mc < 0
        X[7, 1] = 1.5             # q > 1
        X[11, 4] = 0.0            # dL = 0
        X[13, 2] = 1.0            # |chi| = 1
        X[17, 5] = math.nan
        X[19, 6] = math.inf
        X[23, 4] = 20000.0        # outside the prior box but inside the domain: finite logL
    ref = p.loglike_batch(X) if n else np.zeros(0)
    for variant in (0, 1, 2):
        g.set_loglike_variant(variant)
        got = g.nss_loglike_batch(X).cpu().numpy()
        assert got.shape == (n,)
        _close(got, ref)
    if n >= 31:
        assert np.isneginf(ref[[3, 7, 11, 13, 17, 19]]).all() and np.isfinite(ref[23])
    g.close()


def test_k1_large_batch_sampled_and_variant_agreement(nssmod, oracle, wl2):
    """BASELINE config 5 at bench size (N = 1e6, B = 128): a fixed subsample against the oracle plus
    properties that hold at any size (both kernel variants agree; permutation invariance)."""
    import torch
    g = nssmod.Nss(wl2)
    p = oracle.Problem(wl2)
    N = 1_000_000
    X = torch.as_tensor(inputs.draw_prior(wl2, N, 5), device="cuda")
    g.set_loglike_variant(1)
    a = g.nss_loglike_batch(X)
    g.set_loglike_variant(2)
    b = g.nss_loglike_batch(X)
    torch.cuda.synchronize()
    assert torch.all(torch.isfinite(a))
    assert float(torch.max(torch.abs(a - b) / (1e-6 + 1e-9 * torch.abs(a)))) <= 1.0
    sel = np.random.default_rng(0).choice(N, 4000, replace=False)
    ref = p.loglike_batch(X[sel].cpu().numpy())
    _close(a[sel].cpu().numpy(), ref)
    perm = torch.randperm(N, device="cuda")
    g.set_loglike_variant(0)
    c = g.nss_loglike_batch(X[perm])
    assert torch.equal(c, a[perm])
    g.close()


def test_k2_full_grid_matches_oracle(nssmod, oracle):
    w = inputs.make_data(inputs.config4(), oracle.waveform)
    p = oracle.Problem(w)
    g = nssmod.Nss(w)
    X = np.concatenate([inputs.draw_prior(w, 400, 5), _near(w, p, 100, 6), w.theta_fid[w.param_index][None, :]])
    X[5, 1] = 2.0
    ref = p.loglike_batch(X)
    for variant in (0, 1, 2):                  # 1: one thread per point, table streamed in TMA tiles; 2: one warp per point
        g.set_loglike_variant(variant)
        _close(g.nss_loglike_batch(X).cpu().numpy(), ref)
    # config 1 geometry too (one detector)
    w1 = inputs.make_data(inputs.config1(), oracle.waveform)
    w1.kind = 1
    p1, g1 = oracle.Problem(w1), nssmod.Nss(w1)
    X1 = inputs.draw_prior(w1, 777, 2)         # three batches of 256 points, the last one ragged
    ref1 = p1.loglike_batch(X1)
    for variant in (1, 2):
        g1.set_loglike_variant(variant)
        _close(g1.nss_loglike_batch(X1).cpu().numpy(), ref1)
    g.close(); g1.close()


def test_k1_vs_k2_residual_identity_on_gpu(nssmod, oracle):
    """P7 on the GPU: with every grid point an edge, K1 - K2 = +1/2 * (dropped quadratic term) > 0, small."""
    w = inputs.make_data(inputs.config1(n_bins=1968), oracle.waveform)
    g0 = nssmod.Nss(w, kind=0)
    g1 = nssmod.Nss(w, kind=1)
    X = inputs.draw_prior(w, 64, 11)
    a = g0.nss_loglike_batch(X).cpu().numpy()
    b = g1.nss_loglike_batch(X).cpu().numpy()
    p = oracle.Problem(w)
    ref = np.array([p.loglike(x, 0) - p.loglike(x, 1) for x in X])
    assert np.all(a - b > -1e-6)
    assert np.allclose(a - b, ref, atol=2e-6)
    g0.close(); g1.close()


def test_gaussian_kind(nssmod, oracle):
    w = inputs.gaussian_workload(5, sigma=0.07)
    p, g = oracle.Problem(w), nssmod.Nss(w)
    X = inputs.draw_prior(w, 3000, 1)
    X[4, 2] = math.nan
    got = g.nss_loglike_batch(X).cpu().numpy()
    ref = p.loglike_batch(X)
    assert np.isneginf(got[4]) and np.isneginf(ref[4])
    m = np.isfinite(ref)
    assert np.allclose(got[m], ref[m], rtol=1e-13, atol=0)
    g.close()

