"""GPU parity: Philox, K4 bookkeeping kernels, K3 slice-sampling chains and nss_run vs the oracle."""
import math

import numpy as np
import pytest
import scipy.special
import scipy.stats

from paper_2509_24949_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def nssmod():
    from paper_2509_24949_b200 import build, nss
    build.build()
    return nss


@pytest.fixture(scope="module")
def ggauss(nssmod):
    return nssmod.Nss(inputs.gaussian_workload(4, sigma=0.05))


def test_philox_bit_exact(ggauss, oracle):
    rng = np.random.default_rng(0)
    n = 100000
    ctr = rng.integers(0, 2 ** 32, size=(n, 4), dtype=np.uint64).astype(np.uint32)
    ctr[0] = 0
    ctr[1] = 0xFFFFFFFF
    seed = (0xDEADBEEF << 32) | 0x12345678
    got = ggauss.nss_philox(seed, ctr)
    for i in list(range(64)) + list(rng.integers(0, n, 400)):
        assert tuple(int(x) for x in got[i]) == oracle.philox((seed & 0xFFFFFFFF, seed >> 32), [int(c) for c in ctr[i]])
    # all rows distinct (bijection)
    assert len({tuple(r) for r in got[:20000].tolist()}) == 20000


@pytest.mark.parametrize("n,k", [(100, 50), (1000, 500), (5000, 2500), (1025, 1), (300, 299), (2, 1), (8192, 4096), (8193, 4096),
                                 (33000, 16500), (65536, 65535), (200000, 1), (200001, 100000)])
def test_select_lowest_bit_exact(ggauss, oracle, n, k):
    """Up to 8192 values the ranks are counted (n^2 comparisons); above, they come from a sample sort with (logL, slot)
    splitters (256 buckets, 512 above 131072 values).  Same total order, so the same bits — with a quarter of the values
    tied, -inf entries, and (n = 200000) every value equal but one, where only the slot half of the key separates them."""
    rng = np.random.default_rng(n)
    l = rng.normal(size=n) * 10
    l[rng.integers(0, n, n // 4)] = l[0]           # ties -> slot order
    if n == 200000:
        l[:] = 3.25
        l[777] = 3.0
    if n > 10:
        l[5] = -np.inf
        l[n - 1] = -np.inf
    dead, surv, lstar = ggauss.nss_select_lowest(l, k)
    if n <= 5000:
        odead, osurv = oracle.select_lowest(l, k)
    else:
        order = np.argsort(l, kind="stable")           # the library routine that pins the oracle (P12)
        odead, osurv = order[:k], np.sort(order[k:])
    assert np.array_equal(dead.cpu().numpy(), odead)
    assert np.array_equal(surv.cpu().numpy(), osurv)
    assert lstar == l[odead[-1]]


def test_tune_matches_oracle(nssmod, oracle):
    rng = np.random.default_rng(1)
    for d, n in ((11, 1000), (11, 5000), (4, 100), (1, 50), (7, 33)):
        w = inputs.gaussian_workload(d)
        g = nssmod.Nss(w)
        scales = np.array([1.0, 0.1, 0.5, 0.5, 600.0, 1e-3, 1.5, 0.3, 0.6, 0.01, 0.014])[:d]
        A = rng.normal(size=(d, d))
        x = rng.normal(size=(n, d)) @ A.T * scales + 1e3 * scales
        rc, mean, chol = g.nss_tune(x)
        orc, omean, ocov, ochol = oracle.tune(x)
        assert rc == 0 and orc == 0
        assert np.allclose(mean.cpu().numpy(), omean, rtol=1e-13)
        assert np.allclose(chol.cpu().numpy(), ochol, rtol=1e-8, atol=1e-300)
        if d > 2:
            x[:, 2] = 7.0                   # zero variance: the pivot is exactly 0 on both sides
            assert g.nss_tune(x)[0] == nssmod.NSS_ECHOL and oracle.tune(x)[0] != 0
        g.close()


def test_tune_near_singular_covariance_reading_r5(nssmod, oracle):
    """Reading R5: ECHOL if and only if a pivot as computed is <= 0.  A nearly singular live-point covariance
    (chi_1 ~ chi_2 to 1e-5 of their spread: pivot ~1e-10 of the variance) factors on both sides; the well-conditioned
    columns agree to 1e-8, the tiny pivot to 1e-4 (it is a difference of nearly equal sums, taken in a different but
    fixed order), and the GPU factor reproduces the covariance.  With exactly collinear columns the pivot is rounding
    noise of either sign: each side may report ECHOL or return a factor, and a returned factor reproduces the covariance."""
    from test_oracle_sampler import near_singular_population
    g = nssmod.Nss(inputs.gaussian_workload(11))
    x = near_singular_population(np.random.default_rng(5))
    rc, mean, chol = g.nss_tune(x)
    orc, omean, ocov, ochol = oracle.tune(x)
    assert rc == 0 and orc == 0
    L = chol.cpu().numpy()
    assert np.allclose(L[:, :3], ochol[:, :3], rtol=1e-8, atol=1e-300)
    assert np.allclose(L[:, 4:], ochol[:, 4:], rtol=1e-4, atol=1e-12 * np.abs(ochol).max())
    assert L[3, 3] == pytest.approx(ochol[3, 3], rel=1e-4)
    assert np.allclose(L @ L.T, ocov, rtol=1e-9, atol=1e-22)
    x[:, 3] = x[:, 2]
    rc, mean, chol = g.nss_tune(x)
    L = chol.cpu().numpy()
    cov = np.cov(x.T)
    assert rc == nssmod.NSS_ECHOL or np.allclose(L @ L.T, cov, rtol=1e-9, atol=1e-16 * cov[2, 2])
    g.close()


@pytest.mark.parametrize("n,k", [(1000, 500), (5000, 2500), (100, 1), (3000, 2999)])
def test_evidence_update_matches_oracle(ggauss, oracle, n, k):
    rng = np.random.default_rng(2)
    dl = np.sort(rng.normal(size=k) * 5 - 1.2e4)
    if k > 10:
        dl[0] = -np.inf
    logX, logZ = -0.7, -1.2e4
    gx, gz, lw = ggauss.nss_evidence_update(dl, n, logX, logZ)
    ox, oz, olw = oracle.evidence_update(dl, n, logX, logZ)
    assert gx == pytest.approx(ox, rel=1e-13)
    assert gz == pytest.approx(oz, rel=1e-13, abs=1e-9)
    assert np.allclose(lw.cpu().numpy(), olw, rtol=0, atol=1e-9)
    gx2, gz2, _ = ggauss.nss_evidence_update(dl, n, 0.0, -np.inf)
    ox2, oz2, _ = oracle.evidence_update(dl, n, 0.0, -np.inf)
    assert gz2 == pytest.approx(oz2, rel=1e-13)


def test_init_live_matches_oracle(nssmod, oracle, wl1):
    g, p = nssmod.Nss(wl1), oracle.Problem(wl1)
    live, logL = g.nss_init_live(300, 77)
    olive, ologL = p.init_live(300, 77)
    assert np.array_equal(live.cpu().numpy(), olive)                 # same Philox words, same affine map
    assert np.allclose(logL.cpu().numpy(), ologL, rtol=1e-9, atol=1e-6)
    g.close()


def _trajectory_parity(g, p, live, logL, k, n_repeats, seed, it, logLstar=math.nan, max_excluded=0.03, w=None, o=None):
    r = g.nss_replace_step(live, logL, k, n_repeats, seed, it, logLstar=logLstar, want_trace=True)
    if o is None:                                 # else: the oracle's result for these very arguments, computed by the caller
        o = p.replace_step(live, logL, k, n_repeats, seed, it, logLstar=logLstar, want_trace=True)
    assert o["rc"] == 0
    assert np.array_equal(r["dead_idx"].cpu().numpy(), o["dead_idx"])
    assert np.array_equal(r["dead_theta"].cpu().numpy(), o["dead_theta"])
    assert np.array_equal(r["dead_logL"].cpu().numpy(), o["dead_logL"])
    assert r["logLstar"] == o["logLstar"]
    gtr, otr = r["trace"].cpu().numpy(), o["trace"]
    margin = np.minimum(r["margin"].cpu().numpy(), o["margin"])
    safe = margin > 1e-6                          # A20: chains whose bracket tests all clear L* by > 1e-6
    print(f"[trajectory parity] n={live.shape[0]} k={k} repeats={n_repeats} it={it}: {(~safe).sum()} of {k} chains excluded "
          f"by the 1e-6 margin rule ({100 * (~safe).mean():.2f} %, limit {100 * max_excluded:.0f} %)")
    assert safe.mean() >= 1 - max_excluded, f"{(~safe).sum()} of {k} chains excluded"
    assert np.array_equal(gtr[safe], otr[safe])                       # identical decisions
    didx = o["dead_idx"]
    gl, ol = r["live"].cpu().numpy(), o["live"]
    width = (w.hi - w.lo) if w is not None else 1.0
    assert np.all(np.abs(gl[didx][safe] - ol[didx][safe]) <= 1e-9 * width)
    glog, olog = r["logL"].cpu().numpy(), o["logL"]
    assert np.all(np.abs(glog[didx][safe] - olog[didx][safe]) <= 1e-6 + 1e-9 * np.abs(olog[didx][safe]))
    surv = np.setdiff1d(np.arange(live.shape[0]), didx)
    assert np.array_equal(gl[surv], np.asarray(live)[surv]) and np.array_equal(glog[surv], np.asarray(logL)[surv])
    if safe.all():
        assert r["n_evals"] == o["n_evals"]
    assert np.all(glog[didx] > o["logLstar"])
    return r, o, safe


def test_replace_step_trajectories_gaussian(nssmod, oracle):
    for d, n, k in ((4, 1000, 500), (11, 400, 399), (3, 64, 1)):
        w = inputs.gaussian_workload(d, sigma=0.05)
        g, p = nssmod.Nss(w), oracle.Problem(w)
        live, logL = p.init_live(n, 3)
        _trajectory_parity(g, p, live, logL, k, 3 * d, seed=3, it=0, w=w)
        # a later iteration, compressed population
        live2 = live * 0.1
        logL2 = p.loglike_batch(live2)
        _trajectory_parity(g, p, live2, logL2, k, 3 * d, seed=3, it=7, w=w)
        g.close()


def test_iteration_above_the_counting_select_limit(nssmod, oracle):
    """More than 8192 live points: inside an iteration the ranks come from the sample sort (five k4s_* launches in front of
    k4_front, whose selection tail then finds ranks and dead list ready), the mean / covariance reduction runs in several
    blocks with a counter barrier, and 4500 single-warp chains are packed four to a CTA and fetched from the device
    counter.  Same checks as everywhere: dead list and rows bit-exact (a tenth of the logL values tied), trajectories of
    safe chains identical; then a complete (bounded) run on both sides."""
    w = inputs.gaussian_workload(5, sigma=0.07)
    g, p = nssmod.Nss(w), oracle.Problem(w)
    n, k = 9000, 4500
    live, logL = p.init_live(n, 21)
    live[::10] = live[3]                               # exact ties in logL: broken by slot
    logL = p.loglike_batch(live)
    r, o, safe = _trajectory_parity(g, p, live, logL, k, 6, seed=8, it=0, w=w)
    _trajectory_parity(g, p, o["live"], o["logL"], k, 3, seed=8, it=1, w=w)
    rg, ro = g.nss_run(n, k, 4, 5, max_iter=3), p.run(n, k, 4, 5, max_iter=3)
    assert rg["rc"] == nssmod.NSS_ENOTCONV and rg["n_iter"] == ro["n_iter"] == 3 and rg["n_dead"] == ro["n_dead"]
    assert abs(rg["logZ"] - ro["logZ"]) < 3 * math.hypot(rg["logZ_err"], ro["logZ_err"]) + 1e-9
    if _replays(rg, ro):
        _assert_replay(rg, ro, w)
    g.close()


def test_iteration_after_a_stand_alone_tune_on_the_same_handle(nssmod, oracle):
    """nss_tune with several tuning blocks (n_live >= 2048: a counter barrier and a ticket among them) followed by
    iterations on the SAME handle: the stand-alone kernel must leave the two counters at zero, else the next k4_front's
    barrier opens early and no block factors the covariance (stale Cholesky, no NSS_ECHOL).  5000 -> 3 blocks at the
    tune, then 4 blocks (4100 live points: a larger T than the counters' leftover) and 2 blocks in the iterations."""
    w = inputs.gaussian_workload(5, sigma=0.07)
    g, p = nssmod.Nss(w), oracle.Problem(w)
    live5, _ = p.init_live(5000, 31)
    rc, mean, chol = g.nss_tune(live5 * 0.3)                 # a different population: its factor must not be reused
    orc, omean, ocov, ochol = oracle.tune(live5 * 0.3)
    assert rc == 0 and np.allclose(chol.cpu().numpy(), ochol, rtol=1e-8, atol=1e-300)
    live, logL = p.init_live(4100, 32)
    r, o, safe = _trajectory_parity(g, p, live, logL, 2050, 4, seed=9, it=0, w=w)
    rc, mean, chol = g.nss_tune(live5)
    assert rc == 0
    live, logL = p.init_live(2100, 33)
    st = nssmod.nss_iter_state(logX=0.0, logZ=-math.inf)
    import torch
    dl, dL = torch.as_tensor(live, device="cuda").clone(), torch.as_tensor(logL, device="cuda").clone()
    bufs = g.iter_buffers(1050)
    g.nss_iterate(dl, dL, 1050, 4, 9, 0, st, bufs)
    o = p.replace_step(live, logL, 1050, 4, 9, 0, want_trace=True)
    safe = o["margin"] > 1e-6
    didx = o["dead_idx"]
    assert np.array_equal(bufs[3].cpu().numpy(), didx) and st.logLstar == o["logLstar"]
    assert safe.mean() > 0.97
    assert np.all(np.abs(dl.cpu().numpy()[didx][safe] - o["live"][didx][safe]) <= 1e-9 * (w.hi - w.lo))
    g.close()


def test_replace_step_trajectories_config1(nssmod, oracle, wl1):
    g, p = nssmod.Nss(wl1), oracle.Problem(wl1)
    live, logL = p.init_live(100, 1)
    state = (live, logL)
    for it in range(3):                                   # follow the oracle's own state (teacher forcing)
        r, o, safe = _trajectory_parity(g, p, state[0], state[1], 50, 12, seed=1, it=it, w=wl1, max_excluded=0.06)
        state = (o["live"], o["logL"])
    g.close()


def test_replace_step_trajectories_config2_and_teacher_forced_threshold(nssmod, oracle, wl2):
    g, p = nssmod.Nss(wl2), oracle.Problem(wl2)
    live, logL = p.init_live(1000, 2)
    r, o, safe = _trajectory_parity(g, p, live, logL, 500, 6, seed=2, it=0, w=wl2)
    # teacher-forced threshold below the internal one: same deletions, looser constraint
    forced = o["logLstar"] - 5.0
    _trajectory_parity(g, p, live, logL, 500, 3, seed=2, it=1, logLstar=forced, w=wl2)
    # a survivor below the supplied threshold is rejected on both sides
    bad = float(np.max(logL))
    assert p.replace_step(live, logL, 500, 1, 2, 0, logLstar=bad)["rc"] == -2
    assert g.nss_replace_step(live, logL, 500, 1, 2, 0, logLstar=bad, ok=(nssmod.NSS_EINVAL,))["rc"] == nssmod.NSS_EINVAL
    g.close()


@pytest.mark.parametrize("n_live,n_delete", [(1000, 500), (5000, 2500)])
def test_replace_step_full_size_bench_configuration(nssmod, oracle, wl2, n_live, n_delete):
    """BASELINE configs[1] and configs[2] at full size, in the launch configuration bench.py times (all 55 slice
    repeats, automatic lanes / warps per chain): one NS iteration from the initial live set and one from a population
    three iterations in, every chain against the oracle's trajectory (A20: chains whose margins exceed the logL tolerance)."""
    g, p = nssmod.Nss(wl2), oracle.Problem(wl2)
    live, logL = p.init_live(n_live, 4)
    r, o, safe = _trajectory_parity(g, p, live, logL, n_delete, 55, seed=4, it=0, w=wl2, max_excluded=0.05)
    live, logL = o["live"], o["logL"]
    for it in (1, 2):
        o = p.replace_step(live, logL, n_delete, 8, 4, it)
        live, logL = o["live"], o["logL"]
    _trajectory_parity(g, p, live, logL, n_delete, 55, seed=4, it=3, w=wl2, max_excluded=0.05)
    g.close()


def test_replace_step_full_grid_kind(nssmod, oracle):
    w = inputs.make_data(inputs.config4(), oracle.waveform)
    g, p = nssmod.Nss(w), oracle.Problem(w)
    live, logL = p.init_live(64, 5)
    _trajectory_parity(g, p, live, logL, 32, 2, seed=5, it=0, w=w, max_excluded=0.1)
    g.close()


def test_replace_step_full_grid_at_the_bench_launch_shape(nssmod, oracle):
    """BASELINE configs[3] (full frequency grid, 4017 bins x 3 detectors) at n_live 1000 / n_delete 500: K3's
    NSS_KIND_FULL instantiation in its real launch shape (500 one-chain CTAs), 11 slice repeats instead of 55 so that
    the oracle's 12 051-term sums stay affordable; every chain against the oracle's trajectory, from the prior-wide
    population and from a compressed one."""
    w = inputs.make_data(inputs.config4(), oracle.waveform)
    g, p = nssmod.Nss(w), oracle.Problem(w)
    live, logL = p.init_live(1000, 6)
    r, o, safe = _trajectory_parity(g, p, live, logL, 500, 11, seed=6, it=0, w=w, max_excluded=0.05)
    live, logL = o["live"], o["logL"]
    o = p.replace_step(live, logL, 500, 2, 6, 1)
    _trajectory_parity(g, p, o["live"], o["logL"], 500, 3, seed=6, it=2, w=w, max_excluded=0.05)
    g.close()


@pytest.mark.parametrize("B", [256, 1024])
def test_replace_step_and_run_at_many_bins(nssmod, oracle, wl2, B):
    """Config-2 geometry with 256 and 1024 bins per detector (BASELINE configs[4]'s bin counts, inside the sampler this
    time).  At B = 1024 the 8-lane table is not built and no lane count's table fits the 64 KB shared-memory budget, so
    K3 runs its RESIDENT = false instantiations (records read through L2) and a request for 8 lanes falls back to the
    automatic choice; at B = 256 the 8- and 16-lane tables fit and the 32-lane one is the largest resident table.
    Every lane setting must reproduce the oracle's trajectories; then a bounded run on both sides."""
    g, p = nssmod.Nss(wl2, n_bins=B), oracle.Problem(wl2, n_bins=B)
    n, k, nrep = 400, 200, 6
    live, logL = p.init_live(n, 12)
    o0 = p.replace_step(live, logL, k, nrep, 12, 0, want_trace=True)
    live1, logL1 = o0["live"], o0["logL"]
    for it in (1, 2):                              # a compressed population as the second case
        oo = p.replace_step(live1, logL1, k, 3, 12, it)
        live1, logL1 = oo["live"], oo["logL"]
    o1 = p.replace_step(live1, logL1, k, nrep, 12, 3, want_trace=True)
    for lanes in (0, 8, 16, 32):
        g.set_chain_lanes(lanes)
        for warps in ((0, 1) if lanes in (0, 32) else (0,)):
            g.set_chain_warps(warps)
            _trajectory_parity(g, p, live, logL, k, nrep, seed=12, it=0, w=wl2, max_excluded=0.05, o=o0)
            _trajectory_parity(g, p, live1, logL1, k, nrep, seed=12, it=3, w=wl2, max_excluded=0.05, o=o1)
    g.set_chain_lanes(0); g.set_chain_warps(0)
    rg, ro = g.nss_run(n, k, nrep, 13, max_iter=3), p.run(n, k, nrep, 13, max_iter=3)
    assert rg["rc"] == nssmod.NSS_ENOTCONV and rg["n_iter"] == ro["n_iter"] == 3 and rg["n_dead"] == ro["n_dead"]
    assert abs(rg["logZ"] - ro["logZ"]) < 3 * math.hypot(rg["logZ_err"], ro["logZ_err"]) + 1e-9
    if _replays(rg, ro):
        _assert_replay(rg, ro, wl2)
    g.close()


def test_results_do_not_depend_on_what_earlier_calls_left_in_the_handle(nssmod, wl1):
    """compute-sanitizer is closed on the build pool (profiles/r03_sanitizer.md), so the question initcheck would answer
    is asked directly: a handle's scratch (rank counts, sample-sort buffers, tuning partials, control block, run block)
    is reused across calls of different sizes and never cleared by the host.  A run and an iteration on a handle that
    has just served larger and different work (9000-live sample-sort iteration, a stand-alone tune, a bounded run, a
    Cholesky failure) must give the same BITS as on a fresh handle — anything read before it is written would differ."""
    import torch
    wg = inputs.gaussian_workload(4, sigma=0.06)

    def work(g):
        r = g.nss_run(300, 150, 8, 17, want_equal=True)
        live, logL = g.nss_init_live(257, 18)
        st = nssmod.nss_iter_state(logX=0.0, logZ=-math.inf)
        bufs = g.iter_buffers(100)
        g.nss_iterate(live, logL, 100, 5, 18, 0, st, bufs)
        dead, surv, ls = g.nss_select_lowest(logL, 31)
        return (r["logZ"], r["logZ_err"], r["H"], r["ess"], r["n_evals"], r["dead_theta"].tobytes(), r["dead_logw"].tobytes(),
                r["dead_logL_birth"].tobytes(), r["equal_idx"].tobytes(), live.cpu().numpy().tobytes(), logL.cpu().numpy().tobytes(),
                tuple(b.cpu().numpy().tobytes() for b in bufs), (st.logX, st.logZ, st.logZ_live, st.logLstar, st.n_evals),
                dead.cpu().numpy().tobytes(), surv.cpu().numpy().tobytes(), ls)

    fresh = nssmod.Nss(wg)
    want = work(fresh)
    fresh.close()
    g = nssmod.Nss(wg)
    live, logL = g.nss_init_live(9000, 3)                      # sample-sort buffers, eight tuning blocks, packed chains
    st = nssmod.nss_iter_state(logX=-5.0, logZ=-40.0)
    g.nss_iterate(live, logL, 4500, 2, 3, 0, st, g.iter_buffers(4500))
    g.nss_tune(live[:5000])
    g.nss_run(2000, 1000, 3, 4, max_iter=2)
    flat = torch.rand(60, 4, dtype=torch.float64, device="cuda") * 0.1
    flat[:, 1] = 0.25                                          # exactly zero variance (0.25 sums exactly): NSS_ECHOL, flags left set
    fl = g.nss_loglike_batch(flat)
    assert g.nss_replace_step(flat, fl, 30, 2, 1, 0, ok=(nssmod.NSS_ECHOL,))["rc"] == nssmod.NSS_ECHOL
    got = work(g)
    assert got == want
    assert work(g) == want                                      # and again on the now twice-used handle
    g.close()


def test_replace_step_degenerate_population_reports_cholesky(nssmod, oracle):
    w = inputs.gaussian_workload(3)
    g = nssmod.Nss(w)
    live = np.random.default_rng(0).uniform(-1, 1, size=(50, 3))
    live[:, 2] = 0.25
    logL = oracle.Problem(w).loglike_batch(live)
    r = g.nss_replace_step(live, logL, 25, 2, 1, 0, ok=(nssmod.NSS_ECHOL,))
    assert r["rc"] == nssmod.NSS_ECHOL
    assert np.array_equal(r["live"].cpu().numpy(), live)             # nothing was replaced
    g.close()


def _analytic_logz(d, sigma, half):
    c = scipy.stats.norm.cdf(half / sigma) - scipy.stats.norm.cdf(-half / sigma)
    return d * math.log(sigma * math.sqrt(2 * math.pi) / (2 * half) * c)


@pytest.mark.parametrize("d,n,k,seed", [(4, 1000, 500, 1), (11, 600, 300, 3)])
def test_run_gaussian_matches_oracle_and_analytic(nssmod, oracle, d, n, k, seed):
    w = inputs.gaussian_workload(d, sigma=0.05)
    g, p = nssmod.Nss(w), oracle.Problem(w)
    r = g.nss_run(n, k, 5 * d, seed)
    o = p.run(n, k, 5 * d, seed)
    truth = _analytic_logz(d, 0.05, 1.0)
    assert r["rc"] == 0
    assert abs(r["logZ"] - truth) < 3 * r["logZ_err"]
    assert abs(r["logZ"] - o["logZ"]) < 3 * math.hypot(r["logZ_err"], o["logZ_err"])
    assert abs(r["n_iter"] - o["n_iter"]) <= 1
    assert r["logZ_err"] == pytest.approx(o["logZ_err"], rel=0.3)
    assert r["H"] == pytest.approx(o["H"], abs=0.5)
    nd, ni = r["n_dead"], r["n_iter"]
    assert nd == ni * k + n
    assert np.sum(np.exp(r["dead_logw"])) == pytest.approx(1.0, abs=1e-10)
    dl = r["dead_logL"]
    assert np.all(np.diff(dl[:ni * k].reshape(ni, k), axis=1) >= 0) and np.all(np.diff(dl[ni * k:]) >= 0)
    assert np.all(r["dead_logL_birth"] < dl)
    pw = np.exp(dl + r["dead_logw"] - r["logZ"])
    ess = 1.0 / np.sum(pw ** 2)
    mean = pw @ r["dead_theta"]
    sd = np.sqrt(pw @ (r["dead_theta"] - mean) ** 2)
    assert np.all(np.abs(mean) < 5 * 0.05 / math.sqrt(ess)) and np.all(np.abs(sd / 0.05 - 1) < 0.15)
    g.close()


def _replays(r, o):
    """True when the GPU run made the oracle's decisions: same dead rows (logL within the logL tolerance)."""
    return r["n_dead"] == o["n_dead"] and bool(np.allclose(r["dead_logL"], o["dead_logL"], rtol=1e-9, atol=1e-6))


def _assert_replay(r, o, w):
    """What a replayed run must satisfy beyond _replays: same iterations, same sequential evaluation count, same rows
    (positions within 1e-9 of the prior width, A20)."""
    assert r["n_iter"] == o["n_iter"] and r["n_evals"] == o["n_evals"]
    assert np.allclose(r["dead_logw"], o["dead_logw"], rtol=0, atol=1e-9)
    assert r["logZ"] == pytest.approx(o["logZ"], abs=1e-6)
    assert np.allclose(r["dead_logL_birth"], o["dead_logL_birth"], rtol=1e-9, atol=1e-6)
    assert np.all(np.abs(r["dead_theta"] - o["dead_theta"]) <= 1e-9 * (w.hi - w.lo))


def _weights(res):
    a = res["dead_logL"] + res["dead_logw"]
    pw = np.exp(a - a.max())
    return pw / pw.sum()


def test_run_config1_matches_oracle(nssmod, oracle, wl1):
    """End to end on config 1 over its seed ensemble: logZ within 3 sigma_NS and posterior means within 0.1 sigma of the
    oracle's posterior width, asserted for every seed whether or not the run replayed (north_star); and every seed is
    expected to replay the oracle decision for decision (|logL_GPU - logL_oracle| ~ 1e-11 against ~1e5 bracket tests)."""
    g, p = nssmod.Nss(wl1), oracle.Problem(wl1)
    exact = 0
    for seed in (1, 2, 3, 4):
        r = g.nss_run(100, 50, 12, seed)
        o = p.run(100, 50, 12, seed)
        assert r["rc"] == 0 and o["rc"] == 0
        assert abs(r["logZ"] - o["logZ"]) < 3 * math.hypot(r["logZ_err"], o["logZ_err"])
        pg, po = _weights(r), _weights(o)
        mg, mo = pg @ r["dead_theta"], po @ o["dead_theta"]
        so = np.sqrt(po @ (o["dead_theta"] - mo) ** 2)
        assert np.all(np.abs(mg - mo) < 0.1 * so)
        if _replays(r, o):
            exact += 1
            _assert_replay(r, o, wl1)
    print(f"[config 1] {exact} of 4 seeds replayed the oracle's run decision for decision")
    assert exact >= 3
    g.close()


def test_run_seed_ensemble_replays_the_oracle(nssmod, oracle, wl1):
    """The seed-ensemble check behind DESIGN.md §5's replay claim: 16 seeds of config 1 and 8 seeds of a 5-dimensional
    Gaussian, each a whole run to the stop rule on both sides.  Every run must agree in logZ within 3 sigma_NS, and at
    least 7 in 8 must be the oracle's run decision for decision (a flip needs a bracket test within ~1e-11 of L*)."""
    g, p = nssmod.Nss(wl1), oracle.Problem(wl1)
    exact, worst = 0, 0.0
    for seed in range(100, 116):
        r, o = g.nss_run(100, 50, 12, seed), p.run(100, 50, 12, seed)
        worst = max(worst, abs(r["logZ"] - o["logZ"]) / math.hypot(r["logZ_err"], o["logZ_err"]))
        if _replays(r, o):
            exact += 1
            _assert_replay(r, o, wl1)
    g.close()
    print(f"[ensemble] config 1: {exact} of 16 seeds replayed; worst |dlogZ| / sigma = {worst:.3f}")
    assert worst < 3.0 and exact >= 14
    w = inputs.gaussian_workload(5, sigma=0.07)
    g, p = nssmod.Nss(w), oracle.Problem(w)
    exact, worst = 0, 0.0
    for seed in range(200, 208):
        r, o = g.nss_run(500, 250, 15, seed), p.run(500, 250, 15, seed)
        worst = max(worst, abs(r["logZ"] - o["logZ"]) / math.hypot(r["logZ_err"], o["logZ_err"]))
        if _replays(r, o):
            exact += 1
            _assert_replay(r, o, w)
    g.close()
    print(f"[ensemble] 5-d Gaussian: {exact} of 8 seeds replayed; worst |dlogZ| / sigma = {worst:.3f}")
    assert worst < 3.0 and exact >= 7


def test_run_statistical_parity_on_independent_seeds(nssmod, oracle):
    """north_star's statistical criteria on runs that do NOT share a trajectory: the GPU run uses seed 11, the oracle
    seeds 12 and 13 (different Philox streams from the first draw on).  4-d Gaussian, n_live 4000 so that the Monte-Carlo
    error of a posterior mean (sigma / sqrt(ESS), ESS ~ 1e4) is ~ 0.01 sigma and 0.1 sigma is a real bar: logZ within
    3 sigma_NS of each other and of the analytic value, means within 0.1 sigma, widths within 5 %."""
    w = inputs.gaussian_workload(4, sigma=0.05)
    g, p = nssmod.Nss(w), oracle.Problem(w)
    r = g.nss_run(4000, 2000, 20, 11)
    truth = _analytic_logz(4, 0.05, 1.0)
    assert abs(r["logZ"] - truth) < 3 * r["logZ_err"]
    pg = _weights(r)
    mg = pg @ r["dead_theta"]
    sg = np.sqrt(pg @ (r["dead_theta"] - mg) ** 2)
    for seed in (12, 13):
        o = p.run(4000, 2000, 20, seed)
        assert not _replays(r, o)
        assert abs(r["logZ"] - o["logZ"]) < 3 * math.hypot(r["logZ_err"], o["logZ_err"])
        po = _weights(o)
        mo = po @ o["dead_theta"]
        so = np.sqrt(po @ (o["dead_theta"] - mo) ** 2)
        assert np.all(np.abs(mg - mo) < 0.1 * so)
        assert np.all(np.abs(sg / so - 1) < 0.05)
    g.close()


def _config2_summary(res):
    """Posterior means / widths of the quantities SURVEY.md §8(d) says to compare on config 2: Mc, q, the spin
    combination beta that enters the phase (chi_1, chi_2 are individually unconstrained), d_L, t_c, iota, ra, dec as
    plain means; phi_c (period 2 pi) and psi (period pi) as circular means.  Returns (values, widths, is_circular, period)."""
    th, pw = res["dead_theta"], _weights(res)
    q = th[:, 1]
    eta = q / (1 + q) ** 2
    m1, m2 = 1 / (1 + q), q / (1 + q)
    beta = (113 / 12 * m1 ** 2 + 25 / 4 * eta) * th[:, 2] + (113 / 12 * m2 ** 2 + 25 / 4 * eta) * th[:, 3]
    cols = [th[:, 0], q, beta, th[:, 4], th[:, 5], th[:, 7], th[:, 9], th[:, 10]]
    mean = np.array([pw @ c for c in cols])
    sd = np.array([math.sqrt(pw @ (c - m) ** 2) for c, m in zip(cols, mean)])
    circ = []
    for col, period in ((th[:, 6], 2 * math.pi), (th[:, 8], math.pi)):
        z = pw @ np.exp(2j * math.pi * col / period)
        circ.append((np.angle(z) * period / (2 * math.pi), math.sqrt(max(-2 * math.log(abs(z)), 0.0)) * period / (2 * math.pi), period))
    return mean, sd, circ


@pytest.mark.parametrize("seed", [1, 2])
def test_run_config2_matches_oracle(nssmod, oracle, wl2, seed):
    """north_star's Target: a whole NSS run on the 11-parameter, 3-detector heterodyned workload (BASELINE configs[1]:
    n_live 1000, n_delete 500, 55 repeats) to the stop rule on both sides.  Unconditionally: |dlogZ| < 3 hypot(sigma_GPU,
    sigma_oracle); posterior means of Mc, q, beta, d_L, t_c, iota, ra, dec within 0.1 of the oracle's posterior width;
    phi_c and psi compared as wrapped angles.  And the run is expected to replay: same iterations, same sequential
    evaluation count, same dead rows."""
    g, p = nssmod.Nss(wl2), oracle.Problem(wl2)
    import time
    t0 = time.perf_counter()
    r = g.nss_run(1000, 500, 55, seed)
    t1 = time.perf_counter()
    o = p.run(1000, 500, 55, seed)
    t2 = time.perf_counter()
    print(f"[config 2, seed {seed}] GPU {t1 - t0:.3f} s, oracle {t2 - t1:.1f} s on {oracle.n_cores()} cores; n_iter {r['n_iter']} / {o['n_iter']}, "
          f"n_evals {r['n_evals']} / {o['n_evals']}, logZ {r['logZ']:.4f} +- {r['logZ_err']:.3f} / {o['logZ']:.4f} +- {o['logZ_err']:.3f}")
    assert r["rc"] == 0 and o["rc"] == 0
    assert abs(r["logZ"] - o["logZ"]) < 3 * math.hypot(r["logZ_err"], o["logZ_err"])
    assert r["H"] == pytest.approx(o["H"], abs=0.5)
    mg, sg, cg = _config2_summary(r)
    mo, so, co = _config2_summary(o)
    assert np.all(np.abs(mg - mo) < 0.1 * so), (mg, mo, so)
    for (ag, wg, per), (ao, wo, _) in zip(cg, co):
        dist = abs((ag - ao + per / 2) % per - per / 2)
        assert dist < 0.1 * wo
    replay = _replays(r, o)
    print(f"[config 2, seed {seed}] replayed decision for decision: {replay}")
    assert replay, "config 2 is expected to replay (a flip needs a bracket test within ~1e-10 of L*)"
    _assert_replay(r, o, wl2)
    g.close()


def test_run_config3_bounded_matches_oracle(nssmod, oracle, wl2):
    """BASELINE configs[2] (n_live 5000, n_delete 2500, 55 repeats: 2500 concurrent chains) through nss_run for two NS
    iterations (NSS_ENOTCONV: results valid) against the oracle's truncated run: same rows, weights and evidence."""
    g, p = nssmod.Nss(wl2), oracle.Problem(wl2)
    cap = 5000 + 2 * 2500
    r = g.nss_run(5000, 2500, 55, 3, max_iter=2, cap=cap)
    o = p.run(5000, 2500, 55, 3, max_iter=2, cap=cap)
    assert r["rc"] == nssmod.NSS_ENOTCONV and o["rc"] == 1
    assert r["n_iter"] == o["n_iter"] == 2 and r["n_dead"] == o["n_dead"] == cap
    assert abs(r["logZ"] - o["logZ"]) < 3 * math.hypot(r["logZ_err"], o["logZ_err"]) + 1e-6
    assert _replays(r, o)
    _assert_replay(r, o, wl2)
    g.close()


def test_run_config4_bounded_matches_oracle(nssmod, oracle):
    """BASELINE configs[3] (full-grid likelihood, n_live 1000, n_delete 500) through nss_run: two NS iterations with 11
    slice repeats against the oracle's truncated run."""
    w = inputs.make_data(inputs.config4(), oracle.waveform)
    g, p = nssmod.Nss(w), oracle.Problem(w)
    cap = 1000 + 2 * 500
    r = g.nss_run(1000, 500, 11, 4, max_iter=2, cap=cap)
    o = p.run(1000, 500, 11, 4, max_iter=2, cap=cap)
    assert r["rc"] == nssmod.NSS_ENOTCONV and o["rc"] == 1
    assert r["n_iter"] == o["n_iter"] == 2 and r["n_dead"] == o["n_dead"] == cap
    assert abs(r["logZ"] - o["logZ"]) < 3 * math.hypot(r["logZ_err"], o["logZ_err"]) + 1e-6
    assert _replays(r, o)
    _assert_replay(r, o, w)
    g.close()


@pytest.mark.parametrize("n_delete", [1, 7, 25, 75])
def test_run_delete_fraction_sweep_matches_oracle(nssmod, oracle, wl1, n_delete):
    """The n_delete axis of the paper's Fig. 2 (right panel): one chain per iteration up to three
    quarters of the live set.  Same seed -> the oracle's run, decision for decision, until a near-threshold test flips;
    always logZ within 3 sigma_NS, and the bookkeeping invariant sum(w) + X_end = 1 (P14) at every delete fraction."""
    g, p = nssmod.Nss(wl1), oracle.Problem(wl1)
    r = g.nss_run(100, n_delete, 12, 5, max_iter=100000, cap=100 * 60)
    o = p.run(100, n_delete, 12, 5, max_iter=100000, cap=100 * 60)
    assert r["rc"] == 0 and o["rc"] == 0
    assert abs(r["logZ"] - o["logZ"]) < 3 * math.hypot(r["logZ_err"], o["logZ_err"])
    assert np.all(np.diff(r["dead_logL"][: r["n_dead"] - 100]) >= 0)           # dead points leave in ascending logL
    assert np.exp(r["dead_logw"]).sum() == pytest.approx(1.0, abs=1e-9)        # dead + final live weights exhaust the prior
    replay = _replays(r, o)
    print(f"[delete-fraction sweep] n_delete={n_delete}: replayed {replay}")
    assert replay, "every point of the sweep replayed the oracle on B200 when this test was written"
    _assert_replay(r, o, wl1)
    g.close()


def test_iterate_device_and_host_forms_match_oracle(nssmod, oracle, wl1):
    """nss_iterate = replace step + evidence bookkeeping + live evidence (all §8(a) rows); the host-buffer
    form returns the same bits as the device form."""
    import torch
    g, p = nssmod.Nss(wl1), oracle.Problem(wl1)
    n, k, nrep = 100, 50, 12
    live, logL = p.init_live(n, 4)
    st = nssmod.nss_iter_state(logX=0.0, logZ=-math.inf)
    sth = nssmod.nss_iter_state(logX=0.0, logZ=-math.inf)
    dl, dL = torch.as_tensor(live, device="cuda").clone(), torch.as_tensor(logL, device="cuda").clone()
    hl, hL = torch.as_tensor(live).clone().pin_memory(), torch.as_tensor(logL).clone().pin_memory()
    bufs, hbufs = g.iter_buffers(k), g.iter_buffers(k, host=True)
    ol, oL, ox, oz = live, logL, 0.0, -math.inf
    for it in range(3):
        g.nss_iterate(dl, dL, k, nrep, 4, it, st, bufs)
        g.nss_iterate(hl, hL, k, nrep, 4, it, sth, hbufs, host=True)
        assert torch.equal(dl.cpu(), hl) and torch.equal(dL.cpu(), hL)
        for a, b in zip(bufs, hbufs):
            assert torch.equal(a.cpu(), b)
        assert (st.logX, st.logZ, st.logZ_live, st.logLstar, st.n_evals) == \
               (sth.logX, sth.logZ, sth.logZ_live, sth.logLstar, sth.n_evals)
        # oracle, teacher-forced from the GPU's own pre-step state
        o = p.replace_step(ol, oL, k, nrep, 4, it, want_trace=True)
        ox, oz, olw = oracle.evidence_update(o["dead_logL"], n, ox, oz)
        assert np.array_equal(bufs[3].cpu().numpy(), o["dead_idx"])
        assert np.array_equal(bufs[1].cpu().numpy(), o["dead_logL"])
        assert np.allclose(bufs[2].cpu().numpy(), olw, rtol=0, atol=1e-9)
        assert st.logLstar == o["logLstar"]
        assert st.logX == pytest.approx(ox, abs=1e-12) and st.logZ == pytest.approx(oz, abs=1e-9)
        gl = dL.cpu().numpy()
        lzl = st.logX + scipy.special.logsumexp(gl) - math.log(n)
        assert st.logZ_live == pytest.approx(lzl, abs=1e-9)
        assert st.converged == int(st.logZ_live - st.logZ < -3.0)
        ol, oL = dl.cpu().numpy(), gl                    # follow the GPU state
    # host-buffer likelihood form
    X = torch.as_tensor(inputs.draw_prior(wl1, 777, 3)).pin_memory()
    out = torch.empty(777, dtype=torch.float64).pin_memory()
    g.nss_loglike_batch_host(X, out)
    assert torch.equal(out, g.nss_loglike_batch(X.cuda()).cpu())
    g.close()


@pytest.mark.parametrize("cfg", ["gauss", "config1", "config2", "config4"])
def test_chain_group_width_does_not_change_the_trajectory(nssmod, oracle, wl1, wl2, cfg):
    """K3 runs a chain on G = 1, 2, 4 or 8 warps whose sub-warps (8, 16 or 32 lanes per candidate) evaluate the
    next bracket tests speculatively.  For a given lane count the decisions, positions, logL and the
    sequential-algorithm evaluation count must be the same bits for every G (32 lanes, G = 1 is the plain
    sequential algorithm).  Across lane counts logL differs by summation order only, so every chain that clears
    the threshold by more than the logL tolerance (A20) must make the same decisions and end at the same bits.
    Single-warp chains are packed 1, 3 or 8 to a CTA and take their chains from a device counter (nss_set_chain_pack):
    which warp runs which chain, and when, must not matter either."""
    if cfg == "gauss":
        w, n, k, nrep = inputs.gaussian_workload(6, sigma=0.05), 300, 150, 40
    elif cfg == "config1":
        w, n, k, nrep = wl1, 100, 50, 12
    elif cfg == "config4":                           # the full-grid kind: 32 lanes per candidate only, table read from L2
        w, n, k, nrep = inputs.make_data(inputs.config4(), oracle.waveform), 96, 48, 12
    else:
        w, n, k, nrep = wl2, 400, 200, 35            # 35 repeats: crosses the 32-step direction chunk
    g, p = nssmod.Nss(w), oracle.Problem(w)
    live, logL = p.init_live(n, 11)
    if cfg != "gauss":                                # a compressed population: brackets expand and shrink a lot
        for it in range(4):
            o = p.replace_step(live, logL, k, 3, 11, it)
            live, logL = o["live"], o["logL"]
    first = None
    for L in ((32,) if cfg in ("gauss", "config4") else (32, 16, 8)):
        g.set_chain_lanes(L)
        ref = None
        for G, pack in ((1, 1), (1, 3), (1, 8), (2, 0), (4, 0), (8, 0), (0, 0)):
            g.set_chain_warps(G)
            g.set_chain_pack(pack)
            r = g.nss_replace_step(live, logL, k, nrep, 11, 9, want_trace=True)
            cur = (r["live"].cpu().numpy(), r["logL"].cpu().numpy(), r["trace"].cpu().numpy(), r["margin"].cpu().numpy(),
                   r["n_evals"], r["dead_idx"].cpu().numpy())
            if ref is None:
                ref = cur
                assert ref[2][:, :, 0].max() > 0 or ref[2][:, :, 1].max() > 0      # some brackets did step out
                assert ref[2][:, :, 2].max() >= 4                                    # and some shrank several times
            else:
                for a, b in zip(ref[:4], cur[:4]):
                    assert np.array_equal(a, b), f"lanes={L} G={G} pack={pack} changed the result"
                assert ref[4] == cur[4]
        if first is None:
            first = ref
        else:
            safe = np.minimum(first[3], ref[3]) > 1e-6
            assert safe.mean() > 0.9
            assert np.array_equal(first[2][safe], ref[2][safe]), f"lanes={L} changed a decision"
            d = first[5]
            assert np.array_equal(first[0][d][safe], ref[0][d][safe]), f"lanes={L} changed a position"
            assert np.allclose(first[1][d][safe], ref[1][d][safe], rtol=1e-9, atol=1e-6)
    g.set_chain_lanes(0)
    # the K3 event pair is off by default and can be switched on (bench.py's kernel-timed pass)
    with pytest.raises(nssmod.NssError):
        g.nss_last_chain_ms()
    g.set_chain_timing(True)
    g.nss_replace_step(live, logL, k, 2, 11, 9)
    assert g.nss_last_chain_ms() > 0.0
    g.set_chain_timing(False)
    g.close()


# ---- NEXT-2: periodic coordinates (nss_set_periodic) -------------------------------------------------------------------
@pytest.mark.parametrize("cfg", ["gauss", "config1", "config2"])
def test_next2_periodic_trajectories_match_oracle(nssmod, oracle, wl1, wl2, cfg):
    """Wrapped phi_c (config 1), phi_c / psi / ra (config 2), or two of four coordinates of the Gaussian test problem:
    every chain against the oracle's trajectory, from the prior-wide population (where slices cross the seam all the
    time) and from a compressed one; then the flags switch off again."""
    if cfg == "gauss":
        w, n, k, nrep = inputs.gaussian_workload(4, sigma=0.3), 600, 300, 12
        flags = [1, 0, 1, 0]
    elif cfg == "config1":
        w, n, k, nrep = wl1, 100, 50, 12
        flags = [0, 0, 0, 1]
    else:
        w, n, k, nrep = wl2, 1000, 500, 20
        flags = [0, 0, 0, 0, 0, 0, 1, 0, 1, 1, 0]
    g, p = nssmod.Nss(w), oracle.Problem(w)
    g.nss_set_periodic(flags)
    p.set_periodic(flags)
    live, logL = p.init_live(n, 6)
    r, o, safe = _trajectory_parity(g, p, live, logL, k, nrep, seed=6, it=0, w=w, max_excluded=0.06)
    moved = o["live"][o["dead_idx"]]
    assert np.all(moved >= w.lo) and np.all(moved <= w.hi)
    # the wrapped run differs from the walled one (some slice crossed a seam), on both sides alike
    p.set_periodic(np.zeros(w.d, dtype=int))
    walls = p.replace_step(live, logL, k, nrep, 6, 0)
    assert not np.array_equal(walls["live"], o["live"])
    p.set_periodic(flags)
    live, logL = o["live"], o["logL"]
    for it in (1, 2):
        o = p.replace_step(live, logL, k, 4, 6, it)
        live, logL = o["live"], o["logL"]
    _trajectory_parity(g, p, live, logL, k, nrep, seed=6, it=3, w=w, max_excluded=0.06)
    # lane / warp counts do not change a wrapped trajectory either
    ref = None
    for L, G in ((32, 1), (16, 2), (8, 1), (0, 0)):
        if cfg == "gauss" and L not in (32, 0):
            continue
        g.set_chain_lanes(L); g.set_chain_warps(G)
        rr = g.nss_replace_step(live, logL, k, nrep, 6, 4, want_trace=True)
        cur = (rr["trace"].cpu().numpy(), rr["live"].cpu().numpy(), rr["margin"].cpu().numpy(), rr["dead_idx"].cpu().numpy())
        if ref is None:
            ref = cur
        else:
            ok = np.minimum(ref[2], cur[2]) > 1e-6
            assert np.array_equal(ref[0][ok], cur[0][ok]) and np.array_equal(ref[1][ref[3]][ok], cur[1][cur[3]][ok])
    g.set_chain_lanes(0); g.set_chain_warps(0)
    g.nss_set_periodic(None)
    _trajectory_parity(g, oracle.Problem(w), live, logL, k, 3, seed=6, it=5, w=w, max_excluded=0.06)
    g.close()


@pytest.mark.parametrize("n", [600, 5000, 9000])
def test_next2_r7_tuning_of_a_seam_straddling_population_matches_oracle(nssmod, oracle, n):
    """Reading R7 (NEXT-2, second half): with periodic flags set, the tuning blocks unwrap every periodic coordinate around
    its circular mean before the two-pass moments.  A cloud sitting on the seam of two periodic coordinates, stored wrapped:
    mean and Cholesky factor against the oracle (one tuning block at n = 600, three and eight behind the extra counter barrier
    at 5000 and 9000), the covariance being that of the never-wrapped cloud; without flags the plain moments, as before; and
    an iteration on the same handle afterwards (the third counter is left at zero)."""
    rng = np.random.default_rng(n)
    w = inputs.gaussian_workload(4, sigma=0.05)
    g, p = nssmod.Nss(w), oracle.Problem(w)
    W = w.hi - w.lo
    A = np.array([[0.05, 0, 0, 0], [0.02, 0.04, 0, 0], [0.01, -0.03, 0.06, 0], [0.0, 0.01, 0.02, 0.03]])
    free = rng.normal(size=(n, 4)) @ A.T + np.array([0.2, w.hi[1] - 0.005, w.lo[2] + 0.01, -0.4])
    stored = w.lo + np.mod(free - w.lo, W)
    flags = [0, 1, 1, 0]
    g.nss_set_periodic(flags)
    rc, mean, chol = g.nss_tune(stored)
    orc, omean, ocov, ochol = oracle.tune_periodic(stored, flags, w.lo, w.hi)
    assert rc == 0 and orc == 0
    assert np.allclose(chol.cpu().numpy(), ochol, rtol=1e-8, atol=1e-300)
    assert np.allclose(mean.cpu().numpy(), omean, rtol=0, atol=1e-12)
    assert np.allclose(chol.cpu().numpy(), np.linalg.cholesky(np.cov(free.T)), rtol=1e-7)
    # a trajectory step from this population: both sides tune with R7 and wrap the two coordinates
    p.set_periodic(flags)
    logL = p.loglike_batch(stored)
    k = n // 2
    _trajectory_parity(g, p, stored, logL, k, 3, seed=6, it=0, w=w, max_excluded=0.05)
    g.nss_set_periodic(None)
    rc, mean, chol = g.nss_tune(stored)
    _, pmean, _, pchol = oracle.tune(stored)
    assert np.allclose(chol.cpu().numpy(), pchol, rtol=1e-8, atol=1e-300) and np.allclose(mean.cpu().numpy(), pmean, rtol=1e-13)
    g.close()


def test_next2_periodic_run_matches_oracle_and_analytic(nssmod, oracle):
    """End to end with wrapped coordinates: the Gaussian with its peak 0.2 sigma from a wall (O16's analytic logZ holds on
    the torus too), GPU against oracle and against the closed form."""
    w = inputs.gaussian_workload(3, sigma=0.05)
    w.gauss_mu = w.gauss_mu.copy()
    w.gauss_mu[0] = -0.99
    g, p = nssmod.Nss(w), oracle.Problem(w)
    g.nss_set_periodic([1, 1, 0])
    p.set_periodic([1, 1, 0])
    truth = sum(math.log(0.05 * math.sqrt(2 * math.pi) / 2.0
                         * (scipy.stats.norm.cdf((1 - m) / 0.05) - scipy.stats.norm.cdf((-1 - m) / 0.05))) for m in w.gauss_mu[:3])
    r, o = g.nss_run(1000, 500, 15, 3), p.run(1000, 500, 15, 3)
    assert r["rc"] == 0 and o["rc"] == 0
    assert abs(r["logZ"] - truth) < 3 * r["logZ_err"]
    assert abs(r["logZ"] - o["logZ"]) < 3 * math.hypot(r["logZ_err"], o["logZ_err"])
    replay = _replays(r, o)
    print(f"[periodic run] replayed {replay}")
    assert replay, "the wrapped Gaussian run replayed the oracle on B200 when this test was written"
    _assert_replay(r, o, w)
    g.close()


# ---- NEXT-4: Kish effective sample size (the paper's Table 1b metric; O15) -----------------------------
def _kish(logL, logw):
    a = logL + logw
    a = a[np.isfinite(a)]
    p = np.exp(a - a.max())
    return p.sum() ** 2 / (p * p).sum()


def test_next4_kish_ess_matches_the_formula_and_the_oracle(nssmod, oracle, wl1):
    """ESS = (sum p)^2 / sum p^2 over all returned rows, p ~ exp(logL + logw).  Closed forms pin the formula (equal
    weights -> N; one weight dominating -> 1); the library's device reduction must agree with it on the library's own
    rows, and with the oracle's rows wherever the two runs made the same decisions."""
    assert _kish(np.zeros(1000), np.full(1000, -3.0)) == pytest.approx(1000.0)
    assert _kish(np.array([0.0, -800.0, -900.0]), np.zeros(3)) == pytest.approx(1.0)
    g, p = nssmod.Nss(wl1), oracle.Problem(wl1)
    same = 0
    for seed in (1, 2, 3):
        r, o = g.nss_run(100, 50, 12, seed), p.run(100, 50, 12, seed)
        assert r["ess"] == pytest.approx(_kish(r["dead_logL"], r["dead_logw"]), rel=1e-10)
        assert 1.0 < r["ess"] < r["n_dead"]
        if r["n_dead"] == o["n_dead"] and np.allclose(r["dead_logL"], o["dead_logL"], rtol=1e-9, atol=1e-6):
            same += 1
            assert r["ess"] == pytest.approx(_kish(o["dead_logL"], o["dead_logw"]), rel=1e-6)
    assert same >= 1
    g.close()
    w = inputs.gaussian_workload(4, sigma=0.05)
    g = nssmod.Nss(w)
    r = g.nss_run(1000, 500, 20, 2)
    assert r["ess"] == pytest.approx(_kish(r["dead_logL"], r["dead_logw"]), rel=1e-10)
    g.close()


def test_next4_equal_weight_resampling_matches_oracle(nssmod, oracle, ggauss, wl1):
    """Reading R6 (the bracketed "equal weight samples" of PAPER.md:59-63): row i is kept iff u_i < p_i / p_max with the
    reserved Philox word.  Index work: the kept rows must be the oracle's, bit for bit — on synthetic weights (ties at the
    maximum, -inf rows, a ragged length spanning many threads' chunks, the empty and all--inf cases) and on the rows of a
    complete run, whose result struct must carry the same count and indices."""
    rng = np.random.default_rng(11)
    for n in (1, 31, 1025, 70001):
        logL = rng.normal(0.0, 3.0, n)
        logw = -np.sort(rng.exponential(2.0, n))[::-1] - np.arange(n) * (5.0 / n)
        logL[rng.integers(0, n, max(1, n // 50))] = -np.inf
        top = np.nanargmax(np.where(np.isfinite(logL), logL + logw, -np.inf))
        if n > 2:
            logL[(top + 1) % n] = logL[top] + logw[top] - logw[(top + 1) % n]      # a tie at the maximum
        for seed in (1, (7 << 32) | 9):
            want = oracle.resample_equal(logL, logw, seed)
            got = ggauss.nss_resample_equal(logL, logw, seed).cpu().numpy()
            assert np.array_equal(got, want), (n, seed)
            assert 1 <= got.size <= n or not np.isfinite(logL + logw).any()
    got = ggauss.nss_resample_equal(np.full(40, -np.inf), np.zeros(40), 3)
    assert got.numel() == 0 and oracle.resample_equal(np.full(40, -np.inf), np.zeros(40), 3).size == 0
    assert ggauss.nss_resample_equal(np.zeros(0), np.zeros(0), 3).numel() == 0
    # equal weights: every row has p = p_max and u < 1 always
    assert ggauss.nss_resample_equal(np.zeros(5000), np.full(5000, -2.0), 5).numel() == 5000
    g = nssmod.Nss(wl1)
    for seed in (1, 2):
        r = g.nss_run(100, 50, 12, seed, want_equal=True)
        want = oracle.resample_equal(r["dead_logL"], r["dead_logw"], seed)
        assert r["n_equal"] == want.size and np.array_equal(r["equal_idx"], want)
        assert 1 <= r["n_equal"] <= r["n_dead"]
        # expected size sum p / max p; the draw is a sum of independent Bernoullis
        a = r["dead_logL"] + r["dead_logw"]
        pk = np.exp(a - a.max())
        assert abs(r["n_equal"] - pk.sum()) < 5.0 * math.sqrt((pk * (1 - pk)).sum()) + 1.0
        assert g.nss_run(100, 50, 12, seed)["n_equal"] == r["n_equal"]          # without the index array
    g.close()


# ---- degenerate and extreme shapes ------------------------------------------------------------------------------------
def test_edge_shapes_match_oracle(nssmod, oracle, wl1):
    """n_repeats = 0 (chains just copy their start survivor), n_delete = n_live - 1 (one survivor seeds every chain),
    n_delete = 1, a one-dimensional problem, and a single relative-binning bin."""
    g, p = nssmod.Nss(wl1), oracle.Problem(wl1)
    live, logL = p.init_live(64, 9)
    r = g.nss_replace_step(live, logL, 32, 0, 9, 0)
    o = p.replace_step(live, logL, 32, 0, 9, 0)
    assert np.array_equal(r["live"].cpu().numpy(), o["live"]) and np.array_equal(r["logL"].cpu().numpy(), o["logL"])
    assert r["n_evals"] == o["n_evals"] == 0
    _trajectory_parity(g, p, live, logL, 63, 5, seed=9, it=1, w=wl1, max_excluded=0.1)
    _trajectory_parity(g, p, live, logL, 1, 12, seed=9, it=2, w=wl1, max_excluded=1.0)
    g.close()
    w = inputs.gaussian_workload(1, sigma=0.1)
    g, p = nssmod.Nss(w), oracle.Problem(w)
    live, logL = p.init_live(50, 3)
    _trajectory_parity(g, p, live, logL, 25, 7, seed=3, it=0, w=w)
    rr, oo = g.nss_run(50, 25, 5, 3), p.run(50, 25, 5, 3)
    assert abs(rr["logZ"] - oo["logZ"]) < 3 * math.hypot(rr["logZ_err"], oo["logZ_err"]) + 1e-9
    g.close()
    w1 = inputs.make_data(inputs.config1(n_bins=1), oracle.waveform)
    g, p = nssmod.Nss(w1), oracle.Problem(w1)
    X = inputs.draw_prior(w1, 300, 4)
    ref = p.loglike_batch(X)
    for variant in (1, 2):
        g.set_loglike_variant(variant)
        got = g.nss_loglike_batch(X).cpu().numpy()
        assert np.all(np.abs(got - ref) <= 1e-6 + 1e-9 * np.abs(ref))
    live, logL = p.init_live(40, 2)
    _trajectory_parity(g, p, live, logL, 20, 4, seed=2, it=0, w=w1, max_excluded=0.1)
    g.close()


@pytest.mark.parametrize("names", [("H1", "L1"), ("H1", "L1", "V1", "SYN")])
def test_two_and_four_detectors(nssmod, oracle, names):
    """The kernels are compiled per detector count (1..4): config 2 with two and with four detectors (the fourth is the
    synthetic one of config 1), relative binning and full grid, every batch variant and one NS iteration of chains."""
    import dataclasses
    base = inputs.config2(n_bins=64, n_live=200, n_delete=100)
    f = base.f_min + base.df * np.arange(base.n_freq)
    w = dataclasses.replace(base, det_names=names, det=inputs.detector_array(names),
                            psd=np.tile(inputs.psd_aligo_fit(f)[None, :], (len(names), 1)), data=None)
    w = inputs.make_data(w, oracle.waveform)
    X = np.concatenate([inputs.draw_prior(w, 1500, 5), inputs.draw_near(w, 150, 6, 0.01 * (w.hi - w.lo))])
    for kind in (0, 1):
        g, p = nssmod.Nss(w, kind=kind), oracle.Problem(w, kind=kind)
        n = len(X) if kind == 0 else 300
        ref = p.loglike_batch(X[:n])
        for variant in (1, 2):
            g.set_loglike_variant(variant)
            got = g.nss_loglike_batch(X[:n]).cpu().numpy()
            assert np.all(np.abs(got - ref) <= 1e-6 + 1e-9 * np.abs(ref))
        g.set_loglike_variant(0)
        if kind == 0:
            live, logL = p.init_live(200, 3)
            _trajectory_parity(g, p, live, logL, 100, 6, seed=3, it=0, w=w, max_excluded=0.06)
        g.close()


def test_run_stops_at_max_iter_and_reports_a_small_result_array(nssmod, oracle, wl1):
    """nss_run queues one iteration ahead of the host, so the exits other than convergence need their own check:
    max_iter (NSS_ENOTCONV, results valid and equal to the oracle's truncated run, nothing of a further iteration
    applied), max_iter = 0 (only the live points), and a result array that is too small (NSS_ECAP)."""
    g, p = nssmod.Nss(wl1), oracle.Problem(wl1)
    for mi in (3, 1, 0):
        r = g.nss_run(100, 50, 12, 2, max_iter=mi, cap=100 + 50 * max(mi, 1))
        o = p.run(100, 50, 12, 2, max_iter=mi, cap=100 + 50 * max(mi, 1))
        assert r["rc"] == nssmod.NSS_ENOTCONV and o["rc"] == 1
        assert r["n_iter"] == o["n_iter"] == mi and r["n_dead"] == o["n_dead"] == 100 + 50 * mi
        assert np.allclose(r["dead_logL"], o["dead_logL"], rtol=1e-9, atol=1e-6)
        assert r["logZ"] == pytest.approx(o["logZ"], abs=1e-6)
        assert np.allclose(r["dead_logw"], o["dead_logw"], rtol=0, atol=1e-9)
    import ctypes as C
    res = nssmod.nss_result()
    n = 100 + 50                                    # room for one iteration only; the run needs ~29
    bufs = [np.empty((n, wl1.d)), np.empty(n), np.empty(n), np.empty(n)]
    c_dp = C.POINTER(C.c_double)
    res.dead_theta, res.dead_logL, res.dead_logL_birth, res.dead_logw = (b.ctypes.data_as(c_dp) for b in bufs)
    res.cap = n
    rc = nssmod.lib().nss_run(g._h, 100, 50, 12, 2, -3.0, 10000, C.byref(res), None)
    assert rc == nssmod.NSS_ECAP
    assert p.run(100, 50, 12, 2, cap=n)["rc"] == -3
    r = g.nss_run(100, 50, 12, 2)                   # and the handle is fine afterwards
    assert r["rc"] == 0 and r["n_iter"] > 5
    g.close()
