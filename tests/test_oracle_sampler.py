"""Pins for the sampler half of the oracle."""
import math
import os
import shutil
import subprocess
import tempfile

import numpy as np
import pytest
import scipy.special
import scipy.stats

from paper_2509_24949_b200 import inputs


# ---- P10: Philox4x32-10 against cuRAND's own routine (host-compiled from the CUDA header) ---------
_CURAND_HOST = r"""
#include <cstdio>
#include <cuda_runtime.h>
#define QUALIFIERS static inline __host__ __device__
#include <curand_philox4x32_x.h>
int main() {
  unsigned int s = 12345u;
  for (int i = 0; i < 64; ++i) {
    unsigned int v[6];
    for (int j = 0; j < 6; ++j) { s = s * 1664525u + 1013904223u; v[j] = (i < 8 && j != (i % 6)) ? 0u : s; }
    if (i == 8) for (int j = 0; j < 6; ++j) v[j] = 0xFFFFFFFFu;
    uint4 c = make_uint4(v[0], v[1], v[2], v[3]); uint2 k = make_uint2(v[4], v[5]);
    uint4 o = curand_Philox4x32_10(c, k);
    printf("%u %u %u %u %u %u %u %u %u %u\n", v[0], v[1], v[2], v[3], v[4], v[5], o.x, o.y, o.z, o.w);
  }
  return 0;
}
"""


@pytest.mark.skipif(shutil.which("nvcc") is None, reason="nvcc (for the cuRAND header) not found")
def test_p10_philox_matches_curand_host(oracle):
    with tempfile.TemporaryDirectory() as td:
        src, exe = os.path.join(td, "p.cu"), os.path.join(td, "p")
        open(src, "w").write(_CURAND_HOST)
        subprocess.run(["nvcc", "-O1", "-o", exe, src], check=True, capture_output=True)
        out = subprocess.run([exe], check=True, capture_output=True, text=True).stdout
    rows = [list(map(int, ln.split())) for ln in out.strip().splitlines()]
    assert len(rows) == 64
    for r in rows:
        assert oracle.philox(r[4:6], r[0:4]) == tuple(r[6:10])


def test_p10_philox_is_a_bijection_sample_and_key_sensitive(oracle):
    outs = {oracle.philox((1, 2), (i, 0, 0, 0)) for i in range(2000)}
    assert len(outs) == 2000
    assert oracle.philox((1, 2), (5, 6, 7, 8)) != oracle.philox((1, 3), (5, 6, 7, 8))
    # each counter word matters
    base = oracle.philox((9, 9), (1, 1, 1, 1))
    for j in range(4):
        c = [1, 1, 1, 1]; c[j] = 2
        assert oracle.philox((9, 9), c) != base


# ---- P11: uniforms and normals ----------------------------------------------------------------------
def test_p11_uniform_and_normal_moments(oracle):
    n = 40000
    ka = np.array([oracle.draw53(3, 0, s, 1, 0) for s in range(n)], dtype=np.float64)
    u = ka.ravel() * 2.0 ** -53
    assert u.min() >= 0.0 and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 4 * math.sqrt(1 / 12 / u.size)
    assert scipy.stats.kstest(u, "uniform").pvalue > 1e-3
    # 53-bit assembly: ka = (w0 >> 5) * 2^26 + (w1 >> 6)
    w = oracle.philox((3, 0), (0, 17, 1, 0))
    assert oracle.draw53(3, 0, 17, 1, 0) == ((w[0] >> 5) * 2 ** 26 + (w[1] >> 6), (w[2] >> 5) * 2 ** 26 + (w[3] >> 6))
    assert oracle.uniform_a(3, 0, 17, 1, 0) == ((w[0] >> 5) * 2 ** 26 + (w[1] >> 6)) * 2.0 ** -53
    # seed high word is key[1]
    assert oracle.draw53((5 << 32) | 3, 0, 17, 1, 0) != oracle.draw53(3, 0, 17, 1, 0)
    z = np.array([oracle.normal_pair(3, 1, s, 2, 0) for s in range(n)]).ravel()
    assert np.all(np.isfinite(z))
    assert abs(z.mean()) < 4 / math.sqrt(z.size) and abs(z.var() - 1) < 0.03
    assert scipy.stats.kstest(z, "norm").pvalue > 1e-3
    zz = np.array([oracle.normal_pair(3, 1, s, 2, 0) for s in range(2000)])
    assert abs(np.corrcoef(zz[:, 0], zz[:, 1])[0, 1]) < 0.08
    # Box-Muller radius/angle from the documented u's
    ka_, kb_ = oracle.draw53(3, 1, 5, 2, 0)
    r, a = math.sqrt(-2 * math.log((ka_ + 1) * 2.0 ** -53)), 2 * math.pi * kb_ * 2.0 ** -53
    assert oracle.normal_pair(3, 1, 5, 2, 0) == pytest.approx((r * math.cos(a), r * math.sin(a)), rel=1e-14)


# ---- P12: bookkeeping against library routines -------------------------------------------------------
def test_p12_select_lowest_vs_stable_argsort(oracle):
    rng = np.random.default_rng(0)
    for n, k in ((10, 3), (100, 50), (1000, 500), (257, 256), (64, 1)):
        l = rng.normal(size=n)
        l[rng.integers(0, n, n // 5)] = l[0]                 # ties
        if n > 20:
            l[3] = -np.inf
        dead, surv = oracle.select_lowest(l, k)
        order = np.argsort(l, kind="stable")
        assert np.array_equal(dead, order[:k])
        assert np.array_equal(surv, np.sort(order[k:]))


def test_p12_tune_vs_numpy(oracle):
    rng = np.random.default_rng(1)
    scales = np.array([1.0, 0.1, 0.5, 0.5, 600.0, 1e-3, 1.5, 0.3, 0.6, 0.01, 0.014])
    A = rng.normal(size=(11, 11))
    x = rng.normal(size=(1000, 11)) @ A.T * scales + 1e3 * scales
    rc, mean, cov, chol = oracle.tune(x)
    assert rc == 0
    assert np.allclose(mean, x.mean(0), rtol=1e-13)
    assert np.allclose(cov, np.cov(x.T), rtol=1e-10)
    assert np.allclose(chol, np.linalg.cholesky(np.cov(x.T)), rtol=1e-8, atol=0)
    assert np.allclose(chol @ chol.T, cov, rtol=1e-11)
    assert np.all(np.triu(chol, 1) == 0)
    # degenerate population -> pivot failure reported
    x2 = x.copy(); x2[:, 3] = 7.0        # zero variance -> pivot exactly 0
    assert oracle.tune(x2)[0] != 0


def near_singular_population(rng, n=1000, eps=1e-5):
    """The realistic failure late in a run (chi_1 / chi_2 enter the phase only through beta): column 3 is column 2 plus
    a perturbation eps times smaller, so the last-but-one pivot is ~eps^2 of the column variance."""
    scales = np.array([1.0, 0.1, 0.5, 0.5, 600.0, 1e-3, 1.5, 0.3, 0.6, 0.01, 0.014])
    x = rng.normal(size=(n, 11)) * scales + 10 * scales
    x[:, 3] = x[:, 2] + eps * scales[3] * rng.normal(size=n)
    return x


def test_p12_tune_near_singular_covariance_reading_r5(oracle):
    """DESIGN.md reading R5: the Cholesky fails (ECHOL) if and only if a pivot, computed as written (O12.3), is <= 0 — no
    relative epsilon, no jitter (A11).  A nearly singular covariance (pivot ~1e-10 of the variance) must therefore
    factor, and the factor must reproduce the covariance (the only property the slice directions need: v = w L z/|z|
    has covariance proportional to L L^T); NumPy's factor of the same matrix agrees on the well-conditioned columns.
    Exactly collinear columns leave a pivot of the order of the rounding error whose sign is luck: either outcome is
    legal, but a returned factor must still reproduce the covariance."""
    rng = np.random.default_rng(5)
    x = near_singular_population(rng)
    rc, mean, cov, chol = oracle.tune(x)
    assert rc == 0
    assert np.allclose(cov, np.cov(x.T), rtol=1e-9, atol=1e-22)
    assert np.allclose(chol @ chol.T, cov, rtol=1e-11, atol=1e-22)
    ref = np.linalg.cholesky(cov)
    assert np.allclose(chol[:, :3], ref[:, :3], rtol=1e-9, atol=1e-18)
    assert chol[3, 3] == pytest.approx(ref[3, 3], rel=1e-4) and chol[3, 3] < 1e-4 * chol[2, 2]
    x[:, 3] = x[:, 2]
    rc, mean, cov, chol = oracle.tune(x)
    assert rc != 0 or np.allclose(chol @ chol.T, cov, rtol=1e-9, atol=1e-16 * cov[2, 2])


def test_p12_p14_evidence_update(oracle):
    n, k = 1000, 500
    rng = np.random.default_rng(2)
    dl = np.sort(rng.normal(size=k) * 5 - 20)
    logX, logZ, lw = oracle.evidence_update(dl, n, 0.0, -np.inf)
    m = n - np.arange(k)
    assert logX == pytest.approx(-np.sum(1.0 / m), rel=1e-13)
    assert logZ == pytest.approx(scipy.special.logsumexp(dl + lw), rel=1e-13)
    # weights are the shell volumes X_{j-1} - X_j: they and the remaining volume sum to exactly 1
    assert np.sum(np.exp(lw)) + math.exp(logX) == pytest.approx(1.0, abs=1e-13)
    Xs = np.exp(-np.concatenate([[0.0], np.cumsum(1.0 / m)]))
    assert np.allclose(np.exp(lw), Xs[:-1] - Xs[1:], rtol=1e-11)
    # a second batch continues from the first
    logX2, logZ2, lw2 = oracle.evidence_update(dl + 1, n, logX, logZ)
    assert logX2 == pytest.approx(2 * logX, rel=1e-13)
    assert logZ2 == pytest.approx(scipy.special.logsumexp(np.concatenate([dl + lw, dl + 1 + lw2])), rel=1e-13)
    assert oracle.lib().orc_logaddexp(-np.inf, -3.0) == -3.0


# ---- P13: the slice sampler alone -----------------------------------------------------------------------
def test_p13_no_constraint_gives_uniform_in_box(oracle):
    d, n, k = 4, 1000, 500
    w = inputs.gaussian_workload(d, sigma=1.0)
    p = oracle.Problem(w)
    rng = np.random.default_rng(3)
    live = rng.uniform(-0.2, 0.2, size=(n, d))           # concentrated start: must spread to the box
    live[::2] = rng.uniform(-1, 1, size=(n // 2, d))     # (covariance still spans the box)
    logL = p.loglike_batch(live)
    r = p.replace_step(live, logL, k, 40, seed=11, iteration=0, logLstar=-math.inf, want_trace=True)
    assert r["rc"] == 0
    new = r["live"][r["dead_idx"]]
    assert np.all(new >= -1) and np.all(new <= 1)
    for j in range(d):
        assert scipy.stats.kstest((new[:, j] + 1) / 2, "uniform").pvalue > 1e-3
    assert np.all(r["trace"][:, :, 2] >= 0)              # every step accepted something


def test_p13_ball_constraint_gives_uniform_in_ball(oracle):
    d, n, k, R = 4, 2000, 1000, 0.8
    w = inputs.gaussian_workload(d, sigma=1.0)
    p = oracle.Problem(w)
    rng = np.random.default_rng(4)
    x = rng.uniform(-1, 1, size=(12 * n, d))
    x = x[np.sum(x * x, 1) < R * R][:n]
    assert x.shape[0] == n
    logL = p.loglike_batch(x)
    Lstar = -0.5 * R * R
    r = p.replace_step(x, logL, k, 30, seed=5, iteration=3, logLstar=Lstar)
    assert r["rc"] == 0 and r["logLstar"] == Lstar
    new = r["live"][r["dead_idx"]]
    rad = np.sqrt(np.sum(new * new, 1))
    assert rad.max() < R
    assert np.all(r["logL"][r["dead_idx"]] > Lstar)
    assert scipy.stats.kstest((rad / R) ** d, "uniform").pvalue > 1e-3
    # new logL values are the likelihood of the new positions
    assert np.allclose(r["logL"][r["dead_idx"]], p.loglike_batch(new), rtol=0, atol=0)
    # survivors untouched
    surv = np.setdiff1d(np.arange(n), r["dead_idx"])
    assert np.array_equal(r["live"][surv], x[surv])
    # a survivor below the supplied threshold is rejected (teacher-forced contract)
    assert p.replace_step(x, logL, k, 1, 5, 3, logLstar=0.0)["rc"] == -2


def test_p13_determinism_and_thread_independence(oracle):
    w = inputs.gaussian_workload(3, sigma=0.3)
    p = oracle.Problem(w)
    live, logL = p.init_live(200, 9)
    a = p.replace_step(live, logL, 100, 6, 9, 0, nthreads=1, want_trace=True)
    b = p.replace_step(live, logL, 100, 6, 9, 0, nthreads=4, want_trace=True)
    c = p.replace_step(live, logL, 100, 6, 9, 1, nthreads=4)
    assert np.array_equal(a["live"], b["live"]) and np.array_equal(a["trace"], b["trace"]) and a["n_evals"] == b["n_evals"]
    assert not np.array_equal(a["live"], c["live"])
    # initial live points: theta_j = lo + (hi - lo) u with block j/2, lane j%2 (O11 stream layout)
    ka, kb = oracle.draw53(9, 1, 0, 7, 0xFFFFFFFF)
    assert live[7, 2] == -1.0 + 2.0 * (ka * 2.0 ** -53)
    ka, kb = oracle.draw53(9, 0, 0, 7, 0xFFFFFFFF)
    assert live[7, 1] == -1.0 + 2.0 * (kb * 2.0 ** -53)
    # eval count = stepping-out tests + shrink tries inside the box; trace is consistent with it
    tr = a["trace"]
    assert a["n_evals"] <= np.sum(tr[:, :, 0] + 1 + tr[:, :, 1] + 1 + tr[:, :, 2] + 1)


# ---- P14 / P15 / P16: full NS run on the Gaussian test likelihood --------------------------------------
def _analytic_logz(d, sigma, half):
    c = scipy.stats.norm.cdf(half / sigma) - scipy.stats.norm.cdf(-half / sigma)
    return d * math.log(sigma * math.sqrt(2 * math.pi) / (2 * half) * c)


@pytest.mark.parametrize("d,n,k,seed", [(4, 1000, 500, 1), (4, 400, 100, 2), (11, 600, 300, 3)])
def test_p15_p16_gaussian_evidence_and_posterior(oracle, d, n, k, seed):
    sigma = 0.05
    w = inputs.gaussian_workload(d, sigma=sigma)
    p = oracle.Problem(w)
    r = p.run(n, k, 5 * d, seed)
    assert r["rc"] == 0
    truth = _analytic_logz(d, sigma, 1.0)
    assert 0.02 < r["logZ_err"] < 0.6
    assert abs(r["logZ"] - truth) < 3 * r["logZ_err"]
    # closed-form cross-check of the error estimate: sigma^2 ~ H * sum(1/m^2)/sum(1/m) per iteration
    m = n - np.arange(k)
    approx = math.sqrt(r["H"] * np.sum(1.0 / m ** 2) / np.sum(1.0 / m))
    assert 0.5 < r["logZ_err"] / approx < 2.0
    # H of a Gaussian posterior in a wide box: H = -logZ - d/2  (KL(posterior || prior), peak logL = 0)
    assert r["H"] == pytest.approx(-truth - d / 2, abs=0.5)
    # P14 invariants
    nd, ni = r["n_dead"], r["n_iter"]
    assert nd == ni * k + n
    assert np.sum(np.exp(r["dead_logw"])) == pytest.approx(1.0, abs=1e-10)
    dl = r["dead_logL"]
    assert np.all(np.diff(dl[:ni * k]) >= 0) and np.all(np.diff(dl[ni * k:]) >= 0)
    assert np.all(r["dead_logL_birth"] < dl)
    mm = np.concatenate([n - np.arange(k)] * ni)
    assert r["dead_logw"][ni * k] == pytest.approx(-np.sum(1.0 / mm) - math.log(n), rel=1e-12)
    # P16 posterior moments
    pw = np.exp(dl + r["dead_logw"] - r["logZ"])
    assert pw.sum() == pytest.approx(1.0, abs=1e-9)
    ess = 1.0 / np.sum(pw ** 2)
    mean = pw @ r["dead_theta"]
    sd = np.sqrt(pw @ (r["dead_theta"] - mean) ** 2)
    assert np.all(np.abs(mean) < 5 * sigma / math.sqrt(ess))
    assert np.all(np.abs(sd / sigma - 1) < 0.15)


def test_run_matches_stepwise_composition(oracle):
    """orc_run is exactly init_live + repeated replace_step + evidence_update (O12-O14)."""
    w = inputs.gaussian_workload(3, sigma=0.1)
    p = oracle.Problem(w)
    n, k, nr, seed = 200, 100, 9, 4
    r = p.run(n, k, nr, seed)
    live, logL = p.init_live(n, seed)
    logX, logZ, t = 0.0, -np.inf, 0
    # births tracked here, outside the oracle: an initial point is born at -inf, a replacement at the threshold of the
    # iteration that made it (O13); the run must report exactly that value when the point dies or is appended at the end
    birth = np.full(n, -np.inf)
    rows_L, rows_birth, rows_theta = [], [], []
    while True:
        lzl = logX + scipy.special.logsumexp(logL) - math.log(n)
        if t > 0 and lzl - logZ < -3.0:
            break
        s = p.replace_step(live, logL, k, nr, seed, t)
        logX, logZ, lw = oracle.evidence_update(s["dead_logL"], n, logX, logZ)
        di = s["dead_idx"]
        rows_L.append(logL[di]); rows_birth.append(birth[di].copy()); rows_theta.append(live[di])
        birth[di] = s["logLstar"]
        live, logL = s["live"], s["logL"]
        t += 1
    assert t == r["n_iter"]
    assert np.logaddexp(logZ, lzl) == pytest.approx(r["logZ"], rel=1e-13)
    order = np.argsort(logL, kind="stable")                       # the final live points, ascending logL, ties by slot
    rows_L.append(logL[order]); rows_birth.append(birth[order]); rows_theta.append(live[order])
    assert np.array_equal(r["dead_logL"], np.concatenate(rows_L))
    assert np.array_equal(r["dead_theta"], np.concatenate(rows_theta))
    got_birth = r["dead_logL_birth"]
    assert np.array_equal(got_birth, np.concatenate(rows_birth))
    assert np.all(got_birth[:k] == -np.inf) and np.isfinite(got_birth[t * k:]).any()     # both kinds of birth occur


def _replica_sigma(dead_logL, live_logL, n, k, rule, rng, R=400):
    """O15 written out in NumPy with NumPy's own generator: R stochastic-compression replicas of logZ.  `rule` gives the
    number of live points m_j behind the j-th deletion."""
    J = dead_logL.size
    m = rule(np.arange(J))
    lz = np.empty(R)
    for rep in range(R):
        lnt = np.log(1.0 - rng.random(J)) / m                      # t_j = u^(1/m_j), u in (0, 1]
        lX = np.concatenate([[0.0], np.cumsum(lnt)])               # log X before deletion j; lX[J] after the last
        lw = lX[:-1] + np.log1p(-np.exp(lnt))                      # w_j = X_j (1 - t_j)
        dead = scipy.special.logsumexp(dead_logL + lw)
        lz[rep] = np.logaddexp(dead, lX[-1] + scipy.special.logsumexp(live_logL) - math.log(n))
    return lz.std(ddof=1)


def test_p15_replica_error_against_the_closed_form_over_seeds(oracle):
    """O15, tightened.  With k deletions per iteration the log-volume after an iteration has variance sum_j 1/m_j^2,
    m_j = n - (j mod k), and mean -sum_j 1/m_j, so sigma(logZ)^2 ~ H sum(1/m^2) / sum(1/m).  The oracle's replica error,
    averaged over 8 seeds at n_live = 2000, must sit within 12 % of that (measured: 1.005 +- 0.05 per seed).  The same
    replicas written in NumPy from the oracle's dead rows agree too, and with m_j replaced by n — the slip a batched
    deletion invites — they fall to ~0.71 of the closed form, far outside the band."""
    d, n, k, sigma = 4, 2000, 1000, 0.05
    p = oracle.Problem(inputs.gaussian_workload(d, sigma=sigma))
    m = n - np.arange(k)
    ratios, r = [], None
    for seed in range(10, 18):
        r = p.run(n, k, 5 * d, seed)
        assert r["rc"] == 0
        ratios.append(r["logZ_err"] / math.sqrt(r["H"] * np.sum(1.0 / m ** 2) / np.sum(1.0 / m)))
    assert 0.88 < np.mean(ratios) < 1.12, ratios
    assert 0.75 < min(ratios) and max(ratios) < 1.3, ratios
    J = r["n_iter"] * k
    dead, livel = r["dead_logL"][:J], r["dead_logL"][J:]
    approx = math.sqrt(r["H"] * np.sum(1.0 / m ** 2) / np.sum(1.0 / m))
    rng = np.random.default_rng(0)
    right = _replica_sigma(dead, livel, n, k, lambda j: n - (j % k), rng)
    wrong = _replica_sigma(dead, livel, n, k, lambda j: np.full(j.size, float(n)), rng)
    assert 0.85 < right / approx < 1.15 and 0.85 < r["logZ_err"] / right < 1.15
    assert wrong / approx < 0.8


# ---- NEXT-2: periodic coordinates in the slice sampler (R4) ----------------------------------
def test_next2_periodic_slices_stay_uniform_and_in_the_box(oracle):
    """P13 with wrapped coordinates: no constraint (L* = -inf) => still uniform in the box; a wrapped coordinate
    never fails the box test, so its brackets step out to the cap while a walled coordinate stops them."""
    d, n, k = 3, 1000, 500
    w = inputs.gaussian_workload(d, sigma=1.0)
    p = oracle.Problem(w)
    rng = np.random.default_rng(3)
    live = rng.uniform(-1, 1, size=(n, d))
    logL = p.loglike_batch(live)
    p.set_periodic([1, 0, 1])
    r = p.replace_step(live, logL, k, 40, seed=11, iteration=0, logLstar=-math.inf, want_trace=True)
    assert r["rc"] == 0
    new = r["live"][r["dead_idx"]]
    assert np.all(new >= -1) and np.all(new <= 1)
    for j in range(d):
        assert scipy.stats.kstest((new[:, j] + 1) / 2, "uniform").pvalue > 1e-3
    assert np.all(r["trace"][:, :, 2] >= 0)
    walled = r["trace"][:, :, :2].mean()
    p.set_periodic([1, 1, 1])                       # nothing stops a bracket any more: every side reaches the cap of 32
    r2 = p.replace_step(live, logL, k, 5, seed=11, iteration=0, logLstar=-math.inf, want_trace=True)
    assert np.all(r2["trace"][:, :, :2] == 32) and walled < 32
    new2 = r2["live"][r2["dead_idx"]]
    assert np.all(new2 >= -1) and np.all(new2 <= 1)
    p.set_periodic([0, 0, 0])                       # and the flags switch off again: the default walls (A16)
    r3 = p.replace_step(live, logL, k, 5, seed=11, iteration=0, logLstar=-math.inf, want_trace=True)
    r4 = oracle.Problem(w).replace_step(live, logL, k, 5, seed=11, iteration=0, logLstar=-math.inf, want_trace=True)
    assert np.array_equal(r3["live"], r4["live"]) and np.array_equal(r3["trace"], r4["trace"])


def test_next2_r7_tuning_unwraps_around_the_circular_mean(oracle):
    """Reading R7 (NEXT-2, second half).  Pins: (a) the circular mean is SciPy's circmean; (b) a cloud that
    straddles the seam gets the covariance of the UNWRAPPED cloud (NumPy, computed on coordinates that never saw the
    box), not the ~W^2/4 of its stored values; (c) no flag, or a cloud that does not reach across the seam, is orc_tune
    bit for bit; (d) the periodic replace step uses it: directions of a seam-straddling population have the cloud's
    scale, so brackets in the wrapped coordinate stop expanding after a step or two instead of running to the cap."""
    rng = np.random.default_rng(11)
    n, d = 2000, 3
    lo, hi = np.array([-1.0, 0.0, -2.0]), np.array([1.0, 2 * np.pi, 3.0])
    W = hi - lo
    A = np.array([[0.05, 0.0, 0.0], [0.02, 0.04, 0.0], [0.01, -0.03, 0.06]])
    z = rng.normal(size=(n, d)) @ A.T
    centre = np.array([0.3, 2 * np.pi - 0.01, -1.99])             # coordinate 1 sits on its upper seam, 2 on its lower one
    free = z + centre                                             # never wrapped: what the tuning should see
    stored = lo + np.mod(free - lo, W)                            # what the sampler stores
    flags = [0, 1, 1]
    assert np.any(stored[:, 1] < 1.0) and np.any(stored[:, 1] > 5.0)          # really on both sides
    rc, mean, cov, chol = oracle.tune_periodic(stored, flags, lo, hi)
    assert rc == 0
    want = np.cov(free.T)
    assert np.allclose(cov, want, rtol=1e-10, atol=1e-16)
    assert np.allclose(chol, np.linalg.cholesky(want), rtol=1e-9, atol=1e-16)
    _, _, plain, _ = oracle.tune(stored)
    assert plain[1, 1] > 100 * cov[1, 1] and plain[2, 2] > 100 * cov[2, 2]    # what the plain moments would have given
    # (a) the mean it reports is the circular mean's image of the cloud: equal to SciPy's circmean modulo the period
    for j in (1, 2):
        cm = scipy.stats.circmean(stored[:, j], high=hi[j], low=lo[j])
        delta = (mean[j] - cm) / W[j]
        assert abs(delta - round(delta)) < 0.02 / W[j]                         # the two means differ by O(sigma^2 / W)
    # (c) identities, bit for bit
    r0 = oracle.tune_periodic(stored, [0, 0, 0], lo, hi)
    r1 = oracle.tune(stored)
    assert all(np.array_equal(a, b) for a, b in zip(r0[1:], r1[1:]))
    inside = z + np.array([0.3, 3.0, 0.5])                                      # far from every seam
    r2, r3 = oracle.tune_periodic(inside, flags, lo, hi), oracle.tune(inside)
    assert all(np.array_equal(a, b) for a, b in zip(r2[1:], r3[1:]))
    # a uniform population on the circle (no preferred direction) keeps a variance of ~W^2/12 whatever the circular mean is
    u = lo + W * rng.random((4000, d))
    _, _, cu, _ = oracle.tune_periodic(u, flags, lo, hi)
    assert np.allclose(np.diag(cu), W ** 2 / 12, rtol=0.1)
    # (d) inside the sampler: a Gaussian whose peak sits on the seam of a periodic coordinate
    w = inputs.gaussian_workload(2, sigma=0.02)
    w.gauss_mu = w.gauss_mu.copy(); w.gauss_mu[1] = w.hi[1]                     # logL peaks at the upper wall of coordinate 1
    p = oracle.Problem(w)
    Wb = w.hi - w.lo
    cloud = np.column_stack([rng.normal(size=600) * 0.02, w.hi[1] + rng.normal(size=600) * 0.02])
    cloud_stored = w.lo + np.mod(cloud - w.lo, Wb)
    # the likelihood is not periodic here, so give every point the logL of its nearest image (what a periodic one would)
    logL = -0.5 * np.sum(((cloud - w.gauss_mu[:2]) / 0.02) ** 2, axis=1)
    p.set_periodic([0, 1])
    r = p.replace_step(cloud_stored, logL, 300, 4, seed=5, iteration=0, logLstar=-math.inf, want_trace=True)
    assert r["rc"] == 0
    # with L* = -inf every bracket end passes until the cap unless the box stops it: the wall of coordinate 0 does, after
    # (1 - |x0|)/|v0| steps.  R7's directions are ~2 x 0.02 long, the plain moments' (variance ~1 in coordinate 1) are not
    # small in coordinate 0 either only through correlation; what is pinned is the covariance the step used:
    _, _, cov_used, _ = oracle.tune_periodic(cloud_stored, [0, 1], w.lo, w.hi)
    assert cov_used[1, 1] < 4 * 0.02 ** 2 and oracle.tune(cloud_stored)[2][1, 1] > 0.5


def test_next2_wrap_is_the_identity_inside_and_a_shift_by_periods_outside(oracle):
    """A chain that never leaves the box must not notice the flags: with a constraint region well inside the box
    (a tight Gaussian, L* high) the wrapped and the walled sampler make the same decisions and end at the same bits."""
    w = inputs.gaussian_workload(4, sigma=0.02)
    p = oracle.Problem(w)
    rng = np.random.default_rng(5)
    live = rng.normal(size=(400, 4)) * 0.02
    logL = p.loglike_batch(live)
    a = p.replace_step(live, logL, 200, 12, seed=2, iteration=1, want_trace=True)
    p.set_periodic([1, 1, 1, 1])
    b = p.replace_step(live, logL, 200, 12, seed=2, iteration=1, want_trace=True)
    assert np.array_equal(a["live"], b["live"]) and np.array_equal(a["trace"], b["trace"]) and a["n_evals"] == b["n_evals"]


@pytest.mark.parametrize("flags", [(1, 0, 0), (1, 1, 1)])
def test_next2_evidence_does_not_depend_on_the_topology(oracle, flags):
    """The evidence of a likelihood under a uniform prior is the same integral on the box and on the torus, so NS with
    wrapped coordinates must reproduce O16's analytic logZ (here with the peak 0.2 sigma from a wall, where wrapping
    changes most of the slices) within 3 sigma_NS."""
    w = inputs.gaussian_workload(3, sigma=0.05)
    w.gauss_mu = w.gauss_mu.copy()
    w.gauss_mu[0] = -0.99
    p = oracle.Problem(w)
    p.set_periodic(flags)
    truth = sum(math.log(0.05 * math.sqrt(2 * math.pi) / 2.0
                         * (scipy.stats.norm.cdf((1 - m) / 0.05) - scipy.stats.norm.cdf((-1 - m) / 0.05))) for m in w.gauss_mu[:3])
    o = p.run(1000, 500, 15, 3)
    assert o["rc"] == 0
    assert abs(o["logZ"] - truth) < 3 * o["logZ_err"]
    pw = np.exp(o["dead_logL"] + o["dead_logw"] - o["logZ"])
    mean0 = pw @ o["dead_theta"][:, 0]
    # posterior of the first coordinate: a normal truncated at the wall -0.99 - 0.2 sigma ... its mean is known
    a = (-1 - w.gauss_mu[0]) / 0.05
    tm = w.gauss_mu[0] + 0.05 * scipy.stats.norm.pdf(a) / (1 - scipy.stats.norm.cdf(a))
    assert abs(mean0 - tm) < 0.01


def test_next2_bracket_longer_than_one_period_keeps_the_slice_uniform(oracle):
    """A wrapped coordinate never fails the box test, so with a loose constraint a bracket can grow past one period
    (up to 32 widths per side) and wrapped proposals then cover parts of the circle more than once.  The slice is the
    lifted periodic set on the line and stepping-out / shrinkage on it is ordinary slice sampling, so the wrapped draw
    stays uniform on the admissible arc.  1-D circle [-1, 1), threshold admitting the arc |x| < 0.8 (80 % of the circle):
    an end that steps across the seam lands inside the arc again and the bracket keeps growing."""
    w = inputs.gaussian_workload(1, sigma=1.0)
    p = oracle.Problem(w)
    p.set_periodic([1])
    c = 0.8
    Lstar = -0.5 * c * c
    rng = np.random.default_rng(8)
    n, k = 1200, 600
    live = rng.uniform(-c, c, size=(n, 1))
    logL = p.loglike_batch(live)
    r = p.replace_step(live, logL, k, 30, seed=4, iteration=0, logLstar=Lstar, want_trace=True)
    assert r["rc"] == 0
    new = r["live"][r["dead_idx"]][:, 0]
    assert np.all(np.abs(new) < c)
    assert scipy.stats.kstest((new + c) / (2 * c), "uniform").pvalue > 1e-3
    # bracket length in units of the coordinate: (1 + expansions) * |v|, |v| = 2 * s.d. of the live points (A14)
    width = (1 + r["trace"][:, :, 0] + r["trace"][:, :, 1]) * 2.0 * np.std(live[:, 0], ddof=1)
    assert (width > 2.0).mean() > 0.2, "the case must exercise brackets longer than the period"


# ---- NEXT-4 / reading R6: equal-weight posterior samples ---------------------------------------------------------------
def test_r6_equal_weight_resampling_closed_forms(oracle):
    """orc_resample_equal keeps row i iff u_i < p_i / p_max.  What the mathematics fixes: equal weights keep every row;
    a row with the maximum weight is always kept and rows 800 nats below never; weights of exactly half the maximum keep
    about half (binomial); the expected number kept is sum p / p_max; the kept rows are an equally weighted sample of
    the weighted distribution (their plain mean matches the weighted mean); rows of zero weight are never kept; and the
    draw is a function of (seed, row) only."""
    n = 20000
    z = np.zeros(n)
    assert np.array_equal(oracle.resample_equal(z, np.full(n, -7.0), 1), np.arange(n))
    lw = np.full(n, -800.0); lw[[5, 77]] = 0.0
    assert np.array_equal(oracle.resample_equal(z, lw, 2), [5, 77])
    lw = np.full(n, math.log(0.5)); lw[0] = 0.0
    m = oracle.resample_equal(z, lw, 3).size
    assert abs(m - 1 - (n - 1) / 2) < 5 * math.sqrt(n / 4)
    rng = np.random.default_rng(0)
    x = rng.normal(size=n)
    logL = -0.5 * ((x - 0.7) / 0.3) ** 2            # weight ~ N(0.7, 0.3) density ratio over the N(0,1) proposal
    logw = rng.normal(size=n) * 0.0
    logw[::10] = -np.inf
    counts = [oracle.resample_equal(logL, logw, s).size for s in range(40)]
    pw = np.exp(logL + logw - (logL + logw).max())
    assert abs(np.mean(counts) - pw.sum()) < 5 * math.sqrt(pw.sum() / 40)
    idx = oracle.resample_equal(logL, logw, 9)
    assert np.all(np.diff(idx) > 0) and not np.any(np.isin(idx, np.arange(0, n, 10)))
    wmean = (pw * x).sum() / pw.sum()
    wsd = math.sqrt((pw * (x - wmean) ** 2).sum() / pw.sum())
    assert abs(x[idx].mean() - wmean) < 5 * wsd / math.sqrt(idx.size)
    assert abs(x[idx].std() / wsd - 1) < 0.1
    assert np.array_equal(idx, oracle.resample_equal(logL, logw, 9))
    assert not np.array_equal(idx, oracle.resample_equal(logL, logw, 10))
    # u_i is the documented Philox counter: (block 0, step i, chain 0, iteration 0xFFFFFFFD)
    u = np.array([oracle.uniform_a(9, 0, i, 0, 0xFFFFFFFD) for i in range(200)])
    assert np.array_equal(np.flatnonzero(u < pw[:200]), idx[idx < 200])
    assert oracle.resample_equal(z[:3], np.full(3, -np.inf), 1).size == 0


# ---- sanitizers -------------------------------------------------------------------------------------------
def test_oracle_is_clean_under_address_and_undefined_sanitizers(tmp_path):
    """The oracle compiled with -fsanitize=address,undefined (leak check included) walks every entry point on tiny
    problems of all three likelihood kinds (oracle/sanitize_main.c): any out-of-bounds access, leak or undefined
    arithmetic aborts."""
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    exe = str(tmp_path / "orc_sanitized")
    cmd = ["gcc", "-std=c99", "-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-ffp-contract=off",
           "-fopenmp", os.path.join(root, "oracle", "nss_oracle.c"), os.path.join(root, "oracle", "sanitize_main.c"),
           "-o", exe, "-lm"]
    subprocess.run(cmd, check=True)
    r = subprocess.run([exe], capture_output=True, text=True, timeout=300,
                       env=dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", OMP_NUM_THREADS="2"))
    assert r.returncode == 0, r.stdout + r.stderr
    assert "sanitize_main: ok" in r.stdout and "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr
