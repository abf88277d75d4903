"""Pins for the likelihood half of the oracle.

None of these re-types the oracle's formula: each checks a closed form, an invariant, a special
case or an exact identity that a dropped term / wrong sign / transposed operand would break.
"""
import copy
import math
import os

import numpy as np
import pytest

from paper_2509_24949_b200 import inputs

GMSUN = 4.925490947641267e-6


def _canon(**kw):
    th = np.array([30.0, 0.8, 0.1, -0.05, 1000.0, 0.01, 1.0, 0.6, 0.8, 1.5, -0.5])
    for k, v in kw.items():
        th[inputs.SLOT_NAMES.index(k)] = v
    return th


# ---- P1: Newtonian limit ------------------------------------------------------------------------
def test_p1_newtonian_chirp_closed_form(oracle):
    for q in (0.3, 0.8, 1.0):
        th = _canon(q=q)
        for f in (20.0, 57.3, 400.0):
            psi = oracle.phase(f, th, newtonian=True)
            lead = psi - (2 * math.pi * f * th[5] - th[6] - math.pi / 4)
            expect = 3.0 / 128.0 * (math.pi * GMSUN * th[0] * f) ** (-5.0 / 3.0)   # independent of q
            assert lead == pytest.approx(expect, rel=1e-12)


def test_p1_time_frequency_relation(oracle):
    th = _canon()
    mc = GMSUN * th[0]
    for f in (30.0, 100.0):
        h = 1e-3
        dpsi = (oracle.phase(f + h, th, True) - oracle.phase(f - h, th, True)) / (2 * h)
        expect = th[5] - 5.0 / 256.0 * mc ** (-5.0 / 3.0) * (math.pi * f) ** (-8.0 / 3.0)
        assert dpsi / (2 * math.pi) == pytest.approx(expect, rel=1e-7)


def test_p1_full_phase_tends_to_newtonian_at_low_v(oracle):
    # PN corrections are O(v^2) relative to the leading term: ratio -> 1 as f -> 0
    th = _canon(tc=0.0, phic=0.0)
    r = []
    for f in (1e-3, 1e-5):
        full = oracle.phase(f, th) + math.pi / 4
        newt = oracle.phase(f, th, True) + math.pi / 4
        r.append(full / newt - 1.0)
    assert abs(r[1]) < abs(r[0]) < 2e-2
    assert abs(r[1]) < 1e-3


# ---- P2: the higher PN coefficients, recovered numerically and compared with SURVEY.md O3's literals ---------------
def _golden_literals():
    """tests/golden/taylorf2_o3_literals.txt (typed by hand from SURVEY.md:346-355) -> {name: mpmath value}."""
    import mpmath as mp
    sym = {"pi": mp.pi, "pi^2": mp.pi ** 2, "gammaE": mp.mpf("0.5772156649015329")}
    out = {}
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "taylorf2_o3_literals.txt")
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        name, expr = (t.strip() for t in line.split("|"))
        val = mp.mpf(0)
        for term in expr.split(" + "):
            parts = [t.strip() for t in term.split("*")]
            p, q = parts[0].split("/")
            t = mp.mpf(int(p)) / int(q)
            for s in parts[1:]:
                t *= sym[s]
            val += t
        out[name] = val
    return out


def test_p2_pn_literals_recovered_from_the_phase(oracle):
    """S(v) = (128 eta v^5 / 3)(Psi - 2 pi f t_c + phi_c + pi/4) = sum_k phi_k v^k is LINEAR in every literal of O3 once
    the basis (power of v, ln v, power of eta, spin combination) is fixed.  Evaluate orc_phase on a grid of (v, q, spins),
    solve the least-squares problem for the 22 coefficients in 60-digit arithmetic (inputs are the oracle's doubles), and
    compare each with the rational literal stored under tests/golden/ (typed from SURVEY.md O3, not from the oracle).
    A dropped term, a wrong sign or a mistyped digit in any phi_k of oracle/nss_oracle.c changes a recovered
    coefficient by far more than the recovery error (measured: < 3e-9 relative; bar 1e-8)."""
    import mpmath as mp
    mp.mp.dps = 60
    G = _golden_literals()
    rows, rhs = [], []
    Mc = 30.0
    for q in (1.0, 0.8, 0.6, 0.45, 0.3, 0.2, 0.12):
        for c1, c2 in ((0.0, 0.0), (0.7, -0.4), (-0.3, 0.9)):
            for vt in np.geomspace(0.15, 3.0, 24):          # the formula is just a formula: v need not be physical
                f = float(vt ** 3 / (math.pi * Mc * (q / (1 + q) ** 2) ** -0.6 * GMSUN))
                psi = oracle.phase(f, _canon(Mc=Mc, q=q, chi1z=c1, chi2z=c2, tc=0.0, phic=0.0))
                qm = mp.mpf(q)
                eta = qm / (1 + qm) ** 2
                v = mp.cbrt(mp.pi * mp.mpf(Mc) * eta ** (mp.mpf(-3) / 5) * mp.mpf(GMSUN) * mp.mpf(f))
                lv = mp.log(v)
                m1, m2 = 1 / (1 + qm), qm / (1 + qm)
                b_m, b_e = m1 ** 2 * mp.mpf(c1) + m2 ** 2 * mp.mpf(c2), eta * (mp.mpf(c1) + mp.mpf(c2))
                rows.append([1, v, v ** 2, v ** 2 * eta, v ** 3, v ** 3 * b_m, v ** 3 * b_e, v ** 4, v ** 4 * eta, v ** 4 * eta ** 2,
                             v ** 5, v ** 5 * eta, v ** 5 * lv, v ** 5 * lv * eta, v ** 6, v ** 6 * eta, v ** 6 * eta ** 2,
                             v ** 6 * eta ** 3, v ** 6 * lv, v ** 7, v ** 7 * eta, v ** 7 * eta ** 2])
                rhs.append((128 * eta * v ** 5 / 3) * (mp.mpf(psi) + mp.pi / 4))
    A, b = mp.matrix(rows), mp.matrix(rhs)
    x = mp.lu_solve(A.T * A, A.T * b)
    # phi_5 = P5 (1 + 3 ln(v / v_lso)) = P5 (1 + (3/2) ln(1/v_lso^2)) + 3 P5 ln v;   -(6848/21) ln(4v) = phi6_ln (ln 4 + ln v)
    k5 = 1 + G["phi5_ln"] / 2 * mp.log(G["vlso_inv_square"])
    expect = [G["phi0"], G["phi1"], G["phi2_eta0"], G["phi2_eta1"],
              G["phi3_const"], G["phi3_beta"] * G["beta_mass2"], G["phi3_beta"] * G["beta_eta"],
              G["phi4_eta0"], G["phi4_eta1"], G["phi4_eta2"],
              G["phi5_eta0"] * k5, G["phi5_eta1"] * k5, G["phi5_ln"] * G["phi5_eta0"], G["phi5_ln"] * G["phi5_eta1"],
              G["phi6_eta0"] + G["phi6_ln"] * mp.log(G["phi6_ln_arg"]), G["phi6_eta1"], G["phi6_eta2"], G["phi6_eta3"],
              G["phi6_ln"], G["phi7_eta0"], G["phi7_eta1"], G["phi7_eta2"]]
    for i, e in enumerate(expect):
        scale = abs(e) if e != 0 else mp.mpf(1)
        assert abs(x[i] - e) / scale < 1e-8, f"coefficient {i}: recovered {mp.nstr(x[i], 15)}, SURVEY O3 says {mp.nstr(e, 15)}"


# ---- P2 sanity identities -------------------------------------------------------------------------------------------
def test_p2_spin_orbit_enters_only_through_beta(oracle):
    # phi_3 shifts by exactly 4*beta: Psi(chi) - Psi(0) = 3/(128 eta v^5) * 4 beta v^3
    th0, th1 = _canon(chi1z=0.0, chi2z=0.0), _canon(chi1z=0.3, chi2z=-0.2)
    q = th0[1]
    eta = q / (1 + q) ** 2
    M = th0[0] * eta ** -0.6 * GMSUN
    m1, m2 = 1 / (1 + q), q / (1 + q)
    beta = (113 / 12 * m1 * m1 + 25 / 4 * eta) * 0.3 + (113 / 12 * m2 * m2 + 25 / 4 * eta) * (-0.2)
    for f in (25.0, 200.0):
        v = (math.pi * M * f) ** (1 / 3)
        expect = 3 / (128 * eta * v ** 5) * 4 * beta * v ** 3
        got = oracle.phase(f, th1) - oracle.phase(f, th0)
        assert got == pytest.approx(expect, rel=1e-9)


def test_p2_phase_smooth_and_monotone_second_difference(oracle):
    th = _canon()
    f = np.linspace(20.0, 1024.0, 4017)
    psi = np.array([oracle.phase(x, th) for x in f])
    d2 = np.diff(psi, 2)
    assert np.all(np.isfinite(psi))
    assert np.max(np.abs(np.diff(d2))) < 1e-2       # no kinks / jumps


# ---- P3: antenna patterns and delays -------------------------------------------------------------
def test_p3_antenna_invariants(oracle):
    rng = np.random.default_rng(0)
    for name in ("H1", "L1", "V1"):
        det = inputs.detector_array((name,))[0]
        x, y, r = det[3:6], det[6:9], det[0:3]
        assert abs(np.dot(x, x) - 1) < 1e-6 and abs(np.dot(y, y) - 1) < 1e-6 and abs(np.dot(x, y)) < 1e-6
        assert 6.36e6 < np.linalg.norm(r) < 6.38e6
        for _ in range(20):
            ra, dec, psi, gm = rng.uniform(0, 2 * np.pi), np.arcsin(rng.uniform(-1, 1)), rng.uniform(0, np.pi), rng.uniform(0, 2 * np.pi)
            fp, fc, dt = oracle.antenna(det, gm, ra, dec, psi)
            fp2, fc2, dt2 = oracle.antenna(det, gm, ra, dec, psi + 0.37)
            assert fp * fp + fc * fc == pytest.approx(fp2 * fp2 + fc2 * fc2, abs=1e-12)
            fp3, fc3, _ = oracle.antenna(det, gm, ra, dec, psi + np.pi / 2)
            assert fp3 == pytest.approx(-fp, abs=1e-12) and fc3 == pytest.approx(-fc, abs=1e-12)
            fp4, fc4, _ = oracle.antenna(det, gm, ra, dec, psi + np.pi / 4)       # spin-2 rotation
            # O4: dX/dpsi = Y, dY/dpsi = -X  =>  F+(psi+d) = F+ cos2d + Fx sin2d, Fx(psi+d) = Fx cos2d - F+ sin2d
            assert fp4 == pytest.approx(fc, abs=1e-12) and fc4 == pytest.approx(-fp, abs=1e-12)
            assert fp2 == pytest.approx(fp * math.cos(0.74) + fc * math.sin(0.74), abs=1e-12)
            assert abs(fp) <= 1 + 1e-12 and abs(fc) <= 1 + 1e-12
            assert abs(dt) <= np.linalg.norm(r) / 299792458.0 + 1e-15
            assert dt == dt2
            # only ra - gmst matters
            fp5, fc5, dt5 = oracle.antenna(det, gm + 0.5, ra + 0.5, dec, psi)
            assert (fp5, fc5, dt5) == pytest.approx((fp, fc, dt), abs=1e-12)


def test_p3_sky_average_is_one_fifth(oracle):
    rng = np.random.default_rng(1)
    det = inputs.detector_array(("H1",))[0]
    n = 20000
    acc = np.zeros(2)
    for _ in range(n):
        fp, fc, _ = oracle.antenna(det, 0.0, rng.uniform(0, 2 * np.pi), np.arcsin(rng.uniform(-1, 1)), rng.uniform(0, np.pi))
        acc += (fp * fp, fc * fc)
    assert acc[0] / n == pytest.approx(0.2, abs=0.006)
    assert acc[1] / n == pytest.approx(0.2, abs=0.006)


def test_p3_overhead_source_and_delay_sign(oracle):
    det = inputs.detector_array(("SYN",))[0]
    fp, fc, dt = oracle.antenna(det, 0.0, 0.0, math.pi / 2, 0.0)
    assert abs(fp) == pytest.approx(1.0, abs=1e-15) and fc == pytest.approx(0.0, abs=1e-15) and dt == 0.0
    # a detector displaced TOWARDS the source receives the wave earlier: dt = -|r|/c
    d2 = np.array([0, 0, 6.0e6, 1, 0, 0, 0, 1, 0.0])
    assert oracle.antenna(d2, 0.0, 0.3, math.pi / 2, 0.0)[2] == pytest.approx(-6.0e6 / 299792458.0, rel=1e-14)
    # source on the +x axis at gmst = ra: n = (1,0,0)
    d3 = np.array([1.0e6, 0, 0, 0, 1, 0, 0, 0, 1.0])
    assert oracle.antenna(d3, 1.1, 1.1, 0.0, 0.0)[2] == pytest.approx(-1.0e6 / 299792458.0, rel=1e-14)


def test_p3_waveform_amplitude_and_polarisation_mix(oracle):
    # |h| = A f^-7/6 |F+ (1+c^2)/2 - i Fx c| with A from the Newtonian amplitude formula
    th = _canon()
    det = inputs.detector_array(("L1",))[0]
    f = np.array([20.0, 80.0, 512.0])
    h = oracle.waveform(th, det, 0.3, f)
    fp, fc, dt = oracle.antenna(det, 0.3, th[9], th[10], th[8])
    ci = math.cos(th[7])
    A = math.sqrt(5 / 24) * math.pi ** (-2 / 3) * (GMSUN * th[0]) ** (5 / 6) * 299792458.0 / (th[4] * 3.085677581491367e22)
    expect = A * f ** (-7 / 6) * abs(fp * (1 + ci * ci) / 2 - 1j * fc * ci)
    assert np.allclose(np.abs(h), expect, rtol=1e-13)
    # face-on (iota = 0): h ~ F+ - i Fx, and the rotation above gives h(psi + dpsi) = h(psi) e^{+2 i dpsi}
    th0 = _canon(iota=0.0)
    a = oracle.waveform(th0, det, 0.3, f)
    th0[8] += 0.2
    b = oracle.waveform(th0, det, 0.3, f)
    assert np.allclose(b, a * np.exp(2j * 0.2), rtol=1e-11)
    # time shift: tc -> tc + tau multiplies by e^{-2 pi i f tau}
    th1 = _canon()
    th1[5] += 1e-3
    assert np.allclose(oracle.waveform(th1, det, 0.3, f), h * np.exp(-2j * np.pi * f * 1e-3), rtol=1e-10)
    # phic -> phic + delta multiplies by e^{+i delta}
    th2 = _canon()
    th2[6] += 0.3
    assert np.allclose(oracle.waveform(th2, det, 0.3, f), h * np.exp(0.3j), rtol=1e-11)


# ---- P4: noise statistics / inner product ---------------------------------------------------------
def test_p4_noise_inner_product_statistics(oracle, wl2):
    # <n,n> per detector has mean 2 N_f and sd 2 sqrt(N_f); logL(theta_inj) = -1/2 sum <n,n>
    w = copy.copy(wl2)
    p = oracle.Problem(w, kind=1)
    nf = w.n_freq
    l = p.loglike(w.theta_inj[w.param_index])
    assert abs(l + w.n_det * nf) < 4.0 * math.sqrt(w.n_det * nf)
    noise = inputs.make_noise(w)
    direct = -0.5 * np.sum(4 * w.df * np.abs(noise) ** 2 / w.psd)
    assert l == pytest.approx(direct, rel=1e-9)
    # DD is <d,d> summed over detectors, by numpy
    dat = w.data[..., 0] + 1j * w.data[..., 1]
    assert p.DD == pytest.approx(np.sum(4 * w.df * np.abs(dat) ** 2 / w.psd), rel=1e-12)


# ---- P5 / P9: noise-free closed forms, full grid AND relative binning -----------------------------
@pytest.mark.parametrize("cfg,B", [("config1", 32), ("config2", 128), ("config2", 17)])
def test_p5_noise_free_closed_forms(oracle, cfg, B):
    w = getattr(inputs, cfg)(n_bins=B)
    w = inputs.make_data(w, oracle.waveform, noise=False)
    rho2 = w.snr ** 2
    th = w.theta_inj[w.param_index].copy()
    for kind in (0, 1):
        p = oracle.Problem(w, kind=kind)
        assert p.DD == pytest.approx(rho2, rel=1e-12)                      # P9: SNR scaling exact
        assert abs(p.loglike(th)) < 1e-9                                   # logL(theta_inj) = 0
        if "dL" in [inputs.SLOT_NAMES[i] for i in w.param_index]:
            j = list(w.param_index).index(4)
            for fac in (0.5, 1.3, 2.0):
                t2 = th.copy(); t2[j] = th[j] * fac
                assert p.loglike(t2) == pytest.approx(-0.5 * rho2 * (1 / fac - 1) ** 2, rel=1e-9, abs=1e-9)
        j = list(w.param_index).index(6)
        for delta in (0.1, -0.7, 3.0):
            t2 = th.copy(); t2[j] = th[j] + delta
            assert p.loglike(t2) == pytest.approx(-rho2 * (1 - math.cos(delta)), rel=1e-9, abs=1e-9)


# ---- P6: RB exact at the fiducial point ------------------------------------------------------------
def test_p6_rb_equals_full_at_fiducial(oracle, wl1, wl2):
    for w in (wl1, wl2):
        p = oracle.Problem(w, kind=0)
        th = w.theta_fid[w.param_index]
        a, b = p.loglike(th, 0), p.loglike(th, 1)
        assert a == pytest.approx(b, rel=1e-13, abs=1e-9)


# ---- P7: B = N_f - 1 exact residual identity, prior-wide -------------------------------------------
def test_p7_every_grid_point_an_edge(oracle):
    w = inputs.make_data(inputs.config1(n_bins=1968), oracle.waveform)
    p = oracle.Problem(w, kind=0)
    idx, F = p.edges()
    assert np.array_equal(idx, np.arange(1969))
    summ = p.summary()                                   # [n_det, B, 6]
    X = inputs.draw_prior(w, 3, 11)
    for th in X:
        dh_full, hh_full, dh_rb, hh_rb = p.parts(th)
        assert dh_rb == pytest.approx(dh_full, rel=1e-11, abs=1e-9)      # linear interpolation exact at nodes
        # residual: RB drops the quadratic term; bin b owns only node b (last bin owns two):
        # hand-derived identity on the <h,h> part, evaluated here from the oracle's own waveform
        canon = w.theta_fixed.copy(); canon[w.param_index] = th
        r = oracle.waveform(canon, w.det[0], w.gmst, F) / oracle.waveform(w.theta_fid, w.det[0], w.gmst, F)
        h0 = oracle.waveform(w.theta_fid, w.det[0], w.gmst, F)
        wgt = 4 * w.df * np.abs(h0) ** 2 / w.psd[0]      # per-node weight
        # RB's |r|^2 at node k of bin b (first-order expansion about the bin centre, second-order term dropped)
        r0 = 0.5 * (r[:-1] + r[1:]); r1 = (r[1:] - r[:-1]) / np.diff(F)
        fbar = 0.5 * (F[:-1] + F[1:])
        approx = 0.0
        for b in range(1968):
            nodes = [b] if b < 1967 else [b, b + 1]
            for k in nodes:
                dfk = F[k] - fbar[b]
                approx += wgt[k] * (abs(r0[b]) ** 2 + 2 * dfk * (r0[b] * np.conj(r1[b])).real)
        assert hh_rb == pytest.approx(approx, rel=1e-11)
        exact = np.sum(wgt * np.abs(r) ** 2)
        assert hh_full == pytest.approx(exact, rel=1e-11)
        # and the difference is exactly the dropped quadratic term  sum w_k |r1|^2 (f_k - fbar)^2
        drop = 0.0
        for b in range(1968):
            nodes = [b] if b < 1967 else [b, b + 1]
            for k in nodes:
                drop += wgt[k] * abs(r1[b]) ** 2 * (F[k] - fbar[b]) ** 2
        assert hh_full - hh_rb == pytest.approx(drop, rel=1e-6, abs=1e-9)


# ---- P8: RB accuracy near the fiducial, and its B^-2 order -----------------------------------------
def _one_d_widths(p, w, th0):
    """omega_j: 1-D displacement at which the full-grid logL drops by 0.5 (A24)."""
    l0 = p.loglike(th0, 1)
    om = np.zeros(w.d)
    for j in range(w.d):
        step = (w.hi[j] - w.lo[j]) * 1e-6
        for _ in range(60):
            t = th0.copy(); t[j] += step
            if t[j] > w.hi[j] or l0 - p.loglike(t, 1) > 0.5:
                break
            step *= 1.5
        om[j] = step
    return om


def test_p8_rb_matches_full_grid_near_fiducial(oracle, wl2):
    w = wl2
    p = oracle.Problem(w, kind=0)
    th0 = w.theta_fid[w.param_index]
    om = _one_d_widths(p, w, th0)
    X = inputs.draw_near(w, 40, 3, 0.1 * om)
    err = [abs(p.loglike(x, 0) - p.loglike(x, 1)) for x in X]
    assert max(err) < 1e-3                       # north_star: within 1e-3 absolute near the fiducial point


def test_p8_rb_error_is_second_order_in_bins(oracle, wl2):
    w = wl2
    th0 = w.theta_fid[w.param_index]
    om = _one_d_widths(oracle.Problem(w, kind=1), w, th0)
    X = inputs.draw_near(w, 12, 4, 0.5 * om)
    errs = []
    for B in (64, 128, 256):
        p = oracle.Problem(w, kind=0, n_bins=B)
        errs.append(max(abs(p.loglike(x, 0) - p.loglike(x, 1)) for x in X))
    assert 2.5 < errs[0] / errs[1] < 6.0 and 2.5 < errs[1] / errs[2] < 6.0


# ---- O8: bin edges ----------------------------------------------------------------------------------
def test_bin_edges_structure(oracle, wl1, wl2):
    for w, B in ((wl1, 32), (wl2, 128), (wl2, 1024), (wl2, 4016)):
        p = oracle.Problem(w, kind=0, n_bins=B)
        idx, F = p.edges()
        assert idx[0] == 0 and idx[-1] == w.n_freq - 1 and np.all(np.diff(idx) >= 1)
        assert np.allclose(F, w.f_min + w.df * idx)
        if B <= 128:
            # equal increments of a monotone dephasing measure => bins widen with frequency
            assert np.diff(idx)[-1] > np.diff(idx)[0]
    # summary data are partial sums of the full inner product: sum_b A0_b = <d,h0>-like totals
    p = oracle.Problem(wl2, kind=0)
    s = p.summary()
    th = wl2.theta_fid[wl2.param_index]
    dh_full, hh_full, dh_rb, hh_rb = p.parts(th)
    assert s[..., 0].sum() == pytest.approx(dh_full, rel=1e-12)        # Re sum A0 = <d,h0>
    assert s[..., 4].sum() == pytest.approx(hh_full, rel=1e-12)        # sum B0 = <h0,h0>


def _o8_rows(path=None):
    """The hand-typed rows of tests/golden/o8_dephasing.txt: (gamma as an mpmath rational, sign, 'f_min' | 'f_max')."""
    import mpmath as mp
    path = path or os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "o8_dephasing.txt")
    rows = []
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        gam, sign, ref = (t.strip() for t in line.split("|"))
        p_, q_ = gam.split("/")
        rows.append((mp.mpf(int(p_)) / int(q_), int(sign), ref))
    return rows


def _o8_edges(rows, f_min, df, n_freq, B):
    """O8 written out from the fixture in 50-digit arithmetic: (edge indices after the monotonicity passes, raw nearest
    indices, smallest gap by which a raw choice beat its runner-up, relative to the delta range)."""
    import mpmath as mp
    mp.mp.dps = 50
    fmin, fmax = mp.mpf(f_min), mp.mpf(f_min) + (n_freq - 1) * mp.mpf(df)
    ref = {"f_min": fmin, "f_max": fmax}
    delta = [sum(sg * (((fmin + k * mp.mpf(df)) / ref[r]) ** g) for g, sg, r in rows) for k in range(n_freq)]
    d0, d1 = delta[0], delta[-1]
    raw, closest = [], mp.mpf(1)
    up = all(delta[k + 1] > delta[k] for k in range(n_freq - 1))
    for e in range(B + 1):
        t = d0 + mp.mpf(e) / B * (d1 - d0)
        if up:                                   # monotone: the nearest point is one of the two around the target
            lo_, hi_ = 0, n_freq - 1
            while hi_ - lo_ > 1:
                mid = (lo_ + hi_) // 2
                if delta[mid] <= t:
                    lo_ = mid
                else:
                    hi_ = mid
            cand = sorted({max(lo_ - 1, 0), lo_, hi_, min(hi_ + 1, n_freq - 1)})
        else:
            cand = range(n_freq)
        dist = sorted((abs(delta[k] - t), k) for k in cand)          # equal distances: the lower index first
        raw.append(dist[0][1])
        if len(dist) > 1:
            closest = min(closest, (dist[1][0] - dist[0][0]) / abs(d1 - d0))
    ie = list(raw)
    ie[0], ie[B] = 0, n_freq - 1
    for e in range(1, B + 1):
        ie[e] = max(ie[e], ie[e - 1] + 1)
    ie[B] = n_freq - 1
    for e in range(B - 1, -1, -1):
        ie[e] = min(ie[e], ie[e + 1] - 1)
    return np.array(ie), np.array(raw), float(closest)


def test_p17_bin_edges_from_the_dephasing_fixture(oracle, wl1, wl2):
    """P17 (O8, readings A7 / A8).  The power laws, their signs and the f_min / f_max normalisation are read from a
    fixture typed by hand from SURVEY.md:397-403; the edges are rebuilt from it in 50-digit arithmetic (nearest grid
    point to each equal-increment target, ties to the lower index, then the forward / backward passes) and must equal
    the oracle's, index for index, for B in {32, 128, 1024} on both frequency grids (config 1: 20-512 Hz, config 2:
    20-1024 Hz).  A dropped power law, a flipped sign and swapped reference frequencies each give different edges, so
    a slip of that kind in the oracle fails here (before this pin only the GPU's bit-exact edge comparison saw it)."""
    rows = _o8_rows()
    assert len(rows) == 5
    for g_, sg, r in rows:                        # the rule the survey states beside the list
        assert sg == (1 if g_ > 0 else -1) and r == ("f_max" if g_ > 0 else "f_min")
    mutants = {
        "a power law dropped": [x for x in rows if x[0] != 1],
        "a sign flipped": [(g_, -sg if i == 1 else sg, r) for i, (g_, sg, r) in enumerate(rows)],
        "f_min and f_max swapped": [(g_, sg, "f_min" if r == "f_max" else "f_max") for g_, sg, r in rows],
        "an exponent mistyped (5/3 -> 4/3)": [((g_ if i != 3 else g_ - g_ / 5), sg, r) for i, (g_, sg, r) in enumerate(rows)],
    }
    for w in (wl1, wl2):
        for B in (32, 128, 1024):
            idx, F = oracle.Problem(w, kind=0, n_bins=B).edges()
            want, raw, closest = _o8_edges(rows, w.f_min, w.df, w.n_freq, B)
            assert closest > 1e-9, "a target sits within rounding of a tie: fp64 and 50 digits may choose differently"
            assert np.array_equal(idx, want), (w.name, B, np.flatnonzero(idx != want)[:5])
            free = np.flatnonzero((np.diff(idx)[:-1] > 1) & (np.diff(idx)[1:] > 1)) + 1     # edges no pass has moved
            assert free.size > B // 4 and np.array_equal(idx[free], raw[free])              # ... are the nearest points
            assert np.array_equal(F, w.f_min + w.df * idx)
            if B == 128:
                for what, rows_m in mutants.items():
                    bad, _, _ = _o8_edges(rows_m, w.f_min, w.df, w.n_freq, B)
                    assert not np.array_equal(bad, idx), f"{what}: the pin cannot see it"
                    assert np.sum(bad != idx) > B // 4, what


def test_p17_bin_ownership_and_centres(oracle, wl2):
    """A8.  Half-open ownership [i_b, i_b+1) (last bin closed) makes the bins a partition of the grid, and the centre of
    bin b is the mid-point of its two EDGE frequencies: with C_k = 4 df d_k conj(h0_k) / S_k,
    sum_b A0_b = sum_k C_k and sum_b (A1_b + fbar_b A0_b) = sum_k C_k f_k whatever the bins are; likewise B0, B1 with
    |h0_k|^2.  Computed here from the data and the fiducial strain directly, never through a bin.  A closed interval
    (edge points counted twice), a last point left out, or a centre at the mean of the owned frequencies breaks one."""
    w = wl2
    f = w.freqs
    for B in (128, 1000):
        p = oracle.Problem(w, kind=0, n_bins=B)
        idx, F = p.edges()
        fbar = 0.5 * (F[:-1] + F[1:])
        s = p.summary()
        for a in range(w.n_det):
            h0 = oracle.waveform(w.theta_fid, w.det[a], w.gmst, f)
            d = w.data[a, :, 0] + 1j * w.data[a, :, 1]
            C = 4 * w.df * d * np.conj(h0) / w.psd[a]
            Q = 4 * w.df * np.abs(h0) ** 2 / w.psd[a]
            A0, A1 = s[a, :, 0] + 1j * s[a, :, 1], s[a, :, 2] + 1j * s[a, :, 3]
            assert abs(A0.sum() - C.sum()) <= 1e-11 * np.abs(C).sum()
            assert abs((A1 + fbar * A0).sum() - (C * f).sum()) <= 1e-11 * np.abs(C * f).sum()
            assert abs(s[a, :, 4].sum() - Q.sum()) <= 1e-12 * Q.sum()
            assert abs((s[a, :, 5] + fbar * s[a, :, 4]).sum() - (Q * f).sum()) <= 1e-12 * (Q * f).sum()
            # per bin, on the first, a middle and the last bin (the one that also owns i_B)
            for b in (0, B // 2, B - 1):
                own = slice(idx[b], idx[b + 1] + (1 if b == B - 1 else 0))
                assert abs(A0[b] - C[own].sum()) <= 1e-11 * np.abs(C[own]).sum()
                assert abs(A1[b] - (C[own] * (f[own] - fbar[b])).sum()) <= 1e-10 * np.abs(C[own] * (f[own] - fbar[b])).sum() + 1e-300


def test_domain_and_nonfinite(oracle, wl2):
    p = oracle.Problem(wl2)
    th = wl2.theta_fid[wl2.param_index].copy()
    for j, bad in ((0, -1.0), (1, 1.2), (1, 0.0), (2, 1.0), (4, 0.0), (5, float("nan")), (6, float("inf"))):
        t = th.copy(); t[j] = bad
        assert p.loglike(t) == -math.inf
