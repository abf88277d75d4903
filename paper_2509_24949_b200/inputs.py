"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no waveform, no likelihood, no sampler): it
only describes workloads (BASELINE.json configs 1-5) and draws seeded noise and
parameter vectors.  The injected signal is produced by a `waveform_fn` callback supplied by the
caller: the tests pass the oracle's waveform, bench.py passes the CUDA library's own host-side
`nss_waveform`; neither side's data ever comes from the other.

The paper measures on GW150914 public strain with IMRPhenomD; that data set is
not available here.  These inputs stand in for it: multi-detector frequency-domain strain,
coloured Gaussian noise, a compact-binary chirp injection, 4 or 11 sampled parameters, a
heterodyne reference fixed in advance.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Callable, Optional

import numpy as np

NSLOT = 11
SLOT_NAMES = ("Mc", "q", "chi1z", "chi2z", "dL", "tc", "phic", "iota", "psi", "ra", "dec")

# Earth-fixed detector geometry: vertex [m], x-arm, y-arm unit vectors (inputs).
DETECTORS = {
    "H1": ((-2.16141492636e6, -3.83469517889e6, 4.60035022664e6),
           (-0.22389266154, 0.79983062746, 0.55690487831),
           (-0.91397818574, 0.02609403989, -0.40492342125)),
    "L1": ((-7.42760447238e4, -5.49628371971e6, 3.22425701744e6),
           (-0.95457412153, -0.14158077340, -0.26218911324),
           (0.29774156894, -0.48791033647, -0.82054461286)),
    "V1": ((4.54637409900e6, 8.42989697626e5, 4.37857696241e6),
           (-0.70045821479, 0.20848948619, 0.68256166277),
           (-0.05379255368, -0.96908180549, 0.24080451708)),
    # config 1's synthetic detector: |F+| = 1, Fx = 0 at ra=0, dec=pi/2, psi=0, gmst=0
    "SYN": ((0.0, 0.0, 0.0), (1.0, 0.0, 0.0), (0.0, 1.0, 0.0)),
}


def detector_array(names) -> np.ndarray:
    """[n_det, 9] = vertex, xarm, yarm."""
    return np.array([np.concatenate(DETECTORS[n]) for n in names], dtype=np.float64)


def psd_white(f: np.ndarray, level: float = 1e-46) -> np.ndarray:
    return np.full_like(f, level, dtype=np.float64)


def psd_aligo_fit(f: np.ndarray, s0: float = 1e-49) -> np.ndarray:
    """BASELINE.json config 2: S0[x^-4.14 - 5x^-2 + 111(1 - x^2 + x^4/2)/(1 + x^2/2)], x = f/215 Hz."""
    x = np.asarray(f, dtype=np.float64) / 215.0
    return s0 * (x ** -4.14 - 5.0 * x ** -2 + 111.0 * (1.0 - x ** 2 + 0.5 * x ** 4) / (1.0 + 0.5 * x ** 2))


@dataclass
class Workload:
    """Everything nss_create / orc_create needs, plus the sampler settings of the config."""
    name: str
    d: int
    param_index: np.ndarray      # [d] sampled dim -> canonical slot
    theta_fixed: np.ndarray      # [11]
    lo: np.ndarray               # [d]
    hi: np.ndarray               # [d]
    det_names: tuple
    det: np.ndarray              # [n_det, 9]
    gmst: float
    n_freq: int
    f_min: float
    df: float
    psd: np.ndarray              # [n_det, n_freq]
    data: Optional[np.ndarray]   # [n_det, n_freq, 2]; None until make_data()
    theta_fid: np.ndarray        # [11]
    theta_inj: np.ndarray        # [11]
    n_bins: int
    kind: int                    # 0 RB, 1 full grid, 2 Gaussian
    n_live: int
    n_delete: int
    n_repeats: int
    snr: float
    noise_seed: int
    gauss_mu: np.ndarray = field(default_factory=lambda: np.zeros(NSLOT))
    gauss_sigma: np.ndarray = field(default_factory=lambda: np.ones(NSLOT))

    @property
    def n_det(self) -> int:
        return len(self.det_names)

    @property
    def freqs(self) -> np.ndarray:
        return self.f_min + self.df * np.arange(self.n_freq, dtype=np.float64)


def _grid(f_lo: float, f_hi: float, df: float):
    n = int(round((f_hi - f_lo) / df)) + 1
    return n


def config1(n_bins: int = 32) -> Workload:
    """Tiny 4-parameter, one synthetic detector, white PSD (BASELINE.json configs[0])."""
    pidx = np.array([0, 1, 5, 6], dtype=np.int32)
    inj = np.array([30.0, 0.8, 0.0, 0.0, 1000.0, 0.0, 1.0, 0.0, 0.0, 0.0, math.pi / 2], dtype=np.float64)
    n = _grid(20.0, 512.0, 0.25)
    f = 20.0 + 0.25 * np.arange(n)
    return Workload(
        name="config1", d=4, param_index=pidx, theta_fixed=inj.copy(),
        lo=np.array([20.0, 0.3, -0.1, 0.0]), hi=np.array([40.0, 1.0, 0.1, 2 * math.pi]),
        det_names=("SYN",), det=detector_array(("SYN",)), gmst=0.0,
        n_freq=n, f_min=20.0, df=0.25, psd=psd_white(f)[None, :].copy(), data=None,
        theta_fid=inj.copy(), theta_inj=inj.copy(), n_bins=n_bins, kind=0,
        n_live=100, n_delete=50, n_repeats=12, snr=15.0, noise_seed=7)


def config2(n_bins: int = 128, kind: int = 0, n_live: int = 1000, n_delete: int = 500) -> Workload:
    """11-parameter aligned-spin BBH, H1+L1+V1, analytic PSD (BASELINE.json configs[1]);
    configs[2] = n_live 5000 / n_delete 2500; configs[3] = kind 1 (full grid)."""
    pidx = np.arange(11, dtype=np.int32)
    inj = np.array([30.0, 0.8, 0.1, -0.05, 1000.0, 0.0, 1.0, 0.6, 0.8, 1.5, -0.5], dtype=np.float64)
    n = _grid(20.0, 1024.0, 0.25)
    f = 20.0 + 0.25 * np.arange(n)
    names = ("H1", "L1", "V1")
    psd = np.tile(psd_aligo_fit(f)[None, :], (3, 1))
    lo = np.array([20.0, 0.3, -0.9, -0.9, 500.0, -0.1, 0.0, 0.0, 0.0, 0.0, -math.pi / 2])
    hi = np.array([40.0, 1.0, 0.9, 0.9, 8000.0, 0.1, 2 * math.pi, math.pi, math.pi, 2 * math.pi, math.pi / 2])
    return Workload(
        name="config2", d=11, param_index=pidx, theta_fixed=inj.copy(), lo=lo, hi=hi,
        det_names=names, det=detector_array(names), gmst=0.0,
        n_freq=n, f_min=20.0, df=0.25, psd=psd, data=None,
        theta_fid=inj.copy(), theta_inj=inj.copy(), n_bins=n_bins, kind=kind,
        n_live=n_live, n_delete=n_delete, n_repeats=55, snr=20.0, noise_seed=1)


def config3() -> Workload:
    w = config2(n_live=5000, n_delete=2500)
    w.name = "config3"
    return w


def config4() -> Workload:
    w = config2(kind=1)
    w.name = "config4"
    return w


def config5(n_bins: int) -> Workload:
    w = config2(n_bins=n_bins)
    w.name = f"config5_B{n_bins}"
    return w


def gaussian_workload(d: int, sigma: float = 0.05, half_width: float = 1.0,
                      n_live: int = 1000, n_delete: int = 500, n_repeats: Optional[int] = None) -> Workload:
    """O16 test likelihood: d-dim Gaussian (peak 0) in a uniform box; analytic logZ known."""
    z = np.zeros(NSLOT)
    return Workload(
        name=f"gauss{d}", d=d, param_index=np.arange(d, dtype=np.int32), theta_fixed=z.copy(),
        lo=np.full(d, -half_width), hi=np.full(d, half_width), det_names=(), det=np.zeros((0, 9)),
        gmst=0.0, n_freq=0, f_min=0.0, df=0.0, psd=np.zeros((0, 0)), data=np.zeros((0, 0, 2)),
        theta_fid=z.copy(), theta_inj=z.copy(), n_bins=0, kind=2, n_live=n_live, n_delete=n_delete,
        n_repeats=n_repeats if n_repeats is not None else 5 * d, snr=0.0, noise_seed=0,
        gauss_mu=np.concatenate([np.zeros(d), np.zeros(NSLOT - d)]),
        gauss_sigma=np.concatenate([np.full(d, sigma), np.ones(NSLOT - d)]))


def make_noise(w: Workload) -> np.ndarray:
    """O6: n_k = sqrt(S_k / (4 df)) (a_k + i b_k), a, b ~ N(0,1) i.i.d.; [n_det, n_freq] complex128."""
    rng = np.random.Generator(np.random.PCG64(w.noise_seed))
    ab = rng.standard_normal((w.n_det, w.n_freq, 2))
    return np.sqrt(w.psd / (4.0 * w.df)) * (ab[..., 0] + 1j * ab[..., 1])


WaveformFn = Callable[[np.ndarray, np.ndarray, float, np.ndarray], np.ndarray]
"""waveform_fn(theta_canon[11], det9[9], gmst, freqs[n]) -> complex128[n]"""


def make_data(w: Workload, waveform_fn: WaveformFn, noise: bool = True) -> Workload:
    """O6: scale d_L so the network SNR of the injection is w.snr, then data = h(theta_inj) + noise.
    Fiducial = injection.  Fills w.data, w.theta_inj, w.theta_fid, w.theta_fixed in place."""
    f = w.freqs
    d_ref = 1000.0
    th = w.theta_inj.copy()
    th[4] = d_ref
    h = np.stack([waveform_fn(th, w.det[a], w.gmst, f) for a in range(w.n_det)])
    rho_ref = math.sqrt(float(np.sum(4.0 * w.df * np.abs(h) ** 2 / w.psd)))
    dl = d_ref * rho_ref / w.snr
    th[4] = dl
    h = np.stack([waveform_fn(th, w.det[a], w.gmst, f) for a in range(w.n_det)])
    dat = h + (make_noise(w) if noise else 0.0)
    w.data = np.ascontiguousarray(np.stack([dat.real, dat.imag], axis=-1))
    w.theta_inj = th.copy()
    w.theta_fid = th.copy()
    fixed = w.theta_fixed.copy()
    fixed[4] = dl
    w.theta_fixed = fixed
    return w


def draw_prior(w: Workload, n: int, seed: int) -> np.ndarray:
    """n parameter vectors uniform in the prior box; [n, d] float64 (config 5 uses seed 5)."""
    rng = np.random.Generator(np.random.Philox(seed))
    u = rng.random((n, w.d))
    return w.lo[None, :] + (w.hi - w.lo)[None, :] * u


def draw_near(w: Workload, n: int, seed: int, scale: np.ndarray) -> np.ndarray:
    """theta_fid + scale * g / sqrt(d), g ~ N(0, I) (A24), clipped to the box; [n, d]."""
    rng = np.random.Generator(np.random.Philox(seed))
    g = rng.standard_normal((n, w.d))
    centre = w.theta_fid[w.param_index]
    x = centre[None, :] + np.asarray(scale)[None, :] * g / math.sqrt(w.d)
    return np.clip(x, w.lo[None, :], w.hi[None, :])
