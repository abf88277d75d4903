"""ctypes wrapper over oracle/nss_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  It never imports paper_2509_24949_b200.nss (the CUDA binding), and the CUDA path
never imports this.  `build()` compiles the C file with gcc (-O2 -march=native, no fast-math,
-ffp-contract=off so every expression rounds as written).
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nss_oracle.c")
_LIB = os.path.join(_HERE, "libnss_oracle.so")
_lib = None

c_dp = C.POINTER(C.c_double)
c_ip = C.POINTER(C.c_int)


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-std=c99", "-O2", "-march=native", "-ffp-contract=off", "-fopenmp", "-fPIC",
               "-shared", "-Wall", "-Wextra", _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _dp(a):
    return a.ctypes.data_as(c_dp) if a is not None else None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int, c_ip, c_dp, c_dp, c_dp, C.c_int, c_dp, C.c_double, C.c_int,
                                 C.c_double, C.c_double, c_dp, c_dp, c_dp, C.c_int, C.c_int, c_dp, c_dp]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_set_periodic.argtypes = [C.c_void_p, c_ip]
        L.orc_set_periodic.restype = None
        L.orc_loglike.restype = C.c_double
        L.orc_loglike.argtypes = [C.c_void_p, c_dp]
        L.orc_loglike_kind.restype = C.c_double
        L.orc_loglike_kind.argtypes = [C.c_void_p, c_dp, C.c_int]
        L.orc_loglike_batch.argtypes = [C.c_void_p, c_dp, C.c_int64, c_dp, C.c_int]
        L.orc_get_DD.restype = C.c_double
        L.orc_get_DD.argtypes = [C.c_void_p]
        L.orc_get_edges.argtypes = [C.c_void_p, c_ip, c_dp]
        L.orc_get_summary.argtypes = [C.c_void_p, c_dp]
        L.orc_waveform.argtypes = [c_dp, c_dp, C.c_double, c_dp, C.c_int, c_dp]
        L.orc_antenna_flat.argtypes = [c_dp, C.c_double, C.c_double, C.c_double, C.c_double, c_dp]
        L.orc_parts.argtypes = [C.c_void_p, c_dp, c_dp]
        L.orc_phase.restype = C.c_double
        L.orc_phase.argtypes = [C.c_double, c_dp]
        L.orc_phase_newtonian.restype = C.c_double
        L.orc_phase_newtonian.argtypes = [C.c_double, c_dp]
        L.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32)] * 3
        L.orc_draw53.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32,
                                 C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
        L.orc_uniform_a.restype = C.c_double
        L.orc_uniform_a.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32]
        L.orc_normal_pair.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, c_dp, c_dp]
        L.orc_init_live.argtypes = [C.c_void_p, C.c_int, C.c_uint64, c_dp, c_dp, C.c_int]
        L.orc_select_lowest.argtypes = [c_dp, C.c_int, C.c_int, c_ip, c_ip]
        L.orc_logaddexp.restype = C.c_double
        L.orc_logaddexp.argtypes = [C.c_double, C.c_double]
        L.orc_evidence_update.argtypes = [c_dp, C.c_int, C.c_int, c_dp, c_dp, c_dp]
        L.orc_tune.restype = C.c_int
        L.orc_tune_periodic.restype = C.c_int
        L.orc_tune_periodic.argtypes = [c_dp, C.c_int, C.c_int, c_ip, c_dp, c_dp, c_dp, c_dp, c_dp]
        L.orc_tune.argtypes = [c_dp, C.c_int, C.c_int, c_dp, c_dp, c_dp]
        L.orc_replace_step.restype = C.c_int
        L.orc_replace_step.argtypes = [C.c_void_p, c_dp, c_dp, C.c_int, C.c_int, C.c_double, C.c_int,
                                       C.c_uint64, C.c_uint32, c_dp, c_dp, c_ip, c_dp,
                                       C.POINTER(C.c_int64), C.POINTER(C.c_int32), c_dp, C.c_int]
        L.orc_run.restype = C.c_int
        L.orc_run.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_uint64, C.c_double, C.c_int,
                              C.c_int64, c_dp, c_dp, c_dp, c_dp, c_dp, C.c_int]
        L.orc_resample_equal.restype = C.c_int64
        L.orc_resample_equal.argtypes = [c_dp, c_dp, C.c_int64, C.c_uint64, C.POINTER(C.c_int64)]
        _lib = L
    return _lib


def n_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def _f64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def waveform(theta_canon, det9, gmst, freqs) -> np.ndarray:
    """O3/O4 strain of one detector; complex128[n]."""
    th, det9, f = _f64(theta_canon), _f64(det9), _f64(freqs)
    out = np.empty((f.size, 2))
    lib().orc_waveform(_dp(th), _dp(det9), float(gmst), _dp(f), f.size, _dp(out))
    return out[:, 0] + 1j * out[:, 1]


def antenna(det9, gmst, ra, dec, psi):
    """O4: (F+, Fx, dt)."""
    out = np.empty(3)
    lib().orc_antenna_flat(_dp(_f64(det9)), gmst, ra, dec, psi, _dp(out))
    return tuple(out)


def phase(f, theta_canon, newtonian=False) -> float:
    th = _f64(theta_canon)
    fn = lib().orc_phase_newtonian if newtonian else lib().orc_phase
    return fn(float(f), _dp(th))


def philox(key, ctr):
    k = (C.c_uint32 * 2)(*key)
    c = (C.c_uint32 * 4)(*ctr)
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(k, c, o)
    return tuple(int(x) for x in o)


def draw53(seed, block, step, chain, iteration):
    a, b = C.c_uint64(), C.c_uint64()
    lib().orc_draw53(seed, block, step, chain, iteration, C.byref(a), C.byref(b))
    return a.value, b.value


def uniform_a(seed, block, step, chain, iteration) -> float:
    return lib().orc_uniform_a(seed, block, step, chain, iteration)


def normal_pair(seed, block, step, chain, iteration):
    a, b = C.c_double(), C.c_double()
    lib().orc_normal_pair(seed, block, step, chain, iteration, C.byref(a), C.byref(b))
    return a.value, b.value


def select_lowest(logL, k):
    l = _f64(logL)
    dead = np.empty(k, dtype=np.int32)
    surv = np.empty(l.size - k, dtype=np.int32)
    lib().orc_select_lowest(_dp(l), l.size, k, dead.ctypes.data_as(c_ip), surv.ctypes.data_as(c_ip))
    return dead, surv


def evidence_update(dead_logL, n, logX, logZ):
    dl = _f64(dead_logL)
    lw = np.empty(dl.size)
    x, z = C.c_double(logX), C.c_double(logZ)
    lib().orc_evidence_update(_dp(dl), n, dl.size, C.byref(x), C.byref(z), _dp(lw))
    return x.value, z.value, lw


def resample_equal(logL, logw, seed) -> np.ndarray:
    """Reading R6: row indices of the equal-weight posterior sample (ascending)."""
    l, w = _f64(logL), _f64(logw)
    idx = np.empty(l.size, dtype=np.int64)
    m = lib().orc_resample_equal(_dp(l), _dp(w), l.size, int(seed), idx.ctypes.data_as(C.POINTER(C.c_int64)))
    return idx[:m].copy()


def tune(live):
    a = _f64(live)
    n, d = a.shape
    mean, cov, chol = np.empty(d), np.empty((d, d)), np.empty((d, d))
    rc = lib().orc_tune(_dp(a), n, d, _dp(mean), _dp(cov), _dp(chol))
    return rc, mean, cov, chol


def tune_periodic(live, flags, lo, hi):
    """Reading R7: moments of the live points with every flagged coordinate unwrapped around its circular mean."""
    a = _f64(live)
    n, d = a.shape
    f = np.ascontiguousarray(np.asarray(flags, dtype=np.int32)[:d])
    lo_, hi_ = _f64(lo), _f64(hi)
    mean, cov, chol = np.empty(d), np.empty((d, d)), np.empty((d, d))
    rc = lib().orc_tune_periodic(_dp(a), n, d, f.ctypes.data_as(c_ip), _dp(lo_), _dp(hi_), _dp(mean), _dp(cov), _dp(chol))
    return rc, mean, cov, chol


class Problem:
    """One likelihood problem (orc_create); takes a paper_2509_24949_b200.inputs.Workload-like object."""

    def __init__(self, w, kind=None, n_bins=None):
        self.w = w
        self.d = int(w.d)
        kind = int(w.kind if kind is None else kind)
        n_bins = int(w.n_bins if n_bins is None else n_bins)
        self.kind, self.n_bins = kind, n_bins
        pidx = np.ascontiguousarray(w.param_index, dtype=np.int32)
        keep = [_f64(w.theta_fixed), _f64(w.lo), _f64(w.hi), _f64(w.det).ravel(), _f64(w.psd).ravel(),
                _f64(w.data).ravel() if w.data is not None else np.zeros(0), _f64(w.theta_fid),
                _f64(w.gauss_mu), _f64(w.gauss_sigma)]
        self._h = lib().orc_create(self.d, pidx.ctypes.data_as(c_ip), _dp(keep[0]), _dp(keep[1]), _dp(keep[2]),
                                   int(w.n_det), _dp(keep[3]), float(w.gmst), int(w.n_freq), float(w.f_min),
                                   float(w.df), _dp(keep[4]), _dp(keep[5]), _dp(keep[6]), n_bins, kind,
                                   _dp(keep[7]), _dp(keep[8]))
        if not self._h:
            raise ValueError("orc_create rejected the problem")

    def set_periodic(self, flags):
        """NEXT-2: sampled dim j wraps in [lo_j, hi_j) when flags[j] != 0 (default: hard walls, A16)."""
        f = np.zeros(11, dtype=np.int32)
        f[: self.d] = np.asarray(flags, dtype=np.int32)[: self.d]
        lib().orc_set_periodic(self._h, f.ctypes.data_as(c_ip))

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_destroy(self._h)
            self._h = None

    def loglike(self, theta, kind=None) -> float:
        t = _f64(theta)
        if kind is None:
            return lib().orc_loglike(self._h, _dp(t))
        return lib().orc_loglike_kind(self._h, _dp(t), kind)

    def loglike_batch(self, theta, nthreads=None) -> np.ndarray:
        t = _f64(theta).reshape(-1, self.d)
        out = np.empty(t.shape[0])
        lib().orc_loglike_batch(self._h, _dp(t), t.shape[0], _dp(out), nthreads or n_cores())
        return out

    def parts(self, theta):
        """(<d,h>_full, <h,h>_full, <d,h>_RB, <h,h>_RB)."""
        t, out = _f64(theta), np.zeros(4)
        lib().orc_parts(self._h, _dp(t), _dp(out))
        return tuple(out)

    @property
    def DD(self) -> float:
        return lib().orc_get_DD(self._h)

    def edges(self):
        idx = np.empty(self.n_bins + 1, dtype=np.int32)
        f = np.empty(self.n_bins + 1)
        lib().orc_get_edges(self._h, idx.ctypes.data_as(c_ip), _dp(f))
        return idx, f

    def summary(self) -> np.ndarray:
        out = np.empty((self.w.n_det, self.n_bins, 6))
        lib().orc_get_summary(self._h, _dp(out))
        return out

    def init_live(self, n, seed, nthreads=None):
        live, logL = np.empty((n, self.d)), np.empty(n)
        lib().orc_init_live(self._h, n, seed, _dp(live), _dp(logL), nthreads or n_cores())
        return live, logL

    def replace_step(self, live, logL, n_delete, n_repeats, seed, iteration, logLstar=math.nan,
                     want_trace=False, nthreads=None):
        """O12 on copies of (live, logL); returns a dict."""
        live, logL = _f64(live).copy(), _f64(logL).copy()
        n, k = live.shape[0], int(n_delete)
        dth, dl = np.empty((k, self.d)), np.empty(k)
        didx = np.empty(k, dtype=np.int32)
        ls, ne = C.c_double(), C.c_int64()
        trace = np.zeros((k, n_repeats, 3), dtype=np.int32) if want_trace else None
        margin = np.empty(k) if want_trace else None
        rc = lib().orc_replace_step(self._h, _dp(live), _dp(logL), n, k, float(logLstar), int(n_repeats),
                                    int(seed), int(iteration), _dp(dth), _dp(dl), didx.ctypes.data_as(c_ip),
                                    C.byref(ls), C.byref(ne),
                                    trace.ctypes.data_as(C.POINTER(C.c_int32)) if want_trace else None,
                                    _dp(margin), nthreads or n_cores())
        return dict(rc=rc, live=live, logL=logL, dead_theta=dth, dead_logL=dl, dead_idx=didx,
                    logLstar=ls.value, n_evals=ne.value, trace=trace, margin=margin)

    def run(self, n_live, n_delete, n_repeats, seed, stop_dlogz=-3.0, max_iter=10000, nthreads=None, cap=None):
        if cap is None:                      # rows of the caller-side result arrays (no arithmetic depends on it)
            cap = int(n_delete) * int(max_iter) + int(n_live) if max_iter < 400 else 400 * n_delete + n_live
        cap = int(cap)
        dth, dl = np.empty((cap, self.d)), np.empty(cap)
        db, dw, scal = np.empty(cap), np.empty(cap), np.zeros(6)
        rc = lib().orc_run(self._h, n_live, n_delete, n_repeats, int(seed), stop_dlogz, max_iter, cap,
                           _dp(dth), _dp(dl), _dp(db), _dp(dw), _dp(scal), nthreads or n_cores())
        nd = int(scal[4])
        return dict(rc=rc, logZ=scal[0], logZ_err=scal[1], H=scal[2], n_iter=int(scal[3]), n_dead=nd,
                    n_evals=int(scal[5]), dead_theta=dth[:nd], dead_logL=dl[:nd], dead_logL_birth=db[:nd],
                    dead_logw=dw[:nd])
