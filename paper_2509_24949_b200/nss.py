"""Thin ctypes binding over csrc/libnss.so (include/nss.h) — argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; torch is used for device
memory and streams.  There is no CPU fallback: if the library is missing or has not been built,
loading raises.  Function names mirror the C ABI.
"""
from __future__ import annotations

import ctypes as C
import math
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "csrc", "libnss.so")
NSLOT, MAXDET = 11, 4

NSS_OK, NSS_EINVAL, NSS_ENOMEM, NSS_ECUDA, NSS_ECHOL, NSS_ECAP, NSS_ENOTCONV, NSS_ELIMIT = 0, -1, -2, -3, -4, -5, -6, -7
SELECT_STATIC_MAX_LIVE = 8192
KIND_RB, KIND_FULL, KIND_GAUSS = 0, 1, 2


class NssError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        msg = lib().nss_strerror(code).decode()
        if code == NSS_ECUDA:
            msg += ": " + lib().nss_last_cuda_error().decode()
        super().__init__(f"{where}: {msg} ({code})")


class nss_detector(C.Structure):
    _fields_ = [("vertex_m", C.c_double * 3), ("xarm", C.c_double * 3), ("yarm", C.c_double * 3)]


class nss_config(C.Structure):
    _fields_ = [
        ("d", C.c_int32), ("param_index", C.c_int32 * NSLOT), ("theta_fixed", C.c_double * NSLOT),
        ("lo", C.c_double * NSLOT), ("hi", C.c_double * NSLOT), ("n_det", C.c_int32),
        ("det", nss_detector * MAXDET), ("gmst", C.c_double), ("n_freq", C.c_int32),
        ("f_min", C.c_double), ("df", C.c_double), ("psd", C.POINTER(C.c_double)),
        ("data", C.POINTER(C.c_double)), ("theta_fid", C.c_double * NSLOT), ("n_bins", C.c_int32),
        ("kind", C.c_int32), ("gauss_mu", C.c_double * NSLOT), ("gauss_sigma", C.c_double * NSLOT)]


class nss_result(C.Structure):
    _fields_ = [
        ("logZ", C.c_double), ("logZ_err", C.c_double), ("H", C.c_double), ("n_iter", C.c_int32),
        ("n_dead", C.c_int64), ("n_evals", C.c_int64), ("dead_theta", C.POINTER(C.c_double)),
        ("dead_logL", C.POINTER(C.c_double)), ("dead_logL_birth", C.POINTER(C.c_double)),
        ("dead_logw", C.POINTER(C.c_double)), ("cap", C.c_int64), ("gpu_ms", C.c_double), ("ess", C.c_double),
        ("n_equal", C.c_int64), ("equal_idx", C.POINTER(C.c_int64))]


class nss_iter_state(C.Structure):
    _fields_ = [("logX", C.c_double), ("logZ", C.c_double), ("logZ_live", C.c_double), ("logLstar", C.c_double),
                ("n_evals", C.c_int64), ("converged", C.c_int32), ("pad_", C.c_int32)]


EXPORTS = ("nss_create", "nss_destroy", "nss_loglike_batch", "nss_loglike_batch_host", "nss_set_loglike_variant",
           "nss_replace_step", "nss_iterate", "nss_iterate_host",
           "nss_set_trace", "nss_select_lowest", "nss_select_lowest_static", "nss_tune", "nss_evidence_update", "nss_init_live",
           "nss_philox", "nss_run", "nss_resample_equal", "nss_waveform", "nss_get_tables", "nss_fp64_peak", "nss_launch_count",
           "nss_last_chain_ms", "nss_set_chain_timing", "nss_set_chain_warps", "nss_set_chain_lanes", "nss_set_chain_pack", "nss_last_chain_diag", "nss_set_periodic",
           "nss_strerror", "nss_last_cuda_error", "nss_version")

_lib = None
c_dp = C.POINTER(C.c_double)
vp = C.c_void_p


def lib():
    """Load libnss.so; raise loudly if it is missing (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2509_24949_b200.build` "
                              "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        L.nss_create.argtypes = [C.POINTER(nss_config), C.POINTER(vp)]
        L.nss_destroy.argtypes = [vp]
        L.nss_loglike_batch.argtypes = [vp, vp, C.c_int64, vp, vp]
        L.nss_set_loglike_variant.argtypes = [vp, C.c_int32]
        L.nss_replace_step.argtypes = [vp, vp, vp, C.c_int32, C.c_int32, C.c_double, C.c_int32, C.c_uint64,
                                       C.c_uint32, vp, vp, vp, c_dp, C.POINTER(C.c_int64), vp]
        L.nss_set_trace.argtypes = [vp, vp, vp]
        L.nss_iterate.argtypes = [vp, vp, vp, C.c_int32, C.c_int32, C.c_int32, C.c_uint64, C.c_uint32, C.c_double,
                                  vp, vp, vp, vp, C.POINTER(nss_iter_state), vp]
        L.nss_iterate_host.argtypes = L.nss_iterate.argtypes
        L.nss_loglike_batch_host.argtypes = [vp, vp, C.c_int64, vp, vp]
        L.nss_select_lowest.argtypes = [vp, vp, C.c_int32, C.c_int32, vp, vp, c_dp, vp]
        L.nss_select_lowest_static.argtypes = [vp, C.c_int32, C.c_int32, vp, vp, vp, vp]
        L.nss_tune.argtypes = [vp, vp, C.c_int32, vp, vp, vp]
        L.nss_evidence_update.argtypes = [vp, vp, C.c_int32, C.c_int32, vp, c_dp, vp]
        L.nss_init_live.argtypes = [vp, C.c_int32, C.c_uint64, vp, vp, vp]
        L.nss_philox.argtypes = [vp, C.c_uint64, vp, C.c_int64, vp, vp]
        L.nss_run.argtypes = [vp, C.c_int32, C.c_int32, C.c_int32, C.c_uint64, C.c_double, C.c_int32,
                              C.POINTER(nss_result), vp]
        L.nss_resample_equal.argtypes = [vp, vp, vp, C.c_int64, C.c_uint64, vp, C.POINTER(C.c_int64), vp]
        L.nss_waveform.argtypes = [c_dp, C.POINTER(nss_detector), C.c_double, c_dp, C.c_int32, c_dp]
        L.nss_get_tables.argtypes = [vp, vp, c_dp, c_dp]
        L.nss_fp64_peak.argtypes = [C.c_double, c_dp, vp]
        L.nss_launch_count.argtypes = [vp]
        L.nss_last_chain_ms.argtypes = [vp, c_dp]
        L.nss_set_chain_warps.argtypes = [vp, C.c_int32]
        L.nss_set_chain_timing.argtypes = [vp, C.c_int32]
        L.nss_set_chain_lanes.argtypes = [vp, C.c_int32]
        L.nss_set_chain_pack.argtypes = [vp, C.c_int32]
        L.nss_set_periodic.argtypes = [vp, C.POINTER(C.c_int32)]
        L.nss_last_chain_diag.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        L.nss_launch_count.restype = C.c_int64
        L.nss_strerror.argtypes = [C.c_int]
        L.nss_strerror.restype = C.c_char_p
        L.nss_last_cuda_error.restype = C.c_char_p
        _lib = L
    return _lib


def _check(code, where, ok=(NSS_OK,)):
    if code not in ok:
        raise NssError(code, where)
    return code


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _det_struct(det9):
    s = nss_detector()
    for c in range(3):
        s.vertex_m[c], s.xarm[c], s.yarm[c] = float(det9[c]), float(det9[3 + c]), float(det9[6 + c])
    return s


def nss_waveform(theta_canon, det9, gmst, freqs) -> np.ndarray:
    """Host-side strain of one detector (O3, O4); complex128[n].  Signature matches inputs.WaveformFn."""
    th = np.ascontiguousarray(theta_canon, dtype=np.float64)
    f = np.ascontiguousarray(freqs, dtype=np.float64)
    out = np.empty((f.size, 2))
    det = _det_struct(det9)
    _check(lib().nss_waveform(th.ctypes.data_as(c_dp), C.byref(det), float(gmst), f.ctypes.data_as(c_dp), f.size,
                              out.ctypes.data_as(c_dp)), "nss_waveform")
    return out[:, 0] + 1j * out[:, 1]


def nss_fp64_peak(ms: float = 200.0) -> float:
    """Measured fp64 FMA throughput of the device, TFLOP/s (2 flop per FMA)."""
    out = C.c_double()
    _check(lib().nss_fp64_peak(float(ms), C.byref(out), _stream()), "nss_fp64_peak")
    return out.value


def nss_select_lowest_static(logL, n_delete, dead_idx, surv_idx=None, logLstar=None):
    """Delete-select without a handle and without any allocation, here or in the library: every argument is a CUDA tensor
    the caller already owns (logL float64 [n]; dead_idx int32 [n_delete]; surv_idx int32 [n - n_delete] or None; logLstar
    float64 [1] or None), which is the point — a program that has given all device memory to torch's caching allocator
    can still call it.  n <= SELECT_STATIC_MAX_LIVE.  Asynchronous on the current stream; calls must not overlap on the
    GPU (one shared work array per device, see include/nss.h).  Returns the status code for NSS_ELIMIT, raises otherwise."""
    rc = lib().nss_select_lowest_static(logL.data_ptr(), logL.numel(), int(n_delete), dead_idx.data_ptr(),
                                        surv_idx.data_ptr() if surv_idx is not None else None,
                                        logLstar.data_ptr() if logLstar is not None else None, _stream())
    return _check(rc, "nss_select_lowest_static", ok=(NSS_OK, NSS_ELIMIT))


class Nss:
    """One problem instance (nss_create .. nss_destroy).  `w` is an inputs.Workload-like object."""

    def __init__(self, w, kind=None, n_bins=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2509_24949_b200.nss needs a CUDA device; there is no CPU fallback")
        self.torch = torch
        self.d = int(w.d)
        cfg = nss_config()
        cfg.d = self.d
        cfg.kind = int(w.kind if kind is None else kind)
        cfg.n_bins = int(w.n_bins if n_bins is None else n_bins)
        self.kind, self.n_bins = cfg.kind, cfg.n_bins
        cfg.n_det, cfg.gmst = int(w.n_det), float(w.gmst)
        cfg.n_freq, cfg.f_min, cfg.df = int(w.n_freq), float(w.f_min), float(w.df)
        for j in range(self.d):
            cfg.param_index[j] = int(w.param_index[j])
            cfg.lo[j], cfg.hi[j] = float(w.lo[j]), float(w.hi[j])
            cfg.gauss_mu[j], cfg.gauss_sigma[j] = float(w.gauss_mu[j]), float(w.gauss_sigma[j])
        for j in range(NSLOT):
            cfg.theta_fixed[j], cfg.theta_fid[j] = float(w.theta_fixed[j]), float(w.theta_fid[j])
        for a in range(cfg.n_det):
            cfg.det[a] = _det_struct(w.det[a])
        self._psd = np.ascontiguousarray(w.psd, dtype=np.float64)
        self._data = np.ascontiguousarray(w.data if w.data is not None else np.zeros(0), dtype=np.float64)
        cfg.psd = self._psd.ctypes.data_as(c_dp)
        cfg.data = self._data.ctypes.data_as(c_dp)
        self.n_det = cfg.n_det
        h = vp()
        _check(lib().nss_create(C.byref(cfg), C.byref(h)), "nss_create")
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            lib().nss_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- helpers -------------------------------------------------------------------------------------
    def _dev(self, a, dtype=None):
        torch = self.torch
        dtype = dtype or torch.float64
        if isinstance(a, torch.Tensor):
            t = a.to(device="cuda", dtype=dtype).contiguous()
        else:
            t = torch.as_tensor(np.ascontiguousarray(a), dtype=dtype, device="cuda").contiguous()
        return t

    @property
    def launches(self) -> int:
        return int(lib().nss_launch_count(self._h))

    def nss_last_chain_ms(self) -> float:
        ms = C.c_double()
        _check(lib().nss_last_chain_ms(self._h, C.byref(ms)), "nss_last_chain_ms")
        return ms.value

    def set_chain_timing(self, on: bool):
        """Record CUDA events around K3 from now on (nss_last_chain_ms); costs the launch overlap, so off by default."""
        _check(lib().nss_set_chain_timing(self._h, 1 if on else 0), "nss_set_chain_timing")

    def set_chain_warps(self, warps: int):
        _check(lib().nss_set_chain_warps(self._h, int(warps)), "nss_set_chain_warps")

    def nss_last_chain_diag(self):
        """(rounds, evaluated candidates) of the most recent iteration."""
        a, b = C.c_int64(), C.c_int64()
        _check(lib().nss_last_chain_diag(self._h, C.byref(a), C.byref(b)), "nss_last_chain_diag")
        return a.value, b.value

    def nss_set_periodic(self, flags):
        """NEXT-2: sampled dim j wraps in [lo_j, hi_j) in the slice sampler when flags[j] != 0 (None: hard walls)."""
        if flags is None:
            _check(lib().nss_set_periodic(self._h, None), "nss_set_periodic")
            return
        f = np.zeros(11, dtype=np.int32)
        f[: self.d] = np.asarray(flags, dtype=np.int32)[: self.d]
        _check(lib().nss_set_periodic(self._h, f.ctypes.data_as(C.POINTER(C.c_int32))), "nss_set_periodic")

    def set_chain_lanes(self, lanes: int):
        _check(lib().nss_set_chain_lanes(self._h, int(lanes)), "nss_set_chain_lanes")

    def set_chain_pack(self, chains_per_cta: int):
        _check(lib().nss_set_chain_pack(self._h, int(chains_per_cta)), "nss_set_chain_pack")

    def set_loglike_variant(self, variant: int):
        _check(lib().nss_set_loglike_variant(self._h, int(variant)), "nss_set_loglike_variant")

    # ---- the C-ABI calls ---------------------------------------------------------------------------------
    def nss_loglike_batch(self, theta, out=None):
        """theta: [N, d] (torch cuda tensor or array) -> logL torch cuda tensor [N].  Asynchronous."""
        th = self._dev(theta).reshape(-1, self.d)
        n = th.shape[0]
        if out is None:
            out = self.torch.empty(n, dtype=self.torch.float64, device="cuda")
        _check(lib().nss_loglike_batch(self._h, th.data_ptr(), n, out.data_ptr(), _stream()), "nss_loglike_batch")
        return out

    def nss_loglike_batch_host(self, theta_host, out_host):
        """Host-buffer form (torch CPU tensors, pinned recommended): H2D copy, kernel, D2H copy inside the call."""
        n = theta_host.shape[0]
        _check(lib().nss_loglike_batch_host(self._h, theta_host.data_ptr(), n, out_host.data_ptr(), _stream()),
               "nss_loglike_batch_host")
        return out_host

    def iter_buffers(self, n_delete, host=False):
        """Caller-allocated outputs of nss_iterate / nss_iterate_host (dead_theta, dead_logL, dead_logw, dead_idx)."""
        torch = self.torch
        kw = dict(device="cpu", pin_memory=True) if host else dict(device="cuda")
        k = int(n_delete)
        return (torch.empty((k, self.d), dtype=torch.float64, **kw), torch.empty(k, dtype=torch.float64, **kw),
                torch.empty(k, dtype=torch.float64, **kw), torch.empty(k, dtype=torch.int32, **kw))

    def nss_iterate(self, live, logL, n_delete, n_repeats, seed, iteration, state, bufs, stop_dlogz=-3.0, host=False):
        """One complete NS iteration IN PLACE on (live, logL): device tensors, or (host=True) CPU tensors.
        `state` is an nss_iter_state carried between calls; `bufs` from iter_buffers()."""
        fn = lib().nss_iterate_host if host else lib().nss_iterate
        dth, dl, dw, di = bufs
        _check(fn(self._h, live.data_ptr(), logL.data_ptr(), live.shape[0], int(n_delete), int(n_repeats), int(seed),
                  int(iteration), float(stop_dlogz), dth.data_ptr(), dl.data_ptr(), dw.data_ptr(), di.data_ptr(),
                  C.byref(state), _stream()), "nss_iterate_host" if host else "nss_iterate")
        return state

    def nss_init_live(self, n_live, seed):
        torch = self.torch
        live = torch.empty((n_live, self.d), dtype=torch.float64, device="cuda")
        logL = torch.empty(n_live, dtype=torch.float64, device="cuda")
        _check(lib().nss_init_live(self._h, n_live, int(seed), live.data_ptr(), logL.data_ptr(), _stream()), "nss_init_live")
        return live, logL

    def nss_select_lowest(self, logL, n_delete):
        torch = self.torch
        l = self._dev(logL)
        n = l.numel()
        dead = torch.empty(n_delete, dtype=torch.int32, device="cuda")
        surv = torch.empty(n - n_delete, dtype=torch.int32, device="cuda")
        ls = C.c_double()
        _check(lib().nss_select_lowest(self._h, l.data_ptr(), n, int(n_delete), dead.data_ptr(), surv.data_ptr(),
                                       C.byref(ls), _stream()), "nss_select_lowest")
        return dead, surv, ls.value

    def nss_tune(self, live):
        torch = self.torch
        x = self._dev(live)
        mean = torch.empty(self.d, dtype=torch.float64, device="cuda")
        chol = torch.empty((self.d, self.d), dtype=torch.float64, device="cuda")
        rc = lib().nss_tune(self._h, x.data_ptr(), x.shape[0], mean.data_ptr(), chol.data_ptr(), _stream())
        _check(rc, "nss_tune", ok=(NSS_OK, NSS_ECHOL))
        return rc, mean, chol

    def nss_evidence_update(self, dead_logL, n_live, logX, logZ):
        torch = self.torch
        dl = self._dev(dead_logL)
        lw = torch.empty_like(dl)
        st = (C.c_double * 2)(logX, logZ)
        _check(lib().nss_evidence_update(self._h, dl.data_ptr(), int(n_live), dl.numel(), lw.data_ptr(), st, _stream()),
               "nss_evidence_update")
        return st[0], st[1], lw

    def nss_philox(self, seed, ctr):
        torch = self.torch
        c = torch.as_tensor(np.ascontiguousarray(ctr, dtype=np.uint32).view(np.int32), device="cuda")
        out = torch.empty_like(c)
        _check(lib().nss_philox(self._h, int(seed), c.data_ptr(), c.shape[0], out.data_ptr(), _stream()), "nss_philox")
        return out.cpu().numpy().view(np.uint32)

    def nss_replace_step(self, live, logL, n_delete, n_repeats, seed, iteration, logLstar=math.nan, want_trace=False,
                         ok=(NSS_OK,)):
        """One NS iteration on COPIES of (live, logL); returns a dict of torch tensors / scalars."""
        torch = self.torch
        live = self._dev(live).clone()
        logL = self._dev(logL).clone()
        n, k = live.shape[0], int(n_delete)
        dth = torch.empty((k, self.d), dtype=torch.float64, device="cuda")
        dl = torch.empty(k, dtype=torch.float64, device="cuda")
        didx = torch.empty(k, dtype=torch.int32, device="cuda")
        trace = margin = None
        if want_trace:
            trace = torch.zeros((k, max(n_repeats, 1), 3), dtype=torch.int32, device="cuda")
            margin = torch.zeros(k, dtype=torch.float64, device="cuda")
            _check(lib().nss_set_trace(self._h, trace.data_ptr(), margin.data_ptr()), "nss_set_trace")
        ls, ne = C.c_double(), C.c_int64()
        try:
            rc = lib().nss_replace_step(self._h, live.data_ptr(), logL.data_ptr(), n, k, float(logLstar), int(n_repeats),
                                        int(seed), int(iteration), dth.data_ptr(), dl.data_ptr(), didx.data_ptr(),
                                        C.byref(ls), C.byref(ne), _stream())
        finally:
            if want_trace:
                lib().nss_set_trace(self._h, None, None)
        _check(rc, "nss_replace_step", ok=ok)
        return dict(rc=rc, live=live, logL=logL, dead_theta=dth, dead_logL=dl, dead_idx=didx, logLstar=ls.value,
                    n_evals=ne.value, trace=trace[:, :n_repeats] if want_trace else None, margin=margin)

    def nss_resample_equal(self, logL, logw, seed):
        """Reading R6: row indices (ascending, torch int64 on the device) of the equal-weight posterior sample."""
        torch = self.torch
        l, w = self._dev(logL), self._dev(logw)
        idx = torch.empty(l.numel(), dtype=torch.int64, device="cuda")
        m = C.c_int64()
        _check(lib().nss_resample_equal(self._h, l.data_ptr(), w.data_ptr(), l.numel(), int(seed), idx.data_ptr(), C.byref(m),
                                        _stream()), "nss_resample_equal")
        return idx[: m.value]

    def nss_run(self, n_live, n_delete, n_repeats, seed, stop_dlogz=-3.0, max_iter=10000, cap=None, want_equal=False):
        if cap is None:
            cap = min(int(max_iter), 400) * int(n_delete) + int(n_live)
        dth, dl = np.empty((cap, self.d)), np.empty(cap)
        db, dw = np.empty(cap), np.empty(cap)
        res = nss_result()
        res.dead_theta, res.dead_logL = dth.ctypes.data_as(c_dp), dl.ctypes.data_as(c_dp)
        res.dead_logL_birth, res.dead_logw = db.ctypes.data_as(c_dp), dw.ctypes.data_as(c_dp)
        res.cap = cap
        eq = np.empty(cap if want_equal else 0, dtype=np.int64)
        res.equal_idx = eq.ctypes.data_as(C.POINTER(C.c_int64)) if want_equal else None
        rc = lib().nss_run(self._h, int(n_live), int(n_delete), int(n_repeats), int(seed), float(stop_dlogz),
                           int(max_iter), C.byref(res), _stream())
        _check(rc, "nss_run", ok=(NSS_OK, NSS_ENOTCONV))
        nd = int(res.n_dead)
        return dict(rc=rc, logZ=res.logZ, logZ_err=res.logZ_err, H=res.H, n_iter=int(res.n_iter), n_dead=nd,
                    n_evals=int(res.n_evals), gpu_ms=res.gpu_ms, ess=res.ess, n_equal=int(res.n_equal),
                    equal_idx=eq[: int(res.n_equal)] if want_equal else None, dead_theta=dth[:nd], dead_logL=dl[:nd],
                    dead_logL_birth=db[:nd], dead_logw=dw[:nd])

    def nss_get_tables(self):
        B = self.n_bins
        idx = np.empty(B + 1, dtype=np.int32)
        summ = np.empty((self.n_det, B, 6))
        dd = C.c_double()
        _check(lib().nss_get_tables(self._h, idx.ctypes.data, summ.ctypes.data_as(c_dp), C.byref(dd)), "nss_get_tables")
        return idx, summ, dd.value
