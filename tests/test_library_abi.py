"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/nss.h declares,
its host-only routines agree with the oracle, and compute calls fail loudly without a GPU."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2509_24949_b200 import build, inputs, nss

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libnss():
    build.build()
    return nss.lib()


def test_every_declared_symbol_is_exported(libnss):
    hdr = open(os.path.join(ROOT, "include", "nss.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(nss_[a-z0-9_]+)\s*\(", hdr))
    assert {"nss_create", "nss_loglike_batch", "nss_replace_step", "nss_run", "nss_destroy", "nss_strerror"} <= declared
    for name in declared:
        assert hasattr(libnss, name), f"{name} declared in include/nss.h but not exported"
    assert declared == set(nss.EXPORTS)
    assert libnss.nss_version() == 1
    assert libnss.nss_strerror(nss.NSS_ECHOL).decode().startswith("non-positive")


def test_struct_layout_matches_header(libnss):
    # sizes follow from the header's field list with natural alignment
    assert C.sizeof(nss.nss_detector) == 72
    assert C.sizeof(nss.nss_config) % 8 == 0
    assert nss.nss_config.psd.offset % 8 == 0 and nss.nss_config.det.offset % 8 == 0


def test_host_waveform_matches_oracle(libnss, oracle):
    f = 20.0 + 0.25 * np.arange(4017)
    rng = np.random.default_rng(0)
    w = inputs.config2()
    for _ in range(5):
        th = w.theta_inj.copy()
        th[w.param_index] = w.lo + (w.hi - w.lo) * rng.random(11)
        for a in range(3):
            got = nss.nss_waveform(th, w.det[a], 0.3, f)
            ref = oracle.waveform(th, w.det[a], 0.3, f)
            # phases reach ~1e4 rad: absolute phase agreement 1e-10 rad
            assert np.max(np.abs(got - ref) / np.abs(ref)) < 1e-10
    bad = w.theta_inj.copy(); bad[1] = 1.5
    with pytest.raises(nss.NssError):
        nss.nss_waveform(bad, w.det[0], 0.0, f)


def test_argument_validation_and_no_cpu_fallback(libnss):
    import torch
    cfg = nss.nss_config()
    h = C.c_void_p()
    assert libnss.nss_create(None, C.byref(h)) == nss.NSS_EINVAL
    cfg.d = 0
    assert libnss.nss_create(C.byref(cfg), C.byref(h)) == nss.NSS_EINVAL
    cfg.d = 2; cfg.kind = 2
    cfg.lo[0], cfg.hi[0], cfg.lo[1], cfg.hi[1] = 0.0, 1.0, 1.0, 1.0      # lo >= hi
    assert libnss.nss_create(C.byref(cfg), C.byref(h)) == nss.NSS_EINVAL
    assert libnss.nss_destroy(None) == nss.NSS_OK
    if not torch.cuda.is_available():
        # a valid problem cannot be created without a device, and the Python binding refuses too
        cfg.hi[1] = 2.0
        cfg.gauss_sigma[0] = cfg.gauss_sigma[1] = 1.0
        assert libnss.nss_create(C.byref(cfg), C.byref(h)) == nss.NSS_ECUDA
        assert libnss.nss_last_cuda_error().decode() != ""
        with pytest.raises(RuntimeError):
            nss.Nss(inputs.gaussian_workload(2))
