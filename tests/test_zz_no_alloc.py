"""nss_select_lowest_static — the delete-select for callers that must not allocate — against nss_select_lowest.

Why the entry point exists: some users of this library cannot let it call cudaMalloc.  Their device memory belongs to a
pool (torch's caching allocator holding all of HBM, a job with a fixed pre-reserved budget), so an allocation made
behind their back fails although the pool has room; or they run beside other streams and cannot afford the device-wide
stall an allocation causes; or they have to show that nothing can run out of memory once start-up is over.  The static
variant works in a fixed array inside the library image, takes only tensors the caller already owns, and is capped at
nss.SELECT_STATIC_MAX_LIVE live points.

What is checked: the integer outputs (dead list in ascending logL with ties by slot, survivor list in ascending slot) and
the threshold are bit-identical to the handle-based path — the tolerance tests/test_gpu_sampler.py uses for this
operation — on two calls in a row, the second smaller than the first so that it runs over whatever the first left in the
shared array; that the device's free memory does not move across a call; and that oversize requests are refused.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide other tests.
It makes no assumption about what ran before it (it passes alone in a fresh process and after the rest of the suite).
"""
import numpy as np
import pytest

from paper_2509_24949_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def nssmod():
    from paper_2509_24949_b200 import build, nss
    build.build()
    return nss


def _values(n, seed):
    rng = np.random.default_rng(seed)
    l = rng.normal(size=n) * 10
    l[rng.integers(0, n, n // 4)] = l[0]            # a quarter of the values tied: order decided by the slot
    if n > 10:
        l[5] = -np.inf
        l[n - 1] = -np.inf
    return l


def _static_select(nss, torch, l_dev, k, want_surv=True):
    n = l_dev.numel()
    dead = torch.full((k,), -1, dtype=torch.int32, device="cuda")
    surv = torch.full((n - k,), -1, dtype=torch.int32, device="cuda") if want_surv else None
    lstar = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    rc = nss.nss_select_lowest_static(l_dev, k, dead, surv, lstar)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert rc == nss.NSS_OK
    return dead, surv, lstar, free0 - free1


def test_static_select_equals_the_allocating_path_twice_in_a_row(nssmod):
    import torch
    nss = nssmod
    g = nss.Nss(inputs.gaussian_workload(4, sigma=0.05))       # only the existing path needs a handle
    try:
        # first the largest size the array holds (every word of it written), then smaller, odd-sized calls over its remains
        used = []
        for n, k, seed in ((nss.SELECT_STATIC_MAX_LIVE, 4096, 1), (1000, 500, 2), (1025, 1, 3), (300, 299, 4), (2, 1, 5)):
            l = _values(n, seed)
            l_dev = torch.as_tensor(l, device="cuda")
            dead, surv, lstar, delta = _static_select(nss, torch, l_dev, k)
            used.append(delta)
            rdead, rsurv, rlstar = g.nss_select_lowest(l_dev, k)
            assert torch.equal(dead, rdead), (n, k)
            assert torch.equal(surv, rsurv), (n, k)
            assert lstar.item() == rlstar, (n, k)
            order = np.argsort(l, kind="stable")               # and both are the stable sort's answer
            assert np.array_equal(dead.cpu().numpy(), order[:k])
            assert lstar.item() == l[order[k - 1]]
        # after the first call (which may load the module and look the array up) a call leaves free memory where it was
        assert all(u == 0 for u in used[1:]), used
        # the same input again, now without a survivor list: the spare list inside the array takes its place
        l = _values(1000, 2)
        l_dev = torch.as_tensor(l, device="cuda")
        dead, _, lstar, _ = _static_select(nss, torch, l_dev, 500, want_surv=False)
        rdead, _, rlstar = g.nss_select_lowest(l_dev, 500)
        assert torch.equal(dead, rdead) and lstar.item() == rlstar
    finally:
        g.close()


def test_static_select_refuses_what_it_cannot_hold(nssmod):
    import torch
    nss = nssmod
    n = nss.SELECT_STATIC_MAX_LIVE + 1
    l_dev = torch.zeros(n, dtype=torch.float64, device="cuda")
    dead = torch.full((4,), -7, dtype=torch.int32, device="cuda")
    assert nss.nss_select_lowest_static(l_dev, 4, dead) == nss.NSS_ELIMIT
    torch.cuda.synchronize()
    assert bool((dead == -7).all())                            # refused before anything was launched
    assert b"capacity" in nss.lib().nss_strerror(nss.NSS_ELIMIT)
    with pytest.raises(nss.NssError):                          # n_delete >= n_live, as in nss_select_lowest
        nss.nss_select_lowest_static(l_dev[:8], 8, dead)
