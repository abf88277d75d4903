"""Drive every kernel family of libnss.so once, at small sizes, for NVIDIA compute-sanitizer.

    compute-sanitizer --tool memcheck  --error-exitcode 1 python -m paper_2509_24949_b200.sanitize
    compute-sanitizer --tool racecheck --error-exitcode 1 python -m paper_2509_24949_b200.sanitize
    compute-sanitizer --tool initcheck --error-exitcode 1 python -m paper_2509_24949_b200.sanitize
    compute-sanitizer --tool synccheck --error-exitcode 1 python -m paper_2509_24949_b200.sanitize

Set PYTORCH_NO_CUDA_MEMORY_CACHING=1 so that every tensor is its own cudaMalloc block and an out-of-bounds access cannot
land in a neighbouring tensor of torch's pool.  The kernels synchronise through tickets, a spin barrier among the tuning
blocks, volatile flags, double-buffered shared results, sub-warp scratch behind __syncwarp, mbarrier / TMA staging and
programmatic dependent launch; the cases below reach each of those.  Results are only checked for being finite: parity is
tests/'s job, this script exists to be run under the tools.  `--case NAME` runs one case.

State of the tier: on the pool this repository is built on, compute-sanitizer is closed (it exits 86 at once with a notice
that runs under it have left GPUs needing a reset), so NO sanitizer summary exists for this code; profiles/r03_sanitizer.md
records the attempt and what stands in for it.  The script runs clean without a tool (five cases) and is kept for a
machine where the tools may run.
"""
from __future__ import annotations

import argparse
import math
import sys

import numpy as np


def main() -> int:
    import torch
    from . import build, inputs, nss

    ap = argparse.ArgumentParser()
    ap.add_argument("--case", default="all")
    args = ap.parse_args()
    build.build()
    if not torch.cuda.is_available():
        raise SystemExit("needs a CUDA device")
    torch.cuda.set_device(0)
    done = []

    def iterate(g, n, k, nrep, seed, iters=1):
        live, logL = g.nss_init_live(n, seed)
        st = nss.nss_iter_state(logX=0.0, logZ=-math.inf)
        bufs = g.iter_buffers(k)
        for it in range(iters):
            g.nss_iterate(live, logL, k, nrep, seed, it, st, bufs)
        torch.cuda.synchronize()
        assert math.isfinite(st.logLstar) and st.n_evals > 0
        assert bool(torch.isfinite(logL).all())
        return live, logL

    def case_config1():
        """Smoke size: batch likelihood in every variant, two NS iterations, a periodic step, a run to the stop rule."""
        w = inputs.make_data(inputs.config1(), nss.nss_waveform)
        g = nss.Nss(w)
        X = inputs.draw_prior(w, 2048, 5)
        for v in (0, 1, 2):
            g.set_loglike_variant(v)
            assert bool(torch.isfinite(g.nss_loglike_batch(X)).all())
        g.set_loglike_variant(0)
        iterate(g, 100, 50, 12, 1, iters=2)
        for warps, lanes, pack in ((1, 32, 1), (1, 8, 3), (2, 16, 0), (8, 32, 0)):
            g.set_chain_warps(warps); g.set_chain_lanes(lanes); g.set_chain_pack(pack)
            iterate(g, 100, 50, 3, 2)
        g.set_chain_warps(0); g.set_chain_lanes(0); g.set_chain_pack(0)
        g.nss_set_periodic([0, 0, 0, 1])
        iterate(g, 100, 50, 6, 3)
        g.nss_set_periodic(None)
        r = g.nss_run(100, 50, 12, 1, max_iter=3)
        assert r["n_iter"] == 3
        r = g.nss_run(100, 50, 12, 1)
        assert r["rc"] == 0 and math.isfinite(r["logZ"])
        g.close()

    def case_config2():
        """Three detectors, 128 bins: thread and sub-warp batch kernels, one iteration with 8-, 16- and 32-lane candidates;
        1024 bins: the record table read through L2 inside K3."""
        w = inputs.make_data(inputs.config2(), nss.nss_waveform)
        g = nss.Nss(w)
        X = inputs.draw_prior(w, 4096, 5)
        for v in (1, 2):
            g.set_loglike_variant(v)
            assert bool(torch.isfinite(g.nss_loglike_batch(X)).all())
        g.set_loglike_variant(0)
        for lanes in (8, 16, 32):
            g.set_chain_lanes(lanes)
            iterate(g, 200, 100, 2, 4)
        g.close()
        g = nss.Nss(w, n_bins=1024)
        iterate(g, 120, 60, 2, 5)
        g.close()

    def case_full_grid():
        """Full frequency grid (4017 records x 3 detectors): the TMA-streamed thread kernel, the sub-warp kernel, K3 with
        the table read from L2."""
        w = inputs.make_data(inputs.config2(), nss.nss_waveform)
        g = nss.Nss(w, kind=1)
        X = inputs.draw_prior(w, 1024, 6)
        for v in (1, 2):
            g.set_loglike_variant(v)
            assert bool(torch.isfinite(g.nss_loglike_batch(X)).all())
        g.set_loglike_variant(0)
        iterate(g, 64, 32, 1, 6)
        g.close()

    def case_many_live():
        """9000 live points: sample-sort select in front of k4_front, eight tuning blocks behind the spin barrier and the
        ticket, 4500 single-warp chains packed per CTA and fetched from the device counter; then the stand-alone tune
        followed by an iteration on the same handle."""
        w = inputs.gaussian_workload(5, sigma=0.07)
        g = nss.Nss(w)
        live, logL = iterate(g, 9000, 4500, 2, 7)
        rc, mean, chol = g.nss_tune(live[:5000])
        assert rc == 0 and bool(torch.isfinite(chol).all())
        iterate(g, 4100, 2050, 1, 8)
        r = g.nss_run(9000, 4500, 1, 9, max_iter=2)
        assert r["n_iter"] == 2
        g.close()

    def case_hooks():
        """The stand-alone K4 kernels: counting and sample-sort select, the static select, evidence update, resampling,
        Philox."""
        w = inputs.gaussian_workload(4, sigma=0.05)
        g = nss.Nss(w)
        rng = np.random.default_rng(0)
        for n, k in ((1000, 500), (8192, 100), (20000, 10000)):
            l = rng.normal(size=n)
            l[::7] = l[0]
            dead, surv, ls = g.nss_select_lowest(l, k)
            assert int(dead.min()) >= 0 and int(surv.max()) < n
        l = torch.as_tensor(rng.normal(size=3000), device="cuda")
        dead = torch.empty(1500, dtype=torch.int32, device="cuda")
        surv = torch.empty(1500, dtype=torch.int32, device="cuda")
        ls = torch.empty(1, dtype=torch.float64, device="cuda")
        assert nss.nss_select_lowest_static(l, 1500, dead, surv, ls) == nss.NSS_OK
        assert nss.nss_select_lowest_static(l[:77], 5, dead[:5], None, None) == nss.NSS_OK
        torch.cuda.synchronize()
        lx, lz, lw = g.nss_evidence_update(np.sort(rng.normal(size=500)), 1000, 0.0, -math.inf)
        assert math.isfinite(lz)
        idx = g.nss_resample_equal(rng.normal(size=5000), -rng.random(5000) * 3, 3)
        assert idx.numel() > 0
        out = g.nss_philox(12345, rng.integers(0, 2 ** 32, size=(1000, 4), dtype=np.uint64).astype(np.uint32))
        assert out.shape == (1000, 4)
        g.close()

    cases = {"config1": case_config1, "config2": case_config2, "full_grid": case_full_grid, "many_live": case_many_live,
             "hooks": case_hooks}
    for name, fn in cases.items():
        if args.case in ("all", name):
            fn()
            torch.cuda.synchronize()
            done.append(name)
            print(f"[sanitize] case {name}: ran", flush=True)
    print(f"[sanitize] {len(done)} case(s) completed: {', '.join(done)}")
    return 0 if done else 2


if __name__ == "__main__":
    sys.exit(main())
