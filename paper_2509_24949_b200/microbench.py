"""Likelihood-kernel microbenchmark of BASELINE.json configs[4] ("config 5"): batches of N prior-uniform parameter
vectors of the config-2 problem, relative binning with B bins x 3 detectors, through `nss_loglike_batch`.

    python -m paper_2509_24949_b200.microbench

Prints a markdown table: evaluations per second and the fraction of the fp64 DFMA issue peak (measured in the same
process by `nss_fp64_peak`) for the automatic kernel choice and for both kernel forms (one thread per point; one
sub-warp per point).  Parity of the same kernels against the oracle at B = 64, 256, 1024 is in
tests/test_gpu_loglike.py; this script only times (inputs resident in HBM, L2 flushed between launches).

A second table times the FRONT of an NS iteration (k4_front: delete-select by counting ranks, O(n^2) comparisons, beside
mean / covariance / Cholesky) at n_live = 1000 ... 65536 through `nss_replace_step` with zero slice repeats, next to one
full iteration at the same n_live, to show where the counting select stops being negligible (north_star names a radix
select; bit-exact parity of the counting select, ties included, is in tests/test_gpu_sampler.py).

A third table sweeps the schedule of the chain kernel K3 — lanes per candidate, warps per chain, single-warp chains per
CTA (nss_set_chain_lanes / _warps / _pack: they change the schedule only, never a result) — on configs 2 and 3, the
measurements behind the automatic choice.
"""
from __future__ import annotations


def work(B: int, n_det: int):
    """fp64-pipe instructions one evaluation needs."""
    E = B + 1
    return 600 + E * 8 + E * n_det * 25


def main():
    import torch
    from . import build, inputs, nss
    build.build()
    if not torch.cuda.is_available():
        raise SystemExit("microbench.py needs a CUDA device: the product path has no CPU fallback")
    peak = nss.nss_fp64_peak(300.0)                      # TFLOP/s; DFMA issue peak = peak / 2 instructions/s
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    print(f"fp64 DFMA peak measured in this process: {peak:.1f} TFLOP/s\n")
    print("| B | N | kernel | ms | evals/s | fp64 instr./eval | fraction of the DFMA issue peak |")
    print("|---|---|---|---|---|---|---|")
    for B in (64, 128, 256, 1024):
        w = inputs.make_data(inputs.config5(B), nss.nss_waveform)
        g = nss.Nss(w)
        Xall = torch.as_tensor(inputs.draw_prior(w, 1_000_000, 5), device="cuda")
        for N in (1_000, 10_000, 100_000, 1_000_000):
            X = Xall[:N].contiguous()
            out = torch.empty(N, dtype=torch.float64, device="cuda")
            for variant, name in ((0, "automatic"), (1, "thread per point"), (2, "sub-warp per point")):
                g.set_loglike_variant(variant)
                for _ in range(2):
                    g.nss_loglike_batch(X, out)
                ts = []
                for _ in range(5):
                    flush.fill_(1)
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record()
                    g.nss_loglike_batch(X, out)
                    b.record()
                    b.synchronize()
                    ts.append(a.elapsed_time(b))
                ms = sorted(ts)[2]
                rate = N / (ms * 1e-3)
                ins = work(B, w.n_det)
                print(f"| {B} | {N} | {name} | {ms:.4f} | {rate:.3e} | {ins} | {rate * ins / (peak * 1e12 / 2):.3f} |", flush=True)
        g.close()
    front_table(torch, inputs, nss, flush)
    k3_sweep_table(torch, inputs, nss)


def front_table(torch, inputs, nss, flush):
    w = inputs.make_data(inputs.config2(), nss.nss_waveform)
    g = nss.Nss(w)

    def timed(fn, reps=5):
        ts = []
        for _ in range(reps):
            flush.fill_(1)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fn()
            b.record()
            b.synchronize()
            ts.append(a.elapsed_time(b))
        return sorted(ts)[len(ts) // 2]

    print("\n## front of an NS iteration (select + tune + evidence + host synchronisation) vs n_live, n_delete = n_live/2\n")
    print("| n_live | front only ms (0 slice repeats) | full iteration ms (55 repeats) | front / iteration |")
    print("|---|---|---|---|")
    for n in (1000, 5000, 16000, 65536):
        live, logL = g.nss_init_live(n, 1)
        g.nss_replace_step(live, logL, n // 2, 0, 1, 0)
        front = timed(lambda: g.nss_replace_step(live, logL, n // 2, 0, 1, 0))
        g.nss_replace_step(live, logL, n // 2, w.n_repeats, 1, 0)
        full = timed(lambda: g.nss_replace_step(live, logL, n // 2, w.n_repeats, 1, 0), reps=3)
        print(f"| {n} | {front:.4f} | {full:.4f} | {front / full:.4f} |", flush=True)
    g.close()


def k3_sweep_table(torch, inputs, nss):
    import math
    w = inputs.make_data(inputs.config2(), nss.nss_waveform)
    g = nss.Nss(w)
    g.set_chain_timing(True)
    print("\n## K3 schedule sweep (mean over NS iterations 2..25 of a seeded run; kernel ms from the library's event pair)\n")
    print("| n_live | n_delete | lanes/candidate | warps/chain | chains/CTA | K3 ms | step ms | rounds/chain | evaluated/consumed | evals/s (K3) |")
    print("|---|---|---|---|---|---|---|---|---|---|")
    for n, k, combos in ((1000, 500, ((0, 0, 0), (16, 2, 0), (8, 1, 1), (8, 2, 0), (16, 4, 0), (32, 4, 0), (32, 2, 0))),
                         (5000, 2500, ((0, 0, 0), (8, 1, 1), (8, 1, 2), (8, 1, 4), (8, 1, 8), (16, 1, 4), (16, 2, 0)))):
        for L, G, pack in combos:
            g.set_chain_lanes(L); g.set_chain_warps(G); g.set_chain_pack(pack)
            live, logL = g.nss_init_live(n, 1)
            st = nss.nss_iter_state(logX=0.0, logZ=-math.inf)
            bufs = g.iter_buffers(k)
            k3, stp, ev, rd, ex = [], [], 0, 0, 0
            for it in range(26):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                g.nss_iterate(live, logL, k, w.n_repeats, 1, it, st, bufs)
                b.record()
                b.synchronize()
                if it >= 2:
                    k3.append(g.nss_last_chain_ms()); stp.append(a.elapsed_time(b)); ev += st.n_evals
                    r_, e_ = g.nss_last_chain_diag(); rd += r_; ex += e_
            m = len(k3)
            name = lambda v: "auto" if v == 0 else str(v)
            print(f"| {n} | {k} | {name(L)} | {name(G)} | {name(pack)} | {sum(k3) / m:.4f} | {sum(stp) / m:.4f} | {rd / m / k:.1f} | "
                  f"{ex / ev:.3f} | {ev / sum(k3) * 1e3:.3e} |", flush=True)
    g.close()


if __name__ == "__main__":
    main()
