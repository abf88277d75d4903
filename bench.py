#!/usr/bin/env python
"""bench.py — the measurement contract.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A "step" is ONE COMPLETE NESTED-SLICE-SAMPLING ITERATION of BASELINE.json configs[1] (11 parameters,
H1+L1+V1, relative binning with 128 bins per detector, n_live = 1000, n_delete = 500, 55 slice
repeats): delete-select, evidence bookkeeping, covariance + Cholesky, 500 slice chains whose every
bracket test is one heterodyned log-likelihood evaluation, in-place replacement, live-evidence stop
test — one `nss_iterate` call of the C ABI.  Steps are consecutive
iterations of one seeded run (a fresh run is started, untimed, whenever the stop rule fires).

metric  = heterodyned logL evaluations per second (sequential-algorithm count / device time)
value   = device-resident steps (CUDA events around each step on the launching stream)
e2e     = the same through `nss_iterate_host` with pinned HOST buffers (H2D + D2H inside the call)
roofline= the dominant kernel (K3 slice chains): fp64 flop of the likelihood evaluations it made /
          its own CUDA-event duration, against the DFMA peak measured in the same process
extras  = a config-3 step (n_live 5000 / n_delete 2500) with its own K3 roofline object, K1 / K2 batch-likelihood
          microbenchmarks (config 5, N = 1e6; config 4 likelihood), full `nss_run`s to convergence on configs 2, 3, 4
          and on the paper's hyper-parameters (n_live 3000, n_delete 1500, 10 d repeats: PAPER.md:43), the oracle timed
          on the host cores (cpu_baseline: NS iterations; oracle_legs: BASELINE.md section 2's other legs).

`--impl reference` times the ORACLE (oracle/, plain C on the host cores) on a bounded sample of the same
workload; it is the only other place this file executes oracle/ code.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "heterodyned logL evals/s (NSS iteration, config 2)"
NOMINAL_TF = 148 * 64 * 2 * 1.965e9 / 1e12        # 148 SMs x 64 fp64 lanes x 2 flop x 1.965 GHz = 37.2 TFLOP/s
UNIT = "evals/s"
SEED = 1


# ---- algorithmic work of one relative-binning likelihood evaluation -------------------------
def rb_work(B: int, n_det: int):
    """(fp64-pipe instructions, flop) one relative-binning evaluation needs in the regrouped form the kernels
    use: per point; per edge the 8-term phase; per (edge, detector) the arrival-time FMA, sincos
    in turns (17 instructions), T += W conj(z) (4 FMA) and the cross term V Re(z_b conj z_b+1) (3).
    FMA = 1 instruction = 2 flop; add/mul = 1 flop."""
    E = B + 1
    per_point_i, per_point_f = 600, 900
    edge_i, edge_f = 8, 16
    ed_i, ed_f = 1 + 17 + 4 + 3, 2 + 31 + 8 + 5
    instr = per_point_i + E * edge_i + E * n_det * ed_i
    flop = per_point_f + E * edge_f + E * n_det * ed_f
    return instr, flop


K3_PROFILE = os.path.join(ROOT, "profiles", "r03_k3_slice_full.md")


def profile_traffic():
    """DRAM bytes per K3 launch, read from the tracked ncu --set full summary (NOT measured in this run: ncu cannot run
    inside a timed bench).  The summary carries a line `dram_bytes_per_launch: <read + write bytes>` and its capture date."""
    try:
        txt = open(K3_PROFILE).read()
        import re
        m = re.search(r"dram_bytes_per_launch:\s*(\d+)", txt)
        dt = re.search(r"captured:\s*(\S+)", txt)
        if m:
            return int(m.group(1)), (f"from the tracked profile {os.path.relpath(K3_PROFILE, ROOT)} (captured {dt.group(1) if dt else '?'}), "
                                     "dram__bytes_read.sum + dram__bytes_write.sum of one launch; not measured in this run; "
                                     "the kernel is ALU/latency-bound, the live set and tables stay in L2")
    except OSError:
        pass
    return None, "no tracked ncu capture of this build"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled in a thread while the GPU is under load."""

    def __init__(self, index=0, period=0.02):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._t = None
        self.period = period
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                 "hw_power_brake": 0x80, "sync_boost": 0x10, "applications_clocks_setting": 0x2}
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h) if hasattr(nv, "nvmlDeviceGetCurrentClocksEventReasons") \
                    else nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def __enter__(self):
        if self.nv:
            self._t = threading.Thread(target=self._run, daemon=True)
            self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._t:
            self._t.join()

    def summary(self):
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s)}


def oracle_steps(w_oracle, steps, warmup, n_repeats, seed):
    """Times the oracle, as it stands, on the host cores: consecutive NS iterations of config 2 with
    `n_repeats` slice repeats per chain.  Returns (evals, seconds, cores)."""
    from oracle import nss_oracle as orc
    p = orc.Problem(w_oracle)
    cores = orc.n_cores()
    live, logL = p.init_live(w_oracle.n_live, seed, nthreads=cores)
    evals, secs = 0, 0.0
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        o = p.replace_step(live, logL, w_oracle.n_delete, n_repeats, seed, it, nthreads=cores)
        orc.evidence_update(o["dead_logL"], w_oracle.n_live, 0.0, -math.inf)
        dt = time.perf_counter() - t0
        assert o["rc"] == 0
        live, logL = o["live"], o["logL"]
        if it >= warmup:
            evals += o["n_evals"]
            secs += dt
    return evals, secs, cores


def oracle_legs(wo, cores, gpu_small, gpu_large, gpu_run, whole_run, gpu_run1=None):
    """the oracle's batched likelihood on 1 core and on all cores (relative binning N = 1e4, full
    grid N = 1e3), its single-thread config-1 run and its wall clock for one whole config-2 run, beside the GPU figures of
    this run.  gpu_small: the GPU's evals/s measured at the SAME N as the oracle leg; gpu_large: at the microbenchmark N."""
    from oracle import nss_oracle as orc
    from paper_2509_24949_b200 import inputs
    legs = {}
    X = inputs.draw_prior(wo, 10000, 5)
    for name, prob, pts, key in (("loglike_batch_rb_N1e4", orc.Problem(wo), X, "rb"),
                                 ("loglike_batch_full_N1e3", orc.Problem(wo, kind=1), X[:1000], "full")):
        gpu = gpu_small[key]
        leg = {"n_points": int(pts.shape[0]), "gpu_evals_per_s": gpu,
               "gpu_evals_per_s_note": f"measured in this run at N = {int(pts.shape[0])} (same points as the oracle leg), "
                                       "CUDA events, median of 9 launches, automatic kernel variant",
               "gpu_evals_per_s_large_N": gpu_large[key][0], "gpu_large_N": gpu_large[key][1]}
        for label, nt in (("1_core", 1), (f"{cores}_cores", cores)):
            t0 = time.perf_counter()
            prob.loglike_batch(pts, nthreads=nt)
            leg[label + "_evals_per_s"] = pts.shape[0] / (time.perf_counter() - t0)
        leg["gpu_over_all_cores"] = gpu / leg[f"{cores}_cores_evals_per_s"]
        legs[name] = leg
    if gpu_run1 is not None:
        # BASELINE.md section 2, "NSS run, config 1 (single thread)": same seed and stop rule as the GPU's config-1 run
        w1 = inputs.make_data(inputs.config1(), orc.waveform)
        t0 = time.perf_counter()
        o1 = orc.Problem(w1).run(w1.n_live, w1.n_delete, w1.n_repeats, SEED, nthreads=1)
        wall1 = time.perf_counter() - t0
        legs["nss_run_config1"] = {"oracle_wall_s": wall1, "cores": 1, "n_iter": o1["n_iter"], "n_evals": o1["n_evals"],
                                   "logZ": o1["logZ"], "logZ_err": o1["logZ_err"], "gpu_wall_s": gpu_run1["wall_s"],
                                   "gpu_n_iter": gpu_run1["n_iter"], "gpu_n_evals": gpu_run1["n_evals"],
                                   "gpu_logZ": gpu_run1["logZ"], "gpu_over_oracle": wall1 / gpu_run1["wall_s"]}
    if whole_run:
        p = orc.Problem(wo)
        t0 = time.perf_counter()
        o = p.run(wo.n_live, wo.n_delete, wo.n_repeats, SEED, nthreads=cores)
        wall = time.perf_counter() - t0
        legs["nss_run_config2"] = {"oracle_wall_s": wall, "cores": cores, "n_iter": o["n_iter"], "n_evals": o["n_evals"],
                                   "logZ": o["logZ"], "logZ_err": o["logZ_err"], "gpu_wall_s": gpu_run["wall_s"],
                                   "gpu_n_iter": gpu_run["n_iter"], "gpu_n_evals": gpu_run["n_evals"], "gpu_logZ": gpu_run["logZ"],
                                   "gpu_over_oracle": wall / gpu_run["wall_s"],
                                   "note": "same seed, same stop rule; the bench injection comes from the library's own waveform "
                                           "routine and the oracle's from the oracle's, so the two data sets agree to rounding only"}
    return legs


def run_reference(args):
    """--impl reference: the oracle on the host cores, on a bounded sample of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import nss_oracle as orc
    from paper_2509_24949_b200 import inputs
    orc.build()
    w = inputs.make_data(inputs.config2(), orc.waveform)
    n_rep = 5
    w.n_repeats = n_rep                            # the line's config records what this arm ran
    evals, secs, cores = oracle_steps(w, args.steps, args.warmup, n_rep, SEED)
    v = evals / secs
    sample = (f"{args.steps} consecutive NS iterations of config 2 (n_live 1000, n_delete 500) with {n_rep} slice repeats "
              f"per chain instead of 55 (a bounded sample: evals/s is per evaluation), OpenMP over chains on {cores} cores; "
              "the oracle is an unoptimised checker (scalar loops, libm, an allocation per evaluation), not a tuned CPU code")
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(w),
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def config_dict(w):
    return {"workload": "BASELINE.json configs[1]: 11-param aligned-spin BBH, H1+L1+V1, TaylorF2 3.5PN + 1.5PN SO, "
                        "aLIGO-fit PSD, 20-1024 Hz df 0.25 (4017 bins), SNR-20 injection + seeded coloured noise, "
                        f"relative binning B=128/detector, n_live 1000, n_delete 500, {int(w.n_repeats)} slice repeats",
            "n_live": int(w.n_live), "n_delete": int(w.n_delete), "n_repeats": int(w.n_repeats), "n_bins": int(w.n_bins),
            "n_det": int(w.n_det), "d": int(w.d), "seed": SEED,
            "l2": "flushed (256 MiB write) between steps, outside the per-step event pairs; working set < 1 MB, ALU-bound"}


def aggregate_replicas(dist, times, counts, device):
    """Replicas only: every rank ran the same number of steps on its own seeds.  The job's time is
    the MAX over ranks of each timed quantity, its work the SUM over ranks of each count."""
    import torch
    t = torch.tensor(list(times), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor(list(counts), dtype=torch.float64, device=device)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return tuple(float(x) for x in t), tuple(int(x) for x in c)


def run_ours(args):
    import numpy as np
    import torch
    from paper_2509_24949_b200 import build, inputs, nss

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        build.build()
    if dist:
        dist.barrier()

    # inputs: injection synthesised by the CUDA library's own host waveform (never the oracle's)
    w = inputs.make_data(inputs.config2(), nss.nss_waveform)
    g = nss.Nss(w)
    n, k, nrep, d = w.n_live, w.n_delete, w.n_repeats, w.d
    seed = SEED + 1000 * rank                      # replicas only: independent seeds per GPU
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def fresh(sd, n_live=None, g=g):
        live, logL = g.nss_init_live(n if n_live is None else n_live, sd)
        return live, logL, nss.nss_iter_state(logX=0.0, logZ=-math.inf), 0

    def timed_steps(n_live, n_del, steps, warmup, sd, sync_all, kernel_timing=False, g=g):
        """`steps` consecutive NS iterations (one nss_iterate call each) of a seeded run, CUDA events around each step on
        the launching stream, L2 flushed between steps outside the event pairs; a fresh run starts, untimed, whenever the
        stop rule fires.  kernel_timing: the library also records events around K3 (which costs the step ~5 us of launch
        overlap, so the step time is taken from a pass without them and the kernel time from a second, identical pass)."""
        g.set_chain_timing(kernel_timing)
        live, logL, st, it = fresh(sd, n_live, g)
        bufs = g.iter_buffers(n_del)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        r = dict(evals=0, k3_ms=0.0, rounds=0, executed=0, launches=0, wall=0.0, ms=0.0)
        runs, l0, wall0 = 0, 0, None
        if sync_all:
            barrier()
        for s_ in range(warmup + steps):
            if s_ == warmup:
                barrier() if sync_all else torch.cuda.synchronize()
                wall0 = time.perf_counter()
                l0 = g.launches
            if st.converged:
                runs += 1
                live, logL, st, it = fresh(sd + 7919 * runs, n_live, g)
            flush.fill_(s_ & 0xFF)
            if s_ >= warmup:
                ev[s_ - warmup][0].record(stream)
            g.nss_iterate(live, logL, n_del, nrep, sd + 7919 * runs, it, st, bufs)
            if s_ >= warmup:
                ev[s_ - warmup][1].record(stream)
                r["evals"] += st.n_evals
                if kernel_timing:
                    r["k3_ms"] += g.nss_last_chain_ms()
                rd, ex = g.nss_last_chain_diag()
                r["rounds"] += rd; r["executed"] += ex
            it += 1
        barrier() if sync_all else torch.cuda.synchronize()
        r["wall"] = time.perf_counter() - wall0
        r["launches"] = g.launches - l0
        r["ms"] = sum(a.elapsed_time(b) for a, b in ev)
        g.set_chain_timing(False)
        return r

    def barrier():
        torch.cuda.synchronize()
        if dist:
            dist.barrier()
            torch.cuda.synchronize()

    peak_tf = nss.nss_fp64_peak(300.0)

    with ClockSampler(local) as clocks:
        # ---- device-resident steps -----------------------------------------------------------------------
        m2 = timed_steps(n, k, args.steps, args.warmup, seed, True)
        m2k = timed_steps(n, k, args.steps, args.warmup, seed, True, kernel_timing=True)     # the same steps, K3 timed
        assert m2k["evals"] == m2["evals"], "the two passes must make the same evaluations"
        evals, k3_ms, rounds, executed = m2["evals"], m2k["k3_ms"], m2["rounds"], m2["executed"]
        wall, launches, ms = m2["wall"], m2["launches"], m2["ms"]
        ms_with_kernel_events = m2k["ms"]

        # ---- end to end: pinned host buffers through nss_iterate_host ----------------------------------------
        live_d, logL_d, st_h, it_h = fresh(seed + 1)
        live_h = torch.empty((n, d), dtype=torch.float64, pin_memory=True)
        logL_h = torch.empty(n, dtype=torch.float64, pin_memory=True)
        live_h.copy_(live_d); logL_h.copy_(logL_d)
        hb = g.iter_buffers(k, host=True)
        e2e_steps = args.steps
        evals_h, t_h = 0, 0.0
        seed_h = seed + 1
        barrier()
        for s in range(args.warmup + e2e_steps):
            if st_h.converged:
                seed_h = seed + 1 + 104729 * (s + 1)     # a new run: new initial points AND new chain streams
                live_d, logL_d, st_h, it_h = fresh(seed_h)
                live_h.copy_(live_d); logL_h.copy_(logL_d)
                torch.cuda.synchronize()
            flush.fill_(s & 0xFF)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            g.nss_iterate(live_h, logL_h, k, nrep, seed_h, it_h, st_h, hb, host=True)   # synchronous
            dt = time.perf_counter() - t0
            if s >= args.warmup:
                evals_h += st_h.n_evals
                t_h += dt
            it_h += 1
        barrier()
        h2d = n * d * 8 + n * 8
        d2h = n * d * 8 + n * 8 + k * d * 8 + k * 8 + k * 8 + k * 4

        # ---- config 3 (BASELINE.json configs[2]): the same step at n_live 5000 / n_delete 2500 (rank 0 only) ------------
        m3 = None
        if rank == 0 and not args.no_extras:
            m3 = timed_steps(5000, 2500, max(4, args.steps // 2), 3, seed, False)
            m3["k3_ms"] = timed_steps(5000, 2500, max(4, args.steps // 2), 3, seed, False, kernel_timing=True)["k3_ms"]
            m3["steps"] = max(4, args.steps // 2)

        # ---- K1 microbenchmark (config 5): N = 1e6 prior draws, B = 128 x 3 detectors --------------------------
        N1 = 1_000_000
        X = torch.as_tensor(inputs.draw_prior(w, N1, 5), device="cuda")
        out = torch.empty(N1, dtype=torch.float64, device="cuda")
        g.set_loglike_variant(1)
        for _ in range(3):
            g.nss_loglike_batch(X, out)
        k1 = []
        for _ in range(5):
            flush.fill_(1)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            g.nss_loglike_batch(X, out)
            b.record(stream)
            b.synchronize()
            k1.append(a.elapsed_time(b))
        g.set_loglike_variant(0)
        k1_ms = sorted(k1)[len(k1) // 2]

        # ---- K2 microbenchmark (config 4 likelihood): full frequency grid, 4017 bins x 3 detectors, N = 1e5 ---------
        g2 = nss.Nss(w, kind=1)
        N2 = 100_000
        X2, out2 = X[:N2].contiguous(), torch.empty(N2, dtype=torch.float64, device="cuda")
        for _ in range(2):
            g2.nss_loglike_batch(X2, out2)
        k2 = []
        for _ in range(3):
            flush.fill_(2)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            g2.nss_loglike_batch(X2, out2)
            b.record(stream)
            b.synchronize()
            k2.append(a.elapsed_time(b))
        k2_ms = sorted(k2)[len(k2) // 2]

        def batch_rate(gg, pts):
            """evals/s of nss_loglike_batch at exactly this N (automatic variant), median of 9 event-timed launches."""
            o_ = torch.empty(pts.shape[0], dtype=torch.float64, device="cuda")
            for _ in range(3):
                gg.nss_loglike_batch(pts, o_)
            ts = []
            for _ in range(9):
                flush.fill_(3)
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                gg.nss_loglike_batch(pts, o_)
                b.record(stream)
                b.synchronize()
                ts.append(a.elapsed_time(b))
            return pts.shape[0] / (sorted(ts)[len(ts) // 2] * 1e-3)

        Xs = torch.as_tensor(inputs.draw_prior(w, 10000, 5), device="cuda")     # the points oracle_legs uses
        gpu_small = {"rb": batch_rate(g, Xs), "full": batch_rate(g2, Xs[:1000].contiguous())}
        g2.close()

        # ---- full runs to convergence -----------------------------------------------------------------------
        def timed_run(gg, n_live, n_del, n_rep, sd, max_iter=10000):
            gg.nss_run(n_live, n_del, n_rep, sd, max_iter=max_iter)       # warm (allocations of the handle)
            t0 = time.perf_counter()
            rr = gg.nss_run(n_live, n_del, n_rep, sd, max_iter=max_iter)
            wall_s = time.perf_counter() - t0
            return {"wall_s": wall_s, "gpu_ms": rr["gpu_ms"], "n_iter": rr["n_iter"], "n_evals": rr["n_evals"],
                    "evals_per_s": rr["n_evals"] / wall_s, "logZ": rr["logZ"], "logZ_err": rr["logZ_err"], "H": rr["H"],
                    "rc": rr["rc"], "kish_ess": rr["ess"], "ess_per_s": rr["ess"] / wall_s, "n_equal": rr["n_equal"],
                    "n_live": n_live, "n_delete": n_del, "n_repeats": n_rep}

        run2 = timed_run(g, n, k, nrep, seed)
        run1 = None
        if rank == 0 and not args.no_extras:
            w1 = inputs.make_data(inputs.config1(), nss.nss_waveform)
            g1 = nss.Nss(w1)
            run1 = timed_run(g1, w1.n_live, w1.n_delete, w1.n_repeats, SEED)
            g1.close()
        run_wall, r = run2["wall_s"], run2
        runs_extra = {}
        if rank == 0 and not args.no_extras:
            runs_extra["config3"] = timed_run(g, 5000, 2500, nrep, seed)
            # the paper's hyper-parameters on the synthetic config-2 problem (3000 live points, half of
            # them deleted per iteration, chains of 10 d steps); its 207 s / ESS 17490 is IMRPhenomD on
            # GW150914 on an A100: context only
            runs_extra["paper_hyperparameters"] = timed_run(g, 3000, 1500, 10 * d, seed)
            g4 = nss.Nss(w, kind=1)
            runs_extra["config4"] = timed_run(g4, n, k, nrep, seed)
            # config 4 (BASELINE.json configs[3]) as a step: the same iteration with the full-grid likelihood inside K3
            m4 = timed_steps(n, k, 4, 3, seed, False, g=g4)
            m4["k3_ms"] = timed_steps(n, k, 4, 3, seed, False, kernel_timing=True, g=g4)["k3_ms"]
            m4["steps"] = 4
            g4.close()

    # max over ranks of the timed quantities; sum of the work
    if dist:
        (ms, t_h, k3_ms), (evals, evals_h, launches, rounds, executed) = aggregate_replicas(
            dist, (ms, t_h, k3_ms), (evals, evals_h, launches, rounds, executed), "cuda")
    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return 0

    instr, flop = rb_work(w.n_bins, w.n_det)
    traffic, traffic_note = profile_traffic()
    value = evals / (ms * 1e-3)
    k3_tf = (evals / world) * flop / (k3_ms * 1e-3) / 1e12
    k1_rate = N1 / (k1_ms * 1e-3)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": config_dict(w),
        "e2e": {"value": evals_h / t_h, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": 1e3 * t_h / e2e_steps, "timing": "host wall clock around the synchronous nss_iterate_host call"},
        "gpu_launches": launches,
        "evals_per_step": evals / args.steps / world,
        "wall_ms_timed_region": 1e3 * wall,
        "roofline": {"bound": "alu", "kernel": "k3_slice<3 detectors, relative binning, 16 lanes per candidate, table resident in shared "
                                                "memory>: one slice chain per CTA of 2 warps (4 bracket tests per round, "
                                                "speculative beyond the first), directions and likelihood inlined",
                     "achieved": k3_tf, "peak": peak_tf, "unit": "TFLOP/s", "frac": k3_tf / peak_tf,
                     "frac_of_nominal": k3_tf / NOMINAL_TF, "peak_nominal": NOMINAL_TF,
                     "peak_source": "fp64 DFMA chain measured in this process (nss_fp64_peak); nominal 148 SM x 64 lanes x 2 x "
                                    "1.965 GHz = 37.2; MEASURED_PEAKS.json has no fp64 figure",
                     "flop_per_eval": flop, "fp64_instr_per_eval": instr,
                     "pipe_frac": (evals / world) * instr / (k3_ms * 1e-3) / (peak_tf * 1e12 / 2),
                     "kernel_ms_per_step": k3_ms / args.steps, "kernel_share_of_step": k3_ms / ms_with_kernel_events,
                     "kernel_timing": "CUDA events recorded by the library around K3 on the launching stream, in a second pass over "
                                      "the same seeded steps (an event in front of K3 costs the launch overlap, so `ms_per_step` "
                                      "comes from the pass without them)",
                     "ms_per_step_with_kernel_events": ms_with_kernel_events / args.steps,
                     "traffic": traffic, "traffic_note": traffic_note,
                     "rounds_per_chain": rounds / args.steps / k / world, "evaluated_incl_speculative_per_step": executed / args.steps / world,
                     "frac_incl_speculative": (executed / world) * flop / (k3_ms * 1e-3) / 1e12 / peak_tf,
                     "note": "achieved and frac count only the evaluations the sequential algorithm consumed; "
                             "frac_incl_speculative counts every evaluation the kernel performed (the rate the fp64 pipe sees)",
                     # north_star's explicit target: "likelihood kernel >= 50 % of the fp64 roofline" (the batch kernel K1)
                     "likelihood_kernel": {"kernel": "k_rec_thread<3 detectors, cross term> (nss_loglike_batch, one thread per point)",
                                           "workload": "config 5: N=1e6 prior draws, B=128 x 3 detectors", "ms": k1_ms,
                                           "evals_per_s": k1_rate, "achieved": k1_rate * flop / 1e12, "unit": "TFLOP/s",
                                           "frac": k1_rate * flop / 1e12 / peak_tf,
                                           "frac_of_nominal": k1_rate * flop / 1e12 / NOMINAL_TF,
                                           "pipe_frac": k1_rate * instr / (peak_tf * 1e12 / 2)}},
        "loglike_batch": {"workload": "config 5: N=1e6 prior draws, B=128 x 3 detectors, k_rec_thread", "ms": k1_ms,
                          "evals_per_s": k1_rate, "tflops": k1_rate * flop / 1e12, "frac": k1_rate * flop / 1e12 / peak_tf,
                          "frac_of_nominal": k1_rate * flop / 1e12 / NOMINAL_TF,
                          "pipe_frac": k1_rate * instr / (peak_tf * 1e12 / 2)},
        "loglike_batch_full": {"workload": "config 4 likelihood: full grid 4017 bins x 3 detectors, N=1e5 prior draws, k_rec_sub<FULL>",
                               "ms": k2_ms, "evals_per_s": N2 / (k2_ms * 1e-3),
                               "fp64_instr_per_eval": 600 + w.n_freq * (8 + 22 * w.n_det),
                               "pipe_frac": N2 / (k2_ms * 1e-3) * (600 + w.n_freq * (8 + 22 * w.n_det)) / (peak_tf * 1e12 / 2),
                               "pipe_frac_of_nominal": N2 / (k2_ms * 1e-3) * (600 + w.n_freq * (8 + 22 * w.n_det)) / (NOMINAL_TF * 1e12 / 2),
                               "algorithmic_hbm_bytes_per_eval": 96,
                               "note": "the 484 KB record table is shared by every point and stays in L2; HBM GB/s is reported by "
                                       "profiles/r03_k2_full_grid_full.md"},
        "nss_run": run2,
        "clocks": clocks.summary(),
    }
    for key_, v_ in runs_extra.items():
        line["nss_run_" + key_] = v_
    if run1 is not None:
        line["nss_run_config1"] = run1
    if m3 is not None:
        instr4 = 600 + w.n_freq * (8 + 22 * w.n_det)
        line["step_config4"] = {
            "workload": "BASELINE.json configs[3]: config 2 with the full-frequency-grid likelihood (4017 bins x 3 detectors) inside K3",
            "steps": m4["steps"], "ms_per_step": m4["ms"] / m4["steps"], "evals_per_s": m4["evals"] / (m4["ms"] * 1e-3),
            "evals_per_step": m4["evals"] / m4["steps"], "kernel_ms_per_step": m4["k3_ms"] / m4["steps"],
            "fp64_instr_per_eval": instr4, "rounds_per_chain": m4["rounds"] / m4["steps"] / k,
            "pipe_frac": m4["evals"] * instr4 / (m4["k3_ms"] * 1e-3) / (peak_tf * 1e12 / 2),
            "pipe_frac_of_nominal": m4["evals"] * instr4 / (m4["k3_ms"] * 1e-3) / (NOMINAL_TF * 1e12 / 2),
            "note": "k3_slice<3, full grid, 32 lanes per candidate, table read from L2>: fraction of the DFMA issue peak by the "
                    "consumed evaluations only"}
        k3_tf3 = m3["evals"] * flop / (m3["k3_ms"] * 1e-3) / 1e12
        line["step_config3"] = {
            "workload": "BASELINE.json configs[2]: config 2 at n_live 5000, n_delete 2500 (55 repeats)", "steps": m3["steps"],
            "ms_per_step": m3["ms"] / m3["steps"], "evals_per_s": m3["evals"] / (m3["ms"] * 1e-3),
            "evals_per_step": m3["evals"] / m3["steps"], "gpu_launches": m3["launches"],
            "roofline": {"bound": "alu", "kernel": "k3_slice (single-warp chains, 8 lanes per candidate)", "achieved": k3_tf3,
                         "peak": peak_tf, "unit": "TFLOP/s", "frac": k3_tf3 / peak_tf, "frac_of_nominal": k3_tf3 / NOMINAL_TF,
                         "kernel_ms_per_step": m3["k3_ms"] / m3["steps"], "kernel_share_of_step": m3["k3_ms"] / m3["ms"],
                         "frac_incl_speculative": m3["executed"] * flop / (m3["k3_ms"] * 1e-3) / 1e12 / peak_tf,
                         "rounds_per_chain": m3["rounds"] / m3["steps"] / 2500,
                         "evaluated_incl_speculative_per_step": m3["executed"] / m3["steps"]}}
    # ---- CPU baseline: the oracle as it stands, on this box's host cores, bounded sample -----------------------
    if world == 1 and not args.no_cpu_baseline:
        from oracle import nss_oracle as orc
        orc.build()
        wo = inputs.make_data(inputs.config2(), orc.waveform)
        n_it = 16
        ev_o, s_o, cores = oracle_steps(wo, n_it, 0, w.n_repeats, SEED)
        line["cpu_baseline"] = {"value": ev_o / s_o, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"NS iterations 0..{n_it - 1} of the same config-2 run (n_live 1000, n_delete 500, "
                                          f"55 repeats): {ev_o} evaluations in {s_o:.1f} s, OpenMP over chains",
                                "note": "the oracle is an unoptimised checker (scalar loops, libm, an allocation per evaluation): "
                                        "a reported baseline, not a tuned CPU implementation"}
        line["oracle_legs"] = oracle_legs(wo, cores, gpu_small, {"rb": (k1_rate, N1), "full": (N2 / (k2_ms * 1e-3), N2)}, run2,
                                          not args.no_oracle_run, run1)
    print(json.dumps(line))
    g.close()
    if dist:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=("ours", "reference"))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the config-3/4 and paper-hyper-parameter extras")
    ap.add_argument("--no-oracle-run", action="store_true", help="skip the oracle's whole config-2 run (the longest CPU leg)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
