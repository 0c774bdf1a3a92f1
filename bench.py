#!/usr/bin/env python
"""bench.py -- log-lik + gradient evaluations/s of the phylogenetic-Hawkes hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl b200|reference] [--config 1] [--n N_EVENTS]

One "step" = one pass of the whole hot path through the C-ABI call
hawkes_grad: log-likelihood, d/dtheta for all N events and d/d(6 hyperparameters), on the seeded
synthetic events of BASELINE.json configs[1] (N = 23,422).  Rank 0 prints ONE
JSON line.  Timing is on the device (one CUDA-event pair per step on the launching stream, L2 flushed
between steps outside the event pairs), maximum over ranks.  With N > 1 (torchrun) every rank
evaluates its own replica -- the path is single-GPU by design (replicas only),
so `value` is N replicas' evaluations over the slowest rank's time ("scaling": "weak").

--impl reference times the ORACLE (oracle/, plain CPU fp64) on the host cores on a bounded sample of
the same workload; it is a deliberately slow baseline, not the target.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "loglik_grad_evals_per_s"
UNIT = "evals/s"

# Algorithmic FP64 work per pair (SURVEY.md 8(d) table with E = the flop
# count of the exponential actually shipped: 5 DFMA + 2 DADD + 1 DMUL = 8 FP64-pipe instructions, 13 flops).
# SURVEY 8(d) counts the double sum of Eq. 1 as it is written: one background term per ORDERED pair, one excitation
# term per causal pair.  The kernels evaluate the background once per UNORDERED pair (B is symmetric) and add it to
# both events, so the flops they execute are fewer; both figures are reported (roofline.frac uses the algorithmic
# count of SURVEY 8(d), roofline.frac_executed the executed one, fp64_pipe_issue_frac the executed instructions).
EXP_FLOPS, EXP_INSTR = 13, 8
P1_B_FLOPS, P1_S_FLOPS, P2_FLOPS = 15 + EXP_FLOPS, 9 + EXP_FLOPS, 12 + EXP_FLOPS
# executed per unordered pair by the symmetric pass 1: background 15 + E + 5 (second set of three sums), excitation 9 + E
P1_SYM_FLOPS, P1_SYM_INSTR = (15 + EXP_FLOPS + 5) + (9 + EXP_FLOPS), 21 + 13
FP64_LANES_PER_SM = 64


def pass1_flops(n: int) -> float:
    """gradient-level pass 1, algorithmic: every ordered pair carries a background term, every causal
    pair an excitation term"""
    return float(n) * n * P1_B_FLOPS + 0.5 * n * (n - 1) * P1_S_FLOPS


def pass1_flops_executed(n: int) -> float:
    """gradient-level pass 1 as executed: one background + one excitation term per unordered pair"""
    return 0.5 * n * (n - 1) * P1_SYM_FLOPS


def pass2_flops(n: int) -> float:
    return 0.5 * n * (n - 1) * P2_FLOPS


class ClockSampler:
    """Samples SM clock, power and throttle reasons of one GPU while the timed region runs
    (NVML through nvidia_ml_py; falls back to the recipe's nvidia-smi query loop)."""

    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
               0x80: "hw_power_brake", 0x2: "applications_clocks_setting", 0x100: "display_clock_setting",
               0x10: "sync_boost"}

    def __init__(self, index: int, period_s: float = 0.01):
        self.index, self.period = index, period_s
        self.sm, self.power, self.reason_bits = [], [], 0
        self.sm_max = None
        self._stop = threading.Event()
        self._thr = None
        self._proc = None
        self._nvml = None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nvml = pynvml
            uuid_index = self._physical_index()
            self._h = pynvml.nvmlDeviceGetHandleByIndex(uuid_index)
            self.sm_max = int(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()
        except Exception:
            self._nvml = None
            q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
                 "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
                 "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
            try:
                self._proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits",
                                               "-lms", "50", "-i", str(self._physical_index())],
                                              stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            except Exception:
                self._proc = None
        return self

    def _physical_index(self) -> int:
        vis = os.environ.get("CUDA_VISIBLE_DEVICES")
        if vis:
            parts = [p for p in vis.split(",") if p.strip() != ""]
            if self.index < len(parts) and parts[self.index].strip().isdigit():
                return int(parts[self.index])
        return self.index

    def _loop(self):
        nv = self._nvml
        while not self._stop.is_set():
            try:
                self.sm.append(int(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self._h) / 1000.0)
                self.reason_bits |= int(nv.nvmlDeviceGetCurrentClocksEventReasons(self._h))
            except Exception:
                try:
                    self.reason_bits |= int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                except Exception:
                    pass
            self._stop.wait(self.period)

    def stop(self) -> dict:
        self._stop.set()
        if self._thr is not None:
            self._thr.join(timeout=2.0)
        reasons = [name for bit, name in self.REASONS.items() if self.reason_bits & bit]
        if self._proc is not None:
            self._proc.terminate()
            try:
                out, _ = self._proc.communicate(timeout=5)
            except Exception:
                out = ""
            names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
            seen = set()
            for line in out.splitlines():
                f = [s.strip() for s in line.split(",")]
                if len(f) < 9:
                    continue
                try:
                    self.sm.append(int(float(f[1])))
                    self.sm_max = int(float(f[2]))
                    self.power.append(float(f[3]))
                except ValueError:
                    continue
                for name, val in zip(names, f[5:9]):
                    if val.lower().startswith("active"):
                        seen.add(name)
            reasons = sorted(seen)
        if not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": reasons, "samples": 0}
        return {"sm_mhz": int(statistics.median(self.sm)), "sm_min_mhz": min(self.sm), "sm_max_mhz": self.sm_max,
                "power_w_max": round(max(self.power), 1) if self.power else None,
                "reasons": reasons, "samples": len(self.sm)}


# ------------------------------------------------------------------------------------------------
# the oracle, timed on the host cores (cpu_baseline leg and --impl reference)
def oracle_sample_seconds(ev, idx, threads: int) -> float:
    """Seconds the oracle needs for the sampled target rows (lambda_n and its 6 hyper-derivatives: pass 1)
    plus the same number of sampled source columns (c_m, d_m: pass 2).  The column routine needs every
    lambda_n; for timing it is given a vector of ones (same arithmetic, no O(N^2) set-up)."""
    import numpy as np
    import oracle
    t0 = time.perf_counter()
    oracle.rows(ev.x, ev.t, ev.theta, ev.params, idx, derivs=True, threads=threads)
    oracle.cols(ev.x, ev.t, ev.params, np.ones(ev.n), idx, threads=threads)
    return time.perf_counter() - t0


def sample_idx(n: int, r: int):
    import numpy as np
    r = max(1, min(n, r))
    return np.unique(np.linspace(0, n - 1, r).astype(np.int64))


def cpu_baseline(ev, budget_s: float = 15.0) -> dict:
    import oracle
    threads = oracle.max_threads()
    probe = sample_idx(ev.n, 64)
    per_row = oracle_sample_seconds(ev, probe, threads) / len(probe)
    idx = sample_idx(ev.n, int(budget_s / max(per_row, 1e-9)))
    secs = oracle_sample_seconds(ev, idx, threads)
    evals_per_s = (len(idx) / ev.n) / secs
    # the same oracle on ONE thread, on a smaller sample (about 3 s)
    idx1 = sample_idx(ev.n, max(8, int(3.0 / max(per_row * threads, 1e-9))))
    secs1 = oracle_sample_seconds(ev, idx1, 1)
    return {"value": evals_per_s, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": f"{len(idx)} of {ev.n} target rows (lambda_n + 6 hyper-derivatives) and the same {len(idx)} "
                      f"source columns (c_m), evenly strided, {secs:.1f} s on {threads} OpenMP threads; "
                      f"evals/s = (rows/N) / seconds",
            "seconds_per_eval_extrapolated": 1.0 / evals_per_s,
            "single_thread": {"seconds_per_eval_extrapolated": secs1 * ev.n / len(idx1), "cores": 1,
                              "sample": f"{len(idx1)} of {ev.n} rows and columns, {secs1:.1f} s"}}


def run_reference(args, ev, workload: str) -> dict:
    """--impl reference: the oracle as it stands, each step a bounded sample of the workload."""
    import oracle
    threads = oracle.max_threads()
    per_row = oracle_sample_seconds(ev, sample_idx(ev.n, 64), threads) / 64.0
    budget = 150.0 / (args.steps + args.warmup)
    idx = sample_idx(ev.n, max(16, int(budget / max(per_row, 1e-9))))
    for _ in range(args.warmup):
        oracle_sample_seconds(ev, idx, threads)
    secs = [oracle_sample_seconds(ev, idx, threads) for _ in range(args.steps)]
    per_eval = (sum(secs) / len(secs)) * ev.n / len(idx)
    value = 1.0 / per_eval
    sample = (f"each step = {len(idx)} of {ev.n} target rows + the same source columns, evenly strided, "
              f"extrapolated by N/rows; {threads} OpenMP threads")
    return {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": per_eval * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload, "n_events": ev.n, "dim": ev.dim},
            "gpairs_per_s": ev.n * float(ev.n) * value / 1e9,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


# ------------------------------------------------------------------------------------------------
# the CUDA path
def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1)), int(os.environ.get("LOCAL_RANK", 0))


# Multi-GPU = independent replicas: rank r evaluates the problem drawn with seed + r on its own
# GPU, no data-path collective; the only exchange is the MAX over ranks of the timed totals.  These three helpers are
# the whole N > 1 logic and are covered by world-size-2 gloo tests on CPU (tests/test_multiproc.py).
def replica_seed(seed: int, rank: int) -> int:
    return int(seed) + int(rank)


def max_over_ranks(dist, values, device):
    """all-reduce(MAX) of a list of floats; identity when dist is None (single process)."""
    if dist is None:
        return [float(v) for v in values]
    import torch
    v = torch.tensor([float(a) for a in values], dtype=torch.float64, device=device)
    dist.all_reduce(v, op=dist.ReduceOp.MAX)
    return [float(a) for a in v]


def whole_job_value(world: int, steps: int, total_ms_max: float) -> float:
    """evaluations/s of the whole job: every rank did `steps` evaluations within the slowest rank's time."""
    return world * steps / (total_ms_max * 1e-3)


def ncu_record(kernel: str, n: int) -> dict:
    """What the committed `ncu --set full` capture of `kernel` at N = n says (profiles/traffic.csv: kernel, n_events,
    dram_bytes_per_launch, fp64_pipe_pct_active, fp64_pipe_pct_elapsed, source; profiles/traffic.md names the
    commands): DRAM bytes per launch and the FP64-pipe utilisation.  Every value is None when there is no capture of
    this kernel at this N -- a number profiled at another size is not reported."""
    none = {"traffic": None, "ncu_fp64_pipe_pct_active": None, "ncu_fp64_pipe_pct_elapsed": None, "ncu_source": None}
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        with open(path) as fh:
            for line in fh:
                f = [p.strip() for p in line.split(",")]
                if len(f) >= 6 and f[0] == kernel and f[1].isdigit() and int(f[1]) == int(n):
                    return {"traffic": float(f[2]), "ncu_fp64_pipe_pct_active": float(f[3]),
                            "ncu_fp64_pipe_pct_elapsed": float(f[4]), "ncu_source": "profiles/" + f[5]}
    except Exception:
        pass
    return none


def roofline_records(n: int, p1_ms: float, p2_ms: float, sym: bool, peak_nominal: float, peak_dfma, instr_peak: float):
    """`roofline` (pass 1, the dominant kernel) and `roofline_pass2` from the kernels' mean launch durations.
    achieved = algorithmic flops of SURVEY 8(d) per launch / duration; the executed count and the FP64 issue fraction
    depend on which pass-1 form ran (`sym`: background once per unordered pair)."""
    a1 = pass1_flops(n) / (p1_ms * 1e-3) / 1e12
    a2 = pass2_flops(n) / (p2_ms * 1e-3) / 1e12
    if sym:
        kernel1, key1 = "pass1s_kernel<R=2, LEVEL=1> (symmetric background)", "pass1s_kernel"
        x1 = pass1_flops_executed(n)
        i1 = 0.5 * n * (n - 1) * P1_SYM_INSTR
    else:   # dense ordered-pair kernel: executes what SURVEY 8(d) counts (18 / 13 FP64 instructions per term)
        kernel1, key1 = "pass1_kernel<R=2, LEVEL=1> (dense ordered pairs)", "pass1_kernel"
        x1 = pass1_flops(n)
        i1 = float(n) * n * 18 + 0.5 * n * (n - 1) * 13
    a1x = x1 / (p1_ms * 1e-3) / 1e12
    r1 = {"bound": "alu", "kernel": kernel1, "achieved": a1, "peak": peak_nominal, "unit": "TFLOP/s",
          "frac": a1 / peak_nominal,
          "flops_basis": "SURVEY 8(d): N^2 background + N(N-1)/2 excitation terms of Eq. 1, 28 / 22 flops each",
          "achieved_executed": a1x, "frac_executed": a1x / peak_nominal, "flops_executed_per_launch": x1,
          "peak_source": "derived: SMs x 64 FP64 FMA lanes x 2 x clocks.max.sm; MEASURED_PEAKS.json has no FP64 entry",
          "peak_measured_dfma": peak_dfma, "frac_of_measured_dfma": a1 / peak_dfma if peak_dfma else None,
          "fp64_pipe_issue_frac": i1 / (p1_ms * 1e-3) / instr_peak,
          "ms_per_launch": p1_ms, "flops_per_launch": pass1_flops(n)}
    r1.update(ncu_record(key1, n))
    r2 = {"bound": "alu", "kernel": "pass2_kernel", "achieved": a2, "peak": peak_nominal, "unit": "TFLOP/s",
          "frac": a2 / peak_nominal, "frac_of_measured_dfma": a2 / peak_dfma if peak_dfma else None,
          "fp64_pipe_issue_frac": 0.5 * n * (n - 1) * 13 / (p2_ms * 1e-3) / instr_peak,
          "ms_per_launch": p2_ms, "flops_per_launch": pass2_flops(n)}
    r2.update(ncu_record("pass2_kernel", n))
    return r1, r2


def parity_sample(hp, ctx, ev, out, rows: int) -> dict:
    """Parity in this very run: `rows` evenly strided rows of lambda_n and d lambda_n/dp and the same columns of c_m
    against the oracle (scaled as tests/test_parity_gpu.py does)."""
    import numpy as np
    import oracle
    n = ev.n
    sidx = sample_idx(n, rows)
    thr = oracle.max_threads()
    lam_gpu = ctx.get_lambda(n).cpu().numpy()
    d1_gpu = ctx.get_row_moments(n).cpu().numpy()[sidx]
    lam_ref, d1_ref = oracle.rows(ev.x, ev.t, ev.theta, ev.params, sidx, derivs=True, threads=thr)
    c_ref, _ = oracle.cols(ev.x, ev.t, ev.params, lam_gpu, sidx, threads=thr)
    mu0, tx, tt, xi0, h, om = ev.params
    D = ev.dim
    cp = np.array([1 / mu0, D / tx, 1 / tt, 1 / xi0, D / h, 1 / om])
    s1 = np.abs(d1_ref) + cp[None, :] * lam_ref[:, None]
    integ = xi0 * (-np.expm1(-om * (ev.t[-1] - ev.t[sidx])))
    g_gpu = out.grad_theta.cpu().numpy()[sidx]
    return {"rows": int(len(sidx)),
            "max_rel_err_lambda": float(np.max(np.abs(lam_gpu[sidx] - lam_ref) / lam_ref)),
            "max_scaled_err_dlambda_dhyper": float(np.max(np.abs(d1_gpu - d1_ref) / s1)),
            "max_scaled_err_grad_theta": float(np.max(np.abs(g_gpu - (c_ref - integ)) / (np.abs(c_ref) + integ + 1e-300))),
            "tolerance": 1e-10}


def timed_steps(torch, dev, call, steps, flush):
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for e0, e1 in evs:
        flush.zero_()
        e0.record()
        call()
        e1.record()
    torch.cuda.synchronize(dev)
    return [e0.elapsed_time(e1) for e0, e1 in evs]


def sweep_entry(torch, hp, dev, local, n, seed, flush, peaks, with_parity: bool) -> dict:
    """One size of BASELINE.json configs[4]: 3 warm-up + 5 timed hawkes_grad steps on a fresh context."""
    import numpy as np
    from paper_2103_03348_b200 import synth
    ev = synth.config(4, n=n, seed=seed)
    ctx = hp.HawkesContext(n, ev.dim, local)
    f = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    x, t, th = f(ev.x), f(ev.t), f(ev.theta)
    out = ctx.new_outputs(n, hp.WANT_GRAD, dev)
    step = lambda: ctx.grad(x, t, th, ev.params, out=out)
    timed_steps(torch, dev, step, 3, flush)
    assert ctx.last_status() == 0
    sampler = ClockSampler(local).start()
    ctx.profile_enable(True)
    ms = timed_steps(torch, dev, step, 5, flush)
    prof = ctx.profile_read()
    ctx.profile_enable(False)
    clocks = sampler.stop()
    cnt = max(prof["evals"], 1)
    p1_ms, p2_ms = prof["pass1_ms"] / cnt, prof["pass2_ms"] / cnt
    sym = ctx.pass1_is_symmetric(1)
    r1, r2 = roofline_records(n, p1_ms, p2_ms, sym, *peaks)
    ms_step = float(sum(ms)) / len(ms)
    e = {"n_events": n, "steps": 5, "warmup": 3, "ms_per_step": ms_step, "evals_per_s": 1e3 / ms_step,
         "gpairs_per_s": float(n) * n / (ms_step * 1e-3) / 1e9,
         "pass1": {k: r1[k] for k in ("kernel", "ms_per_launch", "frac", "frac_executed", "fp64_pipe_issue_frac",
                                      "traffic", "ncu_fp64_pipe_pct_elapsed")},
         "pass2": {k: r2[k] for k in ("ms_per_launch", "frac", "fp64_pipe_issue_frac", "traffic",
                                      "ncu_fp64_pipe_pct_elapsed")},
         "step_frac_of_fp64_peak": (pass1_flops(n) + pass2_flops(n)) / (ms_step * 1e-3) / 1e12 / peaks[0],
         "ll": float(out.ll.item()), "clocks": clocks}
    if with_parity:
        e["parity_sample"] = parity_sample(hp, ctx, ev, out, 128)
    ctx.close()
    return e


def run_b200(args, ev, workload: str) -> dict:
    import numpy as np
    import torch
    import paper_2103_03348_b200 as hp

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        torch.cuda.synchronize(dev)
        if dist is not None:
            dist.barrier(device_ids=[local])
            torch.cuda.synchronize(dev)

    n, K, W = ev.n, args.steps, args.warmup
    ctx = hp.HawkesContext(n, ev.dim, local)
    x = torch.from_numpy(np.ascontiguousarray(ev.x)).to(dev)
    t = torch.from_numpy(np.ascontiguousarray(ev.t)).to(dev)
    th = torch.from_numpy(np.ascontiguousarray(ev.theta)).to(dev)
    out = ctx.new_outputs(n, hp.WANT_GRAD, dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # 2x the 126 MB L2

    timed = lambda call, steps: timed_steps(torch, dev, call, steps, flush)

    step = lambda: ctx.grad(x, t, th, ev.params, out=out)
    if args.shard:
        # ONE evaluation cut across the ranks (hawkes_shard_*): every rank holds the same events,
        # evaluates its share of both pairwise passes and all-gathers the partial sums (NCCL) -- "scaling": "strong"
        step = lambda: hp.shard_eval(ctx, dist, rank, world, x, t, th, ev.params, hp.WANT_GRAD, out=out)
    # -- device-resident leg ----------------------------------------------------------------------
    timed(step, W)
    assert ctx.last_status() == 0, "evaluation reported a data error"
    barrier()
    sampler = ClockSampler(local).start()
    ctx.profile_enable(True)
    l0 = ctx.launch_count()
    wall0 = time.perf_counter()
    ms = timed(step, K)
    barrier()
    wall = time.perf_counter() - wall0
    launches = ctx.launch_count() - l0
    prof = ctx.profile_read() if not args.shard else None
    ctx.profile_enable(False)
    total_ms = float(sum(ms))
    # -- end-to-end leg: HOST buffers through hawkes_eval_host (H2D of inputs + D2H of results inside) ----
    hx, ht, hth = (a.cpu().pin_memory() for a in (x, t, th))
    hout = ctx.new_outputs(n, hp.WANT_GRAD, "cpu", pinned=True)
    estep = lambda: ctx.eval_host(hx, ht, hth, ev.params, hp.WANT_GRAD, out=hout)
    if args.shard:
        def estep():   # host buffers in, sharded evaluation, replicated results back to the host on every rank
            x.copy_(hx, non_blocking=True); t.copy_(ht, non_blocking=True); th.copy_(hth, non_blocking=True)
            hp.shard_eval(ctx, dist, rank, world, x, t, th, ev.params, hp.WANT_GRAD, out=out)
            hout.ll.copy_(out.ll, non_blocking=True)
            hout.grad_theta.copy_(out.grad_theta, non_blocking=True)
            hout.grad_hyper.copy_(out.grad_hyper, non_blocking=True)
            torch.cuda.current_stream(dev).synchronize()
    timed(estep, W)
    barrier()
    e_ms = timed(estep, K)
    barrier()
    e_total = float(sum(e_ms))
    clocks = sampler.stop()
    total_ms, e_total = max_over_ranks(dist, [total_ms, e_total], dev)
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return {}

    # -- everything below: rank 0 only --------------------------------------------------------------
    ll_dev = float(out.ll.item())
    ll_host = float(hout.ll.item())
    assert ll_dev == ll_host, "device-resident and host-buffer evaluations must be bit-identical"
    # replicas: every rank did K evaluations of its own problem; sharded: the ranks did K evaluations together
    value = whole_job_value(1 if args.shard else world, K, total_ms)
    e_value = whole_job_value(1 if args.shard else world, K, e_total)
    props = torch.cuda.get_device_properties(dev)
    sm_max = clocks.get("sm_max_mhz") or 1965
    peak_nominal = props.multi_processor_count * FP64_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    peak_dfma = ctx.fp64_peak(200.0)
    if args.shard:   # the per-kernel ring belongs to hawkes_eval; a sharded step reports the whole step only
        if dist is not None:
            dist.destroy_process_group()
        return {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": workload, "n_events": n, "dim": ev.dim, "call": "hawkes_shard_pass1/reduce1/pass2/finish",
                           "parallelism": f"one evaluation sharded across {world} ranks (2 all-gathers per evaluation)",
                           "l2": "256 MiB memset between timed steps, outside the per-step event pairs"},
                "gpairs_per_s": float(n) * n * value / 1e9, "gpu_launches": int(launches), "clocks": clocks,
                "e2e": {"value": e_value, "unit": UNIT, "ms_per_step": e_total / K,
                        "h2d_bytes_per_step": int((ev.dim + 2) * n * 8), "d2h_bytes_per_step": int((1 + n + 6) * 8),
                        "call": "pinned host buffers -> shard_eval -> pinned host buffers, on every rank"},
                "ll": ll_dev}
    p1_ms = prof["pass1_ms"] / max(prof["evals"], 1)
    p2_ms = prof["pass2_ms"] / max(prof["evals"], 1)
    inner_ms = prof["total_ms"] / max(prof["evals"], 1)
    instr_peak = props.multi_processor_count * FP64_LANES_PER_SM * sm_max * 1e6
    peaks = (peak_nominal, peak_dfma, instr_peak)
    roof1, roof2 = roofline_records(n, p1_ms, p2_ms, ctx.pass1_is_symmetric(1), *peaks)
    roof1["peak_source"] = (f"derived: {props.multi_processor_count} SMs x {FP64_LANES_PER_SM} FP64 FMA lanes x 2 x "
                            f"{sm_max} MHz (clocks.max.sm); MEASURED_PEAKS.json has no FP64 entry")
    res = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "strong" if args.shard else "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload, "n_events": n, "dim": ev.dim, "outputs": "ll + grad_theta[N] + grad_hyper[6]",
                   "call": "hawkes_grad", "l2": "256 MiB memset between timed steps, outside the per-step event pairs",
                   "parallelism": ("1 GPU" if world == 1 and not args.shard else
                                   f"one evaluation sharded across {world} ranks (2 all-gathers per evaluation)" if args.shard
                                   else f"{world} independent replicas (no collective)")},
        "gpairs_per_s": float(n) * n * value / 1e9,
        "kernel_terms_per_s": (float(n) * n + float(n) * (n - 1)) * value,
        "wall_s_timed_region": wall,
        "gpu_launches": int(launches),
        "clocks": clocks,
        "e2e": {"value": e_value, "unit": UNIT, "ms_per_step": e_total / K,
                "h2d_bytes_per_step": int((ev.dim + 2) * n * 8), "d2h_bytes_per_step": int((1 + n + 6) * 8),
                "call": "hawkes_eval_host (pinned host buffers)"},
        "roofline": roof1,
        "roofline_pass2": roof2,
        "kernel_share": {"pass1": p1_ms / inner_ms, "pass2": p2_ms / inner_ms,
                         "o_n_and_gaps": 1.0 - (p1_ms + p2_ms) / inner_ms, "first_to_last_kernel_ms": inner_ms},
        "ll": ll_dev,
    }
    if args.extras:
        hout_all = ctx.new_outputs(n, hp.WANT_HESS_THETA | hp.WANT_HESS_HYPER, dev)
        hstep = lambda: ctx.hessian(x, t, th, ev.params, out=hout_all)
        timed(hstep, 2)
        hms = timed(hstep, max(3, K // 4))
        # the whole Hessian of configs[0]'s reading: theta-diagonal + 6x6 + the N x 6 cross block (csrc/cross.cuh)
        xout = ctx.new_outputs(n, hp.WANT_HESS_THETA | hp.WANT_HESS_HYPER | hp.WANT_HESS_CROSS, dev)
        xstep = lambda: ctx.hessian(x, t, th, ev.params, cross=True, out=xout)
        timed(xstep, 2)
        xms = timed(xstep, max(3, K // 4))
        conly = ctx.new_outputs(n, hp.WANT_HESS_CROSS, dev)
        cstep = lambda: ctx.eval(x, t, th, ev.params, hp.WANT_HESS_CROSS, out=conly)
        timed(cstep, 2)
        cms = timed(cstep, max(3, K // 4))
        lstep = lambda: ctx.eval(x, t, th, ev.params, hp.WANT_LL | hp.WANT_GRAD_THETA, out=out)
        timed(lstep, 2)
        lms = timed(lstep, max(3, K // 4))
        # same events at the paper's posterior scales (Table 2: tau_x = 194 km, h = 7.37 km, 1/omega = 29.8 d),
        # where no exponential underflows: the kernels are dense, so the time must not depend on the regime
        from paper_2103_03348_b200 import synth as _synth
        t2step = lambda: ctx.grad(x, t, th, _synth.TABLE2_PARAMS, out=out)
        timed(t2step, 2)
        t2ms = timed(t2step, max(3, K // 4))
        # ... and the exact-zero-skipping variant at those scales: the background reaches the whole domain there,
        # only the self-excitation lists shrink (the gain of that variant is data-dependent)
        t2stats = ctx.skip_plan(x, t, _synth.TABLE2_PARAMS)
        t2skip = lambda: ctx.eval_skip(x, t, th, _synth.TABLE2_PARAMS, hp.WANT_GRAD, out=out)
        timed(t2skip, 2)
        t2sms = timed(t2skip, max(3, K // 4))
        # SURVEY 8(e) on one GPU: the phases of every rank of a sharded evaluation timed one after the other (no exchange,
        # no overlap): what each GPU of an N-GPU job would compute; the two all-gathers come on top
        shard = {}
        for wd in (2, 4, 8):
            mk = lambda *sh: torch.empty(*sh, dtype=torch.float64, device=dev)
            parts = mk(wd, ctx.shard_part_doubles(n, hp.WANT_GRAD, 1))
            parts2 = mk(wd, ctx.shard_part_doubles(n, hp.WANT_GRAD, 2))
            sout = ctx.new_outputs(n, hp.WANT_GRAD, dev)
            per = {"pass1": [], "pass2": []}
            for rep in range(2):                      # first repetition = warm-up
                per = {"pass1": [], "pass2": []}
                for r in range(wd):
                    per["pass1"].append(_event_timed(torch, dev, lambda: ctx.shard_pass1(x, t, th, ev.params, hp.WANT_GRAD, r, wd, parts[r]), 1)[0])
                red = _event_timed(torch, dev, lambda: ctx.shard_reduce1(n, ev.params, hp.WANT_GRAD, wd, parts, sout), 1)[0]
                for r in range(wd):
                    per["pass2"].append(_event_timed(torch, dev, lambda: ctx.shard_pass2(n, ev.params, hp.WANT_GRAD, r, wd, parts2[r]), 1)[0])
                fin = _event_timed(torch, dev, lambda: ctx.shard_finish(n, ev.params, hp.WANT_GRAD, wd, parts2, sout), 1)[0]
            slowest = max(per["pass1"]) + red + max(per["pass2"]) + fin
            shard[str(wd)] = {"pass1_ms_per_rank": per["pass1"], "pass2_ms_per_rank": per["pass2"], "reduce1_ms": red,
                              "finish_ms": fin, "slowest_rank_compute_ms": slowest,
                              "all_gather_bytes_per_rank": [int(parts[0].numel() * 8), int(parts2[0].numel() * 8)],
                              "ll_rel_diff_vs_one_gpu": abs(sout.ll.item() - ll_dev) / abs(ll_dev)}
        timed(step, 1)   # leave `out` holding the configs[1] result
        res["shard_emulation_one_gpu"] = shard
        res["extras"] = {"hessian_ms": statistics.median(hms), "ll_grad_theta_only_ms": statistics.median(lms),
                         "hessian_with_cross_block_ms": statistics.median(xms),
                         "cross_block_only_ms": statistics.median(cms),
                         "step_ms_min": min(ms), "step_ms_median": statistics.median(ms),
                         "table2_scales_step_ms": statistics.median(t2ms),
                         "table2_scales_skip_step_ms": statistics.median(t2sms),
                         "table2_scales_skip_tile_pairs": {
                             "pass1_background": t2stats["items_background"] / t2stats["items_dense_pass1"],
                             "pass1_excitation": t2stats["items_excitation"] / t2stats["items_dense_pass1"]}}
    # the O(N) kernels (prep, reduce1, theta) against the measured HBM copy peak: bytes they move per evaluation
    # (records in and out, row-partial slots, column partials: about N^2 * 12 / tile of them), time from the ring
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            hbm_peak = float(json.load(fh)["hbm_gbs"])
    except Exception:
        hbm_peak = 6537.3   # SURVEY.md 8(d) fallback
    tile, w1, w2 = 256, 3 * props.multi_processor_count, 4 * props.multi_processor_count
    n_tiles = (n + tile - 1) // tile
    on_bytes = (n * 64.0                                                      # prep: SoA in, records out
                + (n + w1 * tile) * 6 * 8.0 + 0.5 * n * n_tiles * 3 * 8.0     # reduce1: row slots + column partials
                + n * (32 + 32 + 8 + 34 * 8 / 64.0)                           #          two record streams, lambda, block sums
                + (n + w2 * tile) * 8.0 + n * 16.0)                           # theta: pass-2 slots in, gradient out
    on_ms = (prof["prep_ms"] + prof["mid_ms"] + prof["tail_ms"]) / max(prof["evals"], 1)
    cnt_ = max(prof["evals"], 1)
    res["o_n_kernels"] = {"ms_with_launch_gaps": on_ms, "prep_ms": prof["prep_ms"] / cnt_,
                          "reduce1_to_pass2_ms": prof["mid_ms"] / cnt_, "theta_ms": prof["tail_ms"] / cnt_,
                          "bytes_per_eval_estimate": on_bytes,
                          "achieved_gb_s": on_bytes / (on_ms * 1e-3) / 1e9, "hbm_peak_gb_s": hbm_peak,
                          "frac": on_bytes / (on_ms * 1e-3) / 1e9 / hbm_peak,
                          "note": "launch-latency-bound by nature; the data they touch is L2-resident"}
    if world == 1 and not args.no_cpu_baseline:
        # parity on a sample, in this very run: 256 rows of lambda_n / d lambda_n/dp and 256 columns of c_m
        timed(step, 1)
        res["parity_sample"] = parity_sample(hp, ctx, ev, out, 256)
        res["cpu_baseline"] = cpu_baseline(ev, args.cpu_budget)
    if world == 1:
        # SURVEY 8(f)-4, reported apart from the dense numbers above (the paper's method visits every pair): the same
        # call over the work lists of hawkes_skip_plan, which leave out tile pairs that hold exact zeros only
        t_plan = time.perf_counter()
        stats = ctx.skip_plan(x, t, ev.params)
        plan_ms = (time.perf_counter() - t_plan) * 1e3
        sout = ctx.new_outputs(n, hp.WANT_GRAD, dev)
        sstep = lambda: ctx.eval_skip(x, t, th, ev.params, hp.WANT_GRAD, out=sout)
        timed(sstep, W)
        assert ctx.last_status() == 0
        sms = timed(sstep, K)
        g_d, g_s = out.grad_theta, sout.grad_theta
        res["exact_zero_skipping"] = {
            "call": "hawkes_skip_plan once + hawkes_eval_skip per step (same outputs as hawkes_grad)",
            "ms_per_step": float(sum(sms)) / K, "value": K / (float(sum(sms)) * 1e-3), "unit": UNIT,
            "speedup_over_dense": total_ms / float(sum(sms)), "plan_ms_host_once": plan_ms,
            "tile_pairs_visited": {"pass1_background": stats["items_background"] / stats["items_dense_pass1"],
                                   "pass1_excitation": stats["items_excitation"] / stats["items_dense_pass1"],
                                   "pass2": stats["items_pass2"] / stats["items_dense_pass2"],
                                   "pass1_background_unordered_items": stats["items_background_unordered"]},
            "max_rel_diff_vs_dense": {"ll": abs(sout.ll.item() - ll_dev) / abs(ll_dev),
                                      "grad_theta": float((g_s - g_d).abs().max() / g_d.abs().max()),
                                      "grad_hyper": float((sout.grad_hyper - out.grad_hyper).abs().max()
                                                          / out.grad_hyper.abs().max())},
            "note": "data-dependent: only terms that are exactly +0.0 in fp64 are left out; not the headline"}
    if world == 1 and args.n is None and args.config == 1 and not args.no_sweep:
        # BASELINE.json configs[4] / north_star's second size: N = 50,000 / 100,000 / 250,000 from the same generator,
        # 3 warm-up + 5 timed steps each, with the clocks sampled during each entry's timed region and (unless
        # --no-cpu-baseline) 128 rows and columns of each against the oracle
        ctx.close()
        del ctx
        torch.cuda.empty_cache()
        res["sweep"] = [sweep_entry(torch, hp, dev, local, nn, args.seed, flush, peaks, not args.no_cpu_baseline)
                        for nn in (50000, 100000, 250000)]
        res["configs"] = other_configs(args)
    if dist is not None:
        dist.destroy_process_group()
    return res


# ------------------------------------------------------------------------------------------------
# BASELINE.json configs[2] and configs[3]: secondary bench lines (python bench.py --config 2 | 3)
def _setup_tree_problem(args, torch, hp, dev):
    import numpy as np
    from paper_2103_03348_b200 import synth
    ev, tree, z = synth.config_tree(args.seed)
    to = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    ctx = hp.HawkesContext(ev.n, ev.dim, dev.index)
    tr = hp.HawkesTree(tree.parent, tree.branch, dev.index)
    return ev, tree, z, ctx, tr, to


def _event_timed(torch, dev, call, steps, flush=None):
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for e0, e1 in evs:
        if flush is not None:
            flush.zero_()
        e0.record()
        call()
        e1.record()
    torch.cuda.synchronize(dev)
    return [e0.elapsed_time(e1) for e0, e1 in evs]


def run_posterior(args) -> dict:
    """configs[2]: gradient + Hessian diagonal of the log-likelihood in z plus the tree-diffusion prior and its
    gradient, N = 23,422, M = 1,610: one hawkes_posterior_z call per step."""
    import numpy as np
    import torch
    import paper_2103_03348_b200 as hp
    from paper_2103_03348_b200 import synth
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    ev, tree, z, ctx, tr, to = _setup_tree_problem(args, torch, hp, dev)
    n, M, K, W = ev.n, tree.n_tips, args.steps, args.warmup
    x, t, idx, zd = to(ev.x), to(ev.t), to(ev.free_idx), to(z)
    s2, tau0 = synth.TREE_SIGMA2, synth.TREE_TAU0
    out = ctx.posterior_z(tr, x, t, idx, zd, 0.0, ev.params, s2, tau0, hess=True)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    step = lambda: ctx.posterior_z(tr, x, t, idx, zd, 0.0, ev.params, s2, tau0, hess=True, out=out)
    _event_timed(torch, dev, step, W, flush)
    sampler = ClockSampler(0).start()
    ctx.profile_enable(True)
    l0, t0 = ctx.launch_count(), tr.launch_count()
    ms = _event_timed(torch, dev, step, K, flush)
    launches = ctx.launch_count() - l0 + tr.launch_count() - t0
    prof = ctx.profile_read()
    ctx.profile_enable(False)
    tree_ms = _event_timed(torch, dev, lambda: tr.prior(zd, s2, tau0), K)
    # end to end: z from pinned host memory in, (ell, log prior, sum), grad_z, hess_z back to pinned host memory
    hz = torch.from_numpy(z).pin_memory()
    hout = [torch.empty(k, dtype=torch.float64).pin_memory() for k in (3, M, M)]

    def estep():
        zd.copy_(hz, non_blocking=True)
        ctx.posterior_z(tr, x, t, idx, zd, 0.0, ev.params, s2, tau0, hess=True, out=out)
        for h, d in zip(hout, out):
            h.copy_(d, non_blocking=True)
        torch.cuda.current_stream(dev).synchronize()

    _event_timed(torch, dev, estep, W, flush)
    e_ms = _event_timed(torch, dev, estep, K, flush)
    clocks = sampler.stop()
    total, cnt = float(sum(ms)), max(prof["evals"], 1)
    res = {"metric": "posterior_grad_hess_evals_per_s", "value": K / (total * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": K,
           "warmup": W, "ms_per_step": total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic",
           "config": {"workload": "BASELINE.json configs[2]: N=23,422 events, 1,610 log-rates from Brownian diffusion "
                                  "(sigma^2=0.25, tau0=0.1) on a seeded coalescent tree; ell + log prior, d/dz, "
                                  "diagonal d2 ell/dz2", "n_events": n, "n_tips": M, "tree_levels": tr.levels(),
                      "call": "hawkes_posterior_z", "l2": "256 MiB memset between timed steps", "parallelism": "1 GPU"},
           "gpairs_per_s": float(n) * n * K / (total * 1e-3) / 1e9, "gpu_launches": int(launches), "clocks": clocks,
           "e2e": {"value": K / (float(sum(e_ms)) * 1e-3), "unit": UNIT, "ms_per_step": float(sum(e_ms)) / K,
                   "h2d_bytes_per_step": int(M * 8), "d2h_bytes_per_step": int((3 + 2 * M) * 8),
                   "call": "pinned z -> hawkes_posterior_z -> pinned (out3, grad_z, hess_z)"},
           "breakdown_ms": {"pass1_level0": prof["pass1_ms"] / cnt, "pass2_level1": prof["pass2_ms"] / cnt,
                            "hawkes_eval_first_to_last_kernel": prof["total_ms"] / cnt,
                            "tree_prior_kernel": statistics.median(tree_ms)},
           "out3": [float(v) for v in out[0].cpu()]}
    if not args.no_cpu_baseline:
        import oracle
        from oracle import tree as otree
        threads = oracle.max_threads()
        t0_ = time.perf_counter()
        V = otree.vg(tree.parent, tree.branch, M, tau0)
        otree.log_prior(V, z, s2)
        prior_s = time.perf_counter() - t0_
        cb = cpu_baseline(ev, args.cpu_budget)
        per_eval = cb["seconds_per_eval_extrapolated"] + prior_s
        res["cpu_baseline"] = {"value": 1.0 / per_eval, "unit": UNIT, "cores": threads, "kind": "oracle",
                               "sample": cb["sample"] + f"; plus the dense prior oracle in full (V_G + long-double "
                                                        f"Cholesky, M={M}: {prior_s:.1f} s, 1 thread)"}
    return res


def run_hmc(args, only=None) -> dict:
    """configs[3]: preconditioned HMC on z, 20 leapfrog steps per iteration, preconditioner refreshed every 10
    iterations; --steps = timed iterations (BASELINE: 200).  only: names of the extra variants to run beside the
    headline (None = all)."""
    import numpy as np
    import torch
    import paper_2103_03348_b200 as hp
    from paper_2103_03348_b200 import synth
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    ev, tree, z0, ctx, tr, to = _setup_tree_problem(args, torch, hp, dev)
    n, M, K, W = ev.n, tree.n_tips, args.steps, args.warmup
    x, t, idx = to(ev.x), to(ev.t), to(ev.free_idx)
    s2, tau0, L, every = synth.TREE_SIGMA2, synth.TREE_TAU0, 20, 10
    eps, floor = args.hmc_step, 1.0
    pp = tr.precision_diag(s2, tau0)
    sampler = ClockSampler(0).start()

    def run_variant(cache, step, prior_prec):
        if cache == 3:   # the exact-zero-skipping variants need the plan of these events and hyperparameters
            ctx.skip_plan(x, t, ev.params)
        z, mass = to(z0.copy()), to(np.ones(M))
        nrm = to(synth.normals(args.seed, 500, (W + K) * M).reshape(W + K, M))
        uni = to(synth.uniforms(args.seed, 501, W + K))
        kw = dict(n_leapfrog=L, step=step, precond_every=every, mass=mass, mass_floor=floor, cache_background=cache,
                  prior_prec=prior_prec)
        e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        e0.record()
        ctx.hmc_run(tr, x, t, idx, z, 0.0, ev.params, s2, tau0, n_iter=W, normals=nrm[:W].contiguous(),
                    uniforms=uni[:W].contiguous(), **kw)
        e1.record()
        l0 = ctx.launch_count() + tr.launch_count()
        trace = ctx.hmc_run(tr, x, t, idx, z, 0.0, ev.params, s2, tau0, n_iter=K, normals=nrm[W:].contiguous(),
                            uniforms=uni[W:].contiguous(), n_refresh_done=(W + every - 1) // every, **kw)
        e2.record()
        torch.cuda.synchronize(dev)
        launches = ctx.launch_count() + tr.launch_count() - l0
        tr_h = trace.cpu().numpy()
        n_refresh = len([it for it in range(K) if it % every == 0])
        return {"seconds_per_iteration": e1.elapsed_time(e2) * 1e-3 / K, "accept_rate": float(tr_h[:, 3].mean()),
                "step": step, "preconditioner": "A + P (DESIGN R20)" if prior_prec is not None else "A (PAPER.md:143-145)",
                "log_posterior_last": float(tr_h[-1, 0]), "gpu_launches": int(launches),
                "gpu_launches_per_iteration": launches / K,
                "evals_per_s_implied": (K * L + n_refresh + 1) / (e1.elapsed_time(e2) * 1e-3)}

    # headline: the paper's method (every pair recomputed at every leapfrog step) with the paper's
    # preconditioner (the running average of the likelihood's Hessian diagonal alone); the time per
    # iteration does not depend on the step size, the acceptance rate does (DESIGN R20: this preconditioner needs a
    # far smaller step on a tree with very short branches)
    head = run_variant(0, args.hmc_step_paper, None)
    res_var = {"recompute_all_pairs__paper_preconditioner": head}
    for name, cache in (("recompute_all_pairs", 0), ("cached_background", 1), ("cached_kernel_matrix", 2),
                        ("skip_lists_recompute", 3), ("skip_lists_cached_background", 4),
                        ("sparse_kernel_matrix", 5)):
        if only is None or name + "__plus_prior_curvature" in only:
            res_var[name + "__plus_prior_curvature"] = run_variant(cache, eps, pp)
    if only is None or "sparse_kernel_matrix__paper_preconditioner" in only:
        res_var["sparse_kernel_matrix__paper_preconditioner"] = run_variant(5, args.hmc_step_paper, None)
    clocks = sampler.stop()
    res = {"metric": "hmc_seconds_per_iteration", "value": head["seconds_per_iteration"], "unit": "s/iteration",
           "n_gpus": 1, "steps": K, "warmup": W, "ms_per_step": head["seconds_per_iteration"] * 1e3,
           "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": "BASELINE.json configs[3]: N=23,422, M=1,610 (configs[2] inputs), HMC on z: 20 leapfrog "
                                  "steps per iteration, Hessian preconditioner refreshed every 10 iterations",
                      "n_events": n, "n_tips": M, "step": head["step"], "mass_floor": floor, "call": "hawkes_hmc_run",
                      "variant_of_value": "recompute_all_pairs__paper_preconditioner (cache_background = 0, prior_prec = NULL)",
                      "l2": "working set (0.75 MB) is L2-resident by design: every evaluation re-reads the same events",
                      "parallelism": "1 GPU"},
           "variants": res_var, "gpu_launches": head["gpu_launches"], "clocks": clocks,
           "e2e": {"value": head["seconds_per_iteration"], "unit": "s/iteration", "h2d_bytes_per_step": 0,
                   "d2h_bytes_per_step": 32, "note": "the chain state lives on the device; per iteration only the 4-double "
                   "trace row leaves it (read back once at the end)"}}
    if not args.no_cpu_baseline:
        # the oracle's leapfrog (oracle/hmc.py on the likelihood and prior oracles): a bounded sample of one trajectory
        import oracle
        from oracle import hmc as ohmc
        from oracle import tree as otree
        threads = oracle.max_threads()
        V = otree.vg(tree.parent, tree.branch, M, tau0)
        target = ohmc.hawkes_target(ev.x, ev.t, ev.free_idx, 0.0, ev.params, V, s2, threads=threads)
        lp0, g0, _ = target(z0, False)
        n_steps = 4
        t0_ = time.perf_counter()
        ohmc.leapfrog(target, z0, np.sqrt(np.ones(M)) * synth.normals(args.seed, 500, M), g0, np.ones(M),
                      args.hmc_step_paper, n_steps)
        secs = time.perf_counter() - t0_
        res["cpu_baseline"] = {"value": secs * L / n_steps, "unit": "s/iteration", "cores": threads, "kind": "oracle",
                               "sample": f"{n_steps} of the {L} leapfrog steps of one trajectory (oracle/hmc.py: full "
                                         f"likelihood oracle + dense Cholesky prior oracle per step), {secs:.1f} s on "
                                         f"{threads} OpenMP threads, scaled by {L}/{n_steps}; the preconditioner refresh "
                                         f"(1 Hessian evaluation per 10 iterations) is left out"}
    return res


def run_config0(args) -> dict:
    """configs[0]: N = 1,000, log-lik, full gradient and Hessian -- hawkes_eval with every output (theta-diagonal, 6 x 6,
    N x 6 cross block) plus the dense theta-theta block; every output against the full oracle on the spot."""
    import numpy as np
    import torch
    import paper_2103_03348_b200 as hp
    from paper_2103_03348_b200 import synth
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    ev = synth.config(0, args.seed)
    to = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    x, t, th = to(ev.x), to(ev.t), to(ev.theta)
    ctx = hp.HawkesContext(ev.n, ev.dim, 0)
    out = ctx.eval(x, t, th, ev.params, hp.WANT_ALL)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    step = lambda: ctx.eval(x, t, th, ev.params, hp.WANT_ALL, out=out)
    _event_timed(torch, dev, step, args.warmup, flush)
    l0 = ctx.launch_count()
    ms = _event_timed(torch, dev, step, args.steps, flush)
    launches = ctx.launch_count() - l0
    dense_ms = _event_timed(torch, dev, lambda: ctx.hessian_theta_dense(x, t, th, ev.params), args.steps, flush)
    st = ctx.last_status()
    res = {"workload": "BASELINE.json configs[0]: N=1,000, log-lik + full gradient + Hessian (theta diagonal, 6x6, Nx6 cross block)",
           "call": "hawkes_eval(WANT_ALL)", "steps": args.steps, "warmup": args.warmup, "ms_per_step": statistics.median(ms),
           "evals_per_s": args.steps / (float(sum(ms)) * 1e-3), "gpu_launches_per_step": launches / args.steps,
           "dense_theta_block_ms": statistics.median(dense_ms), "device_status": int(st)}
    if not args.no_cpu_baseline:
        import oracle
        ref = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params, hess=True, cross=True, row_d1=True, threads=oracle.max_threads())
        rel = lambda g, o: float(np.max(np.abs(g.cpu().numpy().reshape(np.shape(o)) - o)) / np.max(np.abs(o)))
        res["parity_vs_full_oracle_max_rel_to_largest_entry"] = {
            "ll": abs(out.ll.item() - ref.ll) / abs(ref.ll), "grad_theta": rel(out.grad_theta, ref.grad_theta),
            "grad_hyper": rel(out.grad_hyper, ref.grad_hyper), "hess_theta_diag": rel(out.hess_theta_diag, ref.hess_theta_diag),
            "hess_hyper": rel(out.hess_hyper, ref.hess_hyper), "hess_cross_per_column": [
                rel(out.hess_cross[:, k], ref.hess_cross[:, k]) for k in range(6) if np.max(np.abs(ref.hess_cross[:, k])) > 0],
            "tolerance": 1e-10}
    ctx.close()
    return res


def other_configs(args) -> dict:
    """BASELINE.json configs[0], [2], [3] inside the default line (configs[1] is the line itself, configs[4] its `sweep`):
    the same measurements `--config 0 | 2 | 3` print on their own, with short step counts and without the oracle-timing legs."""
    sub = lambda **kw: argparse.Namespace(**{**vars(args), **kw})
    c0 = run_config0(sub(steps=20, warmup=5))
    post = run_posterior(sub(steps=20, warmup=5, no_cpu_baseline=True))
    fastest = "sparse_kernel_matrix__plus_prior_curvature"
    hmc = run_hmc(sub(steps=200, warmup=5, no_cpu_baseline=True), only=(fastest,))
    pick = lambda d, keys: {k: d[k] for k in keys if k in d}
    return {
        "configs[0]": c0,
        "configs[2]": {**pick(post, ("metric", "value", "unit", "steps", "warmup", "ms_per_step", "gpu_launches", "breakdown_ms",
                                     "out3", "clocks")),
                       "workload": post["config"]["workload"], "call": post["config"]["call"], "e2e": post["e2e"],
                       "parity": "tests/test_tree_gpu.py::test_posterior_z_config2_full_size (full likelihood oracle + dense Cholesky prior oracle)"},
        "configs[3]": {**pick(hmc, ("metric", "value", "unit", "steps", "warmup", "higher_is_better", "clocks")),
                       "workload": hmc["config"]["workload"], "call": hmc["config"]["call"],
                       "variant_of_value": hmc["config"]["variant_of_value"],
                       "paper_method": hmc["variants"]["recompute_all_pairs__paper_preconditioner"],
                       "fastest_exact_variant": {"name": fastest, **hmc["variants"][fastest]},
                       "parity": "tests/test_hmc_gpu.py (oracle trajectory incl. accept decisions; full-size single iteration)"}}


def workload_of(args):
    from paper_2103_03348_b200 import synth
    rank, world, _ = dist_env()
    if world > 1 and args.impl != "reference" and not getattr(args, "shard", False):   # sharded: the same events on every rank
        args = argparse.Namespace(**{**vars(args), "seed": replica_seed(args.seed, rank)})
    if args.n is not None:
        ev = synth.make_events(args.n, args.seed)
        return ev, f"BASELINE.json configs[4] generator at N={args.n} (seed {args.seed})"
    if args.config == 0:
        return synth.config(0, args.seed), f"BASELINE.json configs[0]: N=1,000 (seed {args.seed})"
    if args.config == 1:
        return synth.config(1, args.seed), (f"BASELINE.json configs[1]: N=23,422 events, 60 clusters, 1,610 non-unit "
                                            f"theta, params (0.3,10,14,0.7,1,1/3), seed {args.seed}")
    raise SystemExit("bench.py times configs[1] (default), configs[0] or --n N for the scaling sweep")


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="timed steps (default 50; --config 3: 200 HMC iterations)")
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--n", type=int, default=None, help="scaling sweep: N events from the same generator")
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--extras", action="store_true", help="also time the Hessian and the theta-only evaluation")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sweep", action="store_true", help="skip the configs[4] sizes in the default line")
    ap.add_argument("--shard", action="store_true",
                    help="N > 1: cut ONE evaluation across the ranks (hawkes_shard_*) instead of running N replicas")
    ap.add_argument("--cpu-budget", type=float, default=15.0, help="seconds of oracle work for cpu_baseline")
    ap.add_argument("--hmc-step", type=float, default=0.2, help="leapfrog step size of --config 3 with the prior curvature in the mass (R20)")
    ap.add_argument("--hmc-step-paper", type=float, default=0.01, help="step size of --config 3 with the paper's preconditioner")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    if args.steps is None:
        args.steps = 200 if (args.config == 3 and args.n is None) else 50
    rank, world, _ = dist_env()
    if args.impl == "reference":
        if rank != 0:
            return 0
        ev, workload = workload_of(args)
        print(json.dumps(run_reference(args, ev, workload)), flush=True)
        return 0
    if world != args.gpus and world > 1:
        args.gpus = world
    if args.config in (2, 3) and args.n is None:
        if rank == 0:
            print(json.dumps(run_posterior(args) if args.config == 2 else run_hmc(args)), flush=True)
        return 0
    ev, workload = workload_of(args)
    res = run_b200(args, ev, workload)
    if rank == 0:
        print(json.dumps(res), flush=True)
    return 0


if __name__ == "__main__":
    sys.exit(main())
