#!/usr/bin/env python
"""bench.py -- headline measurement of the ILE hot path on B200 (BASELINE.json).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-per-config] [--no-cpu-baseline]

A *step* is one pass of the whole hot path over one batch: one integrator iteration of the largest
single-GPU configuration, BASELINE.json configs[2] (3 detectors, 21 modes, 820-bin Q, 400 time bins, source at
SNR 100, AV adaptive-volume integrator, 2^22 samples): draw -> antenna/Y_lm -> coefficients and quadratic term ->
fused lnL over the time grid (contraction on the tensor cores) -> time marginalisation -> weight reduction -> AV
update.  The sampler is reset every 20 steps, as the config's 20-iteration runs are.  Metric: extrinsic lnL
evaluations per second, counted as samples x time bins.

`value`    device-resident: Q/U/V already in HBM; CUDA events around the K steps.
`e2e`      the same step through the C ABI from HOST buffers: every step loads that intrinsic point's Q/U/V from
           pinned host memory (ile_load_quv: host -> device copy + repack + digit image), runs the iteration and
           reads the ile_result struct back to the host.
`roofline` the fused lnL kernel (steps 3-6): algorithmic flop (289.4 per sample-bin) / its
           device time, timed live with CUDA events on the launching stream, against the FP64 peak measured in
           the same process by the library's register-resident DFMA / DMMA chain probes.  The kernel's contraction
           runs on the int8 tensor path (exactly), so the fraction of the FP64 peak can pass 1.
`per_config` configs 2-5 of SURVEY 8(d) at their full BASELINE.json sizes through ile_integrator_run (config 4:
           all 512 intrinsic points): ms per iteration, fused-kernel ms, flop per unit, fraction, n_eff / N.
`cpu_baseline` the oracle (oracle/, numpy fp64, as it stands) on the host cores: one AV iteration of the same
           config on a bounded sample, sample slices fanned out over the cores with multiprocessing.

N > 1 (torchrun): the path does not communicate; rank r runs the same step on intrinsic point r of the config
("replicas", weak scaling); value = total sample-bins / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "extrinsic lnL evals/s (samples x time bins)"
UNIT = "sample-bins/s"
CFG = 3                                   # BASELINE.json configs[2]: the largest single-GPU configuration
KERNEL = "lnl_split_kernel (tcgen05.mma kind::i8 contraction + FP64 epilogue)"


def flop_per_unit(K, M, N_t):
    """Algorithmic flop of the fused kernel per (sample, time bin): contraction +
    interpolation 2 K (2M + 2), plus the U/V quadratic term (K 6 M(M+1)/2 FMA + 8 M(M+1)/2 flop per
    sample) spread over the N_t bins.  264 + 25.4 = 289.4 at K = 3, M = 21, N_t = 400.  (Steps 1-3, which the
    kernel now also does - SURVEY 8(d): 45 K + 15 M + 6 K M flop per sample, 2 more per bin - are not counted.)"""
    pairs = M * (M + 1) // 2
    return 2.0 * K * (2 * M + 2) + (2.0 * K * 6 * pairs + 8.0 * pairs) / N_t


ORACLE_SAMPLE_N = 1 << 14


def ncu_traffic(cfg):
    """dram bytes read + written per launch of the fused kernel on config `cfg`, from the committed ncu summary
    profiles/r2_traffic.csv (one `ncu --set full` capture per config; the command is in profiles/r2_traffic.md)."""
    try:
        with open(os.path.join(ROOT, "profiles", "r2_traffic.csv")) as fh:
            for row in csv.DictReader(fh):
                if int(row["config"]) == cfg:
                    return float(row["dram_bytes_read"]) + float(row["dram_bytes_write"])
    except (OSError, KeyError, ValueError):
        pass
    return None


# ------------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                          "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, reasons, power = [], None, set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 9:
                continue
            try:
                sm.append(float(r[1]))
                smax = float(r[2])
                power.append(float(r[3]))
            except ValueError:
                continue
            for n, v in zip(names, r[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax, "reasons": sorted(reasons),
                "power_w_max": max(power) if power else None, "samples": len(sm)}


# ------------------------------------------------------------------------------- oracle arm
_ORACLE = {}


def _oracle_worker_init(cfg):
    from oracle.ile import IleProblem
    from synth import make_problem
    prob = make_problem(cfg, N=1, n_iter=1)
    _ORACLE["op"] = IleProblem(prob)


def _oracle_lnL_slice(z):
    return _ORACLE["op"].lnL_z(z)


def cpu_model():
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_rate(n_samples, steps=1, warmup=0, procs=None):
    """The oracle as it stands: iterations of config CFG (draw, lnL, weights, reduction, sampler update) on `n_samples`
    samples per step.  The likelihood of the batch is evaluated on sample slices by `procs` worker processes (one per
    host core, SURVEY 8(d) timing protocol); draw, reduction and update run in the parent.  Only oracle/ code runs."""
    import multiprocessing as mp
    from oracle.ile import IleProblem
    from oracle.integrators import make_integrator
    from oracle.reduce import reduce_lnw
    from synth import make_problem
    procs = procs or os.cpu_count() or 1
    prob = make_problem(CFG, N=n_samples, n_iter=1)
    op = IleProblem(prob)
    oo = {k: v for k, v in prob.opts.items() if k != "seed"}
    integ = make_integrator(prob.kind, prob.lo, prob.hi, prob.opts["seed"], **oo)
    pool = mp.get_context("fork").Pool(procs, initializer=_oracle_worker_init, initargs=(CFG,)) if procs > 1 else None

    def one(g):
        z, ln_ps = integ.draw(n_samples, g)
        if pool is not None:
            parts = np.array_split(np.arange(n_samples), procs)
            lnL = np.concatenate(pool.map(_oracle_lnL_slice, [z[:, p] for p in parts]))
        else:
            lnL = op.lnL_z(z)
        with np.errstate(invalid="ignore"):
            lnw = lnL + op.ln_prior(z) - ln_ps
        lnw = np.where(np.isfinite(lnL), lnw, -np.inf)
        reduce_lnw(lnw)
        integ.update(z, lnw, None if integ.kind == "AV" else ln_ps)

    for g in range(warmup):
        one(g)
    t0 = time.perf_counter()
    for g in range(steps):
        one(warmup + g)
    wall = time.perf_counter() - t0
    if pool is not None:
        pool.close()
        pool.join()
    return n_samples * prob.N_t * steps / wall, wall / steps, procs, prob


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n = 1 << 12
    rate, sec, cores, prob = oracle_rate(n, steps=args.steps, warmup=min(args.warmup, 1))
    sample = (f"config {CFG} shapes (K={prob.K}, M={prob.M}, N_t={prob.N_t}, {prob.kind}), {n} samples per step instead of {prob.N}; "
              f"{cores} worker processes on {os.cpu_count()} host cores ({cpu_model()})")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": _config_dict(prob, n),
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def _config_dict(prob, N):
    return {"workload": f"BASELINE.json configs[{CFG - 1}]: {prob.K} detectors, {prob.M} modes (l<=4), N_Q={prob.N_Q}, N_t={prob.N_t}, "
                        f"{prob.kind} integrator in {prob.d} dimensions, {N} samples per iteration, sampler reset every {prob.n_iter} iterations"
                        + (" (source at SNR 100, peak lnL ~ 5000; AV with P_thr 0.999)" if CFG == 3 else ""),
            "samples_per_step": N, "time_bins": prob.N_t, "integrator": prob.kind, "d": prob.d,
            "l2": _l2_note(prob, N)}


def _l2_note(prob, N):
    # per-sample bytes an iteration touches: draws, ln p_s, lnL, ln w, ln prior, u_k, sort keys and indices (two buffers each)
    ws = N * (8 * prob.d + 4 * 8 + 32 + 2 * 12)
    if ws > 126e6:
        return f"per-step working set (draws, densities, weights, u_k, sort buffers: {ws / 1e6:.0f} MB) exceeds the 126 MB L2; no explicit flush"
    return (f"per-step working set {ws / 1e6:.0f} MB fits the 126 MB L2 and is not flushed: the run reuses the same buffers every "
            "iteration, as the production loop does; only the headline configuration is a cold-L2 number")


# ------------------------------------------------------------------------------- our arm
def max_over_ranks(values, world, device):
    """Every multi-GPU number is the maximum over ranks of the per-rank device time."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def aggregate_value(units_per_step_per_rank, steps, world, ms):
    """Whole-job throughput: replicas do not communicate, every rank processes its own units."""
    return world * units_per_step_per_rank * steps / (ms * 1e-3)


def rank_problem(cfg, rank):
    """Rank r works on intrinsic point r of the config (its own seeded Q/U/V; one event: shared network and D_ref)."""
    from synth import make_problem
    prob = make_problem(cfg, P=rank + 1)
    prob.Q, prob.U, prob.V, prob.P = prob.Q[rank:rank + 1].copy(), prob.U[rank:rank + 1].copy(), prob.V[rank:rank + 1].copy(), 1
    return prob


def measure_config(cfg, dev, peak):
    """One full BASELINE.json run of config `cfg` through ile_integrator_run (no host round-trip inside): every
    intrinsic point, every iteration, full batch size.  CUDA events around the run, fused-kernel time from the library."""
    import torch
    from paper_2505_11655_b200 import Ile, Integrator, RESULT_DTYPE
    from synth import make_problem
    prob = make_problem(cfg)
    ile = Ile(int(dev.split(":")[1]))
    ile.load_problem(prob)
    integ = Integrator.from_problem(ile, prob, max_batch=prob.N)
    P, n_iter, N = prob.P, prob.n_iter, prob.N
    out = integ.run(0, min(P, 2), n_iter, N)                            # warm-up: the first points
    torch.cuda.synchronize()
    ile.kernel_timing(True)
    l0 = ile.kernel_launches()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    out = integ.run(0, P, n_iter, N)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    launches = ile.kernel_launches() - l0
    k_ms, k_n = ile.kernel_time()
    ile.kernel_timing(False)
    res = np.frombuffer(out.cpu().numpy().tobytes(), dtype=RESULT_DTYPE).reshape(P, n_iter)
    units = float(P) * n_iter * N * prob.N_t
    fpu = flop_per_unit(prob.K, prob.M, prob.N_t)
    k_avg = k_ms / max(k_n, 1)
    frac = fpu * N * prob.N_t / (k_avg * 1e-3) / 1e12 / peak
    last = res[:, -1]
    integ.close()
    del ile
    torch.cuda.empty_cache()
    return {"config": cfg, "integrator": prob.kind, "points": P, "iterations": n_iter, "samples_per_iteration": N, "time_bins": prob.N_t,
            "ms_per_iteration": ms / (P * n_iter), "value": units / (ms * 1e-3), "fused_kernel_ms": k_avg, "fused_kernel_launches": int(k_n),
            "fused_kernel_share": k_ms / ms, "flop_per_unit": fpu, "frac": frac, "gpu_launches_per_iteration": launches / (P * n_iter),
            "traffic": ncu_traffic(cfg), "l2": _l2_note(prob, N),
            "check": {"n_eff_over_N_last": float(np.mean(last["n_eff"]) / N), "n_eff_cumulative_over_N": float(np.mean(last["cum_n_eff"] / last["cum_n_samples"])),
                      "ln_integral_last": float(last["ln_integral"][0]), "n_nonfinite": int(res["n_nonfinite"].sum())}}


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2505_11655_b200 import Ile, Integrator, RESULT_DTYPE

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    dev = f"cuda:{local}"

    prob = rank_problem(CFG, rank)
    N, n_iter = prob.N, prob.n_iter
    ile = Ile(local)
    ile.load_problem(prob)
    integ = Integrator.from_problem(ile, prob, max_batch=N)
    res_dev = torch.zeros(RESULT_DTYPE.itemsize, dtype=torch.uint8, device=dev)
    units_per_step = N * prob.N_t

    def step(g):
        if g % n_iter == 0:
            integ.reset()
        integ.step(0, N, g % n_iter, out=res_dev)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    # FP64 peaks, measured in this process before the timed region
    peak_dfma, peak_dmma = ile.fp64_peak(0), ile.fp64_peak(1)
    peak = max(peak_dfma, peak_dmma)
    peak_i8, peak_i8_summajor = ile.int8_mma_peak(0), ile.int8_mma_peak(1)      # the tensor path the contraction runs on

    for g in range(args.warmup):
        step(g)
    barrier()

    # ---- device-resident timing
    clocks = ClockSampler(local)
    clocks.start()
    ile.kernel_timing(True)
    launches0 = ile.kernel_launches()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for g in range(args.steps):
        step(args.warmup + g)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = ile.kernel_launches() - launches0
    k_ms, k_n = ile.kernel_time()
    ile.kernel_timing(False)
    clk = clocks.stop()
    last = np.frombuffer(res_dev.cpu().numpy().tobytes(), dtype=RESULT_DTYPE)[0]

    # ---- end to end from host buffers through the C ABI
    Qh = torch.from_numpy(np.ascontiguousarray(prob.Q).view(np.float64)).pin_memory()
    Uh = torch.from_numpy(np.ascontiguousarray(prob.U).view(np.float64)).pin_memory()
    Vh = torch.from_numpy(np.ascontiguousarray(prob.V).view(np.float64)).pin_memory()
    res_host = torch.zeros(RESULT_DTYPE.itemsize, dtype=torch.uint8).pin_memory()
    h2d = Qh.numel() * 8 + Uh.numel() * 8 + Vh.numel() * 8
    d2h = RESULT_DTYPE.itemsize

    def e2e_step(g):
        ile.load_quv_ptr(1, prob.N_Q, prob.fs, prob.t_Q0, Qh.data_ptr(), Uh.data_ptr(), Vh.data_ptr(), prob.D_ref)
        ile.set_time_grid(prob.t_lo, prob.dt, prob.N_t, prob.interp)
        step(g)
        res_host.copy_(res_dev, non_blocking=False)

    for g in range(min(args.warmup, 3)):
        e2e_step(g)
    barrier()
    t0 = time.perf_counter()
    for g in range(args.steps):
        e2e_step(g)
    barrier()
    e2e_s = time.perf_counter() - t0

    ms, e2e_ms = max_over_ranks([ms, e2e_s * 1e3], world, dev)

    if rank == 0:
        value = aggregate_value(units_per_step, args.steps, world, ms)
        e2e_value = aggregate_value(units_per_step, args.steps, world, e2e_ms)
        k_avg_ms = k_ms / max(k_n, 1)
        fpu = flop_per_unit(prob.K, prob.M, prob.N_t)
        achieved = fpu * units_per_step / (k_avg_ms * 1e-3) / 1e12
        integ.close()
        del ile
        torch.cuda.empty_cache()
        # configs 2-5 at full size (rank 0, N = 1 only)
        per_config = None
        if world == 1 and not args.no_per_config:
            per_config = [measure_config(c, dev, peak) for c in (2, 3, 4, 5)]
        # oracle on the host cores (rank 0, N = 1 only), bounded sample
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            rate, sec, cores, _ = oracle_rate(ORACLE_SAMPLE_N)
            cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "host_cores": os.cpu_count(), "cpu_model": cpu_model(),
                   "sample": f"one {prob.kind} iteration of config {CFG} on {ORACLE_SAMPLE_N} samples x {prob.N_t} bins ({sec:.1f} s), "
                             f"likelihood on sample slices in {cores} worker processes"}
        traffic = ncu_traffic(CFG)
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": _config_dict(prob, N),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": e2e_ms / args.steps},
            "gpu_launches": int(launches),
            "clocks": clk,
            "roofline": {"bound": "alu", "kernel": KERNEL, "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                         "frac": achieved / peak, "traffic": traffic,
                         "traffic_note": "dram bytes read + written per launch of this kernel on this config, one ncu --set full capture, "
                                         "profiles/r2_traffic.csv (command in profiles/r2_traffic.md)",
                         "kernel_ms": k_avg_ms, "kernel_launches": int(k_n), "kernel_share_of_step": k_ms / ms,
                         "peak_source": "FP64 peak measured in-process: max(DFMA chain, DMMA chain); the algorithmic FP64 flop of "
                                        "steps 3-6 over the kernel time.  The contraction itself runs exactly on the int8 tensor "
                                        "path (21 digit pairs, tcgen05.mma kind::i8), which is how the fraction can pass 1",
                         "peak_dfma": peak_dfma, "peak_dmma": peak_dmma, "flop_per_unit": fpu,
                         "tensor": {"kind": "tcgen05.mma kind::i8, 128x32x32, A from tensor memory", "peak_tops_measured": peak_i8,
                                    "peak_tops_sum_major_issue": peak_i8_summajor,
                                    "achieved_tops": 2.0 * 1056 * prob.K * units_per_step * (432.0 / prob.N_t) / (k_avg_ms * 1e-3) / 1e12,
                                    "note": "1056 K-bytes per (sample, stored bin, detector), 432 stored bins contracted for 400 time bins"}},
            "cpu_baseline": cpu,
            "per_config": per_config,
            "check": {"ln_integral_last": float(last["ln_integral"]), "n_eff_last": float(last["n_eff"]), "n_eff_over_N_last": float(last["n_eff"]) / N,
                      "samples_per_s": value / prob.N_t},
        }
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def run_precompute(args):
    """Side measurement: ile_precompute_quv on P = 16 intrinsic points, K = 3, M = 21, N_f = 32768,
    N_Q = 1024 stored bins, device-resident spectra; one JSON line, not the headline metric."""
    import torch
    from paper_2505_11655_b200 import Ile
    from synth import make_modes, make_network
    from synth.spectra import make_spectra
    P, K, N_f, N_Q, fs = 16, 3, 32768, 1024, 4096.0
    ell, m = make_modes(4)
    D, pos = make_network(K, np.random.Generator(np.random.Philox(99)))
    h, d, S, df = make_spectra(K, ell, m, N_f, fs, seed=1, P=1)
    ile = Ile(0)
    ile.set_network(D, pos, 0.0)
    ile.set_modes(ell, m)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    hd, dd, Sd = dev(np.repeat(h, P, axis=0)), dev(d), dev(S)
    call = lambda: ile.precompute_quv(hd, dd, Sd, df, 20.0, -(N_Q // 2) / fs, N_Q, 500.0)
    for _ in range(max(args.warmup, 1)):
        call()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        call()                                               # returns after the tables are installed (synchronous)
    ms = (time.perf_counter() - t0) * 1e3 / args.steps
    # roofline of the call (FP64 ALU bound): algorithmic flops of Eq. 6a-c as the kernels evaluate them:
    # U, V: two complex products and 4 K real multiply-adds per (bin, pair a <= b); Q: the product w conj(h) d, N_f / Mq
    # transforms of Mq = 2^ceil(log2 N_Q) points (5 Mq log2 Mq flops each) and one twiddled sum per stored bin
    M = len(ell)
    n_pairs = M * (M + 1) // 2
    Mq = 1 << int(np.ceil(np.log2(N_Q)))
    L = N_f // Mq
    flops_uv = P * N_f * n_pairs * (12 + 8 * K)
    flops_q = P * K * M * (L * 5 * Mq * int(np.log2(Mq)) + 8 * L * N_Q + 6 * N_f)
    peak_dfma = ile.fp64_peak(0)
    achieved = (flops_uv + flops_q) / (ms * 1e-3) / 1e12
    hbm_bytes = 2 * P * M * N_f * 16 + P * K * M * N_Q * 16          # h read by both kernels, Q written
    print(json.dumps({"metric": "Q/U/V precompute (Eq. 6a-c)", "value": P / (ms * 1e-3), "unit": "intrinsic points/s", "ms_per_step": ms,
                      "steps": args.steps, "warmup": args.warmup, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": f"P={P} points, K={K}, M={M}, N_f={N_f}, N_Q={N_Q}, spectra resident in HBM"},
                      "roofline": {"bound": "alu", "achieved": achieved, "peak": peak_dfma, "unit": "TFLOP/s", "frac": achieved / peak_dfma,
                                   "traffic": None, "flops_uv": flops_uv, "flops_q": flops_q,
                                   "peak_source": "FP64 FMA rate measured by ile_fp64_peak(0) in this run",
                                   "hbm_GBps": hbm_bytes / (ms * 1e-3) / 1e9,
                                   "note": "whole call (weights, U/V, Q, install with digit image, final synchronisation), wall clock"}}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the full-size runs of configs 2-5")
    ap.add_argument("--config", type=int, default=3, choices=[2, 3, 4, 5],
                    help="configuration of SURVEY 8(d) the step is taken from (default 3 = BASELINE.json configs[2], the headline; "
                         "the others are for profiling one configuration alone)")
    ap.add_argument("--precompute", action="store_true", help="time the Q/U/V precompute instead of the hot path (side measurement)")
    args = ap.parse_args()
    global CFG
    CFG = args.config
    if args.precompute:
        run_precompute(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
