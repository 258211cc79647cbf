#!/usr/bin/env python
"""bench.py -- headline measurement of the ILE hot path on B200 (BASELINE.json).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A *step* is one pass of the whole hot path over one batch: one integrator iteration of
BASELINE.json configs[1] (3 detectors, 21 modes, 820-bin Q, 400 time bins, AC with 100-bin
marginals, 2^20 samples): draw -> antenna/Y_lm/coefficients/quadratic term -> fused lnL over the
time grid -> time marginalisation -> weight reduction -> AC update.  The sampler is reset every 10
steps, as the config's 10-iteration runs are.  Metric: extrinsic lnL evaluations per second,
counted as samples x time bins.

`value`   device-resident: Q/U/V already in HBM; CUDA events around the K steps.
`e2e`     the same step through the C ABI from HOST buffers: every step loads that intrinsic
          point's Q/U/V from pinned host memory (ile_load_quv: host -> device copy + repack), runs
          the iteration and reads the ile_result struct back to the host.
`roofline` the fused lnL kernel (steps 4-6): algorithmic flop (289.4 per sample-bin, DESIGN.md
          section 6) / its device time, timed live with CUDA events on the launching stream,
          against the FP64 peak measured in the same process by the library's register-resident
          DFMA / DMMA chain probes (bound "alu": the path is FP64-arithmetic bound, not HBM bound).
`cpu_baseline` the oracle (oracle/, numpy fp64, as it stands) on the host cores, one AC iteration
          of the same config on a bounded sample of 2^14 samples.

N > 1 (torchrun): the path does not communicate; each rank runs the same step on its own
intrinsic point ("replicas", weak scaling); value = total sample-bins / max-over-ranks time.
"""
from __future__ import annotations

import argparse
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
CFG = 2


def flop_per_unit(K, M, N_t):
    """Algorithmic flop of the fused kernel per (sample, time bin): contraction +
    interpolation 2 K (2M + 2), plus the U/V quadratic term (K 6 M(M+1)/2 FMA + 8 M(M+1)/2 flop per
    sample) spread over the N_t bins.  264 + 25.4 = 289.4 at K = 3, M = 21, N_t = 400."""
    pairs = M * (M + 1) // 2
    return 2.0 * K * (2 * M + 2) + (2.0 * K * 6 * pairs + 8.0 * pairs) / N_t

ORACLE_SAMPLE_N = 1 << 14
NCU_TRAFFIC_BYTES = 550.80e6 + 15.23e6   # profiles/r1_fused_kernel.md (algorithmic: 512 B in + 8 B out per sample = 545 MB)


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
def oracle_rate(n_samples, steps=1, warmup=0):
    """The oracle as it stands: AC iterations of config 2 on `n_samples` samples per step."""
    from oracle.ile import IleProblem, iteration
    from oracle.integrators import make_integrator
    from synth import make_problem
    prob = make_problem(CFG, N=n_samples, n_iter=1)
    op = IleProblem(prob)
    oo = {k: v for k, v in prob.opts.items() if k != "seed"}
    integ = make_integrator(prob.kind, prob.lo, prob.hi, prob.opts["seed"], **oo)
    for g in range(warmup):
        iteration(op, integ, n_samples, g)
    c0, t0 = time.process_time(), time.perf_counter()
    for g in range(steps):
        iteration(op, integ, n_samples, warmup + g)
    wall, cpu = time.perf_counter() - t0, time.process_time() - c0
    cores = max(1, int(round(cpu / wall)))
    return n_samples * prob.N_t * steps / wall, wall / steps, cores, prob


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n = 1 << 11
    rate, sec, cores, prob = oracle_rate(n, steps=args.steps, warmup=min(args.warmup, 1))
    sample = f"config {CFG} shapes (K=3, M=21, N_t={prob.N_t}, AC), {n} samples per step instead of {1 << 20}"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": _config_dict(prob, n),
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def _config_dict(prob, N):
    return {"workload": f"BASELINE.json configs[1]: {prob.K} detectors, {prob.M} modes (l<=4), N_Q={prob.N_Q}, N_t={prob.N_t}, "
                        f"AC 100 bins, {N} samples per iteration, sampler reset every 10 iterations",
            "samples_per_step": N, "time_bins": prob.N_t, "integrator": prob.kind, "d": prob.d,
            "l2": "per-step working set (draws, per-sample records and Y tiles, ~0.6 GB) exceeds the 126 MB L2; no explicit flush"}


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


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2505_11655_b200 import Ile, Integrator, RESULT_DTYPE
    from synth import make_problem

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    dev = f"cuda:{local}"

    prob = make_problem(CFG, P=1)
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
        peak = max(peak_dfma, peak_dmma)
        # oracle on the host cores (rank 0, N = 1 only), bounded sample
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            rate, sec, cores, _ = oracle_rate(ORACLE_SAMPLE_N)
            cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                   "sample": f"one AC iteration of config {CFG} on {ORACLE_SAMPLE_N} samples x {prob.N_t} bins ({sec:.1f} s)"}
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": _config_dict(prob, N),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": e2e_ms / args.steps},
            "gpu_launches": int(launches),
            "clocks": clk,
            "roofline": {"bound": "alu", "kernel": "lnl_fused2_kernel", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                         "frac": achieved / peak, "traffic": NCU_TRAFFIC_BYTES,
                         "traffic_note": "dram bytes read+written per launch of this kernel, ncu --set full, profiles/r1_fused_kernel.md", "kernel_ms": k_avg_ms, "kernel_launches": int(k_n),
                         "kernel_share_of_step": k_ms / ms, "peak_source": "measured in-process: max(DFMA chain, DMMA chain)",
                         "peak_dfma": peak_dfma, "peak_dmma": peak_dmma, "flop_per_unit": fpu},
            "cpu_baseline": cpu,
            "check": {"ln_integral_last": float(last["ln_integral"]), "n_eff_last": float(last["n_eff"]),
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
    print(json.dumps({"metric": "Q/U/V precompute (Eq. 6a-c)", "value": P / (ms * 1e-3), "unit": "intrinsic points/s", "ms_per_step": ms,
                      "steps": args.steps, "warmup": args.warmup, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": f"P={P} points, K={K}, M={len(ell)}, N_f={N_f}, N_Q={N_Q}, spectra resident in HBM"}}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--precompute", action="store_true", help="time the Q/U/V precompute instead of the hot path (side measurement)")
    args = ap.parse_args()
    if args.precompute:
        run_precompute(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
