#!/usr/bin/env python
"""bench.py - throughput of the BIFROST direct-summation hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config 4|5]

One STEP is one pass of the whole hot path over the workload:
bifrost_acc -> bifrost_grad -> bifrost_dtmin -> bifrost_pn1, all particles active.
Workload at N=1 GPU: BASELINE.json configs[3] ("config4": Plummer N = 2^20, Kroupa masses,
central IMBH + 100 stellar BHs, eps = 0, c = 1e4) - the configuration the metric
"... (acc+FSI grad) at N=1e6" is quoted on.  `--config 5` times the N = 2^21 acc+grad
peak-throughput case instead (no velocities/BHs in that config: dtmin/pn1 are skipped).

Metric: fp64 pair interactions/s for acc + FSI grad = n_sink * n_src / (t_acc + t_grad), one
interaction = one ordered (sink, source) pair evaluated in one pass.
`ms_per_step` is the whole step (all four calls); `passes` lists every call's own time.

Multi-GPU (torchrun, one rank per GPU; strong scaling, total work fixed): the PAIR work of acc and grad is
sharded across ranks (Context.set_shard: every rank evaluates its blocks of the unordered pairs and holds a partial
sum for every particle), with one NCCL all-reduce of double[N][3] after each of the two passes; dtmin is sharded
over sinks (no exchange).

--impl reference times the CPU oracle (oracle/, unmodified) on the host cores on a bounded
sample of the same workload and prints the same JSON line with "impl": "reference".
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

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fp64 pair interactions/s (acc+FSI grad) at N=1e6; % of B200 FP64 peak"
UNIT = "interactions/s"

# EXECUTED FP64-pipe instructions / flops (FMA = 2, ADD/MUL = 1) per INTERACTION (= one ordered (sink, source) pair
# delivered) of the kernels' inner loops (cross-checked against ncu's source page, profiles/).
#   plain kernels (sinks != sources, or a sharded sink range): every ordered pair is evaluated.
#   symmetric kernels (one list on both sides, all-active): every UNORDERED pair is evaluated once - acc 20 + 4.5/8
#   (source-side warp reduction, 8 sinks per thread) = 20.56 instructions / 32.6 flops per unordered pair,
#   grad 33 + 4.5/6 = 33.75 / 52.75 - i.e. half of that per interaction.
#   dtmin: 17 instructions in the hot path (7 DADD + 6 DFMA + 4 DMUL = 23 flops: keys from the unrefined rsqrt seed; the
#   refinement and the exact time-steps run in the rarely taken branch only).
#   Same-list dtmin evaluates every unordered pair once too (both keys are symmetric): 17 / 23 per unordered pair.
FP64_INSTR = {"plain": {"acc": 15, "grad": 28, "dtmin": 17}, "sym": {"acc": 20.5625 / 2, "grad": 33.75 / 2, "dtmin": 17 / 2}}
FP64_FLOPS = {"plain": {"acc": 24, "grad": 44, "dtmin": 23}, "sym": {"acc": 32.5625 / 2, "grad": 52.75 / 2, "dtmin": 23 / 2}}
# SURVEY.md 8(d)'s budget for the minimal ONE-SIDED sequence: flops per ordered pair.  Against it the symmetric
# kernels deliver more interactions than the executed flops alone would ("work-equivalent" fraction, may exceed 1).
SURVEY_8D_FLOPS = {"acc": 26, "grad": 42}
# B200 FP64 ALU peak derived from unit counts and clocks (no fp64 entry in MEASURED_PEAKS.json):
# 148 SMs x 64 FP64 lanes/clk/SM x 2 flop x 1.965 GHz (clocks.max.sm) = 37.2 TFLOP/s.
FP64_LANES_PER_SM = 64


def fp64_peak_tflops(num_sms: int = 148, sm_max_mhz: float = 1965.0) -> float:
    return num_sms * FP64_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200", "-i",
                 str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([t.strip() for t in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); smax.append(float(r[1])); power.append(float(r[2]))
            except ValueError:
                continue
            for name, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def make_workload(cfg: int, n: int = 0):
    from paper_2210_02472_b200 import workloads as W
    return W.CONFIGS[cfg](n=n) if n else W.CONFIGS[cfg]()


def workload_name(cfg: int, n: int) -> str:
    full = {4: 1 << 20, 5: 1 << 21}[cfg]
    if n != full:
        return f"config{cfg} recipe at a REDUCED N={n} (profiling aid, not the benchmark configuration)"
    return {4: f"config4: Plummer N=2^20={n}, Kroupa IMF, IMBH 1e-3 M + 100 stellar BHs, eps=0, c=1e4, all active; "
               "acc + FSI grad + dtmin + PN1.0",
            5: f"config5: Plummer N=2^21={n}, Kroupa IMF, eps=1e-5, all active; acc + FSI grad"}[cfg]


# --------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle, as it stands, on the host cores
# --------------------------------------------------------------------------------------

def oracle_sample(w, n_sample_sinks: int, seed: int = 777):
    """Time oracle acc + grad for a seeded sample of sinks against ALL sources.  Each sink's
    sum is independent, so the sample's rate (pairs/s) is the full problem's rate."""
    import oracle
    rng = np.random.default_rng(seed)
    sinks = np.sort(rng.choice(w.n, size=min(n_sample_sinks, w.n), replace=False)).astype(np.int32)
    fake_acc = np.ascontiguousarray(w.vel)      # any [n][3] field: the cost does not depend on its values
    t0 = time.perf_counter()
    oracle.acc(w.pos, w.mass, w.G, w.eps, sink_idx=sinks)
    t1 = time.perf_counter()
    oracle.grad(w.pos, w.mass, fake_acc, w.G, w.eps, sink_idx=sinks)
    t2 = time.perf_counter()
    pairs = float(sinks.shape[0]) * w.n
    return {"pairs": pairs, "t_acc": t1 - t0, "t_grad": t2 - t1, "n_sinks": int(sinks.shape[0])}


def cpu_baseline(w, n_sample_sinks: int):
    import oracle
    s = oracle_sample(w, n_sample_sinks)
    return {"value": s["pairs"] / (s["t_acc"] + s["t_grad"]), "unit": UNIT, "cores": oracle.n_threads(), "kind": "oracle",
            "sample": f"{s['n_sinks']} seeded sinks x all {w.n} sources, acc then grad "
                      f"({s['pairs']:.3g} pairs per pass; acc {s['t_acc']:.2f} s, grad {s['t_grad']:.2f} s)"}


def cpu_fast_baseline(w, n_sample_sinks: int):
    """the oracle is deliberately slow (compensated sums, -O2, IEEE sqrt + division per pair), so the
    GPU/oracle ratio flatters the GPU.  This times a plain restatement (oracle/cpu_fast.c: uncompensated sums,
    -O3 -mavx2 -mfma, vectorised over sources, OpenMP over sinks; pinned to the oracle at 1e-12 in
    tests/test_oracle_cpu_fast.py) on the same seeded sample.  Context only - neither the parity oracle nor a target."""
    import oracle
    from oracle import cpu_fast
    cpu_fast.build()
    rng = np.random.default_rng(777)
    sinks = np.sort(rng.choice(w.n, size=min(n_sample_sinks, w.n), replace=False)).astype(np.int32)
    fake_acc = np.ascontiguousarray(w.vel)
    cpu_fast.acc(w.pos, w.mass, w.G, w.eps, sinks[:64])            # warm-up (thread pool, page faults)
    t0 = time.perf_counter()
    cpu_fast.acc(w.pos, w.mass, w.G, w.eps, sinks)
    t1 = time.perf_counter()
    cpu_fast.grad(w.pos, w.mass, fake_acc, w.G, w.eps, sinks)
    t2 = time.perf_counter()
    pairs = float(sinks.shape[0]) * w.n
    return {"value": pairs / (t2 - t0), "unit": UNIT, "cores": oracle.n_threads(), "kind": "plain restatement, -O3 AVX2+FMA",
            "sample": f"{sinks.shape[0]} seeded sinks x all {w.n} sources, acc then grad (acc {t1 - t0:.2f} s, grad {t2 - t1:.2f} s)"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    oracle.build()
    w = make_workload(args.config, args.n)
    n_sinks = args.ref_sinks
    for _ in range(args.warmup):
        oracle_sample(w, max(8, n_sinks // 8))
    tot_pairs, tot_t, tot_wall = 0.0, 0.0, 0.0
    for k in range(args.steps):
        t0 = time.perf_counter()
        s = oracle_sample(w, n_sinks, seed=777 + k)
        tot_wall += time.perf_counter() - t0
        tot_pairs += s["pairs"]
        tot_t += s["t_acc"] + s["t_grad"]
    value = tot_pairs / tot_t
    sample = f"each step: {n_sinks} seeded sinks x all {w.n} sources, acc then grad ({n_sinks * w.n:.3g} pairs per pass)"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot_wall / max(1, args.steps), "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config, w.n), "reference_sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.n_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# --------------------------------------------------------------------------------------
# the CUDA arm
# --------------------------------------------------------------------------------------

def run_cuda(args):
    import torch
    import torch.distributed as dist
    from paper_2210_02472_b200 import sharding
    from paper_2210_02472_b200.binding import Context

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    w = make_workload(args.config, args.n)
    n = w.n
    full_path = args.config == 4
    ctx = Context(n)
    pos, vel, mass = (torch.from_numpy(x).to(dev) for x in (w.pos, w.vel, w.mass))
    bh = torch.from_numpy(w.bh_idx).to(dev) if full_path else None
    b, e = sharding.sink_slice(n, rank, world)
    sinks = None if world == 1 else torch.arange(b, e, dtype=torch.int32, device=dev)
    n_loc = e - b
    acc = torch.zeros((n, 3), dtype=torch.float64, device=dev)
    grad = torch.zeros((n, 3), dtype=torch.float64, device=dev)
    dts = (torch.full((n,), float("inf"), dtype=torch.float64, device=dev),
           torch.full((n,), float("inf"), dtype=torch.float64, device=dev),
           torch.full((n,), -1, dtype=torch.int32, device=dev), torch.full((n,), -1, dtype=torch.int32, device=dev))
    apn = torch.empty((n, 3), dtype=torch.float64, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)        # > L2 (126 MB)
    names = ["acc", "exchange_acc", "grad", "exchange_grad", "dtmin", "pn1"]
    if world > 1:
        ctx.set_shard(rank, world)                       # acc / grad: this rank's blocks of the unordered pairs
    ev = {k: [torch.cuda.Event(enable_timing=True) for _ in range(2)] for k in names}

    def step(timed: bool):
        """One pass of the whole hot path; returns per-call device times in ms."""
        flush.fill_(1)                                   # L2 flush, outside the timed events
        rec = {}

        def timed_call(name, fn):
            ev[name][0].record()
            fn()
            ev[name][1].record()

        timed_call("acc", lambda: ctx.acc(pos, mass, w.G, w.eps, out=acc))
        if world > 1:                                    # partial sums of every rank -> the accelerations (the exchange step)
            timed_call("exchange_acc", lambda: sharding.allreduce_sum(acc))
        timed_call("grad", lambda: ctx.grad(pos, mass, acc, w.G, w.eps, out=grad))
        if world > 1:
            timed_call("exchange_grad", lambda: sharding.allreduce_sum(grad))
        if full_path:
            timed_call("dtmin", lambda: ctx.dtmin(pos, vel, mass, w.G, w.eta_ff, w.eta_fb, sinks, None, out=dts))
            # PN1.0 is BH x N work (2e8 pairs): every rank evaluates it redundantly (it is < 0.1 % of a step)
            timed_call("pn1", lambda: ctx.pn1(pos, vel, mass, bh, w.G, w.c, out=apn))
        torch.cuda.synchronize()
        for name in names:
            if name.startswith("exchange") and world == 1:
                continue
            if name in ("dtmin", "pn1") and not full_path:
                continue
            rec[name] = ev[name][0].elapsed_time(ev[name][1])
        return rec

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step(False)
    sampler = ClockSampler(local_rank)
    barrier()
    sampler.start()
    launches0 = ctx.launch_count
    t_wall0 = time.perf_counter()
    recs = [step(True) for _ in range(args.steps)]
    barrier()
    t_wall = time.perf_counter() - t_wall0
    launches = ctx.launch_count - launches0
    clocks = sampler.stop()

    keys = list(recs[0].keys())
    mean_ms = {k: sum(r[k] for r in recs) / len(recs) for k in keys}
    step_ms = sum(mean_ms.values())
    t = torch.tensor([step_ms, mean_ms["acc"] + mean_ms["grad"] + mean_ms.get("exchange_acc", 0.0)
                      + mean_ms.get("exchange_grad", 0.0)] + [mean_ms[k] for k in keys],
                     dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)          # max over ranks
    t = t.cpu().tolist()
    step_ms, accgrad_ms = t[0], t[1]
    mean_ms = dict(zip(keys, t[2:]))
    value = float(n) * n / (accgrad_ms * 1e-3)            # whole job: all ranks' sinks x all sources

    # ---- end-to-end through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if rank == 0 or world > 1:
        def pinned(a):
            tns = torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
            return tns.numpy()
        hpos, hvel, hmass = pinned(w.pos), pinned(w.vel), pinned(w.mass)
        hsinks = None if world == 1 else np.arange(b, e, dtype=np.int32)
        hacc = pinned(np.zeros((n, 3)))
        hgrad = pinned(np.zeros((n, 3)))
        e2e_steps = max(1, min(args.steps, args.e2e_steps))
        t_ag, t_all = 0.0, 0.0
        if world > 1:
            d_pos, d_mass = torch.empty_like(pos), torch.empty_like(mass)
            t_pos, t_mass = torch.from_numpy(hpos), torch.from_numpy(hmass)
            t_acc_rows, t_grad_rows = torch.from_numpy(hacc[b:e]), torch.from_numpy(hgrad[b:e])
        for it in range(1 + e2e_steps):                   # first iteration = warm-up (allocates the mirrors)
            barrier()
            t0 = time.perf_counter()
            if world == 1:
                ctx.acc_host(hpos, hmass, w.G, w.eps, None, None, out=hacc)
                ctx.grad_host(hpos, hmass, hacc, w.G, w.eps, None, None, out=hgrad)
            else:
                # sharded: inputs from pinned host memory, the two all-reduces stay on the device (NCCL), this rank's
                # slice of the result rows back to the host - no device -> host -> device bounce around a collective
                d_pos.copy_(t_pos, non_blocking=True); d_mass.copy_(t_mass, non_blocking=True)
                ctx.acc(d_pos, d_mass, w.G, w.eps, out=acc)
                sharding.allreduce_sum(acc)
                ctx.grad(d_pos, d_mass, acc, w.G, w.eps, out=grad)
                sharding.allreduce_sum(grad)
                t_acc_rows.copy_(acc[b:e], non_blocking=True); t_grad_rows.copy_(grad[b:e], non_blocking=True)
                torch.cuda.synchronize()
            t1 = time.perf_counter()
            if full_path:
                ctx.dtmin_host(hpos, hvel, hmass, w.G, w.eta_ff, w.eta_fb, hsinks, None)
                ctx.pn1_host(hpos, hvel, hmass, w.bh_idx, w.G, w.c)
            t2 = time.perf_counter()
            if it > 0:
                t_ag += t1 - t0
                t_all += t2 - t0
        tt = torch.tensor([t_ag / e2e_steps, t_all / e2e_steps], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        tt = tt.cpu().tolist()
        idx_b = 0 if world == 1 else 4 * n_loc
        h2d = ((32 * n) + (56 * n) if world == 1 else 32 * n) + ((56 * n + idx_b) + (56 * n + 4 * len(w.bh_idx)) if full_path else 0)
        d2h = 24 * n_loc * 2 + ((24 * n_loc) + 24 * n if full_path else 0)
        e2e = {"value": float(n) * n / tt[0], "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "ms_per_step": 1e3 * tt[1], "steps": e2e_steps,
               "how": ("bifrost_*_host entry points on pinned host arrays: H2D copies, kernels, D2H copies per call; "
                       "value = N^2 / host wall time of acc_host + grad_host") if world == 1 else
                      ("per rank: pinned-host -> device copies of pos / mass, bifrost_acc on the rank's pair blocks, NCCL "
                       "all-reduce of acc on the device, bifrost_grad, all-reduce of grad, the rank's slice of the acc / grad "
                       "rows back to pinned host memory; value = N^2 / max over ranks of that wall time")}

    if rank == 0:
        num_sms = torch.cuda.get_device_properties(dev).multi_processor_count
        peak = fp64_peak_tflops(num_sms, clocks.get("sm_max_mhz") or 1965.0)
        # measured FP64-pipe rates of a register-only kernel (outside the timed region; ~0.3 s each)
        probe = {}
        if not args.no_fp64_probe:
            for mix, name in ((0, "dfma"), (1, "acc_mix"), (2, "dfma_3_distinct_operands"), (3, "dfma_accumulate_pattern")):
                ms, rate = ctx.fp64_probe(mix=mix, iters=(1 << 15) if mix < 2 else (1 << 16), ctas_per_sm=32)
                probe[name] = {"ms": ms, "lane_instr_per_s": rate, "frac_of_derived_pipe_peak": rate / (peak * 1e12 / 2)}
        pairs_rank = float(n) * n / world                               # a rank's share of the ordered interactions
        path_ag = path = "sym" if world > 1 or n >= 16384 else "plain"  # which acc / grad kernels these sizes select
        kernel_name = {"acc": {"sym": "sym_pair_kernel<SymAcc, 8, 256, 1>", "plain": "pair_kernel<AccPass, 8, 256, 1, 1>"},
                       "grad": {"sym": "sym_pair_kernel<SymGrad, 6, 256, 1>", "plain": "pair_kernel<GradPass, 5, 128, 2, 2>"},
                       "dtmin": {"sym": "sym_dt_kernel<6, 128, 2, 2>", "plain": "pair_kernel<DtPass, 4, 128, 3, 2>"}}

        def kern(name):
            ms = mean_ms[name]
            path = path_ag if name != "dtmin" else ("sym" if world == 1 and n >= 32768 else "plain")   # dtmin is sink-sharded when world > 1
            tf = pairs_rank * FP64_FLOPS[path][name] / (ms * 1e-3) / 1e12
            pipe = pairs_rank * FP64_INSTR[path][name] / (ms * 1e-3) / (peak * 1e12 / 2)
            out = {"ms": ms, "kernel": kernel_name[name][path], "interactions_per_s": pairs_rank / (ms * 1e-3),
                   "executed_flops_per_interaction": FP64_FLOPS[path][name],
                   "executed_fp64_instr_per_interaction": FP64_INSTR[path][name],
                   "tflops": tf, "frac_of_flop_peak": tf / peak, "fp64_pipe_issue_util": pipe}
            if name in SURVEY_8D_FLOPS:
                out["frac_survey_8d"] = pairs_rank * SURVEY_8D_FLOPS[name] / (ms * 1e-3) / 1e12 / peak
            return out
        passes = {k: kern(k) for k in ("acc", "grad", "dtmin") if k in mean_ms}
        if "pn1" in mean_ms:
            passes["pn1"] = {"ms": mean_ms["pn1"], "interactions_per_s": 2.0 * len(w.bh_idx) * n / (mean_ms["pn1"] * 1e-3)}
        for k in ("exchange_acc", "exchange_grad"):
            if k in mean_ms:
                passes[k] = {"ms": mean_ms[k], "collective": "NCCL all-reduce (sum)", "bytes": 24 * n}
        dom_name = max((k for k in ("acc", "grad", "dtmin") if k in passes), key=lambda k: passes[k]["ms"])
        dom = passes[dom_name]
        roofline = roofline_of(args.config, n, dom_name, dom, passes, peak, num_sms, mean_ms, step_ms, path)
        if probe:
            roofline["measured_fp64_pipe"] = probe
            roofline["pipe_util_vs_measured_dfma"] = (
                dom["fp64_pipe_issue_util"] / probe["dfma"]["frac_of_derived_pipe_peak"])
        extras = run_extras(torch, ctx, w, pos, vel, mass, acc) if world == 1 and args.extras else None
        config5 = None
        if world == 1 and args.config == 4 and not args.no_config5 and not args.n:
            ctx.close()
            del pos, vel, mass, acc, grad, dts, apn
            torch.cuda.empty_cache()
            config5 = run_config5(torch, dev, peak, num_sms)
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": step_ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": workload_name(args.config, n), "n": n, "seed": w.seed,
                           "l2": "flushed between steps (256 MiB device write, outside the timed events)",
                           "parallelism": "1 rank" if world == 1 else
                           f"acc / grad: unordered pairs sharded over {world} ranks + NCCL all-reduce of double[N][3] after each pass; "
                           f"dtmin: sinks sharded over {world} ranks; pn1 redundant on every rank",
                           "timing": "CUDA events per C-ABI call on the launching stream, mean over steps, max over ranks"},
                "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "wall_s_timed_region": t_wall,
                "passes": passes, "roofline": roofline}
        if config5 is not None:
            line["config5"] = config5
        if extras is not None:
            line["extras"] = extras
        if world == 1 and not args.no_cpu_baseline:
            import oracle
            oracle.build()
            line["cpu_baseline"] = cpu_baseline(w, args.cpu_sinks)
            line["cpu_fast"] = cpu_fast_baseline(w, 4 * args.cpu_sinks)
        print(json.dumps(line), flush=True)
    ctx.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def static_traffic(cfg: int, n: int, kernel: str):
    """dram__bytes_read + dram__bytes_write per launch of `kernel` from the committed ncu capture of this workload
    (profiles/r2_traffic_per_launch.csv): a STATIC figure of an earlier run of the same source, not measured now."""
    prof = os.path.join(ROOT, "profiles", "r2_traffic_per_launch.csv")
    if not os.path.exists(prof) or n != {4: 1 << 20, 5: 1 << 21}.get(cfg):
        return None, None
    for row in open(prof).read().splitlines()[1:]:
        f = row.split(",")
        if len(f) >= 4 and f[0] == str(cfg) and f[1] == kernel:
            return int(f[2]) + int(f[3]), f"static: profiles/r2_traffic_per_launch.csv ({f[4] if len(f) > 4 else 'ncu'})"
    return None, None


def roofline_of(cfg, n, dom_name, dom, passes, peak, num_sms, mean_ms, step_ms, path):
    traffic, src = static_traffic(cfg, n, dom["kernel"].split("<")[0] + "_" + dom_name)
    r = {"bound": "alu", "kernel": f"{dom['kernel']} (bifrost_{dom_name}: pack + pair + finish timed together; the pair "
                                   "kernel is > 99.8 % of it)",
         "share_of_step": dom["ms"] / step_ms,
         "achieved": dom["tflops"], "peak": peak, "unit": "TFLOP/s", "frac": dom["tflops"] / peak,
         "frac_is": "EXECUTED flops (2 DFMA + DADD + DMUL, SURVEY.md 8d's convention) / derived FP64 peak",
         "peak_source": f"derived: {num_sms} SMs x 64 FP64 lanes x 2 flop x clocks.max.sm "
                        f"(no FP64 figure in MEASURED_PEAKS.json); a register-only DFMA stream measures 0.997 of it",
         "flops_per_interaction": dom["executed_flops_per_interaction"],
         "fp64_instr_per_interaction": dom["executed_fp64_instr_per_interaction"],
         "fp64_pipe_issue_util": dom["fp64_pipe_issue_util"],
         "traffic": traffic, "traffic_source": src}
    ag = mean_ms["acc"] + mean_ms["grad"]
    pairs = passes["acc"]["interactions_per_s"] * passes["acc"]["ms"] * 1e-3
    r["acc_grad"] = {
        "ms": ag,
        "frac_executed": (FP64_FLOPS[path]["acc"] + FP64_FLOPS[path]["grad"]) * pairs / (1e-3 * ag) / 1e12 / peak,
        "frac_survey_8d": (SURVEY_8D_FLOPS["acc"] + SURVEY_8D_FLOPS["grad"]) * pairs / (1e-3 * ag) / 1e12 / peak,
        "note": "frac_executed counts the flops the kernels execute; frac_survey_8d charges SURVEY.md 8(d)'s one-sided "
                "26 + 42 flops to every ordered interaction delivered - it exceeds frac_executed (and may exceed 1) "
                "because the symmetric kernels evaluate each unordered pair once"}
    return r


def run_config5(torch, dev, peak, num_sms):
    """north_star's peak-throughput case (BASELINE.json configs[4]: N = 2^21, all active, acc + grad), timed in the
    same run: 1 warm-up + 2 timed steps, CUDA events per call, L2 flushed between steps."""
    from paper_2210_02472_b200.binding import Context
    w = make_workload(5)
    n = w.n
    ctx = Context(n)
    pos, mass = (torch.from_numpy(x).to(dev) for x in (w.pos, w.mass))
    acc = torch.zeros((n, 3), dtype=torch.float64, device=dev)
    grad = torch.zeros_like(acc)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    t_acc, t_grad, steps = 0.0, 0.0, 2
    l0 = 0
    for it in range(1 + steps):
        flush.fill_(1)
        if it == 1:
            l0 = ctx.launch_count
        ev[0].record()
        ctx.acc(pos, mass, w.G, w.eps, out=acc)
        ev[1].record()
        ctx.grad(pos, mass, acc, w.G, w.eps, out=grad)
        ev[2].record()
        torch.cuda.synchronize()
        if it > 0:
            t_acc += ev[0].elapsed_time(ev[1]) / steps
            t_grad += ev[1].elapsed_time(ev[2]) / steps
    launches = ctx.launch_count - l0
    ctx.close()
    pairs = float(n) * n
    fl = FP64_FLOPS["sym"]
    return {"workload": workload_name(5, n), "steps": steps, "warmup": 1, "gpu_launches": int(launches),
            "value": pairs / (1e-3 * (t_acc + t_grad)), "unit": UNIT, "acc_ms": t_acc, "grad_ms": t_grad,
            "frac_executed": (fl["acc"] + fl["grad"]) * pairs / (1e-3 * (t_acc + t_grad)) / 1e12 / peak,
            "frac_executed_acc": fl["acc"] * pairs / (1e-3 * t_acc) / 1e12 / peak,
            "frac_executed_grad": fl["grad"] * pairs / (1e-3 * t_grad) / 1e12 / peak,
            "frac_survey_8d": (SURVEY_8D_FLOPS["acc"] + SURVEY_8D_FLOPS["grad"]) * pairs / (1e-3 * (t_acc + t_grad)) / 1e12 / peak,
            "target": "north_star: >= 0.60 of FP64 peak on this case (executed-flop convention)"}


def run_extras(torch, ctx, w, pos, vel, mass, acc):
    from paper_2210_02472_b200.binding import Context
    """Device times of the NEXT rows (SURVEY.md §8f) on the same workload, outside the timed step:
    jerk, potential, neighbour search + components, one FSI cycle.  ms per call, 2 calls each after
    one warm-up, CUDA events on the launching stream."""
    n = w.n
    r_h = 1.30477                                       # Plummer half-mass radius for a_p = 1
    # r_ngb = 1e-3 pc, r_ngb,max = 0.1 pc in a cluster of r_h = 3.1 pc
    par = dict(r_ngb=1e-3 / 3.1 * r_h, r_ngb_max=0.1 / 3.1 * r_h, tau=2.0 ** -10, C=0.5)
    out = {"n": n, "neighbour_parameters": par}
    cnt = torch.zeros(n, dtype=torch.int32, device=pos.device)
    lst = torch.full((n, 16), -1, dtype=torch.int32, device=pos.device)
    jerk = torch.zeros_like(acc)
    acc2 = torch.zeros_like(acc)
    p2, v2 = pos.clone(), vel.clone()
    calls = {
        "jerk": lambda: ctx.jerk(pos, vel, mass, w.G, w.eps, out=jerk),
        "acc_jerk": lambda: ctx.acc_jerk(pos, vel, mass, w.G, w.eps, out=(acc2, jerk)),
        "potential": lambda: ctx.potential(pos, mass, w.G, w.eps, want_phi=False),
        "neighbours": lambda: ctx.neighbours(pos, vel, mass, w.G, par["r_ngb"], par["r_ngb_max"], par["tau"], par["C"],
                                             cap=16, out=(cnt, lst)),
        "dtmin": lambda: ctx.dtmin(pos, vel, mass, w.G, w.eta_ff, w.eta_fb),
        "dtmin_neighbours": lambda: ctx.dtmin_neighbours(pos, vel, mass, w.G, w.eta_ff, w.eta_fb, par["r_ngb"], par["r_ngb_max"],
                                                         par["tau"], par["C"], cap=16),
        "components": lambda: ctx.components(cnt, lst),
        "fsi_step": lambda: ctx.fsi_step(p2, v2, mass, w.G, max(w.eps, 1e-4), 2.0 ** -12),
    }
    for name, fn in calls.items():
        fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        fn(); fn()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / 2
        out[name] = {"ms": ms}
        if name in ("jerk", "acc_jerk", "potential", "neighbours", "dtmin", "dtmin_neighbours"):
            out[name]["interactions_per_s"] = float(n) * n / (ms * 1e-3)
        if name == "fsi_step":
            out[name]["interactions_per_s"] = 4.0 * n * n / (ms * 1e-3)     # four O(N^2) sums
    out["neighbours"]["pairs_found"] = int(cnt.sum().item())
    # one HHS-FSI integration interval (Eq. 11) on config 2 (N = 16384, Kroupa masses): the hierarchy the
    # active-subset sweep stands for; host-steered recursion, so wall time is what counts
    from paper_2210_02472_b200 import workloads as W
    w2 = W.config2()
    p, v, m = (torch.from_numpy(x).to(pos.device) for x in (w2.pos, w2.vel, w2.mass))
    ctx.hhs_fsi(p.clone(), v.clone(), m, w2.G, w2.eps, 0.1, 0.1, 2.0 ** -9, max_depth=12)      # warm-up
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    l0 = ctx.launch_count
    summ, _ = ctx.hhs_fsi(p, v, m, w2.G, w2.eps, 0.1, 0.1, 2.0 ** -9, max_depth=12)
    torch.cuda.synchronize()
    out["hhs_fsi_config2"] = {"ms": 1e3 * (time.perf_counter() - t0), "tau": 2.0 ** -9, "eta": 0.1, "max_depth": 12,
                              "launches": ctx.launch_count - l0, **summ}
    # the inter-level sums of Eq. 12-13 between a slow and a fast set (S = 7/8 of the particles, F = 1/8): one mutual call
    # against the pair of one-sided calls
    ids = torch.randperm(n, device=pos.device, generator=torch.Generator(device=pos.device).manual_seed(5)).to(torch.int32)
    S_, F_ = ids[: n - n // 8].contiguous(), ids[n - n // 8:].contiguous()
    a_m = torch.zeros_like(acc)
    for name, fn in (("acc_mutual", lambda: ctx.acc_mutual(pos, mass, w.G, w.eps, S_, F_, out=a_m)),
                     ("acc_two_calls", lambda: (ctx.acc(pos, mass, w.G, w.eps, S_, F_, out=a_m),
                                                ctx.acc(pos, mass, w.G, w.eps, F_, S_, out=a_m))),
                     ("grad_mutual", lambda: ctx.grad_mutual(pos, mass, acc, w.G, w.eps, S_, F_, out=a_m)),
                     ("grad_two_calls", lambda: (ctx.grad(pos, mass, acc, w.G, w.eps, S_, F_, out=a_m),
                                                 ctx.grad(pos, mass, acc, w.G, w.eps, F_, S_, out=a_m)))):
        fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(); fn(); fn(); e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / 2
        out[name] = {"ms": ms, "n_slow": int(S_.numel()), "n_fast": int(F_.numel()),
                     "interactions_per_s": 2.0 * S_.numel() * F_.numel() / (ms * 1e-3)}
    # one HHS-FSI interval of the paper's softened equal-mass cluster (Fig. 8): N = 161000,
    # eta_ff = eta_fb = 0.2, Eq. 24-29 with eta = 0.1 as dt_cap, tau = 1e-3 Myr; energy error of the interval
    w8 = W.fig8()
    ctx8 = Context(w8.n)
    p, v, m = (torch.from_numpy(x).to(pos.device) for x in (w8.pos, w8.vel, w8.mass))

    def energy():
        return float(ctx8.kinetic_energy(v, m).cpu()) + float(ctx8.potential(p, m, w8.G, w8.eps, want_phi=False)[1].cpu())
    rec8 = {"n": w8.n, "tau": W.fig8_tau(), "eta": 0.2, "eta_criteria": 0.1}
    for it in range(2):                                   # first interval = warm-up (allocates the integrator scratch)
        a8, j8 = ctx8.acc_jerk(p, v, m, w8.G, w8.eps)
        c8 = ctx8.grad(p, m, a8, w8.G, w8.eps)
        cap = torch.full((w8.n,), float("inf"), dtype=torch.float64, device=pos.device)
        ctx8.timestep_criteria(v, a8, c8, j8, 0.1, 0.1, 0.1, inout_dt=cap)
        e_before = energy()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        l0 = ctx8.launch_count
        summ, _ = ctx8.hhs_fsi(p, v, m, w8.G, w8.eps, 0.2, 0.2, W.fig8_tau(), max_depth=40, dt_cap=cap)
        torch.cuda.synchronize()
        rec8.update({"ms": 1e3 * (time.perf_counter() - t0), "launches": ctx8.launch_count - l0, **summ,
                     "rel_energy_error_of_the_interval": abs(energy() - e_before) / abs(e_before)})
    out["hhs_fsi_fig8"] = rec8
    # the same interval (a third one, from the state the second left) with Eq. 24-29 evaluated at EVERY level over the
    # level's own particles (bifrost_set_level_criteria) instead of only as dt_cap at level 0
    ctx8.set_level_criteria(0.1, 0.1, 0.1)
    e_before = energy()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    l0 = ctx8.launch_count
    summ, _ = ctx8.hhs_fsi(p, v, m, w8.G, w8.eps, 0.2, 0.2, W.fig8_tau(), max_depth=40)
    torch.cuda.synchronize()
    out["hhs_fsi_fig8_level_criteria"] = {"ms": 1e3 * (time.perf_counter() - t0), "launches": ctx8.launch_count - l0, **summ,
                                          "rel_energy_error_of_the_interval": abs(energy() - e_before) / abs(e_before)}
    ctx8.close()
    return out


# --------------------------------------------------------------------------------------
# small-active-set sweep (configs 2 and 3): us per call, launch-bound / L2-bound regime
# --------------------------------------------------------------------------------------

def run_sweep(args):
    import torch
    from paper_2210_02472_b200 import workloads as W
    from paper_2210_02472_b200.binding import Context
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    out = {"metric": "us per C-ABI call vs active-set size (configs 2, 3)", "unit": "us", "data": "synthetic",
           "timing": "CUDA events around 20 back-to-back calls after 3 warm-ups, sources L2-resident; *_graph_us = the same 20 calls captured in one CUDA graph and replayed", "cases": []}
    for cfg, sizes in ((2, [W.config2_sink_list(k) for k in range(0, 15)]),
                       (3, [W.config3_sink_list(k) for k in range(10, -1, -1)])):
        w = W.CONFIGS[cfg]()
        ctx = Context(w.n)
        pos, vel, mass = (torch.from_numpy(x).to(dev) for x in (w.pos, w.vel, w.mass))
        acc = ctx.acc(pos, mass, w.G, w.eps)
        outs = {"acc": torch.zeros_like(acc), "grad": torch.zeros_like(acc)}
        dt_out = (torch.empty(w.n, dtype=torch.float64, device=dev), torch.empty(w.n, dtype=torch.float64, device=dev),
                  torch.empty(w.n, dtype=torch.int32, device=dev), torch.empty(w.n, dtype=torch.int32, device=dev))
        for sinks in sizes:
            si = torch.from_numpy(sinks).to(dev)
            ns = int(sinks.shape[0])
            calls = {"acc": lambda: ctx.acc(pos, mass, w.G, w.eps, si, None, out=outs["acc"]),
                     "grad": lambda: ctx.grad(pos, mass, acc, w.G, w.eps, si, None, out=outs["grad"]),
                     "dtmin": lambda: ctx.dtmin(pos, vel, mass, w.G, w.eta_ff, w.eta_fb, si, None, out=dt_out)}
            rec = {"config": cfg, "n_src": w.n, "n_sink": ns}
            reps = 20 if ns * w.n < 2e9 else 3
            for name, fn in calls.items():
                for _ in range(3):
                    fn()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                e0.record()
                for _ in range(reps):
                    fn()
                e1.record()
                torch.cuda.synchronize()
                us = 1e3 * e0.elapsed_time(e1) / reps
                rec[name + "_us"] = round(us, 2)
                rec[name + "_pairs_per_s"] = ns * float(w.n) / (us * 1e-6)
                # the same calls captured in a CUDA graph and replayed: device time without the
                # host's launch cost (the calls are asynchronous and capture-safe)
                graph = torch.cuda.CUDAGraph()
                with torch.cuda.graph(graph):
                    for _ in range(reps):
                        fn()
                graph.replay()
                torch.cuda.synchronize()
                e0.record()
                graph.replay()
                e1.record()
                torch.cuda.synchronize()
                rec[name + "_graph_us"] = round(1e3 * e0.elapsed_time(e1) / reps, 2)
                del graph
            # a1 gather traffic: the acc pack reads 32 B and writes 48 B per source
            rec["acc_source_bytes"] = 80 * w.n
            out["cases"].append(rec)
        ctx.close()
    # same-list (all-active) acc / grad over the list length m: the symmetric kernels (every unordered pair once)
    # against the plain ones, switched with bifrost_set_tuning; config 4's recipe at reduced N
    out["same_list"] = []
    ctx = Context(1 << 18)
    for m in (4096, 8192, 12288, 16384, 24576, 32768, 65536, 131072, 262144):
        w = W.config4(n=m, n_sbh=10)
        pos, vel, mass = (torch.from_numpy(x).to(dev) for x in (w.pos, w.vel, w.mass))
        rec = {"m": m}
        for mode, thr in (("sym", 0), ("plain", 1 << 40)):
            ctx.set_tuning(Context.TUNE_SYM_MIN_N, thr)
            a = ctx.acc(pos, mass, w.G, w.eps)
            for name, fn in (("acc", lambda: ctx.acc(pos, mass, w.G, w.eps)), ("grad", lambda: ctx.grad(pos, mass, a, w.G, w.eps)),
                             ("dtmin", lambda: ctx.dtmin(pos, vel, mass, w.G, w.eta_ff, w.eta_fb))):
                reps = 20 if m <= 65536 else 4
                for _ in range(reps):
                    fn()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                e0.record()
                for _ in range(reps):
                    fn()
                e1.record()
                torch.cuda.synchronize()
                rec[f"{name}_{mode}_us"] = round(1e3 * e0.elapsed_time(e1) / reps, 1)
        out["same_list"].append(rec)
    ctx.close()
    print(json.dumps(out), flush=True)
    return 0


def run_small(args):
    """Profiling aid: config 2 (N = 16384 sources), 2^k seeded sinks, acc / grad / dtmin three times each (one fused
    launch per call) - the command the ncu captures of pair_fused_kernel in profiles/ were taken with."""
    import torch
    from paper_2210_02472_b200 import workloads as W
    from paper_2210_02472_b200.binding import Context
    torch.cuda.set_device(0)
    w = W.config2()
    ctx = Context(w.n)
    pos, vel, mass = (torch.from_numpy(x).cuda() for x in (w.pos, w.vel, w.mass))
    acc = ctx.acc(pos, mass, w.G, w.eps)
    si = torch.from_numpy(W.config2_sink_list(args.small)).cuda()
    for _ in range(3):
        ctx.acc(pos, mass, w.G, w.eps, si, None)
        ctx.grad(pos, mass, acc, w.G, w.eps, si, None)
        ctx.dtmin(pos, vel, mass, w.G, w.eta_ff, w.eta_fb, si, None)
    torch.cuda.synchronize()
    print(json.dumps({"small": args.small, "n_sink": int(si.numel()), "launches": ctx.launch_count}))
    ctx.close()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", type=int, default=4, choices=[4, 5])
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--cpu-sinks", type=int, default=2048, help="oracle sample size (sinks) for cpu_baseline")
    ap.add_argument("--ref-sinks", type=int, default=1024, help="oracle sample size (sinks) per reference step")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--n", type=int, default=0, help="override the workload's N (profiling aid; NOT the benchmark configuration)")
    ap.add_argument("--extras", action="store_true", help="also time the NEXT rows (jerk, potential, neighbours, components, one FSI cycle) once, outside the timed step")
    ap.add_argument("--sweep", action="store_true", help="small-active-set sweep of configs 2 and 3 (us per call); prints one JSON line")
    ap.add_argument("--no-fp64-probe", action="store_true", help="skip the register-only FP64-pipe peak probe")
    ap.add_argument("--no-config5", action="store_true", help="skip the N = 2^21 acc + grad block of the default line")
    ap.add_argument("--small", type=int, default=-1, help="profiling aid: config 2 with 2^k sinks, acc / grad / dtmin three times each")
    args = ap.parse_args()
    if args.small >= 0:
        return run_small(args)
    if args.impl == "reference":
        return run_reference(args)
    if args.sweep:
        return run_sweep(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
