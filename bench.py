#!/usr/bin/env python
"""bench.py -- throughput of the epoch-substitution-model hot path on B200 (one JSON line on stdout, rank 0).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl cuda|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

A STEP is one pass of the whole hot path (segmenter, eigensystems, segment exponentials +
chain convolution, pruning, root reduction) over BASELINE.json config 2 (`configs[1]`: HKY, 10 epochs, 2 000 tips,
10 000 site patterns, 4 rate categories), seeded synthetic input.  BASELINE.json's metric has two halves:
  * "pruning partials GB/s"     -> the headline `value`: algorithmic bytes of a5+a6
                                   divided by the time of the WHOLE step;
  * "epoch branch matrices/s"   -> the `matrices` object: config 5 (61-state convolution microbenchmark, a1..a4), the
                                   largest single-GPU matrix workload, with its own (FP64 ALU) roofline.
Multi-GPU: the path does not shard (replicas only) -- every rank runs an independent replica
of the same problem, no data-path collective; value = N x units / max-over-ranks time ("weak" scaling).

`--impl reference` times the CPU oracle (oracle/, as it stands, long-double build, OpenMP) on a bounded sample of the same
workload on the box's host cores; rank 0 only.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402  (input generators only; shared with the oracle, holds no arithmetic of the method)

# dram__bytes_read.sum + dram__bytes_write.sum of the pruning launches of one config-2 step, from the committed
# `ncu --set full` capture named here (re-captured whenever the pruning kernel changes; `--traffic` overrides it)
NCU_TRAFFIC = {"bytes_per_step": 2.6034e9, "profile": "profiles/r2_prune4_lane_ncu.md", "commit": "0aeab7f",
               "kernel": "prune4_lane_kernel<4, 1, false> + <4, 1, true>"}

METRIC = "pruning partials GB/s (fp64) over the whole a1..a6 log-likelihood step; epoch branch matrices/s in `matrices`"
UNIT = "GB/s"


# ---------------------------------------------------------------------------------------------- algorithmic work
def pruning_bytes(prob) -> dict:
    """Algorithmic HBM bytes of a5: every internal node writes its partials [C][L][K] f64 and its
    scale exponents [L] i32, reads per child either partials + exponents (internal child) or one byte per pattern
    (tip child), and the two children's C K x K matrices; a6 re-reads the root partials + exponents, reads the
    pattern weights and writes the site log-likelihoods."""
    K, C, L, N = prob.K, prob.C, prob.L, prob.N
    part = C * L * K * 8
    n_int = N - 1
    is_child_internal = np.zeros(2 * N - 1, dtype=bool)
    is_child_internal[N:] = True
    par = np.asarray(prob.parent)
    children = np.nonzero(par >= 0)[0]
    n_int_children = int(np.sum(children >= N))
    n_tip_children = int(np.sum(children < N))
    a5 = n_int * (part + 4 * L + 2 * C * K * K * 8) + n_int_children * (part + 4 * L) + n_tip_children * L
    a6 = part + 4 * L + 8 * L + 8 * L
    flops = n_int * C * L * (4 * K * K + K)
    return {"a5": a5, "a6": a6, "flops": flops}


def compulsory_bytes(prob) -> dict:
    """HBM bytes the depth-first pruning has to move: every internal node's partials [C][L][K] f64 and
    scale exponents [L] i32 are WRITTEN once (they are outputs: epx_get_partials, the incremental path) and never read back
    -- a child's vector is handed to its parent in registers / shared memory --; every tip state is read once (1 B per tip
    and pattern); the two children's C K x K matrices once per node.  a6 as in pruning_bytes()."""
    K, C, L, N = prob.K, prob.C, prob.L, prob.N
    part = C * L * K * 8
    n_int = N - 1
    a5 = n_int * (part + 4 * L + 2 * C * K * K * 8) + N * L
    a6 = part + 4 * L + 8 * L + 8 * L
    return {"a5": a5, "a6": a6}


def tree_levels(parent, N: int) -> int:
    """Post-order levels of the tree (host integer work on the input; a workload property for `config`)."""
    par = np.asarray(parent)
    n = par.shape[0]
    kids = [[] for _ in range(n)]
    root = -1
    for v in range(n):
        if par[v] >= 0:
            kids[par[v]].append(v)
        else:
            root = v
    level = np.zeros(n, dtype=np.int64)
    order, stack = [], [root]
    while stack:
        u = stack.pop()
        order.append(u)
        stack.extend(kids[u])
    for u in reversed(order):
        if kids[u]:
            level[u] = 1 + max(level[k] for k in kids[u])
    return int(level.max())


def workload_config(prob, cid: int, world: int) -> dict:
    """`config` of the JSON line: the workload and how the timing treats L2 -- identical for both arms."""
    cfg = {"workload": W.CONFIG_NAMES[cid], "K": prob.K, "M": prob.M, "C": prob.C, "seed": W.config_seed(cid),
           "parallelism": f"replicas x{world} (no collective)"}
    if prob.N:
        part_gb = (prob.N - 1) * prob.C * prob.L * prob.K * 8 / 1e9
        cfg.update({"N_tips": prob.N, "L": prob.L, "tree_levels": tree_levels(prob.parent, prob.N),
                    "l2": f"inputs larger than L2: {part_gb:.2f} GB of partials rewritten every step vs 126 MB L2"
                          if part_gb > 0.126 else f"working set {part_gb * 1e3:.1f} MB of partials fits the 126 MB L2 (latency-bound "
                                                "configuration; no flush, steps run back to back)"})
    else:
        p_gb = prob.n_br * prob.C * prob.K * prob.K * 8 / 1e9
        cfg.update({"n_br": prob.n_br, "l2": f"inputs larger than L2: {p_gb:.2f} GB of P written per step vs 126 MB L2"})
    return cfg


def chain_flops(K: int, C: int, n_seg: np.ndarray) -> dict:
    """Executed useful flops of the eigenbasis chain (one K^3 product per segment and category, K not padded) and the
    straightforward exp-then-convolve count of SURVEY.md 8(d) for context."""
    nseg = n_seg.astype(np.int64)
    executed = int(nseg.sum()) * C * 2 * K ** 3
    straightforward = int((2 * nseg - (nseg > 0)).sum()) * C * 2 * K ** 3
    return {"executed": executed, "straightforward": straightforward}


def cached_chain_flops(K: int, C: int, M: int, n_seg: np.ndarray) -> dict:
    """Executed useful flops with the cached products of consecutive full epochs (EPX_OPT_EPOCH_PRODUCTS):
    a chain over >= 2 full epochs (n_seg >= 4) costs 3 products, the table costs a products for each (a, category), a = 1..M-2."""
    nseg = n_seg.astype(np.int64)
    chain = int(np.where(nseg >= 4, 3, nseg).sum()) * C * 2 * K ** 3
    table = sum(range(1, M - 1)) * C * 2 * K ** 3
    return {"chain": chain, "table": table, "executed": chain + table}


def n_segments(prob) -> np.ndarray:
    """Segment count per matrix slot from the inputs (host integer arithmetic for the flop count only)."""
    ch, ph = prob.branch_heights()
    tau = np.asarray(prob.tau)
    e_lo = np.searchsorted(tau, ch, side="right")
    e_hi = np.searchsorted(tau, ph, side="left")
    return np.where(ph > ch, e_hi - e_lo + 1, 0)


# ---------------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples SM clock, power and clock-event reasons of one GPU through NVML while the timed regions run."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, index: int, period_s: float = 0.02):
        self.samples, self.reason_bits, self.power = [], 0, []
        self.period, self._stop, self._thr, self.h, self.max_mhz = period_s, threading.Event(), None, None, None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as e:  # NVML missing: the JSON line says so instead of inventing clocks
            self.err = repr(e)

    def _loop(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    bits = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    bits = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                self.reason_bits |= int(bits)
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:
                pass
            self._stop.wait(self.period)

    def start(self):
        if self.h is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()

    def stop(self) -> dict:
        if self._thr is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml unavailable"]}
        self._stop.set()
        self._thr.join()
        reasons = [name for bit, name in self.REASONS.items() if self.reason_bits & bit]
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None, "sm_max_mhz": self.max_mhz,
                "reasons": reasons, "samples": len(self.samples),
                "power_w_max": max(self.power) if self.power else None}


# ---------------------------------------------------------------------------------------------- reference arm
def oracle_sample_problem(prob, L_s: int):
    """The same workload restricted to its first L_s site patterns (full tree, every branch matrix)."""
    import copy
    q = copy.copy(prob)
    q.L = L_s
    q.tip_states = np.ascontiguousarray(prob.tip_states[:, :L_s])
    q.pattern_weights = np.ascontiguousarray(prob.pattern_weights[:L_s])
    return q


def time_oracle(prob, target_s: float, steps: int = 1, warmup: int = 0):
    """Time the oracle's evaluate() on a pattern sample sized (from a 32-pattern probe) to ~target_s per step.
    The long-double build is timed: the oracle does no rescaling (reading A12), so its double build
    underflows on a 2000-tip tree (site likelihoods ~1e-1200) and cannot run this workload."""
    import oracle
    orc = oracle.Oracle("ld")
    cores = int(os.environ.get("OMP_NUM_THREADS", 0)) or len(os.sched_getaffinity(0))
    probe = oracle_sample_problem(prob, min(32, prob.L))
    t0 = time.perf_counter()
    orc.evaluate(probe)
    t_probe = time.perf_counter() - t0
    L_s = int(min(prob.L, max(32, 32 * target_s / max(t_probe, 1e-6))))
    sample = oracle_sample_problem(prob, L_s)
    for _ in range(warmup):
        orc.evaluate(sample)
    times = []
    for _ in range(steps):
        t0 = time.perf_counter()
        out = orc.evaluate(sample)
        times.append(time.perf_counter() - t0)
    nbytes = compulsory_bytes(sample)
    sec = float(np.mean(times))
    return {"value": (nbytes["a5"] + nbytes["a6"]) / sec / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"first {L_s} of {prob.L} site patterns of config 2, full 2000-tip tree, all {prob.n_br} x {prob.C} "
                      f"branch matrices; oracle long-double build with OpenMP, {sec:.2f} s per pass",
            "seconds_per_step": sec, "lnl_sample": float(out["lnl"])}


def run_reference(args) -> None:
    if int(os.environ.get("RANK", "0")) != 0:
        return
    prob = W.make_config(2)
    world = int(os.environ.get("WORLD_SIZE", "1"))
    # bounded: (steps + warmup) passes of ~target seconds each, the whole run within a few minutes
    target = min(10.0, 150.0 / max(1, args.steps + args.warmup))
    r = time_oracle(prob, target, steps=args.steps, warmup=args.warmup)
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": r["seconds_per_step"] * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(prob, 2, world),
            "note": "CPU oracle (long-double build, OpenMP) on a bounded pattern sample of the config; rank 0 only",
            "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------- CUDA arm
def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def bracket(torch, stream, fn, steps):
    """Device time in ms of `steps` calls of fn(), CUDA events on the launching stream, synchronised on both sides."""
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stream.synchronize()
    e0.record(stream)
    for _ in range(steps):
        fn()
    e1.record(stream)
    stream.synchronize()
    return e0.elapsed_time(e1)


def max_over_ranks(x: float, world: int, device: str = "cuda") -> float:
    """Max of a per-rank device time over all ranks (the only cross-rank exchange of the bench: replicas only)."""
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(unit_bytes: float, ms_step: float, world: int) -> float:
    """GB/s of `world` independent replicas that each moved `unit_bytes` per step, the slowest taking ms_step."""
    return world * unit_bytes / (ms_step * 1e-3) / 1e9


def taylor_chain_flops(prob) -> dict:
    """Useful flops (K not padded, 2 K^3 per dense product) the componentwise-Taylor chain kernel executes for a tree-mode
    codon problem (A21): per dense exponential 6 products (powers M^2..M^4, three Horner steps) + s squarings with
    2^s >= r d max|q_ii|; a (slot, category) exponentiates its first and last segment, takes interior epochs from the
    full-epoch table, and multiplies its n_seg factors together.  Host integer / scalar bookkeeping for the flop count."""
    K, C, M = prob.K, prob.C, prob.M
    ch, ph = prob.branch_heights()
    tau = np.asarray(prob.tau)
    e_lo = np.searchsorted(tau, ch, side="right")
    e_hi = np.searchsorted(tau, ph, side="left")
    nseg = np.where(ph > ch, e_hi - e_lo + 1, 0)
    qmax = np.max(-np.diagonal(prob.Q, axis1=1, axis2=2), axis=1)          # max_i |q_ii| per epoch

    def products(e, d):       # dense exponential of epoch e over duration d, per category
        n = 0
        for r in prob.rates:
            mu = r * d * qmax[e]
            n += 6 + (int(np.ceil(np.log2(mu))) if mu > 1.0 else 0)
        return n

    total = 0
    for b in range(len(ch)):
        n = int(nseg[b])
        if n == 0:
            continue
        if n == 1:
            total += products(e_hi[b], ph[b] - ch[b])
        else:
            total += products(e_hi[b], ph[b] - tau[e_hi[b] - 1]) + products(e_lo[b], tau[e_lo[b]] - ch[b]) + (n - 1) * C
    table = sum(products(e, tau[e] - tau[e - 1]) for e in range(1, M - 1)) if M >= 3 else 0
    return {"chain_products": int(total), "table_products": int(table), "flops": int(total + table) * 2 * K ** 3}


def run_cuda(args) -> None:
    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the hot path has no CPU fallback (use --impl reference for the oracle)")
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    from paper_1309_3075_b200 import build as B
    if rank == 0:
        B.build_library()
    if world > 1:
        dist.barrier()
    import paper_1309_3075_b200 as epx
    legs = set(args.legs.split(","))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    K, Wm = args.steps, max(3, args.warmup)
    prob = W.make_config(2)
    comp, lvl = compulsory_bytes(prob), pruning_bytes(prob)
    unit_bytes = comp["a5"] + comp["a6"]
    ctx = epx.from_problem(prob, device=local)
    for opt, val in args.opt:
        ctx.set_option(opt, val)
    ctx.set_option(epx.EPX_OPT_STAGE_EVENTS, 1)
    stream = ctx.stream
    lnl = None
    for _ in range(Wm):
        lnl = ctx.log_likelihood()
    assert ctx.status() == 0 and np.isfinite(lnl)

    clocks = ClockSampler(local)
    clocks.start()
    # (1) headline: K steps back to back, inputs resident in HBM; every step re-runs a1..a6 (nothing is cached)
    launches0 = ctx.launch_count()
    barrier()
    ms_total = bracket(torch, stream, ctx.enqueue_log_likelihood, K)
    barrier()
    gpu_launches = ctx.launch_count() - launches0
    assert abs(ctx.fetch_log_likelihood() - lnl) <= 1e-12 * abs(lnl)
    ms_step = max_over_ranks(ms_total / K, world)

    # (2) roofline of the dominant kernel: the same K steps with the per-stage CUDA events read after every step
    stage_ms = np.zeros(5)
    stage_launches = None
    for _ in range(K):
        ctx.enqueue_log_likelihood()
        ms, stage_launches = ctx.get_stage_ms()
        stage_ms += ms
    stage_ms /= K

    # (3) end to end through the C ABI with HOST buffers: every setter (host -> device copies) + log_likelihood
    #     (device -> host read of logL and the status word) inside the timed region
    e2e = None
    if "e2e" in legs:
        tips_u8 = np.ascontiguousarray(prob.tip_states, dtype=np.uint8)    # the alignment as host BYTES (epx_set_tip_states_u8)

        def e2e_step():
            epx.set_problem(ctx, prob, tip_states_u8=tips_u8)
            return ctx.log_likelihood()
        Ke = max(3, min(K, 20))
        for _ in range(2):
            e2e_step()
        barrier()
        ms_e2e = bracket(torch, stream, e2e_step, Ke) / Ke
        barrier()
        ms_e2e = max_over_ranks(ms_e2e, world)
        n_nodes = prob.n_nodes
        # tip states as bytes (rows padded to 32), pattern weights, parent + height, the two pruning plans (32 B per node
        # each), models, boundaries, category rates + weights, root frequencies
        h2d = (prob.N * ((prob.L + 31) // 32 * 32) + 8 * prob.L + 4 * n_nodes + 8 * n_nodes + 64 * (prob.N - 1) +
               8 * prob.M * prob.K * prob.K + 8 * prob.M * prob.K + 8 * (prob.M - 1) + 16 * prob.C + 8 * prob.K)
        e2e = {"value": whole_job_value(unit_bytes, ms_e2e, world), "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": 12, "ms_per_step": ms_e2e, "steps": Ke,
               "what": "all epx_set_* calls from host arrays (tip states as host bytes through epx_set_tip_states_u8) + epx_log_likelihood (syncs, reads logL + status)"}
    # (4) SURVEY.md 8(f) f1, reported beside the headline: one MCMC-style move (one random internal node slides between its
    #     children and its parent) followed by an incremental re-evaluation, host call to host result
    inc = bench_incremental(torch, epx, ctx, prob, stream) if "incremental" in legs else None
    clk = clocks.stop()
    plan = ctx.plan_info()
    ws_bytes = ctx.workspace_bytes()
    ctx.close()

    hbm_peak, peak_src = load_peaks()
    prune_ms = float(stage_ms[3])
    prune_launches = int(stage_launches[3])
    traffic_step = args.traffic * prune_launches if args.traffic is not None else NCU_TRAFFIC["bytes_per_step"]
    gbs = lambda nbytes: nbytes / (prune_ms * 1e-3) / 1e9      # noqa: E731
    roofline = {"bound": "hbm", "kernel": prune_kernel_name(args.opt, prob.L) + " (a5; depth-first walk, bottom pieces + top piece)",
                # algorithmic bytes of the depth-first pruning = its compulsory HBM traffic: partials +
                # exponents written once, tips and matrices read once; a physical rate, comparable with the copy peak
                "achieved": gbs(comp["a5"]), "peak": hbm_peak, "unit": "GB/s", "frac": gbs(comp["a5"]) / hbm_peak,
                "compulsory_bytes": comp["a5"],
                "traffic": traffic_step / prune_launches,
                "dram_gbs": gbs(traffic_step), "dram_frac": gbs(traffic_step) / hbm_peak,
                "traffic_source": ("--traffic" if args.traffic is not None else
                                   f"dram__bytes_read.sum + dram__bytes_write.sum per launch (step total / launches), "
                                   f"{NCU_TRAFFIC['profile']} ({NCU_TRAFFIC['kernel']}, captured at commit {NCU_TRAFFIC['commit']})"),
                # SURVEY.md 8(d)'s level-by-level byte model (every child block read back once by its parent): NOT a physical
                # rate -- the walk never performs those reads -- kept for comparison with round 1 and with level kernels
                "level_model_bytes": lvl["a5"], "level_model_gbs": gbs(lvl["a5"]), "level_model_frac": gbs(lvl["a5"]) / hbm_peak,
                "peak_source": peak_src, "launches_per_step": prune_launches,
                "algorithmic_bytes_per_launch": comp["a5"] / prune_launches,
                "avg_launch_ms": prune_ms / prune_launches, "share_of_step": prune_ms / float(stage_ms.sum()),
                "stage_ms": {n: float(v) for n, v in zip(epx.STAGE_NAMES, stage_ms)},
                "stage_ms_flat": "segment/eigen/chain/prune/root = " + "/".join("%.4f" % v for v in stage_ms),
                # (K = 4, graph replay: a1 runs on a second branch beside a2..a5, so its stage reads ~0 ms: hidden, not measured)
                "stage_note": "segment ~0: a1 overlaps a2-a5 on a second graph branch at K=4, its time is not measured"}

    cfg = workload_config(prob, 2, world)
    assert cfg["tree_levels"] == plan["levels"]
    line = {"metric": METRIC, "value": whole_job_value(unit_bytes, ms_step, world), "unit": UNIT, "n_gpus": world,
            "steps": K, "warmup": Wm, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg,
            "value_definition": "compulsory HBM bytes of a5 + a6 (partials + exponents written once, tips / matrices read "
                                "once; DESIGN.md section 5) x replicas / time of the WHOLE a1..a6 step",
            "value_level_model": whole_job_value(lvl["a5"] + lvl["a6"], ms_step, world),
            "workspace_bytes": ws_bytes, "plan": plan,
            "roofline": roofline, "gpu_launches": int(gpu_launches), "clocks": clk, "log_likelihood": lnl,
            "matrices_per_s_cfg2": world * prob.n_br * prob.C / (float(stage_ms[:3].sum()) * 1e-3)}
    if e2e is not None:
        line["e2e"] = e2e
    if inc is not None:
        line["incremental"] = inc
    peaks = None
    if rank == 0 and ("matrices" in legs or "other" in legs):
        peaks = {"dfma": epx.measure_fp64_peak(0, 200.0, local), "dmma": epx.measure_fp64_peak(1, 200.0, local)}
    if rank == 0 and "matrices" in legs:
        line["matrices"] = bench_matrices(torch, epx, local, K, peaks, sustain_s=args.sustain)
        # SURVEY.md 8(f) f1, reported separately (it changes the algorithmic flops; config 5's text asks for the full chain)
        line["matrices_cached"] = bench_matrices(torch, epx, local, K, peaks, options=[(epx.EPX_OPT_EPOCH_PRODUCTS, 1)],
                                                 label=", products of consecutive full epochs cached (SURVEY.md 8(f) f1)")
    if rank == 0 and "other" in legs:
        line["other_configs"] = bench_other_configs(torch, epx, local, K, peaks)
    if rank == 0 and "batch" in legs:
        line["batch"] = bench_batch(torch, epx, local)
    if rank == 0 and "cpu" in legs and world == 1:
        r = time_oracle(prob, 15.0)
        line["cpu_baseline"] = {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")}
        line["cpu_baseline"]["cfg1_single_thread_s"] = time_oracle_single_thread_cfg1()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(finalise_line(line)), flush=True)


def _r(x, digits: int = 4):
    """Round to `digits` significant digits (the compact copies only; the full objects keep every digit)."""
    if x is None:
        return None
    x = float(x)
    return 0.0 if x == 0 else float(f"{x:.{digits}g}")


def compact_numbers(line: dict) -> dict:
    """The numbers of the optional legs that BASELINE.json's metric and north_star name -- config 5's matrices/s and its share of
    the FP64 tensor peak, the rooflines of configs 3 and 6, the latencies of configs 1 and 4 -- as one flat dict of short keys
    and scalars.  Missing legs leave their keys out."""
    out = {}

    def put(k, v, digits=4):
        if v is not None:
            if isinstance(v, (int, np.integer)) and not isinstance(v, bool):
                out[k] = int(v)
            else:
                out[k] = _r(v, digits) if isinstance(v, (float, np.floating)) else v

    for tag, key in (("cfg5", "matrices"), ("cfg5c", "matrices_cached")):     # cfg5c: products of consecutive full epochs cached (f1)
        m = line.get(key)
        if not m:
            continue
        rf = m["roofline"]
        put(tag + "_ms", m["ms_per_step"]); put(tag + "_Mmat_per_s", m["value"] / 1e6)
        put(tag + "_chain_ms", rf["stage_ms"]["chain"]); put(tag + "_eigen_ms", rf["stage_ms"]["eigen"])
        put(tag + "_chain_tflops", rf["achieved"]); put(tag + "_dmma_peak", rf["peak"]); put(tag + "_chain_frac", rf["frac"])
        put(tag + "_sm_mhz", m["clocks"].get("sm_mhz")); put(tag + "_reasons", ",".join(m["clocks"].get("reasons") or []) or "none")
        su = m.get("sustained")
        if su:
            put(tag + "_sus_s", su["seconds"], 3); put(tag + "_sus_ms", su["ms_per_step"]); put(tag + "_sus_Mmat_per_s", su["matrices_per_s"] / 1e6)
            put(tag + "_sus_tflops", su["whole_step_useful_tflops"]); put(tag + "_sus_dmma_peak", su["dmma_peak_sustained"])
            put(tag + "_sus_frac", su["whole_step_frac_of_sustained_peak"]); put(tag + "_sus_sm_mhz", su["clocks"].get("sm_mhz"))
            put(tag + "_sus_peak_sm_mhz", su["peak_probe_clocks"].get("sm_mhz"))
            put(tag + "_sus_reasons", ",".join(su["clocks"].get("reasons") or []) or "none")
    other = line.get("other_configs") or {}
    for name, o in other.items():
        if not isinstance(o, dict) or "config" not in o:
            continue
        tag = name.split("_")[0]                       # cfg1, cfg3, cfg4, cfg6
        put(tag + "_ms", o["ms_per_step"]); put(tag + "_launches", o["gpu_launches_per_step"])
        for leg in ("prune", "chain"):
            rf = o.get("roofline_" + leg)
            if rf:
                put(f"{tag}_{leg}_ms", o["stage_ms"][leg]); put(f"{tag}_{leg}_tflops", rf["achieved"]); put(f"{tag}_{leg}_frac", rf["frac"])
                put(f"{tag}_{leg}_launches", rf["launches"])
        if "us_per_step" in o and "roofline_prune" not in o:
            put(tag + "_dep_ops", o["plan"]["largest_piece_ops"] + o["plan"]["top_piece_ops"] if o["plan"]["depth_first"] else o["plan"]["levels"])
        if "alternative" in o:
            put(tag + "_taylor_ms", o["alternative"]["ms_per_step"])
    inc = line.get("incremental")
    if inc and "ms_per_move" in inc:
        put("inc_ms_per_move", inc["ms_per_move"])
    return out


def finalise_line(line: dict) -> dict:
    """What the driver keeps of the JSON line is `roofline` (scalars, strings cut at ~120 characters) and the last ~1 500
    characters.  So the numbers of compact_numbers() go (a) as flat scalars into `roofline` and (b) into a `summary` object that is
    the LAST key of the line and stays under 1 200 characters; the full objects stay where they were."""
    nums = compact_numbers(line)
    out = dict(line)
    out["roofline"] = dict(line["roofline"], **nums)
    head = {"cfg2_ms": _r(line["ms_per_step"]), "cfg2_GBps": _r(line["value"]), "cfg2_prune_frac": _r(line["roofline"]["frac"]),
            "cfg2_prune_GBps": _r(line["roofline"]["achieved"]), "hbm_peak": _r(line["roofline"]["peak"])}
    if line.get("e2e"):
        head["cfg2_e2e_ms"] = _r(line["e2e"]["ms_per_step"])
    summary = dict(head, **nums)
    # shortest-first trimming if a future key pushes it over: drop the least important tails, never the cfg5 / cfg3 / cfg6 fractions
    for k in ("cfg3_chain_launches", "cfg1_launches", "cfg4_launches", "cfg6_launches", "cfg3_launches", "cfg5c_dmma_peak", "cfg5c_eigen_ms",
              "cfg4_taylor_ms", "cfg5c_chain_tflops", "cfg3_chain_tflops", "cfg3_prune_tflops", "cfg6_prune_tflops", "cfg5c_reasons",
              "cfg5_sus_peak_sm_mhz", "cfg5_sus_tflops", "cfg5_reasons", "cfg5_sus_reasons"):
        if len(json.dumps(summary)) <= 1200:
            break
        summary.pop(k, None)
    out.pop("summary", None)
    out["summary"] = summary
    return out


def prune_kernel_name(opts, L: int) -> str:
    """Name of the K = 4 pruning kernel the config-2 context launches under the EPX_OPT overrides of --opt."""
    o = dict(opts)
    kernel, ppl = o.get(3, 0), o.get(6, 0)
    if kernel == 5:
        return "prune4_dfs_kernel<4, %d>" % (ppl or (2 if L >= 4096 else 1))
    if kernel == 3:
        return "prune4_mma_kernel<4>"
    if kernel == 2:
        return "prune4_kernel<4> (level by level)"
    if kernel == 1:
        return "prune_generic_kernel (level by level)"
    return "prune4_lane_kernel<4, %d, false> + <4, 1, true>" % (ppl or 1)


def time_oracle_single_thread_cfg1() -> float:
    """Seconds of one oracle evaluation of config 1 (16 tips, 500 patterns) on ONE host thread."""
    import ctypes
    import oracle
    orc = oracle.Oracle("ld")
    gomp = ctypes.CDLL("libgomp.so.1")
    gomp.omp_get_max_threads.restype = ctypes.c_int
    before = gomp.omp_get_max_threads()
    gomp.omp_set_num_threads(1)
    try:
        prob = W.make_config(1)
        orc.evaluate(prob)
        t0 = time.perf_counter()
        orc.evaluate(prob)
        return time.perf_counter() - t0
    finally:
        gomp.omp_set_num_threads(before)


def bench_incremental(torch, epx, ctx, prob, stream, moves: int = 64) -> dict:
    """Average time of epx_set_node_heights (1 node) + epx_log_likelihood_incremental, which synchronises and returns logL."""
    rng = np.random.default_rng(W.config_seed(2) + 1)
    par = np.asarray(prob.parent)
    h = np.asarray(prob.height, dtype=np.float64).copy()
    kids = [[] for _ in range(prob.n_nodes)]
    for v, p in enumerate(par):
        if p >= 0:
            kids[p].append(v)
    ctx.set_tree(prob.parent, h)
    ctx.log_likelihood()

    def one_move():
        u = int(rng.integers(prob.N, prob.n_nodes))
        lo = max(h[kids[u][0]], h[kids[u][1]])
        hi = h[par[u]] if par[u] >= 0 else h[u] * 1.02
        h[u] = lo + (hi - lo) * rng.uniform(0.1, 0.9)
        ctx.set_node_heights(np.array([u], dtype=np.int32), np.array([h[u]]))
        return ctx.log_likelihood_incremental()
    for _ in range(5):
        one_move()
    n0 = ctx.launch_count()
    t0 = time.perf_counter()
    ms_dev = bracket(torch, stream, one_move, moves) / moves
    ms_wall = (time.perf_counter() - t0) / moves * 1e3
    launches = (ctx.launch_count() - n0) / moves
    lnl_inc = one_move()
    ctx.set_tree(prob.parent, h)                      # full evaluation of the same final state: must agree bit for bit
    lnl_full = ctx.log_likelihood()
    assert lnl_inc == lnl_full, (lnl_inc, lnl_full)
    ctx.set_tree(prob.parent, prob.height)
    ctx.log_likelihood()
    return {"what": "one random internal node moved (epx_set_node_heights) + epx_log_likelihood_incremental, host call to host "
                    "result; bit-identical to a full evaluation", "ms_per_move": ms_dev, "ms_per_move_wall": ms_wall,
            "kernel_launches_per_move": launches, "moves": moves}


def bench_matrices(torch, epx, device: int, K: int, peaks: dict, options=(), label: str = "", sustain_s: float = 0.0) -> dict:
    """Second half of the metric: config 5 (61-state matrix-convolution microbenchmark, a1..a4 only)."""
    prob = W.make_config(5)
    nseg = n_segments(prob)
    fl = chain_flops(prob.K, prob.C, nseg)
    cached = dict(options).get(epx.EPX_OPT_EPOCH_PRODUCTS, 0) == 1
    if cached:
        cf = cached_chain_flops(prob.K, prob.C, prob.M, nseg)
        fl = dict(fl, executed=cf["executed"], table=cf["table"])
    ctx = epx.from_problem(prob, device=device)
    for opt, val in options:
        ctx.set_option(opt, val)
    ctx.set_option(epx.EPX_OPT_STAGE_EVENTS, 1)
    steps = max(3, min(K, 10))
    for _ in range(3):
        ctx.update_matrices()
    assert ctx.status() == 0
    clocks = ClockSampler(device)
    clocks.start()
    n0 = ctx.launch_count()
    ms = bracket(torch, ctx.stream, ctx.update_matrices, steps) / steps
    launches = ctx.launch_count() - n0
    stage = np.zeros(5)
    for _ in range(steps):
        ctx.update_matrices()
        m, _ = ctx.get_stage_ms()
        stage += m
    stage /= steps
    clk = clocks.stop()
    sustained = None
    if not cached and sustain_s > 0:
        # the burst above is ~50 ms of work; a tensor-pipe load held for seconds drops this box's SM clock (MEASURED_PEAKS.json:
        # 1 342 MHz median under a 4 s bf16 matmul), so the same step is also timed back to back for >= sustain_s seconds, with
        # its own clock samples, against a DMMA peak probe that runs as long
        n_s = max(steps, int(np.ceil(sustain_s * 1e3 / ms)))
        cs = ClockSampler(device)
        cs.start()
        ms_s = bracket(torch, ctx.stream, ctx.update_matrices, n_s) / n_s
        clk_s = cs.stop()
        cs = ClockSampler(device)
        cs.start()
        dmma_s = epx.measure_fp64_peak(1, sustain_s * 1e3, device)
        clk_p = cs.stop()
        sustained = {"seconds": ms_s * n_s * 1e-3, "steps": n_s, "ms_per_step": ms_s, "matrices_per_s": prob.n_br * prob.C / (ms_s * 1e-3),
                     "whole_step_useful_tflops": fl["executed"] / (ms_s * 1e-3) / 1e12, "dmma_peak_sustained": dmma_s,
                     "whole_step_frac_of_sustained_peak": fl["executed"] / (ms_s * 1e-3) / 1e12 / dmma_s,
                     "clocks": clk_s, "peak_probe_clocks": clk_p}
    ctx.close()
    dfma, dmma = peaks["dfma"], peaks["dmma"]
    chain_ms = float(stage[2])
    achieved = fl["executed"] / (chain_ms * 1e-3) / 1e12
    n_mat = prob.n_br * prob.C
    kernel = ("epoch_product_table_kernel + chain_dmma64_kernel<1, 4> (a3+a4 fused; chains over >= 2 full epochs multiply by the "
              "tabulated product of those epochs: 3 products per branch at most)" if cached else
              "chain_dmma64_kernel<1, 4> (a3+a4 fused, mma.sync m8n8k4 f64, one product per segment)")
    return {"metric": "epoch branch matrices/s (fp64)" + label, "value": n_mat / (ms * 1e-3), "unit": "matrices/s",
            "ms_per_step": ms, "steps": steps, "gpu_launches": int(launches), "clocks": clk, "sustained": sustained,
            "config": dict(workload_config(prob, 5, 1), segments=int(nseg.sum())),
            "whole_step_useful_tflops": fl["executed"] / (ms * 1e-3) / 1e12,
            "roofline": {"bound": "alu", "kernel": kernel,
                         "achieved": achieved, "peak": dmma, "unit": "TFLOP/s", "frac": achieved / dmma,
                         "traffic": None, "peak_source": "measured in this run by epx_measure_fp64_peak "
                                                         "(register-only DMMA m8n8k4 loop); DFMA peak beside it",
                         "peak_dfma": dfma, "frac_of_dfma": achieved / dfma,
                         "flops_executed_useful": fl["executed"], "flops_straightforward": fl["straightforward"],
                         "output_GBps": n_mat * prob.K * prob.K * 8 / (chain_ms * 1e-3) / 1e9,
                         "stage_ms": {n: float(v) for n, v in zip(epx.STAGE_NAMES, stage)}}}


def bench_other_configs(torch, epx, device: int, K: int, peaks: dict) -> dict:
    """Configs 1, 3 and 4 (BASELINE.json; PAPER.md:L224 names the shapes of 3 and 4) and the 20-state amino-acid workload of
    SURVEY.md 8(f) f3 ("config 6"): whole a1..a6 step on the device, per-stage CUDA-event times, launches.  The pruning kernels of
    configs 3 and 6 (and config 3's chain kernel) get an `alu` roofline against the fp64 peak measured in this run; configs 1
    and 4 are latency-bound: time, tree levels and the dependent-operation chain."""
    out = {}
    clocks = ClockSampler(device)
    clocks.start()
    for cid in (1, 3, 4, 6):
        prob = W.make_config(cid)
        ctx = epx.from_problem(prob, device=device)
        ctx.set_option(epx.EPX_OPT_STAGE_EVENTS, 1)
        lnl = None
        for _ in range(3):
            lnl = ctx.log_likelihood()
        assert ctx.status() == 0 and np.isfinite(lnl)
        steps = max(5, min(K, 50))
        n0 = ctx.launch_count()
        ms = bracket(torch, ctx.stream, ctx.enqueue_log_likelihood, steps) / steps
        launches = (ctx.launch_count() - n0) // steps
        stage = np.zeros(5)
        sl = None
        for _ in range(steps):
            ctx.enqueue_log_likelihood()
            m, sl = ctx.get_stage_ms()
            stage += m
        stage /= steps
        plan = ctx.plan_info()
        alt = None
        if cid == 4:
            # the same step with the asymmetric exponentials by the componentwise-accurate shifted Taylor series instead of Pade 13
            # (EPX_OPT_EXP_METHOD = 2: no Gauss-Jordan solve; north_star names Pade for asymmetric Q, so it stays the default)
            ctx.set_option(epx.EPX_OPT_EXP_METHOD, 2)
            for _ in range(3):
                lnl_alt = ctx.log_likelihood()
            ms_alt = bracket(torch, ctx.stream, ctx.enqueue_log_likelihood, steps) / steps
            ctx.enqueue_log_likelihood()
            m_alt, _ = ctx.get_stage_ms()
            alt = {"exp_method": "componentwise shifted Taylor (EPX_OPT_EXP_METHOD = 2)", "ms_per_step": ms_alt,
                   "chain_ms": float(m_alt[2]), "log_likelihood": lnl_alt}
        ctx.close()
        o = {"config": workload_config(prob, cid, 1), "ms_per_step": ms, "steps": steps, "gpu_launches_per_step": int(launches),
             "log_likelihood": lnl, "stage_ms": {n: float(v) for n, v in zip(epx.STAGE_NAMES, stage)},
             "stage_launches": {n: int(v) for n, v in zip(epx.STAGE_NAMES, sl)}, "plan": plan}
        if alt is not None:
            o["alternative"] = alt
        if cid in (3, 6):
            Kc, C, L, n_int = prob.K, prob.C, prob.L, prob.N - 1
            pf = n_int * C * L * (4 * Kc * Kc + Kc)              # O(K^2 N C L) with both children counted
            prune_ms, chain_ms = float(stage[3]), float(stage[2])
            kp = (Kc + 7) // 8 * 8
            o["roofline_prune"] = {"bound": "alu", "kernel": "prune_mma_kernel<%d> + pb_swizzle_kernel<%d> (a5, %d states padded to %d "
                                                             "on the FP64 tensor pipe)" % (kp, kp, Kc, kp),
                                   "achieved": pf / (prune_ms * 1e-3) / 1e12, "peak": peaks["dmma"], "unit": "TFLOP/s",
                                   "frac": pf / (prune_ms * 1e-3) / 1e12 / peaks["dmma"], "traffic": None, "flops": pf,
                                   "flops_definition": "n_int C L (4 K^2 + K), K = %d (tip children counted like internal ones)" % Kc,
                                   "peak_source": "DMMA m8n8k4 register-only loop measured in this run",
                                   "launches": int(sl[3]), "avg_launch_ms": prune_ms / max(1, int(sl[3]))}
        if cid == 3:
            tf = taylor_chain_flops(prob)
            o["roofline_chain"] = {"bound": "alu", "kernel": "pade_chain_kernel<1> + pade_full_epoch_kernel<1> (a3+a4, "
                                                             "componentwise Taylor exponentials, reading A21)",
                                   "achieved": tf["flops"] / (chain_ms * 1e-3) / 1e12, "peak": peaks["dmma"], "unit": "TFLOP/s",
                                   "frac": tf["flops"] / (chain_ms * 1e-3) / 1e12 / peaks["dmma"], "traffic": None,
                                   "flops": tf["flops"], "dense_products": tf["chain_products"] + tf["table_products"],
                                   "launches": int(sl[2])}
        else:
            o["bound"] = ("latency: %d dependent operations (the largest piece of every tier of the walk, one launch per tier) of %d, %d tree levels"
                          % (plan["largest_piece_ops"] + plan["top_piece_ops"], plan["operations"], plan["levels"])
                          if plan["depth_first"] else "latency: %d tree levels, one launch each" % plan["levels"])
            o["us_per_step"] = ms * 1e3
        out[W.CONFIG_NAMES[cid]] = o
    out["clocks"] = clocks.stop()
    return out




def bench_batch(torch, epx, device: int) -> dict:
    """many independent instances through epx_log_likelihood_batch (every context on its own stream, all
    enqueued before the first fetch) against the same contexts evaluated one after the other.  Host wall clock around
    synchronised calls: the API-level cost a caller sees."""
    import dataclasses
    out = {}
    for label, cid, count in (("8 x config 3 (eight codon data sets, PAPER.md:L157-L161)", 3, 8), ("64 x config 1", 1, 64),
                              ("16 x config 4", 4, 16)):
        base = W.make_config(cid)
        rng = np.random.default_rng(W.config_seed(cid) + 7)
        ctxs = []
        for k in range(count):                           # same shapes, different data per instance
            tips = rng.integers(0, base.K, base.tip_states.shape).astype(np.int32)
            ctxs.append(epx.from_problem(dataclasses.replace(base, tip_states=tips), device=device))
        single = [c.log_likelihood() for c in ctxs]
        for _ in range(3):
            got = epx.log_likelihood_batch(ctxs)
        assert np.array_equal(got, np.array(single))
        reps = 20
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(reps):
            for c in ctxs:
                c.log_likelihood()
        t_seq = (time.perf_counter() - t0) / reps
        t0 = time.perf_counter()
        for _ in range(reps):
            epx.log_likelihood_batch(ctxs)
        t_batch = (time.perf_counter() - t0) / reps
        for c in ctxs:
            c.close()
        out[label] = {"instances": count, "ms_one_after_the_other": t_seq * 1e3, "ms_batch": t_batch * 1e3,
                      "instances_per_s_batch": count / t_batch, "speedup": t_seq / t_batch}
    return out


def parse_opts(text: str):
    """--opt 3=1,6=2 -> [(3, 1), (6, 2)]: EPX_OPT_* overrides for the config-2 context (kernel comparisons, ncu captures)."""
    out = []
    for item in filter(None, text.split(",")):
        k, v = item.split("=")
        out.append((int(k), int(v)))
    return out


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", choices=["cuda", "reference"], default="cuda")
    ap.add_argument("--legs", default="e2e,incremental,matrices,other,batch,cpu",
                    help="optional legs beside the config-2 headline + roofline: e2e, incremental, matrices (config 5), "
                         "other (configs 1, 3, 4, 6), batch (many instances, f4), cpu (oracle on the host cores)")
    ap.add_argument("--no-matrices", action="store_true", help="skip the config-5 matrices/s leg")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip timing the oracle on the host cores")
    ap.add_argument("--opt", type=parse_opts, default=[], help="EPX_OPT overrides for the config-2 context, e.g. 3=2,6=1")
    ap.add_argument("--sustain", type=float, default=2.0,
                    help="seconds of back-to-back config-5 steps (and of the DMMA peak probe) for the sustained matrices/s figure; 0 = skip")
    ap.add_argument("--traffic", type=float, default=None,
                    help="dram bytes per launch of the dominant kernel from the committed ncu capture (profiles/)")
    args = ap.parse_args()
    legs = [x for x in args.legs.split(",") if x]
    if args.no_matrices and "matrices" in legs:
        legs.remove("matrices")
    if args.no_cpu_baseline and "cpu" in legs:
        legs.remove("cpu")
    args.legs = ",".join(legs)
    if args.impl == "reference":
        if args.steps == 100 and args.warmup == 5:
            args.steps, args.warmup = 5, 1
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
