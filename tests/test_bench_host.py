"""Host-side logic of bench.py (no GPU): the algorithmic byte / flop counts, and the N > 1 path -- replicas only, the one
cross-rank exchange is a MAX all-reduce of the device time -- on a world_size-2 gloo group."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_pruning_bytes_formula_matches_a_node_by_node_count():
    import bench
    prob = W.make_config(2, N=37, L=123)
    K, C, L, N = prob.K, prob.C, prob.L, prob.N
    total = 0
    for u in range(N, 2 * N - 1):                       # node-by-node restatement of DESIGN.md section 5
        total += C * L * K * 8 + 4 * L + 2 * C * K * K * 8
        for ch in np.nonzero(prob.parent == u)[0]:
            total += L if ch < N else C * L * K * 8 + 4 * L
    got = bench.pruning_bytes(prob)
    assert got["a5"] == total
    assert got["a6"] == C * L * K * 8 + 4 * L + 16 * L
    assert got["flops"] == (N - 1) * C * L * (4 * K * K + K)


def test_config2_algorithmic_bytes_is_the_surveyed_5_2_GB():
    import bench
    nb = bench.pruning_bytes(W.make_config(2))
    assert 5.1e9 < nb["a5"] + nb["a6"] < 5.4e9          # ~5.20 GB


def test_compulsory_bytes_is_what_the_walk_has_to_move():
    # every node's partials + exponents written once, every tip byte and every matrix read once;
    # for config 2 that is the 2.56 GB of partials + 80 MB of exponents + 20 MB of tips + 2 MB of matrices
    import bench
    prob = W.make_config(2)
    cb = bench.compulsory_bytes(prob)
    assert cb["a5"] == 1999 * (4 * 10000 * 4 * 8 + 4 * 10000 + 2 * 4 * 16 * 8) + 2000 * 10000
    assert 2.6e9 < cb["a5"] < 2.7e9
    assert cb["a5"] < bench.pruning_bytes(prob)["a5"]            # the level model counts each child block a second time


def test_workload_config_is_shared_by_both_arms():
    import bench
    prob = W.make_config(2, N=50, L=64)
    cfg = bench.workload_config(prob, 2, 1)
    assert cfg["workload"] == W.CONFIG_NAMES[2] and cfg["N_tips"] == 50 and cfg["L"] == 64 and "l2" in cfg
    # post-order levels restated with the heights-free definition: longest tip-to-root path in edges
    depth = 0
    for t in range(prob.N):
        d, v = 0, t
        while prob.parent[v] >= 0:
            v = prob.parent[v]; d += 1
        depth = max(depth, d)
    assert cfg["tree_levels"] == depth
    assert bench.workload_config(W.make_config(5, n_br=10), 5, 2)["parallelism"].startswith("replicas x2")


def test_taylor_chain_flop_count_small_case():
    import bench
    prob = W.make_config(3, N=4, L=2)
    tf = bench.taylor_chain_flops(prob)
    nseg = bench.n_segments(prob)
    # at least 6 dense products per exponential, one or two exponentials per (slot, category), n_seg - 1 chain products
    lo = sum((6 * min(int(n), 2) + int(n) - 1) * prob.C for n in nseg if n > 0)
    assert tf["chain_products"] >= lo and tf["table_products"] >= 6 * prob.C * (prob.M - 2)
    assert tf["flops"] == (tf["chain_products"] + tf["table_products"]) * 2 * 61 ** 3


def test_segment_counts_and_chain_flops(orc_ld):
    import bench
    prob = W.make_config(5, n_br=500)
    nseg = bench.n_segments(prob)
    off, _, _ = orc_ld.segments(prob.child_height, prob.parent_height, prob.tau)
    assert np.array_equal(nseg, np.diff(off))
    fl = bench.chain_flops(61, 4, nseg)
    assert fl["executed"] == int(nseg.sum()) * 4 * 2 * 61 ** 3
    assert fl["straightforward"] > fl["executed"]


_WORKER = r"""
import os, sys
sys.path.insert(0, sys.argv[1])
import torch.distributed as dist
import bench
rank = int(os.environ["RANK"])
dist.init_process_group("gloo")
mine = 1.5 if rank == 0 else 2.25                      # rank 1 is the slow replica
ms = bench.max_over_ranks(mine, 2, device="cpu")
val = bench.whole_job_value(1e9, ms, 2)
print(f"RESULT {rank} {ms} {val}", flush=True)
dist.destroy_process_group()
"""


def test_replicas_aggregate_with_gloo_world_size_2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29533", WORLD_SIZE="2")
    procs = [subprocess.Popen([sys.executable, str(script), ROOT], env=dict(env, RANK=str(r)), stdout=subprocess.PIPE,
                              stderr=subprocess.PIPE, text=True) for r in range(2)]
    outs = [p.communicate(timeout=120) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e
    for o, _ in outs:
        line = [x for x in o.splitlines() if x.startswith("RESULT")][0].split()
        assert float(line[2]) == 2.25                                  # max over ranks on every rank
        assert abs(float(line[3]) - 2 * 1e9 / 2.25e-3 / 1e9) < 1e-9    # 2 replicas / slowest time


def test_reference_arm_only_rank0_prints(tmp_path):
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_reference_arm_prints_the_contract_line():
    """`bench.py --impl reference` (the oracle on the host cores, bounded sample): one JSON line with the base contract's keys
    plus impl / cpu_baseline / e2e as the tier rules ask."""
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0"],
                       env=dict(os.environ, RANK="0", WORLD_SIZE="1"), capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr
    lines = [x for x in r.stdout.splitlines() if x.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "impl", "cpu_baseline", "e2e"):
        assert key in d, key
    assert d["impl"] == "reference" and d["dtype"] == "f64" and d["vs_baseline"] is None and d["unit"] == "GB/s"
    assert d["config"]["workload"] == W.CONFIG_NAMES[2]
    import bench
    assert d["config"] == bench.workload_config(W.make_config(2), 2, 1)      # the CUDA arm prints the same dict
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"] and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["value"] > 0


def _stub_line():
    """A JSON line of the shape run_cuda() assembles, with made-up numbers and strings as long as the real ones."""
    import bench
    long = "x" * 150
    clk = {"sm_mhz": 1965.0, "sm_max_mhz": 1965, "reasons": [], "samples": 6, "power_w_max": 480.0}
    stage = {n: 0.1 * (i + 1) for i, n in enumerate(("segment", "eigen", "chain", "prune", "root"))}

    def matrices(ms, cached):
        return {"metric": long, "value": 8e4 / (ms * 1e-3), "unit": "matrices/s", "ms_per_step": ms, "steps": 10, "gpu_launches": 50,
                "clocks": clk, "config": {"workload": long}, "whole_step_useful_tflops": 25.0,
                "sustained": None if cached else {"seconds": 2.01, "steps": 400, "ms_per_step": ms * 1.2, "matrices_per_s": 8e4 / (ms * 1.2e-3),
                                                  "whole_step_useful_tflops": 21.0, "dmma_peak_sustained": 30.0,
                                                  "whole_step_frac_of_sustained_peak": 0.7, "clocks": dict(clk, reasons=["sw_power_cap"]),
                                                  "peak_probe_clocks": clk},
                "roofline": {"bound": "alu", "kernel": long, "achieved": 26.9, "peak": 37.05, "unit": "TFLOP/s", "frac": 0.726,
                             "traffic": None, "peak_source": long, "stage_ms": dict(stage, chain=ms * 0.94, eigen=0.246)}}

    def other(cid, K, rf):
        o = {"config": {"workload": long}, "ms_per_step": 0.4, "steps": 20, "gpu_launches_per_step": 20, "log_likelihood": -1.0,
             "stage_ms": stage, "stage_launches": {n: 1 for n in stage},
             "plan": {"levels": 17, "operations": 199, "depth_first": 0, "bottom_pieces": 0, "largest_piece_ops": 0, "top_piece_ops": 0,
                      "stack_slots": 0, "prune_launches": 18}}
        for leg in rf:
            o["roofline_" + leg] = {"bound": "alu", "kernel": long, "achieved": 12.6, "peak": 37.05, "unit": "TFLOP/s", "frac": 0.34,
                                    "traffic": None, "flops": 2.5e9, "flops_definition": long, "peak_source": long, "launches": 18,
                                    "avg_launch_ms": 0.011}
        if not rf:
            o["bound"] = long; o["us_per_step"] = 400.0
        if cid == 4:
            o["alternative"] = {"exp_method": long, "ms_per_step": 0.3, "chain_ms": 0.1, "log_likelihood": -1.0}
        return o

    line = {"metric": bench.METRIC, "value": 5139.0, "unit": "GB/s", "n_gpus": 1, "steps": 20, "warmup": 5, "ms_per_step": 0.5178,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": long}, "value_definition": long, "workspace_bytes": 1, "plan": {},
            "roofline": {"bound": "hbm", "kernel": long, "achieved": 5559.0, "peak": 6517.6, "unit": "GB/s", "frac": 0.853, "traffic": 1.3e9,
                         "stage_ms": stage},
            "gpu_launches": 100, "clocks": clk, "log_likelihood": -1.0,
            "e2e": {"value": 2000.0, "unit": "GB/s", "h2d_bytes_per_step": 1, "d2h_bytes_per_step": 12, "ms_per_step": 1.18, "what": long},
            "incremental": {"ms_per_move": 0.105, "what": long},
            "matrices": matrices(5.02, False), "matrices_cached": matrices(3.53, True),
            "other_configs": {W.CONFIG_NAMES[1]: other(1, 4, ()), W.CONFIG_NAMES[3]: other(3, 61, ("prune", "chain")),
                              W.CONFIG_NAMES[4]: other(4, 24, ()), W.CONFIG_NAMES[6]: other(6, 20, ("prune",)), "clocks": clk},
            "batch": {long: {"instances": 8, "speedup": 1.3}},
            "cpu_baseline": {"value": 5.1, "unit": "GB/s", "cores": 16, "kind": "oracle", "sample": long * 2}}
    return line


def test_second_half_of_the_metric_stays_in_what_the_driver_keeps():
    """The driver's record keeps `roofline` (scalars) and the last ~1 500 characters of the line.  Config 5's matrices/s and
    tensor-peak fraction (the second half of BASELINE.json's metric), its sustained figure, and the rooflines of configs 3
    and 6 must therefore sit inside `roofline` as flat scalars AND inside a trailing `summary` of at most 1 200 characters."""
    import bench
    out = bench.finalise_line(_stub_line())
    text = json.dumps(out)
    assert list(out.keys())[-1] == "summary" and len(json.dumps(out["summary"])) <= 1200
    tail = text[-1500:]
    need = ("cfg5_ms", "cfg5_Mmat_per_s", "cfg5_chain_ms", "cfg5_chain_tflops", "cfg5_dmma_peak", "cfg5_chain_frac", "cfg5_eigen_ms",
            "cfg5_sm_mhz", "cfg5_sus_ms", "cfg5_sus_Mmat_per_s", "cfg5_sus_frac", "cfg5_sus_sm_mhz", "cfg5c_ms", "cfg5c_Mmat_per_s",
            "cfg5c_chain_frac", "cfg3_prune_ms", "cfg3_prune_frac", "cfg3_chain_ms", "cfg3_chain_frac", "cfg6_prune_ms",
            "cfg6_prune_frac", "cfg6_prune_launches", "cfg1_ms", "cfg4_ms", "cfg4_dep_ops", "inc_ms_per_move", "cfg5_sus_reasons")
    for k in need:
        assert k in out["roofline"], k
        assert not isinstance(out["roofline"][k], (dict, list)), k
        assert '"%s":' % k in tail, k
    assert out["roofline"]["cfg5_Mmat_per_s"] == pytest.approx(8e4 / 5.02e-3 / 1e6, rel=1e-3)
    assert out["summary"]["cfg2_prune_frac"] == pytest.approx(0.853)
    # the full objects are still there, untouched
    assert out["matrices"] == _stub_line()["matrices"] and out["roofline"]["frac"] == 0.853
    # a line without the optional legs still finalises
    bare = {k: v for k, v in _stub_line().items() if k not in ("matrices", "matrices_cached", "other_configs", "incremental", "e2e")}
    assert "cfg5_ms" not in bench.finalise_line(bare)["summary"]


def test_ncu_traffic_constant_is_the_number_in_the_profile_it_names():
    """bench.py's NCU_TRAFFIC (bytes per step of the pruning launches) is a constant taken from a committed ncu capture: it must
    be the figure that profile states, so that a re-capture that forgets one of the two cannot go unnoticed."""
    import re
    import bench
    text = open(os.path.join(ROOT, bench.NCU_TRAFFIC["profile"])).read()
    m = re.findall(r"DRAM bytes per step = \*\*([0-9 \u00a0\u202f.]+) MB\*\*", text)
    assert m, "the profile no longer states 'DRAM bytes per step = **... MB**'"
    mb = float(re.sub(r"[^0-9.]", "", m[-1]))
    assert abs(mb * 1e6 - bench.NCU_TRAFFIC["bytes_per_step"]) <= 1e-4 * bench.NCU_TRAFFIC["bytes_per_step"]
    assert bench.NCU_TRAFFIC["kernel"].split("<")[0] in text
