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
