"""Stored long-double oracle values (tests/golden/oracle_values.txt, written by tests/golden/make_golden.py from oracle/
only).  CPU: the oracle still reproduces them (a change of the oracle's arithmetic must be deliberate).  GPU: the CUDA
path matches them to the north_star tolerance without the oracle in the loop."""
import os

import numpy as np
import pytest

import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))
CASES = {"cfg1": (1, {}), "cfg2_N150_L777": (2, {"N": 150, "L": 777}), "cfg2": (2, {}), "cfg3_N12_L70": (3, {"N": 12, "L": 70}),
         "cfg3": (3, {}), "cfg4_N60_L3": (4, {"N": 60, "L": 3}), "cfg4": (4, {}), "cfg6_N30_L100": (6, {"N": 30, "L": 100}),
         "cfg6": (6, {})}


def golden():
    out = {}
    for line in open(os.path.join(HERE, "golden", "oracle_values.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, kind, value = line.split()
        out[(name, kind)] = np.longdouble(value)
    return out


@pytest.mark.parametrize("name", ["cfg1", "cfg2_N150_L777", "cfg3_N12_L70", "cfg4_N60_L3", "cfg6_N30_L100"])
def test_oracle_reproduces_golden(orc_ld, name):
    g = golden()
    cid, kw = CASES[name]
    ref = orc_ld.evaluate(W.make_config(cid, **kw))
    assert abs(ref["lnl"] - g[(name, "logL")]) <= 1e-15 * abs(g[(name, "logL")])
    assert abs(ref["P"].sum(dtype=np.longdouble) - g[(name, "sumP")]) <= 1e-15 * abs(g[(name, "sumP")])
    assert int(ref["seg_off"][-1]) == int(g[(name, "n_segments")])


@pytest.mark.gpu
@pytest.mark.parametrize("name", list(CASES))
def test_cuda_matches_golden_loglik(name):
    import paper_1309_3075_b200 as epx
    g = golden()
    cid, kw = CASES[name]
    prob = W.make_config(cid, **kw)
    ctx = epx.from_problem(prob)
    lnl = ctx.log_likelihood()
    want = g[(name, "logL")]
    assert abs(np.longdouble(lnl) - want) <= 1e-9 * abs(want)
    off, _, _ = ctx.get_all_segments()
    assert int(off[-1]) == int(g[(name, "n_segments")])
    P = ctx.get_all_matrices()
    assert abs(np.longdouble(P.sum()) - g[(name, "sumP")]) <= 1e-9     # every row of every P sums to 1
    assert ctx.status() == 0
    ctx.close()


@pytest.mark.gpu
def test_cuda_matches_golden_config5_sample():
    import paper_1309_3075_b200 as epx
    g = golden()
    prob = W.make_config(5)
    ctx = epx.from_problem(prob)
    ctx.update_matrices()
    off, _, _ = ctx.get_all_segments()
    assert int(off[-1]) == int(g[("cfg5", "n_segments")])
    P = ctx.get_all_matrices()[np.arange(0, prob.n_br, 997)]
    w = np.cos(np.arange(P.size, dtype=np.float64)).reshape(P.shape)
    got = (P.astype(np.longdouble) * w).sum(dtype=np.longdouble)
    assert abs(got - g[("cfg5_every997", "wsumP")]) <= 1e-12 * P.size ** 0.5 * 10     # 1e-12 per entry, random-sign sum
    ctx.close()
