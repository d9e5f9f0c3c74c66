"""Writes tests/golden/oracle_values.txt: results of the long-double CPU oracle on the seeded workloads.

Calls only `oracle/` and the input generators in `workloads/` -- never the CUDA path.  Run from the repo root:
    python tests/golden/make_golden.py
Config 2 at full size takes about a minute.  The paper prints no worked numeric example, so these are
regression values of the pinned oracle, not paper values; each line says what it is.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402
import workloads as W  # noqa: E402

CASES = [("cfg1", 1, {}), ("cfg2_N150_L777", 2, {"N": 150, "L": 777}), ("cfg2", 2, {}), ("cfg3_N12_L70", 3, {"N": 12, "L": 70}),
         ("cfg3", 3, {}), ("cfg4_N60_L3", 4, {"N": 60, "L": 3}), ("cfg4", 4, {}), ("cfg6_N30_L100", 6, {"N": 30, "L": 100}), ("cfg6", 6, {})]


def main():
    orc = oracle.Oracle("ld")
    lines = ["# name kind value      (long-double oracle, PAPER.md Eq. 3-7 + L72; written by make_golden.py)"]
    for name, cid, kw in CASES:
        prob = W.make_config(cid, **kw)
        ref = orc.evaluate(prob)
        lines.append(f"{name} logL {np.format_float_scientific(ref['lnl'], precision=20, unique=False)}")
        lines.append(f"{name} sumP {np.format_float_scientific(ref['P'].sum(dtype=np.longdouble), precision=20, unique=False)}")
        lines.append(f"{name} n_segments {int(ref['seg_off'][-1])}")
    prob = W.make_config(5)
    sample = np.arange(0, prob.n_br, 997)
    ref = orc.evaluate(prob, branches=sample)
    w = np.cos(np.arange(ref["P"].size, dtype=np.float64)).reshape(ref["P"].shape)      # position-sensitive checksum
    lines.append(f"cfg5_every997 wsumP {np.format_float_scientific((ref['P'] * w).sum(dtype=np.longdouble), precision=20, unique=False)}")
    off, _, _ = orc.segments(prob.child_height, prob.parent_height, prob.tau)
    lines.append(f"cfg5 n_segments {int(off[-1])}")
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_values.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")
    print("\n".join(lines))


if __name__ == "__main__":
    main()
