"""Per-stage device times of BASELINE.json configs 1, 3 and 4 (the configs bench.py does not time), through the public binding.

    python -m paper_1309_3075_b200.examples.other_configs [steps]

Prints one line per config: log-likelihood, CUDA-event time of each stage (EPX_OPT_STAGE_EVENTS), launches per stage."""
import sys

import numpy as np


def main(steps: int = 10) -> None:
    import workloads as W
    import paper_1309_3075_b200 as epx
    for cid in (1, 3, 4):
        prob = W.make_config(cid)
        ctx = epx.from_problem(prob)
        ctx.set_option(epx.EPX_OPT_STAGE_EVENTS, 1)
        for _ in range(3):
            lnl = ctx.log_likelihood()
        acc = np.zeros(5)
        for _ in range(steps):
            ctx.enqueue_log_likelihood()
            ms, launches = ctx.get_stage_ms()
            acc += ms
        acc /= steps
        print(f"{prob.name}: logL={lnl:.9f} step={acc.sum():.4f} ms " +
              " ".join(f"{n}={v:.4f}" for n, v in zip(epx.STAGE_NAMES, acc)) + f" launches={launches.tolist()} levels={ctx.tree_levels()}",
              flush=True)
        ctx.close()


if __name__ == "__main__":
    import os
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
    main(int(sys.argv[1]) if len(sys.argv) > 1 else 10)
