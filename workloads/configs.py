"""The five BASELINE.json workloads as seeded generators, plus reduced-size variants of the same recipe.

The paper's own workloads (H3N2, 522 taxa, K=7, 13 epochs; HIV patient 3, 109 taxa,
516 sites, K=61, 2 epochs) are empirical data sets that are not available; these synthetic inputs have
their shapes (dated-tip coalescent trees, HKY/GY94/discrete-trait Q, 2..24 epochs) and stand in for them.
Recipe and the readings of BASELINE.json's gaps: DESIGN.md "Input recipe".
"""
from __future__ import annotations

import numpy as np

from . import models, trees
from .problem import EpochProblem

CONFIG_NAMES = {
    1: "cfg1_gtr4_2epoch_16tips_500pat",
    2: "cfg2_hky4_10epoch_2000tips_10000pat",
    3: "cfg3_gy94_61_3epoch_100tips_1000pat",
    4: "cfg4_trait24_asym_24epoch_1500tips_1pat",
    5: "cfg5_conv61_16epoch_20000branches",
    6: "cfg6_aa20_3epoch_200tips_2000pat",      # not in BASELINE.json: SURVEY.md 8(f) f3, the 20-state amino-acid workload
}


def config_seed(config_id: int) -> int:
    return 13093075 * 10 + config_id


def _streams(config_id: int):
    ss = np.random.SeedSequence(config_seed(config_id))
    return [np.random.default_rng(s) for s in ss.spawn(4)]  # tree, models, tips, weights


def _gy94_epoch(rng, omega, kappa=2.0):
    pos = rng.dirichlet(np.full(4, 5.0), size=3)
    pi = models.f3x4(pos)
    return models.gy94(omega, kappa, pi), pi


def make_config(config_id: int, *, N: int | None = None, L: int | None = None,
                n_br: int | None = None) -> EpochProblem:
    """Build config `config_id` (1..5 = BASELINE.json; 6 = the 20-state workload of SURVEY.md 8(f) f3). N / L / n_br override the
    size (same recipe, same seed) for tests."""
    r_tree, r_model, r_tips, r_wt = _streams(config_id)
    if config_id == 1:
        K, M, C = 4, 2, 4
        N = 16 if N is None else N
        L = 500 if L is None else L
        parent, height = trees.coalescent(r_tree, np.zeros(N))
        height = height / height.max()
        height[np.argmax(height)] = 1.0
        tau = np.array([0.5])
        Q = np.zeros((M, K, K)); F = np.zeros((M, K))
        for e in range(M):
            exch = r_model.gamma(1.0, 1.0, size=6)
            F[e] = r_model.dirichlet(np.ones(4))
            Q[e] = models.gtr(exch, F[e])
        rates, weights = models.discrete_gamma(0.5, C)
        tips = r_tips.integers(0, K, size=(N, L)).astype(np.int32)
        wt = np.ones(L)
        return EpochProblem(CONFIG_NAMES[1], K, M, C, N, L, tau, Q, F, True, rates, weights,
                            parent=parent, height=height, tip_states=tips, pattern_weights=wt)
    if config_id == 2:
        K, M, C = 4, 10, 4
        N = 2000 if N is None else N
        L = 10000 if L is None else L
        tip_h = r_tree.uniform(0.0, 0.2, size=N)
        tip_h[np.argmin(tip_h)] = 0.0
        parent, height = trees.coalescent(r_tree, tip_h, ne=0.5)
        height = trees.stretch_above(height, 0.2, 1.0)
        tau = np.arange(1, M) / M
        Q = np.zeros((M, K, K)); F = np.zeros((M, K))
        for e in range(M):
            kappa = r_model.lognormal(1.0, 0.5)
            F[e] = r_model.dirichlet(np.full(4, 2.0))
            Q[e] = models.hky(kappa, F[e])
        rates, weights = models.discrete_gamma(0.3, C)
        tips = r_tips.integers(0, K, size=(N, L)).astype(np.int32)
        wt = (r_wt.poisson(3.0, size=L) + 1).astype(np.float64)
        return EpochProblem(CONFIG_NAMES[2], K, M, C, N, L, tau, Q, F, True, rates, weights,
                            parent=parent, height=height, tip_states=tips, pattern_weights=wt)
    if config_id == 3:
        K, M, C = 61, 3, 4
        N = 100 if N is None else N
        L = 1000 if L is None else L
        parent, height = trees.coalescent(r_tree, np.zeros(N))
        height = height / height.max()
        height[np.argmax(height)] = 1.0
        tau = np.array([1.0 / 3.0, 2.0 / 3.0])
        omegas = [0.2, 1.0, 2.5]        # epoch 0 = most recent ... epoch 2 = oldest
        Q = np.zeros((M, K, K)); F = np.zeros((M, K))
        for e in range(M):
            Q[e], F[e] = _gy94_epoch(r_model, omegas[e])
        rates, weights = models.discrete_gamma(1.0, C)
        tips = r_tips.integers(0, K, size=(N, L)).astype(np.int32)
        wt = np.ones(L)
        return EpochProblem(CONFIG_NAMES[3], K, M, C, N, L, tau, Q, F, True, rates, weights,
                            parent=parent, height=height, tip_states=tips, pattern_weights=wt)
    if config_id == 4:
        K, M, C = 24, 24, 1
        N = 1500 if N is None else N
        L = 1 if L is None else L
        tip_h = r_tree.uniform(0.0, 10.0, size=N)
        tip_h[np.argmin(tip_h)] = 0.0
        parent, height = trees.coalescent(r_tree, tip_h, ne=1.0)
        height = trees.stretch_above(height, 10.0, 12.0)
        tau = 0.5 * np.arange(1, M)
        regimes = [models.asymmetric_trait(r_model, K), models.asymmetric_trait(r_model, K)]
        stat = [models.stationary(q) for q in regimes]
        Q = np.stack([regimes[e % 2] for e in range(M)])
        F = np.stack([stat[e % 2] for e in range(M)])
        root_epoch = int(np.sum(tau < height.max()))
        rates, weights = np.ones(1), np.ones(1)
        tips = r_tips.integers(0, K, size=(N, L)).astype(np.int32)
        wt = np.ones(L)
        return EpochProblem(CONFIG_NAMES[4], K, M, C, N, L, tau, Q, F, False, rates, weights,
                            parent=parent, height=height, tip_states=tips, pattern_weights=wt,
                            root_freqs=F[root_epoch].copy())
    if config_id == 5:
        K, M, C = 61, 16, 4
        n_br = 20000 if n_br is None else n_br
        tau = np.sort(r_tree.uniform(0.0, 1.0, size=M - 1))
        child = r_tree.uniform(0.0, 1.0, size=n_br)
        par = np.minimum(child + r_tree.exponential(0.25, size=n_br), 1.0)
        Q = np.zeros((M, K, K)); F = np.zeros((M, K))
        for e in range(M):
            omega = r_model.lognormal(0.0, 0.7)
            Q[e], F[e] = _gy94_epoch(r_model, omega)
        rates, weights = models.discrete_gamma(1.0, C)
        return EpochProblem(CONFIG_NAMES[5], K, M, C, 0, 0, tau, Q, F, True, rates, weights,
                            child_height=child, parent_height=par)
    if config_id == 6:
        # SURVEY.md 8(f) f3 / north_star "tiles for 20-61-state": an amino-acid shaped workload (PAPER.md:L26 finite state
        # spaces).  Reversible GTR-like Q per epoch: 190 exchangeabilities ~ Gamma(1,1), pi ~ Dirichlet(5,...,5) (empirical
        # amino-acid frequencies span about one decade), normalised; 3 epochs at thirds of the root height; 4 gamma
        # categories (alpha = 0.7); 200 tips from a serially-sampled coalescent (tip dates over 20 % of the root height);
        # 2 000 site patterns, tips uniform over the 20 states with 2 % missing, weights Poisson(2) + 1.
        K, M, C = 20, 3, 4
        N = 200 if N is None else N
        L = 2000 if L is None else L
        tip_h = r_tree.uniform(0.0, 0.2, size=N)
        tip_h[np.argmin(tip_h)] = 0.0
        parent, height = trees.coalescent(r_tree, tip_h, ne=0.5)
        height = trees.stretch_above(height, 0.2, 1.0)
        tau = np.array([1.0 / 3.0, 2.0 / 3.0])
        Q = np.zeros((M, K, K)); F = np.zeros((M, K))
        for e in range(M):
            F[e] = r_model.dirichlet(np.full(K, 5.0))
            Q[e] = models.gtr_k(r_model.gamma(1.0, 1.0, size=K * (K - 1) // 2), F[e])
        rates, weights = models.discrete_gamma(0.7, C)
        tips = r_tips.integers(0, K, size=(N, L)).astype(np.int32)
        tips[r_tips.random((N, L)) < 0.02] = -1
        wt = (r_wt.poisson(2.0, size=L) + 1).astype(np.float64)
        return EpochProblem(CONFIG_NAMES[6], K, M, C, N, L, tau, Q, F, True, rates, weights,
                            parent=parent, height=height, tip_states=tips, pattern_weights=wt)
    raise ValueError(f"unknown config {config_id}")
