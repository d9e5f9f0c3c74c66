"""GPU parity on the degenerate and edge cases of the method (through the C ABI, against the long-double oracle):
odd state counts on every kernel family, a single epoch, boundaries outside the tree, zero-length branches, all tips
missing, relabelled trees, an overridden root distribution, and re-evaluation after inputs change (the MCMC use of the
library: the cached CUDA graph and the dirty-upload logic must not serve stale data)."""
import dataclasses

import numpy as np
import pytest

import workloads as W
from workloads import models, trees

from test_gpu_parity import run_tree, check_matrices, check_segments, P_TOL, LNL_RTOL
from test_oracle_pins import _small_problem

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def epx():
    import torch
    assert torch.cuda.is_available()
    import paper_1309_3075_b200 as m
    m.lib()
    return m


@pytest.mark.parametrize("K,C,L,reversible", [(2, 1, 5, True), (7, 3, 45, True), (24, 2, 33, True), (33, 1, 40, True),
                                              (34, 2, 11, True), (40, 3, 45, True), (62, 1, 9, True), (64, 2, 37, True),
                                              (7, 2, 9, False), (20, 1, 3, False)])
def test_state_counts_across_kernel_families(epx, orc_ld, K, C, L, reversible):
    # K = 2, 7, 24: generic shared-memory kernels; 33 .. 64: DMMA chain + DMMA pruning with padding columns; 33 .. 62 take the
    # cluster Jacobi (odd K: a dummy player; 62: the largest it serves), 64 round 1's kernel;
    # asymmetric: Pade.  L is never a multiple of the pattern tile; some tips are missing.
    rng = np.random.default_rng(1000 + K)
    prob = _small_problem(rng, K=K, M=4, C=C, N=9, L=L, reversible=reversible, tip_h=rng.uniform(0, 0.3, 9))
    tips = prob.tip_states.copy()
    tips[::2, ::5] = -1
    prob = dataclasses.replace(prob, tip_states=tips)
    if not reversible:
        prob = dataclasses.replace(prob, root_freqs=prob.freqs[-1].copy())
    run_tree(epx, orc_ld, prob)
    run_tree(epx, orc_ld, prob, options=[(epx.EPX_OPT_CHAIN_KERNEL, 1), (epx.EPX_OPT_PRUNE_KERNEL, 1)])


@pytest.mark.parametrize("K,C,L,reversible", [(24, 1, 5, False), (24, 3, 7, True), (9, 3, 4, True), (16, 1, 2, True), (31, 2, 3, True)])
def test_few_pattern_walk_instances(epx, orc_ld, K, C, L, reversible):
    # pruneK_dfs_kernel (L C <= 64, N >= 8): the compile-time instances K = 24 with C = 1 / runtime C, the generic ones,
    # matrices staged by TMA bulk copies (C K^2 even) and by cp.async (K = 9, C = 3: odd), several pieces + a top piece;
    # every node's partials against the oracle, then the level kernels on the same problem
    rng = np.random.default_rng(2000 + 10 * K + C)
    prob = _small_problem(rng, K=K, M=3, C=C, N=41, L=L, reversible=reversible, tip_h=rng.uniform(0, 0.2, 41))
    tips = prob.tip_states.copy()
    tips[::7, 0] = -1
    prob = dataclasses.replace(prob, tip_states=tips)
    if not reversible:
        prob = dataclasses.replace(prob, root_freqs=prob.freqs[-1].copy())
    # (reversible models: componentwise exponential, so that every node's partials meet the RELATIVE bound -- DESIGN.md A21)
    exp_opt = [(epx.EPX_OPT_EXP_METHOD, 2)] if reversible else []
    lnl, _ = run_tree(epx, orc_ld, prob, options=exp_opt)
    info = epx.from_problem(prob).plan_info()
    assert info["depth_first"] == 1 and info["bottom_pieces"] >= 2
    lnl_level, _ = run_tree(epx, orc_ld, prob, options=exp_opt + [(epx.EPX_OPT_PRUNE_KERNEL, 1)])
    assert lnl == lnl_level                  # same summation order: bit-identical


def test_set_tree_same_topology_fast_path(epx, orc_ld):
    # epx_set_tree with an unchanged parent array keeps the pruning plans and the CUDA graphs and only replaces the heights:
    # the result must be that of a fresh context, bad heights must be rejected and leave the context usable
    prob = W.make_config(2, N=60, L=70)
    ctx = epx.from_problem(prob)
    ctx.log_likelihood()
    rng = np.random.default_rng(3)
    h2 = prob.height.copy()
    h2[prob.N:] *= 1.0 + 0.05 * rng.random(prob.n_nodes - prob.N).cumsum() / (prob.n_nodes - prob.N)   # monotone stretch: order kept
    order_ok = all(h2[prob.parent[i]] >= h2[i] for i in range(prob.n_nodes) if prob.parent[i] >= 0)
    assert order_ok
    ctx.set_tree(prob.parent, h2)
    lnl = ctx.log_likelihood_incremental()          # no complete evaluation of these heights: falls back to a full one
    prob2 = dataclasses.replace(prob, height=h2)
    fresh = epx.from_problem(prob2)
    assert lnl == fresh.log_likelihood()
    ref = orc_ld.evaluate(prob2)
    assert abs(np.longdouble(lnl) - ref["lnl"]) <= LNL_RTOL * abs(ref["lnl"])
    bad = h2.copy()
    bad[prob.N] = h2.max() + 1.0                    # an internal node above the root
    with pytest.raises(Exception):
        ctx.set_tree(prob.parent, bad)
    assert ctx.log_likelihood() == lnl              # the old tree is still in place
    ctx.close(); fresh.close()


def test_single_epoch_and_boundaries_outside_the_tree(epx, orc_ld):
    rng = np.random.default_rng(7)
    one = _small_problem(rng, K=4, M=1, C=2, N=10, L=50)                    # M = 1: no boundary at all (homogeneous model)
    lnl_one, _ = run_tree(epx, orc_ld, one)
    # the same model with two unused boundaries (one below every node, one above the root): same answer (reading A4)
    three = dataclasses.replace(one, M=3, tau=np.array([-0.5, 2.0]), Q=np.repeat(one.Q, 3, 0), freqs=np.repeat(one.freqs, 3, 0))
    lnl_three, ref = run_tree(epx, orc_ld, three)
    assert abs(lnl_one - lnl_three) <= 1e-12 * abs(lnl_one)
    assert np.all(np.diff(ref["seg_off"]) <= 1)


def test_zero_length_branches_and_nodes_on_boundaries(epx, orc_ld):
    # ((0,1)4, 2)5, 3)6 with node 4, node 5 and tip 2 all at height 0.25 = the first boundary: the branches 4->5 and 2->5
    # have length zero (no segment, P = I, reading A3) and sit exactly on a boundary
    rng = np.random.default_rng(8)
    base = _small_problem(rng, K=4, M=3, C=2, N=4, L=20, tau=[0.25, 0.5])
    parent = np.array([4, 4, 5, 6, 5, 6, -1], dtype=np.int32)
    height = np.array([0.0, 0.0, 0.25, 0.0, 0.25, 0.25, 1.0])
    prob = dataclasses.replace(base, parent=parent, height=height)
    lnl, ref = run_tree(epx, orc_ld, prob)
    nseg = np.diff(ref["seg_off"])
    assert nseg[2] == 0 and nseg[4] == 0 and nseg[6] == 0          # tip 2, node 4, root slot
    assert nseg[0] == 1 and nseg[5] == 2                           # [0, 0.25) is one epoch; 0.25 -> 1.0 is epochs 2 and 1 (a node ON a boundary starts the older epoch)
    ctx = epx.from_problem(prob)
    ctx.update_matrices()
    assert np.array_equal(ctx.get_matrix(4, 1), np.eye(4))
    ctx.close()


def test_all_tips_missing_gives_zero(epx, orc_ld):
    prob = W.make_config(2, N=64, L=100)
    prob = dataclasses.replace(prob, tip_states=np.full_like(prob.tip_states, -1))
    ctx = epx.from_problem(prob)
    lnl = ctx.log_likelihood()
    assert abs(lnl) < 1e-9                              # every site likelihood is 1 (rows of P sum to 1); exercises the rescaling
    assert ctx.status() == 0
    ctx.close()


def test_relabelled_tree_and_root_override(epx, orc_ld):
    rng = np.random.default_rng(9)
    prob = W.make_config(1, N=20, L=64)
    lnl0, _ = run_tree(epx, orc_ld, prob)
    parent, height = trees.relabel_internal(rng, prob.parent, prob.height)      # the root is no longer the last node
    lnl1, _ = run_tree(epx, orc_ld, dataclasses.replace(prob, parent=parent, height=height))
    assert abs(lnl0 - lnl1) <= 1e-12 * abs(lnl0)
    rf = rng.dirichlet(np.ones(4))
    run_tree(epx, orc_ld, dataclasses.replace(prob, root_freqs=rf))


def test_reevaluation_after_inputs_change(epx, orc_ld):
    """One context, many evaluations: heights, models, rates, tips, weights, then the topology change; after each change
    the result must equal a fresh oracle evaluation (no stale graph, no stale upload)."""
    rng = np.random.default_rng(10)
    prob = W.make_config(2, N=60, L=300)
    ctx = epx.from_problem(prob)

    def check(p):
        lnl = ctx.log_likelihood()
        ref = orc_ld.evaluate(p)
        assert abs(np.longdouble(lnl) - ref["lnl"]) <= LNL_RTOL * abs(ref["lnl"])
        check_segments(ctx, ref)
        check_matrices(ctx, ref)
        assert ctx.status() == 0

    check(prob)
    # 1. node heights move (same topology: the cached graph is replayed)
    h = prob.height.copy()
    internal = h > 0.2
    h[internal] = 0.2 + (h[internal] - 0.2) * 0.9
    prob = dataclasses.replace(prob, height=h)
    ctx.set_tree(prob.parent, prob.height)
    check(prob)
    # 2. one epoch's model changes
    pi = rng.dirichlet(np.full(4, 3.0))
    Q, F = prob.Q.copy(), prob.freqs.copy()
    Q[3], F[3] = models.hky(4.2, pi), pi
    prob = dataclasses.replace(prob, Q=Q, freqs=F)
    ctx.set_epoch_model(3, Q[3], F[3], True)
    check(prob)
    # 3. boundaries and category rates
    prob = dataclasses.replace(prob, tau=prob.tau * 0.95)
    ctx.set_epoch_boundaries(prob.tau)
    rates, weights = models.discrete_gamma(0.9, 4)
    prob = dataclasses.replace(prob, rates=rates, weights=weights)
    ctx.set_category_rates(rates, weights)
    check(prob)
    # 4. tips and pattern weights
    tips = prob.tip_states.copy(); tips[:, ::3] = (tips[:, ::3] + 1) % 4
    wt = rng.poisson(2.0, prob.L) + 1.0
    prob = dataclasses.replace(prob, tip_states=tips, pattern_weights=wt)
    ctx.set_tip_states(tips); ctx.set_pattern_weights(wt)
    check(prob)
    # 5. a different topology (graph must be rebuilt)
    parent, height = trees.coalescent(rng, np.sort(rng.uniform(0, 0.2, prob.N)))
    height = trees.stretch_above(height, 0.2, 1.0)
    prob = dataclasses.replace(prob, parent=parent, height=height)
    ctx.set_tree(parent, height)
    check(prob)
    ctx.close()


@pytest.mark.parametrize("cid,kw", [(2, {"N": 60, "L": 100}), (3, {"N": 8, "L": 24}), (4, {"N": 40, "L": 2}), (5, {"n_br": 150})])
def test_shared_processes(epx, orc_ld, cid, kw):
    """f2 (PAPER.md L78 phi_m): epochs with identical (Q, freqs) share one eigensystem / one full-epoch exponential.  Parity with
    the oracle (which knows nothing of the sharing), and bit-identical to computing one per epoch."""
    prob = W.make_config(cid, **kw)
    Q, F = prob.Q.copy(), prob.freqs.copy()
    for e in range(2, prob.M):                          # three processes at most: epochs 2.. repeat the first two
        Q[e], F[e] = Q[e % 2], F[e % 2]
    prob = dataclasses.replace(prob, Q=Q, freqs=F)
    if prob.root_freqs is not None:
        prob = dataclasses.replace(prob, root_freqs=F[int(np.sum(prob.tau < prob.height.max()))].copy())
    outs = []
    for share in (1, 0):
        ctx = epx.from_problem(prob)
        ctx.set_option(epx.EPX_OPT_SHARE_PROCESSES, share)
        phi, S = ctx.epoch_processes()
        assert S == (min(2, prob.M) if share else prob.M)
        if prob.N:
            lnl = ctx.log_likelihood()
        else:
            ctx.update_matrices(); lnl = 0.0
        assert ctx.status() == 0
        outs.append((lnl, ctx.get_all_matrices()))
        ctx.close()
    assert outs[0][0] == outs[1][0] and np.array_equal(outs[0][1], outs[1][1])
    ref = orc_ld.evaluate(prob)
    assert np.max(np.abs(outs[0][1].astype(np.longdouble) - ref["P"])) <= P_TOL
    if prob.N:
        assert abs(np.longdouble(outs[0][0]) - ref["lnl"]) <= LNL_RTOL * abs(ref["lnl"])


def test_stage_events_and_launch_count(epx):
    prob = W.make_config(1)
    ctx = epx.from_problem(prob)
    with pytest.raises(epx.EpxError):
        ctx.get_stage_ms()                               # option off
    ctx.set_option(epx.EPX_OPT_STAGE_EVENTS, 1)
    n0 = ctx.launch_count()
    ctx.log_likelihood()
    ms, launches = ctx.get_stage_ms()
    assert np.all(ms >= 0) and ms[3] > 0 and launches.sum() == ctx.launch_count() - n0
    assert launches[0] == 1 and launches[4] == 0          # small problem: fused segmenter; K = 4: the root reduction runs inside the walk
    ctx.set_option(epx.EPX_OPT_PRUNE_KERNEL, 2)           # level kernels: a root kernel of its own (last-block final sum)
    lnl_walk = ctx.get_site_log_likelihoods().copy()
    ctx.log_likelihood()
    _, launches = ctx.get_stage_ms()
    assert launches[4] == 1
    assert np.allclose(ctx.get_site_log_likelihoods(), lnl_walk, rtol=1e-13, atol=0)   # the same quantities from either reduction
    ctx.set_option(epx.EPX_OPT_PRUNE_KERNEL, 0)
    ctx.update_matrices()
    ms, launches = ctx.get_stage_ms()
    assert launches[3] == 0 and launches[4] == 0 and ms[3] == 0
    ctx.close()


def _oracle_with_branch_rates(orc, prob, brates):
    """Oracle evaluation with per-branch rate scalars r_v: the oracle's own routines, fed segment
    durations multiplied by the branch's rate (effective time r_v * t, reading A6) -- its arithmetic is untouched."""
    ch, ph = prob.branch_heights()
    off, ep, du = orc.segments(ch, ph, prob.tau)
    scaled = du * np.repeat(np.asarray(brates, dtype=np.float64), np.diff(off))
    P = orc.branch_matrices(prob.Q, prob.rates, off, ep, scaled)
    out = {"seg_off": off, "seg_epoch": ep, "seg_dur": scaled, "P": P}
    if prob.N > 0:
        rf = prob.root_freqs if prob.root_freqs is not None else prob.freqs[orc.epoch_of_parent_end(np.max(prob.height), prob.tau)]
        out.update(orc.log_likelihood(prob.parent, P, prob.tip_states, rf, prob.weights, prob.pattern_weights))
    return out


@pytest.mark.parametrize("cid,kw", [(2, {"N": 80, "L": 130}), (3, {"N": 8, "L": 20}), (4, {"N": 50, "L": 2}), (5, {"n_br": 120})])
def test_branch_rates(epx, orc_ld, cid, kw):
    # every path: K=4 registers, componentwise Taylor (codon likelihood), Pade (the full-epoch table must be bypassed),
    # eigenbasis DMMA chain (branch list); rates include 0 (P = I) and 1
    rng = np.random.default_rng(40 + cid)
    prob = W.make_config(cid, **kw)
    br = rng.lognormal(0.0, 0.6, prob.n_br)
    br[1], br[2] = 0.0, 1.0
    ctx = epx.from_problem(prob)
    ctx.set_branch_rates(br)
    ref = _oracle_with_branch_rates(orc_ld, prob, br)
    if prob.N > 0:
        lnl = ctx.log_likelihood()
        assert abs(np.longdouble(lnl) - ref["lnl"]) <= LNL_RTOL * abs(ref["lnl"])
    else:
        ctx.update_matrices()
    off, ep, du = ctx.get_all_segments()
    assert np.array_equal(off, ref["seg_off"]) and np.array_equal(ep, ref["seg_epoch"])
    assert np.all(np.abs(du - ref["seg_dur"]) <= 2 * np.spacing(np.abs(ref["seg_dur"])))
    check_matrices(ctx, ref)
    assert ctx.status() == 0
    # back to unit rates: identical to a context that never had them
    ctx.set_branch_rates(None)
    ref1 = orc_ld.evaluate(prob)
    if prob.N > 0:
        lnl1 = ctx.log_likelihood()
        assert abs(np.longdouble(lnl1) - ref1["lnl"]) <= LNL_RTOL * abs(ref1["lnl"])
    else:
        ctx.update_matrices()
    check_matrices(ctx, ref1)
    with pytest.raises(epx.EpxError):
        ctx.set_branch_rates(np.full(prob.n_br, -1.0))
    ctx.close()


def _move_nodes(rng, prob, k):
    """New heights for k random nodes, each strictly inside the interval its children and parent allow."""
    left, right = trees.children_of(prob.parent)
    nodes = rng.choice(prob.n_nodes, size=k, replace=False)
    h = prob.height.copy()
    out = []
    for u in nodes:
        lo = max(h[left[u]], h[right[u]]) if left[u] >= 0 else max(0.0, h[u] - 0.05)
        hi = h[prob.parent[u]] if prob.parent[u] >= 0 else h[u] * 1.1
        if left[u] < 0:
            hi = min(hi, h[u] + 0.05)
        h[u] = lo + (hi - lo) * rng.uniform(0.05, 0.95)
        out.append(h[u])
    return nodes.astype(np.int32), np.array(out), h


@pytest.mark.parametrize("cid,kw,opts", [(2, {"N": 120, "L": 333}, ()), (2, {"N": 120, "L": 333}, ((3, 2),)), (2, {"N": 120, "L": 333}, ((3, 5),)),
                                         (2, {"N": 120, "L": 333}, ((6, 2),)), (1, {}, ()),
                                         (3, {"N": 10, "L": 40}, ()), (4, {"N": 70, "L": 3}, ())])
def test_incremental_reevaluation(epx, orc_ld, cid, kw, opts):
    """f1: after epx_set_node_heights only the touched matrices and the partials above them are recomputed; the result must
    be BIT-identical to a full evaluation of the same inputs on a fresh context, and match the oracle."""
    rng = np.random.default_rng(70 + cid)
    prob = W.make_config(cid, **kw)
    ctx = epx.from_problem(prob)
    for o, v in opts:
        ctx.set_option(o, v)
    ctx.log_likelihood()
    for it in range(6):
        nodes, new_h, h = _move_nodes(rng, prob, 1 if it < 3 else 4)
        if it == 5:
            nodes, new_h = np.array([prob.n_nodes - 1], dtype=np.int32), np.array([prob.height.max() * 1.07])   # the root
            h = prob.height.copy(); h[nodes[0]] = new_h[0]
        prob = dataclasses.replace(prob, height=h)
        n0 = ctx.launch_count()
        ctx.set_node_heights(nodes, new_h)
        lnl = ctx.log_likelihood_incremental()
        used = ctx.launch_count() - n0
        seg = 1 if prob.n_br <= 2048 else 3
        full_cost = seg + 6 if (prob.K == 4 and not opts) else seg + 2 + 2 + ctx.tree_levels() + 1     # (+1: fragment-order copies)
        if prob.K == 4 and (not opts or opts[0][0] == 6 or opts[0] == (3, 5)):
            root = 1 if (opts and opts[0] == (3, 5)) or prob.L > 4096 else 0    # up to 4096 patterns the lane walk does the root reduction itself
            assert used == seg + 1 + 1 + root       # segmenter, chain, ONE pruning walk over the dirty path (, root kernel)
        else:
            assert used < full_cost                  # no eigensystems / tables, only the dirty levels
        fresh = epx.from_problem(prob)
        for o, v in opts:
            fresh.set_option(o, v)
        full = fresh.log_likelihood()
        assert lnl == full, (it, lnl, full)
        assert np.array_equal(ctx.get_site_log_likelihoods(), fresh.get_site_log_likelihoods())
        assert np.array_equal(ctx.get_all_matrices(), fresh.get_all_matrices())
        for node in (prob.n_nodes - 1, prob.N + 1):
            a, ea = ctx.get_partials(node); b, eb = fresh.get_partials(node)
            assert np.array_equal(a, b) and np.array_equal(ea, eb)
        fresh.close()
        ref = orc_ld.evaluate(prob)
        assert abs(np.longdouble(lnl) - ref["lnl"]) <= LNL_RTOL * abs(ref["lnl"])
        assert ctx.status() == 0
    # an invalid move is refused and changes nothing
    with pytest.raises(epx.EpxError) as ei:
        ctx.set_node_heights(np.array([prob.N], dtype=np.int32), np.array([prob.height.max() * 5]))
    assert ei.value.code == epx.EPX_E_TREE
    assert ctx.log_likelihood_incremental() == lnl
    # any other change falls back to a full evaluation
    ctx.set_pattern_weights(np.full(prob.L, 2.0))
    assert abs(ctx.log_likelihood_incremental() - 2.0 * float(orc_ld.evaluate(dataclasses.replace(prob, pattern_weights=np.ones(prob.L)))["lnl"])) <= 1e-9 * abs(2 * lnl)
    ctx.close()


@pytest.mark.parametrize("variant", ["taylor", "pade"])
def test_incremental_k4_off_the_spectral_path(epx, orc_ld, variant):
    """f1 at K = 4 when a3 is NOT done by eigensystems (EPX_OPT_EXP_METHOD = 2 on a reversible model; an asymmetric model on
    the Pade path).  Those chain kernels read the segment lists and take their grid from the host-side slot count, so the
    incremental call must neither replay a graph captured for another move's slot count nor run the segmenter beside them:
    1-node, 4-node and root moves in one sequence (3 -> 12 -> 2 touched slots), each bit-identical to a fresh full evaluation."""
    rng = np.random.default_rng(170)
    prob = W.make_config(2, N=90, L=257)
    opts = ()
    if variant == "taylor":
        opts = ((epx.EPX_OPT_EXP_METHOD, 2),)
    else:
        regimes = [models.asymmetric_trait(rng, 4, keep=0.9) for _ in range(2)]
        Q = np.stack([regimes[e % 2] for e in range(prob.M)])
        F = np.stack([models.stationary(regimes[e % 2]) for e in range(prob.M)])
        prob = dataclasses.replace(prob, Q=Q, freqs=F, reversible=False, root_freqs=F[0].copy())
    ctx = epx.from_problem(prob)
    for o, v in opts:
        ctx.set_option(o, v)
    ctx.log_likelihood()
    for it, k in enumerate((1, 4, 1, 4, 0, 1)):
        if k == 0:
            nodes, new_h = np.array([prob.n_nodes - 1], dtype=np.int32), np.array([prob.height.max() * 1.07])   # the root
            h = prob.height.copy(); h[nodes[0]] = new_h[0]
        else:
            nodes, new_h, h = _move_nodes(rng, prob, k)
        prob = dataclasses.replace(prob, height=h)
        ctx.set_node_heights(nodes, new_h)
        lnl = ctx.log_likelihood_incremental()
        fresh = epx.from_problem(prob)
        for o, v in opts:
            fresh.set_option(o, v)
        full = fresh.log_likelihood()
        assert lnl == full, (variant, it, lnl, full)
        assert np.array_equal(ctx.get_site_log_likelihoods(), fresh.get_site_log_likelihoods())
        assert np.array_equal(ctx.get_all_matrices(), fresh.get_all_matrices())
        for x, y in zip(ctx.get_all_segments(), fresh.get_all_segments()):
            assert np.array_equal(x, y)
        fresh.close()
        ref = orc_ld.evaluate(prob)
        assert abs(np.longdouble(lnl) - ref["lnl"]) <= LNL_RTOL * abs(ref["lnl"])
        assert ctx.status() == 0
    ctx.close()


def test_tip_states_from_bytes_and_two_contexts_on_two_streams(epx, orc_ld):
    """epx_set_tip_states_u8 == epx_set_tip_states; two contexts on their own streams, interleaved call by call, do not
    disturb each other (independent instances are independent contexts)."""
    pa, pb = W.make_config(2, N=50, L=200), W.make_config(1, N=12, L=90)
    ta = pa.tip_states.copy(); ta[::4, ::3] = -1
    pa = dataclasses.replace(pa, tip_states=ta)
    a, b = epx.from_problem(pa), epx.from_problem(pb)
    la0 = a.log_likelihood()
    a.set_tip_states_u8(np.where(ta >= 0, ta, 255).astype(np.uint8))
    a.enqueue_log_likelihood(); b.enqueue_log_likelihood()
    a.enqueue_log_likelihood(); b.enqueue_log_likelihood()
    la, lb = a.fetch_log_likelihood(), b.fetch_log_likelihood()
    assert la == la0
    ra, rb = orc_ld.evaluate(pa), orc_ld.evaluate(pb)
    assert abs(np.longdouble(la) - ra["lnl"]) <= LNL_RTOL * abs(ra["lnl"])
    assert abs(np.longdouble(lb) - rb["lnl"]) <= LNL_RTOL * abs(rb["lnl"])
    a.close(); b.close()


def test_batch_of_independent_instances(epx, orc_ld):
    """f4 (eight patients, one codon model each): epx_log_likelihood_batch over contexts of different
    shapes, each on its own stream; bit-identical to single calls, parity with the oracle, errors reported per context."""
    rng = np.random.default_rng(44)
    probs = []
    for k in range(8):                                   # eight codon data sets with their own trees, tips and sizes
        p = W.make_config(3, N=6 + k, L=24 + 5 * k)
        probs.append(dataclasses.replace(p, tip_states=rng.integers(0, 61, p.tip_states.shape).astype(np.int32)))
    probs += [W.make_config(1), W.make_config(2, N=40, L=90), W.make_config(4, N=30, L=2)]
    ctxs = [epx.from_problem(p) for p in probs]
    single = np.array([c.log_likelihood() for c in ctxs])
    for _ in range(3):
        got = epx.log_likelihood_batch(ctxs)
        assert np.array_equal(got, single)
    for k in (0, 7, 9):
        ref = orc_ld.evaluate(probs[k])
        assert abs(np.longdouble(got[k]) - ref["lnl"]) <= LNL_RTOL * abs(ref["lnl"])
    assert epx.log_likelihood_batch([]).size == 0
    # a context that cannot run is reported, the others are unaffected
    broken = epx.Epx(4, 2, 2, 3, 5)
    with pytest.raises(epx.EpxError) as e:
        epx.log_likelihood_batch(ctxs[:2] + [broken])
    assert e.value.code == epx.EPX_E_STATE
    broken.close()
    for c in ctxs:
        c.close()


@pytest.mark.parametrize("cid,kw,opts", [(2, {"N": 60, "L": 203}, ()), (2, {"N": 60, "L": 203}, ((6, 2),)), (2, {"N": 60, "L": 203}, ((3, 5),)),
                                         (2, {"N": 60, "L": 203}, ((3, 2),)), (2, {"N": 60, "L": 203}, ((3, 3),)),
                                         (2, {"N": 60, "L": 203}, ((3, 1), (1, 1))), (3, {"N": 9, "L": 40}, ()), (4, {"N": 40, "L": 3}, ())])
def test_partially_observed_tips(epx, orc_ld, cid, kw, opts):
    """f3: tips given as vectors -- ambiguity sets (0/1) and general weights -- on every pruning kernel."""
    rng = np.random.default_rng(90 + cid)
    prob = W.make_config(cid, **kw)
    K, L = prob.K, prob.L
    ctx = epx.from_problem(prob, tip_partials=4)
    for o, v in opts:
        ctx.set_option(o, v)
    tp = {}
    for t in (0, 3, 7):                                 # ambiguity sets of 2..K states, different per pattern
        v = (rng.random((L, K)) < 0.5).astype(np.float64)
        v[np.arange(L), rng.integers(0, K, L)] = 1.0    # never empty
        tp[t] = v
    tp[5] = rng.uniform(0.0, 1.0, (L, K))               # general weights
    for t, v in tp.items():
        ctx.set_tip_partials(t, v)
    with pytest.raises(epx.EpxError):
        ctx.set_tip_partials(6, np.ones((L, K)))         # only 4 blocks were reserved
    lnl = ctx.log_likelihood()
    ref = orc_ld.evaluate(prob, tip_partials=tp, want_partials=True)
    assert abs(np.longdouble(lnl) - ref["lnl"]) <= LNL_RTOL * abs(ref["lnl"])
    site = ctx.get_site_log_likelihoods()
    assert np.max(np.abs(site.astype(np.longdouble) - ref["site_lnl"]) / np.abs(ref["site_lnl"])) <= LNL_RTOL
    out, ex = ctx.get_partials(prob.n_nodes - 1)
    got = np.ldexp(out.astype(np.longdouble), ex[None, :, None])
    want = ref["partials"][prob.n_nodes - 1]
    assert np.max(np.abs(got - want) / np.max(want, axis=(0, 2), keepdims=True)) <= 1e-10
    o5, e5 = ctx.get_partials(5)
    assert np.array_equal(o5[0], tp[5]) and not e5.any()
    assert ctx.status() == 0
    # clear one, change another: a different plan, new values
    ctx.set_tip_partials(3, None)
    tp.pop(3)
    tp[0] = np.ones((L, K))                             # all ones == missing
    ctx.set_tip_partials(0, tp[0])
    lnl2 = ctx.log_likelihood()
    ref2 = orc_ld.evaluate(prob, tip_partials=tp)
    assert abs(np.longdouble(lnl2) - ref2["lnl"]) <= LNL_RTOL * abs(ref2["lnl"])
    t = prob.tip_states.copy(); t[0, :] = -1
    ref3 = orc_ld.evaluate(dataclasses.replace(prob, tip_states=t), tip_partials={k: v for k, v in tp.items() if k != 0})
    assert abs(ref2["lnl"] - ref3["lnl"]) <= 1e-15 * abs(ref3["lnl"])
    # an incremental move on top of it
    nodes, new_h, h = _move_nodes(np.random.default_rng(5), prob, 2)
    ctx.set_node_heights(nodes, new_h)
    lnl3 = ctx.log_likelihood_incremental()
    ref4 = orc_ld.evaluate(dataclasses.replace(prob, height=h), tip_partials=tp)
    assert abs(np.longdouble(lnl3) - ref4["lnl"]) <= LNL_RTOL * abs(ref4["lnl"])
    ctx.close()
