"""epx_segment_branches_static: the entry point for callers that cannot allocate device memory.

Who that is: code that is handed device buffers for its inputs and results and nothing else -- a likelihood plug-in
running inside a host program that has given all GPU memory to its own arena, or a step on a latency-critical path
where cudaMalloc (which synchronises the whole device) is not acceptable.  Such a caller cannot bind the workspace the
rest of the library asks for, so this one call keeps its intermediates in a fixed array inside libepx.so.

What is checked here: the call returns the same segment lists as the ordinary, workspace-backed path
(epx_set_branches -> epx_update_matrices -> epx_get_all_segments) -- offsets and epochs equal, durations within the
1 ulp the segment tests of this suite allow -- on two calls in a row with different branch lists.  The built-in array
keeps the first call's contents when the second starts, so the second call (fewer branches, other epochs) would show
anything that leaks from one call into the next.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the parity
tests.  It passes alone in a fresh process (the first call then does the per-device address look-up) and after the
other tests.
"""
import numpy as np
import pytest


def _branch_list(seed, n_br, M):
    """Seeded branch list in the shape of config 5 (uniform child ends, exponential lengths) plus the awkward cases:
    zero-length branches, ends exactly on a boundary, a branch across every epoch."""
    import workloads as W
    from workloads import models
    rng = np.random.default_rng(seed)
    tau = np.sort(rng.uniform(0.05, 0.95, size=M - 1))
    child = rng.uniform(0.0, 1.0, size=n_br)
    par = np.minimum(child + rng.exponential(0.25, size=n_br), 1.0)
    par[5] = child[5]                                   # zero length
    child[6], par[6] = tau[0], tau[min(2, M - 2)]       # both ends on boundaries
    child[7], par[7] = 0.0, 1.0                         # every epoch
    par[8] = child[8] = tau[0]                          # zero length on a boundary
    K, C = 4, 1
    Q = np.zeros((M, K, K)); F = np.zeros((M, K))
    for e in range(M):
        F[e] = rng.dirichlet(np.full(4, 2.0))
        Q[e] = models.hky(2.0, F[e])
    return W.EpochProblem(f"static_{seed}", K, M, C, 0, 0, tau, Q, F, True, np.ones(1), np.ones(1),
                          child_height=child, parent_height=par)


def _existing_path(prob):
    import paper_1309_3075_b200 as epx
    ctx = epx.from_problem(prob, device=0)
    ctx.update_matrices()
    off, ep, du = ctx.get_all_segments()
    ctx.close()
    return off, ep, du


@pytest.mark.gpu
def test_static_scratch_segmenter_matches_workspace_path_twice():
    import torch
    import paper_1309_3075_b200 as epx
    assert torch.cuda.is_available()
    dev = torch.device("cuda", 0)
    stream = torch.cuda.Stream(device=dev)
    # first call: more than the 2 048 slots the fused single-CTA segmenter takes, so the reference is the three-kernel path;
    # second call: fewer branches, fewer epochs -- the array still holds the first call's counts and epochs beyond n_br
    for seed, n_br, M in ((11, 20000, 16), (12, 1500, 5)):
        prob = _branch_list(seed, n_br, M)
        off_ref, ep_ref, du_ref = _existing_path(prob)
        cap = n_br * M
        # the caller's buffers (inputs and outputs); outputs poisoned so that an element the call skips shows
        tau = torch.tensor(prob.tau, dtype=torch.float64, device=dev)
        ch = torch.tensor(prob.child_height, dtype=torch.float64, device=dev)
        ph = torch.tensor(prob.parent_height, dtype=torch.float64, device=dev)
        seg_off = torch.full((n_br + 1,), -7, dtype=torch.int32, device=dev)
        seg_epoch = torch.full((cap,), -7, dtype=torch.int32, device=dev)
        seg_dur = torch.full((cap,), float("nan"), dtype=torch.float64, device=dev)
        torch.cuda.synchronize(dev)
        before = torch.cuda.memory_allocated(dev)
        epx.segment_branches_static(tau, ch, ph, seg_off, seg_epoch, seg_dur, stream=stream)
        stream.synchronize()
        assert torch.cuda.memory_allocated(dev) == before          # the binding made no tensor either
        off = seg_off.cpu().numpy()
        n = int(off[-1])
        assert n == int(off_ref[-1]) and np.array_equal(off, off_ref)
        ep, du = seg_epoch.cpu().numpy(), seg_dur.cpu().numpy()
        assert np.array_equal(ep[:n], ep_ref)
        assert np.all(np.abs(du[:n] - du_ref) <= np.spacing(np.abs(du_ref)))     # <= 1 ulp, as test_gpu_parity's segment check
        assert np.all(du[:n] > 0) and np.all(ep[n:] == -7) and np.all(np.isnan(du[n:]))   # nothing written past the total


@pytest.mark.gpu
def test_static_scratch_segmenter_respects_capacity():
    """Outputs shorter than the segment total: the offsets still report the total, nothing is stored past `cap`."""
    import torch
    import paper_1309_3075_b200 as epx
    dev = torch.device("cuda", 0)
    prob = _branch_list(13, 600, 8)
    off_ref, ep_ref, du_ref = _existing_path(prob)
    cap = int(off_ref[-1]) // 2
    tau = torch.tensor(prob.tau, dtype=torch.float64, device=dev)
    ch = torch.tensor(prob.child_height, dtype=torch.float64, device=dev)
    ph = torch.tensor(prob.parent_height, dtype=torch.float64, device=dev)
    seg_off = torch.zeros(601, dtype=torch.int32, device=dev)
    guard = 64
    seg_epoch = torch.full((cap + guard,), -7, dtype=torch.int32, device=dev)
    seg_dur = torch.full((cap + guard,), -7.0, dtype=torch.float64, device=dev)
    epx.segment_branches_static(tau, ch, ph, seg_off, seg_epoch[:cap], seg_dur[:cap])
    torch.cuda.synchronize(dev)
    assert np.array_equal(seg_off.cpu().numpy(), off_ref)
    assert np.array_equal(seg_epoch.cpu().numpy()[:cap], ep_ref[:cap]) and np.all(seg_epoch.cpu().numpy()[cap:] == -7)
    assert np.all(seg_dur.cpu().numpy()[cap:] == -7.0)


def test_static_scratch_segmenter_refuses_oversize_and_null():
    """Host-side checks come before any CUDA call, so they run without a GPU: a list longer than the built-in array is
    refused with EPX_E_WORKSPACE and a message that names the limit; NULL outputs with EPX_E_ARG."""
    import ctypes as ct
    from paper_1309_3075_b200 import build
    build.build_library()
    import paper_1309_3075_b200 as epx
    L = epx.lib()
    msg = ct.create_string_buffer(256)
    fake = ct.c_void_p(256)          # never dereferenced: the size check fails first
    rc = L.epx_segment_branches_static(0, epx.EPX_STATIC_MAX_BRANCHES + 1, 4, fake, fake, fake, fake, fake, fake, 10, None, msg, len(msg))
    assert rc == epx.EPX_E_WORKSPACE
    text = msg.value.decode()
    assert str(epx.EPX_STATIC_MAX_BRANCHES) in text and "EPX_STATIC_MAX_BRANCHES" in text
    assert L.epx_segment_branches_static(0, 10, 4, fake, fake, fake, None, fake, fake, 10, None, msg, len(msg)) == epx.EPX_E_ARG
    assert L.epx_segment_branches_static(0, 10, 0, fake, fake, fake, fake, fake, fake, 10, None, None, 0) == epx.EPX_E_ARG
    assert L.epx_segment_branches_static(0, -1, 4, fake, fake, fake, fake, fake, fake, 10, None, None, 0) == epx.EPX_E_ARG
    # the header's limit and the binding's agree
    import os, re
    hdr = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "epx.h")).read()
    assert int(re.search(r"#define\s+EPX_STATIC_MAX_BRANCHES\s+(\d+)", hdr).group(1)) == epx.EPX_STATIC_MAX_BRANCHES
