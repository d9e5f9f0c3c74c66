"""CPU-side checks of the C-ABI boundary: libepx.so builds, loads, and exports every symbol include/epx.h declares;
host-side validation (no kernels are launched, no GPU needed)."""
import ctypes as ct
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_1309_3075_b200 import build
    build.build_library()
    import paper_1309_3075_b200 as epx
    return epx.lib()


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "epx.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(epx_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(L):
    names = _declared_symbols()
    assert len(names) >= 25
    for n in names:
        assert hasattr(L, n), f"libepx.so does not export {n}"


def test_binding_covers_every_symbol(L):
    import paper_1309_3075_b200 as epx
    for n in _declared_symbols():
        short = n[len("epx_"):]
        assert hasattr(epx.Epx, short) or hasattr(epx, short) or n in ("epx_create", "epx_destroy", "epx_measure_fp64_peak"), n


def test_no_torch_types_in_signatures():
    src = open(os.path.join(ROOT, "include", "epx.h")).read()
    assert "torch" not in src.lower() and "at::" not in src and "#include <cuda" not in src


def test_create_argument_checks(L):
    import paper_1309_3075_b200 as epx
    for args in [(1, 1, 1, 2, 1), (65, 1, 1, 2, 1), (4, 0, 1, 2, 1), (4, 1, 9, 2, 1), (4, 1, 1, 1, 1), (4, 1, 1, 2, 0)]:
        with pytest.raises(epx.EpxError):
            epx.Epx(*args)
    c = epx.Epx(4, 2, 2, 3, 5)
    assert c.workspace_bytes() > 0
    c.close()


def test_host_validation_rules(L):
    import paper_1309_3075_b200 as epx
    c = epx.Epx(4, 3, 2, 3, 5)
    # boundaries: strictly increasing, finite
    for bad in ([0.5, 0.5], [0.6, 0.5], [0.1, np.inf], [np.nan, 1.0]):
        with pytest.raises(epx.EpxError) as ei:
            c.set_epoch_boundaries(bad)
        assert ei.value.code == epx.EPX_E_ARG
    c.set_epoch_boundaries([0.1, 0.5])
    # models
    pi = np.array([0.1, 0.2, 0.3, 0.4])
    Q = np.tile(pi, (4, 1)); np.fill_diagonal(Q, 0); np.fill_diagonal(Q, -Q.sum(1))
    c.set_epoch_model(0, Q, pi, True)
    Qbad = Q.copy(); Qbad[0, 1] += 1e-3
    with pytest.raises(epx.EpxError) as ei:
        c.set_epoch_model(1, Qbad, pi, True)          # row does not sum to 0
    assert ei.value.code == epx.EPX_E_MODEL
    Qneg = Q.copy(); Qneg[0, 1] = -0.1; Qneg[0, 0] = -(Qneg[0, 1] + Qneg[0, 2] + Qneg[0, 3])
    with pytest.raises(epx.EpxError):
        c.set_epoch_model(1, Qneg, pi, True)
    Qasym = Q.copy(); Qasym[0, 1] += 0.2; Qasym[0, 0] -= 0.2
    with pytest.raises(epx.EpxError):
        c.set_epoch_model(1, Qasym, pi, True)         # detailed balance violated
    with pytest.raises(epx.EpxError):
        c.set_epoch_model(1, Qasym, pi, False)        # mixing reversible flags within a ctx
    with pytest.raises(epx.EpxError):
        c.set_epoch_model(1, Q, pi * 1.1, True)       # freqs not a distribution
    with pytest.raises(epx.EpxError):
        c.set_epoch_model(3, Q, pi, True)             # epoch out of range
    # category rates
    with pytest.raises(epx.EpxError):
        c.set_category_rates([1.0, -1.0], [0.5, 0.5])
    with pytest.raises(epx.EpxError):
        c.set_category_rates([1.0, 1.0], [0.5, 0.6])
    c.set_category_rates([0.5, 1.5], [0.5, 0.5])
    # trees: N = 3 tips, nodes 0..4
    good_parent, good_h = [3, 3, 4, 4, -1], [0.0, 0.0, 0.0, 0.3, 1.0]
    c.set_tree(good_parent, good_h)
    for parent, h in [([3, 3, 4, 4, 4], good_h),            # no root
                      ([3, 3, 3, 4, -1], good_h),           # trifurcation
                      ([3, 3, 4, -1, -1], good_h),          # two roots
                      ([3, 3, 4, 4, -1], [0, 0, 0, 1.3, 1.0]),  # child above parent
                      ([1, 3, 4, 4, -1], good_h),           # tip as a parent
                      ([3, 3, 4, 4, -1], [0, 0, np.nan, 0.3, 1.0])]:
        with pytest.raises(epx.EpxError) as ei:
            c.set_tree(parent, h)
        assert ei.value.code == epx.EPX_E_TREE
    # a call with the CURRENT topology only replaces the heights; if it is refused the tree stays in place
    c.set_tree(good_parent, good_h)
    c.set_tree(good_parent, [0.0, 0.0, 0.1, 0.4, 2.0])
    with pytest.raises(epx.EpxError) as ei:
        c.set_tree(good_parent, [0.0, 0.0, 0.1, 2.4, 2.0])
    assert ei.value.code == epx.EPX_E_TREE
    assert c.plan_info()["operations"] == 2          # still planned: the refused call changed nothing
    with pytest.raises(epx.EpxError):
        c.set_tree([3, 3, 3, 4, -1], good_h)         # a NEW topology that fails leaves the context without a tree ...
    with pytest.raises(epx.EpxError):
        c.plan_info()                                # ... (EPX_E_STATE)
    # moving nodes (f1): a node must stay between its children and its parent; a refused move changes nothing
    c.set_tree(good_parent, good_h)
    c.set_node_heights([3], [0.5])
    for nodes, hs in [([3], [1.5]), ([3], [-0.1]), ([4], [0.2]), ([9], [0.1]), ([3], [np.nan])]:
        with pytest.raises(epx.EpxError):
            c.set_node_heights(nodes, hs)
    c.set_node_heights([3, 4], [0.9, 2.0])           # consistent as a set
    # compute before bind -> state error, not a crash
    with pytest.raises(epx.EpxError) as ei:
        c.log_likelihood()
    assert ei.value.code == epx.EPX_E_STATE
    # branch-list setters are refused in tree mode and vice versa
    with pytest.raises(epx.EpxError):
        c.set_branches([0.0], [1.0])
    b = epx.Epx(4, 1, 1, 0, 0)
    with pytest.raises(epx.EpxError):
        b.workspace_bytes()                            # needs set_branches first
    with pytest.raises(epx.EpxError):
        b.set_branches([0.5], [0.1])                   # parent below child
    b.set_branches([0.0, 0.1], [1.0, 0.1])
    assert b.workspace_bytes() > 0
    with pytest.raises(epx.EpxError):
        b.set_tree(good_parent, good_h)
    c.close(); b.close()


def test_workspace_scales_with_problem(L):
    import paper_1309_3075_b200 as epx
    a = epx.Epx(4, 10, 4, 2000, 10000)
    need = a.workspace_bytes()
    partials = 1999 * 4 * 10000 * 4 * 8
    assert partials < need < partials * 1.2          # the partials buffer dominates (cfg 2: 2.56 GB)
    a.close()


def test_plan_info_and_tip_partial_reservation_state(L):
    import paper_1309_3075_b200 as epx
    import workloads as W
    prob = W.make_config(2, N=33, L=40)
    c = epx.Epx(prob.K, prob.M, prob.C, prob.N, prob.L)
    with pytest.raises(epx.EpxError) as e:
        c.plan_info()                                   # no tree yet
    assert e.value.code == epx.EPX_E_STATE
    c.set_tree(prob.parent, prob.height)
    info = c.plan_info()
    assert info["operations"] == prob.N - 1 and info["levels"] >= 6 and info["depth_first"] == 1
    assert info["bottom_pieces"] >= 1 and info["stack_slots"] >= 1
    assert info["largest_piece_ops"] + info["top_piece_ops"] <= prob.N - 1
    # a second reservation while a tip still carries a vector would orphan its block: refused
    c.reserve_tip_partials(2)
    c.set_tip_partials(3, np.ones((prob.L, prob.K)))
    with pytest.raises(epx.EpxError) as e:
        c.reserve_tip_partials(4)
    assert e.value.code == epx.EPX_E_STATE
    c.set_tip_partials(3, None)
    c.reserve_tip_partials(4)
    c.close()


def test_shared_processes_are_detected(L):
    """S processes, M epochs, phi_m.  Config 4 alternates two seasonal regimes over 24 epochs; config 2 has ten
    different HKY models."""
    import paper_1309_3075_b200 as epx
    import workloads as W
    p4 = W.make_config(4, N=10, L=1)
    c = epx.Epx(p4.K, p4.M, p4.C, p4.N, p4.L)
    with pytest.raises(epx.EpxError):
        c.epoch_processes()                              # models not set yet
    for e in range(p4.M):
        c.set_epoch_model(e, p4.Q[e], p4.freqs[e], False)
    phi, S = c.epoch_processes()
    assert S == 2 and phi.tolist() == [e % 2 for e in range(24)]
    c.close()
    p2 = W.make_config(2, N=10, L=4)
    c = epx.Epx(p2.K, p2.M, p2.C, p2.N, p2.L)
    for e in range(p2.M):
        c.set_epoch_model(e, p2.Q[e], p2.freqs[e], True)
    phi, S = c.epoch_processes()
    assert S == 10 and phi.tolist() == list(range(10))
    c.set_epoch_model(7, p2.Q[2], p2.freqs[2], True)     # epoch 7 now runs process 2
    phi, S = c.epoch_processes()
    assert S == 9 and phi.tolist() == [0, 1, 2, 3, 4, 5, 6, 2, 7, 8]
    c.close()


def test_tip_state_pool_survives_fork(L):
    """The host thread pool behind epx_set_tip_states is process-wide.  A child forked while another thread is inside a
    repacking job must still be able to set tip states (its own pool, no mutex left locked by a thread that does not exist
    in the child); the parent's pool must keep working after the forks.  No GPU: an unbound ctx repacks into host memory."""
    import signal
    import threading
    import time
    import warnings
    import paper_1309_3075_b200 as epx
    N, Lp = 1100, 4000                       # 4.4 M states: above the 4 M threshold of the pooled path
    rng = np.random.default_rng(5)
    states = rng.integers(0, 4, size=(N, Lp), dtype=np.uint8)
    a = epx.Epx(4, 1, 1, N, Lp)
    a.set_tip_states_u8(states)              # creates the pool in the parent
    stop = threading.Event()

    def hammer():
        while not stop.is_set():
            a.set_tip_states_u8(states)

    t = threading.Thread(target=hammer)
    t.start()
    try:
        for k in range(6):
            time.sleep(0.003 * k)
            with warnings.catch_warnings():
                warnings.simplefilter("ignore", DeprecationWarning)      # fork() in a multi-threaded process: the case under test
                pid = os.fork()
            if pid == 0:
                code = 1
                try:
                    signal.alarm(20)         # a deadlocked child dies by SIGALRM instead of hanging the suite
                    b = epx.Epx(4, 1, 1, N, Lp)
                    b.set_tip_states_u8(states)
                    b.set_tip_states(states.astype(np.int32))
                    code = 0
                finally:
                    os._exit(code)
            _, status = os.waitpid(pid, 0)
            assert os.WIFEXITED(status) and os.WEXITSTATUS(status) == 0, f"forked child {k}: status {status:#x}"
    finally:
        stop.set()
        t.join(30)
    assert not t.is_alive()
    a.set_tip_states_u8(states)              # the parent's pool still serves
    a.close()
