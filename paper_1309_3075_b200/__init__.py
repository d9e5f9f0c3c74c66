"""B200-native epoch substitution model hot path (arxiv 1309.3075) -- thin Python binding of the C ABI in
``include/epx.h``.

Argument marshalling only: every step of the path (segmenter, eigensystems / Pade, segment exponentials + chain
convolution, pruning, root reduction) runs in the CUDA kernels of ``libepx.so``.  PyTorch provides the device
workspace and the stream, nothing else.  There is no CPU fallback: loading fails loudly if ``libepx.so`` is missing.
Method names are the C names without the ``epx_`` prefix.
"""
from __future__ import annotations

import ctypes as ct
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libepx.so")

EPX_OK, EPX_E_ARG, EPX_E_STATE, EPX_E_TREE, EPX_E_MODEL, EPX_E_WORKSPACE, EPX_E_CUDA, EPX_E_NUMERIC = 0, -1, -2, -3, -4, -5, -6, -7
EPX_OPT_CHAIN_KERNEL, EPX_OPT_USE_GRAPH, EPX_OPT_PRUNE_KERNEL, EPX_OPT_EXP_METHOD = 1, 2, 3, 4
EPX_OPT_STAGE_EVENTS, EPX_OPT_DFS_PPL, EPX_OPT_DFS_PIECES, EPX_OPT_MMA_CHUNK, EPX_OPT_JACOBI_KERNEL = 5, 6, 7, 8, 9
EPX_OPT_SHARE_PROCESSES, EPX_OPT_EPOCH_PRODUCTS = 10, 11
STAGE_NAMES = ("segment", "eigen", "chain", "prune", "root")
EPX_STATIC_MAX_BRANCHES = 32768   # epx.h: most branches one epx_segment_branches_static call takes

_lib = None


class EpxError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"epx error {code}: {message}")
        self.code = code


def _sig(lib, name, restype, *argtypes):
    fn = getattr(lib, name)
    fn.restype = restype
    fn.argtypes = list(argtypes)


def lib():
    """Load libepx.so (built by ``paper_1309_3075_b200.build``). Raises if it is missing -- no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_1309_3075_b200.build` "
                           "(the CUDA library is the product; there is no CPU fallback)")
    L = ct.CDLL(LIB_PATH)
    vp, i, dp, ip = ct.c_void_p, ct.c_int, ct.c_void_p, ct.c_void_p
    _sig(L, "epx_create", i, ct.POINTER(vp), i, i, i, i, i, i)
    _sig(L, "epx_destroy", None, vp)
    _sig(L, "epx_workspace_bytes", i, vp, ct.POINTER(ct.c_size_t))
    _sig(L, "epx_bind", i, vp, vp, ct.c_size_t, vp)
    _sig(L, "epx_set_epoch_boundaries", i, vp, dp)
    _sig(L, "epx_set_epoch_model", i, vp, i, dp, dp, i)
    _sig(L, "epx_set_category_rates", i, vp, dp, dp)
    _sig(L, "epx_set_tree", i, vp, ip, dp)
    _sig(L, "epx_set_tip_states", i, vp, ip)
    _sig(L, "epx_set_tip_states_u8", i, vp, ip)
    _sig(L, "epx_set_pattern_weights", i, vp, dp)
    _sig(L, "epx_reserve_tip_partials", i, vp, i)
    _sig(L, "epx_set_tip_partials", i, vp, i, dp)
    _sig(L, "epx_set_root_frequencies", i, vp, dp)
    _sig(L, "epx_set_branches", i, vp, i, dp, dp)
    _sig(L, "epx_set_branch_rates", i, vp, dp)
    _sig(L, "epx_set_node_heights", i, vp, i, ip, dp)
    _sig(L, "epx_log_likelihood_incremental", i, vp, ct.POINTER(ct.c_double))
    _sig(L, "epx_update_matrices", i, vp)
    _sig(L, "epx_enqueue_log_likelihood", i, vp)
    _sig(L, "epx_log_likelihood", i, vp, ct.POINTER(ct.c_double))
    _sig(L, "epx_fetch_log_likelihood", i, vp, ct.POINTER(ct.c_double))
    _sig(L, "epx_log_likelihood_batch", i, vp, i, dp, ip)
    _sig(L, "epx_get_segments", i, vp, i, ct.POINTER(i), ip, dp)
    _sig(L, "epx_get_all_segments", i, vp, ip, ip, dp, i)
    _sig(L, "epx_get_matrix", i, vp, i, i, dp)
    _sig(L, "epx_matrices_device", i, vp, ct.POINTER(vp))
    _sig(L, "epx_get_partials", i, vp, i, dp, ip)
    _sig(L, "epx_get_site_log_likelihoods", i, vp, dp)
    _sig(L, "epx_launch_count", i, vp, ct.POINTER(ct.c_longlong))
    _sig(L, "epx_tree_levels", i, vp, ct.POINTER(i))
    _sig(L, "epx_plan_info", i, vp, ip)
    _sig(L, "epx_epoch_processes", i, vp, ip, ct.POINTER(i))
    _sig(L, "epx_get_stage_ms", i, vp, ct.c_void_p, ct.c_void_p)
    _sig(L, "epx_status", i, vp, ct.POINTER(i))
    _sig(L, "epx_set_option", i, vp, i, i)
    _sig(L, "epx_last_error", ct.c_char_p, vp)
    _sig(L, "epx_measure_fp64_peak", i, i, i, ct.c_double, vp, vp, ct.POINTER(ct.c_double))
    _sig(L, "epx_segment_branches_static", i, i, i, i, dp, dp, dp, ip, ip, dp, i, vp, ct.c_char_p, ct.c_size_t)
    _lib = L
    return L


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ct.c_void_p)


class Epx:
    """One epx_ctx. ``bind`` allocates the device workspace with torch and borrows a torch stream."""

    def __init__(self, K: int, M: int, C: int, N_tips: int, L: int, device: int = 0):
        self._L = lib()
        self._ctx = ct.c_void_p()
        self.K, self.M, self.C, self.N, self.L, self.device = K, M, C, N_tips, (L if N_tips else 0), device
        self.n_slots = 2 * N_tips - 1 if N_tips else 0
        self._ws = None
        self._stream = None
        rc = self._L.epx_create(ct.byref(self._ctx), K, M, C, N_tips, L, device)
        if rc != EPX_OK:
            self._ctx = ct.c_void_p()
            raise EpxError(rc, "epx_create: bad argument")

    # ---- plumbing
    def _check(self, rc: int) -> None:
        if rc != EPX_OK:
            raise EpxError(rc, self.last_error())

    def last_error(self) -> str:
        return self._L.epx_last_error(self._ctx).decode()

    def close(self) -> None:
        if self._ctx:
            self._L.epx_destroy(self._ctx)
            self._ctx = ct.c_void_p()
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def workspace_bytes(self) -> int:
        n = ct.c_size_t()
        self._check(self._L.epx_workspace_bytes(self._ctx, ct.byref(n)))
        return int(n.value)

    def bind(self, stream=None, workspace=None) -> None:
        """Allocate (or take) a torch uint8 CUDA tensor as workspace and bind it with `stream` (a torch.cuda.Stream;
        None = a new non-default stream, so that the library replays its kernels from a CUDA graph)."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("CUDA device required: the epoch hot path has no CPU fallback")
        dev = torch.device("cuda", self.device)
        need = self.workspace_bytes()
        if workspace is None:
            workspace = torch.empty(need + 256, dtype=torch.uint8, device=dev)
        base = workspace.data_ptr()
        aligned = (base + 255) & ~255
        if stream is None:
            stream = torch.cuda.Stream(device=dev)
        self._ws, self._stream = workspace, stream
        self._check(self._L.epx_bind(self._ctx, ct.c_void_p(aligned), workspace.numel() - (aligned - base),
                                     ct.c_void_p(stream.cuda_stream)))

    @property
    def stream(self):
        return self._stream

    # ---- setters
    def set_epoch_boundaries(self, tau) -> None:
        tau = _f64(tau)
        self._check(self._L.epx_set_epoch_boundaries(self._ctx, _ptr(tau) if tau.size else None))

    def set_epoch_model(self, epoch: int, Q, freqs, reversible: bool) -> None:
        Q, freqs = _f64(Q), _f64(freqs)
        assert Q.shape == (self.K, self.K) and freqs.shape == (self.K,)
        self._check(self._L.epx_set_epoch_model(self._ctx, epoch, _ptr(Q), _ptr(freqs), int(bool(reversible))))

    def set_category_rates(self, rates, weights) -> None:
        rates, weights = _f64(rates), _f64(weights)
        assert rates.shape == (self.C,) and weights.shape == (self.C,)
        self._check(self._L.epx_set_category_rates(self._ctx, _ptr(rates), _ptr(weights)))

    def set_tree(self, parent, height) -> None:
        parent, height = _i32(parent), _f64(height)
        assert self.N == 0 or (parent.shape == (2 * self.N - 1,) and height.shape == parent.shape)
        self._check(self._L.epx_set_tree(self._ctx, _ptr(parent), _ptr(height)))

    def set_tip_states(self, states) -> None:
        states = _i32(states)
        assert states.shape == (self.N, self.L)
        self._check(self._L.epx_set_tip_states(self._ctx, _ptr(states)))

    def set_tip_states_u8(self, states) -> None:
        states = np.ascontiguousarray(states, dtype=np.uint8)
        assert states.shape == (self.N, self.L)
        self._check(self._L.epx_set_tip_states_u8(self._ctx, _ptr(states)))

    def reserve_tip_partials(self, max_tips: int) -> None:
        self._check(self._L.epx_reserve_tip_partials(self._ctx, int(max_tips)))

    def set_tip_partials(self, tip: int, partials) -> None:
        partials = None if partials is None else _f64(partials)
        assert partials is None or partials.shape == (self.L, self.K)
        self._check(self._L.epx_set_tip_partials(self._ctx, int(tip), _ptr(partials)))

    def set_pattern_weights(self, wt) -> None:
        wt = None if wt is None else _f64(wt)
        self._check(self._L.epx_set_pattern_weights(self._ctx, _ptr(wt)))

    def set_root_frequencies(self, freqs) -> None:
        freqs = None if freqs is None else _f64(freqs)
        self._check(self._L.epx_set_root_frequencies(self._ctx, _ptr(freqs)))

    def set_branches(self, child_height, parent_height) -> None:
        ch, ph = _f64(child_height), _f64(parent_height)
        assert ch.shape == ph.shape and ch.ndim == 1
        self._check(self._L.epx_set_branches(self._ctx, ch.shape[0], _ptr(ch), _ptr(ph)))
        self.n_slots = ch.shape[0]

    def set_branch_rates(self, rates) -> None:
        rates = None if rates is None else _f64(rates)
        assert rates is None or rates.shape == (self.n_slots,)
        self._check(self._L.epx_set_branch_rates(self._ctx, _ptr(rates)))

    def set_node_heights(self, nodes, heights) -> None:
        nodes, heights = _i32(nodes), _f64(heights)
        assert nodes.shape == heights.shape and nodes.ndim == 1
        self._check(self._L.epx_set_node_heights(self._ctx, nodes.shape[0], _ptr(nodes), _ptr(heights)))

    def log_likelihood_incremental(self) -> float:
        v = ct.c_double()
        self._check(self._L.epx_log_likelihood_incremental(self._ctx, ct.byref(v)))
        return v.value

    def set_option(self, option: int, value: int) -> None:
        self._check(self._L.epx_set_option(self._ctx, option, value))

    # ---- compute
    def update_matrices(self) -> None:
        self._check(self._L.epx_update_matrices(self._ctx))

    def enqueue_log_likelihood(self) -> None:
        self._check(self._L.epx_enqueue_log_likelihood(self._ctx))

    def log_likelihood(self) -> float:
        v = ct.c_double()
        self._check(self._L.epx_log_likelihood(self._ctx, ct.byref(v)))
        return v.value

    def fetch_log_likelihood(self) -> float:
        v = ct.c_double()
        self._check(self._L.epx_fetch_log_likelihood(self._ctx, ct.byref(v)))
        return v.value

    # ---- read-back
    def get_segments(self, slot: int):
        n = ct.c_int()
        ep = np.zeros(max(self.M, 1), dtype=np.int32)
        du = np.zeros(max(self.M, 1), dtype=np.float64)
        self._check(self._L.epx_get_segments(self._ctx, slot, ct.byref(n), _ptr(ep), _ptr(du)))
        return ep[:n.value].copy(), du[:n.value].copy()

    def get_all_segments(self):
        cap = self.n_slots * self.M + 1
        off = np.zeros(self.n_slots + 1, dtype=np.int32)
        ep = np.zeros(cap, dtype=np.int32)
        du = np.zeros(cap, dtype=np.float64)
        self._check(self._L.epx_get_all_segments(self._ctx, _ptr(off), _ptr(ep), _ptr(du), cap))
        n = int(off[-1])
        return off, ep[:n].copy(), du[:n].copy()

    def get_matrix(self, slot: int, category: int):
        out = np.zeros((self.K, self.K), dtype=np.float64)
        self._check(self._L.epx_get_matrix(self._ctx, slot, category, _ptr(out)))
        return out

    def matrices_device(self) -> int:
        p = ct.c_void_p()
        self._check(self._L.epx_matrices_device(self._ctx, ct.byref(p)))
        return int(p.value)

    def get_all_matrices(self):
        """All matrices [slot][C][K][K] as a host array (one device->host copy of the borrowed device buffer)."""
        import torch
        ptr = self.matrices_device()
        n = self.n_slots * self.C * self.K * self.K
        out = np.empty(n, dtype=np.float64)
        self._stream.synchronize()
        # wrap the borrowed pointer without copying, then copy to host
        base = self._ws.data_ptr()
        off = ptr - base
        view = self._ws[off:off + 8 * n].view(torch.float64)
        out[:] = view.cpu().numpy()
        return out.reshape(self.n_slots, self.C, self.K, self.K)

    def get_partials(self, node: int):
        out = np.zeros((self.C, self.L, self.K), dtype=np.float64)
        ex = np.zeros(self.L, dtype=np.int32)
        self._check(self._L.epx_get_partials(self._ctx, node, _ptr(out), _ptr(ex)))
        return out, ex

    def get_site_log_likelihoods(self):
        out = np.zeros(self.L, dtype=np.float64)
        self._check(self._L.epx_get_site_log_likelihoods(self._ctx, _ptr(out)))
        return out

    def launch_count(self) -> int:
        n = ct.c_longlong()
        self._check(self._L.epx_launch_count(self._ctx, ct.byref(n)))
        return int(n.value)

    def get_stage_ms(self):
        """(ms[5], launches[5]) of the last compute call's stages (needs EPX_OPT_STAGE_EVENTS = 1); synchronises."""
        ms = np.zeros(5, dtype=np.float32)
        ln = np.zeros(5, dtype=np.int32)
        self._check(self._L.epx_get_stage_ms(self._ctx, _ptr(ms), _ptr(ln)))
        return ms, ln

    def tree_levels(self) -> int:
        n = ct.c_int()
        self._check(self._L.epx_tree_levels(self._ctx, ct.byref(n)))
        return n.value

    def epoch_processes(self):
        """(phi[M], S): the detected process of every epoch and the number of distinct processes."""
        phi = np.zeros(self.M, dtype=np.int32)
        n = ct.c_int()
        self._check(self._L.epx_epoch_processes(self._ctx, _ptr(phi), ct.byref(n)))
        return phi, n.value

    def plan_info(self) -> dict:
        info = np.zeros(8, dtype=np.int32)
        self._check(self._L.epx_plan_info(self._ctx, _ptr(info)))
        keys = ("levels", "operations", "depth_first", "bottom_pieces", "largest_piece_ops", "top_piece_ops", "stack_slots",
                "prune_launches")
        return {k: int(v) for k, v in zip(keys, info)}

    def status(self) -> int:
        n = ct.c_int()
        self._check(self._L.epx_status(self._ctx, ct.byref(n)))
        return n.value


def set_problem(ctx: Epx, prob, tip_states_u8=None) -> None:
    """Call every setter of `ctx` from a problem object (attributes as in workloads.EpochProblem; read by
    attribute, nothing is imported).  `tip_states_u8`: the tip states as a host uint8 array, passed through
    epx_set_tip_states_u8 instead of the int32 form."""
    if prob.N > 0:
        # the largest input first: on a bound ctx its host -> device copy is pipelined with the repacking and then runs
        # behind the host work of the other setters (validation, pruning plan)
        if tip_states_u8 is not None:
            ctx.set_tip_states_u8(tip_states_u8)
        else:
            ctx.set_tip_states(prob.tip_states)
    ctx.set_epoch_boundaries(prob.tau)
    for e in range(prob.M):
        ctx.set_epoch_model(e, prob.Q[e], prob.freqs[e], prob.reversible)
    ctx.set_category_rates(prob.rates, prob.weights)
    if prob.N > 0:
        ctx.set_tree(prob.parent, prob.height)
        ctx.set_pattern_weights(prob.pattern_weights)
        ctx.set_root_frequencies(prob.root_freqs)
    else:
        ctx.set_branches(prob.child_height, prob.parent_height)


def from_problem(prob, device: int = 0, stream=None, tip_partials: int = 0) -> Epx:
    """Create, fill and bind a context for `prob` (`tip_partials`: blocks to reserve for partially observed tips)."""
    ctx = Epx(prob.K, prob.M, prob.C, prob.N, prob.L if prob.N else 1, device)
    if tip_partials:
        ctx.reserve_tip_partials(tip_partials)
    if prob.N == 0:
        ctx.set_branches(prob.child_height, prob.parent_height)
    ctx.bind(stream)
    set_problem(ctx, prob)
    return ctx


def log_likelihood_batch(ctxs) -> np.ndarray:
    """epx_log_likelihood_batch: every context's work is enqueued before the first result is fetched."""
    n = len(ctxs)
    arr = (ct.c_void_p * n)(*[c._ctx for c in ctxs])
    out = np.zeros(n, dtype=np.float64)
    rc = np.zeros(n, dtype=np.int32)
    code = lib().epx_log_likelihood_batch(arr, n, _ptr(out), _ptr(rc))
    if code != EPX_OK:
        bad = int(np.nonzero(rc)[0][0])
        raise EpxError(int(rc[bad]), f"context {bad}: {ctxs[bad].last_error()}")
    return out


def measure_fp64_peak(kind: int, ms_target: float = 50.0, device: int = 0) -> float:
    """TFLOP/s of the DFMA (kind 0) or DMMA m8n8k4 (kind 1) pipe, measured by a register-only kernel."""
    import torch
    scratch = torch.zeros(8, dtype=torch.uint8, device=torch.device("cuda", device))
    v = ct.c_double()
    rc = lib().epx_measure_fp64_peak(device, kind, float(ms_target), ct.c_void_p(scratch.data_ptr()),
                                     ct.c_void_p(torch.cuda.current_stream(device).cuda_stream), ct.byref(v))
    if rc != EPX_OK:
        raise EpxError(rc, "epx_measure_fp64_peak")
    return v.value


def segment_branches_static(tau, child_height, parent_height, seg_off, seg_epoch, seg_dur, stream=None) -> None:
    """epx_segment_branches_static: split a branch list into per-epoch segments without allocating anything on the device.

    For code that has device buffers for its inputs and results but may not ask CUDA for more memory (it runs under a host
    program's fixed memory budget, or where an allocation's device-wide synchronisation is unwelcome).  Every argument is
    a CUDA tensor the CALLER made, all on one device: ``tau`` float64 [M-1] (may be empty), ``child_height`` /
    ``parent_height`` float64 [n_br], outputs ``seg_off`` int32 [n_br+1], ``seg_epoch`` int32 [cap], ``seg_dur`` float64
    [cap].  This wrapper passes their addresses and sizes on and creates no tensor; the intermediates live in a fixed array
    inside libepx.so, so n_br <= EPX_STATIC_MAX_BRANCHES (EpxError with code EPX_E_WORKSPACE otherwise).  Work is enqueued
    on ``stream`` (default: the device's current torch stream) and not synchronised.  The first call on a device also looks
    the array's address up: make it at start-up, outside stream capture.  Calls that can overlap on the GPU share that
    array and race; calls that run one after the other are independent (see include/epx.h)."""
    import torch
    dev = child_height.device
    for t, dt in ((tau, torch.float64), (child_height, torch.float64), (parent_height, torch.float64),
                  (seg_off, torch.int32), (seg_epoch, torch.int32), (seg_dur, torch.float64)):
        if not (t.is_cuda and t.device == dev and t.dtype == dt and t.is_contiguous() and t.dim() == 1):
            raise ValueError("segment_branches_static takes contiguous 1-d CUDA tensors on one device (float64 / int32 as documented)")
    n_br, M = child_height.numel(), tau.numel() + 1
    if parent_height.numel() != n_br or seg_off.numel() != n_br + 1 or seg_epoch.numel() != seg_dur.numel():
        raise ValueError("segment_branches_static: tensor sizes do not match")
    cap = seg_epoch.numel()
    if stream is None:
        stream = torch.cuda.current_stream(dev)
    msg = ct.create_string_buffer(256)
    rc = lib().epx_segment_branches_static(
        dev.index, n_br, M, ct.c_void_p(tau.data_ptr() if M > 1 else None),
        ct.c_void_p(child_height.data_ptr() if n_br else None), ct.c_void_p(parent_height.data_ptr() if n_br else None),
        ct.c_void_p(seg_off.data_ptr()), ct.c_void_p(seg_epoch.data_ptr() if cap else None),
        ct.c_void_p(seg_dur.data_ptr() if cap else None), cap, ct.c_void_p(stream.cuda_stream), msg, len(msg))
    if rc != EPX_OK:
        raise EpxError(rc, msg.value.decode())
