"""ctypes front-end of the CPU oracle (``epoch_oracle.c``) -- TEST INFRASTRUCTURE ONLY.

Only tests/, ``__graft_entry__.smoke()`` and bench.py's ``cpu_baseline`` / ``--impl reference`` legs may import
this package.  It imports nothing from the CUDA product and nothing from ``workloads`` (problems are read by
attribute).  Two builds of the one C source: ``"ld"`` (80-bit long double, the parity referee) and ``"d"``
(double, the timed CPU baseline, "as it stands"); a third, ``"q"`` (binary128), exists only to pin the referee's own
rounding error (tests/test_oracle_pins.py).
"""
from __future__ import annotations

import ctypes as ct
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "epoch_oracle.c")
_LIBS = {"ld": os.path.join(_HERE, "liborc_ld.so"), "d": os.path.join(_HERE, "liborc_d.so"), "q": os.path.join(_HERE, "liborc_q.so")}
_FLAGS = {"ld": ["-DORC_LONG_DOUBLE"], "d": [], "q": ["-DORC_QUAD"]}
_REAL_BYTES = {"ld": 16, "d": 8, "q": 16}
# ORC_SANITIZE=1: separate builds with AddressSanitizer + UndefinedBehaviorSanitizer (the process must preload libasan;
# tests/test_oracle_pins.py runs the pins' inputs through them in a subprocess).  Same source, same arithmetic.
_SAN = os.environ.get("ORC_SANITIZE") == "1"
if _SAN:
    _LIBS = {k: v.replace(".so", "_san.so") for k, v in _LIBS.items()}
    _FLAGS = {k: v + ["-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer", "-g"]
              for k, v in _FLAGS.items()}
_lock = threading.Lock()
_loaded: dict = {}


def build(force: bool = False) -> None:
    """Compile both builds of the oracle with gcc (no GPU, no nvcc)."""
    for prec, path in _LIBS.items():
        if not force and os.path.exists(path) and os.path.getmtime(path) >= os.path.getmtime(_SRC):
            continue
        cmd = ["gcc"] + _FLAGS[prec] + ["-O2", "-fopenmp", "-fPIC", "-shared", "-o", path, _SRC, "-lm"]
        if prec == "q":
            cmd.append("-lquadmath")
        subprocess.run(cmd, check=True)


def _lib(prec: str):
    with _lock:
        if prec not in _loaded:
            build()
            lib = ct.CDLL(_LIBS[prec])
            lib.orc_real_bytes.restype = ct.c_int
            want = _REAL_BYTES[prec]
            if lib.orc_real_bytes() != want:
                raise RuntimeError(f"oracle build {prec}: REAL is {lib.orc_real_bytes()} bytes, expected {want}")
            _loaded[prec] = lib
        return _loaded[prec]


def _p(a):
    return a.ctypes.data_as(ct.c_void_p)


class Oracle:
    """One precision of the oracle. ``real`` is the numpy dtype its REAL arrays use."""

    def __init__(self, precision: str = "ld"):
        assert precision in ("ld", "d", "q")
        self.precision = precision
        self.lib = _lib(precision)
        # "q" (binary128): numpy has no such type, so REAL arrays are opaque 16-byte cells on the Python side and results are
        # read back rounded to long double (_out); only evaluate() / branch_matrices / log_likelihood serve this build
        self.real = {"ld": np.longdouble, "d": np.float64, "q": np.dtype("V16")}[precision]

    def _out(self, a):
        """A REAL array as numbers numpy can compute with (binary128 -> long double by orc_real_to_ld; others unchanged)."""
        if self.precision != "q" or a is None:
            return a
        a = np.ascontiguousarray(a)
        out = np.zeros(a.shape, dtype=np.longdouble)
        self.lib.orc_real_to_ld(ct.c_size_t(a.size), _p(a), _p(out))
        return out

    # ---- O2
    def segments(self, child_h, parent_h, tau):
        child_h = np.ascontiguousarray(child_h, dtype=np.float64)
        parent_h = np.ascontiguousarray(parent_h, dtype=np.float64)
        tau = np.ascontiguousarray(tau, dtype=np.float64)
        n_br, M = child_h.shape[0], tau.shape[0] + 1
        cap = n_br * M + 1
        off = np.zeros(n_br + 1, dtype=np.int32)
        ep = np.zeros(cap, dtype=np.int32)
        du = np.zeros(cap, dtype=np.float64)
        n = self.lib.orc_segments(n_br, _p(child_h), _p(parent_h), M, _p(tau), _p(off), _p(ep), _p(du), cap)
        if n < 0:
            raise RuntimeError("orc_segments: capacity")
        return off, ep[:n].copy(), du[:n].copy()

    def epoch_of_parent_end(self, h, tau) -> int:
        tau = np.ascontiguousarray(tau, dtype=np.float64)
        return int(self.lib.orc_epoch_of_parent_end(ct.c_double(float(h)), tau.shape[0] + 1, _p(tau)))

    # ---- O3 / O3'
    def expm(self, A, method: str = "taylor"):
        A = np.ascontiguousarray(A, dtype=self.real)
        K = A.shape[0]
        out = np.zeros((K, K), dtype=self.real)
        if method == "taylor":
            self.lib.orc_expm_taylor(K, _p(A), _p(out))
        elif method == "uniformisation":
            it = self.lib.orc_expm_uniformisation(K, _p(A), _p(out), 100000)
            if it < 0:
                raise RuntimeError("uniformisation did not converge")
        else:
            raise ValueError(method)
        return out

    # ---- O3 + O4
    def branch_matrices(self, Q, rates, seg_off, seg_epoch, seg_dur, raw: bool = False):
        Q = np.ascontiguousarray(Q, dtype=np.float64)
        rates = np.ascontiguousarray(rates, dtype=np.float64)
        seg_off = np.ascontiguousarray(seg_off, dtype=np.int32)
        seg_epoch = np.ascontiguousarray(seg_epoch, dtype=np.int32)
        seg_dur = np.ascontiguousarray(seg_dur, dtype=np.float64)
        M, K = Q.shape[0], Q.shape[1]
        C, n_br = rates.shape[0], seg_off.shape[0] - 1
        P = np.zeros((n_br, C, K, K), dtype=self.real)
        rc = self.lib.orc_branch_matrices(K, M, C, _p(Q), _p(rates), n_br, _p(seg_off), _p(seg_epoch), _p(seg_dur), _p(P))
        if rc != 0:
            raise RuntimeError(f"orc_branch_matrices rc={rc}")
        return P if raw else self._out(P)       # raw: REAL cells as the C side wrote them (input of log_likelihood)

    # ---- O5 + O6
    def log_likelihood(self, parent, P, tip_states, root_freqs, cat_weights, pattern_weights=None,
                       want_partials: bool = False, tip_partials=None):
        """`tip_partials`: {tip index: array [L][K]} -- tip vectors of partially observed tips, used
        instead of the indicator of the tip's state."""
        parent = np.ascontiguousarray(parent, dtype=np.int32)
        P = np.ascontiguousarray(P, dtype=self.real)
        tips = np.ascontiguousarray(tip_states, dtype=np.int32)
        root_freqs = np.ascontiguousarray(root_freqs, dtype=np.float64)
        cat_weights = np.ascontiguousarray(cat_weights, dtype=np.float64)
        N, L = tips.shape
        n_nodes, C, K = P.shape[0], P.shape[1], P.shape[2]
        assert n_nodes == 2 * N - 1 and parent.shape[0] == n_nodes
        wt = None if pattern_weights is None else np.ascontiguousarray(pattern_weights, dtype=np.float64)
        site = np.zeros(L, dtype=self.real)
        lnl = np.zeros(1, dtype=self.real)
        partials = np.zeros((n_nodes, C, L, K), dtype=self.real) if want_partials else None
        tp = has = None
        if tip_partials:
            tp = np.zeros((N, L, K), dtype=np.float64)
            has = np.zeros(N, dtype=np.uint8)
            for t, v in tip_partials.items():
                tp[t] = np.asarray(v, dtype=np.float64).reshape(L, K)
                has[t] = 1
        rc = self.lib.orc_log_likelihood_tp(K, C, N, L, _p(parent), _p(P), _p(tips), _p(root_freqs), _p(cat_weights),
                                            None if wt is None else _p(wt), _p(site), _p(lnl),
                                            None if partials is None else _p(partials),
                                            None if tp is None else _p(tp), None if has is None else _p(has))
        if rc != 0:
            raise RuntimeError(f"orc_log_likelihood rc={rc}")
        return {"lnl": self._out(lnl)[0], "site_lnl": self._out(site), "partials": self._out(partials)}

    # ---- O1
    def validate_model(self, Q, freqs, reversible: bool) -> int:
        Q = np.ascontiguousarray(Q, dtype=np.float64)
        freqs = np.ascontiguousarray(freqs, dtype=np.float64)
        return int(self.lib.orc_validate_model(Q.shape[0], _p(Q), _p(freqs), int(bool(reversible))))

    def validate_tree(self, parent, height) -> int:
        parent = np.ascontiguousarray(parent, dtype=np.int32)
        height = np.ascontiguousarray(height, dtype=np.float64)
        return int(self.lib.orc_validate_tree((parent.shape[0] + 1) // 2, _p(parent), _p(height)))

    # ---- whole path on a problem object (duck-typed: tau, Q, rates, parent, height, ...)
    def evaluate(self, prob, want_partials: bool = False, branches=None, tip_partials=None):
        """Run O2..O6 on a problem. `branches` (index array) restricts O3/O4 to a sample of matrix slots
        (branch-list problems / sampled parity); the likelihood is then skipped."""
        if prob.N > 0:
            ch = np.asarray(prob.height, dtype=np.float64).copy()
            ph = ch.copy()
            par = np.asarray(prob.parent)
            nz = par >= 0
            ph[nz] = ch[par[nz]]
        else:
            ch, ph = prob.child_height, prob.parent_height
        if branches is not None:
            ch, ph = np.asarray(ch)[branches], np.asarray(ph)[branches]
        off, ep, du = self.segments(ch, ph, prob.tau)
        P = self.branch_matrices(prob.Q, prob.rates, off, ep, du, raw=True)
        out = {"seg_off": off, "seg_epoch": ep, "seg_dur": du, "P": self._out(P)}
        if prob.N > 0 and branches is None:
            if prob.root_freqs is not None:
                rf = prob.root_freqs
            else:
                rf = prob.freqs[self.epoch_of_parent_end(np.max(prob.height), prob.tau)]
            out.update(self.log_likelihood(prob.parent, P, prob.tip_states, rf, prob.weights,
                                           prob.pattern_weights, want_partials, tip_partials))
            out["root_freqs"] = np.asarray(rf, dtype=np.float64)
        return out
