"""Container for one epoch-model likelihood problem (inputs only).

Conventions: time is measured as
HEIGHT, backwards from the most recent tip; parents are higher than children;
epoch e in 0..M-1 covers heights [tau_e, tau_{e+1}) with tau_0=-inf, tau_M=+inf,
so epoch 0 is the most recent one (PAPER.md:L78 read backwards in time).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np


@dataclass
class EpochProblem:
    name: str
    K: int                      # states
    M: int                      # epochs
    C: int                      # rate categories
    N: int                      # tips (0 = branch-list mode, no tree / likelihood)
    L: int                      # site patterns
    tau: np.ndarray             # (M-1,) f64 strictly increasing epoch boundaries (heights)
    Q: np.ndarray               # (M,K,K) f64 row-major, rows sum to 0
    freqs: np.ndarray           # (M,K) f64 equilibrium frequencies of each epoch's process
    reversible: bool            # all epochs reversible (Jacobi path) or not (Pade path)
    rates: np.ndarray           # (C,) category rates r_c
    weights: np.ndarray         # (C,) category weights w_c
    parent: Optional[np.ndarray] = None          # (2N-1,) i32, root = -1, tips are 0..N-1
    height: Optional[np.ndarray] = None          # (2N-1,) f64
    tip_states: Optional[np.ndarray] = None      # (N,L) i32; outside 0..K-1 = missing
    pattern_weights: Optional[np.ndarray] = None  # (L,) f64
    root_freqs: Optional[np.ndarray] = None      # (K,) f64 or None = freqs of the root's epoch
    child_height: Optional[np.ndarray] = None    # (n_br,) f64, branch-list mode
    parent_height: Optional[np.ndarray] = None   # (n_br,) f64, branch-list mode
    meta: dict = field(default_factory=dict)

    @property
    def n_nodes(self) -> int:
        return 2 * self.N - 1 if self.N > 0 else 0

    @property
    def n_br(self) -> int:
        """Number of matrix slots: one per node in tree mode (the root's is unused), else the branch list."""
        return self.n_nodes if self.N > 0 else int(self.child_height.shape[0])

    def branch_heights(self):
        """(child_height, parent_height) per matrix slot; the root slot gets parent = child (zero length)."""
        if self.N == 0:
            return self.child_height, self.parent_height
        ch = self.height.copy()
        ph = self.height.copy()
        nz = self.parent >= 0
        ph[nz] = self.height[self.parent[nz]]
        return ch, ph
