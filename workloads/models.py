"""Textbook substitution-model INPUT builders (rate matrices, frequencies, gamma rates).

The paper only names these models (HKY PAPER.md:L139, GY94 L147, asymmetric
discrete-trait Q L26, "rate mixtures with C categories" L72); the library takes a
finished Q per epoch, so these live with the input generators, not with the method.
"""
from __future__ import annotations

import numpy as np
from scipy import special, stats

NUCS = "TCAG"
# universal genetic code, codons in TCAG order (first position slowest)
AA_TCAG = "FFLLSSSSYY**CC*WLLLLPPPPHHQQRRRRIIIMTTTTNNKKSSRRVVVVAAAADDEEGGGG"
assert len(AA_TCAG) == 64 and AA_TCAG.count("*") == 3


def complete_diagonal(Q: np.ndarray) -> np.ndarray:
    Q = np.array(Q, dtype=np.float64, copy=True)
    np.fill_diagonal(Q, 0.0)
    np.fill_diagonal(Q, -Q.sum(axis=1))
    return Q


def normalise(Q: np.ndarray, pi: np.ndarray) -> np.ndarray:
    """Scale Q to one expected substitution per unit time: -sum_i pi_i q_ii = 1."""
    Q = complete_diagonal(Q)
    rate = -float(np.dot(pi, np.diag(Q)))
    return complete_diagonal(Q / rate)


def gtr(exch6: np.ndarray, pi: np.ndarray) -> np.ndarray:
    """General time-reversible 4-state Q: q_ij = s_ij * pi_j, s symmetric (6 exchangeabilities)."""
    S = np.zeros((4, 4))
    iu = np.triu_indices(4, 1)
    S[iu] = exch6
    S = S + S.T
    return normalise(S * pi[None, :], pi)


def gtr_k(exch: np.ndarray, pi: np.ndarray) -> np.ndarray:
    """General time-reversible K-state Q (amino-acid style): q_ij = s_ij * pi_j with K (K-1) / 2 exchangeabilities."""
    K = pi.shape[0]
    S = np.zeros((K, K))
    iu = np.triu_indices(K, 1)
    S[iu] = exch
    S = S + S.T
    return normalise(S * pi[None, :], pi)


def hky(kappa: float, pi: np.ndarray) -> np.ndarray:
    """HKY85 in TCAG order: transitions T<->C and A<->G get kappa."""
    S = np.ones((4, 4))
    S[0, 1] = S[1, 0] = kappa
    S[2, 3] = S[3, 2] = kappa
    return normalise(S * pi[None, :], pi)


def jc69() -> np.ndarray:
    return normalise(np.ones((4, 4)), np.full(4, 0.25))


def equal_input(pi: np.ndarray) -> np.ndarray:
    """K-state F81 / equal-input model: q_ij = pi_j (i != j), normalised."""
    K = pi.shape[0]
    return normalise(np.tile(pi[None, :], (K, 1)), pi)


def sense_codons():
    """List of the 61 sense codons as (n1,n2,n3) index triples in TCAG order, plus their amino acids."""
    trip, aa = [], []
    for c in range(64):
        if AA_TCAG[c] != "*":
            trip.append((c // 16, (c // 4) % 4, c % 4))
            aa.append(AA_TCAG[c])
    return trip, aa


def f3x4(pos_freqs: np.ndarray) -> np.ndarray:
    """Codon frequencies from 3 per-position nucleotide distributions, renormalised over sense codons."""
    trip, _ = sense_codons()
    pi = np.array([pos_freqs[0, a] * pos_freqs[1, b] * pos_freqs[2, c] for a, b, c in trip])
    return pi / pi.sum()


def _is_transition(a: int, b: int) -> bool:
    return {a, b} in ({0, 1}, {2, 3})  # T<->C, A<->G


def gy94(omega: float, kappa: float, pi: np.ndarray) -> np.ndarray:
    """Goldman-Yang 1994 codon model (61 sense codons): q_ij = 0 if the codons differ at more than one
    position, else pi_j * (kappa if transition) * (omega if non-synonymous); normalised."""
    trip, aa = sense_codons()
    K = len(trip)
    Q = np.zeros((K, K))
    for i in range(K):
        for j in range(K):
            if i == j:
                continue
            diff = [p for p in range(3) if trip[i][p] != trip[j][p]]
            if len(diff) != 1:
                continue
            p = diff[0]
            r = pi[j]
            if _is_transition(trip[i][p], trip[j][p]):
                r *= kappa
            if aa[i] != aa[j]:
                r *= omega
            Q[i, j] = r
    return normalise(Q, pi)


def asymmetric_trait(rng: np.random.Generator, K: int, shape: float = 0.5, keep: float = 0.3) -> np.ndarray:
    """Sparse asymmetric discrete-trait Q: Gamma(shape,1) rates times a Bernoulli(keep) mask, with the cycle
    i -> (i+1) mod K forced on so the chain is irreducible; NOT normalised."""
    R = rng.gamma(shape, 1.0, size=(K, K))
    mask = rng.random((K, K)) < keep
    for i in range(K):
        mask[i, (i + 1) % K] = True
    R = np.where(mask, R, 0.0)
    # a forced-on entry that drew (numerically) zero would break irreducibility
    for i in range(K):
        j = (i + 1) % K
        if R[i, j] < 1e-3:
            R[i, j] = 1e-3
    return complete_diagonal(R)


def stationary(Q: np.ndarray) -> np.ndarray:
    """Stationary vector of an irreducible Q: pi Q = 0, sum pi = 1 (least squares on the augmented system)."""
    K = Q.shape[0]
    A = np.vstack([Q.T, np.ones((1, K))])
    b = np.zeros(K + 1)
    b[-1] = 1.0
    pi, *_ = np.linalg.lstsq(A, b, rcond=None)
    pi = np.clip(pi, 0.0, None)
    return pi / pi.sum()


def discrete_gamma(alpha: float, C: int):
    """Yang (1994) discrete gamma, mean of each equal-probability category; mean rate 1. Returns (rates, weights)."""
    if C == 1:
        return np.ones(1), np.ones(1)
    cuts = stats.gamma.ppf(np.arange(1, C) / C, a=alpha, scale=1.0 / alpha)
    cuts = np.concatenate([[0.0], cuts, [np.inf]])
    # integral of x*g(x) over [a,b] with g = Gamma(alpha, rate alpha) equals I(b*alpha; alpha+1) - I(a*alpha; alpha+1)
    upper = special.gammainc(alpha + 1.0, cuts[1:] * alpha)
    lower = special.gammainc(alpha + 1.0, cuts[:-1] * alpha)
    rates = (upper - lower) * C
    return rates.astype(np.float64), np.full(C, 1.0 / C)
