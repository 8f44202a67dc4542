"""CPU oracle for WEST's per-sample steps -- TEST INFRASTRUCTURE ONLY.

Plain numpy, fp64, in the paper's order and notation; shares nothing with the CUDA path. Only
tests/ may import it.

What it states:

* PAPER.md:89-94 (Sec. 4.1.1, Eq. 1) / Alg. 1 l.9-10: block significance
      S(u,v) = (1/B^2) * sum_{p in B_u} sum_{q in B_v} A(p,q),   A = softmax(scale * Q K^T)
  of one head of one calibration sample (rows of A sum to 1 over the valid keys).
* Alg. 1 l.12-17, "Local Threshold Discovery" and "Topology Union":
      sort S and compute the cumulative sum C;
      for each p in P find the cutoff tau s.t. C[tau] ~ p;
      L(u,v) = min{p in P | block (u,v) is active at p};      T <- min(T, L).

Readings taken (P18-P20):
  - keys >= n_valid carry zero weight and query rows >= n_valid are left out of the block sums
    (they are padding, not calibration data); the divisor stays B^2 as printed.
  - the sort is descending (largest blocks first), ties in flat-index order (stable); C is the
    inclusive cumulative sum divided by its total, so that p in (0,1] is a fraction of the head's
    attention mass ("C[tau] ~ p" with C a cumulative sum only makes sense for a mass fraction).
  - tau(p) is the FIRST position with C[tau] >= p (the smallest prefix that reaches p; when rounding
    keeps the last C below p, tau is the last position); the blocks at sorted positions 0..tau are
    active at p. A block active at no p in P keeps L = 1.0, the map's initial "max value"
    (PAPER.md:389).
"""
import numpy as np


def softmax_rows(q, k, scale, n_valid):
    """A = softmax(scale * q k^T) over the valid keys, fp64. q, k: [N][D] float64."""
    s = scale * (q @ k.T)
    s[:, n_valid:] = -np.inf
    m = s.max(axis=1, keepdims=True)
    e = np.exp(s - m)
    return e / e.sum(axis=1, keepdims=True)


def block_significance(q, k, scale, B, n_valid=None):
    """Eq. 1 for one head of one sample. q, k: [N][D] (any float dtype; widened to fp64).
    Returns S float64 [N/B][N/B]."""
    q = np.asarray(q, dtype=np.float64)
    k = np.asarray(k, dtype=np.float64)
    N = q.shape[0]
    assert N % B == 0
    n_valid = N if n_valid is None else int(n_valid)
    A = softmax_rows(q, k, float(scale), n_valid)
    nb = N // B
    S = np.zeros((nb, nb), dtype=np.float64)
    for u in range(nb):
        for v in range(nb):
            acc = 0.0
            for p in range(u * B, min((u + 1) * B, n_valid)):     # padded query rows are left out
                acc += A[p, v * B:(v + 1) * B].sum()
            S[u, v] = acc / (B * B)
    return S


def local_threshold_map(S, P):
    """Alg. 1 l.12-15 for one head of one sample: the local map L. S [nbq][nbk] (non-negative),
    P the candidate thresholds (ascending, in (0,1])."""
    S = np.asarray(S, dtype=np.float64)
    P = [float(p) for p in P]
    assert all(0.0 < p <= 1.0 for p in P) and P == sorted(P)
    flat = S.reshape(-1)
    order = np.argsort(-flat, kind="stable")          # descending, ties in flat-index order
    C = np.cumsum(flat[order])
    C = C / C[-1]
    L = np.ones(flat.shape[0], dtype=np.float64)       # "max value" for blocks active at no p
    for p in reversed(P):                               # descending p: the smallest p is written last
        reach = np.nonzero(C >= p)[0]
        tau = int(reach[0]) if reach.size else flat.shape[0] - 1
        for r in range(tau + 1):
            L[order[r]] = p
    return L.reshape(S.shape)


def threshold_map_update(T, S, P):
    """Alg. 1 l.17: T <- min(T, L), L the local map of this sample."""
    return np.minimum(np.asarray(T, dtype=np.float64), local_threshold_map(S, P))
