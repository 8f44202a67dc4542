"""CPU oracle for FAST's fidelity score -- TEST INFRASTRUCTURE ONLY.

Plain numpy, fp64, the definitions written out; shares nothing with the CUDA path. Only tests/
may import it.

What it states:

* PAPER.md:113-116 (Sec. 4.2.1, Eq. 3): Hellinger distance of two discrete distributions,
      H(P, Q) = (1 / sqrt(2)) * sqrt( sum_i (sqrt(p_i) - sqrt(q_i))^2 ).
* PAPER.md:132-134 (Eq. 4): Fidelity Score  F(P, P~) = 1 - H(P, P~)  of the dense attention
  distribution P of a query row and its sparse approximation P~.
* PAPER.md:155-159 (Sec. 4.2.3): the score is evaluated on a stratified sample of rows (the row
  indices are drawn by the caller and passed in) and averaged.

Reading taken (P17): P~ is the softmax over the KEPT keys only (the
distribution the sparse kernel actually applies: its weights sum to 1), zero elsewhere.
"""
import math

import numpy as np


def hellinger(p, q):
    """Eq. 3, as printed."""
    p = np.asarray(p, dtype=np.float64)
    q = np.asarray(q, dtype=np.float64)
    assert p.shape == q.shape
    acc = 0.0
    for pi, qi in zip(p.tolist(), q.tolist()):
        d = math.sqrt(pi) - math.sqrt(qi)
        acc += d * d
    return math.sqrt(acc) / math.sqrt(2.0)


def fidelity(p, q):
    """Eq. 4."""
    return 1.0 - hellinger(p, q)


def mean_fidelity(P_rows, Pt_rows):
    """Average Fidelity Score over the sampled rows (Sec. 4.2.3). P_rows, Pt_rows: [n][N]."""
    assert len(P_rows) == len(Pt_rows) and len(P_rows) > 0
    return sum(fidelity(p, q) for p, q in zip(P_rows, Pt_rows)) / len(P_rows)
