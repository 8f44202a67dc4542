"""CPU oracle for mask instantiation from a threshold map -- TEST INFRASTRUCTURE ONLY.

Plain numpy, fp64, written out in the paper's order and notation; shares nothing with the CUDA
path and imports nothing from paper_2606_23019_b200. Only tests/ may import it.

What it states:

* PAPER.md:103 (Sec. 4.1.2) / Alg. 1 l.31: a binary mask for a target density p is
  instantiated by the comparison  M_p = 1(T <= p),  T the threshold map of one head.
* PAPER.md:165-171 (Sec. 4.3.1, Eq. 7): a map built at a base resolution is reused at a target
  resolution by "conservative bilinear interpolation with a ceiling rule",
      R_target(u, v) = ceil( Phi(R_base, u / s_h, v / s_w) ),
  "ensuring that any overlap with active regions is preserved".

Readings taken (P14-P16):
  - R in Eq. 7 is the binary ACTIVE-REGION mask R_base = M_p at the base resolution (the sentence
    after Eq. 7 speaks of "active regions", and rounding a threshold UP would drop blocks, the
    opposite of conservative); the brackets, garbled to [ ] in the extracted text, are the
    ceiling the sentence before Eq. 7 names. ceil of a bilinear blend of 0/1 values is 1 exactly
    when some base cell with positive interpolation weight is active.
  - s_h = NQB / nbq and s_w = NKB / nbk (target / base size along the query-block and key-block
    axes); Phi samples at the point (u / s_h, v / s_w) = (u * nbq / NQB, v * nbk / NKB) in base
    index coordinates (no half-cell offset: Eq. 7 has none), the right / lower neighbour clamped
    to the last cell.
  - the comparison T <= p is done on the fp32 values as given (both sides receive fp32).
"""
import math

import numpy as np


def mask_at(T, p):
    """M_p = 1(T <= p) for one head. T float32 [nbq][nbk], p float32 scalar."""
    T = np.asarray(T, dtype=np.float32)
    return (T <= np.float32(p)).astype(np.float64)


def phi(R, x, y):
    """Bilinear interpolation Phi(R, x, y) of the 2-D array R at the real-valued index point
    (x, y) (row coordinate x, column coordinate y), neighbours clamped to the last cell."""
    n0, n1 = R.shape
    x0 = int(math.floor(x))
    y0 = int(math.floor(y))
    fx = x - x0
    fy = y - y0
    x1 = min(x0 + 1, n0 - 1)
    y1 = min(y0 + 1, n1 - 1)
    return ((1.0 - fx) * (1.0 - fy) * R[x0, y0] + (1.0 - fx) * fy * R[x0, y1]
            + fx * (1.0 - fy) * R[x1, y0] + fx * fy * R[x1, y1])


def resize_conservative(R_base, NQB, NKB):
    """Eq. 7: R_target(u,v) = ceil(Phi(R_base, u/s_h, v/s_w)) for a 0/1 map."""
    R_base = np.asarray(R_base, dtype=np.float64)
    nbq, nbk = R_base.shape
    out = np.zeros((NQB, NKB), dtype=np.float64)
    for u in range(NQB):
        x = (u * nbq) / NQB            # = u / s_h with s_h = NQB / nbq
        for v in range(NKB):
            y = (v * nbk) / NKB        # = v / s_w
            out[u, v] = math.ceil(phi(R_base, x, y))
    return out


def mask_from_threshold(T_base, p_star, NQB, NKB, force_diag):
    """Dense 0/1 block mask [H][NQB][NKB] (uint8) of every head at the target resolution:
    M_{p*_h} at the base resolution, resized by Eq. 7 when the sizes differ;
    force_diag sets (u,u) afterwards (BASELINE.json: "diagonal always on")."""
    T_base = np.asarray(T_base, dtype=np.float32)
    p_star = np.asarray(p_star, dtype=np.float32)
    H, nbq, nbk = T_base.shape
    assert p_star.shape == (H,)
    out = np.zeros((H, NQB, NKB), dtype=np.uint8)
    for h in range(H):
        R = mask_at(T_base[h], p_star[h])
        if (nbq, nbk) != (NQB, NKB):
            R = resize_conservative(R, NQB, NKB)
        out[h] = R.astype(np.uint8)
        if force_diag:
            for u in range(min(NQB, NKB)):
                out[h, u, u] = 1
    return out
