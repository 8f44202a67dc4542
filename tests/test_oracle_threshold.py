"""Pins for oracle/threshold.py (mask instantiation M_p = 1(T <= p), and the
conservative resize of Eq. 7) against things other than itself: a library
interpolation routine, brute-force restatements in integer arithmetic, closed forms and the
invariants the paper states ("any overlap with active regions is preserved"; nested masks)."""
import numpy as np
import pytest
import torch

from oracle import threshold as th


def _rand_T(H, nbq, nbk, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    # thresholds on a discrete grid of levels, as the paper's candidate set P
    return (rng.integers(1, 49, size=(H, nbq, nbk)) / 48.0).astype(np.float32)


def test_same_size_is_the_plain_comparison():
    T = _rand_T(3, 7, 9, 0)
    p = np.array([0.25, 0.5, 1.0], dtype=np.float32)
    got = th.mask_from_threshold(T, p, 7, 9, force_diag=False)
    for h in range(3):
        for u in range(7):
            for v in range(9):
                assert got[h, u, v] == (1 if T[h, u, v] <= p[h] else 0)
    # p = 1 keeps every block (thresholds are <= 1, PAPER.md:389 initial value 1.0)
    assert got[2].all()


def test_masks_are_nested_in_p():
    # Eq. 2 "encodes the full sparsity hierarchy": p1 <= p2 => M_p1 subset of M_p2, at any size
    T = _rand_T(1, 6, 6, 1)
    prev = np.zeros((1, 15, 15), dtype=np.uint8)
    for p in (0.1, 0.3, 0.6, 0.9, 1.0):
        cur = th.mask_from_threshold(T, np.array([p], np.float32), 15, 15, force_diag=False)
        assert (cur >= prev).all()
        prev = cur


def test_phi_matches_torch_grid_sample():
    # Phi is plain bilinear interpolation at the point (x, y): torch's grid_sample with
    # align_corners=True samples exactly at normalised coordinates 2x/(n-1) - 1, border-clamped.
    rng = np.random.Generator(np.random.PCG64(2))
    R = rng.random((5, 7))
    pts = [(0.0, 0.0), (1.25, 3.5), (3.999, 5.2), (4.0, 6.0), (2.5, 0.75), (0.3, 5.9)]
    grid = torch.tensor([[[[2 * y / 6 - 1, 2 * x / 4 - 1] for (x, y) in pts]]], dtype=torch.float64)
    ref = torch.nn.functional.grid_sample(torch.from_numpy(R)[None, None], grid, mode="bilinear",
                                          padding_mode="border", align_corners=True)[0, 0, 0]
    for (x, y), r in zip(pts, ref.tolist()):
        assert abs(th.phi(R, x, y) - r) < 1e-12


def _dilate_integer(Rb, NQB, NKB):
    """Independent restatement in integer arithmetic: the target cell is on iff one of the base
    cells with positive bilinear weight is on. Cell a0 = (u*nbq)//NQB always has positive weight;
    its successor has positive weight iff (u*nbq) % NQB != 0 (and it exists)."""
    nbq, nbk = Rb.shape
    out = np.zeros((NQB, NKB), dtype=np.uint8)
    for u in range(NQB):
        a0, ra = divmod(u * nbq, NQB)
        rows = [a0] + ([a0 + 1] if ra != 0 and a0 + 1 < nbq else [])
        for v in range(NKB):
            b0, rb = divmod(v * nbk, NKB)
            cols = [b0] + ([b0 + 1] if rb != 0 and b0 + 1 < nbk else [])
            out[u, v] = 1 if any(Rb[a, b] for a in rows for b in cols) else 0
    return out


@pytest.mark.parametrize("nbq,nbk,NQB,NKB", [(4, 4, 8, 8), (5, 7, 12, 9), (8, 8, 5, 3), (6, 6, 6, 13),
                                             (1, 1, 4, 4), (16, 16, 37, 37)])
def test_resize_equals_integer_dilation(nbq, nbk, NQB, NKB):
    rng = np.random.Generator(np.random.PCG64(nbq * 100 + NQB))
    Rb = (rng.random((nbq, nbk)) < 0.3).astype(np.float64)
    got = th.resize_conservative(Rb, NQB, NKB)
    assert set(np.unique(got)) <= {0.0, 1.0}
    assert (got.astype(np.uint8) == _dilate_integer(Rb, NQB, NKB)).all()


def test_resize_preserves_every_active_region():
    # "ensuring that any overlap with active regions is preserved": every target
    # cell whose sampling point falls inside an active base cell is active.
    rng = np.random.Generator(np.random.PCG64(5))
    Rb = (rng.random((9, 9)) < 0.2).astype(np.float64)
    for NB in (9, 14, 27, 40):
        got = th.resize_conservative(Rb, NB, NB)
        for u in range(NB):
            for v in range(NB):
                if Rb[(u * 9) // NB, (v * 9) // NB]:
                    assert got[u, v] == 1.0
        # and never more than the 2x2 neighbourhood allows: an all-zero map stays all-zero
    assert not th.resize_conservative(np.zeros((4, 4)), 11, 11).any()
    assert th.resize_conservative(np.ones((4, 4)), 11, 11).all()


def test_integer_upscale_by_two_closed_form():
    # s = 2: even target indices sit exactly on base cells, odd ones half-way between two.
    Rb = np.zeros((4, 4))
    Rb[1, 2] = 1.0
    got = th.resize_conservative(Rb, 8, 8)
    on = {(u, v) for u in range(8) for v in range(8) if got[u, v]}
    assert on == {(u, v) for u in (1, 2, 3) for v in (3, 4, 5)}


def test_force_diag_and_per_head_threshold():
    T = np.ones((2, 3, 3), dtype=np.float32)
    T[0, 0, 2] = 0.25
    T[1, 2, 0] = 0.5
    got = th.mask_from_threshold(T, np.array([0.25, 0.25], np.float32), 3, 3, force_diag=True)
    assert got[0].tolist() == [[1, 0, 1], [0, 1, 0], [0, 0, 1]]
    assert got[1].tolist() == [[1, 0, 0], [0, 1, 0], [0, 0, 1]]
