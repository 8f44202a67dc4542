"""Pins for oracle/fidelity.py (Hellinger distance Eq. 3 and Fidelity Score Eq. 4)
against a library routine, closed forms, the metric's stated properties (symmetric, bounded,
well-defined with zero-mass entries) and the identity the CUDA path relies on:
with P~ the softmax renormalised over the kept keys, H = sqrt(1 - sqrt(rho)), rho the retained
attention mass = exp(lse_sparse - lse_dense)."""
import math

import numpy as np
import scipy.spatial.distance as ssd

import oracle
from oracle import fidelity as fd
from paper_2606_23019_b200 import inputs


def _rand_dist(rng, n, zeros=0):
    p = rng.random(n) ** 3
    if zeros:
        p[rng.choice(n, size=zeros, replace=False)] = 0.0
    return p / p.sum()


def test_matches_scipy_euclidean_of_square_roots():
    rng = np.random.Generator(np.random.PCG64(0))
    for n in (2, 7, 300):
        p, q = _rand_dist(rng, n), _rand_dist(rng, n, zeros=n // 3)
        ref = ssd.euclidean(np.sqrt(p), np.sqrt(q)) / math.sqrt(2.0)
        assert abs(fd.hellinger(p, q) - ref) < 1e-14


def test_closed_forms_and_properties():
    rng = np.random.Generator(np.random.PCG64(1))
    p, q = _rand_dist(rng, 50), _rand_dist(rng, 50, zeros=20)
    assert fd.hellinger(p, p) == 0.0 and fd.fidelity(p, p) == 1.0
    assert abs(fd.hellinger(p, q) - fd.hellinger(q, p)) < 1e-15          # symmetric
    assert 0.0 <= fd.hellinger(p, q) <= 1.0                              # bounded
    assert abs(fd.hellinger([1, 0, 0], [0, 0.5, 0.5]) - 1.0) < 1e-15     # disjoint support
    # two-point distributions: H^2 = 1 - sqrt(ab) - sqrt((1-a)(1-b))
    a, b = 0.3, 0.8
    assert abs(fd.hellinger([a, 1 - a], [b, 1 - b]) ** 2
               - (1 - math.sqrt(a * b) - math.sqrt((1 - a) * (1 - b)))) < 1e-15
    # uniform over n vs uniform over the first m of them: H^2 = 1 - sqrt(m/n)
    n, m = 64, 16
    u, w = np.full(n, 1 / n), np.concatenate([np.full(m, 1 / m), np.zeros(n - m)])
    assert abs(fd.hellinger(u, w) ** 2 - (1 - math.sqrt(m / n))) < 1e-14


def test_retained_mass_identity_on_attention_rows():
    # dense softmax row P and its renormalised restriction P~ to the kept key blocks, both from the
    # attention oracle: H(P, P~) = sqrt(1 - sqrt(rho)), rho = exp(lse_sparse - lse_dense)
    D, blk, H, nblk = 16, 8, 2, 6
    N = blk * nblk
    g = np.random.Generator(np.random.PCG64(2))
    import torch
    q, k, v = [torch.from_numpy(g.standard_normal((1, H, N, D)).astype(np.float32)).to(torch.bfloat16)
               for _ in range(3)]
    m = g.random((H, nblk, nblk)) < 0.4
    m[:, np.arange(nblk), np.arange(nblk)] = True
    bits_s = oracle.pack_bool(m)
    bits_d = oracle.pack_bool(np.ones_like(m))
    qa, ka, va = inputs.as_u16(q), inputs.as_u16(k), inputs.as_u16(v)
    for h in range(H):
        for i in (0, 13, N - 1):
            Pd, _, lse_d = oracle.attn_row_weights(qa, ka, va, bits_d, blk, blk, 0.25, 0, h, i)
            Ps, _, lse_s = oracle.attn_row_weights(qa, ka, va, bits_s, blk, blk, 0.25, 0, h, i)
            assert abs(Pd.sum() - 1) < 1e-12 and abs(Ps.sum() - 1) < 1e-12
            rho = math.exp(lse_s - lse_d)
            assert 0 < rho <= 1 + 1e-15
            assert abs(fd.hellinger(Pd, Ps) - math.sqrt(max(0.0, 1 - math.sqrt(rho)))) < 1e-9


def test_mean_fidelity_is_the_plain_average():
    rng = np.random.Generator(np.random.PCG64(3))
    P = [_rand_dist(rng, 10) for _ in range(4)]
    Q = [_rand_dist(rng, 10, zeros=3) for _ in range(4)]
    assert abs(fd.mean_fidelity(P, Q) - np.mean([1 - fd.hellinger(p, q) for p, q in zip(P, Q)])) < 1e-15
