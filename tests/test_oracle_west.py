"""Pins for oracle/west.py: block significance (Eq. 1) and the per-sample
threshold-map update (Alg. 1 l.12-17), against library routines, brute-force
restatements, closed forms and the invariants the definitions imply."""
import numpy as np
import torch

from oracle import west


def _qk(N, D, seed, scale_q=1.0):
    rng = np.random.Generator(np.random.PCG64(seed))
    return rng.standard_normal((N, D)) * scale_q, rng.standard_normal((N, D))


def test_block_significance_matches_torch_softmax_and_avg_pool():
    # Eq. 1 is the B x B average pooling of the attention matrix: two library routines
    N, D, B = 48, 8, 8
    q, k = _qk(N, D, 0, 1.5)
    A = torch.softmax(torch.from_numpy(0.3 * (q @ k.T)), dim=1)
    ref = torch.nn.functional.avg_pool2d(A[None, None], B)[0, 0].numpy()
    assert np.abs(west.block_significance(q, k, 0.3, B) - ref).max() < 1e-15


def test_block_significance_row_mass_and_padding():
    N, D, B, n_valid = 40, 4, 8, 35
    q, k = _qk(N, D, 1)
    S = west.block_significance(q, k, 0.5, B, n_valid)
    nb = N // B
    # every valid query row spreads mass 1 over the key blocks: row u of S sums to
    # (#valid rows in block u) / B^2
    for u in range(nb):
        rows = max(0, min((u + 1) * B, n_valid) - u * B)
        assert abs(S[u].sum() - rows / (B * B)) < 1e-14
    # padded keys get nothing: the last key block only holds keys 32..34
    A = west.softmax_rows(q, k, 0.5, n_valid)
    assert (A[:, n_valid:] == 0).all() and abs(A[:n_valid].sum() - n_valid) < 1e-12
    # closed form: q = 0 gives uniform rows, S(u,v) = rows_u * keys_v / (B^2 * n_valid)
    S0 = west.block_significance(np.zeros((N, D)), k, 0.5, B, n_valid)
    for u in range(nb):
        for v in range(nb):
            rows = max(0, min((u + 1) * B, n_valid) - u * B)
            keys = max(0, min((v + 1) * B, n_valid) - v * B)
            assert abs(S0[u, v] - rows * keys / (B * B * n_valid)) < 1e-15


def _local_map_brute(S, P):
    """Independent restatement: for every p decide the active set by its definition (the
    shortest prefix of the descending order whose mass fraction reaches p), then L = min p."""
    flat = S.reshape(-1).astype(np.float64)
    idx = sorted(range(flat.size), key=lambda i: (-flat[i], i))
    total = sum(flat[i] for i in idx)
    L = np.ones(flat.size)
    for p in P:
        acc, active = 0.0, []
        for i in idx:
            active.append(i)
            acc += flat[i]
            if acc / total >= p:
                break
        for i in active:
            L[i] = min(L[i], p)
    return L.reshape(S.shape)


def test_local_threshold_map_matches_brute_force_and_invariants():
    rng = np.random.Generator(np.random.PCG64(2))
    P = [float(np.float32(x)) for x in np.linspace(0.05, 0.95, 19)]
    for shape in [(4, 4), (7, 5), (12, 12)]:
        S = rng.random(shape) ** 4            # heavy-tailed, like attention mass
        S[0, 0] = S[1, 1]                     # a tie
        L = west.local_threshold_map(S, P)
        assert np.array_equal(L, _local_map_brute(S, P))
        flat, Lf = S.reshape(-1), L.reshape(-1)
        for p in P:
            act = Lf <= p
            assert flat[act].sum() / flat.sum() >= p - 1e-12            # the active set reaches p ...
            order = np.argsort(-flat, kind="stable")
            kept = int(act.sum())
            assert set(order[:kept].tolist()) == set(np.nonzero(act)[0].tolist())   # ... is a prefix ...
            if kept > 1:
                assert flat[order[:kept - 1]].sum() / flat.sum() < p            # ... and the shortest one
        # larger blocks never get a larger threshold
        o = np.argsort(-flat, kind="stable")
        assert (np.diff(Lf[o]) >= 0).all()
        assert L.flat[int(np.argmax(flat))] == P[0]


def test_local_map_closed_forms():
    # one dominant block holding 90% of the mass: it alone is active up to p = 0.9
    S = np.full((3, 3), 0.1 / 8)
    S[1, 2] = 0.9
    P = [0.5, 0.9, 0.95, 1.0]
    L = west.local_threshold_map(S, P)
    assert L[1, 2] == 0.5
    assert sorted(L.reshape(-1).tolist()) == [0.5] + [0.95] * 4 + [1.0] * 4
    # equal blocks: ties go in flat-index order
    L = west.local_threshold_map(np.ones((2, 2)), [0.25, 0.5, 0.75, 1.0])
    assert L.tolist() == [[0.25, 0.5], [0.75, 1.0]]
    # a block active at no p keeps the initial value 1.0
    L = west.local_threshold_map(np.array([[0.6, 0.4]]), [0.5])
    assert L.tolist() == [[0.5, 1.0]]


def test_topology_union_is_elementwise_min():
    rng = np.random.Generator(np.random.PCG64(3))
    P = [0.2, 0.4, 0.6, 0.8, 1.0]
    T = np.ones((5, 5))
    maps = []
    for _ in range(3):
        S = rng.random((5, 5)) ** 3
        maps.append(west.local_threshold_map(S, P))
        T = west.threshold_map_update(T, S, P)
    assert np.array_equal(T, np.minimum.reduce(maps))
    # "include block if active in any sample": M_p(T) is the union of the samples' active sets
    for p in P:
        union = np.zeros((5, 5), dtype=bool)
        for L in maps:
            union |= L <= p
        assert np.array_equal(T <= p, union)
