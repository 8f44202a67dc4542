"""Pins for the mask-packing oracle and the CRM bit layout. CPU only."""
import os

import numpy as np
import pytest
import torch

import oracle
from paper_2606_23019_b200 import inputs

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def alg2_iterate(words):
    """Algorithm 2 (CRM Forward Iterator) restated line by line; returns the
    sequence of INDEX values until the end sentinel. Test-local; not shared with any side."""
    ptr, end, val, base = 0, len(words), 0, -32

    def advance():
        nonlocal ptr, val, base
        while val == 0 and ptr != end:          # l.14
            val = int(words[ptr])               # l.15
            ptr += 1                            # l.16
            base += 32                          # l.17

    advance()                                   # INIT l.9
    seq = []
    while val != 0:                             # INDEX != sentinel, l.29
        bit = (val & -val).bit_length() - 1     # CTZ, l.32
        seq.append(base + bit)                  # l.33
        val &= val - 1                          # NEXT l.22
        if val == 0:
            advance()                           # l.24
    return seq


def _golden_rows():
    rows = []
    with open(os.path.join(GOLDEN, "crm_bit_order.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            nkb, blocks, words = [x.strip() for x in line.split("|")]
            blocks = [] if blocks == "-" else [int(x) for x in blocks.split()]
            rows.append((int(nkb), blocks, [int(w, 16) for w in words.split()]))
    return rows


@pytest.mark.parametrize("nkb,blocks,words", _golden_rows())
def test_golden_bit_order(nkb, blocks, words):
    assert len(words) == (nkb + 31) // 32
    # the hand-written words decode, by the paper's iterator, to the listed blocks
    assert alg2_iterate(words) == blocks
    # the oracle's pack and unpack (plain shifts) agree with both
    dense = np.zeros((1, 1, nkb), dtype=bool)
    dense[0, 0, blocks] = True
    bits = oracle.pack_bool(dense)
    assert bits.shape == (1, 1, len(words))
    assert bits[0, 0].tolist() == words
    assert (oracle.unpack_mask(np.asarray(words, dtype=np.uint32).reshape(1, 1, -1), nkb)[0, 0]
            == dense[0, 0]).all()


def test_paper_sizes():
    vals = {}
    with open(os.path.join(GOLDEN, "paper_sizes.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                name, val, _ = [x.strip() for x in line.split("|")]
                vals[name.split(" ")[0]] = int(val)
    assert 21 * 1560 == vals["tokens_wan1.3b_480p"] == inputs.C2.n_valid == inputs.C3.n_valid
    assert 21 * 3600 == vals["tokens_wan14b_720p"] == inputs.C4.n_valid
    for cfg in (inputs.C2, inputs.C3, inputs.C4):
        T, Hl, Wl = cfg.grid
        assert T * Hl * Wl == cfg.n_valid and cfg.Bq == cfg.Bk == vals["block_size"]
        assert cfg.N % 128 == 0 and 0 <= cfg.N - cfg.n_valid < 128
    assert oracle.words_per_row(262144, 128) == vals["words_per_row"] == 64
    assert oracle.words_per_row(inputs.C4.N, 128) == 19 and inputs.C4.NKB == 591
    assert oracle.words_per_row(inputs.C2.N, 128) == 8
    assert oracle.words_per_row(1024, 64) == 1


@pytest.mark.parametrize("nkb", [1, 31, 32, 33, 64, 591])
def test_pack_unpack_round_trip_and_iterator(nkb):
    rng = np.random.Generator(np.random.PCG64(nkb))
    dense = rng.random((3, 5, nkb)) < 0.4
    dense[0, 0] = False
    dense[0, 1] = True
    dense[1, 2] = False
    dense[1, 2, nkb - 1] = True
    bits = oracle.pack_bool(dense)
    assert (oracle.unpack_mask(bits, nkb) == dense).all()
    # stray-bit freedom: nothing at positions >= NKB
    if nkb % 32:
        assert (bits[:, :, -1] >> (nkb % 32) == 0).all()
    # density = popcount / total
    pop = sum(bin(int(w)).count("1") for w in bits.reshape(-1))
    assert pop == int(dense.sum())
    for h in range(3):
        for u in range(5):
            assert alg2_iterate(bits[h, u]) == np.nonzero(dense[h, u])[0].tolist()


def _topk_ref(scores, density, force_diag):
    """Library routine: torch.sort(stable=True, descending=True) top-k_h per head."""
    H, NQB, NKB = scores.shape
    out = np.zeros((H, NQB, NKB), dtype=bool)
    for h in range(H):
        key = torch.from_numpy(scores[h].astype(np.float64)).reshape(-1).clone()
        if force_diag:
            for u in range(min(NQB, NKB)):
                key[u * NKB + u] = float("inf")
        order = torch.sort(key, stable=True, descending=True).indices.numpy()
        kh = int(np.floor(float(np.float64(density[h])) * NQB * NKB + 0.5))
        kh = max(1, min(NQB * NKB, kh))
        if force_diag:
            kh = max(kh, min(NQB, NKB))
        flat = out[h].reshape(-1)
        flat[order[:kh]] = True
    return out


@pytest.mark.parametrize("NQB,NKB,force_diag", [(16, 16, 1), (16, 16, 0), (40, 40, 1), (7, 45, 0)])
def test_pack_mask_equals_stable_sort_topk(NQB, NKB, force_diag):
    rng = np.random.Generator(np.random.PCG64(NQB * 100 + NKB))
    H = 4
    scores = rng.random((H, NQB, NKB)).astype(np.float32)
    scores[1] = np.round(scores[1] * 4) / 4          # heavy ties -> index tie-break matters
    scores[2] = -scores[2]                           # negative scores
    scores[3, :, ::2] = 0.0
    scores[3, :, 1::4] = -0.0                        # signed zeros compare equal
    density = np.asarray([0.5, 0.3, 0.11, 0.6], dtype=np.float32)
    bits = oracle.pack_mask(scores, density, force_diag)
    got = oracle.unpack_mask(bits, NKB).astype(bool)
    ref = _topk_ref(scores, density, force_diag)
    assert (got == ref).all()
    for h in range(H):
        kh = oracle.keep_count(density[h], NQB, NKB, force_diag)
        assert got[h].sum() == kh                                  # exactly k_h bits
        if force_diag:
            assert got[h][np.arange(min(NQB, NKB)), np.arange(min(NQB, NKB))].all()
        # order statistic: min kept >= max dropped under (score desc, index asc)
        key = scores[h].astype(np.float64).copy()
        if force_diag:
            key[np.arange(min(NQB, NKB)), np.arange(min(NQB, NKB))] = np.inf
        if got[h].any() and (~got[h]).any():
            kmin, dmax = key[got[h]].min(), key[~got[h]].max()
            assert kmin >= dmax
            if kmin == dmax:   # ties at the cut: kept indices all below dropped ones
                flat_k = np.nonzero((got[h] & (key == kmin)).reshape(-1))[0]
                flat_d = np.nonzero((~got[h] & (key == kmin)).reshape(-1))[0]
                assert flat_k.max() < flat_d.min()
    if NKB % 32:
        assert (bits[:, :, -1] >> (NKB % 32) == 0).all()


def test_keep_count_rounding():
    # DESIGN.md P2: round half up in fp64 from the fp32 density, clamp to [1,total]; P3: >= NQB
    assert oracle.keep_count(0.5, 16, 16, 0) == 128
    assert oracle.keep_count(1.0, 591, 591, 1) == 591 * 591
    assert oracle.keep_count(1e-9, 16, 16, 0) == 1
    assert oracle.keep_count(1e-9, 16, 16, 1) == 16
    assert oracle.keep_count(0.25, 3, 2, 0) == 2          # 1.5 -> 2 (half up)
    assert oracle.keep_count(0.41666666, 3, 2, 0) == 2    # 2.4999 -> 2
    d = np.float32(0.1)
    assert oracle.keep_count(d, 591, 591, 0) == int(np.floor(float(d) * 591 * 591 + 0.5))


def test_density_one_sets_every_bit():
    scores = np.random.Generator(np.random.PCG64(5)).random((2, 33, 33)).astype(np.float32)
    bits = oracle.pack_mask(scores, np.ones(2, dtype=np.float32), 1)
    assert oracle.unpack_mask(bits, 33).all()
    assert (bits[:, :, 0] == 0xFFFFFFFF).all() and (bits[:, :, 1] == 1).all()


def test_bool_mask_as_scores_reproduces_mask():
    # the input helper that lets sa_pack_mask realise an explicit boolean mask
    m = inputs.iid_block_mask(2, 16, 16, 0.5, seed=0)
    assert m[:, np.arange(16), np.arange(16)].all()
    scores, density = inputs.bool_mask_as_scores(m)
    bits = oracle.pack_mask(scores, density, 1)
    assert (oracle.unpack_mask(bits, 16).astype(bool) == m).all()
    adv = inputs.adversarial_block_mask(2, 591, 0.1, seed=105)
    assert abs(adv.mean() - 0.1015) < 2e-3
    scores, density = inputs.bool_mask_as_scores(adv)
    bits = oracle.pack_mask(scores, density, 1)
    assert (oracle.unpack_mask(bits, 591).astype(bool) == adv).all()


def test_pack_rejects_non_finite():
    scores = np.zeros((1, 4, 4), dtype=np.float32)
    scores[0, 1, 1] = np.nan
    with pytest.raises(ValueError):
        oracle.pack_mask(scores, np.asarray([0.5], dtype=np.float32), 0)


def test_structured_scores_recipe():
    # The synthetic recipe gives local + sink structure and per-head densities in range.
    cfg = inputs.scaled(inputs.C2, H=3)
    scores, density, sigma = inputs.make_block_scores(cfg)
    assert scores.shape == (3, 256, 256) and scores.dtype == np.float32
    assert ((density >= 0.1) & (density <= 0.4)).all() and ((sigma >= 1) & (sigma <= 16)).all()
    bits = oracle.pack_mask(scores, density, 1)
    dense = oracle.unpack_mask(bits, 256).astype(bool)
    for h in range(3):
        assert dense[h].sum() == oracle.keep_count(density[h], 256, 256, 1)
        assert dense[h][np.arange(256), np.arange(256)].all()
        assert (dense[h].sum(axis=0) == 256).sum() >= 2       # the two sink columns are full
    s2, d2, _ = inputs.make_block_scores(cfg)
    assert (s2 == scores).all() and (d2 == density).all()       # seeded
