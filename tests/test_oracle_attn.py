"""Pins for the attention oracle (oracle/sa_oracle.cpp) against things other than itself:
library routines (torch SDPA / logsumexp in fp64), special cases, closed forms, invariants and a
long-double brute force. CPU only. See DESIGN.md "What pins each part"."""
import math

import numpy as np
import pytest
import torch

import oracle
from paper_2606_23019_b200 import inputs


def _rand_qkv(B, H, N, D, seed, scale_q=1.0):
    g = torch.Generator().manual_seed(seed)
    q = (torch.randn((B, H, N, D), generator=g) * scale_q).to(torch.bfloat16)
    k = torch.randn((B, H, N, D), generator=g).to(torch.bfloat16)
    v = torch.randn((B, H, N, D), generator=g).to(torch.bfloat16)
    return q, k, v


def _rand_block_mask(H, NQB, NKB, p, seed, diag=True):
    rng = np.random.Generator(np.random.PCG64(seed))
    m = rng.random((H, NQB, NKB)) < p
    if diag:
        for u in range(min(NQB, NKB)):
            m[:, u, u] = True
    return m


def _token_mask(m, Bq, Bk, n_valid=None):
    """block mask [H][NQB][NKB] -> token-level boolean [H][N][N] by repeat_interleave."""
    t = torch.from_numpy(m).repeat_interleave(Bq, dim=1).repeat_interleave(Bk, dim=2)
    if n_valid is not None:
        t = t.clone()
        t[:, :, n_valid:] = False
    return t


def _sdpa_ref(q, k, v, tok_mask, scale):
    """Second, differently written routine: torch SDPA + logsumexp in fp64."""
    qd, kd, vd = q.double(), k.double(), v.double()
    am = None if tok_mask is None else tok_mask[None]
    out = torch.nn.functional.scaled_dot_product_attention(qd, kd, vd, attn_mask=am, scale=scale)
    s = torch.einsum("bhid,bhjd->bhij", qd, kd) * scale
    if am is not None:
        s = s.masked_fill(~am, float("-inf"))
    lse = torch.logsumexp(s, dim=-1)
    return out.numpy(), lse.numpy()


@pytest.mark.parametrize("D,Bq", [(64, 64), (128, 128), (16, 32)])
def test_dense_equals_sdpa(D, Bq):
    # Special case ("fully dense setting"): all bits set == ordinary attention.
    B, H, N = 2, 2, 256
    q, k, v = _rand_qkv(B, H, N, D, seed=11)
    scale = float(np.float32(1 / math.sqrt(D)))
    bits = oracle.pack_bool(np.ones((H, N // Bq, N // Bq), dtype=bool))
    out, lse = oracle.attn(inputs.as_u16(q), inputs.as_u16(k), inputs.as_u16(v), bits, Bq, Bq, scale)
    ref_o, ref_l = _sdpa_ref(q, k, v, None, scale)
    assert np.abs(out - ref_o).max() < 1e-12
    assert np.abs(lse - ref_l).max() < 1e-12


@pytest.mark.parametrize("seed,p", [(0, 0.5), (1, 0.15), (2, 0.9)])
def test_arbitrary_mask_equals_sdpa_with_token_mask(seed, p):
    B, H, N, D, Bq = 1, 3, 320, 32, 32
    q, k, v = _rand_qkv(B, H, N, D, seed=20 + seed)
    scale = 0.2
    m = _rand_block_mask(H, N // Bq, N // Bq, p, seed)
    bits = oracle.pack_bool(m)
    out, lse = oracle.attn(inputs.as_u16(q), inputs.as_u16(k), inputs.as_u16(v), bits, Bq, Bq, scale)
    ref_o, ref_l = _sdpa_ref(q, k, v, _token_mask(m, Bq, Bq), float(np.float32(scale)))
    assert np.abs(out - ref_o).max() < 1e-12
    assert np.abs(lse - ref_l).max() < 1e-12


def test_rectangular_blocks_and_padding_vs_sdpa():
    # Bq != Bk and n_valid < N: padded keys carry exactly zero weight even when they hold
    # enormous values (P8).
    B, H, N, D, Bq, Bk, n_valid = 1, 2, 256, 16, 64, 32, 250
    q, k, v = _rand_qkv(B, H, N, D, seed=31)
    k[:, :, n_valid:] = 64.0
    v[:, :, n_valid:] = 1000.0
    m = _rand_block_mask(H, N // Bq, N // Bk, 0.5, 5, diag=False)
    m[:, :, -1] = True  # every row sees the ragged last key block
    bits = oracle.pack_bool(m)
    out, lse = oracle.attn(inputs.as_u16(q), inputs.as_u16(k), inputs.as_u16(v), bits, Bq, Bk,
                           0.25, n_valid=n_valid)
    ref_o, ref_l = _sdpa_ref(q, k, v, _token_mask(m, Bq, Bk, n_valid), 0.25)
    assert np.abs(out - ref_o).max() < 1e-12
    assert np.abs(lse - ref_l).max() < 1e-12
    assert np.abs(out).max() < 10.0  # nothing leaked from v = 1000


def test_block_diagonal_equals_independent_blocks():
    # BASELINE.json: with a block-diagonal mask the result is NQB independent attentions.
    B, H, N, D, Bq = 1, 2, 256, 64, 64
    q, k, v = _rand_qkv(B, H, N, D, seed=41)
    scale = 0.125
    m = np.zeros((H, N // Bq, N // Bq), dtype=bool)
    for u in range(N // Bq):
        m[:, u, u] = True
    out, lse = oracle.attn(inputs.as_u16(q), inputs.as_u16(k), inputs.as_u16(v),
                           oracle.pack_bool(m), Bq, Bq, scale)
    for u in range(N // Bq):
        sl = slice(u * Bq, (u + 1) * Bq)
        o_u, l_u = _sdpa_ref(q[:, :, sl], k[:, :, sl], v[:, :, sl], None, scale)
        assert np.abs(out[:, :, sl] - o_u).max() < 1e-12
        assert np.abs(lse[:, :, sl] - l_u).max() < 1e-12


def test_weights_sum_to_one_and_reproduce_output():
    B, H, N, D, Bq = 1, 2, 256, 32, 32
    q, k, v = _rand_qkv(B, H, N, D, seed=51, scale_q=3.0)
    m = _rand_block_mask(H, N // Bq, N // Bq, 0.4, 7)
    bits = oracle.pack_bool(m)
    qa, ka, va = inputs.as_u16(q), inputs.as_u16(k), inputs.as_u16(v)
    out, lse = oracle.attn(qa, ka, va, bits, Bq, Bq, 0.3)
    vd = v.double().numpy()
    for h in range(H):
        for i in range(0, N, 7):
            w, o, l = oracle.attn_row_weights(qa, ka, va, bits, Bq, Bq, 0.3, 0, h, i)
            assert abs(w.sum() - 1.0) < 1e-12
            assert (w >= 0).all()
            # weights vanish exactly outside the active blocks
            tok = np.repeat(m[h, i // Bq], Bq)
            assert (w[~tok] == 0).all() and (w[tok] > 0).all()
            assert np.abs(w @ vd[0, h] - out[0, h, i]).max() < 1e-12
            assert l == lse[0, h, i]


def test_brute_force_long_double_tiny():
    # Two-pass double loop in long double, no max subtraction (scores are O(1)).
    B, H, N, D, Bq = 1, 2, 64, 8, 16
    q, k, v = _rand_qkv(B, H, N, D, seed=61)
    scale = float(np.float32(0.35))
    m = _rand_block_mask(H, N // Bq, N // Bq, 0.5, 9)
    out, lse = oracle.attn(inputs.as_u16(q), inputs.as_u16(k), inputs.as_u16(v),
                           oracle.pack_bool(m), Bq, Bq, scale)
    ql = q.float().numpy().astype(np.longdouble)
    kl = k.float().numpy().astype(np.longdouble)
    vl = v.float().numpy().astype(np.longdouble)
    for h in range(H):
        for i in range(N):
            Z = np.longdouble(0)
            acc = np.zeros(D, dtype=np.longdouble)
            for j in range(N):
                if not m[h, i // Bq, j // Bq]:
                    continue
                s = np.longdouble(0)
                for d in range(D):
                    s += ql[0, h, i, d] * kl[0, h, j, d]
                e = np.exp(np.longdouble(scale) * s)
                Z += e
                acc += e * vl[0, h, j]
            assert np.abs((acc / Z).astype(np.float64) - out[0, h, i]).max() < 1e-13
            assert abs(float(np.log(Z)) - lse[0, h, i]) < 1e-13


def test_closed_form_constant_v():
    # V == c per column  =>  out[i,:] = c for every non-empty row, whatever Q, K and the mask.
    B, H, N, D, Bq = 1, 2, 256, 16, 32
    q, k, v = _rand_qkv(B, H, N, D, seed=71)
    c = torch.linspace(-2, 2, D).to(torch.bfloat16)
    v[:] = c
    m = _rand_block_mask(H, N // Bq, N // Bq, 0.3, 3)
    out, _ = oracle.attn(inputs.as_u16(q), inputs.as_u16(k), inputs.as_u16(v),
                         oracle.pack_bool(m), Bq, Bq, 0.25)
    assert np.abs(out - c.double().numpy()).max() < 1e-13


def test_closed_form_zero_q():
    # Q == 0  =>  uniform weights: out = mean of the valid active V rows,
    # lse = ln(#valid active keys) -- depends only on the mask, so it checks the bit layout.
    B, H, N, D, Bq, n_valid = 1, 3, 40 * 16, 8, 16, 40 * 16 - 5     # NKB = 40: two mask words
    q, k, v = _rand_qkv(B, H, N, D, seed=81)
    q.zero_()
    m = _rand_block_mask(H, N // Bq, N // Bq, 0.3, 4)
    out, lse = oracle.attn(inputs.as_u16(q), inputs.as_u16(k), inputs.as_u16(v),
                           oracle.pack_bool(m), Bq, Bq, 0.5, n_valid=n_valid)
    vd = v.double().numpy()
    for h in range(H):
        for u in range(N // Bq):
            tok = np.repeat(m[h, u], Bq)
            tok[n_valid:] = False
            cnt = int(tok.sum())
            assert cnt == int(m[h, u].sum()) * Bq - (5 if m[h, u, -1] else 0)
            i = u * Bq + 3
            assert abs(lse[0, h, i] - math.log(cnt)) < 1e-13
            assert np.abs(out[0, h, i] - vd[0, h][tok].mean(axis=0)).max() < 1e-13


def test_key_block_permutation_invariance():
    # Permuting key blocks together with their mask bits leaves out and lse unchanged (up to
    # fp64 summation order).
    B, H, N, D, Bq = 1, 2, 256, 16, 32
    q, k, v = _rand_qkv(B, H, N, D, seed=91)
    nb = N // Bq
    m = _rand_block_mask(H, nb, nb, 0.4, 6, diag=False)
    perm = np.random.Generator(np.random.PCG64(1)).permutation(nb)
    tok_perm = (perm[:, None] * Bq + np.arange(Bq)[None, :]).reshape(-1)
    k2, v2, m2 = k[:, :, tok_perm], v[:, :, tok_perm], m[:, :, perm]
    a = oracle.attn(inputs.as_u16(q), inputs.as_u16(k), inputs.as_u16(v), oracle.pack_bool(m), Bq, Bq, 0.25)
    b = oracle.attn(inputs.as_u16(q), inputs.as_u16(k2), inputs.as_u16(v2), oracle.pack_bool(m2), Bq, Bq, 0.25)
    ne = np.isfinite(a[1])
    assert (np.isfinite(b[1]) == ne).all()
    assert np.abs(a[0] - b[0]).max() < 1e-12
    assert np.abs(a[1][ne] - b[1][ne]).max() < 1e-12


def test_empty_row_definition():
    # DESIGN.md P7 (Alg. 2 returns the end sentinel at once): out = 0, lse = -inf.
    B, H, N, D, Bq = 1, 1, 128, 8, 32
    q, k, v = _rand_qkv(B, H, N, D, seed=101)
    m = np.ones((1, 4, 4), dtype=bool)
    m[0, 2, :] = False
    out, lse = oracle.attn(inputs.as_u16(q), inputs.as_u16(k), inputs.as_u16(v),
                           oracle.pack_bool(m), Bq, Bq, 1.0)
    assert (out[0, 0, 64:96] == 0).all()
    assert np.isneginf(lse[0, 0, 64:96]).all()
    assert np.isfinite(lse[0, 0, :64]).all() and np.isfinite(lse[0, 0, 96:]).all()
    # a row whose only active block holds no valid key is empty too
    m2 = np.zeros((1, 4, 4), dtype=bool)
    m2[0, :, 3] = True
    out2, lse2 = oracle.attn(inputs.as_u16(q), inputs.as_u16(k), inputs.as_u16(v),
                             oracle.pack_bool(m2), Bq, Bq, 1.0, n_valid=96)
    assert (out2 == 0).all() and np.isneginf(lse2).all()


def test_units_variant_matches_full():
    B, H, N, D, Bq = 2, 2, 256, 16, 64
    q, k, v = _rand_qkv(B, H, N, D, seed=111)
    m = _rand_block_mask(H, N // Bq, N // Bq, 0.5, 8)
    bits = oracle.pack_bool(m)
    qa, ka, va = inputs.as_u16(q), inputs.as_u16(k), inputs.as_u16(v)
    out, lse = oracle.attn(qa, ka, va, bits, Bq, Bq, 0.25, n_valid=250)
    units = [(0, 0, 0), (1, 1, 3), (0, 1, 2), (1, 0, 1)]
    uo, ul = oracle.attn_units(qa, ka, va, bits, units, Bq, Bq, 0.25, n_valid=250)
    for t, (b, h, u) in enumerate(units):
        assert (uo[t] == out[b, h, u * Bq:(u + 1) * Bq]).all()
        assert (ul[t] == lse[b, h, u * Bq:(u + 1) * Bq]).all()


def test_mask_is_shared_across_batch_and_per_head():
    # DESIGN.md P10: bits are [H][NQB][W]; batch entries use the same mask, heads their own.
    B, H, N, D, Bq = 2, 2, 128, 8, 32
    q, k, v = _rand_qkv(B, H, N, D, seed=121)
    m = _rand_block_mask(H, 4, 4, 0.5, 10)
    assert (m[0] != m[1]).any()
    out, lse = oracle.attn(inputs.as_u16(q), inputs.as_u16(k), inputs.as_u16(v),
                           oracle.pack_bool(m), Bq, Bq, 0.3)
    ref_o, ref_l = _sdpa_ref(q, k, v, _token_mask(m, Bq, Bq), float(np.float32(0.3)))
    assert np.abs(out - ref_o).max() < 1e-12 and np.abs(lse - ref_l).max() < 1e-12
