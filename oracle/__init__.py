"""CPU oracle for the ScalingAttention hot path -- TEST INFRASTRUCTURE ONLY.

Thin ctypes/numpy wrapper over oracle/sa_oracle.cpp (fp64, plain definition; see that file's
header for what it states and which PAPER.md passages it follows). Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package. It imports nothing from paper_2606_23019_b200 and the product never imports it.

All arrays are numpy, C-contiguous:
  q, k, v   : uint16 [B][H][N][D]  (bf16 bit patterns)
  mask_bits : uint32 [H][NQB][W],  W = ceil((N/Bk)/32), bit v%32 of word v/32 <-> key block v
  scores    : float32 [H][NQB][NKB];  density: float32 [H]
"""
import ctypes as C

import numpy as np

from .build import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.oracle_keep_count.restype = C.c_longlong
        _lib.oracle_keep_count.argtypes = [C.c_float, C.c_int, C.c_int, C.c_int]
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _chk(a, dtype, ndim=None):
    a = np.ascontiguousarray(a)
    assert a.dtype == dtype, (a.dtype, dtype)
    if ndim is not None:
        assert a.ndim == ndim, (a.ndim, ndim)
    return a


def hardware_threads() -> int:
    return int(lib().oracle_hardware_threads())


def words_per_row(N: int, Bk: int) -> int:
    return int(lib().oracle_words_per_row(C.c_int(N), C.c_int(Bk)))


def unpack_mask(mask_bits, NKB: int):
    bits = _chk(mask_bits, np.uint32, 3)
    H, NQB, W = bits.shape
    assert W == (NKB + 31) // 32
    dense = np.zeros((H, NQB, NKB), dtype=np.uint8)
    lib().oracle_unpack_mask(_p(bits), _p(dense), C.c_int(H), C.c_int(NQB), C.c_int(NKB))
    return dense


def pack_bool(dense):
    dense = _chk(np.asarray(dense).astype(np.uint8), np.uint8, 3)
    H, NQB, NKB = dense.shape
    bits = np.zeros((H, NQB, (NKB + 31) // 32), dtype=np.uint32)
    lib().oracle_pack_bool(_p(dense), _p(bits), C.c_int(H), C.c_int(NQB), C.c_int(NKB))
    return bits


def keep_count(density: float, NQB: int, NKB: int, force_diag: bool) -> int:
    return int(lib().oracle_keep_count(C.c_float(float(density)), C.c_int(NQB), C.c_int(NKB),
                                       C.c_int(int(bool(force_diag)))))


def pack_mask(scores, density, force_diag: bool):
    scores = _chk(scores, np.float32, 3)
    H, NQB, NKB = scores.shape
    density = _chk(density, np.float32, 1)
    assert density.shape[0] == H
    bits = np.zeros((H, NQB, (NKB + 31) // 32), dtype=np.uint32)
    rc = lib().oracle_pack_mask(_p(scores), _p(density), _p(bits), C.c_int(H), C.c_int(NQB),
                                C.c_int(NKB), C.c_int(int(bool(force_diag))))
    if rc != 0:
        raise ValueError("oracle_pack_mask: scores must be finite")
    return bits


def _attn_args(q, k, v, mask_bits, Bq, Bk):
    q = _chk(q, np.uint16, 4)
    k = _chk(k, np.uint16, 4)
    v = _chk(v, np.uint16, 4)
    assert q.shape == k.shape == v.shape
    B, H, N, D = q.shape
    assert N % Bq == 0 and N % Bk == 0
    bits = _chk(mask_bits, np.uint32, 3)
    assert bits.shape == (H, N // Bq, (N // Bk + 31) // 32), bits.shape
    return q, k, v, bits, B, H, N, D


def attn(q, k, v, mask_bits, Bq, Bk, scale, n_valid=None, n_threads=0):
    """Full oracle. Returns (out float64 [B][H][N][D], lse float64 [B][H][N])."""
    q, k, v, bits, B, H, N, D = _attn_args(q, k, v, mask_bits, Bq, Bk)
    n_valid = N if n_valid is None else int(n_valid)
    out = np.zeros((B, H, N, D), dtype=np.float64)
    lse = np.zeros((B, H, N), dtype=np.float64)
    lib().oracle_attn(_p(q), _p(k), _p(v), _p(bits), _p(out), _p(lse), C.c_int(B), C.c_int(H),
                      C.c_int(N), C.c_int(D), C.c_int(Bq), C.c_int(Bk), C.c_int(n_valid),
                      C.c_float(float(scale)), C.c_int(n_threads))
    return out, lse


def attn_units(q, k, v, mask_bits, units, Bq, Bk, scale, n_valid=None, n_threads=0):
    """Oracle on a list of units (b, h, u). Returns (out [n][Bq][D], lse [n][Bq]) in fp64."""
    q, k, v, bits, B, H, N, D = _attn_args(q, k, v, mask_bits, Bq, Bk)
    n_valid = N if n_valid is None else int(n_valid)
    units = _chk(np.asarray(units, dtype=np.int32).reshape(-1, 3), np.int32, 2)
    n = units.shape[0]
    for b, h, u in units:
        assert 0 <= b < B and 0 <= h < H and 0 <= u < N // Bq
    out = np.zeros((n, Bq, D), dtype=np.float64)
    lse = np.zeros((n, Bq), dtype=np.float64)
    lib().oracle_attn_units(_p(q), _p(k), _p(v), _p(bits), _p(units), C.c_int(n), _p(out),
                            _p(lse), C.c_int(B), C.c_int(H), C.c_int(N), C.c_int(D),
                            C.c_int(Bq), C.c_int(Bk), C.c_int(n_valid), C.c_float(float(scale)),
                            C.c_int(n_threads))
    return out, lse


def attn_row_weights(q, k, v, mask_bits, Bq, Bk, scale, b, h, i, n_valid=None):
    """Softmax weights (length N), output row and lse of one query token."""
    q, k, v, bits, B, H, N, D = _attn_args(q, k, v, mask_bits, Bq, Bk)
    n_valid = N if n_valid is None else int(n_valid)
    w = np.zeros(N, dtype=np.float64)
    o = np.zeros(D, dtype=np.float64)
    lse = np.zeros(1, dtype=np.float64)
    lib().oracle_attn_row_weights(_p(q), _p(k), _p(v), _p(bits), C.c_int(H), C.c_int(N),
                                  C.c_int(D), C.c_int(Bq), C.c_int(Bk), C.c_int(n_valid),
                                  C.c_float(float(scale)), C.c_int(b), C.c_int(h), C.c_int(i),
                                  _p(w), _p(o), _p(lse))
    return w, o, float(lse[0])
