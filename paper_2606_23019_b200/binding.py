"""Thin ctypes binding over libscalingattn.so (include/scalingattn.h), same names as the C ABI.

Argument marshalling only: every step of the hot path runs in the CUDA kernels of the library.
torch is used for device memory and streams. There is no CPU fallback: if the library cannot be
loaded, or a call returns a non-OK status, SAError is raised.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libscalingattn.so")
_lib = None

SA_OK = 0


class SAError(RuntimeError):
    def __init__(self, status: int, name: str, detail: str):
        super().__init__(f"{name} ({status}): {detail}")
        self.status = status
        self.name = name
        self.detail = detail


def library_path() -> str:
    return _LIB_PATH


def load_library() -> C.CDLL:
    """dlopen the in-tree library; fails loudly if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise SAError(-1, "SA_ERR_NOT_BUILT",
                      f"{_LIB_PATH} missing: run `python -m paper_2606_23019_b200.build` "
                      "(there is no CPU fallback)")
    lib = C.CDLL(_LIB_PATH)
    vp, ip, fp, sz = C.c_void_p, C.c_int, C.c_float, C.c_size_t
    lib.sa_mask_words_per_row.restype = ip
    lib.sa_mask_words_per_row.argtypes = [ip, ip]
    lib.sa_pack_mask_workspace_bytes.restype = sz
    lib.sa_pack_mask_workspace_bytes.argtypes = [ip, ip, ip]
    lib.sa_fwd_workspace_bytes.restype = sz
    lib.sa_fwd_workspace_bytes.argtypes = [ip, ip, ip, ip]
    lib.sa_fwd_host_scratch_bytes.restype = sz
    lib.sa_fwd_host_scratch_bytes.argtypes = [ip] * 6
    lib.sa_pack_mask.restype = ip
    lib.sa_pack_mask.argtypes = [vp, vp, vp, ip, ip, ip, ip, vp, sz, vp]
    lib.sa_pack_mask_static.restype = ip
    lib.sa_pack_mask_static.argtypes = [vp, vp, vp, ip, ip, ip, ip, vp]
    lib.sa_mask_from_threshold.restype = ip
    lib.sa_mask_from_threshold.argtypes = [vp, vp, vp, ip, ip, ip, ip, ip, ip, vp]
    lib.sa_block_significance.restype = ip
    lib.sa_block_significance.argtypes = [vp, vp, vp, vp, ip, ip, ip, ip, ip, ip, ip, fp, vp]
    lib.sa_threshold_map_update_workspace_bytes.restype = sz
    lib.sa_threshold_map_update_workspace_bytes.argtypes = [ip, ip, ip, ip]
    lib.sa_threshold_map_update.restype = ip
    lib.sa_threshold_map_update.argtypes = [vp, vp, ip, vp, ip, ip, ip, ip, vp, sz, vp]
    lib.sa_fidelity_from_lse.restype = ip
    lib.sa_fidelity_from_lse.argtypes = [vp, vp, vp, ip, ip, ip, ip, vp, vp, vp]
    lib.sa_block_sparse_attn_fwd.restype = ip
    lib.sa_block_sparse_attn_fwd.argtypes = [vp, vp, vp, vp, vp, vp, ip, ip, ip, ip, ip, ip, fp, vp]
    lib.sa_block_sparse_attn_fwd_ex.restype = ip
    lib.sa_block_sparse_attn_fwd_ex.argtypes = [vp, vp, vp, vp, vp, vp, ip, ip, ip, ip, ip, ip, ip,
                                                fp, vp, sz, vp]
    lib.sa_block_sparse_attn_fwd_reuse.restype = ip
    lib.sa_block_sparse_attn_fwd_reuse.argtypes = lib.sa_block_sparse_attn_fwd_ex.argtypes
    lib.sa_fwd_softmax_path_counts.restype = ip
    lib.sa_fwd_softmax_path_counts.argtypes = [vp, vp, vp, vp]
    lib.sa_debug_tail_plan.restype = ip
    lib.sa_debug_tail_plan.argtypes = [ip, ip, ip, ip, ip, ip, vp, vp]
    lib.sa_debug_l2_fill_rate.restype = ip
    lib.sa_debug_l2_fill_rate.argtypes = [vp, sz, ip, vp, vp, vp]
    lib.sa_debug_ex2_rate.restype = ip
    lib.sa_debug_ex2_rate.argtypes = [ip, vp, vp, vp, vp]
    lib.sa_debug_fwd_walk_log_bytes.restype = sz
    lib.sa_debug_fwd_walk_log_bytes.argtypes = [ip] * 5
    lib.sa_debug_fwd_walk.restype = ip
    lib.sa_debug_fwd_walk.argtypes = [vp, vp, vp, vp, vp, vp, ip, ip, ip, ip, ip, ip, ip, fp, vp, sz,
                                      vp, sz, vp]
    lib.sa_block_sparse_attn_fwd_host.restype = ip
    lib.sa_block_sparse_attn_fwd_host.argtypes = [vp, vp, vp, vp, vp, vp, ip, ip, ip, ip, ip, ip,
                                                  ip, fp, vp, sz, vp]
    lib.sa_hot_path_host_scratch_bytes.restype = sz
    lib.sa_hot_path_host_scratch_bytes.argtypes = [ip] * 6
    lib.sa_hot_path_host.restype = ip
    lib.sa_hot_path_host.argtypes = [vp, vp, ip, vp, vp, vp, vp, vp, vp, ip, ip, ip, ip, ip, ip,
                                     ip, fp, vp, sz, vp]
    lib.sa_profile_enable.restype = ip
    lib.sa_profile_enable.argtypes = [ip]
    lib.sa_profile_collect.restype = ip
    lib.sa_profile_collect.argtypes = [vp, ip, vp]
    lib.sa_enumerate_active_blocks.restype = ip
    lib.sa_enumerate_active_blocks.argtypes = [vp, ip, ip, ip, vp, vp, vp]
    lib.sa_set_fwd_variant.restype = ip
    lib.sa_set_fwd_variant.argtypes = [ip]
    lib.sa_get_fwd_variant.restype = ip
    lib.sa_last_launch_count.restype = ip
    lib.sa_status_string.restype = C.c_char_p
    lib.sa_status_string.argtypes = [ip]
    lib.sa_last_error.restype = C.c_char_p
    _lib = lib
    return lib


def _check(status: int) -> None:
    if status != SA_OK:
        lib = load_library()
        raise SAError(status, lib.sa_status_string(status).decode(), lib.sa_last_error().decode())


def _ptr(t) -> int:
    return 0 if t is None else t.data_ptr()


def _stream(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


def _scratch(nbytes: int, device, stream):
    """A temporary device buffer for one call. The caching allocator ties a block to the stream that
    was current when it was allocated; when the call runs on another stream the block is marked as
    in use there (record_stream), so that it is not handed out again while the kernels are pending."""
    t = torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=device)
    if stream is not None:
        s = stream if isinstance(stream, torch.cuda.Stream) else torch.cuda.ExternalStream(int(stream))
        t.record_stream(s)
    return t


def sa_status_string(status: int) -> str:
    return load_library().sa_status_string(status).decode()


def sa_last_error() -> str:
    return load_library().sa_last_error().decode()


def sa_mask_words_per_row(N: int, Bk: int) -> int:
    return load_library().sa_mask_words_per_row(N, Bk)


def sa_pack_mask_workspace_bytes(H: int, NQB: int, NKB: int) -> int:
    return load_library().sa_pack_mask_workspace_bytes(H, NQB, NKB)


def sa_fwd_workspace_bytes(B: int, H: int, N: int, Bq: int) -> int:
    return load_library().sa_fwd_workspace_bytes(B, H, N, Bq)


def sa_fwd_host_scratch_bytes(B: int, H: int, N: int, D: int, Bq: int, Bk: int) -> int:
    return load_library().sa_fwd_host_scratch_bytes(B, H, N, D, Bq, Bk)


def sa_set_fwd_variant(variant: int) -> None:
    _check(load_library().sa_set_fwd_variant(variant))


def sa_get_fwd_variant() -> int:
    return load_library().sa_get_fwd_variant()


def sa_last_launch_count() -> int:
    return load_library().sa_last_launch_count()


def sa_pack_mask(scores, density, force_diag: bool = True, mask_bits=None, workspace=None,
                 stream=None):
    """scores fp32 [H][NQB][NKB], density fp32 [H] (device) -> mask_bits int32 [H][NQB][W]
    (uint32 bit patterns; torch has no general uint32 support, so the storage dtype is int32)."""
    lib = load_library()
    assert scores.dtype == torch.float32 and scores.is_contiguous() and scores.dim() == 3
    assert density.dtype == torch.float32 and density.is_contiguous()
    H, NQB, NKB = scores.shape
    assert density.shape == (H,)
    W = (NKB + 31) // 32
    if mask_bits is None:
        mask_bits = torch.empty((H, NQB, W), dtype=torch.int32, device=scores.device)
    need = lib.sa_pack_mask_workspace_bytes(H, NQB, NKB)
    if workspace is None:
        workspace = _scratch(need, scores.device, stream)
    _check(lib.sa_pack_mask(_ptr(scores), _ptr(density), _ptr(mask_bits), H, NQB, NKB,
                            int(bool(force_diag)), _ptr(workspace), workspace.numel(),
                            _stream(stream)))
    return mask_bits


SA_STATIC_SCRATCH_BYTES = 2304 * 1024      # include/scalingattn.h


def sa_pack_mask_static(scores, density, mask_bits, force_diag: bool = True, stream=None):
    """sa_pack_mask with the library's fixed scratch array as its workspace: allocates nothing (the
    caller passes the output tensor). Raises SAError(SA_ERR_WORKSPACE) beyond SA_STATIC_SCRATCH_BYTES."""
    lib = load_library()
    assert scores.dtype == torch.float32 and scores.is_contiguous() and scores.dim() == 3
    assert density.dtype == torch.float32 and density.is_contiguous()
    H, NQB, NKB = scores.shape
    assert density.shape == (H,)
    assert mask_bits.dtype == torch.int32 and mask_bits.is_contiguous()
    assert tuple(mask_bits.shape) == (H, NQB, (NKB + 31) // 32)
    _check(lib.sa_pack_mask_static(_ptr(scores), _ptr(density), _ptr(mask_bits), H, NQB, NKB,
                                   int(bool(force_diag)), _stream(stream)))
    return mask_bits


def sa_mask_from_threshold(tmap, p_star, NQB: int, NKB: int, force_diag: bool = True,
                           mask_bits=None, stream=None):
    """tmap fp32 [H][nbq][nbk], p_star fp32 [H] (device) -> mask_bits int32 [H][NQB][W] (uint32 bit
    patterns): 1(T <= p*) at the base resolution, conservatively resized to NQB x NKB (Eq. 7)."""
    lib = load_library()
    assert tmap.dtype == torch.float32 and tmap.is_contiguous() and tmap.dim() == 3
    assert p_star.dtype == torch.float32 and p_star.is_contiguous()
    H, nbq, nbk = tmap.shape
    assert p_star.shape == (H,)
    W = (NKB + 31) // 32
    if mask_bits is None:
        mask_bits = torch.empty((H, NQB, W), dtype=torch.int32, device=tmap.device)
    _check(lib.sa_mask_from_threshold(_ptr(tmap), _ptr(p_star), _ptr(mask_bits), H, nbq, nbk,
                                      int(NQB), int(NKB), int(bool(force_diag)), _stream(stream)))
    return mask_bits


def sa_block_significance(q, k, lse, Bq: int, Bk: int, scale: float, n_valid=None, sig=None,
                          stream=None):
    """q, k bf16 [B][H][N][D], lse fp32 [B][H][N] (of a dense forward call) -> block significance
    fp32 [B][H][N/Bq][N/Bk] (Eq. 1)."""
    lib = load_library()
    assert q.dtype == k.dtype == torch.bfloat16 and q.is_contiguous() and k.is_contiguous()
    assert q.shape == k.shape and q.dim() == 4
    B, H, N, D = q.shape
    assert lse.dtype == torch.float32 and tuple(lse.shape) == (B, H, N) and lse.is_contiguous()
    n_valid = N if n_valid is None else int(n_valid)
    if sig is None:
        sig = torch.empty((B, H, N // Bq, N // Bk), dtype=torch.float32, device=q.device)
    _check(lib.sa_block_significance(_ptr(q), _ptr(k), _ptr(lse), _ptr(sig), B, H, N, n_valid, D, Bq,
                                     Bk, float(scale), _stream(stream)))
    return sig


def sa_threshold_map_update(sig, levels, tmap, workspace=None, stream=None):
    """sig fp32 [B][H][NQB][NKB], levels fp32 [n_levels] ascending in (0,1], tmap fp32 [H][NQB][NKB]
    (in/out, device): tmap <- min(tmap, local map of every sample) (Alg. 1 l.12-17)."""
    lib = load_library()
    assert sig.dtype == torch.float32 and sig.is_contiguous() and sig.dim() == 4
    assert levels.dtype == torch.float32 and levels.is_contiguous() and levels.dim() == 1
    B, H, NQB, NKB = sig.shape
    assert tmap.dtype == torch.float32 and tmap.is_contiguous() and tuple(tmap.shape) == (H, NQB, NKB)
    need = lib.sa_threshold_map_update_workspace_bytes(B, H, NQB, NKB)
    if workspace is None:
        workspace = _scratch(need, sig.device, stream)
    _check(lib.sa_threshold_map_update(_ptr(sig), _ptr(levels), levels.numel(), _ptr(tmap), B, H, NQB,
                                       NKB, _ptr(workspace), workspace.numel(), _stream(stream)))
    return tmap


def sa_fidelity_from_lse(lse_dense, lse_sparse, rows, per_row: bool = False, stream=None):
    """lse_dense, lse_sparse fp32 [B][H][N], rows int32 [n_rows] (device) -> fidelity fp32 [B][H]
    (and the per-row scores fp32 [B][H][n_rows] if per_row)."""
    lib = load_library()
    assert lse_dense.dtype == lse_sparse.dtype == torch.float32 and lse_dense.shape == lse_sparse.shape
    assert lse_dense.is_contiguous() and lse_sparse.is_contiguous() and lse_dense.dim() == 3
    assert rows.dtype == torch.int32 and rows.is_contiguous() and rows.dim() == 1
    B, H, N = lse_dense.shape
    fid = torch.empty((B, H), dtype=torch.float32, device=lse_dense.device)
    pr = (torch.empty((B, H, rows.numel()), dtype=torch.float32, device=lse_dense.device)
          if per_row else None)
    _check(lib.sa_fidelity_from_lse(_ptr(lse_dense), _ptr(lse_sparse), _ptr(rows), rows.numel(), B, H,
                                    N, _ptr(fid), _ptr(pr), _stream(stream)))
    return (fid, pr) if per_row else fid


def _fwd_shapes(q, k, v, mask_bits, Bq, Bk):
    assert q.dtype == k.dtype == v.dtype == torch.bfloat16
    assert q.is_contiguous() and k.is_contiguous() and v.is_contiguous()
    assert q.shape == k.shape == v.shape and q.dim() == 4
    B, H, N, D = q.shape
    assert mask_bits.dtype == torch.int32 and mask_bits.is_contiguous()
    if N % Bq == 0 and N % Bk == 0:
        assert tuple(mask_bits.shape) == (H, N // Bq, (N // Bk + 31) // 32), mask_bits.shape
    return B, H, N, D


def sa_block_sparse_attn_fwd(q, k, v, mask_bits, Bq: int, Bk: int, scale: float, out=None,
                             lse=None, stream=None):
    """The signature BASELINE.json names (internal workspace, all N tokens real)."""
    lib = load_library()
    B, H, N, D = _fwd_shapes(q, k, v, mask_bits, Bq, Bk)
    if out is None:
        out = torch.empty_like(q)
    if lse is None:
        lse = torch.empty((B, H, N), dtype=torch.float32, device=q.device)
    _check(lib.sa_block_sparse_attn_fwd(_ptr(q), _ptr(k), _ptr(v), _ptr(mask_bits), _ptr(out),
                                        _ptr(lse), B, H, N, D, Bq, Bk, float(scale),
                                        _stream(stream)))
    return out, lse


def sa_block_sparse_attn_fwd_ex(q, k, v, mask_bits, Bq: int, Bk: int, scale: float,
                                n_valid=None, out=None, lse=None, workspace=None, stream=None,
                                reuse_schedule: bool = False):
    """reuse_schedule=True calls sa_block_sparse_attn_fwd_reuse: `workspace` must hold the work list
    of an earlier call with the same mask and shape."""
    lib = load_library()
    B, H, N, D = _fwd_shapes(q, k, v, mask_bits, Bq, Bk)
    n_valid = N if n_valid is None else int(n_valid)
    if out is None:
        out = torch.empty_like(q)
    if lse is None:
        lse = torch.empty((B, H, N), dtype=torch.float32, device=q.device)
    if workspace is None:
        if reuse_schedule:
            raise ValueError("reuse_schedule=True needs the caller-owned workspace of the earlier call "
                             "(a fresh workspace holds no work list)")
        workspace = _scratch(lib.sa_fwd_workspace_bytes(B, H, N, Bq), q.device, stream)
    fn = lib.sa_block_sparse_attn_fwd_reuse if reuse_schedule else lib.sa_block_sparse_attn_fwd_ex
    _check(fn(_ptr(q), _ptr(k), _ptr(v), _ptr(mask_bits), _ptr(out),
                                           _ptr(lse), B, H, N, n_valid, D, Bq, Bk, float(scale),
                                           _ptr(workspace), workspace.numel(), _stream(stream)))
    return out, lse


def sa_fwd_softmax_path_counts(workspace, stream=None):
    """(fixed, exact): (softmax warp, work item) counts of the last tcgen05 forward call on `workspace`
    by softmax path (fixed Cauchy-Schwarz reference point / exact running max)."""
    a, b = C.c_longlong(0), C.c_longlong(0)
    _check(load_library().sa_fwd_softmax_path_counts(_ptr(workspace), C.addressof(a), C.addressof(b),
                                                     _stream(stream)))
    return a.value, b.value


def sa_debug_tail_plan(B: int, H: int, N: int, Bq: int, Bk: int, n_sm: int):
    """(rem, parts): how many work items a forward call of this shape issues in how many parts each
    on a device with n_sm SMs (host arithmetic only)."""
    rem, parts = C.c_int(0), C.c_int(0)
    _check(load_library().sa_debug_tail_plan(B, H, N, Bq, Bk, n_sm, C.addressof(rem), C.addressof(parts)))
    return rem.value, parts.value


def sa_debug_l2_fill_rate(buf_mb: int = 40, seconds: float = 0.3, iters: int = 4096, device=None, stream=None):
    """Measured L2 -> shared-memory fill rate in GB/s (every SM streaming 32 KB tiles of a `buf_mb` MB
    buffer with bulk copies), sustained over about `seconds`. Returns (GB/s, launches)."""
    import time
    lib = load_library()
    device = torch.device("cuda", torch.cuda.current_device()) if device is None else device
    buf = torch.zeros(buf_mb << 20, dtype=torch.uint8, device=device)
    ms, nbytes = C.c_float(0.0), C.c_double(0.0)
    tot_ms = tot_b = 0.0
    n = 0
    t0 = time.time()
    while True:
        _check(lib.sa_debug_l2_fill_rate(_ptr(buf), buf.numel(), int(iters), C.addressof(ms), C.addressof(nbytes),
                                         _stream(stream)))
        n += 1
        if n > 1:                                  # the first launch fills L2
            tot_ms += ms.value
            tot_b += nbytes.value
        if time.time() - t0 > seconds and n >= 3:
            break
    return tot_b / (tot_ms * 1e-3) / 1e9, n


def sa_debug_ex2_rate(seconds: float = 0.5, iters: int = 4096, device=None, stream=None):
    """Measured MUFU.EX2 rate (exponentials per second) under sustained load: launches of the library's
    ex2-only kernel back to back for about `seconds`; the median rate of the second half is returned."""
    import time
    lib = load_library()
    sink = torch.zeros(8 * 1024, dtype=torch.float32, device=device or "cuda")
    ms, n = C.c_float(0), C.c_double(0)
    rates = []
    t0 = time.time()
    while time.time() - t0 < seconds or len(rates) < 4:
        _check(lib.sa_debug_ex2_rate(int(iters), _ptr(sink), C.addressof(ms), C.addressof(n), _stream(stream)))
        rates.append(n.value / (ms.value * 1e-3))
    tail = sorted(rates[len(rates) // 2:])
    return tail[len(tail) // 2]


def sa_debug_fwd_walk(q, k, v, mask_bits, Bq: int, Bk: int, scale: float, n_valid=None, stream=None):
    """Debug hook (include/scalingattn.h): the forward call on the walk-recording build of the tcgen05
    kernel. Returns out, lse and the log regions as int32 tensors
    (wg_cnt [R], wg_info [R], wg_seq [R][NKB], is_cnt [R], is_seq [R][2*NKB]), R = B*H*N/Bq."""
    lib = load_library()
    B, H, N, D = _fwd_shapes(q, k, v, mask_bits, Bq, Bk)
    n_valid = N if n_valid is None else int(n_valid)
    out = torch.empty_like(q)
    lse = torch.empty((B, H, N), dtype=torch.float32, device=q.device)
    workspace = _scratch(lib.sa_fwd_workspace_bytes(B, H, N, Bq), q.device, stream)
    log = torch.zeros(lib.sa_debug_fwd_walk_log_bytes(B, H, N, Bq, Bk) // 4, dtype=torch.int32,
                      device=q.device)
    if stream is not None:      # the zero fill ran on the current stream
        torch.cuda.current_stream().synchronize()
    _check(lib.sa_debug_fwd_walk(_ptr(q), _ptr(k), _ptr(v), _ptr(mask_bits), _ptr(out), _ptr(lse), B, H, N,
                                 n_valid, D, Bq, Bk, float(scale), _ptr(workspace), workspace.numel(),
                                 _ptr(log), log.numel() * 4, _stream(stream)))
    R, NKB = B * H * (N // Bq), N // Bk
    o = 0
    regions = []
    for n, shape in ((R, (R,)), (R, (R,)), (R * NKB, (R, NKB)), (R, (R,)), (2 * R * NKB, (R, 2 * NKB))):
        regions.append(log[o:o + n].view(shape))
        o += n
    return (out, lse) + tuple(regions)


def sa_block_sparse_attn_fwd_host(q, k, v, mask_bits, out, lse, Bq: int, Bk: int, scale: float,
                                  n_valid, scratch, stream=None):
    """End-to-end form: q, k, v, mask_bits, out, lse are HOST (pinned) tensors, scratch is device."""
    lib = load_library()
    B, H, N, D = _fwd_shapes(q, k, v, mask_bits, Bq, Bk)
    for t in (q, k, v, mask_bits, out, lse):
        assert t.device.type == "cpu"
    assert out.dtype == torch.bfloat16 and out.shape == q.shape and out.is_contiguous()
    assert lse.dtype == torch.float32 and tuple(lse.shape) == (B, H, N) and lse.is_contiguous()
    _check(lib.sa_block_sparse_attn_fwd_host(_ptr(q), _ptr(k), _ptr(v), _ptr(mask_bits), _ptr(out),
                                             _ptr(lse), B, H, N, int(n_valid), D, Bq, Bk,
                                             float(scale), _ptr(scratch), scratch.numel(),
                                             _stream(stream)))
    return out, lse


def sa_hot_path_host_scratch_bytes(B: int, H: int, N: int, D: int, Bq: int, Bk: int) -> int:
    return load_library().sa_hot_path_host_scratch_bytes(B, H, N, D, Bq, Bk)


def sa_hot_path_host(scores, density, q, k, v, mask_bits, out, lse, Bq: int, Bk: int,
                     scale: float, n_valid, scratch, force_diag: bool = True, stream=None):
    """Whole hot path with HOST (pinned) tensors: scores, density -> mask_bits (out, host);
    q, k, v -> out, lse (host). scratch is a device uint8 tensor."""
    lib = load_library()
    B, H, N, D = _fwd_shapes(q, k, v, mask_bits, Bq, Bk)
    for t in (scores, density, q, k, v, mask_bits, out, lse):
        assert t.device.type == "cpu" and t.is_contiguous()
    assert scores.dtype == torch.float32 and tuple(scores.shape) == (H, N // Bq, N // Bk)
    assert density.dtype == torch.float32 and tuple(density.shape) == (H,)
    assert out.dtype == torch.bfloat16 and out.shape == q.shape
    assert lse.dtype == torch.float32 and tuple(lse.shape) == (B, H, N)
    _check(lib.sa_hot_path_host(_ptr(scores), _ptr(density), int(bool(force_diag)), _ptr(q),
                                _ptr(k), _ptr(v), _ptr(mask_bits), _ptr(out), _ptr(lse), B, H, N,
                                int(n_valid), D, Bq, Bk, float(scale), _ptr(scratch),
                                scratch.numel(), _stream(stream)))
    return mask_bits, out, lse


def sa_profile_enable(capacity: int) -> None:
    _check(load_library().sa_profile_enable(int(capacity)))


def sa_profile_collect(capacity: int):
    """Elapsed milliseconds of the attention kernel of each forward call recorded since the last
    collect (synchronises on them)."""
    ms = (C.c_float * max(capacity, 1))()
    n = C.c_int(0)
    _check(load_library().sa_profile_collect(C.addressof(ms), capacity, C.addressof(n)))
    return [float(ms[i]) for i in range(n.value)]


def sa_enumerate_active_blocks(mask_bits, NKB: int, stream=None):
    lib = load_library()
    H, NQB, W = mask_bits.shape
    assert mask_bits.dtype == torch.int32 and mask_bits.is_contiguous()
    idx = torch.full((H, NQB, NKB), -1, dtype=torch.int32, device=mask_bits.device)
    cnt = torch.zeros((H, NQB), dtype=torch.int32, device=mask_bits.device)
    _check(lib.sa_enumerate_active_blocks(_ptr(mask_bits), H, NQB, NKB, _ptr(idx), _ptr(cnt),
                                          _stream(stream)))
    return idx, cnt
