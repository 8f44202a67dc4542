"""C-ABI library: loads, exports every symbol include/scalingattn.h declares, host helpers and
argument validation (no kernel is launched: validation fails before any CUDA call). CPU only."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_23019_b200 import build
    build.build()
    from paper_2606_23019_b200 import binding
    return binding.load_library()


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "scalingattn.h")).read()
    return re.findall(r"SA_API\s+[\w\s\*]+?\b(sa_\w+)\s*\(", src)


def test_header_symbols_exported(lib):
    names = _declared_symbols()
    assert len(names) >= 14 and "sa_pack_mask" in names and "sa_block_sparse_attn_fwd" in names
    for n in names:
        assert hasattr(lib, n), n


def test_no_torch_or_python_types_in_abi():
    src = open(os.path.join(ROOT, "include", "scalingattn.h")).read()
    assert "torch" not in src.lower() and "PyObject" not in src and "at::" not in src
    assert 'extern "C"' in src


def test_host_helpers(lib):
    assert lib.sa_mask_words_per_row(262144, 128) == 64
    assert lib.sa_mask_words_per_row(75648, 128) == 19
    assert lib.sa_mask_words_per_row(1024, 64) == 1
    assert lib.sa_mask_words_per_row(1000, 64) == -1
    assert lib.sa_mask_words_per_row(0, 64) == -1
    assert lib.sa_fwd_workspace_bytes(1, 40, 75648, 128) >= 4 * (16 + 2 * 40 + 2 * 40 * 591)
    assert lib.sa_fwd_workspace_bytes(1, 40, 75648, 100) == 0
    assert lib.sa_pack_mask_workspace_bytes(40, 591, 591) > 40 * 4 * 256 * 4
    assert lib.sa_pack_mask_workspace_bytes(0, 591, 591) == 0
    t = 40 * 75648 * 128 * 2
    assert lib.sa_fwd_host_scratch_bytes(1, 40, 75648, 128, 128, 128) >= 4 * t + 40 * 75648 * 4
    assert lib.sa_status_string(0) == b"SA_OK"
    assert lib.sa_status_string(2) == b"SA_ERR_UNSUPPORTED"


def test_tail_plan_host_logic():
    # DESIGN.md K2: P pair items on n SMs; rem = P mod n items run in `parts` parts when that makes the
    # last round ceil(rem * parts / n) / parts of a pair long, saves >= 3% of the launch, and a dense row
    # has 32 key blocks per part. Worked by hand:
    from paper_2606_23019_b200 import binding as sa
    plan = lambda H, N, n=148, B=1: sa.sa_debug_tail_plan(B, H, N, 128, 128, n)
    assert plan(12, 16384) == (28, 4)        # 768 pairs = 5 x 148 + 28; 112 quarter items fill 3/4 of a round
    assert plan(12, 32768) == (56, 2)        # 1536 = 10 x 148 + 56; halves and quarters both give 1/2: fewer parts
    assert plan(12, 8192) == (0, 0)          # 384 = 2 x 148 + 88, 64 key blocks: halves only, 176 halves = a whole round
    assert plan(12, 65536) == (0, 0)         # 3072 = 20 x 148 + 112: no split shortens the round
    assert plan(40, 75648) == (0, 0)         # C4: 11840 pairs = 80 rounds exactly
    assert plan(24, 44672) == (0, 0)         # HunyuanVideo shape: 4200 = 28 x 148 + 56: half a round of 29 is < 3%
    assert plan(12, 4096) == (0, 0)          # below two waves of pairs: split items instead (api.cu)
    assert plan(8, 9600) == (8, 2)           # 304 pairs; 75 key blocks allow two parts
    assert plan(5, 16384) == (24, 4)
    # 29 rounds + 1 item: one quarter of a round saved is < 3% of 30 rounds
    assert plan(1, 128 * 2 * (148 * 29 + 1)) == (0, 0)
    with pytest.raises(sa.SAError):
        sa.sa_debug_tail_plan(1, 12, 1000, 128, 128, 148)


def _fwd_ex(lib, q=16, k=16, v=16, m=16, o=16, l=16, B=1, H=2, N=1024, nv=1024, D=64, Bq=64,
            Bk=64, scale=0.125, ws=16, wsb=1 << 20):
    return lib.sa_block_sparse_attn_fwd_ex(q, k, v, m, o, l, B, H, N, nv, D, Bq, Bk, scale, ws,
                                           wsb, None)


def test_fwd_validation_errors_before_any_cuda_call(lib):
    INVALID, UNSUPPORTED, WORKSPACE = 1, 2, 4
    assert _fwd_ex(lib, q=None) == INVALID
    assert b"null" in lib.sa_last_error()
    assert _fwd_ex(lib, N=1000) == INVALID
    assert _fwd_ex(lib, N=0) == INVALID
    assert _fwd_ex(lib, nv=0) == INVALID
    assert _fwd_ex(lib, nv=1025) == INVALID
    assert _fwd_ex(lib, scale=0.0) == INVALID
    assert _fwd_ex(lib, scale=float("nan")) == INVALID
    assert _fwd_ex(lib, q=24) == INVALID                    # misaligned
    assert _fwd_ex(lib, D=128) == UNSUPPORTED               # (128,64,64)
    assert _fwd_ex(lib, D=32, Bq=32, Bk=32) == UNSUPPORTED
    assert _fwd_ex(lib, Bq=128, D=128) == UNSUPPORTED       # Bq != Bk
    assert b"unsupported" in lib.sa_last_error()
    assert _fwd_ex(lib, ws=None) == WORKSPACE
    assert _fwd_ex(lib, wsb=8) == WORKSPACE


def test_pack_and_misc_validation(lib):
    INVALID, WORKSPACE = 1, 4
    assert lib.sa_pack_mask(None, 16, 16, 2, 16, 16, 1, 16, 1 << 20, None) == INVALID
    assert lib.sa_pack_mask(16, 16, 16, 0, 16, 16, 1, 16, 1 << 20, None) == INVALID
    assert lib.sa_pack_mask(16, 16, 16, 2, 16, 16, 1, 16, 8, None) == WORKSPACE
    assert lib.sa_pack_mask(16, 16, 16, 2, 16, 16, 1, None, 1 << 20, None) == WORKSPACE
    assert lib.sa_enumerate_active_blocks(None, 1, 1, 1, 16, 16, None) == INVALID
    assert lib.sa_set_fwd_variant(7) == INVALID and lib.sa_set_fwd_variant(-1) == INVALID
    assert lib.sa_set_fwd_variant(3) == 0 and lib.sa_set_fwd_variant(2) == 0
    assert lib.sa_set_fwd_variant(1) == 0 and lib.sa_get_fwd_variant() == 1
    assert lib.sa_set_fwd_variant(0) == 0 and lib.sa_get_fwd_variant() == 0
    host = lib.sa_block_sparse_attn_fwd_host
    assert host(16, 16, 16, 16, 16, 16, 1, 2, 1024, 1024, 64, 64, 64, 0.125, None, 0, None) == WORKSPACE
    assert host(None, 16, 16, 16, 16, 16, 1, 2, 1024, 1024, 64, 64, 64, 0.125, 256, 1 << 30, None) == INVALID


def test_offline_entry_points_validation(lib):
    INVALID, UNSUPPORTED, WORKSPACE = 1, 2, 4
    mft = lib.sa_mask_from_threshold
    assert mft(None, 16, 16, 2, 4, 4, 8, 8, 1, None) == INVALID
    assert mft(16, 16, 16, 2, 0, 4, 8, 8, 1, None) == INVALID
    assert mft(24, 16, 16, 2, 4, 4, 8, 8, 1, None) == INVALID            # misaligned map
    assert mft(16, 16, 16, 2, 4, 4, 40000, 8, 1, None) == UNSUPPORTED    # grid side > 32768
    sig = lib.sa_block_significance
    assert sig(None, 16, 16, 16, 1, 2, 1024, 1024, 128, 128, 128, 0.1, None) == INVALID
    assert sig(16, 16, 16, 16, 1, 2, 1000, 1000, 128, 128, 128, 0.1, None) == INVALID
    assert sig(16, 16, 16, 16, 1, 2, 1024, 1024, 64, 64, 64, 0.1, None) == UNSUPPORTED
    upd = lib.sa_threshold_map_update
    assert lib.sa_threshold_map_update_workspace_bytes(2, 3, 40, 40) > 2 * 2 * 3 * 1600 * 8
    assert lib.sa_threshold_map_update_workspace_bytes(0, 3, 40, 40) == 0
    assert upd(None, 16, 4, 16, 1, 2, 8, 8, 256, 1 << 30, None) == INVALID
    assert upd(16, 16, 0, 16, 1, 2, 8, 8, 256, 1 << 30, None) == INVALID
    assert upd(16, 16, 300, 16, 1, 2, 8, 8, 256, 1 << 30, None) == UNSUPPORTED
    assert upd(16, 16, 4, 16, 1, 2, 8, 8, 256, 8, None) == WORKSPACE
    assert upd(16, 16, 4, 16, 1, 2, 8, 8, 8, 1 << 30, None) == WORKSPACE   # not 256 B aligned
    fid = lib.sa_fidelity_from_lse
    assert fid(None, 16, 16, 4, 1, 2, 1024, 16, None, None) == INVALID
    assert fid(16, 16, 16, 0, 1, 2, 1024, 16, None, None) == INVALID


def test_binding_refuses_schedule_reuse_without_workspace(lib):
    # a fresh workspace holds no work list: the binding must not hand one to the _reuse entry point
    import torch
    from paper_2606_23019_b200 import binding
    q = torch.zeros((1, 1, 128, 128), dtype=torch.bfloat16)
    bits = torch.zeros((1, 1, 1), dtype=torch.int32)
    with pytest.raises(ValueError):
        binding.sa_block_sparse_attn_fwd_ex(q, q, q, bits, 128, 128, 0.1, reuse_schedule=True)


def test_debug_and_stats_entry_points_validation(lib):
    lib.sa_debug_fwd_walk_log_bytes.restype = C.c_size_t
    assert lib.sa_debug_fwd_walk_log_bytes(1, 2, 1024, 128, 128) == (3 * 16 + 3 * 16 * 8) * 4
    assert lib.sa_debug_fwd_walk_log_bytes(1, 2, 1000, 128, 128) == 0
    # (64,64,64) has no walk-recording kernel; a short log is refused before any CUDA call
    assert lib.sa_debug_fwd_walk(16, 16, 16, 16, 16, 16, 1, 2, 1024, 1024, 64, 64, 64, 0.125, 16, 1 << 20,
                                 16, 1 << 20, None) == 2
    assert lib.sa_debug_fwd_walk(16, 16, 16, 16, 16, 16, 1, 2, 1024, 1024, 128, 128, 128, 0.125, 16, 1 << 20,
                                 16, 64, None) == 4
    assert lib.sa_fwd_softmax_path_counts(None, None, None, None) == 1


def test_product_does_not_import_oracle():
    # the product path must not route through the oracle (or any CPU fallback)
    pkg = os.path.join(ROOT, "paper_2606_23019_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
                assert "sa_oracle" not in src, f
    osrc = open(os.path.join(ROOT, "oracle", "sa_oracle.cpp")).read()
    assert "#include \"" not in osrc          # the oracle includes no project header
    assert "paper_2606_23019_b200" not in open(os.path.join(ROOT, "oracle", "__init__.py")).read().replace(
        "paper_2606_23019_b200 and the product never imports it", "")
