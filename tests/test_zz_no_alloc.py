"""sa_pack_mask_static: the mask pack with the library's fixed scratch array as its workspace (for
callers that cannot allocate device memory). Collected last on purpose (pytest -x).
Checks the entry point against the existing path (sa_pack_mask with a caller's workspace) and the
oracle: bit-exact, on two calls in a row, with no device allocation during the calls."""
import os
import sys

import numpy as np
import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2606_23019_b200 import inputs  # noqa: E402


def _host_bits(t):
    return t.cpu().numpy().view(np.uint32)


@pytest.mark.gpu
def test_pack_mask_static_matches_existing_path_two_calls_in_a_row():
    from paper_2606_23019_b200 import binding as sa
    sa.load_library()
    assert torch.cuda.is_available()
    dev = torch.device("cuda", 0)
    rng = np.random.Generator(np.random.PCG64(2024))
    # first call: a head grid with heavy ties (the tie-count scratch is used) and a forced diagonal;
    # second call: a different, larger shape with real-valued scores, right behind it on the stream,
    # so anything the first call left in the shared array would show
    H1, NQB1, NKB1 = 6, 70, 90
    s1 = np.round(rng.random((H1, NQB1, NKB1)).astype(np.float32) * 4) / 4
    d1 = rng.uniform(0.05, 0.9, size=H1).astype(np.float32)
    cfg = inputs.scaled(inputs.C4, H=8)
    s2, d2, _ = inputs.make_block_scores(cfg)
    cases = []
    for s, d, fd in ((s1, d1, True), (s2, d2, True), (s1, d1, False)):
        st, dt = torch.from_numpy(s).to(dev), torch.from_numpy(d).to(dev)
        out = torch.zeros((s.shape[0], s.shape[1], (s.shape[2] + 31) // 32), dtype=torch.int32, device=dev)
        cases.append((s, d, fd, st, dt, out))
    want = [sa.sa_pack_mask(st, dt, fd) for (_, _, fd, st, dt, _) in cases]      # the existing path
    torch.cuda.synchronize()
    for (_, _, fd, st, dt, out) in cases:                                        # back to back, one stream
        sa.sa_pack_mask_static(st, dt, out, fd)
        assert sa.sa_last_launch_count() == 5
    torch.cuda.synchronize()
    for (s, d, fd, _, _, out), w in zip(cases, want):
        assert torch.equal(out, w)                          # bit-exact against sa_pack_mask
        assert (_host_bits(out) == oracle.pack_mask(s, d, 1 if fd else 0)).all()
    # and once more, from the array as the calls above left it: the same results, and no device memory
    # taken (the first call on a device may make the driver load the library's module, array included;
    # from then on neither torch's allocator nor the driver's free-memory figure moves)
    for (_, _, _, _, _, out) in cases:
        out.zero_()
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated(dev)
    free_before, _ = torch.cuda.mem_get_info(dev)
    for (_, _, fd, st, dt, out) in cases:
        sa.sa_pack_mask_static(st, dt, out, fd)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated(dev) == before
    free_after, _ = torch.cuda.mem_get_info(dev)
    assert free_after >= free_before
    for (_, _, _, _, _, out), w in zip(cases, want):
        assert torch.equal(out, w)


@pytest.mark.gpu
def test_pack_mask_static_rejects_sizes_beyond_the_array():
    from paper_2606_23019_b200 import binding as sa
    sa.load_library()
    dev = torch.device("cuda", 0)
    H, NQB, NKB = 128, 8, 8                                  # 128 heads of histograms: 3 MiB > 2.25 MiB
    assert sa.sa_pack_mask_workspace_bytes(H, NQB, NKB) > sa.SA_STATIC_SCRATCH_BYTES
    s = torch.rand((H, NQB, NKB), device=dev)
    d = torch.full((H,), 0.5, device=dev)
    out = torch.zeros((H, NQB, 1), dtype=torch.int32, device=dev)
    with pytest.raises(sa.SAError) as ei:
        sa.sa_pack_mask_static(s, d, out)
    assert "SA_ERR_WORKSPACE" in str(ei.value) and "fixed array" in str(ei.value)
    assert (out == 0).all()                                  # nothing ran
    # the largest documented case fits: H = 64 at 2048 x 2048 blocks
    assert sa.sa_pack_mask_workspace_bytes(64, 2048, 2048) <= sa.SA_STATIC_SCRATCH_BYTES
