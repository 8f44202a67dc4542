"""Host-side logic of bench.py: metric arithmetic, clock-log parsing, and the max-over-ranks /
sum-over-ranks aggregation of the replicas-only multi-GPU mode, covered with a world_size-2 gloo
run on CPU. No GPU needed."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import bench  # noqa: E402


def test_effective_tflops_arithmetic():
    # one active 128x128x128 block = 4*128*128*128 = 8 388 608 FLOP
    assert 4 * 128 * 128 * 128 == 8388608
    # 2.79 M blocks in 23.8 ms is the "60% of 1643 TFLOP/s" budget of BASELINE.md section 4
    tf = bench.effective_tflops(2_790_000, 8388608, 23.8)
    assert abs(tf - 983.4) < 1.0
    assert bench.effective_tflops(1, 10 ** 12, 1000.0) == pytest.approx(1.0)


def test_parse_clock_csv():
    text = (
        "index, clocks.current.sm [MHz], clocks.max.sm [MHz], power.draw [W], clocks_event_reasons.active, "
        "hw_slowdown, hw_thermal_slowdown, sw_thermal_slowdown, sw_power_cap\n"
        "0, 1965 MHz, 1965 MHz, 310.2 W, 0x0000000000000000, Not Active, Not Active, Not Active, Not Active\n"
        "0, 1410 MHz, 1965 MHz, 998.1 W, 0x0000000000000004, Not Active, Not Active, Not Active, Active\n"
        "0, 1335 MHz, 1965 MHz, 1000.5 W, 0x0000000000000004, Not Active, Not Active, Not Active, Active\n")
    s = bench.parse_clock_csv(text)
    assert s["samples"] == 3 and s["sm_mhz"] == 1410.0 and s["sm_max_mhz"] == 1965.0
    assert s["reasons"] == ["sw_power_cap"]
    assert bench.parse_clock_csv("garbage\n")["samples"] == 0
    # timestamped form (what ClockSampler asks for) and a time window
    import datetime
    t0 = datetime.datetime(2026, 11, 5, 1, 2, 3).timestamp()
    rows = "".join(
        f"2026/11/05 01:02:0{3 + i}.500, 0, {1500 + 10 * i} MHz, 1965 MHz, {900 + i}.0 W, 0x4, Not Active, "
        f"Not Active, Not Active, Active\n" for i in range(5))
    s = bench.parse_clock_csv("timestamp, index, ...\n" + rows)
    assert s["samples"] == 5 and s["sm_mhz"] == 1520.0 and s["power_w_median"] == 902.0
    w = bench.parse_clock_csv(rows, t0 + 1.0, t0 + 3.0)         # samples at +1.5 and +2.5 s
    assert w["samples"] == 2 and w["sm_mhz"] == 1515.0


def test_load_peaks_has_measured_or_fallback():
    p = bench.load_peaks()
    assert p["source"] in ("measured", "fallback")
    assert 1000 < p["bf16_tflops"] < 2500 and 3000 < p["hbm_gbs"] < 9000


def test_aggregate_single_process_is_identity():
    v, ms, blocks = bench.aggregate_replicas(1000, 8388608, 2.0)
    assert ms == 2.0 and blocks == 1000
    assert v == pytest.approx(bench.effective_tflops(1000, 8388608, 2.0))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group(backend="gloo", rank=rank, world_size=world)
    try:
        # rank 0 is the slow replica: whole-job time is the max, units are the sum
        ms_local = 30.0 if rank == 0 else 20.0
        blocks_local = 1000 + rank
        v, ms, blocks = bench.aggregate_replicas(blocks_local, 8388608, ms_local, dist)
        q.put((rank, v, ms, blocks))
    finally:
        dist.destroy_process_group()


def test_replica_aggregation_world_size_2_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, v, ms, blocks in res:
        assert ms == 30.0 and blocks == 2001
        assert v == pytest.approx(bench.effective_tflops(2001, 8388608, 30.0))
