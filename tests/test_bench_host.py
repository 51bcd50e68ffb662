"""Host logic of bench.py that runs without a GPU: the replica aggregation (DESIGN.md section 9:
replicas only - the single cross-rank step is a MAX over the device-timed milliseconds), exercised
with two gloo ranks on CPU, and the flop accounting."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = 100.0 + 25.0 * rank                      # rank 1 is the slow replica
    dist.barrier()
    worst = bench.max_over_ranks(dist, ms, torch.device("cpu"))
    out[rank] = (worst, bench.aggregate_value(world, 1000, worst))
    dist.destroy_process_group()


def test_replica_timing_is_max_over_ranks_gloo():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1] == (125.0, 2 * 1000 / 0.125)


def test_single_process_path_and_flop_accounting():
    import bench
    import workloads
    assert bench.max_over_ranks(None, 7.5, torch.device("cpu")) == 7.5
    c = workloads.config(2)
    tot, row, per_w = bench.algorithmic_flops(c)
    npair = 80
    assert row == npair * 120000 * 5.0 * 256 * 8
    assert per_w[5] == (120000 - 64 + 1) * npair * (256 * 5.0 * 128 * 7 + 5.0 * 128 * 256)
    assert abs(tot - 2.21e13) < 0.02e13                     # 2.21e13 algorithmic flops
    assert abs(bench.nominal_flops(c) - 4.36e13) < 0.03e13  # ... and 4.36e13 nominal


def test_traffic_table_and_executed_flops():
    import bench
    import workloads
    tab = bench.ncu_traffic_table()
    assert (2, "slide", 64) in tab and tab[(2, "slide", 64)][0] > 1e9 and "profiles/" in tab[(2, "slide", 64)][1]
    c = workloads.config(2)
    # sliding kernel, w = 64 (Nt 128, Nf 256): 7.9 flops per bin per window (ncu-pinned), 5 launches
    ex = bench.executed_flops_per_launch(c, 6, 5, 5, 80, c["nap"], 1.0)
    assert ex == (120000 - 64 + 1) * 80 * 128 * 256 * 7.9 / 5
    # k_colfft2 at Nt = 512: the counter-pinned flops per (window, column); kernels without a capture: the algorithmic count
    c4 = workloads.config(4)
    assert bench.executed_flops_per_launch(c4, 7, 0, 7, 84, 20000, 123.0) == 1247 * 84 * 2048 * 13700.0 / 7
    assert bench.executed_flops_per_launch(c4, 1, -1, 7, 84, 20000, 123.0) == 123.0
    # the same launches as FP32 lane-operations (the pipe-level view); kernels without a capture give None
    assert bench.executed_ops_per_launch(c, 6, 5, 5, 80, c["nap"]) == (120000 - 64 + 1) * 80 * 128 * 256 * 5.17 / 5
    assert bench.executed_ops_per_launch(c4, 7, 2, 7, 84, 20000) == 309 * 84 * 2048 * 14178.0 / 7
    assert bench.executed_ops_per_launch(c4, 1, -1, 7, 84, 20000) is None
    # the folded sliding sum (kind 14): 1.22 flops, 0.81 lane-operations and 0.045 warp instructions per bin per window
    bins = (120000 - 64 + 1) * 80 * 128 * 256
    assert bench.executed_flops_per_launch(c, 14, 5, 5, 80, c["nap"], 1.0) == bins * 1.22 / 5
    assert bench.executed_ops_per_launch(c, 14, 5, 5, 80, c["nap"]) == bins * 0.81 / 5
    assert abs(bench.executed_warp_inst_per_launch(c, 14, 5, 5, 80, c["nap"]) - bins * 0.04497 / 5) < 1e-3 * bins * 0.045 / 5
    assert bench.executed_warp_inst_per_launch(c, 6, 0, 5, 80, c["nap"]) is None     # the narrow widths: no capture
    assert bench.executed_warp_inst_per_launch(c, 1, -1, 5, 80, c["nap"]) is None
