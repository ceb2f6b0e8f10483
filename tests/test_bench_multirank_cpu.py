"""The N > 1 path of bench.py on CPU: two gloo ranks, each a replica with its own seed, timings
reduced with MAX over ranks, bytes summed (weak scaling; the data path has no collective)."""
import os
import socket

import numpy as np
import torch
import torch.multiprocessing as mp

import bench


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.distributed.init_process_group("gloo", rank=rank, world_size=world)
    try:
        times = [10.0 + rank, 20.0 - rank, 1.5 * (rank + 1)]        # rank-dependent "timings"
        red = bench.max_over_ranks(times, world, "cpu")
        wl = bench._workload(1, rank)
        out.put((rank, red, int(wl.seed), wl.ctx_lens.tolist(), wl.block_tables.shape))
    finally:
        torch.distributed.destroy_process_group()


def test_two_gloo_ranks_reduce_max_and_shard_by_replica():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_rank_main, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, red, seed, lens, shape in res:
        assert red == [11.0, 20.0, 3.0]                            # MAX over ranks, identical on every rank
    assert res[0][2] != res[1][2]                                  # each replica draws its own values ...
    assert res[0][3] == res[1][3] and res[0][4] == res[1][4]       # ... with the same structure


def test_whole_job_value_is_aggregate_over_replicas():
    one = bench.whole_job_value(10**9, 1, 1.0)
    assert one == 1000.0                                           # 1 GB per ms = 1000 GB/s
    assert bench.whole_job_value(10**9, 8, 1.0) == 8 * one


def test_step_bytes_accounting_matches_survey_figures():
    wl = bench._workload(2, 0)
    total, decode = bench.step_bytes(wl, 9, wl.ctx_lens.astype(np.int32), 1)
    kv = 32 * 32768 * 4 * 136                                      # 136 B per (token, kv head)
    assert kv == 570_425_344 and decode > kv and total > decode
    assert decode - kv == 4 * 32 * 2048 + 32 * 64 * 128 + 32 * 64 * 9 * 520
