"""N > 1 host logic on CPU: two processes over gloo (127.0.0.1).  The data path has no collective, so what
there is to test is the sharding rule (every rank gets its own sequences) and the timing reduction bench.py reports
(max over ranks, whole-job tokens / s)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_04511_b200 import shard, synth


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = shard.rank_config(synth.CFG1_TINY, rank)
    L = synth.decode_layer(cfg, 0, device="cpu")
    # each rank's own step time; the job's step time is the slowest rank's
    ms_local = 10.0 + 5.0 * rank
    ms = shard.max_over_ranks(ms_local)
    # gather the rank seeds and a checksum of the rank's sequences to rank 0
    info = [None] * world
    dist.all_gather_object(info, (cfg.seed, float(L["kv"].float().sum()), ms))
    if rank == 0:
        out.put(info)
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_shard_by_sequence_and_reduce_time_by_max():
    world = 2
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    info = out.get(timeout=120)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    seeds = [i[0] for i in info]
    sums = [i[1] for i in info]
    assert seeds[0] != seeds[1] and sums[0] != sums[1], "ranks must decode different sequences"
    assert all(i[2] == 15.0 for i in info), "step time of the job = max over ranks on every rank"
    v = shard.whole_job_value(synth.CFG3_128K.batch, world, 15.0)
    assert abs(v - 2 * 4 / 0.015) < 1e-9


def test_single_process_is_identity():
    assert shard.max_over_ranks(3.5) == 3.5
    assert shard.rank_config(synth.CFG3_128K, 0) == synth.CFG3_128K
