"""world_size-2 gloo test of the N>1 host logic: shards are independent (no data-path collective),
seeds differ per rank, and the job time is the MAX over ranks while units are SUMMED."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_11867_b200 import multi, synth


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    assert multi.env_rank() == (rank, rank, world)
    assert multi.init("gloo")
    cfg = synth.config(1, seed=multi.shard_seed(0, rank))
    ids, w, mb_off = synth.gen_trace(cfg, "cpu")
    multi.barrier()
    t, u = multi.aggregate(10.0 + 5.0 * rank, float(cfg.T * cfg.L))
    # every rank's trace differs (its own shard), gathered only for this assertion
    sums = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(sums, ids.to(torch.int64).sum().reshape(1))
    out.put((rank, t, u, [int(s) for s in sums]))
    dist.destroy_process_group()


def test_gloo_world2_aggregate():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = [out.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    cfg = synth.config(1)
    for rank, t, u, sums in res:
        assert t == 15.0                        # max over ranks
        assert u == 2.0 * cfg.T * cfg.L         # sum over ranks
        assert sums[0] != sums[1]               # independent shards


def test_single_process_passthrough():
    assert multi.aggregate(3.0, 7.0) == (3.0, 7.0)
    assert multi.shard_seed(0, 0) == 0 and multi.shard_seed(0, 1) != multi.shard_seed(0, 2)
