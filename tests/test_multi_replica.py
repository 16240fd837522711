"""N > 1 path of bench.py on CPU (gloo, world_size 2).  The method runs on one GPU with no data-path collective (BASELINE.json;
DESIGN.md section 7: "replicas only"), so the multi-rank logic is: barrier, max over ranks of the device-timed region, value = N x
one replica's work / that time.  Rendezvous on 127.0.0.1."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import bench


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dist.barrier()
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, "cpu")      # rank 1 is the slow replica
    val = bench.aggregate_value(3.0e9, ms / 5, world)
    out.put((rank, ms, val))
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_report_the_slowest_time_and_the_summed_throughput():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, val in res:
        assert ms == 15.0                                             # max over ranks, identical on every rank
        assert abs(val - 2 * 3.0e9 / (3.0e-3) / 1e9) < 1e-9           # 2 replicas x 3 GFLOP per step / 3 ms
    assert bench.max_over_ranks(7.0, 1, "cpu") == 7.0 and torch.distributed.is_available()
