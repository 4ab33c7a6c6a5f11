"""N > 1 path of bench.py on CPU: two gloo ranks.  The hot path does not shard across GPUs ("replicas only",
DESIGN.md §8): each rank draws its own clusters and there is no data-path collective; the only exchange is the
MAX-over-ranks of the device time and the SUM of the units processed, after the timed region."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import bench
from workloads import make_cluster


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q) -> None:
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    specs = bench.workload_specs("config0", rank)
    flops = sum(bench.alg_flops(s)["total"] for s in specs)
    ms, units = bench.reduce_over_ranks(10.0 + 5.0 * rank, flops, world, torch.device("cpu"))
    x = make_cluster(specs[0])
    q.put((rank, ms, units, flops, specs[0].cluster_id, float(x.e_occ[0])))
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_max_time_sum_units():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, ms0, u0, f0, c0, e0), (r1, ms1, u1, f1, c1, e1) = out
    assert ms0 == ms1 == 15.0                      # MAX over ranks
    assert u0 == u1 == f0 + f1                     # whole-job units
    assert c0 != c1 and e0 != e1                   # each replica draws its own cluster


def test_single_process_is_identity():
    assert bench.reduce_over_ranks(3.0, 7.0, 1, None) == (3.0, 7.0)
