"""world_size-2 gloo test of the N > 1 host logic ("replicas only": barrier + max-over-ranks timing)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2605_25863_b200 import replicas
    import linac_inputs as gen
    seed = replicas.replica_seed(4, rank)
    a = gen.uniform_matrix(8, 8, 2147483647, seed)
    my_time = 1.0 + rank            # rank 1 is the slow one
    dist.barrier()
    tmax = replicas.max_over_ranks(my_time)
    agg = replicas.aggregate_throughput(100.0, tmax, world)
    out.put((rank, seed, int(a[0, 0]), tmax, agg))
    dist.destroy_process_group()


def test_two_rank_replicas_timing_and_seeds():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, v0, t0, a0), (r1, s1, v1, t1, a1) = res
    assert (s0, s1) == (4, 1004) and v0 != v1          # independent matrices per rank
    assert t0 == t1 == 2.0                             # max over ranks
    assert a0 == a1 == 2 * 100.0 / 2.0                 # whole-job units / slowest rank


def test_single_process_is_identity():
    from paper_2605_25863_b200 import replicas
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.aggregate_throughput(10.0, 2.0, 1) == 5.0
