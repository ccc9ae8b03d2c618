"""N > 1 host logic on CPU: world_size 2, gloo backend (the data path itself never communicates)."""
import os
import socket

import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1802_04449_b200 import replicas
    ms_local = 10.0 + 5.0 * rank                       # rank 1 is the slow one
    rate, ms = replicas.aggregate_rate(1000, 4, ms_local, world)
    dist.barrier()
    out.put((rank, rate, ms, replicas.rank_seed(4, rank)))
    dist.destroy_process_group()


def test_two_rank_aggregate_and_seeds():
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
    (r0, rate0, ms0, seed0), (r1, rate1, ms1, seed1) = res
    assert ms0 == ms1 == 15.0                          # max over ranks
    assert rate0 == rate1 == 2 * 1000 * 4 / 15e-3      # whole-job aggregate
    assert seed0 != seed1 and seed1 == seed0 + 1       # one seeded event per rank


def test_single_process_is_identity():
    from paper_1802_04449_b200 import replicas
    rate, ms = replicas.aggregate_rate(10, 2, 4.0, 1)
    assert ms == 4.0 and rate == 10 * 2 / 4e-3
