"""World-size-2 gloo test (CPU) of the only multi-GPU logic the path has: independent replicas,
barrier, max-over-ranks timing and summed units ("replicas only")."""
import os
import socket

import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_1610_05329_b200 import replicas
    r, lr, w = replicas.init(backend="gloo")
    replicas.barrier()
    seconds = 2.0 + rank            # rank 1 is the slow one
    units = 10.0 * (rank + 1)
    value, t = replicas.aggregate_throughput(units, seconds)
    q.put((r, w, value, t, replicas.max_over_ranks(rank), replicas.replica_seed(4, rank)))
    replicas.barrier()
    replicas.shutdown()


def test_two_replicas_aggregate_by_max_time_and_summed_units():
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
    for rank, (r, w, value, t, mx, seed) in enumerate(res):
        assert (r, w) == (rank, 2)
        assert t == 3.0                     # max over ranks
        assert abs(value - 30.0 / 3.0) < 1e-12   # (10 + 20) units / slowest time
        assert mx == 1.0
        assert seed == 4 + 1000 * rank


def test_single_process_needs_no_process_group():
    from paper_1610_05329_b200 import replicas
    assert replicas.env_world()[2] >= 1
    assert replicas.max_over_ranks(1.5) == 1.5
    v, t = replicas.aggregate_throughput(8.0, 2.0)
    assert (v, t) == (4.0, 2.0)
