"""The N > 1 path of bench.py ("replicas only"): barrier, max-over-ranks and the whole-job
aggregate, exercised with world_size 2 on CPU over gloo."""
import os
import socket

import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    from paper_2012_06144_b200 import replicas
    r, lr, w = replicas.init("gloo")
    assert (r, lr, w) == (rank, rank, world)
    replicas.barrier()
    ms = replicas.max_over_ranks(10.0 + 5.0 * rank)          # rank 1 is the slow one
    replicas.barrier()
    q.put((rank, ms, replicas.aggregate_mlups(1000, 20, ms, w)))
    replicas.shutdown()


def test_two_rank_replicas_over_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, mlups in out:
        assert ms == 15.0                                      # max over ranks, on every rank
        assert abs(mlups - 2 * 1000 * 20 / 15e-3 / 1e6) < 1e-12


def test_single_process_is_passthrough():
    from paper_2012_06144_b200 import replicas
    os.environ.pop("WORLD_SIZE", None)
    assert replicas.env_ranks()[2] == 1
    assert replicas.max_over_ranks(3.5) == 3.5
    replicas.barrier()
    assert replicas.aggregate_mlups(10 ** 6, 10, 1.0, 1) == 10 ** 4
