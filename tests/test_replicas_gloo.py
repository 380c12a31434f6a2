"""world_size-2 CPU test (gloo) of the only multi-rank logic on the path: the replicas-only timing
protocol used by bench.py --gpus N (barrier, MAX over ranks, whole-job throughput)."""
import os
import socket

import pytest
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, size, port, out):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(size), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    from paper_1008_2042_b200 import replicas
    replicas.init("gloo")
    assert replicas.world() == (rank, size, rank)
    replicas.barrier()
    seconds = 2.0 if rank == 0 else 3.0                      # rank 1 is the slow replica
    mx = replicas.max_over_ranks(seconds)
    thr = replicas.job_throughput(60.0, seconds)
    replicas.barrier()
    replicas.shutdown()
    out.put((rank, mx, thr))


def test_two_replicas_take_the_slowest_time():
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
    for rank, mx, thr in res:
        assert mx == 3.0                                     # MAX over ranks, on every rank
        assert thr == pytest.approx(2 * 60.0 / 3.0)         # 2 replicas x 60 units / slowest 3 s


def test_single_process_is_a_no_op():
    from paper_1008_2042_b200 import replicas
    assert replicas.max_over_ranks(1.5) == 1.5
    assert replicas.job_throughput(10.0, 2.0) == 5.0
    replicas.barrier()
