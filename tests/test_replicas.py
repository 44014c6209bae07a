"""N > 1 = independent replicas: the bench's cross-rank timing protocol on world_size-2 gloo (CPU)."""
import os
import socket

import torch.multiprocessing as mp

from paper_2502_02040_b200 import replicas


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    r = replicas.init_from_env(backend="gloo")
    replicas.barrier(r)
    # rank 0 took 10 ms for 256 tokens, rank 1 took 16 ms for 256 tokens
    ms = 10.0 if rank == 0 else 16.0
    t, u = replicas.aggregate(r, ms, 256)
    v = replicas.whole_job_throughput(r, ms, 256)
    out.put((rank, r.world, t, u, v, replicas.replica_seed(1000, r)))
    replicas.barrier(r)
    replicas.shutdown(r)


def test_two_rank_gloo_max_time_sum_units():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(i, 2, port, q)) for i in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    for rank, world, t, u, v, seed in res:
        assert world == 2
        assert t == 16.0                     # MAX over ranks
        assert u == 512.0                    # SUM of units
        assert abs(v - 512.0 / 0.016) < 1e-6  # whole-job tokens/s
    assert res[0][5] != res[1][5]            # each replica decodes its own prompt stream


def test_single_rank_needs_no_process_group():
    for k in ("WORLD_SIZE", "RANK", "LOCAL_RANK"):
        os.environ.pop(k, None)
    r = replicas.init_from_env()
    assert r.world == 1 and r.group is None
    replicas.barrier(r)
    assert replicas.aggregate(r, 5.0, 7) == (5.0, 7.0)
    assert replicas.whole_job_throughput(r, 5.0, 10) == 2000.0
