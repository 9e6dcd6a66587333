"""N > 1 path of bench.py on CPU: world_size 2, gloo.  The path has no exchange step (replicas only), so what is
covered is the plumbing: rendezvous, barrier, max-over-ranks timing, whole-job aggregation, rank-0 reporting."""
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
    from paper_1411_3396_b200.replicas import Replicas
    r = Replicas(backend="gloo")
    r.barrier()
    t_local = 100.0 + 50.0 * rank                      # rank 1 is the slow one
    value, t_max = r.aggregate_rate(1.0e9, 4, t_local)
    q.put((rank, r.world, value, t_max, r.is_reporter()))
    r.barrier()
    r.close()


def test_replicas_world2_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, world, value, t_max, rep in out:
        assert world == 2 and t_max == 150.0                       # max over ranks, not the local time
        assert abs(value - 2 * 4 * 1.0e9 / 0.150) < 1e-3           # units of ALL ranks / max time
        assert rep == (rank == 0)


def test_replicas_single_process():
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        os.environ.pop(k, None)
    from paper_1411_3396_b200.replicas import Replicas
    r = Replicas()
    assert r.world == 1 and r.is_reporter()
    v, t = r.aggregate_rate(10.0, 5, 1000.0)
    assert v == 50.0 and t == 1000.0
