"""N > 1 path of bench.py on CPU: two gloo processes run the replica protocol (barrier, max over
ranks of the duration, sum of the units) - DESIGN.md section 8, "replicas only"."""
import os
import socket
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_1210_1017_b200 import replicas as R
    r = R.init("gloo")
    assert (r.rank, r.world, r.is_root) == (rank, world, rank == 0)
    R.barrier(r)
    # rank k "took" 10 + 5k ms for 1000 (k + 1) units
    ms_local = 10.0 + 5.0 * rank
    units_local = 1000.0 * (rank + 1)
    rate, ms = R.aggregate_rate(r, units_local, ms_local)
    mx = R.max_over_ranks(r, float(rank))
    sm = R.sum_over_ranks(r, 1.0)
    R.barrier(r)
    R.finalize(r)
    q.put((rank, rate, ms, mx, sm))


def test_two_replicas_gloo():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(k, world, port, q)) for k in range(world)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, rate, ms, mx, sm in out:
        assert ms == 15.0                       # slowest rank
        assert rate == 3000.0 / 15e-3           # all units / slowest time
        assert mx == 1.0 and sm == 2.0


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        os.environ.pop(k, None)
    from paper_1210_1017_b200 import replicas as R
    r = R.init()
    assert r.world == 1 and r.backend is None and r.is_root
    assert R.aggregate_rate(r, 500.0, 2.0) == (250000.0, 2.0)
    R.barrier(r)
    R.finalize(r)
