"""world_size-2 CPU test (gloo) of the only multi-process logic this build has:
"replicas only" bookkeeping (sum of lattice updates, max of device time)."""
import os
import socket
import sys

import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    from paper_1011_2613_b200 import replicas
    r, w, _ = replicas.init_from_env(backend="gloo")
    replicas.barrier()
    units, ms = replicas.aggregate(1000.0 * (rank + 1), 10.0 + 5.0 * rank)
    q.put((r, w, units, ms, replicas.mlups(units, ms)))
    replicas.barrier()
    replicas.shutdown()


def test_two_replicas_aggregate_sum_and_max():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, (r, w, units, ms, ml) in enumerate(res):
        assert (r, w) == (rank, 2)
        assert units == 3000.0 and ms == 15.0
        assert ml == pytest.approx(3000.0 / 0.015 / 1e6)


def test_aggregate_is_identity_without_a_process_group():
    sys.path.insert(0, ROOT)
    from paper_1011_2613_b200 import replicas
    assert replicas.aggregate(5.0, 2.0) == (5.0, 2.0)
