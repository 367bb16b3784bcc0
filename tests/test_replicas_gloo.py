"""N > 1 path of bench.py ("replicas only") on CPU: world_size 2, gloo.  Checks that the whole-job
value is (units of all ranks) / (MAX over ranks of the time) and that no rank needs anything from another
beyond that scalar."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    import torch.distributed as dist
    from paper_2512_18010_b200 import replicas
    assert replicas.env_rank_world_local() == (rank, world, rank)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        local_ms = 10.0 * (rank + 1)                 # rank 1 is the slow one: 20 ms over 4 steps
        value, ms_per_step = replicas.whole_job_value(1000.0, 4, local_ms)
        mx = replicas.max_over_ranks(float(rank))
        q.put((rank, value, ms_per_step, mx))
    finally:
        dist.destroy_process_group()


def test_replicas_world2_gloo():
    import torch.multiprocessing as mp
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
    for rank, value, ms_per_step, mx in res:
        assert ms_per_step == pytest.approx(5.0)              # max(10, 20) ms / 4 steps
        assert value == pytest.approx(2 * 1000.0 / 5e-3)      # both ranks' units over the slower rank's time
        assert mx == 1.0


def test_single_process_identity():
    sys.path.insert(0, ROOT)
    from paper_2512_18010_b200 import replicas
    value, ms = replicas.whole_job_value(500.0, 5, 10.0)
    assert ms == pytest.approx(2.0) and value == pytest.approx(500.0 / 2e-3)
