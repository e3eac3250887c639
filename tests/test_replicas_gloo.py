"""-m "not gpu": the N > 1 path of bench.py is "replicas only" — independent solves, timing
aggregated as MAX over ranks, value = all ranks' units / that time.  Covered here with 2 gloo processes."""
import os
import socket

import pytest
import torch
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    from paper_1108_2045_b200 import replicas
    r, w = replicas.init("gloo")
    assert (r, w) == (rank, world)
    replicas.barrier()
    # rank r "measures" (10 + r) ms of solve time and (1 + 2 r) s end to end
    total_ms, e2e_s = replicas.max_over_ranks([10.0 + rank, 1.0 + 2.0 * rank])
    val = replicas.job_value(1000, 5, w, total_ms)
    q.put((rank, total_ms, e2e_s, val))
    replicas.barrier()
    torch.distributed.destroy_process_group()


def test_two_replicas_aggregate_by_max_over_ranks():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    out = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    for rank, total_ms, e2e_s, val in out:
        assert total_ms == 11.0 and e2e_s == 3.0                 # the slower rank decides, on every rank
        assert val == pytest.approx(1000 * 5 * 2 / 11e-3)         # units of BOTH ranks / max time


def test_single_process_is_a_noop():
    from paper_1108_2045_b200 import replicas
    assert replicas.max_over_ranks([3.5, 1.25]) == [3.5, 1.25]
    assert replicas.job_value(10, 2, 1, 4.0) == pytest.approx(10 * 2 / 4e-3)
