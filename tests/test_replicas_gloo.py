"""N > 1 path on CPU: world_size 2 over gloo (127.0.0.1).  Replicas exchange only timing scalars."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2607_02043_b200 import replicas as R
    from paper_2607_02043_b200 import workloads as W
    local_ms = 10.0 + 5.0 * rank                      # rank 1 is the slow one
    us = R.whole_job_us_per_step(local_ms, steps=5, world=world)
    a = W.make_inputs("t", 7 + R.replica_seed_shift(rank), [70, 130], 8, 3)
    sig = int(a.pool[:2].astype("int64").sum())
    sigs = [None] * world
    dist.all_gather_object(sigs, (sig, a.pool.shape, int(a.dec_ctx_lens.sum())))
    dist.barrier()
    q.put((rank, us, sigs))
    dist.destroy_process_group()


def test_two_replicas_aggregate_by_slowest_rank():
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
    for rank, us, sigs in res:
        assert abs(us - 15.0 * 1e3 / (5 * 2)) < 1e-9          # max over ranks, 2 replicas advance per iteration
        assert sigs[0][1:] == sigs[1][1:]                      # same shapes / lengths
        assert sigs[0][0] != sigs[1][0]                        # independent data


def test_single_process_needs_no_group():
    from paper_2607_02043_b200 import replicas as R
    assert not dist.is_initialized()
    assert R.whole_job_us_per_step(2.0, steps=4, world=1) == 500.0
