"""world_size-2 gloo test of the replica mode's host logic: per-rank seeds, the
max-over-ranks timing reduction and the whole-job value.  CPU only."""
import os
import socket

import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp

from paper_2411_11725_b200 import replicas, workloads as wl


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        r, w, l = replicas.rank_info()
        assert (r, w, l) == (rank, world, rank)
        sec = 1.0 + 0.5 * rank                       # rank 1 is the slow one
        slow = replicas.max_over_ranks(sec)
        seed = replicas.replica_seed(16, rank)
        m0 = wl.random_unit_field((17, 17, 17), seed)
        out.put((rank, slow, seed, float(m0[0, 0, 0, 0]),
                 replicas.job_value(world, 6, 16 ** 3, 10, slow)))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_replicas_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, slow0, seed0, v0, job0), (r1, slow1, seed1, v1, job1) = res
    assert slow0 == slow1 == 1.5                     # both ranks report the slowest rank's time
    assert seed0 == 20 and seed1 == 21 and v0 != v1  # replica 0 is config 4's own input
    assert job0 == job1 == 2 * 6 * 16 ** 3 * 10 / 1.5 / 1e6


def test_single_process_defaults():
    assert replicas.rank_info({}) == (0, 1, 0)
    assert replicas.max_over_ranks(0.25) == 0.25
    assert wl.config4_sweep(16).seed == replicas.replica_seed(16, 0)
