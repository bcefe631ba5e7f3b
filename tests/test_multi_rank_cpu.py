"""N > 1 host logic of bench.py on CPU: world_size 2, gloo.  The path partitions by plot (one
independent plot per rank), so there is no data-path collective to test -- only the
per-rank key derivation, the max-over-ranks of the device times and the whole-job aggregate."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    sys.path.insert(0, ROOT)
    import bench
    import vx_inputs
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # every rank plots under its own key
        seed = bench.rank_seed(31, rank)
        key = vx_inputs.key_from_seed(seed)
        keys = [None] * world
        dist.all_gather_object(keys, key)
        # rank r "measured" (10 + r) ms in total, e2e (0.5 - 0.1 r) s: the job's numbers are the MAX
        got = bench.max_over_ranks([10.0 + rank, 0.5 - 0.1 * rank], world)
        if rank == 0:
            out.put((keys, got, bench.whole_job_value(31, world, got[0])))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(120)
def test_two_ranks_gloo_keys_and_max_reduction():
    world = 2
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    keys, got, value = out.get(timeout=100)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert len(set(keys)) == world and all(len(k) == 32 for k in keys)
    import vx_inputs
    assert keys[0] == vx_inputs.config_key(31)           # rank 0 plots the BASELINE.json configuration
    assert got == [11.0, 0.5]                             # max over ranks, element-wise
    assert value == pytest.approx(2 * (1 << 31) / 11.0e-3)
