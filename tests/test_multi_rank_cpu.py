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


# ------------------------------------------------------------------ one plot over G ranks
# The sharded build's exchange step, with the CPU standing in for the kernels: every rank takes its
# nonce share and its bucket range from the library's own ownership arithmetic (vx_shard_owner: host
# code of libvx, no GPU needed), hashes its share with the oracle, sends every record to the rank that
# owns its bucket (one all-to-all, spelled with gloo's all_gather), and the owner puts what it received into canonical form.
# The union of the ranks' slices must be the oracle's one-process Table 1, and their Table 2 its Table 2.
def _shard_worker(rank: int, world: int, port: int, K: int, B: int, seed: int, out):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import numpy as np
    import oracle
    import paper_2606_14007_b200 as vx
    import vx_inputs
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        key = vx_inputs.key_from_seed(seed)
        n0, n1, b0, b1 = vx.shard_owner(K, B, world, rank)
        ranges = [None] * world
        dist.all_gather_object(ranges, (n0, n1, b0, b1))
        H = oracle.hash_range(key, oracle.nonce_size(K), n0, n1 - n0)
        nonces = np.arange(n0, n1, dtype=np.uint64)
        bucket = (H >> np.uint64(64 - B)).astype(np.int64)
        send = []
        for g in range(world):
            gb0, gb1 = ranges[g][2], ranges[g][3]
            sel = (bucket >= gb0) & (bucket < gb1)
            send.append(torch.from_numpy(np.stack([nonces[sel], H[sel]]).view(np.int64).copy()))
        # gloo has no all-to-all: every rank publishes its per-destination lists and takes its own column
        everyone = [None] * world
        dist.all_gather_object(everyone, [t.numpy() for t in send])
        recv = [torch.from_numpy(everyone[g][rank]) for g in range(world)]
        got = torch.cat(recv, dim=1).numpy().view(np.uint64)
        off, non, has = oracle.table1_from_records(B, b0, b1, got[0], got[1])
        t2o, p1, p2 = oracle.table2(K, off, non, has, 1)
        out.put((rank, ranges[rank], off, non, has, t2o, p1, p2))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(180)
@pytest.mark.parametrize("world", [2, 4])
def test_sharded_plot_ownership_and_exchange_gloo(world):
    import numpy as np
    sys.path.insert(0, ROOT)
    import oracle
    import vx_inputs
    K, B, seed = 14, 9, 5
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_shard_worker, args=(r, world, port, K, B, seed, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted([out.get(timeout=150) for _ in range(world)], key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # ownership: nonce shares and bucket ranges tile [0, 2^K) and [0, 2^B) with no gap and no overlap
    assert res[0][1][0] == 0 and res[-1][1][1] == 1 << K and res[0][1][2] == 0 and res[-1][1][3] == 1 << B
    for a, b in zip(res[:-1], res[1:]):
        assert a[1][1] == b[1][0] and a[1][3] == b[1][2]
    key = vx_inputs.key_from_seed(seed)
    o_off, o_non, o_has = oracle.table1(K, key, B)
    o_t2o, o_n1, o_n2 = oracle.table2(K, o_off, o_non, o_has, 1)
    for rank, (n0, n1, b0, b1), off, non, has, t2o, p1, p2 in res:
        lo, hi = int(o_off[b0]), int(o_off[b1])
        assert np.array_equal(off, o_off[b0:b1 + 1] - o_off[b0])
        assert np.array_equal(non, o_non[lo:hi]) and np.array_equal(has, o_has[lo:hi])
        l2, h2 = int(o_t2o[b0]), int(o_t2o[b1])
        assert np.array_equal(t2o, o_t2o[b0:b1 + 1] - o_t2o[b0])
        assert np.array_equal(p1, o_n1[l2:h2]) and np.array_equal(p2, o_n2[l2:h2])
