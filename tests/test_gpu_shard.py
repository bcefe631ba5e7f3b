"""One plot over G GPUs -- the fused exchange + first partition pass, on ONE
device: G plots with the same key and G workspaces stand for G ranks and their peer-mapped memory
(only one GPU is available to this build; DESIGN.md says "unmeasured on hardware").  Every "rank"
hashes its nonce share and stores each record into its owner's workspace through the peer table;
after the barriers each rank sorts and matches its slice alone.  The union of the slices must be the
oracle's tables, bit for bit."""
import numpy as np
import pytest

import oracle
import vx_inputs
from vx_testlib import canon_t2, decode_t2, oracle_tables

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def vx():
    import paper_2606_14007_b200 as m
    m.load_library()
    return m


@pytest.mark.parametrize("world", [2, 4, 8])
@pytest.mark.parametrize("big", [0, 2])
@pytest.mark.parametrize("K,B,seed", [(16, 12, 1), (18, 24, 3), (20, 24, 1), (22, 24, 22)])
def test_sharded_build_union_equals_oracle(vx, K, B, seed, big, world):
    import torch
    wl = world.bit_length() - 1
    if K - (13 if big else 12) < wl:
        pytest.skip("fewer partitions than ranks")
    key = vx_inputs.key_from_seed(seed)
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_tables(K, key, B)
    plots = [vx.Plot(K, key, B, flags=big | vx.VX_CREATE_PASSES_LOG(wl)) for _ in range(world)]
    peers = [p.workspace.data_ptr() for p in plots]
    streams = [torch.cuda.Stream() for _ in range(world)]
    for r, p in enumerate(plots):
        p.shard_begin(r, world, streams[r])
    torch.cuda.synchronize()                              # BARRIER: every rank's cursors are zero
    for r, p in enumerate(plots):
        p.shard_scatter(r, world, peers, streams[r])      # the "ranks" scatter concurrently
    torch.cuda.synchronize()                              # BARRIER: every record has reached its owner
    t1 = t2 = 0
    for r, p in enumerate(plots):
        p.shard_finish(streams[r])
        p.sort_match_table2(streams[r])
    for r, p in enumerate(plots):
        n0, n1, b0, b1 = vx.shard_owner(K, B, world, r)
        assert (b0, b1) == p.pass_buckets()
        lo, hi = int(o_off[b0]), int(o_off[b1])
        off1, raw1 = p.read_tables(1)
        assert np.array_equal(off1, o_off[b0:b1 + 1] - o_off[b0])
        assert np.array_equal(raw1, oracle.serialize_t1(4, o_non[lo:hi], o_has[lo:hi]))
        off2, raw2 = p.read_tables(2)
        l2, h2 = int(o_t2o[b0]), int(o_t2o[b1])
        assert np.array_equal(off2, o_t2o[b0:b1 + 1] - o_t2o[b0])
        g1, g2 = canon_t2(off2, *decode_t2(raw2, 4))
        assert np.array_equal(g1, o_n1[l2:h2]) and np.array_equal(g2, o_n2[l2:h2])
        st = p.get_stats()
        t1 += st["t1_records"]
        t2 += st["t2_records"]
    assert t1 == 1 << K and t2 == len(o_n1)
    # a second round on the same handles gives the same slices (cursors reset by shard_begin)
    for r, p in enumerate(plots):
        p.shard_begin(r, world, streams[r])
    torch.cuda.synchronize()
    for r, p in enumerate(plots):
        p.shard_scatter(r, world, peers, streams[r])
    torch.cuda.synchronize()
    for r, p in enumerate(plots):
        p.shard_finish(streams[r])
        p.sort_match_table2(streams[r])
        assert p.get_stats()["t1_records"] == int(o_off[p.pass_buckets()[1]] - o_off[p.pass_buckets()[0]])
    for p in plots:
        p.free()


def test_shard_arguments(vx):
    key = vx_inputs.key_from_seed(1)
    one = vx.Plot(18, key, 12)                               # a one-pass plot cannot be a shard
    with pytest.raises(vx.VxError) as ei:
        one.shard_begin(0, 2)
    assert ei.value.status == -1
    one.free()
    p = vx.Plot(18, key, 12, flags=vx.VX_CREATE_PASSES_LOG(1))
    with pytest.raises(vx.VxError):
        p.shard_begin(2, 2)                                  # rank outside the world
    p.shard_begin(1, 2)
    with pytest.raises(vx.VxError):
        p.shard_scatter(0, 2, [p.workspace.data_ptr()] * 2)  # begun as rank 1
    with pytest.raises(vx.VxError):
        p.shard_scatter(1, 2, [p.workspace.data_ptr(), 0])   # NULL peer / own entry wrong
    p.free()
    w = vx.Plot(18, key, 12, flags=vx.VX_CREATE_WIDE_LAYOUT | vx.VX_CREATE_PASSES_LOG(1))
    with pytest.raises(vx.VxError) as ei:
        w.shard_begin(0, 2)
    assert ei.value.status == -7
    w.free()
    assert vx.shard_owner(31, 24, 8, 3) == (3 << 28, 4 << 28, 3 << 21, 4 << 21)
    with pytest.raises(vx.VxError):
        vx.shard_owner(31, 24, 3, 0)                         # world must be a power of two


# ------------------------------------------------------------------ the ranks as separate processes
# Two processes on the ONE GPU of this box, each with its own plot and workspace; the workspaces are mapped
# into each other with CUDA IPC (vx_ipc_export / vx_ipc_open), the barriers are torch.distributed's (gloo:
# NCCL does not take two ranks on one device).  This is the multi-process path of a multi-GPU node
# (paper_2606_14007_b200.ShardedPlot) with the two "GPUs" being one; the kernels never wait on one another.
def _ipc_worker(rank, world, port, K, B, seed, out):
    import os
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sys.path.insert(0, root)
    sys.path.insert(0, os.path.join(root, "tests"))
    import torch
    import torch.distributed as dist
    import paper_2606_14007_b200 as vxm
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        torch.cuda.set_device(0)
        key = vx_inputs.key_from_seed(seed)
        sp = vxm.ShardedPlot(K, key, rank, world, "cuda:0", bucket_bits=B)
        for _ in range(2):                                   # twice: the second build reuses everything
            sp.build_table1()
            sp.plot.sort_match_table2()
        off1, raw1 = sp.plot.read_tables(1)
        off2, raw2 = sp.plot.read_tables(2)
        st = sp.plot.get_stats()
        b0, b1 = sp.plot.pass_buckets()
        sp.close()
        out.put((rank, b0, b1, off1, raw1, off2, raw2, st))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
@pytest.mark.parametrize("K,B,seed", [(18, 12, 9), (22, 24, 22)])
def test_sharded_build_two_processes_cuda_ipc(vx, K, B, seed):
    import socket
    import torch.multiprocessing as mp
    world = 2
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_ipc_worker, args=(r, world, port, K, B, seed, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted([out.get(timeout=240) for _ in range(world)], key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    key = vx_inputs.key_from_seed(seed)
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_tables(K, key, B)
    t1 = t2 = 0
    for rank, b0, b1, off1, raw1, off2, raw2, st in res:
        assert (b0, b1) == (rank << (B - 1), (rank + 1) << (B - 1))
        lo, hi = int(o_off[b0]), int(o_off[b1])
        assert np.array_equal(off1, o_off[b0:b1 + 1] - o_off[b0])
        assert np.array_equal(raw1, oracle.serialize_t1(4, o_non[lo:hi], o_has[lo:hi]))
        l2, h2 = int(o_t2o[b0]), int(o_t2o[b1])
        assert np.array_equal(off2, o_t2o[b0:b1 + 1] - o_t2o[b0])
        g1, g2 = canon_t2(off2, *decode_t2(raw2, 4))
        assert np.array_equal(g1, o_n1[l2:h2]) and np.array_equal(g2, o_n2[l2:h2])
        t1 += st["t1_records"]
        t2 += st["t2_records"]
    assert t1 == 1 << K and t2 == len(o_n1)
