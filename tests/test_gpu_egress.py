"""GPU parity of the Table-2 egress pipeline (include/vx.h
vx_sort_match_table2_to_host / _to_file): stage 2 run as partition-range slices with Table 2
streamed to the host must give exactly the tables of the one-launch path, i.e. the oracle's.
Bit-exact (integer work); Table-2 buckets are compared after canonical (n1, n2) ordering (A13)."""
import os

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


def pinned(nbytes):
    import torch
    return torch.empty(max(nbytes, 1), dtype=torch.uint8, pin_memory=True)


CASES = [(4, 2, 3, 1), (12, 8, 1, 4), (14, 9, 5, 3), (16, 12, 1, 16), (18, 24, 3, 7), (20, 24, 1, 256),
         (21, 12, 2, 5), (22, 24, 22, 16)]


@pytest.mark.parametrize("K,B,seed,slices", CASES)
@pytest.mark.parametrize("flags", [0, 1, 2])   # narrow, VX_CREATE_WIDE_LAYOUT, VX_CREATE_BIG_TILES
def test_streamed_table2_to_host_is_the_oracles(vx, K, B, seed, slices, flags):
    import torch
    key = vx_inputs.key_from_seed(seed)
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_tables(K, key, B)
    plot = vx.Plot(K, key, B, flags=flags)
    copy = torch.cuda.Stream()
    rec = pinned(8 * len(o_n1) + 64)
    off = torch.empty((1 << B) + 1, dtype=torch.int64, pin_memory=True)
    rec.fill_(0xEE); off.fill_(-1)
    plot.build_table1()
    got = plot.sort_match_table2_to_host(copy, rec.data_ptr(), rec.numel(), off.data_ptr(), slices=slices)
    assert got == 8 * len(o_n1)
    off2 = off.numpy().view(np.uint64)
    assert np.array_equal(off2, o_t2o)
    raw2 = rec.numpy()[:got]
    g1, g2 = canon_t2(off2, *decode_t2(raw2, 4))
    assert np.array_equal(g1, o_n1) and np.array_equal(g2, o_n2)
    assert np.all(rec.numpy()[got:] == 0xEE)                       # nothing written past the end
    # the resident tables are the ones the one-launch path leaves: Table 1 sorted in place, stats
    off1, raw1 = plot.read_tables(1)
    assert np.array_equal(off1, o_off)
    assert np.array_equal(raw1, oracle.serialize_t1(4, o_non, o_has))
    offr, rawr = plot.read_tables(2)
    assert np.array_equal(offr, o_t2o) and np.array_equal(rawr, raw2)
    assert plot.get_stats() == {"t1_records": 1 << K, "t2_records": len(o_n1),
                                "max_bucket": int(np.diff(o_off).max())}
    plot.free()


def test_streamed_table2_to_host_capacity_and_argument_errors(vx):
    import torch
    key = vx_inputs.key_from_seed(1)
    plot = vx.Plot(16, key, 12)
    copy = torch.cuda.Stream()
    rec = pinned(1024)
    with pytest.raises(vx.VxError, match="VX_ERR_STATE"):
        plot.sort_match_table2_to_host(copy, rec.data_ptr(), rec.numel())
    plot.build_table1()
    with pytest.raises(vx.VxError, match="VX_ERR_RANGE"):
        plot.sort_match_table2_to_host(copy, rec.data_ptr(), rec.numel(), slices=4)
    with pytest.raises(vx.VxError, match="VX_ERR_ARG"):
        plot.sort_match_table2_to_host(torch.cuda.current_stream(), rec.data_ptr(), rec.numel())
    plot.free()


@pytest.mark.parametrize("K,B,seed,slices,ring_chunks", [(12, 8, 1, 2, 2), (20, 24, 1, 8, 3), (22, 24, 22, 16, 2)])
def test_streamed_table2_to_file(vx, tmp_path, K, B, seed, slices, ring_chunks):
    """records || offsets || trailer, written through a ring of 4 MB chunks smaller than the data
    (K=22: 33 MB of records + 134 MB of offsets through 8 MB)."""
    import torch
    key = vx_inputs.key_from_seed(seed)
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_tables(K, key, B)
    plot = vx.Plot(K, key, B)
    copy = torch.cuda.Stream()
    ring = pinned(ring_chunks << 22)
    path = tmp_path / "t2.bin"
    fd = os.open(path, os.O_WRONLY | os.O_CREAT | os.O_TRUNC, 0o600)
    try:
        plot.build_table1()
        nbytes = plot.sort_match_table2_to_file(copy, fd, ring.data_ptr(), ring.numel(), slices=slices)
    finally:
        os.close(fd)
    plot.free()
    m = len(o_n1)
    assert nbytes == os.path.getsize(path) == 8 * m + 8 * ((1 << B) + 1) + 32
    data = np.fromfile(path, dtype=np.uint8)
    off2 = data[8 * m: 8 * m + 8 * ((1 << B) + 1)].view(np.uint64)
    assert np.array_equal(off2, o_t2o)
    g1, g2 = canon_t2(off2, *decode_t2(data[:8 * m], 4))
    assert np.array_equal(g1, o_n1) and np.array_equal(g2, o_n2)
    tr = data[-32:]
    assert bytes(tr[:8]) == b"VXT2\0\0\0\1"
    assert list(tr[8:24].view(np.uint32)) == [K, B, 4, 0] and int(tr[24:].view(np.uint64)[0]) == m


def test_two_plots_in_flight_from_two_threads(vx):
    """bench.py's e2e.two_plots_in_flight path: two host threads, each with its own plot, workspace,
    streams and pinned buffers, plotting end to end at the same time (shared: the library's mailbox
    pool and the copy engines).  Every plot of both threads must be the oracle's."""
    import threading
    import torch
    cases = [(20, 24, 1), (19, 12, 9)]
    want = [oracle_tables(K, vx_inputs.key_from_seed(seed), B) for K, B, seed in cases]
    errors = []

    def worker(i):
        try:
            K, B, seed = cases[i]
            o_off, o_non, o_has, o_t2o, o_n1, o_n2 = want[i]
            key = vx_inputs.key_from_seed(seed)
            comp, copy = torch.cuda.Stream(), torch.cuda.Stream()
            rec = pinned(8 * len(o_n1) + 64)
            off = torch.empty((1 << B) + 1, dtype=torch.int64, pin_memory=True)
            ws = None
            for rep in range(4):
                plot = vx.Plot(K, key, B, workspace=ws)
                ws = plot.workspace
                rec.fill_(0); off.fill_(-1)
                plot.build_table1(comp)
                got = plot.sort_match_table2_to_host(copy, rec.data_ptr(), rec.numel(), off.data_ptr(),
                                                     slices=5 + rep, stream=comp)
                assert got == 8 * len(o_n1)
                off2 = off.numpy().view(np.uint64)
                assert np.array_equal(off2, o_t2o)
                g1, g2 = canon_t2(off2, *decode_t2(rec.numpy()[:got], 4))
                assert np.array_equal(g1, o_n1) and np.array_equal(g2, o_n2)
                plot.free()
        except BaseException as ex:   # noqa: BLE001 - reported by the main thread
            errors.append(f"thread {i}: {ex!r}")

    threads = [threading.Thread(target=worker, args=(i,)) for i in range(2)]
    for t in threads: t.start()
    for t in threads: t.join()
    assert not errors, errors
