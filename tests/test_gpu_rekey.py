"""Table-2 re-keying and the plot file (readings A19-A21): the CUDA path against the
oracle's Step 6, bit for bit.  The order of pairs with equal H2 inside a bucket is not part of the
contract (A20): both sides are put into (H2, n1, n2) order before comparing, and the CUDA path's own
order is checked to be non-decreasing in H2 (the oracle's pair hash, recomputed record by record)."""
import os
import tempfile

import numpy as np
import pytest

import oracle
import vx_inputs
from vx_testlib import bucket_ids, decode_t2, oracle_tables

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def vx():
    import paper_2606_14007_b200 as m
    m.load_library()
    return m


def canon_rekeyed(off, n1, n2, h2):
    order = np.lexsort((n2, n1, h2, bucket_ids(off)))
    return n1[order], n2[order], h2[order]


@pytest.mark.parametrize("big", [0, 2, 1, 3])      # narrow / big tiles / wide / big + wide (vx.VX_CREATE_* flags)
@pytest.mark.parametrize("K,B,seed", [(10, 6, 2), (12, 8, 1), (14, 9, 5), (16, 12, 1), (16, 7, 6), (18, 24, 3),
                                      (20, 24, 1), (21, 12, 2), (22, 24, 22)])
def test_rekeyed_table2_and_plot_file_vs_oracle(vx, K, B, seed, big):
    import torch
    key = vx_inputs.key_from_seed(seed)
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_tables(K, key, B)
    r_off, r_n1, r_n2, r_h2 = oracle.table2_rekey(K, key, B, o_n1, o_n2)
    plot = vx.Plot(K, key, B, flags=big)
    plot.build_table1()
    with pytest.raises(vx.VxError) as ei:
        plot.rekey_table2()
    assert ei.value.status == -2                                  # before the match step
    plot.sort_match_table2()
    plot.rekey_table2()
    off, raw = plot.read_tables(vx.VX_TABLE2_REKEYED)
    assert np.array_equal(off, r_off), "CSR offsets of the re-keyed table differ from the oracle's"
    g1, g2 = decode_t2(raw, 4)
    # the CUDA path's order: bucket-major, H2 non-decreasing inside every bucket
    h = None
    if len(g1) <= 300000:
        h = np.array([oracle.hash_pair(key, int(a), int(b), 4) for a, b in zip(g1, g2)], dtype=np.uint64)
    if h is not None:
        assert np.array_equal(h >> np.uint64(64 - B), bucket_ids(off).astype(np.uint64))
        same = bucket_ids(off)[1:] == bucket_ids(off)[:-1]
        assert bool(np.all(h[1:][same] >= h[:-1][same]))
        c1, c2, ch = canon_rekeyed(off, g1, g2, h)
        assert np.array_equal(c1, r_n1) and np.array_equal(c2, r_n2) and np.array_equal(ch, r_h2)
    else:
        # large case: no 64-bit H2 tie in the oracle's table => the order is unique => compare directly
        if len(np.unique(r_h2)) == len(r_h2):
            assert np.array_equal(g1, r_n1) and np.array_equal(g2, r_n2)
        else:
            a = np.sort((g1 << np.uint64(32)) | g2)
            b = np.sort((r_n1 << np.uint64(32)) | r_n2)
            assert np.array_equal(a, b)
    # Table 2 itself is still there; Table 1 is gone; the stats still count both
    off2, raw2 = plot.read_tables(2)
    assert np.array_equal(off2, o_t2o)
    with pytest.raises(vx.VxError) as ei:
        plot.read_tables(1)
    assert ei.value.status == -2
    st = plot.get_stats()
    assert st["t1_records"] == 1 << K and st["t2_records"] == len(o_n1)
    # ranged read
    nbk = 1 << B
    b0, b1 = nbk // 3, nbk // 3 + max(1, nbk // 5)
    offr, rawr = plot.read_tables(vx.VX_TABLE2_REKEYED, b0, b1)
    assert np.array_equal(offr, r_off[b0:b1 + 1] - r_off[b0])
    assert np.array_equal(rawr, raw[8 * int(r_off[b0]): 8 * int(r_off[b1])])
    # the plot file: the oracle's bytes when the order is unique, else header + offsets + same pairs
    ring = torch.empty(2 << 20, dtype=torch.uint8, pin_memory=True)
    with tempfile.TemporaryFile() as f:
        n = plot.write_plot_file(f.fileno(), ring.data_ptr(), ring.numel())
        f.seek(0)
        blob = np.frombuffer(f.read(), dtype=np.uint8)
    want = oracle.plot_file(K, key, B, r_off, r_n1, r_n2)
    assert n == len(blob) == len(want)
    head = 64 + 8 * (nbk + 1)
    assert np.array_equal(blob[:head], want[:head])
    assert np.array_equal(blob[head:], raw)
    if len(np.unique(r_h2)) == len(r_h2):
        assert np.array_equal(blob, want), "plot file bytes differ from the oracle's"
    # a fresh build on the same handle works again
    plot.build_table1()
    plot.sort_match_table2()
    off1, raw1 = plot.read_tables(1)
    assert np.array_equal(raw1, oracle.serialize_t1(4, o_non, o_has))
    plot.free()


def test_rekey_unsupported_layouts_and_errors(vx):
    import torch
    key = vx_inputs.key_from_seed(1)
    for flags in (vx.VX_CREATE_PASSES_LOG(1), vx.VX_CREATE_PASSES_LOG(1) | vx.VX_CREATE_WIDE_LAYOUT):
        p = vx.Plot(16, key, 12, flags=flags)
        p.build_table1()
        p.sort_match_table2()
        with pytest.raises(vx.VxError) as ei:
            p.rekey_table2()
        assert ei.value.status == -7
        p.free()
    p = vx.Plot(14, key, 9)
    ring = torch.empty(2 << 20, dtype=torch.uint8, pin_memory=True)
    p.build_table1()
    p.sort_match_table2()
    with pytest.raises(vx.VxError) as ei:
        p.write_plot_file(1, ring.data_ptr(), ring.numel())        # before the re-keying
    assert ei.value.status == -2
    p.rekey_table2()
    with pytest.raises(vx.VxError):
        p.rekey_table2()                                           # twice
    fd = os.open("/dev/full", os.O_WRONLY) if os.path.exists("/dev/full") else -1
    if fd >= 0:
        try:
            with pytest.raises(vx.VxError) as ei:
                p.write_plot_file(fd, ring.data_ptr(), ring.numel())
            assert ei.value.status == -8
        finally:
            os.close(fd)
    p.free()
