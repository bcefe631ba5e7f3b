"""Bucket-range passes ("chunked VRAM tiling"): a plot made in 2^l
hash-prefix slices, each slice hashing all nonces and keeping its own buckets, must give exactly the
one-pass tables.  The pass count is forced (VX_CREATE_PASSES_LOG, the test-only "VRAM budget") so that
the path K >= 34 takes is compared with the oracle, bit for bit, on full small tables, in every
internal layout.  Integer work: no tolerance."""
import numpy as np
import pytest

import oracle
import vx_inputs
from vx_testlib import canon_t1, canon_t2, decode_t1, decode_t2, oracle_tables

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def vx():
    import paper_2606_14007_b200 as m
    m.load_library()
    return m


LAYOUTS = [("narrow", 0), ("wide", 1), ("big", 2), ("big+wide", 3)]
CASES = [(14, 9, 5), (16, 12, 1), (16, 7, 6), (18, 12, 9), (18, 24, 3), (20, 24, 1), (21, 12, 2), (22, 24, 22)]


@pytest.mark.parametrize("passes_log", [1, 2])
@pytest.mark.parametrize("layout,lflags", LAYOUTS)
@pytest.mark.parametrize("K,B,seed", CASES)
def test_every_pass_holds_its_slice_of_the_oracle_tables(vx, K, B, seed, layout, lflags, passes_log):
    tile_log = 13 if lflags & 2 else 12
    if K - tile_log < passes_log:
        pytest.skip("fewer partitions than passes")
    key = vx_inputs.key_from_seed(seed)
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_tables(K, key, B)
    plot = vx.Plot(K, key, B, flags=lflags | vx.VX_CREATE_PASSES_LOG(passes_log))
    assert plot.passes == 1 << passes_log
    nsize = plot.nonce_size
    NB = 1 << B
    t1_total = t2_total = 0
    for s in range(plot.passes):
        plot.select_pass(s)
        b0, b1 = plot.pass_buckets()
        assert (b0, b1) == (s * NB // plot.passes, (s + 1) * NB // plot.passes)
        plot.build_table1()
        # Table 1 after stage 1 alone (in-bucket order unspecified, A9)
        off_b, raw_b = plot.read_tables(1)
        lo, hi = int(o_off[b0]), int(o_off[b1])
        assert np.array_equal(off_b, o_off[b0:b1 + 1] - o_off[b0])
        nb, hb = canon_t1(off_b, *decode_t1(raw_b, nsize))
        assert np.array_equal(nb, o_non[lo:hi]) and np.array_equal(hb, o_has[lo:hi])
        plot.sort_match_table2()
        off1, raw1 = plot.read_tables(1)
        assert np.array_equal(off1, o_off[b0:b1 + 1] - o_off[b0])
        assert np.array_equal(raw1, oracle.serialize_t1(nsize, o_non[lo:hi], o_has[lo:hi]))
        off2, raw2 = plot.read_tables(2)
        l2, h2 = int(o_t2o[b0]), int(o_t2o[b1])
        assert np.array_equal(off2, o_t2o[b0:b1 + 1] - o_t2o[b0])
        g1, g2 = canon_t2(off2, *decode_t2(raw2, nsize))
        assert np.array_equal(g1, o_n1[l2:h2]) and np.array_equal(g2, o_n2[l2:h2])
        # a sub-range, and a range outside the pass
        mid = (b0 + b1) // 2
        offm, rawm = plot.read_tables(1, mid, b1)
        assert np.array_equal(rawm, oracle.serialize_t1(nsize, o_non[int(o_off[mid]):hi], o_has[int(o_off[mid]):hi]))
        other = (b1, min(NB, b1 + 1)) if s + 1 < plot.passes else (0, 1)
        with pytest.raises(vx.VxError) as ei:
            plot.read_tables(1, *other)
        assert ei.value.status == -6
        st = plot.get_stats()
        assert st["t1_records"] == hi - lo and st["t2_records"] == h2 - l2
        t1_total += st["t1_records"]
        t2_total += st["t2_records"]
    assert t1_total == 1 << K and t2_total == len(o_n1)      # every nonce in exactly one pass
    plot.free()


@pytest.mark.parametrize("passes_log,slices", [(1, 1), (2, 3), (3, 16)])
@pytest.mark.parametrize("layout,lflags", LAYOUTS)
@pytest.mark.parametrize("K,B,seed", [(16, 12, 1), (18, 24, 3), (20, 24, 1), (22, 24, 22)])
def test_all_passes_to_host_is_the_one_pass_table2(vx, K, B, seed, layout, lflags, passes_log, slices):
    import torch
    tile_log = 13 if lflags & 2 else 12
    if K - tile_log < passes_log:
        pytest.skip("fewer partitions than passes")
    key = vx_inputs.key_from_seed(seed)
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_tables(K, key, B)
    plot = vx.Plot(K, key, B, flags=lflags | vx.VX_CREATE_PASSES_LOG(passes_log))
    cap = 8 * len(o_n1) + 4096
    rec = torch.zeros(cap, dtype=torch.uint8, pin_memory=True)
    off = torch.full(((1 << B) + 1,), -1, dtype=torch.int64, pin_memory=True)
    nbytes, t1 = plot.all_passes_to_host(torch.cuda.Stream(), rec.data_ptr(), cap, off.data_ptr(), slices=slices)
    assert t1 == 1 << K
    assert nbytes == 8 * len(o_n1)
    got_off = off.numpy().view(np.uint64)
    assert np.array_equal(got_off, o_t2o), "global CSR offsets differ from the oracle's"
    g1, g2 = canon_t2(got_off, *decode_t2(rec.numpy()[:nbytes], 4))
    assert np.array_equal(g1, o_n1) and np.array_equal(g2, o_n2)
    # too small a host buffer is an error, not a truncation
    with pytest.raises(vx.VxError) as ei:
        plot.all_passes_to_host(torch.cuda.Stream(), rec.data_ptr(), 8 * (len(o_n1) // 2), off.data_ptr(), slices=slices)
    assert ei.value.status == -6
    plot.free()


def test_pass_arguments(vx):
    key = vx_inputs.key_from_seed(1)
    with pytest.raises(vx.VxError):
        vx.Plot(12, key, 24, flags=vx.VX_CREATE_PASSES_LOG(1))      # one partition cannot be split
    plot = vx.Plot(18, key, 12, flags=vx.VX_CREATE_PASSES_LOG(2))
    with pytest.raises(vx.VxError) as ei:
        plot.select_pass(4)
    assert ei.value.status == -1
    # the file sink writes the selected pass's slice: records, its 2^B / passes + 1 offsets, trailer
    import os
    import tempfile
    import torch
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_tables(18, key, 12)
    ring = torch.empty(16 << 20, dtype=torch.uint8, pin_memory=True)
    plot.select_pass(2)
    b0, b1 = plot.pass_buckets()
    with tempfile.TemporaryFile() as f:
        plot.build_table1()
        n = plot.sort_match_table2_to_file(torch.cuda.Stream(), f.fileno(), ring.data_ptr(), ring.numel(), slices=3)
        f.seek(0)
        blob = np.frombuffer(f.read(), dtype=np.uint8)
    m = int(o_t2o[b1] - o_t2o[b0])
    assert n == len(blob) == 8 * m + 8 * (b1 - b0 + 1) + 32
    offs = blob[8 * m: 8 * m + 8 * (b1 - b0 + 1)].view(np.uint64)
    assert np.array_equal(offs, o_t2o[b0:b1 + 1] - o_t2o[b0])
    g1, g2 = canon_t2(offs, *decode_t2(blob[:8 * m], 4))
    assert np.array_equal(g1, o_n1[int(o_t2o[b0]):int(o_t2o[b1])]) and np.array_equal(g2, o_n2[int(o_t2o[b0]):int(o_t2o[b1])])
    tr = blob[-32:]
    assert bytes(tr[:8]) == b"VXT2\0\0\0\1"
    assert list(tr[8:24].view(np.uint32)) == [18, 12, 4, 2 | (2 << 16)] and int(tr[24:].view(np.uint64)[0]) == m
    plot.free()
