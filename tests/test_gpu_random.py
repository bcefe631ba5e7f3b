"""Seeded random geometries through the whole CUDA path against the oracle: K, bucket bits, key, internal
layout (narrow / wide / big tiles) and pass count drawn per case, tiny and ragged sizes included
(K = 1 ... 19; empty buckets, buckets larger than a tile's bins, single-partition plots).  Table 1 byte for
byte, Table 2 after canonical ordering, the re-keyed Table 2 where it applies.  Integer work: no tolerance."""
import numpy as np
import pytest

import oracle
import vx_inputs
from vx_testlib import bucket_ids, canon_t2, decode_t2, oracle_tables

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def vx():
    import paper_2606_14007_b200 as m
    m.load_library()
    return m


def draw_cases(n, seed):
    rng = np.random.default_rng(seed)
    cases = [(1, 1, 0, 0), (2, 1, 0, 0), (2, 2, 1, 0), (3, 2, 0, 0), (3, 3, 3, 0), (5, 1, 2, 0), (9, 1, 1, 0), (9, 9, 3, 0)]
    while len(cases) < n:
        K = int(rng.integers(4, 20))
        B = int(rng.integers(max(1, K - 9), min(24, K + 5) + 1))
        flags = int(rng.integers(0, 4))
        tile_log = 13 if flags & 2 else 12
        pl = int(rng.integers(0, 3))
        if K - tile_log < pl or B < pl:
            pl = 0
        cases.append((K, B, flags, pl))
    return [(i,) + c for i, c in enumerate(cases)]


@pytest.mark.parametrize("case,K,B,flags,passes_log", draw_cases(160, 20260614))
def test_random_geometry_vs_oracle(vx, case, K, B, flags, passes_log):
    key = vx_inputs.key_from_seed(1000 + case)
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_tables(K, key, B)
    plot = vx.Plot(K, key, B, flags=flags | vx.VX_CREATE_PASSES_LOG(passes_log))
    nsize = plot.nonce_size
    opt = np.random.default_rng(77 + case)
    if opt.integers(0, 3) == 0:
        plot.set_option(vx.VX_OPT_FORCE_EXACT_RANK, 1)            # the exact (H, n) ranking path
    elif opt.integers(0, 2) == 0:
        plot.set_option(vx.VX_OPT_SUBKEY_BITS, int(opt.integers(0, 9)))   # the tie -> redo path
    slices = int(opt.integers(1, 40))
    t1 = t2 = 0
    for s in range(plot.passes):
        if plot.passes > 1:
            plot.select_pass(s)
        b0, b1 = plot.pass_buckets()
        plot.build_table1()
        plot.sort_match_table2()
        off1, raw1 = plot.read_tables(1)
        lo, hi = int(o_off[b0]), int(o_off[b1])
        assert np.array_equal(off1, o_off[b0:b1 + 1] - o_off[b0])
        assert np.array_equal(raw1, oracle.serialize_t1(nsize, o_non[lo:hi], o_has[lo:hi]))
        off2, raw2 = plot.read_tables(2)
        l2, h2 = int(o_t2o[b0]), int(o_t2o[b1])
        assert np.array_equal(off2, o_t2o[b0:b1 + 1] - o_t2o[b0])
        g1, g2 = canon_t2(off2, *decode_t2(raw2, nsize))
        assert np.array_equal(g1, o_n1[l2:h2]) and np.array_equal(g2, o_n2[l2:h2])
        st = plot.get_stats()
        t1 += st["t1_records"]
        t2 += st["t2_records"]
        # the same slice again through the streamed egress, a random number of stage-2 launches
        import torch
        rec = torch.zeros(raw2.nbytes + 64, dtype=torch.uint8, pin_memory=True)
        off = torch.full((b1 - b0 + 1,), -1, dtype=torch.int64, pin_memory=True)
        plot.build_table1()
        n = plot.sort_match_table2_to_host(torch.cuda.Stream(), rec.data_ptr(), rec.numel(), off.data_ptr(), slices=slices)
        assert n == raw2.nbytes and np.array_equal(off.numpy().view(np.uint64), off2)
        e1, e2 = canon_t2(off2, *decode_t2(rec.numpy()[:n], nsize))
        assert np.array_equal(e1, g1) and np.array_equal(e2, g2)
    assert t1 == 1 << K and t2 == len(o_n1)
    if plot.passes == 1:
        plot.rekey_table2()
        r_off, r_n1, r_n2, r_h2 = oracle.table2_rekey(K, key, B, o_n1, o_n2)
        off3, raw3 = plot.read_tables(vx.VX_TABLE2_REKEYED)
        assert np.array_equal(off3, r_off)
        g1, g2 = decode_t2(raw3, nsize)
        h = np.array([oracle.hash_pair(key, int(a), int(b), nsize) for a, b in zip(g1, g2)], dtype=np.uint64)
        order = np.lexsort((g2, g1, h, bucket_ids(off3)))
        assert np.array_equal(g1[order], r_n1) and np.array_equal(g2[order], r_n2) and np.array_equal(h[order], r_h2)
        ids = bucket_ids(off3)
        same = ids[1:] == ids[:-1]
        assert bool(np.all(h[1:][same] >= h[:-1][same])), "re-keyed buckets are not in H2 order"
    plot.free()
