"""GPU parity: the CUDA path (through the C ABI, via the ctypes binding) against the CPU oracle,
element by element on the same seeded inputs.  Bit-exact: everything here is integer work.

Tolerance: none (north_star: "GPU results must be bit-exact against the oracle, comparing bucket
contents after canonical ordering").
"""
import numpy as np
import pytest

import oracle
import vx_inputs
from vx_testlib import bucket_ids, canon_t1, canon_t2, decode_t1, decode_t2, oracle_tables

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def vx():
    import paper_2606_14007_b200 as m
    m.load_library()
    return m


def u64(t):
    return t.cpu().numpy().view(np.uint64)


# ------------------------------------------------------------------ hash kernel alone (a2-a4)
@pytest.mark.parametrize("K,seed", [(20, 1), (27, 27), (31, 31), (32, 5), (33, 33)])
def test_hash_range_vs_oracle(vx, K, seed):
    key = vx_inputs.key_from_seed(seed)
    N = 1 << K
    nsize = oracle.nonce_size(K)                 # 5-byte nonces from K = 33 (reading A1)
    for begin, count in ((0, 70001), (N - 4099, 4099), (N // 2 - 17, 1025), (min(N, 1 << 32) - 600, 1200 if K > 32 else 600)):
        got = u64(vx.hash_range(K, key, begin, count))
        want = oracle.hash_range(key, nsize, begin, count)
        assert np.array_equal(got, want)


def test_hash_range_vs_blake3_library(vx):
    blake3 = pytest.importorskip("blake3")
    key = vx_inputs.key_from_seed(31)
    got = u64(vx.hash_range(31, key, (1 << 31) - 300, 300))
    for i in range(300):
        n = (1 << 31) - 300 + i
        want = int.from_bytes(blake3.blake3(n.to_bytes(4, "little"), key=key).digest(8), "big")
        assert int(got[i]) == want


def test_hash_worked_values(vx):
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "blake3_worked_values.txt")
    for ln in open(path):
        if ln.startswith("#") or not ln.strip():
            continue
        K, seed, n, hx = ln.split()
        got = u64(vx.hash_range(int(K), vx_inputs.key_from_seed(int(seed)), int(n), 1))
        assert f"{int(got[0]):016x}" == hx


# ------------------------------------------------------------------ full tables, small K
def run_plot(vx, K, key, B, force_exact=False, flags=0, subkey_bits=None, counters=None, s2_kernel=None):
    plot = vx.Plot(K, key, B, flags=flags)
    if s2_kernel is not None:
        plot.set_option(vx.VX_OPT_STAGE2_KERNEL, s2_kernel)
    if force_exact:
        plot.set_option(vx.VX_OPT_FORCE_EXACT_RANK, 1)
    if subkey_bits is not None:
        plot.set_option(vx.VX_OPT_SUBKEY_BITS, subkey_bits)
    plot.build_table1()
    # Table 1 straight after stage 1: bucket order unspecified (A9) -> canonicalise
    off_b, raw_b = plot.read_tables(1)
    plot.sort_match_table2()
    off1, raw1 = plot.read_tables(1)
    off2, raw2 = plot.read_tables(2)
    stats = plot.get_stats()
    if counters is not None:
        counters.update(plot.get_counters())
    nsize = plot.nonce_size
    plot.free()
    return (off_b, raw_b), (off1, raw1), (off2, raw2), stats, nsize


FULL_CASES = [
    # (K, B, seed): tiny brute-force geometries, one partition, ragged sizes, several partitions
    (4, 2, 3), (8, 4, 1), (10, 6, 2), (12, 8, 1), (12, 12, 7), (10, 24, 8),
    (13, 8, 4), (14, 9, 5), (16, 12, 1), (16, 7, 6), (18, 12, 9), (18, 24, 3), (20, 24, 1),
    (21, 12, 2), (22, 24, 22),
]


@pytest.mark.parametrize("K,B,seed", FULL_CASES + [(13, 4, 11), (15, 8, 12), (17, 8, 13), (19, 10, 14), (20, 12, 15), (23, 20, 16)])
def test_tables_bit_exact_vs_oracle(vx, K, B, seed):
    key = vx_inputs.key_from_seed(seed)
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_tables(K, key, B)
    (off_b, raw_b), (off1, raw1), (off2, raw2), stats, nsize = run_plot(vx, K, key, B)

    # Table 1 after build only
    assert np.array_equal(off_b, o_off)
    nb, hb = canon_t1(off_b, *decode_t1(raw_b, nsize))
    assert np.array_equal(nb, o_non) and np.array_equal(hb, o_has)

    # Table 1 after sort+match: sorted in place, byte-exact with the oracle's serialisation
    assert np.array_equal(off1, o_off)
    assert np.array_equal(raw1, oracle.serialize_t1(nsize, o_non, o_has))

    # Table 2: offsets exact; bucket contents equal after canonical (n1, n2) ordering
    assert np.array_equal(off2, o_t2o)
    g1, g2 = canon_t2(off2, *decode_t2(raw2, nsize))
    assert np.array_equal(g1, o_n1) and np.array_equal(g2, o_n2)
    # and as raw bytes: the multiset of 8-byte external records is the oracle's
    assert nsize == 4
    assert np.array_equal(np.sort(raw2.view(np.uint64)),
                          np.sort(oracle.serialize_t2(nsize, o_n1, o_n2).view(np.uint64)))

    sizes = np.diff(o_off)
    assert stats == {"t1_records": 1 << K, "t2_records": len(o_n1), "max_bucket": int(sizes.max())}


@pytest.mark.parametrize("K,B,seed", [(12, 8, 1), (16, 7, 6), (18, 24, 3), (21, 12, 2)])
def test_exact_rerank_path_gives_the_same_tables(vx, K, B, seed):
    """The (H, n) re-ranking path the kernel takes when a tile holds two equal 64-bit hashes
    (reading A10), forced on every tile: the tables must still be the oracle's."""
    key = vx_inputs.key_from_seed(seed)
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_tables(K, key, B)
    _, (off1, raw1), (off2, raw2), stats, nsize = run_plot(vx, K, key, B, force_exact=True)
    assert np.array_equal(off1, o_off)
    assert np.array_equal(raw1, oracle.serialize_t1(nsize, o_non, o_has))
    assert np.array_equal(off2, o_t2o)
    g1, g2 = canon_t2(off2, *decode_t2(raw2, nsize))
    assert np.array_equal(g1, o_n1) and np.array_equal(g2, o_n2)


# The fast ranking pass of the fused kernel compares 32 hash bits below the bin index; two records of
# one bin that tie on them (about once per 2^21 tiles) may come out in the wrong order, which the
# kernel sees as keys that do not strictly increase, and the tile is then redone with exact (H, n)
# ranks -- with the deferred emit of the CTA's previous tile already spent.  VX_OPT_SUBKEY_BITS narrows
# the compared bits so that this redo runs on most tiles; the tables must still be the oracle's.
RETRY_LAYOUTS = [("narrow", 0), ("wide", 1), ("big", 2), ("big+wide", 3)]


@pytest.mark.parametrize("bits", [0, 3])
@pytest.mark.parametrize("layout,flags", RETRY_LAYOUTS)
@pytest.mark.parametrize("K,B,seed", [(12, 8, 1), (13, 8, 4), (16, 12, 1), (16, 7, 6), (18, 12, 9), (18, 24, 3),
                                      (20, 24, 1), (21, 12, 2), (22, 24, 22)])
def test_tie_retry_path_gives_the_same_tables(vx, K, B, seed, layout, flags, bits):
    key = vx_inputs.key_from_seed(seed)
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_tables(K, key, B)
    ctr = {}
    _, (off1, raw1), (off2, raw2), stats, nsize = run_plot(vx, K, key, B, flags=flags, subkey_bits=bits, counters=ctr)
    assert np.array_equal(off1, o_off)
    assert np.array_equal(raw1, oracle.serialize_t1(nsize, o_non, o_has))
    assert np.array_equal(off2, o_t2o)
    g1, g2 = canon_t2(off2, *decode_t2(raw2, nsize))
    assert np.array_equal(g1, o_n1) and np.array_equal(g2, o_n2)
    assert stats["t2_records"] == len(o_n1)
    # dense tiles (several records per bin somewhere in nearly every tile): the redo did run
    tile_log = 13 if flags & 2 else 12
    tiles = 1 << max(K - tile_log, 0)
    if K >= tile_log:
        assert ctr["tile_retries"] >= tiles // 2, ctr
    assert ctr["tile_retries"] <= tiles


def test_default_subkey_bits_take_no_retry(vx):
    K, B = 20, 24
    key = vx_inputs.key_from_seed(1)
    ctr = {}
    run_plot(vx, K, key, B, counters=ctr)
    assert ctr["tile_retries"] == 0


WIDE_CASES = [(4, 2, 3), (10, 6, 2), (12, 8, 1), (12, 12, 7), (13, 8, 4), (16, 12, 1), (16, 7, 6),
              (18, 24, 3), (20, 24, 1), (21, 12, 2), (22, 24, 22)]


@pytest.mark.parametrize("K,B,seed", [(10, 6, 2), (13, 8, 4), (14, 9, 5), (16, 12, 1), (16, 7, 6), (18, 24, 3),
                                      (20, 24, 1), (21, 12, 2), (22, 24, 22)])
@pytest.mark.parametrize("wide", [False, True])
def test_big_tile_geometry_gives_the_same_tables(vx, K, B, seed, wide):
    """The K >= 32 geometry (2^13-record partitions, one 1024-thread CTA per SM), forced at small K,
    in both record layouts: bit-exact against the oracle."""
    key = vx_inputs.key_from_seed(seed)
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_tables(K, key, B)
    flags = vx.VX_CREATE_BIG_TILES | (vx.VX_CREATE_WIDE_LAYOUT if wide else 0)
    (off_b, raw_b), (off1, raw1), (off2, raw2), stats, nsize = run_plot(vx, K, key, B, flags=flags)
    assert np.array_equal(off_b, o_off)
    nb, hb = canon_t1(off_b, *decode_t1(raw_b, nsize))
    assert np.array_equal(nb, o_non) and np.array_equal(hb, o_has)
    assert np.array_equal(off1, o_off)
    assert np.array_equal(raw1, oracle.serialize_t1(nsize, o_non, o_has))
    assert np.array_equal(off2, o_t2o)
    g1, g2 = canon_t2(off2, *decode_t2(raw2, nsize))
    assert np.array_equal(g1, o_n1) and np.array_equal(g2, o_n2)
    assert stats["t2_records"] == len(o_n1)


@pytest.mark.parametrize("force_exact", [False, True])
@pytest.mark.parametrize("K,B,seed", WIDE_CASES)
def test_wide_layout_gives_the_same_tables(vx, K, B, seed, force_exact):
    """The K >= 33 internal layout (10-byte Table-1 records a = (H << pb) | (n >> 12), b = n & 0xfff;
    Table-2 records with a high-bits byte), forced at small K: bit-exact against the oracle."""
    key = vx_inputs.key_from_seed(seed)
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_tables(K, key, B)
    (off_b, raw_b), (off1, raw1), (off2, raw2), stats, nsize = run_plot(
        vx, K, key, B, force_exact=force_exact, flags=vx.VX_CREATE_WIDE_LAYOUT)
    assert nsize == 4
    assert np.array_equal(off_b, o_off)
    nb, hb = canon_t1(off_b, *decode_t1(raw_b, nsize))
    assert np.array_equal(nb, o_non) and np.array_equal(hb, o_has)
    assert np.array_equal(off1, o_off)
    assert np.array_equal(raw1, oracle.serialize_t1(nsize, o_non, o_has))
    assert np.array_equal(off2, o_t2o)
    g1, g2 = canon_t2(off2, *decode_t2(raw2, nsize))
    assert np.array_equal(g1, o_n1) and np.array_equal(g2, o_n2)
    sizes = np.diff(o_off)
    assert stats == {"t1_records": 1 << K, "t2_records": len(o_n1), "max_bucket": int(sizes.max())}


def test_device_tables_layout(vx):
    """vx_device_tables: Table 1 sorted in place in the partition array, as include/vx.h states."""
    import torch
    K, B = 16, 12
    key = vx_inputs.key_from_seed(1)
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_tables(K, key, B)
    plot = vx.Plot(K, key, B)
    plot.build_table1()
    plot.sort_match_table2()
    plot.synchronize()
    t1, t1o, t2, t2o, pbase = plot.device_tables()
    ws = plot.workspace
    base = ws.data_ptr()
    P, cap = 1 << plot.partition_bits, plot.partition_capacity
    part = ws[t1 - base: t1 - base + P * cap * 16].cpu().numpy().view(np.uint32).reshape(P, cap, 4)
    pb = ws[pbase - base: pbase - base + (P + 1) * 8].cpu().numpy().view(np.uint64)
    offs = ws[t1o - base: t1o - base + ((1 << B) + 1) * 8].cpu().numpy().view(np.uint64)
    assert np.array_equal(offs, o_off)
    fb = B - plot.partition_bits
    for b in (0, 1, 77, 2048, 4095):
        q = b >> fb
        lo = int(offs[b] - pb[q]); hi = int(offs[b + 1] - pb[q])
        rec = part[q, lo:hi]
        H = (rec[:, 1].astype(np.uint64) << np.uint64(32)) | rec[:, 0].astype(np.uint64)
        assert np.array_equal(H, o_has[int(o_off[b]):int(o_off[b + 1])])
        assert np.array_equal(rec[:, 2].astype(np.uint64), o_non[int(o_off[b]):int(o_off[b + 1])])
    t2r = ws[t2 - base: t2 - base + len(o_n1) * 8].cpu().numpy()
    assert np.array_equal(np.sort(t2r.view(np.uint64)), np.sort(oracle.serialize_t2(4, o_n1, o_n2).view(np.uint64)))
    plot.free()


def test_ranged_reads(vx):
    K, B, seed = 16, 12, 1
    key = vx_inputs.key_from_seed(seed)
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_tables(K, key, B)
    plot = vx.Plot(K, key, B)
    plot.build_table1()
    plot.sort_match_table2()
    for b0, b1 in ((0, 1), (5, 5), (100, 1000), (4095, 4096), (0, 4096)):
        off, raw = plot.read_tables(1, b0, b1)
        lo, hi = int(o_off[b0]), int(o_off[b1])
        assert np.array_equal(off, o_off[b0:b1 + 1] - o_off[b0])
        assert np.array_equal(raw, oracle.serialize_t1(4, o_non[lo:hi], o_has[lo:hi]))
        off, raw = plot.read_tables(2, b0, b1)
        lo, hi = int(o_t2o[b0]), int(o_t2o[b1])
        assert np.array_equal(off, o_t2o[b0:b1 + 1] - o_t2o[b0])
        g1, g2 = canon_t2(off, *decode_t2(raw, 4))
        assert np.array_equal(g1, o_n1[lo:hi]) and np.array_equal(g2, o_n2[lo:hi])
    with pytest.raises(vx.VxError) as ei:
        plot.read_tables(1, 10, 5)
    assert ei.value.status == -6
    with pytest.raises(vx.VxError):
        plot.read_tables(2, 0, 4097)
    with pytest.raises(vx.VxError) as ei:
        plot.read_tables(1, 0, 4096, records_out=np.empty(8, dtype=np.uint8))
    assert ei.value.status == -6
    plot.free()


def test_state_machine_and_rebuild(vx):
    import torch
    K, B = 14, 9
    key = vx_inputs.key_from_seed(5)
    plot = vx.Plot(K, key, B)
    with pytest.raises(vx.VxError) as ei:
        plot.sort_match_table2()
    assert ei.value.status == -2
    plot.build_table1()
    with pytest.raises(vx.VxError) as ei:
        plot.read_tables(2)
    assert ei.value.status == -2
    plot.sort_match_table2()
    a = plot.read_tables(2)
    # a second full run on a side stream gives the same tables (buffers fully reset)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        plot.build_table1()
        plot.sort_match_table2()
    b = plot.read_tables(2)
    assert np.array_equal(a[0], b[0])
    assert np.array_equal(np.sort(a[1].view(np.uint64)), np.sort(b[1].view(np.uint64)))
    with pytest.raises(vx.VxError) as ei:
        vx.Plot(K, key, B, workspace=torch.empty(1024, dtype=torch.uint8, device="cuda"))
    assert ei.value.status == -3
    plot.free()


def test_two_plots_with_different_keys_coexist(vx):
    K, B = 13, 8
    k1, k2 = vx_inputs.key_from_seed(101), vx_inputs.key_from_seed(202)
    p1, p2 = vx.Plot(K, k1, B), vx.Plot(K, k2, B)
    p1.build_table1(); p2.build_table1()
    p1.sort_match_table2(); p2.sort_match_table2()
    for p, k in ((p1, k1), (p2, k2)):
        o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_tables(K, k, B)
        off1, raw1 = p.read_tables(1)
        assert np.array_equal(off1, o_off) and np.array_equal(raw1, oracle.serialize_t1(4, o_non, o_has))
        off2, raw2 = p.read_tables(2)
        g1, g2 = canon_t2(off2, *decode_t2(raw2, 4))
        assert np.array_equal(off2, o_t2o) and np.array_equal(g1, o_n1) and np.array_equal(g2, o_n2)
    p1.free(); p2.free()


# ------------------------------------------------------------------ K = 24: mean one record per bucket
def test_K24_full_parity(vx):
    K, B = 24, 24
    key = vx_inputs.config_key(K)
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_tables(K, key, B)
    plot = vx.Plot(K, key, B)
    plot.build_table1()
    plot.sort_match_table2()
    off1, raw1 = plot.read_tables(1)
    assert np.array_equal(off1, o_off)
    assert np.array_equal(raw1, oracle.serialize_t1(4, o_non, o_has))
    off2, raw2 = plot.read_tables(2)
    assert np.array_equal(off2, o_t2o)
    g1, g2 = canon_t2(off2, *decode_t2(raw2, 4))
    assert np.array_equal(g1, o_n1) and np.array_equal(g2, o_n2)
    assert plot.get_stats()["t2_records"] == 8386097        # tests/golden/match_counts.txt
    plot.free()


# ------------------------------------------------------------------ overflow is an error, never a silent drop (A8)
@pytest.mark.parametrize("flags", [0, 1])    # narrow; wide (stage 1 in rounds + compaction)
def test_partition_overflow_raises(vx, flags):
    key = vx_inputs.key_from_seed(5)
    plot = vx.Plot(16, key, 12, flags=flags)            # 16 partitions of mean 4096, capacity 4608
    plot.set_option(vx.VX_OPT_PARTITION_CAPACITY_LIMIT, 4000)
    plot.build_table1()
    with pytest.raises(vx.VxError, match="VX_ERR_OVERFLOW"):
        plot.synchronize()
    with pytest.raises(vx.VxError, match="VX_ERR_OVERFLOW"):
        plot.read_tables(1)
    # the same handle recovers once the capacity is back
    plot.set_option(vx.VX_OPT_PARTITION_CAPACITY_LIMIT, plot.partition_capacity)
    plot.build_table1()
    plot.sort_match_table2()
    assert plot.get_stats()["t1_records"] == 1 << 16
    with pytest.raises(vx.VxError, match="VX_ERR_ARG"):
        plot.set_option(vx.VX_OPT_PARTITION_CAPACITY_LIMIT, plot.partition_capacity + 1)
    plot.free()


def test_table2_overflow_raises(vx):
    import torch
    key = vx_inputs.key_from_seed(5)
    plot = vx.Plot(16, key, 12)
    plot.set_option(vx.VX_OPT_TABLE2_CAPACITY_LIMIT, 1000)   # |T2| ~ 2^16
    plot.build_table1()
    plot.sort_match_table2()
    with pytest.raises(vx.VxError, match="VX_ERR_OVERFLOW"):
        plot.synchronize()
    # streamed egress reports it too
    rec = torch.empty(1 << 20, dtype=torch.uint8, pin_memory=True)
    plot.build_table1()
    with pytest.raises(vx.VxError, match="VX_ERR_OVERFLOW"):
        plot.sort_match_table2_to_host(torch.cuda.Stream(), rec.data_ptr(), rec.numel(), slices=4)
    plot.set_option(vx.VX_OPT_TABLE2_CAPACITY_LIMIT, plot.t2_capacity)
    plot.build_table1()
    plot.sort_match_table2()
    assert plot.get_stats()["t2_records"] > 60000
    plot.free()
