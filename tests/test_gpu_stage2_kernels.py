"""GPU parity of the two fused stage-2 kernels.

Stage 2 has the classic kernel (phases separated by CTA-wide barriers; the default) and the warp-local
one (`vx_k_sort_match_wl`: from the scatter on every warp finishes its own hash range of the tile alone;
VX_OPT_STAGE2_KERNEL = 1), which applies to the narrow layout when a warp's range is a whole number of
buckets (log2(warps) <= B - partition bits <= 9).  Every geometry below is eligible; each is run through
both kernels, in the fast-rank,
forced-exact and tie-retry modes, against the oracle.  Bit-exact: integer work.
"""
import numpy as np
import pytest

import oracle
import vx_inputs
from test_gpu_parity import run_plot
from vx_testlib import canon_t1, canon_t2, decode_t1, decode_t2, oracle_tables

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def vx():
    import paper_2606_14007_b200 as m
    m.load_library()
    return m


# (K, B, seed, flags): flags 0 -> 2^12-record tiles, 16 warps (needs 4 <= fb <= 9, fb = B - max(K - 12, 0));
# flags 2 (VX_CREATE_BIG_TILES) -> 2^13-record tiles, 32 warps (needs 5 <= fb <= 9, fb = B - max(K - 13, 0))
ELIGIBLE = [
    (8, 4, 1, 0), (10, 6, 2, 0), (12, 8, 1, 0), (13, 8, 4, 0), (14, 9, 5, 0), (15, 8, 12, 0), (16, 12, 1, 0),
    (18, 12, 9, 0), (20, 12, 15, 0), (20, 16, 3, 0), (22, 16, 7, 0), (22, 18, 8, 0),
    (9, 5, 2, 2), (13, 8, 4, 2), (16, 12, 1, 2), (18, 12, 9, 2), (20, 12, 15, 2), (22, 16, 7, 2),
]

_oracle_cache = {}


def oracle_cached(K, B, seed):
    k = (K, B, seed)
    if k not in _oracle_cache:
        _oracle_cache[k] = oracle_tables(K, vx_inputs.key_from_seed(seed), B)
    return _oracle_cache[k]


def check(vx, K, B, seed, flags, **kw):
    key = vx_inputs.key_from_seed(seed)
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_cached(K, B, seed)
    (off_b, raw_b), (off1, raw1), (off2, raw2), stats, nsize = run_plot(vx, K, key, B, flags=flags, **kw)
    assert np.array_equal(off1, o_off)
    assert np.array_equal(raw1, oracle.serialize_t1(nsize, o_non, o_has))
    assert np.array_equal(off2, o_t2o)
    g1, g2 = canon_t2(off2, *decode_t2(raw2, nsize))
    assert np.array_equal(g1, o_n1) and np.array_equal(g2, o_n2)
    sizes = np.diff(o_off)
    assert stats == {"t1_records": 1 << K, "t2_records": len(o_n1), "max_bucket": int(sizes.max())}


@pytest.mark.parametrize("s2_kernel", [0, 1])
@pytest.mark.parametrize("K,B,seed,flags", ELIGIBLE)
def test_both_kernels_fast_rank(vx, K, B, seed, flags, s2_kernel):
    ctr = {}
    check(vx, K, B, seed, flags, s2_kernel=s2_kernel, counters=ctr)
    assert ctr["tile_retries"] <= 1 << max(K - 12, 0)


@pytest.mark.parametrize("s2_kernel", [0, 1])
@pytest.mark.parametrize("K,B,seed,flags", ELIGIBLE)
def test_both_kernels_forced_exact(vx, K, B, seed, flags, s2_kernel):
    check(vx, K, B, seed, flags, s2_kernel=s2_kernel, force_exact=True)


@pytest.mark.parametrize("bits", [0, 3])
@pytest.mark.parametrize("s2_kernel", [0, 1])
@pytest.mark.parametrize("K,B,seed,flags", ELIGIBLE)
def test_both_kernels_tie_retry(vx, K, B, seed, flags, s2_kernel, bits):
    """Narrowed ranking keys: records of a bin tie, come out in the wrong order and the tile is redone with
    exact ranks (in the warp-local kernel: after every warp has written its range back)."""
    ctr = {}
    check(vx, K, B, seed, flags, s2_kernel=s2_kernel, subkey_bits=bits, counters=ctr)
    tile_log = 13 if flags & 2 else 12
    tiles = 1 << max(K - tile_log, 0)
    if K >= tile_log:
        assert ctr["tile_retries"] >= tiles // 2, ctr
    assert ctr["tile_retries"] <= tiles


def test_unknown_kernel_choice_is_rejected(vx):
    plot = vx.Plot(12, vx_inputs.key_from_seed(1), 8)
    with pytest.raises(Exception):
        plot.set_option(vx.VX_OPT_STAGE2_KERNEL, 2)
    plot.free()


@pytest.mark.parametrize("K,B,seed,flags,slices", [(14, 9, 5, 0, 3), (16, 12, 1, 0, 16), (20, 16, 3, 0, 7),
                                                   (22, 16, 7, 0, 64), (18, 12, 9, 2, 5), (22, 16, 7, 2, 16)])
def test_warp_local_kernel_in_slices_streamed_to_host(vx, K, B, seed, flags, slices):
    """The warp-local kernel launched as partition-range slices (vx_sort_match_table2_to_host: the look-back
    state carries over from slice to slice, the last tile of a slice reports the running |Table 2|)."""
    import torch
    key = vx_inputs.key_from_seed(seed)
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_cached(K, B, seed)
    plot = vx.Plot(K, key, B, flags=flags)
    plot.set_option(vx.VX_OPT_STAGE2_KERNEL, 1)
    copy = torch.cuda.Stream()
    rec = torch.empty(8 * len(o_n1) + 64, dtype=torch.uint8, pin_memory=True)
    off = torch.empty((1 << B) + 1, dtype=torch.int64, pin_memory=True)
    rec.fill_(0xEE); off.fill_(-1)
    plot.build_table1()
    got = plot.sort_match_table2_to_host(copy, rec.data_ptr(), rec.numel(), off.data_ptr(), slices=slices)
    assert got == 8 * len(o_n1)
    off2 = off.numpy().view(np.uint64)
    assert np.array_equal(off2, o_t2o)
    g1, g2 = canon_t2(off2, *decode_t2(rec.numpy()[:got], 4))
    assert np.array_equal(g1, o_n1) and np.array_equal(g2, o_n2)
    assert np.all(rec.numpy()[got:] == 0xEE)
    off1, raw1 = plot.read_tables(1)
    assert np.array_equal(off1, o_off)
    assert np.array_equal(raw1, oracle.serialize_t1(4, o_non, o_has))
    plot.free()


@pytest.mark.parametrize("K,B,seed,passes_log", [(16, 12, 1, 1), (20, 16, 3, 2), (22, 18, 8, 1)])
def test_warp_local_kernel_in_bucket_range_passes(vx, K, B, seed, passes_log):
    """... and on the passes of a plot made in 2^l bucket-range passes (tile and bucket indices relative to the pass)."""
    key = vx_inputs.key_from_seed(seed)
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_cached(K, B, seed)
    plot = vx.Plot(K, key, B, flags=vx.VX_CREATE_PASSES_LOG(passes_log))
    plot.set_option(vx.VX_OPT_STAGE2_KERNEL, 1)
    nb = (1 << B) >> passes_log
    for s in range(1 << passes_log):
        plot.select_pass(s)
        plot.build_table1()
        plot.sort_match_table2()
        off1, raw1 = plot.read_tables(1)
        off2, raw2 = plot.read_tables(2)
        lo, hi = s * nb, (s + 1) * nb
        assert np.array_equal(off1, o_off[lo:hi + 1] - o_off[lo])
        a, b = int(o_off[lo]), int(o_off[hi])
        assert np.array_equal(raw1, oracle.serialize_t1(4, o_non[a:b], o_has[a:b]))
        assert np.array_equal(off2, o_t2o[lo:hi + 1] - o_t2o[lo])
        g1, g2 = canon_t2(off2, *decode_t2(raw2, 4))
        a2, b2 = int(o_t2o[lo]), int(o_t2o[hi])
        assert np.array_equal(g1, o_n1[a2:b2]) and np.array_equal(g2, o_n2[a2:b2])
    plot.free()
