"""The torch restatement of the match step that the full-size GPU tests use (tests/vx_testlib.py) is
itself checked here, on the CPU, against the oracle's Table-2 digest mode."""
import numpy as np
import pytest

import oracle
import vx_inputs
from vx_testlib import t_mix64, torch_match_digest_chunk, torch_table2_digest

torch = pytest.importorskip("torch")


def _i64(a):
    return torch.from_numpy(a.view(np.int64).copy())


def test_t_mix64_is_the_oracles_finaliser():
    z = np.array([0, 1, 0x0123456789abcdef, (1 << 64) - 1, 1 << 63], dtype=np.uint64)
    got = t_mix64(_i64(z)).numpy().view(np.uint64)
    assert [int(x) for x in got] == [oracle.mix64(int(x)) for x in z]


@pytest.mark.parametrize("K,B,seed", [(10, 4, 3), (14, 8, 2), (16, 12, 1), (12, 12, 6), (13, 24, 4), (6, 1, 9)])
def test_torch_matcher_equals_oracle_digest(K, B, seed):
    key = vx_inputs.key_from_seed(seed)
    off, non, has = oracle.table1(K, key, B)
    c2, D2 = oracle.table2_digest(K, off, non, has, 1)
    NB = 1 << B
    tc, tD = torch.zeros(NB, dtype=torch.int64), torch.zeros(NB, dtype=torch.int64)
    # in several chunks of whole buckets
    cuts = sorted({0, NB // 3, NB // 2, NB})
    total = 0
    for b0, b1 in zip(cuts[:-1], cuts[1:]):
        lo, hi = int(off[b0]), int(off[b1])
        total += torch_match_digest_chunk(_i64(has[lo:hi]), _i64(non[lo:hi]), K, B, tc, tD)
    assert total == int(c2.sum())
    assert np.array_equal(tc.numpy().view(np.uint64), c2)
    assert np.array_equal(tD.numpy().view(np.uint64), D2)
    # and the digest of a Table 2 given as records
    t2o, n1, n2 = oracle.table2(K, off, non, has, 1)
    rc, rD = torch.zeros(NB, dtype=torch.int64), torch.zeros(NB, dtype=torch.int64)
    half = len(n1) // 2
    o2 = _i64(t2o)
    torch_table2_digest(_i64(n1[:half]), _i64(n2[:half]), o2, 0, rc, rD)
    torch_table2_digest(_i64(n1[half:]), _i64(n2[half:]), o2, half, rc, rD)
    assert np.array_equal(rc.numpy().view(np.uint64), c2)
    assert np.array_equal(rD.numpy().view(np.uint64), D2)
