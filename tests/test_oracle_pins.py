"""Pins of the CPU oracle (oracle/vx_oracle.c) against things OTHER than itself.

Every check here is against (a) the independent `blake3` Python package (official BLAKE3 crate),
(b) values stored under tests/golden/ with their citation, (c) closed forms / invariants, or
(d) an independent numpy brute force.  None of it touches the CUDA path.
"""
import math
import os
import random

import numpy as np
import pytest

import oracle
import vx_inputs

blake3 = pytest.importorskip("blake3")

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    with open(os.path.join(GOLD, name)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


def lib_hash_u64(key: bytes, n: int, nsize: int) -> int:
    """H(n) via the blake3 library: first 8 digest bytes read big-endian (readings A2-A5)."""
    return int.from_bytes(blake3.blake3(n.to_bytes(nsize, "little"), key=key).digest(8), "big")


def lib_hashes(key: bytes, K: int) -> np.ndarray:
    nsize = 4 if K <= 32 else 5
    return np.array([lib_hash_u64(key, n, nsize) for n in range(1 << K)], dtype=np.uint64)


# ------------------------------------------------------------------ Step 1: SplitMix64 / keys
def test_splitmix64_published_sequence():
    want = [int(r[0]) for r in _rows("splitmix64_seed1234567.txt")]
    assert [oracle.splitmix64(1234567, i) for i in range(5)] == want
    assert vx_inputs.splitmix64_stream(1234567, 5) == want


def test_config_keys():
    for seed, hexkey in _rows("config_keys.txt"):
        assert oracle.key_from_seed(int(seed)).hex() == hexkey
        assert vx_inputs.key_from_seed(int(seed)).hex() == hexkey
    assert vx_inputs.config_key(20) == vx_inputs.key_from_seed(1)
    assert vx_inputs.config_key(31) == vx_inputs.key_from_seed(31)
    assert vx_inputs.config_key(25) == vx_inputs.key_from_seed(25)


# ------------------------------------------------------------------ Step 2: BLAKE3 keyed hash
def test_blake3_vs_library_all_lengths():
    rng = random.Random(20260614)
    for trial in range(40):
        key = rng.randbytes(32)
        for ln in range(0, 65):
            msg = rng.randbytes(ln)
            want = blake3.blake3(msg, key=key).digest(64)
            assert oracle.blake3_keyed(key, msg, 64) == want, (trial, ln)


def test_blake3_vs_library_structured_inputs():
    # inputs with a single non-zero byte / word at every position catch a wrong message-word
    # index or permutation entry; all-ones catches dropped carries
    key = bytes(range(32))
    for ln in (1, 4, 5, 8, 33, 64):
        for pos in range(ln):
            for val in (1, 0x80, 0xFF):
                msg = bytearray(ln)
                msg[pos] = val
                assert oracle.blake3_keyed(key, bytes(msg), 64) == blake3.blake3(bytes(msg), key=key).digest(64)
    for key in (bytes(32), b"\xff" * 32):
        for msg in (b"", b"\xff" * 64, b"\x00" * 64):
            assert oracle.blake3_keyed(key, msg, 64) == blake3.blake3(msg, key=key).digest(64)


def test_blake3_rejects_long_input():
    with pytest.raises(ValueError):
        oracle.blake3_keyed(bytes(32), bytes(65), 8)


def test_nonce_size_reading_A1():
    assert [oracle.nonce_size(K) for K in (1, 20, 31, 32, 33, 40)] == [4, 4, 4, 4, 5, 5]


def test_worked_hash_values():
    for K, seed, n, hx in _rows("blake3_worked_values.txt"):
        K, seed, n = int(K), int(seed), int(n)
        key = vx_inputs.key_from_seed(seed)
        nsize = oracle.nonce_size(K)
        assert f"{oracle.hash_nonce(key, n, nsize):016x}" == hx
        assert f"{lib_hash_u64(key, n, nsize):016x}" == hx      # the fixture agrees with the library


def test_hash_range_vs_library_random_nonces():
    rng = random.Random(7)
    for nsize, hi in ((4, 1 << 32), (5, 1 << 40)):
        key = rng.randbytes(32)
        for _ in range(300):
            n = rng.randrange(hi)
            assert oracle.hash_nonce(key, n, nsize) == lib_hash_u64(key, n, nsize)
        h = oracle.hash_range(key, nsize, hi - 50, 50)
        assert [int(x) for x in h] == [lib_hash_u64(key, hi - 50 + i, nsize) for i in range(50)]


# ------------------------------------------------------------------ Step 3: Table 1
def _check_table1_invariants(K, B, off, non, has):
    N = 1 << K
    assert off[0] == 0 and off[-1] == N and len(off) == (1 << B) + 1
    assert np.all(np.diff(off.astype(np.int64)) >= 0)
    assert np.array_equal(np.sort(non), np.arange(N, dtype=np.uint64))      # every nonce once
    bucket_of_slot = np.repeat(np.arange(1 << B, dtype=np.uint64), np.diff(off).astype(np.int64))
    assert np.array_equal(has >> np.uint64(64 - B), bucket_of_slot)          # bucket = hash prefix
    # buckets sorted by (H, n): globally (bucket-major) H is non-decreasing, ties by n
    dH = has[1:] >= has[:-1]
    assert np.all(dH)
    ties = has[1:] == has[:-1]
    assert np.all(non[1:][ties] > non[:-1][ties])


def test_table1_vs_library_small():
    for K, B, seed in ((8, 4, 3), (10, 6, 4), (12, 8, 1), (13, 24, 5)):
        key = vx_inputs.key_from_seed(seed)
        off, non, has = oracle.table1(K, key, B)
        _check_table1_invariants(K, B, off, non, has)
        H = lib_hashes(key, K)                                   # independent hashes
        assert np.array_equal(has, H[non.astype(np.int64)])
        order = np.lexsort((np.arange(1 << K), H))               # global (H, n) order == bucket-major
        assert np.array_equal(non, order.astype(np.uint64))
        cnt = np.bincount((H >> np.uint64(64 - B)).astype(np.int64), minlength=1 << B)
        assert np.array_equal(np.diff(off).astype(np.int64), cnt)


def test_table1_K20_golden_histogram_and_checksums():
    (row,) = [r for r in _rows("bucket_histograms.txt") if r[0] == "20"]
    K, seed, B = int(row[0]), int(row[1]), int(row[2])
    sumH, xorH, sumHn1 = (int(x, 16) for x in row[3:6])
    hist = {int(a): int(b) for a, b in (t.split(":") for t in row[7:])}
    off, non, has = oracle.table1(K, vx_inputs.key_from_seed(seed), B)
    _check_table1_invariants(K, B, off, non, has)
    sizes = np.diff(off).astype(np.int64)
    got = {int(s): int(c) for s, c in enumerate(np.bincount(sizes)) if c}
    assert got == hist
    assert int(np.sum(has, dtype=np.uint64)) == sumH
    assert int(np.bitwise_xor.reduce(has)) == xorH
    assert int(np.sum(has * (non + np.uint64(1)), dtype=np.uint64)) == sumHn1
    # Poisson closed form: #buckets of size s ~ 2^B e^-lam lam^s / s!, lam = 2^(K-B)
    lam = 2.0 ** (K - B)
    for s in range(0, 4):
        exp = (1 << B) * math.exp(-lam) * lam ** s / math.factorial(s)
        assert abs(got.get(s, 0) - exp) < 6 * math.sqrt(exp) + 1


def test_serialize_t1_bytes_are_nonce_le_then_digest_bytes():
    K, B = 10, 6
    key = vx_inputs.key_from_seed(9)
    off, non, has = oracle.table1(K, key, B)
    for nsize in (4, 5):
        raw = oracle.serialize_t1(nsize, non, has).tobytes()
        R = nsize + 8
        for i in (0, 1, 17, len(non) - 1):
            n = int(non[i])
            want = n.to_bytes(nsize, "little") + blake3.blake3(n.to_bytes(4, "little"), key=key).digest(8)
            assert raw[i * R:(i + 1) * R] == want


def test_serialize_t2_bytes():
    n1 = np.array([1, 0x0102030405], dtype=np.uint64)
    n2 = np.array([0xAABBCCDD, 7], dtype=np.uint64)
    assert oracle.serialize_t2(4, n1, n2).tobytes() == bytes.fromhex("01000000ddccbbaa" "0504030207000000")
    assert oracle.serialize_t2(5, n1, n2).tobytes() == bytes.fromhex("0100000000ddccbbaa00" "05040302010700000000")


# ------------------------------------------------------------------ Step 4: Table 2
def numpy_bruteforce_table2(K, B, H):
    """Independent statement of Step 4 on library hashes: all same-bucket pairs with |dH| < T.
    Python ints for the arithmetic (no u64 wrap); returns a sorted list of (bucket, n1, n2)."""
    T = 1 << (64 - K)
    Hl = [int(x) for x in H]
    by_bucket = {}
    for n, h in enumerate(Hl):
        by_bucket.setdefault(h >> (64 - B), []).append(n)
    out = []
    for b, ns in by_bucket.items():
        for i in range(len(ns)):
            for j in range(i + 1, len(ns)):
                r, s = ns[i], ns[j]
                if abs(Hl[r] - Hl[s]) < T:
                    first, second = (r, s) if (Hl[r], r) < (Hl[s], s) else (s, r)
                    out.append((b, first, second))
    return sorted(out)


def oracle_table2_triples(K, off, non, has, mode):
    t2o, n1, n2 = oracle.table2(K, off, non, has, mode)
    b = np.repeat(np.arange(len(t2o) - 1), np.diff(t2o).astype(np.int64))
    return list(zip(b.tolist(), n1.tolist(), n2.tolist())), t2o


@pytest.mark.parametrize("K,B,seed", [(8, 4, 1), (9, 5, 2), (10, 4, 3), (11, 7, 4), (12, 8, 1), (12, 12, 6), (10, 24, 8)])
def test_table2_definition_vs_independent_bruteforce(K, B, seed):
    key = vx_inputs.key_from_seed(seed)
    off, non, has = oracle.table1(K, key, B)
    want = numpy_bruteforce_table2(K, B, lib_hashes(key, K))
    got0, _ = oracle_table2_triples(K, off, non, has, 0)
    got1, _ = oracle_table2_triples(K, off, non, has, 1)
    assert got0 == want          # Step 4 (all pairs) == independent brute force
    assert got1 == want          # Step 4' (sorted scan) == the same


@pytest.mark.parametrize("K,B", [(8, 4), (10, 5), (12, 6), (13, 8), (14, 9), (15, 10), (16, 12), (14, 4)])
def test_sorted_scan_equals_all_pairs(K, B):
    for seed in (11, 12):
        key = vx_inputs.key_from_seed(seed * 100 + K)
        off, non, has = oracle.table1(K, key, B)
        t0, a1, a2 = oracle.table2(K, off, non, has, 0)
        t1, b1, b2 = oracle.table2(K, off, non, has, 1)
        assert np.array_equal(t0, t1) and np.array_equal(a1, b1) and np.array_equal(a2, b2)


def test_all_pairs_accepts_any_input_order_and_ties():
    # hand-made bucket with equal hashes (A10, A15): dH = 0 matches, first = smaller nonce
    K = 60                                     # T = 16
    non = np.array([5, 3, 9, 1], dtype=np.uint64)
    has = np.array([100, 100, 115, 116], dtype=np.uint64)
    n1, n2 = oracle.match_allpairs(K, non, has)
    # pairs: (3,5) dH=0; (3,9),(5,9) dH=15; (3,1)? dH=16 no; (9,1) dH=1 -> first=9 (H=115<116)
    assert list(zip(n1.tolist(), n2.tolist())) == [(3, 5), (3, 9), (5, 9), (9, 1)]
    order = np.lexsort((non, has))
    s1, s2 = oracle.match_sorted(K, non[order], has[order])
    assert list(zip(s1.tolist(), s2.tolist())) == [(3, 5), (3, 9), (5, 9), (9, 1)]


def test_match_threshold_is_strict_and_bucket_local():
    K, B = 4, 1                                # T = 2^60, buckets split at 2^63
    T = 1 << 60
    has = np.array([0, T - 1, T, (1 << 63) - 1, 1 << 63], dtype=np.uint64)
    non = np.arange(5, dtype=np.uint64)
    off = np.array([0, 4, 5], dtype=np.uint64)
    t2o, n1, n2 = oracle.table2(K, off, non, has, 0)
    # (0,1): dH = T-1 match; (0,2): dH = T no; (1,2): dH = 1 match; (3,4): dH = 1 but other bucket
    assert list(zip(n1.tolist(), n2.tolist())) == [(0, 1), (1, 2)]
    assert t2o.tolist() == [0, 2, 2]


def test_match_golden_counts():
    for K, seed, B, m, s1, s2 in _rows("match_counts.txt"):
        K, seed, B = int(K), int(seed), int(B)
        if K > 20:
            continue                            # K=24 takes the plain oracle ~20 s: see the slow test
        off, non, has = oracle.table1(K, vx_inputs.key_from_seed(seed), B)
        t2o, n1, n2 = oracle.table2(K, off, non, has, 1)
        assert (len(n1), int(n1.sum()), int(n2.sum())) == (int(m), int(s1), int(s2))


def test_expected_table2_size_closed_form():
    # E|T2| = 2^K (1 - 2^(B-K-1)) for K >= B ; 2^(2K-1-B) for K < B, sd ~ sqrt(E)
    for K, B in ((16, 12), (16, 8), (14, 14), (12, 16), (18, 10)):
        tot = 0
        for seed in (1, 2, 3, 4):
            off, non, has = oracle.table1(K, vx_inputs.key_from_seed(1000 * K + seed), B)
            tot += int(oracle.table2(K, off, non, has, 1)[0][-1])
        E = 4 * (2.0 ** K * (1 - 2.0 ** (B - K - 1)) if K >= B else 2.0 ** (2 * K - 1 - B))
        assert abs(tot - E) < 6 * math.sqrt(E), (K, B, tot, E)


# ------------------------------------------------------------------ slice / digest modes
def test_slice_and_digest_modes_agree_with_full_table():
    K, B = 14, 8
    key = vx_inputs.key_from_seed(77)
    off, non, has = oracle.table1(K, key, B)
    so, sn, sh = oracle.table1_slice(K, key, B, 37, 101, 1 << K)
    lo, hi = int(off[37]), int(off[101])
    assert np.array_equal(so, off[37:102] - off[37])
    assert np.array_equal(sn, non[lo:hi]) and np.array_equal(sh, has[lo:hi])
    c1, D1 = oracle.table1_digest(K, key, B)
    assert np.array_equal(c1, np.diff(off))
    # the digest, recomputed with numpy from its definition: D1[b] = sum f(H ^ f(n))
    def f(z):
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return z ^ (z >> np.uint64(31))
    with np.errstate(over="ignore"):
        d = f(has ^ f(non))
        want = np.array([np.sum(d[int(off[b]):int(off[b + 1])], dtype=np.uint64) for b in range(1 << B)],
                        dtype=np.uint64)
    assert np.array_equal(D1, want)
    with np.errstate(over="ignore"):
        assert oracle.mix64(0) == 0 and oracle.mix64(1) == int(f(np.array([1], dtype=np.uint64))[0])


def _py_mix64(z: int) -> int:
    """SplitMix64 finaliser in plain Python integers (the digest function f of SURVEY.md 8(c))."""
    M = (1 << 64) - 1
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M
    return z ^ (z >> 31)


@pytest.mark.parametrize("K,B,seed,mode", [(10, 4, 3, 0), (12, 8, 1, 0), (12, 8, 1, 1), (16, 12, 1, 1), (14, 24, 5, 1)])
def test_table2_digest_mode_agrees_with_full_table(K, B, seed, mode):
    """count2[b] / D2[b] = sum f(f(n1) ^ n2) against the same quantities worked out in plain Python
    from the full-table mode (itself pinned by brute force and the golden counts above)."""
    key = vx_inputs.key_from_seed(seed)
    off, non, has = oracle.table1(K, key, B)
    t2o, n1, n2 = oracle.table2(K, off, non, has, mode)
    c2, D2 = oracle.table2_digest(K, off, non, has, mode)
    assert np.array_equal(c2, np.diff(t2o))
    M = (1 << 64) - 1
    want = [0] * (1 << B)
    for b in np.flatnonzero(np.diff(t2o)):
        acc = 0
        for i in range(int(t2o[b]), int(t2o[b + 1])):
            acc = (acc + _py_mix64(_py_mix64(int(n1[i])) ^ int(n2[i]))) & M
        want[int(b)] = acc
    assert [int(x) for x in D2] == want
    # a bucket range gives the same entries
    lo, hi = (1 << B) // 3, (1 << B) // 3 + min(50, (1 << B) // 2)
    c2r, D2r = oracle.table2_digest(K, off, non, has, mode, lo, hi)
    assert np.array_equal(c2r, c2[lo:hi]) and np.array_equal(D2r, D2[lo:hi])
    # swapping the two nonces of a pair changes the digest (it is not symmetric in n1, n2)
    assert _py_mix64(_py_mix64(5) ^ 9) != _py_mix64(_py_mix64(9) ^ 5)


def test_slice_halves_and_parallel_helpers_agree_with_full_table():
    """vxo_filter_range + vxo_table1_from_records (the two halves of the slice mode, used by the
    large-K GPU tests with the hashing shared by several threads) against the full table."""
    K, B = 15, 9
    key = vx_inputs.key_from_seed(91)
    off, non, has = oracle.table1(K, key, B)
    b0, b1 = 100, 333
    lo, hi = int(off[b0]), int(off[b1])
    # records of a nonce range, in nonce order, with their library hashes
    rn, rh = oracle.filter_range(key, 4, B, b0, b1, 1000, 20000, 1 << K)
    H = lib_hashes(key, K)
    sel = [n for n in range(1000, 20000) if b0 <= (int(H[n]) >> (64 - B)) < b1]
    assert [int(x) for x in rn] == sel and [int(x) for x in rh] == [int(H[n]) for n in sel]
    with pytest.raises(RuntimeError):
        oracle.filter_range(key, 4, B, b0, b1, 0, 1 << K, 10)          # capacity too small
    # any input order -> canonical form
    an, ah = oracle.filter_range(key, 4, B, b0, b1, 0, 1 << K, 1 << K)
    perm = np.random.default_rng(5).permutation(len(an))
    so, sn, sh = oracle.table1_from_records(B, b0, b1, an[perm], ah[perm])
    assert np.array_equal(so, off[b0:b1 + 1] - off[b0])
    assert np.array_equal(sn, non[lo:hi]) and np.array_equal(sh, has[lo:hi])
    with pytest.raises(RuntimeError):
        oracle.table1_from_records(B, b0 + 1, b1, an, ah)              # a record outside the range
    for workers in (1, 3):
        po, pn, ph = oracle.table1_slice_parallel(K, key, B, b0, b1, workers)
        assert np.array_equal(po, so) and np.array_equal(pn, sn) and np.array_equal(ph, sh)
        assert np.array_equal(oracle.hash_range_parallel(key, 4, 77, 5000, workers), H[77:5077])
    # the whole table through the halves
    fo, fn, fh = oracle.table1_from_records(B, 0, 1 << B, np.arange(1 << K, dtype=np.uint64), H)
    assert np.array_equal(fo, off) and np.array_equal(fn, non) and np.array_equal(fh, has)


# ------------------------------------------------------------------ Step 6: re-keyed Table 2 (A19-A21)
def lib_pair_hash(key: bytes, n1: int, n2: int, nsize: int) -> int:
    """A19 with the independent `blake3` package: keyed hash of nonce1 LE || nonce2 LE, first 8 bytes BE."""
    blake3 = pytest.importorskip("blake3")
    msg = int(n1).to_bytes(nsize, "little") + int(n2).to_bytes(nsize, "little")
    return int.from_bytes(blake3.blake3(msg, key=key).digest(8), "big")


def test_pair_hash_vs_library():
    rng = random.Random(19)
    for seed in (1, 31, 33):
        key = vx_inputs.key_from_seed(seed)
        for nsize in (4, 5):
            top = (1 << (8 * nsize)) - 1
            cases = [(0, 0), (0, 1), (1, 0), (top, top), (top, 0), (0x01020304, 0x05060708)]
            cases += [(rng.randrange(top + 1), rng.randrange(top + 1)) for _ in range(200)]
            for n1, n2 in cases:
                assert oracle.hash_pair(key, n1, n2, nsize) == lib_pair_hash(key, n1, n2, nsize)
    # not symmetric, and not the hash of either nonce alone
    key = vx_inputs.key_from_seed(1)
    assert oracle.hash_pair(key, 5, 9, 4) != oracle.hash_pair(key, 9, 5, 4)
    assert oracle.hash_pair(key, 5, 0, 4) != oracle.hash_nonce(key, 5, 4)


@pytest.mark.parametrize("K,B,seed", [(10, 4, 3), (12, 8, 1), (14, 24, 5), (16, 12, 1)])
def test_rekeyed_table2_vs_library_and_lexsort(K, B, seed):
    """A20 against an independent construction: library pair hashes + numpy lexsort."""
    key = vx_inputs.key_from_seed(seed)
    off, non, has = oracle.table1(K, key, B)
    t2o, n1, n2 = oracle.table2(K, off, non, has, 1)
    ro, r1, r2, rh = oracle.table2_rekey(K, key, B, n1, n2)
    H2 = np.array([lib_pair_hash(key, a, b, 4) for a, b in zip(n1, n2)], dtype=np.uint64)
    order = np.lexsort((n2, n1, H2))                      # H2 major; bucket = H2 prefix, so bucket-major too
    assert np.array_equal(r1, n1[order]) and np.array_equal(r2, n2[order]) and np.array_equal(rh, H2[order])
    want_off = np.concatenate(([0], np.cumsum(np.bincount((H2 >> np.uint64(64 - B)).astype(np.int64),
                                                          minlength=1 << B)))).astype(np.uint64)
    assert np.array_equal(ro, want_off)
    # any input order gives the same table; the pairs are a permutation of Table 2
    perm = np.random.default_rng(seed).permutation(len(n1))
    po, p1, p2, ph = oracle.table2_rekey(K, key, B, n1[perm], n2[perm])
    assert np.array_equal(po, ro) and np.array_equal(p1, r1) and np.array_equal(p2, r2) and np.array_equal(ph, rh)
    a = np.sort((n1 << np.uint64(32)) | n2)
    b = np.sort((r1 << np.uint64(32)) | r2)
    assert np.array_equal(a, b)


def test_rekeyed_bucket_histogram_closed_form():
    """Pair hashes are uniform: bucket loads of the re-keyed table ~ Poisson(|T2| / 2^B)."""
    K, B, seed = 16, 12, 1
    key = vx_inputs.key_from_seed(seed)
    off, non, has = oracle.table1(K, key, B)
    t2o, n1, n2 = oracle.table2(K, off, non, has, 1)
    ro, r1, r2, rh = oracle.table2_rekey(K, key, B, n1, n2)
    sizes = np.diff(ro).astype(np.int64)
    lam = len(n1) / (1 << B)
    hist = np.bincount(sizes)
    for s_ in range(min(len(hist), 30)):
        expect = (1 << B) * math.exp(-lam) * lam ** s_ / math.factorial(s_)
        assert abs(hist[s_] - expect) < 6 * math.sqrt(expect) + 6
    # and the re-keyed buckets are not the source buckets (the pair hash is a fresh key)
    assert not np.array_equal(ro, t2o)


def test_plot_file_bytes_spelled_out():
    key = bytes(range(32))
    offsets = np.array([0, 1, 1, 3], dtype=np.uint64)        # B = 1 would need 3 entries; use B = 1 -> 2^1 + 1 = 3
    offsets = np.array([0, 1, 3], dtype=np.uint64)
    n1 = np.array([0x01020304, 5, 6], dtype=np.uint64)
    n2 = np.array([0x0a0b0c0d, 7, 8], dtype=np.uint64)
    f = oracle.plot_file(12, key, 1, offsets, n1, n2)
    want = (b"VXPLOT\x00\x01" + (12).to_bytes(4, "little") + (1).to_bytes(4, "little") + (4).to_bytes(4, "little")
            + (0).to_bytes(4, "little") + key + (3).to_bytes(8, "little")
            + b"".join(int(o).to_bytes(8, "little") for o in offsets)
            + bytes([4, 3, 2, 1, 0x0d, 0x0c, 0x0b, 0x0a]) + (5).to_bytes(4, "little") + (7).to_bytes(4, "little")
            + (6).to_bytes(4, "little") + (8).to_bytes(4, "little"))
    assert bytes(f) == want
    # 5-byte nonces
    f5 = oracle.plot_file(33, key, 1, offsets, n1, n2)
    assert len(f5) == 64 + 24 + 30 and bytes(f5[16:20]) == (5).to_bytes(4, "little")
    assert bytes(f5[88:98]) == bytes([4, 3, 2, 1, 0, 0x0d, 0x0c, 0x0b, 0x0a, 0])


def test_K24_golden_histogram_and_match_count():
    # the plain oracle needs ~15 s here; this is the largest full-table pin (mean 1 record/bucket)
    (row,) = [r for r in _rows("bucket_histograms.txt") if r[0] == "24"]
    K, seed, B = int(row[0]), int(row[1]), int(row[2])
    sumH, xorH, sumHn1 = (int(x, 16) for x in row[3:6])
    hist = {int(a): int(b) for a, b in (t.split(":") for t in row[7:])}
    off, non, has = oracle.table1(K, vx_inputs.key_from_seed(seed), B)
    sizes = np.diff(off).astype(np.int64)
    assert {int(s): int(c) for s, c in enumerate(np.bincount(sizes)) if c} == hist
    assert int(np.sum(has, dtype=np.uint64)) == sumH
    assert int(np.bitwise_xor.reduce(has)) == xorH
    assert int(np.sum(has * (non + np.uint64(1)), dtype=np.uint64)) == sumHn1
    (m,) = [r for r in _rows("match_counts.txt") if r[0] == "24"]
    t2o, n1, n2 = oracle.table2(K, off, non, has, 1)
    assert (len(n1), int(n1.sum()), int(n2.sum())) == (int(m[3]), int(m[4]), int(m[5]))
