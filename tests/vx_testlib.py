"""Shared helpers of the GPU parity tests: decode external records, canonicalise, compare."""
import numpy as np

import oracle


def decode_t1(raw: np.ndarray, nsize: int):
    """external Table-1 bytes -> (nonces u64, hashes u64)."""
    R = nsize + 8
    rec = raw.reshape(-1, R)
    non = np.zeros(len(rec), dtype=np.uint64)
    for j in range(nsize):
        non |= rec[:, j].astype(np.uint64) << np.uint64(8 * j)
    has = np.zeros(len(rec), dtype=np.uint64)
    for j in range(8):
        has |= rec[:, nsize + j].astype(np.uint64) << np.uint64(8 * (7 - j))
    return non, has


def decode_t2(raw: np.ndarray, nsize: int):
    rec = raw.reshape(-1, 2 * nsize)
    n1 = np.zeros(len(rec), dtype=np.uint64)
    n2 = np.zeros(len(rec), dtype=np.uint64)
    for j in range(nsize):
        n1 |= rec[:, j].astype(np.uint64) << np.uint64(8 * j)
        n2 |= rec[:, nsize + j].astype(np.uint64) << np.uint64(8 * j)
    return n1, n2


def bucket_ids(offsets: np.ndarray) -> np.ndarray:
    return np.repeat(np.arange(len(offsets) - 1, dtype=np.int64), np.diff(offsets).astype(np.int64))


def canon_t1(offsets, non, has):
    """sort every bucket by (H, n) (reading A9/A10)."""
    order = np.lexsort((non, has, bucket_ids(offsets)))
    return non[order], has[order]


def canon_t2(offsets, n1, n2):
    """sort every bucket by (n1, n2) (reading A13)."""
    order = np.lexsort((n2, n1, bucket_ids(offsets)))
    return n1[order], n2[order]


def oracle_tables(K, key, B):
    off, non, has = oracle.table1(K, key, B)
    t2o, n1, n2 = oracle.table2(K, off, non, has, 1)
    return off, non, has, t2o, n1, n2


# ------------------------------------------------------------------ whole-table Table-2 check on the device
# An independent (torch) statement of the match step, used where the oracle cannot hold the tables
# (K >= 29): given a hash-sorted run of Table-1 records it derives, with searchsorted, how many
# successors of every record lie within T (and inside the record's bucket), expands the pairs and
# folds them into the per-bucket digest of SURVEY.md 8(c) "Large-K parity" (iii):
#   count2[b], D2[b] = sum over the pairs of bucket b of f(f(n1) ^ n2) mod 2^64, f = SplitMix64 finaliser.
# tests/test_gpu_large.py compares it (a) with the oracle's vxo_table2_digest at K = 27 and (b) with the
# same digest of the CUDA path's Table 2, bucket by bucket over all 2^24 buckets.
SIGN = -(1 << 63)
_C1 = 0xBF58476D1CE4E5B9 - (1 << 64)
_C2 = 0x94D049BB133111EB - (1 << 64)


def t_lsr(z, s):
    """logical right shift of int64 bit patterns"""
    return (z >> s) & ((1 << (64 - s)) - 1)


def t_mix64(z):
    z = (z ^ t_lsr(z, 30)) * _C1
    z = (z ^ t_lsr(z, 27)) * _C2
    return z ^ t_lsr(z, 31)


def torch_match_digest_chunk(H, non, K, B, count2, D2):
    """H: int64 bit patterns of u64 hashes of consecutive WHOLE buckets, ascending (unsigned); non: their
    nonces (int64).  Adds the chunk's matches into count2 / D2 (int64[2^B])."""
    import torch
    n = H.numel()
    if n == 0:
        return 0
    T = 1 << (64 - K)
    bmask = (1 << (64 - B)) - 1
    room = (~H) & bmask                                   # last hash of the bucket - H, 0 <= room < 2^(64-B)
    reach = torch.clamp(room, max=T - 1) if T - 1 < (1 << 62) else room
    lim = H + reach                                       # no wrap: H + room = H | bmask
    ks = H ^ SIGN                                         # unsigned order through a signed compare
    hi = torch.searchsorted(ks, lim ^ SIGN, right=True)
    idx = torch.arange(n, device=H.device)
    cnt = hi - (idx + 1)
    assert bool((cnt >= 0).all())
    total = int(cnt.sum())
    bucket = t_lsr(H, 64 - B)
    count2.index_add_(0, bucket, cnt)
    if total:
        src = torch.repeat_interleave(idx, cnt)
        start = torch.cumsum(cnt, 0) - cnt
        t = torch.arange(total, device=H.device) - start[src]
        dst = src + 1 + t
        term = t_mix64(t_mix64(non[src]) ^ non[dst])
        D2.index_add_(0, bucket[src], term)
    return total


def torch_table2_digest(n1, n2, offsets2, first, count2, D2):
    """Digest of Table-2 records [first, first + len) given as int64 nonces; offsets2 = int64 CSR offsets."""
    import torch
    r = torch.arange(first, first + n1.numel(), device=n1.device)
    bucket = torch.searchsorted(offsets2, r, right=True) - 1
    D2.index_add_(0, bucket, t_mix64(t_mix64(n1) ^ n2))
    count2.index_add_(0, bucket, torch.ones_like(bucket))
