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
