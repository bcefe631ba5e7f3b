"""ctypes binding of the CPU oracle (oracle/vx_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  The product package never imports this module and this
module never imports the product package.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "vx_oracle.c")
_LIB = os.path.join(_HERE, "libvxoracle.so")
_BIN = os.path.join(_HERE, "vx_oracle")

U64 = ctypes.c_uint64
_p64 = ctypes.POINTER(ctypes.c_uint64)
_p8 = ctypes.POINTER(ctypes.c_uint8)
UINT64_MAX = (1 << 64) - 1


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 (no SIMD intrinsics, single thread). Returns the .so path."""
    stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
    if force or stale:
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-Wall", "-Wextra", "-fPIC", "-shared",
                               "-o", _LIB, _SRC])
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-Wall", "-Wextra", "-DVXO_MAIN",
                               "-o", _BIN, _SRC])
    return _LIB


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        L.vxo_splitmix64.restype = U64
        L.vxo_splitmix64.argtypes = [U64, ctypes.c_int]
        L.vxo_key_from_seed.restype = None
        L.vxo_key_from_seed.argtypes = [U64, ctypes.c_char_p]
        L.vxo_blake3_keyed.restype = ctypes.c_int
        L.vxo_blake3_keyed.argtypes = [ctypes.c_char_p, ctypes.c_char_p, ctypes.c_size_t,
                                       ctypes.c_char_p, ctypes.c_size_t]
        L.vxo_nonce_size.restype = ctypes.c_int
        L.vxo_nonce_size.argtypes = [ctypes.c_int]
        L.vxo_hash_nonce.restype = U64
        L.vxo_hash_nonce.argtypes = [ctypes.c_char_p, U64, ctypes.c_int]
        L.vxo_hash_range.restype = None
        L.vxo_hash_range.argtypes = [ctypes.c_char_p, ctypes.c_int, U64, U64, _p64]
        L.vxo_table1.restype = ctypes.c_int
        L.vxo_table1.argtypes = [ctypes.c_int, ctypes.c_char_p, ctypes.c_int, _p64, _p64, _p64]
        for f in (L.vxo_match_allpairs, L.vxo_match_sorted):
            f.restype = U64
            f.argtypes = [ctypes.c_int, U64, _p64, _p64, _p64, _p64, U64]
        L.vxo_table2.restype = U64
        L.vxo_table2.argtypes = [ctypes.c_int, ctypes.c_int, U64, U64, _p64, _p64, _p64,
                                 _p64, _p64, _p64, U64]
        L.vxo_serialize_t1.restype = None
        L.vxo_serialize_t1.argtypes = [ctypes.c_int, U64, _p64, _p64, _p8]
        L.vxo_serialize_t2.restype = None
        L.vxo_serialize_t2.argtypes = [ctypes.c_int, U64, _p64, _p64, _p8]
        L.vxo_mix64.restype = U64
        L.vxo_mix64.argtypes = [U64]
        L.vxo_table1_slice.restype = U64
        L.vxo_table1_slice.argtypes = [ctypes.c_int, ctypes.c_char_p, ctypes.c_int, U64, U64,
                                       _p64, _p64, _p64, U64]
        L.vxo_filter_range.restype = U64
        L.vxo_filter_range.argtypes = [ctypes.c_char_p, ctypes.c_int, ctypes.c_int, U64, U64, U64, U64,
                                       _p64, _p64, U64]
        L.vxo_table1_from_records.restype = ctypes.c_int
        L.vxo_table1_from_records.argtypes = [ctypes.c_int, U64, U64, U64, _p64, _p64, _p64, _p64, _p64]
        L.vxo_table2_digest.restype = U64
        L.vxo_table2_digest.argtypes = [ctypes.c_int, ctypes.c_int, U64, U64, _p64, _p64, _p64, _p64, _p64]
        L.vxo_hash_pair.restype = U64
        L.vxo_hash_pair.argtypes = [ctypes.c_char_p, U64, U64, ctypes.c_int]
        L.vxo_table2_rekey.restype = ctypes.c_int
        L.vxo_table2_rekey.argtypes = [ctypes.c_int, ctypes.c_char_p, ctypes.c_int, U64, _p64, _p64,
                                       _p64, _p64, _p64, _p64]
        L.vxo_plot_file_bytes.restype = U64
        L.vxo_plot_file_bytes.argtypes = [ctypes.c_int, ctypes.c_int, U64]
        L.vxo_plot_file.restype = None
        L.vxo_plot_file.argtypes = [ctypes.c_int, ctypes.c_char_p, ctypes.c_int, U64, _p64, _p64, _p64, _p8]
        L.vxo_table1_digest.restype = ctypes.c_int
        L.vxo_table1_digest.argtypes = [ctypes.c_int, ctypes.c_char_p, ctypes.c_int, _p64, _p64]
        _lib = L
    return _lib


def _ptr(a: np.ndarray):
    assert a.dtype == np.uint64 and a.flags.c_contiguous
    return a.ctypes.data_as(_p64)


def _ptr8(a: np.ndarray):
    assert a.dtype == np.uint8 and a.flags.c_contiguous
    return a.ctypes.data_as(_p8)


def _null():
    return ctypes.cast(None, _p64)


# ------------------------------------------------------------------------------- Step 1
def splitmix64(seed: int, index: int) -> int:
    return int(lib().vxo_splitmix64(seed, index))


def key_from_seed(seed: int) -> bytes:
    buf = ctypes.create_string_buffer(32)
    lib().vxo_key_from_seed(seed, buf)
    return buf.raw


# ------------------------------------------------------------------------------- Step 2
def blake3_keyed(key: bytes, msg: bytes, outlen: int = 32) -> bytes:
    assert len(key) == 32
    out = ctypes.create_string_buffer(max(outlen, 1))
    rc = lib().vxo_blake3_keyed(key, msg, len(msg), out, outlen)
    if rc != 0:
        raise ValueError("vxo_blake3_keyed: message or output longer than 64 bytes")
    return out.raw[:outlen]


def nonce_size(K: int) -> int:
    return int(lib().vxo_nonce_size(K))


def hash_nonce(key: bytes, n: int, nsize: int) -> int:
    return int(lib().vxo_hash_nonce(key, n, nsize))


def hash_range(key: bytes, nsize: int, n_begin: int, count: int) -> np.ndarray:
    out = np.empty(count, dtype=np.uint64)
    lib().vxo_hash_range(key, nsize, n_begin, count, _ptr(out))
    return out


# ------------------------------------------------------------------------------- Step 3
def table1(K: int, key: bytes, bucket_bits: int = 24):
    """Canonical Table 1: (offsets[2^B+1], nonces[2^K], hashes[2^K]) as uint64 arrays."""
    offsets = np.empty((1 << bucket_bits) + 1, dtype=np.uint64)
    nonces = np.empty(1 << K, dtype=np.uint64)
    hashes = np.empty(1 << K, dtype=np.uint64)
    rc = lib().vxo_table1(K, key, bucket_bits, _ptr(offsets), _ptr(nonces), _ptr(hashes))
    if rc != 0:
        raise RuntimeError(f"vxo_table1 failed: {rc}")
    return offsets, nonces, hashes


def table1_slice(K: int, key: bytes, bucket_bits: int, b_begin: int, b_end: int, cap: int):
    offsets = np.empty(b_end - b_begin + 1, dtype=np.uint64)
    nonces = np.empty(cap, dtype=np.uint64)
    hashes = np.empty(cap, dtype=np.uint64)
    kept = lib().vxo_table1_slice(K, key, bucket_bits, b_begin, b_end,
                                  _ptr(offsets), _ptr(nonces), _ptr(hashes), cap)
    if kept == UINT64_MAX:
        raise RuntimeError("vxo_table1_slice: capacity too small or out of memory")
    return offsets, nonces[:kept].copy(), hashes[:kept].copy()


def filter_range(key: bytes, nsize: int, bucket_bits: int, b_begin: int, b_end: int, n_begin: int, n_end: int,
                 cap: int):
    """Records (nonces, hashes) of the nonces [n_begin, n_end) whose bucket lies in [b_begin, b_end)."""
    nonces = np.empty(max(cap, 1), dtype=np.uint64)
    hashes = np.empty(max(cap, 1), dtype=np.uint64)
    kept = lib().vxo_filter_range(key, nsize, bucket_bits, b_begin, b_end, n_begin, n_end,
                                  _ptr(nonces), _ptr(hashes), cap)
    if kept == UINT64_MAX:
        raise RuntimeError("vxo_filter_range: capacity too small")
    return nonces[:kept].copy(), hashes[:kept].copy()


def table1_from_records(bucket_bits: int, b_begin: int, b_end: int, nonces_in, hashes_in):
    """Canonical Table 1 of the bucket range from its records in any order: (offsets, nonces, hashes)."""
    nonces_in = np.ascontiguousarray(nonces_in, dtype=np.uint64)
    hashes_in = np.ascontiguousarray(hashes_in, dtype=np.uint64)
    cnt = len(nonces_in)
    assert len(hashes_in) == cnt
    offsets = np.empty(b_end - b_begin + 1, dtype=np.uint64)
    nonces = np.empty(max(cnt, 1), dtype=np.uint64)
    hashes = np.empty(max(cnt, 1), dtype=np.uint64)
    rc = lib().vxo_table1_from_records(bucket_bits, b_begin, b_end, cnt, _ptr(nonces_in), _ptr(hashes_in),
                                       _ptr(offsets), _ptr(nonces), _ptr(hashes))
    if rc != 0:
        raise RuntimeError(f"vxo_table1_from_records failed: {rc}")
    return offsets, nonces[:cnt], hashes[:cnt]


def table1_slice_parallel(K: int, key: bytes, bucket_bits: int, b_begin: int, b_end: int, workers: int):
    """vxo_table1_slice with the hashing shared by `workers` threads, each running the single-threaded
    vxo_filter_range on its own nonce range (ctypes releases the GIL for the call; the C code keeps no
    global state).  Same result as table1_slice."""
    from concurrent.futures import ThreadPoolExecutor
    N = 1 << K
    nsize = nonce_size(K)
    pieces = max(workers * 4, 1)
    bounds = [N * i // pieces for i in range(pieces + 1)]
    expect = (N >> bucket_bits) * (b_end - b_begin) if K >= bucket_bits else (b_end - b_begin)
    cap = max(1024, (2 * expect) // pieces + 8 * int((expect / pieces) ** 0.5) + 64)
    lib()

    def work(i):
        return filter_range(key, nsize, bucket_bits, b_begin, b_end, bounds[i], bounds[i + 1], cap)

    with ThreadPoolExecutor(max_workers=max(workers, 1)) as ex:
        parts = list(ex.map(work, range(pieces)))
    non = np.concatenate([p[0] for p in parts]) if parts else np.empty(0, dtype=np.uint64)
    has = np.concatenate([p[1] for p in parts]) if parts else np.empty(0, dtype=np.uint64)
    return table1_from_records(bucket_bits, b_begin, b_end, non, has)


def hash_range_parallel(key: bytes, nsize: int, n_begin: int, count: int, workers: int) -> np.ndarray:
    """hash_range with the range split over `workers` threads (each call is the single-threaded C loop)."""
    from concurrent.futures import ThreadPoolExecutor
    out = np.empty(count, dtype=np.uint64)
    pieces = max(workers * 4, 1)
    bounds = [count * i // pieces for i in range(pieces + 1)]
    L = lib()

    def work(i):
        lo, hi = bounds[i], bounds[i + 1]
        if hi > lo:
            L.vxo_hash_range(key, nsize, n_begin + lo, hi - lo, _ptr(out[lo:hi]))

    with ThreadPoolExecutor(max_workers=max(workers, 1)) as ex:
        list(ex.map(work, range(pieces)))
    return out


def table2_digest(K: int, t1_offsets, nonces, hashes, mode: int = 1, b_begin: int = 0, b_end: int | None = None):
    """(count2[nb], D2[nb]) of the bucket range of a canonical Table 1: D2[b] = sum f(f(n1) ^ n2) mod 2^64."""
    if b_end is None:
        b_end = len(t1_offsets) - 1
    nb = b_end - b_begin
    count2 = np.empty(max(nb, 1), dtype=np.uint64)
    D2 = np.empty(max(nb, 1), dtype=np.uint64)
    total = lib().vxo_table2_digest(K, mode, b_begin, b_end, _ptr(t1_offsets), _ptr(nonces), _ptr(hashes),
                                    _ptr(count2), _ptr(D2))
    if total == UINT64_MAX:
        raise MemoryError
    return count2[:nb], D2[:nb]


def table1_digest(K: int, key: bytes, bucket_bits: int = 24):
    count1 = np.empty(1 << bucket_bits, dtype=np.uint64)
    D1 = np.empty(1 << bucket_bits, dtype=np.uint64)
    rc = lib().vxo_table1_digest(K, key, bucket_bits, _ptr(count1), _ptr(D1))
    if rc != 0:
        raise RuntimeError(f"vxo_table1_digest failed: {rc}")
    return count1, D1


# ------------------------------------------------------------------------------- Step 4
def _match(fn, K, nonces, hashes):
    nonces = np.ascontiguousarray(nonces, dtype=np.uint64)
    hashes = np.ascontiguousarray(hashes, dtype=np.uint64)
    cnt = len(nonces)
    m = fn(K, cnt, _ptr(nonces), _ptr(hashes), _null(), _null(), 0)
    if m == UINT64_MAX:
        raise MemoryError
    n1 = np.empty(m, dtype=np.uint64)
    n2 = np.empty(m, dtype=np.uint64)
    if m:
        fn(K, cnt, _ptr(nonces), _ptr(hashes), _ptr(n1), _ptr(n2), m)
    return n1, n2


def match_allpairs(K: int, nonces, hashes):
    """Step 4 (definition) on one bucket given in any order -> canonical (n1, n2) arrays."""
    return _match(lib().vxo_match_allpairs, K, nonces, hashes)


def match_sorted(K: int, nonces, hashes):
    """Step 4' (fast form) on one bucket sorted by (H, n) -> canonical (n1, n2) arrays."""
    return _match(lib().vxo_match_sorted, K, nonces, hashes)


def table2(K: int, t1_offsets, nonces, hashes, mode: int = 1, b_begin: int = 0, b_end: int | None = None):
    """Table 2 of the bucket range: (t2_offsets[nb+1] relative to the range, n1, n2)."""
    if b_end is None:
        b_end = len(t1_offsets) - 1
    nb = b_end - b_begin
    t2_off = np.empty(nb + 1, dtype=np.uint64)
    total = lib().vxo_table2(K, mode, b_begin, b_end, _ptr(t1_offsets), _ptr(nonces), _ptr(hashes),
                             _ptr(t2_off), _null(), _null(), 0)
    if total == UINT64_MAX:
        raise MemoryError
    n1 = np.empty(total, dtype=np.uint64)
    n2 = np.empty(total, dtype=np.uint64)
    if total:
        got = lib().vxo_table2(K, mode, b_begin, b_end, _ptr(t1_offsets), _ptr(nonces), _ptr(hashes),
                               _ptr(t2_off), _ptr(n1), _ptr(n2), total)
        assert got == total
    return t2_off, n1, n2


# ------------------------------------------------------------------------------- Step 5
def serialize_t1(nsize: int, nonces, hashes) -> np.ndarray:
    nonces = np.ascontiguousarray(nonces, dtype=np.uint64)
    hashes = np.ascontiguousarray(hashes, dtype=np.uint64)
    out = np.empty(len(nonces) * (nsize + 8), dtype=np.uint8)
    lib().vxo_serialize_t1(nsize, len(nonces), _ptr(nonces), _ptr(hashes), _ptr8(out))
    return out


def serialize_t2(nsize: int, n1, n2) -> np.ndarray:
    n1 = np.ascontiguousarray(n1, dtype=np.uint64)
    n2 = np.ascontiguousarray(n2, dtype=np.uint64)
    out = np.empty(len(n1) * 2 * nsize, dtype=np.uint8)
    lib().vxo_serialize_t2(nsize, len(n1), _ptr(n1), _ptr(n2), _ptr8(out))
    return out


# ------------------------------------------------------------------------------- Step 6
def hash_pair(key: bytes, n1: int, n2: int, nsize: int) -> int:
    return int(lib().vxo_hash_pair(key, n1, n2, nsize))


def table2_rekey(K: int, key: bytes, bucket_bits: int, n1, n2):
    """Re-keyed Table 2 (A19, A20): (offsets[2^B+1], n1, n2, H2), buckets sorted by (H2, n1, n2)."""
    n1 = np.ascontiguousarray(n1, dtype=np.uint64)
    n2 = np.ascontiguousarray(n2, dtype=np.uint64)
    cnt = len(n1)
    offsets = np.empty((1 << bucket_bits) + 1, dtype=np.uint64)
    o1 = np.empty(max(cnt, 1), dtype=np.uint64)
    o2 = np.empty(max(cnt, 1), dtype=np.uint64)
    oh = np.empty(max(cnt, 1), dtype=np.uint64)
    rc = lib().vxo_table2_rekey(K, key, bucket_bits, cnt, _ptr(n1), _ptr(n2), _ptr(offsets), _ptr(o1), _ptr(o2), _ptr(oh))
    if rc != 0:
        raise RuntimeError(f"vxo_table2_rekey failed: {rc}")
    return offsets, o1[:cnt], o2[:cnt], oh[:cnt]


def plot_file(K: int, key: bytes, bucket_bits: int, offsets, n1, n2) -> np.ndarray:
    """The plot file bytes (A21) of a re-keyed Table 2."""
    offsets = np.ascontiguousarray(offsets, dtype=np.uint64)
    n1 = np.ascontiguousarray(n1, dtype=np.uint64)
    n2 = np.ascontiguousarray(n2, dtype=np.uint64)
    out = np.empty(int(lib().vxo_plot_file_bytes(K, bucket_bits, len(n1))), dtype=np.uint8)
    lib().vxo_plot_file(K, key, bucket_bits, len(n1), _ptr(offsets), _ptr(n1), _ptr(n2), _ptr8(out))
    return out


def mix64(z: int) -> int:
    return int(lib().vxo_mix64(z))
