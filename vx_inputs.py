"""Seeded synthetic inputs shared by the oracle tests and the CUDA path's tests/bench.

Holds none of the method's arithmetic (no hashing, bucketing or matching): only the plot
configurations BASELINE.json names and the SplitMix64 key derivation they are defined with
("256-bit plot key from SplitMix64(seed=...)").  The workload itself is self-generating: the
nonces are 0 .. 2^K - 1, so a configuration is just (K, key).
"""
from __future__ import annotations

MASK64 = (1 << 64) - 1

#: BASELINE.json `configs`: K -> SplitMix64 seed.  Any other K in the 20..33 sweep uses seed = K
#: (SURVEY.md 8(d) "Inputs").
CONFIG_SEEDS = {20: 1, 27: 27, 29: 29, 31: 31, 33: 33}

#: the paper's setting: 2^24 buckets
BUCKET_BITS = 24


def splitmix64_stream(seed: int, count: int) -> list[int]:
    """First `count` outputs of SplitMix64 started at `seed` (Steele, Lea & Flood 2014)."""
    s = seed & MASK64
    out = []
    for _ in range(count):
        s = (s + 0x9E3779B97F4A7C15) & MASK64
        z = s
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & MASK64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & MASK64
        out.append(z ^ (z >> 31))
    return out


def key_from_seed(seed: int) -> bytes:
    """256-bit plot key: four successive SplitMix64 outputs, each little-endian, concatenated."""
    return b"".join(w.to_bytes(8, "little") for w in splitmix64_stream(seed, 4))


def seed_for_K(K: int) -> int:
    return CONFIG_SEEDS.get(K, K)


def config_key(K: int) -> bytes:
    """The plot key of the BASELINE.json configuration for this K."""
    return key_from_seed(seed_for_K(K))
