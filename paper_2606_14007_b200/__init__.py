"""paper_2606_14007_b200 -- B200-native VaultxGPU plotting hot path.

BLAKE3 keyed hash of every nonce -> bucketed Table 1 in HBM -> fused per-bucket sort + match ->
Table 2.  All arithmetic runs in the hand-written sm_100a kernels of
`libvx.so` (C ABI: include/vx.h); this package is the thin ctypes binding.  PyTorch provides the
device memory and streams only.  There is no CPU fallback.
"""
from .binding import (Plot, VxError, build_library, hash_range, library_path, load_library,  # noqa: F401
                      workspace_bytes, shard_owner, ipc_open, ipc_close, probe_alu, PROBE_KINDS, EXPORTS, VX_OPT_FORCE_EXACT_RANK, VX_OPT_PARTITION_CAPACITY_LIMIT,
                      VX_OPT_TABLE2_CAPACITY_LIMIT, VX_OPT_SUBKEY_BITS, VX_OPT_STAGE2_KERNEL, VX_TABLE2_REKEYED, VX_CREATE_WIDE_LAYOUT, VX_CREATE_BIG_TILES, VX_CREATE_PASSES_LOG)
from .sharded import ShardedPlot  # noqa: F401,E402
