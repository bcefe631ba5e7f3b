"""One plot over G processes / GPUs (include/vx.h "One plot over G GPUs").

Plumbing only: every rank creates the same plot (same key) with one bucket-range slice per rank, the
ranks exchange CUDA IPC handles of their workspaces through torch.distributed and map each other's
memory, and a build is the three C-ABI calls with a barrier over all ranks between them.  All
arithmetic -- hashing, the peer stores and peer atomics of the fused exchange, the per-rank sort +
match -- runs in the kernels behind vx_shard_* and vx_sort_match_table2*.
"""
from __future__ import annotations

from . import binding as _b


class ShardedPlot:
    """Rank `rank` of `world` (a power of two <= 8): owns the buckets [rank 2^B / world, (rank+1) 2^B / world)."""

    def __init__(self, K: int, key: bytes, rank: int, world: int, device, bucket_bits: int = 24, flags: int = 0):
        import torch
        import torch.distributed as dist
        if world < 2 or world & (world - 1) or world > 8:
            raise ValueError("world must be 2, 4 or 8")
        self.rank, self.world = rank, world
        self.plot = _b.Plot(K, key, bucket_bits, device=device,
                            flags=flags | _b.VX_CREATE_PASSES_LOG(world.bit_length() - 1))
        self.device = self.plot.device
        mine = self.plot.ipc_export()
        everyone = [None] * world
        dist.all_gather_object(everyone, mine)
        self._mapped = []
        self.peers = []
        with torch.cuda.device(self.device):
            for g, (handle, offset) in enumerate(everyone):
                if g == rank:
                    self.peers.append(self.plot.workspace.data_ptr())
                else:
                    base, ws = _b.ipc_open(handle, offset)
                    self._mapped.append(base)
                    self.peers.append(ws)
        dist.barrier()

    def _barrier(self, stream):
        import torch.distributed as dist
        stream.synchronize()        # this rank's kernels (its stores into the peers) have completed ...
        dist.barrier()              # ... on every rank

    def build_table1(self, stream=None):
        """The sharded stage 1: after it this rank holds its slice of Table 1 (vx_shard_finish)."""
        import torch
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        p = self.plot
        p.shard_begin(self.rank, self.world, stream)
        self._barrier(stream)
        p.shard_scatter(self.rank, self.world, self.peers, stream)
        self._barrier(stream)
        p.shard_finish(stream)

    def close(self):
        import torch
        import torch.distributed as dist
        torch.cuda.synchronize(self.device)
        dist.barrier()              # nobody unmaps memory a peer may still be writing
        with torch.cuda.device(self.device):
            for base in self._mapped:
                _b.ipc_close(base)
        self._mapped = []
        dist.barrier()
        self.plot.free()
