"""ctypes binding of libvx.so with the same names as include/vx.h (argument marshalling only).

Every step of the hot path runs in the CUDA kernels behind the C ABI.  PyTorch supplies the
device workspace (a uint8 CUDA tensor) and the stream.  If the library or a CUDA device is
missing, calls raise: nothing here computes on the CPU.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import build as _build

VX_OK = 0
VX_OPT_FORCE_EXACT_RANK = 1
VX_OPT_PARTITION_CAPACITY_LIMIT = 2
VX_OPT_TABLE2_CAPACITY_LIMIT = 3
VX_OPT_SUBKEY_BITS = 4
VX_OPT_STAGE2_KERNEL = 5
VX_TABLE2_REKEYED = 3
VX_CREATE_WIDE_LAYOUT = 1
VX_CREATE_BIG_TILES = 2


def VX_CREATE_PASSES_LOG(l: int) -> int:
    return l << 8

STATUS = {0: "VX_OK", -1: "VX_ERR_ARG", -2: "VX_ERR_STATE", -3: "VX_ERR_WORKSPACE", -4: "VX_ERR_CUDA",
          -5: "VX_ERR_OVERFLOW", -6: "VX_ERR_RANGE", -7: "VX_ERR_UNSUPPORTED", -8: "VX_ERR_IO", -9: "VX_ERR_NOMEM"}

#: every symbol include/vx.h declares
EXPORTS = ["vx_workspace_bytes", "vx_workspace_bytes_ex", "vx_workspace_bytes_opts", "vx_plot_create",
           "vx_plot_create_ex", "vx_plot_create_opts",
           "vx_plot_bind", "vx_build_table1", "vx_sort_match_table2", "vx_sort_match_table2_to_host",
           "vx_sort_match_table2_to_file", "vx_read_tables", "vx_plot_passes", "vx_plot_select_pass",
           "vx_plot_all_passes_to_host", "vx_rekey_table2", "vx_write_plot_file", "vx_shard_owner", "vx_shard_begin", "vx_shard_scatter", "vx_shard_finish",
           "vx_ipc_export", "vx_ipc_open", "vx_ipc_close",
           "vx_device_tables", "vx_plot_set_option", "vx_get_stats", "vx_get_counters", "vx_synchronize", "vx_hash_range",
           "vx_hash_sink", "vx_probe_alu", "vx_hash_fold_noalloc",
           "vx_plot_info", "vx_plot_layout", "vx_plot_launches", "vx_last_error", "vx_status_string", "vx_free"]

_u64 = ctypes.c_uint64
_u32 = ctypes.c_uint32
_vp = ctypes.c_void_p
_sz = ctypes.c_size_t


class VxError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__(f"{STATUS.get(status, status)}: {text}")
        self.status = status


def library_path() -> str:
    return _build.LIB


def build_library(force: bool = False) -> str:
    return _build.build(force=force)


_lib = None


def load_library() -> ctypes.CDLL:
    """Load (building first if the sources are newer) libvx.so.  Raises if it cannot be had."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if _build.is_stale():
        path = _build.build()
    L = ctypes.CDLL(path)
    L.vx_workspace_bytes.restype = _sz
    L.vx_workspace_bytes.argtypes = [_u32]
    L.vx_workspace_bytes_ex.restype = _sz
    L.vx_workspace_bytes_ex.argtypes = [_u32, _u32]
    L.vx_plot_create.restype = ctypes.c_int
    L.vx_plot_create.argtypes = [_u32, ctypes.c_char_p, ctypes.POINTER(_vp)]
    L.vx_plot_create_ex.restype = ctypes.c_int
    L.vx_plot_create_ex.argtypes = [_u32, ctypes.c_char_p, _u32, ctypes.POINTER(_vp)]
    L.vx_workspace_bytes_opts.restype = _sz
    L.vx_workspace_bytes_opts.argtypes = [_u32, _u32, _u32]
    L.vx_plot_create_opts.restype = ctypes.c_int
    L.vx_plot_create_opts.argtypes = [_u32, ctypes.c_char_p, _u32, _u32, ctypes.POINTER(_vp)]
    L.vx_plot_bind.restype = ctypes.c_int
    L.vx_plot_bind.argtypes = [_vp, _vp, _sz]
    L.vx_build_table1.restype = ctypes.c_int
    L.vx_build_table1.argtypes = [_vp, _vp]
    L.vx_sort_match_table2.restype = ctypes.c_int
    L.vx_sort_match_table2.argtypes = [_vp, _vp]
    L.vx_sort_match_table2_to_host.restype = ctypes.c_int
    L.vx_sort_match_table2_to_host.argtypes = [_vp, _vp, _vp, _u32, _vp, _sz, _vp, ctypes.POINTER(_sz)]
    L.vx_sort_match_table2_to_file.restype = ctypes.c_int
    L.vx_sort_match_table2_to_file.argtypes = [_vp, _vp, _vp, _u32, ctypes.c_int, _vp, _sz, ctypes.POINTER(_u64)]
    L.vx_plot_passes.restype = ctypes.c_int
    L.vx_plot_passes.argtypes = [_vp, ctypes.POINTER(_u32), ctypes.POINTER(_u32), ctypes.POINTER(_u64),
                                 ctypes.POINTER(_u64)]
    L.vx_plot_select_pass.restype = ctypes.c_int
    L.vx_plot_select_pass.argtypes = [_vp, _u32]
    L.vx_plot_all_passes_to_host.restype = ctypes.c_int
    L.vx_plot_all_passes_to_host.argtypes = [_vp, _vp, _vp, _u32, _vp, _sz, _vp, ctypes.POINTER(_sz),
                                             ctypes.POINTER(_u64)]
    L.vx_shard_owner.restype = ctypes.c_int
    L.vx_shard_owner.argtypes = [_u32, _u32, _u32, _u32] + [ctypes.POINTER(_u64)] * 4
    L.vx_shard_begin.restype = ctypes.c_int
    L.vx_shard_begin.argtypes = [_vp, _u32, _u32, _vp]
    L.vx_shard_scatter.restype = ctypes.c_int
    L.vx_shard_scatter.argtypes = [_vp, _u32, _u32, ctypes.POINTER(_vp), _vp]
    L.vx_shard_finish.restype = ctypes.c_int
    L.vx_shard_finish.argtypes = [_vp, _vp]
    L.vx_rekey_table2.restype = ctypes.c_int
    L.vx_rekey_table2.argtypes = [_vp, _vp]
    L.vx_write_plot_file.restype = ctypes.c_int
    L.vx_write_plot_file.argtypes = [_vp, ctypes.c_int, _vp, _sz, ctypes.POINTER(_u64)]
    L.vx_ipc_export.restype = ctypes.c_int
    L.vx_ipc_export.argtypes = [_vp, ctypes.c_char_p, ctypes.POINTER(_u64)]
    L.vx_ipc_open.restype = ctypes.c_int
    L.vx_ipc_open.argtypes = [ctypes.c_char_p, _u64, ctypes.POINTER(_vp), ctypes.POINTER(_vp)]
    L.vx_ipc_close.restype = ctypes.c_int
    L.vx_ipc_close.argtypes = [_vp]
    L.vx_read_tables.restype = ctypes.c_int
    L.vx_read_tables.argtypes = [_vp, ctypes.c_int, _u64, _u64, _vp, _vp, _sz, ctypes.POINTER(_sz)]
    L.vx_device_tables.restype = ctypes.c_int
    L.vx_device_tables.argtypes = [_vp] + [ctypes.POINTER(_vp)] * 5
    L.vx_plot_set_option.restype = ctypes.c_int
    L.vx_plot_set_option.argtypes = [_vp, ctypes.c_int, _u64]
    L.vx_get_stats.restype = ctypes.c_int
    L.vx_get_stats.argtypes = [_vp, ctypes.POINTER(_u64), ctypes.POINTER(_u64), ctypes.POINTER(_u32)]
    L.vx_get_counters.restype = ctypes.c_int
    L.vx_get_counters.argtypes = [_vp, ctypes.POINTER(_u64)]
    L.vx_synchronize.restype = ctypes.c_int
    L.vx_synchronize.argtypes = [_vp]
    L.vx_hash_range.restype = ctypes.c_int
    L.vx_hash_range.argtypes = [_vp, _u64, _u64, _vp, _vp]
    L.vx_hash_sink.restype = ctypes.c_int
    L.vx_hash_sink.argtypes = [_vp, _u64, _vp, _sz, _vp]
    L.vx_hash_fold_noalloc.restype = ctypes.c_int
    L.vx_hash_fold_noalloc.argtypes = [_vp, _u64, _u64, _vp, _vp]
    L.vx_probe_alu.restype = ctypes.c_int
    L.vx_probe_alu.argtypes = [ctypes.c_int, _u32, _u32, _vp, _sz, _vp, ctypes.POINTER(_u64)]
    L.vx_plot_info.restype = ctypes.c_int
    L.vx_plot_info.argtypes = [_vp] + [ctypes.POINTER(_u32)] * 5 + [ctypes.POINTER(_u64)]
    L.vx_plot_layout.restype = ctypes.c_int
    L.vx_plot_layout.argtypes = [_vp, ctypes.POINTER(_u32), ctypes.POINTER(_u32)]
    L.vx_plot_launches.restype = ctypes.c_int
    L.vx_plot_launches.argtypes = [_vp, ctypes.POINTER(_u32), ctypes.POINTER(_u32)]
    L.vx_last_error.restype = ctypes.c_char_p
    L.vx_last_error.argtypes = [_vp]
    L.vx_status_string.restype = ctypes.c_char_p
    L.vx_status_string.argtypes = [ctypes.c_int]
    L.vx_free.restype = None
    L.vx_free.argtypes = [_vp]
    _lib = L
    return L


def workspace_bytes(K: int, bucket_bits: int = 24, flags: int = 0) -> int:
    return int(load_library().vx_workspace_bytes_opts(K, bucket_bits, flags))


def _stream_ptr(stream, device=None) -> int:
    import torch
    if stream is None:
        stream = torch.cuda.current_stream(device)
    return int(stream.cuda_stream)


class Plot:
    """One plot (K, key): vx_plot_create + vx_plot_bind on a torch-owned workspace."""

    def __init__(self, K: int, key: bytes, bucket_bits: int = 24, device="cuda:0", workspace=None,
                 flags: int = 0):
        import torch
        if len(key) != 32:
            raise ValueError("key must be 32 bytes")
        self._L = load_library()
        self._h = _vp()
        st = self._L.vx_plot_create_opts(K, bytes(key), bucket_bits, flags, ctypes.byref(self._h))
        if st != VX_OK:
            raise VxError(st, f"vx_plot_create_opts(K={K}, bucket_bits={bucket_bits}, flags={flags})")
        self.K, self.bucket_bits = K, bucket_bits
        info = [_u32() for _ in range(5)]
        t2cap = _u64()
        self._L.vx_plot_info(self._h, *[ctypes.byref(x) for x in info], ctypes.byref(t2cap))
        self.nonce_size = info[2].value
        self.partition_bits = info[3].value
        self.partition_capacity = info[4].value
        self.t2_capacity = t2cap.value
        wide, tlog = _u32(), _u32()
        self._L.vx_plot_layout(self._h, ctypes.byref(wide), ctypes.byref(tlog))
        self.wide, self.tile_log = bool(wide.value), tlog.value
        l1, l2 = _u32(), _u32()
        self._L.vx_plot_launches(self._h, ctypes.byref(l1), ctypes.byref(l2))
        self.launches_per_plot = l1.value + l2.value
        np_, sel = _u32(), _u32()
        self._L.vx_plot_passes(self._h, ctypes.byref(np_), ctypes.byref(sel), None, None)
        self.passes = np_.value
        self.rec1_bytes = self.nonce_size + 8
        self.rec2_bytes = 2 * self.nonce_size
        need = int(self._L.vx_workspace_bytes_opts(K, bucket_bits, flags))
        if not torch.cuda.is_available():
            self.free()
            raise VxError(-4, "no CUDA device: libvx has no CPU fallback")
        self.device = torch.device(device)
        if workspace is None:
            workspace = torch.empty(need, dtype=torch.uint8, device=self.device)
        self.workspace = workspace
        self.workspace_bytes = need
        with torch.cuda.device(self.device):
            self._check(self._L.vx_plot_bind(self._h, workspace.data_ptr(), workspace.numel()))

    # -- plumbing -------------------------------------------------------------------------------
    def _dev(self):
        """Every ABI call runs with the plot's device current (kernels launch on the current device)."""
        import torch
        return torch.cuda.device(self.device)

    def _sp(self, stream) -> int:
        return _stream_ptr(stream, self.device)

    def _check(self, st: int):
        if st != VX_OK:
            raise VxError(st, self._L.vx_last_error(self._h).decode())

    def free(self):
        if getattr(self, "_h", None):
            self._L.vx_free(self._h)
            self._h = None
        self.workspace = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.free()

    # -- the hot path ---------------------------------------------------------------------------
    def build_table1(self, stream=None):
        with self._dev():
            self._check(self._L.vx_build_table1(self._h, self._sp(stream)))

    def sort_match_table2(self, stream=None):
        with self._dev():
            self._check(self._L.vx_sort_match_table2(self._h, self._sp(stream)))

    def sort_match_table2_to_host(self, copy_stream, records_ptr: int, records_capacity: int,
                                  offsets_ptr: int = 0, slices: int = 16, stream=None) -> int:
        """Stage 2 in `slices` launches with Table 2 streamed to host memory on copy_stream
        (vx_sort_match_table2_to_host); raw host pointers (pinned torch tensors); returns record bytes."""
        need = _sz()
        with self._dev():
            self._check(self._L.vx_sort_match_table2_to_host(
                self._h, self._sp(stream), self._sp(copy_stream), slices, records_ptr, records_capacity,
                offsets_ptr or None, ctypes.byref(need)))
        return need.value

    def sort_match_table2_to_file(self, copy_stream, fd: int, staging_ptr: int, staging_bytes: int,
                                  slices: int = 16, stream=None) -> int:
        """Same, to a file descriptor through a pinned ring of 4 MB chunks; returns the bytes written."""
        n = _u64()
        with self._dev():
            self._check(self._L.vx_sort_match_table2_to_file(
                self._h, self._sp(stream), self._sp(copy_stream), slices, fd, staging_ptr, staging_bytes,
                ctypes.byref(n)))
        return n.value

    def select_pass(self, s: int):
        with self._dev():
            self._check(self._L.vx_plot_select_pass(self._h, s))

    def pass_buckets(self):
        """(bucket_begin, bucket_end) of the selected pass."""
        b0, b1 = _u64(), _u64()
        self._L.vx_plot_passes(self._h, None, None, ctypes.byref(b0), ctypes.byref(b1))
        return b0.value, b1.value

    def all_passes_to_host(self, copy_stream, records_ptr: int, records_capacity: int, offsets_ptr: int = 0,
                           slices: int = 16, stream=None):
        """The whole plot, pass by pass, Table 2 streamed to host memory: (record bytes, Table-1 records)."""
        need, t1 = _sz(), _u64()
        with self._dev():
            self._check(self._L.vx_plot_all_passes_to_host(
                self._h, self._sp(stream), self._sp(copy_stream), slices, records_ptr, records_capacity,
                offsets_ptr or None, ctypes.byref(need), ctypes.byref(t1)))
        return need.value, t1.value

    # -- re-keying + plot file (8(f2)) -------------------------------------------------------------
    def rekey_table2(self, stream=None):
        with self._dev():
            self._check(self._L.vx_rekey_table2(self._h, self._sp(stream)))

    def write_plot_file(self, fd: int, staging_ptr: int, staging_bytes: int) -> int:
        n = _u64()
        with self._dev():
            self._check(self._L.vx_write_plot_file(self._h, fd, staging_ptr, staging_bytes, ctypes.byref(n)))
        return n.value

    # -- one plot over G GPUs (8(f4)) ------------------------------------------------------------
    def shard_begin(self, rank: int, world: int, stream=None):
        with self._dev():
            self._check(self._L.vx_shard_begin(self._h, rank, world, self._sp(stream)))

    def shard_scatter(self, rank: int, world: int, peer_ptrs, stream=None):
        arr = (_vp * world)(*[int(x) for x in peer_ptrs])
        with self._dev():
            self._check(self._L.vx_shard_scatter(self._h, rank, world, arr, self._sp(stream)))

    def ipc_export(self):
        """(64-byte CUDA IPC handle, offset) of the workspace, for a peer process (vx_ipc_export)."""
        buf = ctypes.create_string_buffer(64)
        off = _u64()
        with self._dev():
            self._check(self._L.vx_ipc_export(self._h, buf, ctypes.byref(off)))
        return buf.raw, off.value

    def shard_finish(self, stream=None):
        with self._dev():
            self._check(self._L.vx_shard_finish(self._h, self._sp(stream)))

    def synchronize(self):
        with self._dev():
            self._check(self._L.vx_synchronize(self._h))

    def get_stats(self):
        t1, t2, mb = _u64(), _u64(), _u32()
        with self._dev():
            self._check(self._L.vx_get_stats(self._h, ctypes.byref(t1), ctypes.byref(t2), ctypes.byref(mb)))
        return {"t1_records": t1.value, "t2_records": t2.value, "max_bucket": mb.value}

    def get_counters(self):
        r = _u64()
        with self._dev():
            self._check(self._L.vx_get_counters(self._h, ctypes.byref(r)))
        return {"tile_retries": r.value}

    def read_tables(self, table: int, bucket_begin: int | None = None, bucket_end: int | None = None,
                    records_out: np.ndarray | None = None):
        """(offsets uint64[nb+1] relative to the range, records uint8[...]) copied to the host.
        Default range: all buckets of the selected pass (= all 2^B buckets of a one-pass plot)."""
        if bucket_begin is None:
            bucket_begin = self.pass_buckets()[0]
        if bucket_end is None:
            bucket_end = self.pass_buckets()[1]
        nb = bucket_end - bucket_begin
        offsets = np.empty(max(nb, 0) + 1, dtype=np.uint64)
        need = _sz()
        with self._dev():
            self._check(self._L.vx_read_tables(self._h, table, bucket_begin, bucket_end,
                                               offsets.ctypes.data, None, 0, ctypes.byref(need)))
            if records_out is None:
                records_out = np.empty(need.value, dtype=np.uint8)
            assert records_out.dtype == np.uint8 and records_out.flags.c_contiguous
            self._check(self._L.vx_read_tables(self._h, table, bucket_begin, bucket_end,
                                               offsets.ctypes.data, records_out.ctypes.data,
                                               records_out.nbytes, ctypes.byref(need)))
        return offsets, records_out[:need.value]

    def read_tables_into(self, table: int, bucket_begin: int, bucket_end: int,
                         offsets_ptr: int, records_ptr: int, records_capacity: int) -> int:
        """Raw-pointer form (e.g. pinned torch tensors): returns the record bytes written."""
        need = _sz()
        with self._dev():
            self._check(self._L.vx_read_tables(self._h, table, bucket_begin, bucket_end,
                                               offsets_ptr, records_ptr, records_capacity, ctypes.byref(need)))
        return need.value

    def set_option(self, option: int, value: int):
        self._check(self._L.vx_plot_set_option(self._h, option, value))

    def device_tables(self):
        """[t1 partition array, t1 offsets, t2 records, t2 offsets, partition base] device pointers."""
        ptrs = [_vp() for _ in range(5)]
        self._check(self._L.vx_device_tables(self._h, *[ctypes.byref(x) for x in ptrs]))
        return [x.value for x in ptrs]

    def hash_range(self, nonce_begin: int, count: int, stream=None):
        """H(n) for n in [nonce_begin, nonce_begin+count) as a torch int64 CUDA tensor (bit pattern of u64)."""
        import torch
        out = torch.empty(count, dtype=torch.int64, device=self.device)
        with self._dev():
            self._check(self._L.vx_hash_range(self._h, nonce_begin, count, out.data_ptr(), self._sp(stream)))
        return out

    def hash_fold_noalloc(self, nonce_begin: int, count: int, out, stream=None):
        """vx_hash_fold_noalloc: xor of H(n) over the range -> out[0] (a 1-element int64 CUDA tensor the caller
        owns); the library's scratch is a static device array, nothing is allocated."""
        with self._dev():
            self._check(self._L.vx_hash_fold_noalloc(self._h, nonce_begin, count, out.data_ptr(), self._sp(stream)))

    def hash_sink(self, count: int, sink, stream=None):
        with self._dev():
            self._check(self._L.vx_hash_sink(self._h, count, sink.data_ptr(), sink.numel(), self._sp(stream)))


PROBE_KINDS = {"lop3": 0, "shf": 1, "add": 2, "imad": 3, "prmt": 4, "arx": 5}


def probe_alu(kind: str, iters: int, scratch, ctas_per_sm: int = 8, stream=None) -> int:
    """vx_probe_alu: enqueue one dependent-free chain kernel; returns the lane-ops it executes."""
    ops = _u64()
    st = load_library().vx_probe_alu(PROBE_KINDS[kind], iters, ctas_per_sm, scratch.data_ptr(), scratch.numel(),
                                     _stream_ptr(stream, scratch.device), ctypes.byref(ops))
    if st != VX_OK:
        raise VxError(st, f"vx_probe_alu({kind})")
    return ops.value


def ipc_open(handle: bytes, offset: int):
    """Map a peer process's workspace (vx_ipc_open) on the current device: (mapped base, workspace pointer)."""
    base, ws = _vp(), _vp()
    st = load_library().vx_ipc_open(handle, offset, ctypes.byref(base), ctypes.byref(ws))
    if st != VX_OK:
        raise VxError(st, "vx_ipc_open")
    return base.value, ws.value


def ipc_close(mapped_base: int):
    st = load_library().vx_ipc_close(mapped_base)
    if st != VX_OK:
        raise VxError(st, "vx_ipc_close")


def shard_owner(K: int, bucket_bits: int, world: int, rank: int):
    """(nonce_begin, nonce_end, bucket_begin, bucket_end) of a rank of a plot sharded over `world` GPUs."""
    v = [_u64() for _ in range(4)]
    st = load_library().vx_shard_owner(K, bucket_bits, world, rank, *[ctypes.byref(x) for x in v])
    if st != VX_OK:
        raise VxError(st, f"vx_shard_owner(K={K}, B={bucket_bits}, world={world}, rank={rank})")
    return tuple(x.value for x in v)


def hash_range(K: int, key: bytes, nonce_begin: int, count: int):
    """Convenience: H(n) for a nonce range without building tables (no workspace needed)."""
    import torch
    L = load_library()
    h = _vp()
    st = L.vx_plot_create(K, bytes(key), ctypes.byref(h))
    if st != VX_OK:
        raise VxError(st, f"vx_plot_create(K={K})")
    try:
        if not torch.cuda.is_available():
            raise VxError(-4, "no CUDA device: libvx has no CPU fallback")
        out = torch.empty(count, dtype=torch.int64, device="cuda:0")
        st = L.vx_hash_range(h, nonce_begin, count, out.data_ptr(), _stream_ptr(None))
        if st != VX_OK:
            raise VxError(st, L.vx_last_error(h).decode())
        torch.cuda.synchronize()
        return out
    finally:
        L.vx_free(h)
