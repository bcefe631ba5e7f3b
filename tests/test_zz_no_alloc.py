"""vx_hash_fold_noalloc: the entry point that allocates nothing (its scratch is a file-scope device array of
libvx.so, 256 KB, at most 2^25 nonces per call) against the existing paths -- vx_hash_sink with caller-owned
scratch and vx_hash_range -- on two calls in a row, which share that array.  Bit-exact: integer work.
Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

import vx_inputs

pytestmark = pytest.mark.gpu

MAX_NONCES = 1 << 25


def xor_all(t):
    return int(np.bitwise_xor.reduce(t.cpu().numpy().view(np.uint64))) if t.numel() else 0


class P33:
    """vx_plot_create without vx_plot_bind (vx_hash_fold_noalloc, like vx_hash_range, needs no workspace)."""

    def __init__(self, vx, key):
        import ctypes
        self.L = vx.load_library()
        self.h = ctypes.c_void_p()
        assert self.L.vx_plot_create(33, bytes(key), ctypes.byref(self.h)) == 0

    def hash_fold_noalloc(self, begin, count, out, stream):
        st = self.L.vx_hash_fold_noalloc(self.h, begin, count, out.data_ptr(), int(stream.cuda_stream))
        assert st == 0, self.L.vx_last_error(self.h)

    def free(self):
        self.L.vx_free(self.h)


def test_no_alloc_fold_matches_the_existing_paths_on_two_calls_in_a_row():
    import torch
    import paper_2606_14007_b200 as vx
    vx.load_library()
    dev = torch.device("cuda:0")
    out = torch.full((1,), -1, dtype=torch.int64, device=dev)
    stream = torch.cuda.current_stream(dev)

    # call 1: the full limit, from nonce 0 -- against vx_hash_sink (caller-owned scratch, folded here)
    # (the hash depends on K only through NONCE_SIZE: K = 26 hashes 4-byte nonces like K = 31 and needs a small workspace)
    K1, n1 = 26, MAX_NONCES
    p1 = vx.Plot(K1, vx_inputs.config_key(31))
    sink = torch.zeros((n1 + 1023) // 1024, dtype=torch.int64, device=dev)
    p1.hash_sink(n1, sink, stream)
    want1 = xor_all(sink)
    before = torch.cuda.memory_allocated(dev)
    p1.hash_fold_noalloc(0, n1, out, stream)
    # call 2, right behind it on the same stream, SMALLER (the array still holds call 1's partials), another key,
    # 5-byte nonces and a range across 2^32 -- against vx_hash_range
    K2, b2, n2 = 33, (1 << 32) - 70001, 150001
    p2 = P33(vx, vx_inputs.config_key(K2))                # a handle without a workspace: K = 33's would be 171 GB
    out2 = torch.full((1,), -1, dtype=torch.int64, device=dev)
    base = torch.cuda.memory_allocated(dev)
    p2.hash_fold_noalloc(b2, n2, out2, stream)
    torch.cuda.synchronize(dev)
    assert torch.cuda.memory_allocated(dev) == base and base - before <= 512     # only out2 was allocated, by the test
    got1, got2 = xor_all(out), xor_all(out2)
    assert got1 == want1, "call 1 differs from vx_hash_sink"
    want2 = xor_all(vx.hash_range(K2, vx_inputs.config_key(K2), b2, n2))
    assert got2 == want2, "call 2 differs from vx_hash_range"
    # call 3: the first range again -- same answer after the array was reused
    p1.hash_fold_noalloc(0, n1, out, stream)
    torch.cuda.synchronize(dev)
    assert xor_all(out) == want1
    # ragged and empty ranges
    for begin, count in ((5, 1), (12345, 1023), (7, 1025), (0, 0)):
        p1.hash_fold_noalloc(begin, count, out, stream)
        torch.cuda.synchronize(dev)
        assert xor_all(out) == xor_all(p1.hash_range(begin, count, stream)), (begin, count)
    # beyond the limit: a clear error, nothing launched, the output untouched
    out.fill_(-7)
    with pytest.raises(vx.VxError) as ei:
        p1.hash_fold_noalloc(0, MAX_NONCES + 1, out, stream)
    assert ei.value.status == -6 and "2^25" in str(ei.value)
    torch.cuda.synchronize(dev)
    assert int(out[0]) == -7
    p1.free()
    p2.free()
