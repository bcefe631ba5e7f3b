"""Make a plot file on one B200: the paper's whole program (Fig. 1, L81 Fig. 3: hash ->
Table 1 -> sort + match -> Table 2 -> file) as calls into the C ABI.

    python -m paper_2606_14007_b200.plotter --K 27 --seed 27 --out plot.vx          # re-keyed plot file (A21)
    python -m paper_2606_14007_b200.plotter --K 31 --key <64 hex digits> --out t2.vx --table2

--table2 writes Table 2 as the match step leaves it (grouped by the Table-1 bucket), streamed to the file
while later slices are still being matched (vx_sort_match_table2_to_file, 4 MB sequential writes through a
pinned ring: the paper's egress, L81/L91/L165); the default also re-keys it by the hash of each pair so that a
prover can look a challenge up (vx_rekey_table2 + vx_write_plot_file; K <= 33).  Argument marshalling only:
every step runs in the kernels of libvx.so.  File layouts: include/vx.h.
"""
from __future__ import annotations

import argparse
import os
import sys
import time


def main(argv=None) -> int:
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("--K", type=int, required=True)
    g = ap.add_mutually_exclusive_group(required=True)
    g.add_argument("--key", help="256-bit plot key, 64 hex digits")
    g.add_argument("--seed", type=int, help="plot key = four SplitMix64(seed) outputs, as BASELINE.json's configs")
    ap.add_argument("--out", required=True)
    ap.add_argument("--table2", action="store_true", help="write Table 2 by source bucket instead of the re-keyed plot file")
    ap.add_argument("--device", default="cuda:0")
    ap.add_argument("--slices", type=int, default=64)
    args = ap.parse_args(argv)

    import torch

    from . import binding as vx
    if args.key is not None:
        key = bytes.fromhex(args.key)
        if len(key) != 32:
            ap.error("--key must be 64 hex digits")
    else:
        sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
        import vx_inputs
        key = vx_inputs.key_from_seed(args.seed)
    if not torch.cuda.is_available():
        raise SystemExit("plotter: no CUDA device (libvx has no CPU fallback)")
    dev = torch.device(args.device)
    torch.cuda.set_device(dev)
    plot = vx.Plot(args.K, key, device=dev)
    if not args.table2 and plot.passes > 1:
        raise SystemExit("plotter: a re-keyed plot file needs the whole Table 2 resident (K <= 33); use --table2")
    ring = torch.empty(256 << 20, dtype=torch.uint8, pin_memory=True)
    stream, copy = torch.cuda.current_stream(dev), torch.cuda.Stream(dev)
    t0 = time.perf_counter()
    written = 0
    fd = os.open(args.out, os.O_WRONLY | os.O_CREAT | os.O_TRUNC, 0o644)
    try:
        if args.table2:
            for s in range(plot.passes):                  # K >= 34: one slice file section per bucket-range pass
                if plot.passes > 1:
                    plot.select_pass(s)
                plot.build_table1(stream)
                written += plot.sort_match_table2_to_file(copy, fd, ring.data_ptr(), ring.numel(),
                                                          slices=args.slices, stream=stream)
        else:
            plot.build_table1(stream)
            plot.sort_match_table2(stream)
            plot.rekey_table2(stream)
            written = plot.write_plot_file(fd, ring.data_ptr(), ring.numel())
    finally:
        os.close(fd)
    dt = time.perf_counter() - t0
    st = plot.get_stats()
    plot.free()
    print(f"K={args.K}: {st['t1_records']} Table-1 records, {st['t2_records']} Table-2 records"
          f"{' (last pass)' if plot.passes > 1 else ''}, {written} bytes -> {args.out} in {dt:.3f} s")
    return 0


if __name__ == "__main__":
    sys.exit(main())
