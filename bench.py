#!/usr/bin/env python
"""bench.py -- the plotting hot path on N B200s, one JSON line.

A "step" is one pass of the whole hot path over one plot: vx_build_table1 (BLAKE3 keyed hash of
all 2^K nonces + bucket construction) followed by vx_sort_match_table2 (fused per-bucket sort +
match, Table 1 sorted + Table 2 written), through the C ABI.

  metric  nonces hashed + bucketed + sorted + matched per second for the whole plot (BASELINE.json:
          "nonces hashed+bucketed/s; end-to-end K=31 Table1+Table2 plot time (s), 1 B200"); the plot
          seconds and the per-stage nonces/s ride along in "plot_seconds" and "stages".
  value   device-timed, tables stay resident in HBM (the input is (K, key); nothing else exists).
  e2e     the same through the C ABI with HOST buffers: every step also copies the key in and
          streams Table 2 + its offsets to pinned host memory with vx_read_tables (the paper's
          egress, minus the disk), inside the timed region.
  roofline  the dominant kernel of the step; "stages" carries both kernels.
  cpu_baseline  the oracle as it stands on this box's host cores, bounded sample (N=1 only).

--impl reference times the CPU oracle itself (this tier's reference arm).
N > 1: independent plots, one per rank (the path partitions by plot; no data-path collective),
"scaling": "weak"; launched by torch.distributed.run.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "nonces hashed+bucketed+sorted+matched per second (whole Table1+Table2 plot)"
UNIT = "nonces/s"
BUCKET_BITS = 24
# algorithmic work per nonce: SURVEY.md 8(d)
ALU_OPS_PER_NONCE = 415            # xor / rotate / byte-swap lane-ops that need the ALU pipe
S2_BYTES_PER_NONCE = 12 + 12 + 8   # read record, write sorted record, write ~1 Table-2 record
S1_BYTES_PER_NONCE = 12            # write the record once
# integer ALU pipe: warp instructions issue at one per 2 clocks per SM sub-partition = 16 lanes/clk, measured
# with dependent-free LOP3 / SHF chains (bench.py --probe-alu; profiles/r02_alu_probe.md)
ALU_LANES_PER_SMSP = 16
# roofline.traffic: DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) per nonce of one launch
# from an ncu --set full capture of THIS tree's kernels, per kernel geometry (layout, tile_log); the
# bytes per nonce depend on the geometry, not on K.  Each entry names the summary under profiles/ it was
# read from (with the full ncu command); a geometry with no capture reports traffic = null rather than
# another geometry's number.
NCU_TRAFFIC = {
    # (layout, tile_log): B/nonce of stage 1 (vx_k_hash_scatter [+ vx_k_compact]) and of stage 2 (vx_k_sort_match)
    ("narrow", 12): {"s1": 21.91, "s2": 40.31, "source": "profiles/r02_ncu.md (narrow layout, 2^12-record tiles; ncu --set full at K=29)"},
    ("narrow", 13): {"s1": 17.18, "s2": 40.55, "source": "profiles/r02_ncu.md (narrow layout, 2^13-record tiles; ncu --set full at K=28)"},
    ("wide", 13): {"s1": 41.22, "s2": 29.54, "source": "profiles/r02_ncu.md (wide layout, 2^13-record tiles; ncu --set full at K=28)"},
}


def load_ncu_traffic():
    """(the table above is final for this tree; kept as a function so that run_cuda reads one place)"""
    return NCU_TRAFFIC


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)),
                "source": "MEASURED_PEAKS.json"}
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback (B200_PROFILING.md)"}


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.when = []
        self.t_mark = 0.0
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())
            self.when.append(time.perf_counter())     # a line is printed right after its sample is taken

    def mark(self):
        """Samples before this moment are dropped (the sampler is started ahead of the timed region so
        that nvidia-smi's start-up does not eat a short run)."""
        self.t_mark = time.perf_counter()

    def count(self):
        return sum(1 for t in self.when if t >= self.t_mark)

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r, t in zip(self.rows, self.when):
            if t < self.t_mark:
                continue
            parts = [x.strip() for x in r.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1]))
            except ValueError:
                continue
            for nm, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        busy = [x for x in sm if x >= 0.5 * max(sm)] or sm
        return {"sm_mhz": statistics.median(busy), "sm_max_mhz": max(mx), "samples": len(sm),
                "reasons": sorted(reasons)}


def rank_seed(K: int, rank: int) -> int:
    """Independent plots: rank r plots under key SplitMix64(seed_for_K + 1000 r)."""
    import vx_inputs
    return vx_inputs.seed_for_K(K) + 1000 * rank


def max_over_ranks(values, world: int, device=None):
    """Element-wise MAX over ranks of a list of floats (times are max-over-ranks, never summed)."""
    import torch
    t = torch.tensor(values, dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.tolist()]


def whole_job_value(K: int, world: int, ms_per_step: float) -> float:
    """nonces/s over all ranks: every rank makes one whole plot per step (weak scaling)."""
    return world * (1 << K) / (ms_per_step * 1e-3)


def make_config(K: int):
    import vx_inputs
    idx = {20: 0, 27: 1, 29: 2, 31: 3, 33: 4}.get(K, "-")
    return {"workload": f"K={K} plot: 2^{K} nonces, key SplitMix64({vx_inputs.seed_for_K(K)}), 2^24 buckets "
                        f"(BASELINE.json configs[{idx}])",
            "K": K, "bucket_bits": BUCKET_BITS, "plots_per_gpu": 1,
            "passes": 1 if K <= 33 else 1 << (K - 33),
            "l2": "inputs larger than L2 (tens of GB of tables are rewritten every step)"}


# --------------------------------------------------------------------------- CPU oracle legs
def oracle_plot_seconds(K: int, seed: int):
    """One whole plot with the oracle, single thread: (seconds, stage1 s, stage2 s, |T2|)."""
    import oracle
    import vx_inputs
    key = vx_inputs.key_from_seed(seed)
    t0 = time.perf_counter()
    off, non, has = oracle.table1(K, key, BUCKET_BITS)
    t1 = time.perf_counter()
    t2o, n1, n2 = oracle.table2(K, off, non, has, 1)
    t2 = time.perf_counter()
    return t2 - t0, t1 - t0, t2 - t1, len(n1)


def cpu_model() -> str:
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_plot_parallel_hash(K: int, seed: int, workers: int):
    """One whole plot with the oracle, the hashing shared by `workers` threads, each running the
    single-threaded C loop on its own nonce range (ctypes releases the GIL; the oracle keeps no global
    state); bucketing, sorting and matching on one thread.  (seconds hash, bucket+sort, match, |T2|)."""
    import numpy as np
    import oracle
    import vx_inputs
    key = vx_inputs.key_from_seed(seed)
    N = 1 << K
    t0 = time.perf_counter()
    H = oracle.hash_range_parallel(key, oracle.nonce_size(K), 0, N, workers)
    t1 = time.perf_counter()
    off, non, has = oracle.table1_from_records(BUCKET_BITS, 0, 1 << BUCKET_BITS, np.arange(N, dtype=np.uint64), H)
    t2 = time.perf_counter()
    t2o, n1, n2 = oracle.table2(K, off, non, has, 1)
    t3 = time.perf_counter()
    return t1 - t0, t2 - t1, t3 - t2, len(n1)


def cpu_baseline(full_K: int):
    """BASELINE.md section 4 / SURVEY 8(d): the oracle as it stands (gcc -O2, no intrinsics) on this box's
    host cores: K=20 in full on one thread, per stage; K=`full_K` (27) in full, per stage, the hashing
    as P = nproc single-threaded workers over disjoint nonce ranges; K=31 extrapolated from the measured
    K=27 rates and labelled so."""
    P = os.cpu_count() or 1
    t20, s1_20, s2_20, m20 = oracle_plot_seconds(20, 1)
    h, b, m, nt2 = oracle_plot_parallel_hash(full_K, full_K, P)
    N = 1 << full_K
    total = h + b + m
    per_thread_hash = N / (h * P)
    rows = [
        {"K": 20, "threads": 1, "seconds": t20, "table1_s": s1_20, "table2_s": s2_20, "t2_records": m20,
         "nonces_per_s": (1 << 20) / t20, "kind": "measured, whole plot"},
        {"K": full_K, "threads": P, "seconds": total, "hash_s": h, "bucket_sort_s": b, "table1_s": h + b,
         "table2_s": m, "t2_records": nt2, "nonces_per_s": N / total,
         "hash_nonces_per_s_per_thread": per_thread_hash,
         "kind": f"measured, whole plot; hashing on {P} threads over disjoint nonce ranges, "
                 "bucketing + sort + match on one thread"},
        {"K": 31, "threads": P, "seconds": total * (1 << (31 - full_K)), "nonces_per_s": N / total,
         "kind": f"extrapolated from the K={full_K} row (x 2^{31 - full_K}); one thread would take about "
                 f"{(h * P + b + m) * (1 << (31 - full_K)):.0f} s"},
    ]
    return {"value": N / total, "unit": UNIT, "cores": P, "kind": "oracle", "cpu": cpu_model(),
            "sample": f"whole plot at K={full_K} (2^{full_K} nonces, key SplitMix64({full_K}), B=24): hash "
                      f"{h:.1f} s on {P} threads + bucket/sort {b:.1f} s + match {m:.1f} s on one thread; "
                      f"K=20 whole plot on one thread {t20:.2f} s",
            "seconds": total, "single_thread_nonces_per_s": (1 << 20) / t20, "rows": rows}


def run_reference(args):
    """--impl reference: the oracle as it stands, on the host cores, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    K = args.ref_K
    for _ in range(args.warmup):
        oracle_plot_seconds(K, K)
    times = []
    for _ in range(args.steps):
        times.append(oracle_plot_seconds(K, K)[0])
    total = sum(times)
    value = args.steps * (1 << K) / total
    sample = (f"each step = one whole oracle plot at K={K} (2^{K} nonces, B=24), single thread; "
              f"bounded sample of the K={args.K} workload")
    ref_config = make_config(args.K)
    ref_config["workload"] += (f"; REFERENCE ARM: each step is a bounded sample of that workload, one whole oracle "
                               f"plot at K={K} (2^{K} nonces, key SplitMix64({K}), B=24) on one host thread -- "
                               f"value and ms_per_step are the sample's, not a K={args.K} plot's")
    ref_config["reference_sample_K"] = K
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32/u64",
        "data": "synthetic", "gpu_launches": 0,
        "config": ref_config,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                         "cpu": cpu_model()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)
    return 0


# --------------------------------------------------------------------------- the CUDA arm
def run_cuda(args):
    import torch
    import torch.distributed as dist

    import paper_2606_14007_b200 as vx
    import vx_inputs

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    K = args.K
    # independent plots: rank r plots under key SplitMix64(seed_for_K + 1000 r)
    key = vx_inputs.key_from_seed(rank_seed(K, rank))
    def new_plot(**kw):
        p = vx.Plot(K, key, BUCKET_BITS, device=dev, flags=args.flags, **kw)
        if args.s2_kernel:      # measurement: the warp-local stage-2 kernel instead of the default
            p.set_option(vx.VX_OPT_STAGE2_KERNEL, args.s2_kernel)
        return p

    plot = new_plot()
    N = 1 << K
    stream = torch.cuda.current_stream()

    passes = plot.passes          # > 1 from K = 34: bucket-range passes, each hashing all nonces

    def step(evs=None):
        for s in range(passes):
            if passes > 1:
                plot.select_pass(s)
            if evs: evs[3 * s].record(stream)
            plot.build_table1(stream)
            if evs: evs[3 * s + 1].record(stream)
            plot.sort_match_table2(stream)
            if evs: evs[3 * s + 2].record(stream)

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()                 # ahead of the warm-up: nvidia-smi needs a moment to print its first line
    for _ in range(args.warmup):
        step()
    barrier()
    stats = plot.get_stats()
    stats.update(plot.get_counters())   # tiles of the last stage 2 that took the exact re-rank

    # ---- device-timed region -------------------------------------------------------------
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3 * passes)] for _ in range(args.steps)]
    barrier()
    sampler.mark()                      # only samples taken from here on count
    for i in range(args.steps):
        step(evs[i])
    barrier()
    # a short run (small K) ends before nvidia-smi has printed a line: keep the same workload running,
    # untimed, until there are three samples, and say so
    extra = 0
    if rank == 0:
        t_end = time.perf_counter() + 3.0
        while sampler.count() < 3 and time.perf_counter() < t_end:
            step(); extra += 1
            torch.cuda.synchronize()
    clocks = sampler.stop() if rank == 0 else None
    if clocks is not None:
        clocks["sampled_during"] = ("the timed region" if extra == 0 else
                                    f"the timed region + {extra} untimed steps of the same workload right behind it")
    barrier()
    total_ms = evs[0][0].elapsed_time(evs[-1][-1])
    s1_ms = [sum(e[3 * s].elapsed_time(e[3 * s + 1]) for s in range(passes)) for e in evs]
    s2_ms = [sum(e[3 * s + 1].elapsed_time(e[3 * s + 2]) for s in range(passes)) for e in evs]
    plot.synchronize()

    # ---- end to end through the C ABI with host buffers -----------------------------------
    # per step: key (32 B) in; Table 2 + its offsets out, streamed through a pinned staging buffer
    nb = 1 << BUCKET_BITS
    e2e_steps = max(1, args.e2e_steps if args.e2e_steps > 0 else args.steps)
    d2h = 0
    streamed = not args.e2e_serial
    if passes > 1:
        # K >= 34: the whole Table 2 (172 GB at K = 34) does not fit this box's host memory, so every pass
        # streams its slice through a pinned ring of 4 MB chunks to a file descriptor (/dev/null here)
        streamed = False
        ring = torch.empty(256 << 20, dtype=torch.uint8, pin_memory=True)
        copy_stream = torch.cuda.Stream()
        devnull = os.open("/dev/null", os.O_WRONLY)
        e2e_what = (f"vx_plot_create(key) + per pass ({passes}): vx_build_table1 + vx_sort_match_table2_to_file(Table 2 + "
                    f"offsets through a 256 MB pinned ring of 4 MB chunks to /dev/null, {args.e2e_slices} slices)")

        def e2e_step():
            nonlocal d2h
            p2 = new_plot(workspace=plot.workspace)
            moved = 0
            for s in range(passes):
                p2.select_pass(s)
                p2.build_table1(stream)
                moved += p2.sort_match_table2_to_file(copy_stream, devnull, ring.data_ptr(), ring.numel(),
                                                      slices=args.e2e_slices, stream=stream)
            d2h = moved
            p2.free()
    elif streamed:
        # vx_sort_match_table2_to_host: stage 2 in slices, each finished slice copied
        # on a second stream straight into place in one pinned buffer while later slices are matched
        rec_cap = plot.rec2_bytes * plot.t2_capacity
        try:
            # every local rank pins a whole Table 2 (K=31: 17 GB, K=33: 86 GB): only with room to spare
            import psutil
            local_world = int(os.environ.get("LOCAL_WORLD_SIZE", str(world)))
            if psutil.virtual_memory().available < 1.5 * rec_cap * local_world + (8 << 30):
                raise RuntimeError("host memory")
            pinned_rec = torch.empty(rec_cap, dtype=torch.uint8, pin_memory=True)
        except (RuntimeError, ImportError):
            streamed = False                         # not enough pinnable host memory: ranged reads
    if passes > 1:
        pass
    elif streamed:
        copy_stream = torch.cuda.Stream()
        pinned_off = torch.empty(nb + 1, dtype=torch.int64, pin_memory=True)
        e2e_what = ("vx_plot_create(key) + vx_build_table1 + vx_sort_match_table2_to_host(Table 2 + offsets into "
                    f"pinned host memory on a second stream, {args.e2e_slices} slices overlapped with the matching)")

        def e2e_step():
            nonlocal d2h
            p2 = new_plot(workspace=plot.workspace)  # key -> kernel params
            p2.build_table1(stream)
            d2h = p2.sort_match_table2_to_host(copy_stream, pinned_rec.data_ptr(), rec_cap, pinned_off.data_ptr(),
                                               slices=args.e2e_slices, stream=stream) + (nb + 1) * 8
            p2.free()
    else:
        # vx_read_tables copies (5-byte nonces: converts and copies) Table 2 range by range after the plot
        chunks = args.e2e_chunks
        per = nb // chunks
        rec_cap = int(1.25 * plot.rec2_bytes * (N // chunks)) + (1 << 20)
        pinned_rec = torch.empty(rec_cap, dtype=torch.uint8, pin_memory=True)
        pinned_off = torch.empty(per + 1, dtype=torch.int64, pin_memory=True)
        e2e_what = ("vx_plot_create(key) + vx_build_table1 + vx_sort_match_table2 + vx_read_tables(Table 2, "
                    f"{chunks} bucket ranges) into pinned host memory")

        def e2e_step():
            nonlocal d2h
            p2 = new_plot(workspace=plot.workspace)  # key -> kernel params
            p2.build_table1(stream)
            p2.sort_match_table2(stream)
            moved = 0
            for c in range(chunks):
                moved += p2.read_tables_into(2, c * per, (c + 1) * per, pinned_off.data_ptr(),
                                             pinned_rec.data_ptr(), rec_cap) + (per + 1) * 8
            d2h = moved
            p2.free()

    e2e_step()                      # warm the pinned path
    barrier()
    e2e_each = []
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        t1 = time.perf_counter()
        e2e_step()                  # blocks until Table 2 is in host memory
        e2e_each.append(time.perf_counter() - t1)
    barrier()
    e2e_s = (time.perf_counter() - t0) / e2e_steps

    # ---- plot farm: two plots in flight (N=1 only; needs two workspaces + two pinned buffers) ----
    # plot B is hashed, sorted and matched while plot A's Table 2 is still crossing PCIe
    farm = None
    free_b, _ = torch.cuda.mem_get_info()
    host_ok = False
    try:
        import psutil
        host_ok = psutil.virtual_memory().available > 1.5 * plot.rec2_bytes * plot.t2_capacity + (8 << 30)
    except ImportError:
        pass
    if (world == 1 and streamed and host_ok and args.e2e_inflight > 1
            and free_b > plot.workspace_bytes + (2 << 30)):
        try:
            farm = run_farm(vx, torch, K, key, dev, plot, pinned_rec, pinned_off, rec_cap, nb,
                            args.e2e_slices, max(8, e2e_steps))
        except Exception as ex:                      # e.g. not enough pinned host memory
            farm = {"unavailable": repr(ex)[:200]}

    # ---- Table-2 re-keying, outside the step: one more stage a plot file needs ---------
    rekey_ms = None
    if rank == 0 and passes == 1:
        plot.build_table1(stream)
        plot.sort_match_table2(stream)
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        r0.record(stream)
        plot.rekey_table2(stream)
        r1.record(stream)
        plot.synchronize()
        rekey_ms = r0.elapsed_time(r1)

    # ---- max over ranks -------------------------------------------------------------------
    total_ms, e2e_s, s1, s2 = max_over_ranks(
        [total_ms, e2e_s, statistics.mean(s1_ms), statistics.mean(s2_ms)], world, dev)
    ms_per_step = total_ms / args.steps

    if rank == 0:
        peaks = measured_peaks()
        load_ncu_traffic()
        geom = ("wide" if plot.wide else "narrow", plot.tile_log)
        tr = NCU_TRAFFIC.get(geom)
        alu_peak = 148 * 4 * ALU_LANES_PER_SMSP * peaks["sm_max_mhz"] * 1e6 / 1e12     # T lane-ops/s on the ALU pipe
        r1 = {"kernel": "vx_k_hash_scatter", "bound": "alu", "achieved": ALU_OPS_PER_NONCE * N / (s1 * 1e-3) / 1e12,
              "peak": alu_peak, "unit": "Tlaneop/s", "traffic": tr["s1"] * N if tr else None, "ms": s1,
              "hbm_algorithmic_GBps": S1_BYTES_PER_NONCE * N / (s1 * 1e-3) / 1e9}
        r1["frac"] = r1["achieved"] / r1["peak"]
        r2 = {"kernel": "vx_k_sort_match", "bound": "hbm", "achieved": S2_BYTES_PER_NONCE * N / (s2 * 1e-3) / 1e9,
              "peak": peaks["hbm_gbs"], "unit": "GB/s", "traffic": tr["s2"] * N if tr else None, "ms": s2}
        r2["frac"] = r2["achieved"] / r2["peak"]
        dominant = dict(r1 if s1 >= s2 else r2)
        dominant["traffic_source"] = (f"{tr['source']}: DRAM read+write bytes per nonce of this kernel in the "
                                      f"{geom[0]} layout with 2^{geom[1]}-record tiles x 2^K" if tr else
                                      f"no ncu capture of the {geom[0]} layout with 2^{geom[1]}-record tiles")
        dominant["peak_source"] = peaks["source"] + (" (hbm_gbs, burst copy)" if dominant["bound"] == "hbm" else
                                                     f" (sm_max_mhz) x 148 SM x 4 SMSP x {ALU_LANES_PER_SMSP} ALU lanes/clk: "
                                                     "profiles/r02_alu_probe.md (bench.py --probe-alu)")
        line = {
            "metric": METRIC, "value": whole_job_value(K, world, ms_per_step), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32/u64",
            "data": "synthetic",
            "config": dict(make_config(K), **({"stage2_kernel": "warp-local variant (VX_OPT_STAGE2_KERNEL = 1)"} if args.s2_kernel else {})),
            "plot_seconds": ms_per_step * 1e-3, "workspace_GB": plot.workspace_bytes / 1e9,
            "stages": {"build_table1": {"ms": s1, "nonces_per_s": N / (s1 * 1e-3), "roofline": r1},
                       "sort_match_table2": {"ms": s2, "nonces_per_s": N / (s2 * 1e-3), "roofline": r2}},
            "table_stats": stats,
            "rekey_table2_ms": rekey_ms,
            "roofline": {k: dominant[k] for k in ("bound", "achieved", "peak", "unit", "frac", "traffic", "kernel", "peak_source", "traffic_source")},
            "e2e": {"value": world * N / e2e_s, "unit": UNIT, "h2d_bytes_per_step": 32,
                    "d2h_bytes_per_step": d2h, "seconds_per_step": e2e_s, "steps": e2e_steps,
                    "seconds_each_rank0": [round(x, 4) for x in e2e_each],
                    "what": e2e_what, "two_plots_in_flight": farm},
            "gpu_launches": plot.launches_per_plot * passes * args.steps,
            "clocks": clocks,
        }
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(args.cpu_K)
        print(json.dumps(line), flush=True)
    plot.free()
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_probe_alu(args):
    """Issue rate of the integer pipes: dependent-free chains of one instruction kind, 2048 threads per
    SM, timed with CUDA events; lane-ops per clock per SM at the SM clock sampled during the run."""
    import torch

    import paper_2606_14007_b200 as vx
    torch.cuda.set_device(0)
    scratch = torch.zeros(1024, dtype=torch.int32, device="cuda:0")
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    iters = 1 << 14
    out = {}
    sampler = ClockSampler(0)
    sampler.start()
    for kind in ("lop3", "shf", "arx", "prmt", "add", "imad"):
        for _ in range(2):
            vx.probe_alu(kind, iters, scratch)
        torch.cuda.synchronize()
        best = None
        for _ in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            ops = vx.probe_alu(kind, iters, scratch)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            best = ms if best is None else min(best, ms)
        out[kind] = {"lane_ops": ops, "ms": best, "Tlaneop_per_s": ops / (best * 1e-3) / 1e12}
    clocks = sampler.stop()
    mhz = clocks.get("sm_mhz") or measured_peaks()["sm_max_mhz"]
    for v in out.values():
        v["lanes_per_clk_per_sm"] = v["Tlaneop_per_s"] * 1e12 / (mhz * 1e6) / sms
        v["lanes_per_clk_per_smsp"] = v["lanes_per_clk_per_sm"] / 4
    print(json.dumps({"probe": "alu", "sms": sms, "sm_mhz": mhz, "clocks": clocks, "kinds": out}), flush=True)
    return 0


def run_one_plot(args):
    """--one-plot: ONE plot over the N ranks instead of one plot per rank: rank r hashes
    its nonce share, the records cross to their owners inside stage 1 (peer stores over NVLink), every rank
    sorts and matches its bucket range.  "scaling": "strong".  Ranks that must share a device (a one-GPU
    box) run over gloo: a functional check, not a measurement."""
    import torch
    import torch.distributed as dist

    import paper_2606_14007_b200 as vx
    import vx_inputs
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world < 2:
        raise SystemExit("bench.py --one-plot needs --gpus 2, 4 or 8 (torch.distributed.run)")
    shared = torch.cuda.device_count() < int(os.environ.get("LOCAL_WORLD_SIZE", str(world)))
    dev = torch.device("cuda", 0 if shared else local)
    torch.cuda.set_device(dev)
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    dist.init_process_group("gloo" if shared else "nccl", **({} if shared else {"device_id": dev}))
    K = args.K
    key = vx_inputs.config_key(K)
    sp = vx.ShardedPlot(K, key, rank, world, dev, bucket_bits=BUCKET_BITS)
    stream = torch.cuda.current_stream()

    def step(evs=None):
        if evs: evs[0].record(stream)
        sp.build_table1(stream)
        if evs: evs[1].record(stream)
        sp.plot.sort_match_table2(stream)
        if evs: evs[2].record(stream)

    def barrier():
        torch.cuda.synchronize()
        dist.barrier()

    for _ in range(args.warmup):
        step()
    barrier()
    stats = sp.plot.get_stats()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    sampler = ClockSampler(dev.index)
    if rank == 0:
        sampler.start()
    barrier()
    sampler.mark()
    for i in range(args.steps):
        step(evs[i])
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    total_ms = evs[0][0].elapsed_time(evs[-1][2])
    s1 = statistics.mean(e[0].elapsed_time(e[1]) for e in evs)
    s2 = statistics.mean(e[1].elapsed_time(e[2]) for e in evs)
    t = torch.tensor([total_ms, s1, s2], dtype=torch.float64, device=None if shared else dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    cnt = torch.tensor([stats["t1_records"], stats["t2_records"]], dtype=torch.int64, device=None if shared else dev)
    dist.all_reduce(cnt, op=dist.ReduceOp.SUM)
    total_ms, s1, s2 = (float(x) for x in t.tolist())
    if rank == 0:
        ms = total_ms / args.steps
        cfg = make_config(K)
        cfg["plots_per_gpu"] = f"1/{world} (one plot over {world} ranks)"
        cfg["parallelism"] = (f"nonce range split {world} ways, buckets owned by hash range, all-to-all fused with "
                              "stage 1 (peer stores + peer atomics), bucket-local sort + match")
        line = {"metric": METRIC, "value": (1 << K) / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "strong",
                "vs_baseline": None, "dtype": "u32/u64", "data": "synthetic", "config": cfg,
                "stages": {"build_table1_sharded": {"ms": s1}, "sort_match_table2": {"ms": s2}},
                "table_stats": {"t1_records": int(cnt[0]), "t2_records": int(cnt[1])},
                "ranks_share_one_device": shared,
                "note": ("functional run: the ranks share one GPU, gloo barriers" if shared else
                         "device time per rank between CUDA events, max over ranks; host barriers inside the step"),
                "gpu_launches": 5 * args.steps, "clocks": clocks}
        print(json.dumps(line), flush=True)
    sp.close()
    dist.destroy_process_group()
    return 0


def run_farm(vx, torch, K, key, dev, plot, rec_a, off_a, rec_cap, nb, slices, steps_each):
    """Two host threads, each plotting end to end into its own workspace and pinned buffers:
    whole-plot throughput with the PCIe egress of one plot hidden behind the kernels of the other."""
    ws_b = torch.empty(plot.workspace_bytes, dtype=torch.uint8, device=dev)
    rec_b = torch.empty(rec_cap, dtype=torch.uint8, pin_memory=True)
    off_b = torch.empty(nb + 1, dtype=torch.int64, pin_memory=True)
    lanes = [(plot.workspace, rec_a, off_a), (ws_b, rec_b, off_b)]
    streams = [(torch.cuda.Stream(), torch.cuda.Stream()) for _ in lanes]
    errors = []

    def worker(i, n):
        try:
            torch.cuda.set_device(dev)
            ws, rec, off = lanes[i]
            comp, copy = streams[i]
            for _ in range(n):
                p = vx.Plot(K, key, BUCKET_BITS, device=dev, workspace=ws)
                p.build_table1(comp)
                p.sort_match_table2_to_host(copy, rec.data_ptr(), rec_cap, off.data_ptr(), slices=slices, stream=comp)
                p.free()
        except Exception as ex:
            errors.append(repr(ex))

    def run(n):
        th = [threading.Thread(target=worker, args=(i, n)) for i in range(len(lanes))]
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for t in th: t.start()
        for t in th: t.join()
        torch.cuda.synchronize()
        return time.perf_counter() - t0

    run(1)                                           # warm both lanes
    dt = run(steps_each)
    if errors:
        raise RuntimeError(errors[0])
    plots = len(lanes) * steps_each
    return {"plots": plots, "seconds_per_plot": dt / plots, "value": plots * (1 << K) / dt, "unit": UNIT,
            "what": "two host threads, one plot each in flight (own workspace, streams and pinned buffers): "
                    "vx_build_table1 + vx_sort_match_table2_to_host back to back"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--K", type=int, default=31, help="plot size; 31 = the configuration the metric is quoted on")
    ap.add_argument("--cpu-K", dest="cpu_K", type=int, default=27,
                    help="cpu_baseline: the oracle makes this plot in full (hashing on nproc threads), and K=20 on one")
    ap.add_argument("--flags", type=int, default=0,
                    help="test-only layout flags (1 wide layout, 2 big tiles): ncu captures of the K>=32 geometries at small K")
    ap.add_argument("--s2-kernel", dest="s2_kernel", type=int, default=0, choices=[0, 1],
                    help="VX_OPT_STAGE2_KERNEL: 0 = the default fused kernel, 1 = its warp-local variant (a measured alternative)")
    ap.add_argument("--one-plot", dest="one_plot", action="store_true",
                    help="with --gpus N > 1: ONE plot sharded over the N ranks (strong scaling) instead of one plot per rank")
    ap.add_argument("--probe-alu", dest="probe_alu", action="store_true",
                    help="integer-pipe issue rates from dependent-free instruction chains (vx_probe_alu), one JSON line")
    ap.add_argument("--ref-K", dest="ref_K", type=int, default=22, help="oracle sample size per --impl reference step")
    ap.add_argument("--e2e-steps", dest="e2e_steps", type=int, default=0, help="0 = as many as --steps")
    ap.add_argument("--e2e-chunks", dest="e2e_chunks", type=int, default=32)
    ap.add_argument("--e2e-slices", dest="e2e_slices", type=int, default=64)
    ap.add_argument("--e2e-inflight", dest="e2e_inflight", type=int, default=2,
                    help="2: also report end-to-end throughput with two plots in flight (N=1, K<=31)")
    ap.add_argument("--e2e-serial", dest="e2e_serial", action="store_true",
                    help="e2e with vx_read_tables after the plot instead of the streamed egress")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "cuda":
        print("bench.py: note: warmup < 3 breaks the timing rules", file=sys.stderr)
    if args.impl == "reference":
        return run_reference(args)
    if args.probe_alu:
        return run_probe_alu(args)
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus != world:
        if world == 1 and args.gpus > 1:
            # convenience: relaunch under torch.distributed.run
            cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
                   "--master-addr", "127.0.0.1", "--master-port", "29541", os.path.abspath(__file__)] + sys.argv[1:]
            return subprocess.call(cmd)
    if args.one_plot:
        return run_one_plot(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
