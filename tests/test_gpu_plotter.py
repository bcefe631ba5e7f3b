"""The plotter command (paper_2606_14007_b200.plotter: hash -> Table 1 -> sort + match -> Table 2 -> file, the
paper's whole program) against the oracle's file bytes."""
import os
import subprocess
import sys

import numpy as np
import pytest

import oracle
import vx_inputs
from vx_testlib import canon_t2, decode_t2, oracle_tables

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run(args):
    return subprocess.check_output([sys.executable, "-m", "paper_2606_14007_b200.plotter"] + args, cwd=ROOT, text=True)


def test_plotter_writes_the_oracles_plot_file(tmp_path):
    K, seed, B = 20, 1, 24
    key = vx_inputs.key_from_seed(seed)
    o_off, o_non, o_has, o_t2o, o_n1, o_n2 = oracle_tables(K, key, B)
    out = tmp_path / "plot.vx"
    msg = run(["--K", str(K), "--seed", str(seed), "--out", str(out)])
    assert f"{len(o_n1)} Table-2 records" in msg
    blob = np.fromfile(out, dtype=np.uint8)
    r_off, r_n1, r_n2, r_h2 = oracle.table2_rekey(K, key, B, o_n1, o_n2)
    assert len(np.unique(r_h2)) == len(r_h2)                   # no 64-bit tie: the file is unique
    assert np.array_equal(blob, oracle.plot_file(K, key, B, r_off, r_n1, r_n2)), "plot file differs from the oracle's"
    # Table 2 by source bucket, same key given as hex
    out2 = tmp_path / "t2.vx"
    run(["--K", str(K), "--key", key.hex(), "--out", str(out2), "--table2", "--slices", "5"])
    blob = np.fromfile(out2, dtype=np.uint8)
    m = len(o_n1)
    assert len(blob) == 8 * m + 8 * ((1 << B) + 1) + 32
    offs = blob[8 * m: 8 * m + 8 * ((1 << B) + 1)].view(np.uint64)
    assert np.array_equal(offs, o_t2o)
    g1, g2 = canon_t2(offs, *decode_t2(blob[:8 * m], 4))
    assert np.array_equal(g1, o_n1) and np.array_equal(g2, o_n2)
    assert bytes(blob[-32:-24]) == b"VXT2\0\0\0\1" and int(blob[-8:].view(np.uint64)[0]) == m
