"""Host logic of bench.py (`-m "not gpu"`): the per-call algorithmic bytes partition SURVEY.md §8(d)'s step bytes, and both
arms print the same `config`."""
import argparse
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402
import workloads as W  # noqa: E402


def test_call_bytes_partition_the_compulsory_bytes():
    for (R, E, U, H, D, b, dedup) in [(200000, 9855146, 504390, 8, 16, 2, 1), (1800, 13283, 13283, 2, 50, 4, 0),
                                      (50000, 99006221, 2148670, 2, 64, 4, 1), (12000, 192533, 40567, 4, 32, 2, 1), (0, 0, 0, 2, 50, 4, 1)]:
        f, g = bench.compulsory_bytes(R, E, U, H, D, b, dedup)
        cb = bench.call_bytes(R, E, U, H, D, b, dedup)
        assert sum(cb.values()) == f + g and cb["fwd"] == f
        assert all(v >= 0 for v in cb.values())
    # SURVEY.md §8(d)'s worked figures for config 4 (realised sizes of this generator): forward 407.2 MB, backward 809.2 MB
    f, g = bench.compulsory_bytes(200000, 9855146, 504390, 8, 16, 2, 1)
    assert abs(f / 1e6 - 407.3) < 0.2 and abs(g / 1e6 - 809.4) < 0.2


def test_gathered_bytes():
    gb = bench.gathered_bytes(1000, 8, 16, 2)
    assert gb["fwd"] == gb["bwd_dst"] == 2 * 1000 * 128 * 2 and gb["bwd_src"] == gb["fwd"] + 8 * 8 * 1000


def test_config_dict_is_the_same_for_both_arms():
    args = argparse.Namespace(config=1, seed=0)
    ws = [W.config1(0)]
    U = ws[0].num_unique_rows()
    c1, comp = bench.config_dict(args, ws, [U])
    c2, _ = bench.config_dict(args, ws, [np.int64(U)])
    assert c1 == c2 and c1["workload"].startswith("config1:") and c1["E"] == ws[0].E and c1["U"] == U
    assert set(c1) == {"workload", "R", "E", "U", "H", "D", "storage", "accumulate", "dedup_mode", "seed", "per_rank", "l2"}
    assert comp == sum(bench.compulsory_bytes(ws[0].R, ws[0].E, U, 2, 50, 4, 0))
