"""The seeded inputs are pinned by hash: every rank, both bench arms and every parity test read these very arrays."""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.join(HERE, "golden"))

import make_window_hashes  # noqa: E402


def test_window_arrays_match_recorded_sha256():
    with open(os.path.join(HERE, "golden", "window_sha256.txt")) as fh:
        recorded = [l.strip() for l in fh if l.strip()]
    assert recorded == make_window_hashes.lines()


def test_rank_window_sets_differ_and_set0_is_the_config():
    import numpy as np
    from paper_2602_15605_b200 import shard, windows
    base = windows.config(3, lmax=50)
    s0 = windows.pol_windows(50, (0.4, 80.0, 2.0), (0.35, 100.0, 2.4), 0.05, shard.window_seed(3, 0))
    s1 = windows.pol_windows(50, (0.4, 80.0, 2.0), (0.35, 100.0, 2.4), 0.05, shard.window_seed(3, 1))
    assert np.array_equal(s0[0], base.Wtt) and np.array_equal(s0[2], base.Wpp)
    assert not np.array_equal(s1[0], base.Wtt)
