"""Pins for the threshold form of the assignment and its calibration (Eq. 2).
The rank form `oracle.assign` is pinned in test_oracle_assign.py; here the threshold oracle is tied to it, to
closed forms and to plain numpy counts."""
import numpy as np
import pytest

import oracle
from paper_2606_23419_b200 import synth


def _mag(x):
    return np.ascontiguousarray(x).view(np.uint16) & 0x7FFF


def test_calibration_closed_form():
    """two vectors whose level-separating magnitudes are 1.0 / 3.0 (8-bit cut) and 0.25 / 0.75 (4-bit cut):
    theta = their means 2.0 and 0.5, exactly representable; unused widths inherit the cut of the next used one"""
    K = 256
    counts = np.zeros(9, np.uint32)
    counts[8], counts[4], counts[0] = 64, 64, 128
    xs = np.zeros((2, K), np.float16)
    for s, (hi, lo) in enumerate([(1.0, 0.25), (3.0, 0.75)]):
        xs[s, :64] = hi * (1 + np.arange(64)[::-1] / 64.0)     # 64 largest, the smallest of them is exactly hi
        xs[s, 64:128] = lo * (1 + np.arange(64)[::-1] / 64.0)   # next 64, the smallest is lo
        xs[s, 128:] = lo / 4
        xs[s] *= np.where(np.arange(K) % 2, -1, 1)              # signs must not matter
    theta = oracle.calibrate_thresholds(xs, counts)
    f = theta.view(np.float16)
    assert all(f[w] == np.float16(2.0) for w in (5, 6, 7, 8)) and all(f[w] == np.float16(0.5) for w in (1, 2, 3, 4))
    counts2 = counts.copy()
    counts2[8], counts2[4] = 0, 128                             # no 8-bit level: widths 5..8 unreachable
    theta2 = oracle.calibrate_thresholds(xs, counts2)
    assert all(theta2[w] == 0x8000 for w in (5, 6, 7, 8))


@pytest.mark.parametrize("K,mix,seed", [(1024, "4", 0), (4096, "2", 1), (2048, "3.25", 2)])
def test_self_calibrated_thresholds_reproduce_the_rank_partition_up_to_ties(K, mix, seed):
    x = synth.make_x(1, K, seed, "student_t")
    counts = oracle.mix_to_counts(K, synth.MIXES[mix])
    theta = oracle.calibrate_thresholds(x, counts)
    a, r = oracle.assign_thresholds(x, theta), oracle.assign(x, counts)
    m = _mag(x)[0]
    diff = a["bits"][0] != r["bits"][0]
    # only keys exactly equal to a threshold may differ (the rank form breaks ties by index), and only upwards
    assert np.all(np.isin(m[diff], theta[1:]))
    assert np.all(a["bits"][0][diff] > r["bits"][0][diff])
    assert diff.sum() < 16


def test_threshold_widths_are_plain_counts_and_lists_are_consistent():
    T, K = 3, 1536
    x = synth.make_x(T, K, 9, "normal")
    theta = np.array([0, 0x2000, 0x2000, 0x3000, 0x3400, 0x3800, 0x3C00, 0x4000, 0x8000], np.uint16)
    a = oracle.assign_thresholds(x, theta)
    m = _mag(x)
    expect = sum((m >= int(theta[w])).astype(np.uint8) for w in range(1, 9))
    assert np.array_equal(a["bits"], expect)
    assert a["bits"].max() <= 7                                  # width 8 is unreachable (0x8000)
    assert np.array_equal(a["bits_union"], a["bits"].max(axis=0))
    rows = a["rows"]
    assert np.array_equal(np.sort(rows), np.arange(K))
    bu = a["bits_union"][rows]
    assert np.all(bu[:-1] >= bu[1:])
    same = bu[:-1] == bu[1:]
    assert np.all(rows[1:][same] > rows[:-1][same])
    assert np.array_equal(a["cnt_ge"], [(a["bits_union"] >= w).sum() for w in range(10)])


def test_threshold_extremes_and_monotonicity_check():
    K = 256
    x = synth.make_x(1, K, 4)
    assert np.all(oracle.assign_thresholds(x, np.zeros(9, np.uint16))["bits"] == 8)
    assert np.all(oracle.assign_thresholds(x, np.full(9, 0x8000, np.uint16))["bits"] == 0)
    bad = np.array([0, 0x3C00, 0x3800, 0x3C00, 0x3C00, 0x3C00, 0x3C00, 0x3C00, 0x3C00], np.uint16)
    with pytest.raises(ValueError):
        oracle.assign_thresholds(x, bad)
