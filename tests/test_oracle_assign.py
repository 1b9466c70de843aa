"""Pins for the oracle's rank assignment and compacted lists (c.2).  CPU only."""
import os

import numpy as np
import pytest

import oracle
from paper_2606_23419_b200 import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden", "table3_bmax8_rows.txt")


def _table3():
    rows = []
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        f = line.split()
        rows.append((int(f[0]), [float(v) for v in f[1:]]))
    return rows


def test_mix_to_counts_config_mixes_exact():
    # BASELINE.json config 1: {8:25%,4:37.5%,2:25%,0:12.5%} of 256 rows
    c = oracle.mix_to_counts(256, synth.MIXES["4"])
    assert list(c) == [32, 0, 64, 0, 96, 0, 0, 0, 64]
    for name, K in [("2", 4096), ("3", 4096), ("3.25", 12288), ("4", 14336), ("5", 8192), ("8", 28672)]:
        frac = synth.MIXES[name]
        c = oracle.mix_to_counts(K, frac)
        assert int(c.sum()) == K
        assert np.array_equal(c, np.array(frac) * K)      # fractions are multiples of 1/32 -> exact
        assert np.isclose(sum(w * int(c[w]) for w in range(9)) / K, synth.mix_avg_bits(frac))
    assert synth.mix_avg_bits(synth.MIXES["3.25"]) == 3.25   # reading #15
    assert synth.mix_avg_bits(synth.MIXES["3"]) == 3.0


def test_table3_rows_effective_bits():
    """PAPER.md:262-266 Eq. 1: effective bits = sum p_i b_i; Table 3 caption: 2 <= b <= 7 for sampled rows."""
    for K in (4096, 14336, 1000 * 128):
        for row, p in _table3():
            frac = [0.0] * 9
            for i, v in enumerate(p):
                frac[2 * i] = v
            assert abs(sum(p) - 1.0) < 1e-9
            c = oracle.mix_to_counts(K, frac)
            assert int(c.sum()) == K
            eff = sum(w * int(c[w]) for w in range(9)) / K
            target = sum(2 * i * v for i, v in enumerate(p))
            assert abs(eff - target) <= 8.0 * 4.5 / K + 1e-12      # <= half a row per cut, 8 bits each
            if row not in (28, 57, 60):
                assert 2.0 <= target <= 7.0
            # every cumulative cut is within half a row of its fraction
            C = np.cumsum(c[::-1])[::-1]
            F = np.cumsum(np.array(frac)[::-1])[::-1]
            assert np.all(np.abs(C[1:] - F[1:] * K) <= 0.5 + 1e-9)
    assert {r: round(sum(2 * i * v for i, v in enumerate(p)), 2) for r, p in _table3()}[1] == 2.24
    assert {r: sum(2 * i * v for i, v in enumerate(p)) for r, p in _table3()}[60] == 8.0


def test_mix_to_counts_rejects_bad_mix():
    with pytest.raises(ValueError):
        oracle.mix_to_counts(256, [0.5] * 9)
    with pytest.raises(ValueError):
        oracle.mix_to_counts(256, [1.5, -0.5, 0, 0, 0, 0, 0, 0, 0])


def _check_lists(a, K, G=128):
    bu = a["bits_union"].astype(np.int64)
    rows = a["rows"]
    assert np.array_equal(np.sort(rows), np.arange(K))                  # permutation
    w = bu[rows]
    assert np.all(np.diff(w) <= 0)                                      # non-increasing width
    same = np.diff(w) == 0
    assert np.all(np.diff(rows)[same] > 0)                              # ascending index inside a width
    hist = np.bincount(bu, minlength=9)
    assert np.array_equal(a["cnt_ge"][:9], np.cumsum(hist[::-1])[::-1])  # suffix sums
    assert a["cnt_ge"][0] == K and a["cnt_ge"][9] == 0
    for j in range(8):                                                  # prefix = rows needing plane j
        assert set(rows[:a["cnt_ge"][j + 1]].tolist()) == set(np.nonzero(bu > j)[0].tolist())
    for g in range(K // G):
        loc = a["grows"][g * G:(g + 1) * G].astype(np.int64)
        assert np.array_equal(np.sort(loc), np.arange(G))
        wg = bu[g * G + loc]
        assert np.all(np.diff(wg) <= 0)
        assert np.all(np.diff(loc)[np.diff(wg) == 0] > 0)
        hg = np.bincount(bu[g * G:(g + 1) * G], minlength=9)
        assert np.array_equal(a["gcnt_ge"][g, :9], np.cumsum(hg[::-1])[::-1])
        assert np.all(a["gcnt_ge"][g, 9:] == 0)


@pytest.mark.parametrize("K,mix,seed", [(256, "4", 0), (1024, "2", 1), (4096, "3.25", 2), (1536, "5", 3)])
def test_assign_invariants_and_bruteforce_rank(K, mix, seed):
    x = synth.make_x(1, K, seed, "student_t")
    x[0, 5:9] = x[0, 4]                       # force ties
    x[0, 100] = np.float16(-0.0)
    x[0, 101] = np.float16(0.0)
    counts = oracle.mix_to_counts(K, synth.MIXES[mix])
    a = oracle.assign(x, counts)
    b = a["bits"][0].astype(np.int64)
    assert np.array_equal(np.bincount(b, minlength=9), counts)           # histogram == counts
    m = (x.view(np.uint16)[0] & 0x7FFF).astype(np.int64)
    order = np.lexsort((np.arange(K), -m))                               # numpy library sort: (m desc, k asc)
    assert np.all(np.diff(b[order]) <= 0)                                # larger |x| never gets fewer bits
    r = oracle.rank_bruteforce(x)                                        # O(K^2) definition
    assert np.array_equal(np.argsort(r, kind="stable"), order)
    C = np.cumsum(counts[::-1])[::-1]                                    # C_w
    expect = np.array([max([w for w in range(1, 9) if rk < C[w]], default=0) for rk in r])
    assert np.array_equal(b, expect)
    assert np.array_equal(a["bits_union"], a["bits"][0])
    _check_lists(a, K)


def test_assign_all_equal_is_index_order():
    K = 512
    x = np.full((1, K), 1.5, dtype=np.float16)
    x[0, ::2] *= -1                                                       # sign must not matter
    counts = oracle.mix_to_counts(K, synth.MIXES["4"])
    a = oracle.assign(x, counts)
    expect = np.concatenate([np.full(counts[w], w) for w in range(8, -1, -1)])
    assert np.array_equal(a["bits"][0], expect)
    assert np.array_equal(a["rows"], np.arange(K))


def test_assign_tiny_config_outliers_get_8_bits():
    W, x, mix = synth.tiny_config(0)
    counts = oracle.mix_to_counts(256, mix)
    a = oracle.assign(x, counts)
    top4 = np.argsort(-np.abs(x[0].astype(np.float32)))[:4]
    assert np.all(a["bits"][0][top4] == 8)
    assert sum(w * int(c) for w, c in enumerate(counts)) / 256 == 4.0


def test_assign_inf_sorts_above_finite_and_zero_last():
    K = 256
    x = synth.make_x(1, K, 9)
    x[0, 17] = np.float16(np.inf)
    x[0, 200] = np.float16(0.0)
    counts = np.array([1, 0, 0, 0, 0, 0, 0, 0, K - 1], dtype=np.uint32)   # exactly one row dropped
    a = oracle.assign(x, counts)
    assert a["bits"][0][17] == 8 and a["bits"][0][200] == 0


def test_assign_multi_token_union():
    K, T = 1024, 4
    x = synth.make_x(T, K, 4, "student_t")
    counts = oracle.mix_to_counts(K, synth.MIXES["4"])
    a = oracle.assign(x, counts)
    for t in range(T):
        solo = oracle.assign(x[t:t + 1], counts)
        assert np.array_equal(a["bits"][t], solo["bits"][0])               # tokens are independent
    assert np.array_equal(a["bits_union"], a["bits"].max(axis=0))
    _check_lists(a, K)
    assert a["bits_union"].mean() > 4.0                                    # union fetches more than one token
