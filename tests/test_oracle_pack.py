"""Pins for oracle fp16 conversions, quantiser (c.1) and bit-plane split.  CPU only."""
import numpy as np
import pytest

import oracle
from paper_2606_23419_b200 import synth
from tests.helpers import np_unpack_codes


# ------------------------------------------------------------------ fp16 conversions vs numpy float16
def test_half_to_float_all_patterns_match_numpy():
    pats = np.arange(65536, dtype=np.uint16)
    ref = pats.view(np.float16).astype(np.float32)
    got = np.array([oracle.half_to_float(int(p)) for p in pats], dtype=np.float32)
    finite = np.isfinite(ref)
    assert np.array_equal(got[finite], ref[finite])
    assert np.array_equal(np.isnan(got), np.isnan(ref))
    assert np.array_equal(np.isinf(got), np.isinf(ref))


def test_float_to_half_roundtrip_identity_for_non_nan():
    pats = np.arange(65536, dtype=np.uint16)
    f = pats.view(np.float16).astype(np.float32)
    for p, v in zip(pats[::7], f[::7]):
        if np.isnan(v):
            continue
        assert oracle.float_to_half(float(v)) == int(p)


def test_float_to_half_rounding_matches_numpy_on_ties_and_random():
    rng = np.random.default_rng(1)
    vals = []
    # exact ties between neighbouring halfs (normal and subnormal), and values one fp32 ulp either side
    for p in list(range(0, 0x7BFF, 37)) + [0, 1, 2, 0x3FF, 0x400, 0x7BFE, 0x7BFF]:
        a = np.uint16(p).view(np.float16).astype(np.float64)
        b = np.uint16(p + 1).view(np.float16).astype(np.float64)
        mid = np.float32((a + b) / 2)
        vals += [mid, np.nextafter(mid, np.float32(0)), np.nextafter(mid, np.float32(1e9))]
    vals += list(rng.standard_normal(2000).astype(np.float32) * np.float32(3.0))
    vals += list((rng.standard_normal(500) * 1e-6).astype(np.float32))
    vals += [np.float32(65519.9), np.float32(65520.0), np.float32(70000.0), np.float32(2.0 ** -25),
             np.float32(2.0 ** -25 * 1.0001), np.float32(2.0 ** -24 * 1.5)]
    vals = np.array(vals, dtype=np.float32)
    vals = np.concatenate([vals, -vals])
    with np.errstate(over="ignore"):
        ref = vals.astype(np.float16).view(np.uint16)
    got = np.array([oracle.float_to_half(float(v)) for v in vals], dtype=np.uint16)
    assert np.array_equal(got, ref)


# ------------------------------------------------------------------ quantiser closed forms
def _ramp_matrix(rng, K=256, N=64, s=2.0 ** -10, z=-0.125):
    """Each (group, column) holds z + s*j for 128 distinct j in 0..255 including 0 and 255:
    s and z are exact in fp16, (max-min)/255 == s exactly -> the quantiser must return q == j."""
    J = np.zeros((K, N), dtype=np.int64)
    for g in range(K // 128):
        for n in range(N):
            mid = rng.choice(np.arange(1, 255), size=126, replace=False)
            j = np.concatenate([[0, 255], mid])
            rng.shuffle(j)
            J[g * 128:(g + 1) * 128, n] = j
    W = (z + s * J).astype(np.float16)
    assert np.array_equal(W.astype(np.float64), z + s * J)  # exactly representable
    return W, J


def test_pack_ramp_groups_closed_form():
    rng = np.random.default_rng(0)
    W, J = _ramp_matrix(rng)
    planes, scales, zeros = oracle.pack(W)
    assert np.all(scales.astype(np.float64) == 2.0 ** -10)
    assert np.all(zeros.astype(np.float64) == -0.125)
    assert np.array_equal(np_unpack_codes(planes), J)        # numpy unpack pins plane order + bit order
    assert np.array_equal(oracle.codes(planes).astype(np.int64), J)


def test_pack_constant_group_and_zero_canonical():
    W = np.full((128, 32), 0.5, dtype=np.float16)
    W[:, 1] = np.float16(-0.0)
    W[::2, 2] = np.float16(0.0)
    W[1::2, 2] = np.float16(-0.0)
    planes, scales, zeros = oracle.pack(W)
    assert np.all(scales.view(np.uint16)[0, :3] == 0)
    assert np.all(planes[:, :, 0] & 0x7 == 0)
    assert zeros[0, 0] == np.float16(0.5)
    assert zeros.view(np.uint16)[0, 1] == 0 and zeros.view(np.uint16)[0, 2] == 0   # zero canonicalised to +0
    w8 = oracle.dequant(planes, scales, zeros, 8)
    assert np.all(w8[:, 0] == 0.5) and np.all(w8[:, 1] == 0.0)


@pytest.mark.parametrize("std,seed", [(0.02, 0), (0.015, 3), (1.0, 5)])
def test_pack_error_bound_and_extremes(std, seed):
    W = synth.make_weights(256, 96, std, seed)
    planes, scales, zeros = oracle.pack(W)
    q = np_unpack_codes(planes)
    s = np.repeat(scales.astype(np.float64), 128, axis=0)
    z = np.repeat(zeros.astype(np.float64), 128, axis=0)
    w = W.astype(np.float64)
    assert np.all(s >= 6.2e-5)  # normal fp16 scales for these distributions
    err = np.abs(w - (s * q + z))
    assert np.all(err <= s / 2 * (1 + 2.0 ** -10))
    # min -> code 0, max -> code >= 254, z is the group minimum
    for g in range(2):
        blk = w[g * 128:(g + 1) * 128]
        qb = q[g * 128:(g + 1) * 128]
        assert np.array_equal(zeros[g].astype(np.float64), blk.min(axis=0))
        assert np.all(qb[blk.argmin(axis=0), np.arange(96)] == 0)
        assert np.all(qb[blk.argmax(axis=0), np.arange(96)] >= 254)
    assert q.min() >= 0 and q.max() <= 255


def test_pack_matches_numpy_minmax_rtn():
    """Cross-implementation: textbook asymmetric min-max RTN written with numpy float32 library ops."""
    W = synth.make_weights(384, 64, 0.02, 11)
    planes, scales, zeros = oracle.pack(W)
    w = W.astype(np.float32).reshape(3, 128, 64)
    lo, hi = w.min(axis=1), w.max(axis=1)
    s = ((hi - lo) / np.float32(255.0)).astype(np.float16)
    t = (w - lo[:, None, :]) / s.astype(np.float32)[:, None, :]
    q = np.clip(np.rint(t), 0, 255).astype(np.int64).reshape(384, 64)
    assert np.array_equal(scales.view(np.uint16), s.view(np.uint16))
    assert np.array_equal(zeros.astype(np.float32), lo)
    assert np.array_equal(np_unpack_codes(planes), q)


def test_nested_property_and_popcounts():
    """the b-bit code is the top b bits of the 8-bit code."""
    W = synth.make_weights(128, 64, 0.02, 2)
    planes, _, _ = oracle.pack(W)
    q8 = np_unpack_codes(planes)
    for b in range(0, 9):
        qb = np_unpack_codes(planes, upto=b)
        assert np.array_equal(qb >> (8 - b) if b else qb, q8 >> (8 - b) if b else np.zeros_like(q8))
        assert np.array_equal(qb, q8 & ((0xFF << (8 - b)) & 0xFF))
    for j in range(8):
        pop = sum(bin(int(v)).count("1") for v in planes[j].reshape(-1))
        assert pop == int(((q8 >> (7 - j)) & 1).sum())


def test_code_prime_error_closed_forms():
    """|q - code'(q,b)| <= 2^(7-b); over all 256 codes MSE_b = (4^(8-b) + 2)/12 (b=1..7), 0 at b=8."""
    q = np.arange(256)
    for b in range(1, 9):
        c = np.array([oracle.code_prime(int(v), b) for v in q])
        e = (q - c).astype(np.float64)
        if b == 8:
            assert np.all(e == 0)
        else:
            assert np.max(np.abs(e)) <= 2 ** (7 - b)
            assert np.isclose(np.mean(e * e), (4.0 ** (8 - b) + 2) / 12)
            assert np.isclose(np.mean(e), -0.5)     # reading #6: phi overshoots the bin centre by 0.5
            # printed equation: q_b * 2^(8-b) + 2^(8-b-1)
            assert np.array_equal(c, (q >> (8 - b)) * 2 ** (8 - b) + 2 ** (8 - b - 1))
    assert all(oracle.code_prime(int(v), 0) == 0 for v in q)
