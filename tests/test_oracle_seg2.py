"""Pins of the oracle's 2-bit-segment store (SURVEY.md 8f2; PAPER.md:79-81 segments, :85 reconstruction with the store's
own b_max, :95 b_max in {4, 6, 8}, :442 sixteen 2-bit chunks per uint32).  Each pin is something other than the oracle
itself: an independent numpy unpacker / quantiser, closed forms, the printed equation, and — for b_max = 8 — the 1-bit
plane store of the same weights, which must agree exactly wherever both are defined."""
import numpy as np
import pytest

import oracle
from paper_2606_23419_b200 import synth


def np_codes_from_segs(segs, bmax, upto_segments=None):
    """independent numpy unpacker: column n's pair of segment sigma sits at bits 2 (n & 15) + {1, 0} of word n >> 4"""
    nseg, K, words = segs.shape
    n = np.arange(words * 16)
    q = np.zeros((K, words * 16), np.int64)
    for sg in range(nseg if upto_segments is None else upto_segments):
        pair = (segs[sg][:, n >> 4] >> (2 * (n & 15)).astype(np.uint32)) & 3
        q |= pair.astype(np.int64) << (bmax - 2 - 2 * sg)
    return q


def np_rtn(W, bmax, G=128):
    """textbook asymmetric min-max RTN with 2^bmax - 1 steps, fp32 ops, fp16 scale, quantised against the stored scale"""
    K, N = W.shape
    Wf = W.astype(np.float32).reshape(K // G, G, N)
    lo, hi = Wf.min(1), Wf.max(1)
    s16 = ((hi - lo) / np.float32((1 << bmax) - 1)).astype(np.float16)
    s = s16.astype(np.float32)
    with np.errstate(divide="ignore", invalid="ignore"):
        t = (Wf - lo[:, None, :]) / s[:, None, :]
    q = np.where(s[:, None, :] != 0, np.clip(np.rint(t), 0, (1 << bmax) - 1), 0).astype(np.int64)
    return q.reshape(K, N), s16, lo.astype(np.float16)


@pytest.mark.parametrize("bmax", [4, 6, 8])
def test_pack2_codes_equal_independent_rtn_and_round_trip(bmax):
    W = synth.make_weights(256, 96, 0.02, 10 + bmax)
    W[:128, 0] = np.float16(0.25)                       # constant group -> s = 0, codes 0
    segs, s, z = oracle.pack2(W, bmax)
    q_ref, s_ref, z_ref = np_rtn(W, bmax)
    assert np.array_equal(np_codes_from_segs(segs, bmax), q_ref)
    assert np.array_equal(oracle.codes2(segs, bmax), q_ref)
    assert np.array_equal(s.view(np.uint16), s_ref.view(np.uint16))
    assert np.array_equal(z.astype(np.float32), z_ref.astype(np.float32))
    assert q_ref.min() == 0 and q_ref.max() == (1 << bmax) - 1 and not q_ref[:128, 0].any()
    err = np.abs(W.astype(np.float64) - (s.astype(np.float64).repeat(128, 0) * q_ref + z.astype(np.float64).repeat(128, 0)))
    assert np.all(err <= s.astype(np.float64).repeat(128, 0) / 2 * (1 + 2 ** -9) + 1e-12)   # RTN error bound


@pytest.mark.parametrize("bmax", [4, 6, 8])
def test_nested_property_per_segment(bmax):
    """the b-bit code is the top b bits of the b_max-bit code — here: the first b/2 segments"""
    W = synth.make_weights(128, 64, 0.02, 3)
    segs, _, _ = oracle.pack2(W, bmax)
    q = np_codes_from_segs(segs, bmax)
    for b in range(0, bmax + 1, 2):
        top = np_codes_from_segs(segs, bmax, b // 2)
        assert np.array_equal(top, (q >> (bmax - b)) << (bmax - b))


def test_bmax8_segments_are_pairs_of_the_one_bit_planes():
    """b_max = 8: same quantiser as the 1-bit store, segment sigma = planes 2 sigma (high bit) and 2 sigma + 1"""
    W = synth.make_weights(256, 64, 0.02, 5)
    planes, s1, z1 = oracle.pack(W)
    segs, s2, z2 = oracle.pack2(W, 8)
    assert np.array_equal(s1.view(np.uint16), s2.view(np.uint16)) and np.array_equal(z1.view(np.uint16), z2.view(np.uint16))
    n = np.arange(64)
    for sg in range(4):
        hi = (planes[2 * sg][:, n >> 5] >> (n & 31).astype(np.uint32)) & 1
        lo = (planes[2 * sg + 1][:, n >> 5] >> (n & 31).astype(np.uint32)) & 1
        pair = (segs[sg][:, n >> 4] >> (2 * (n & 15)).astype(np.uint32)) & 3
        assert np.array_equal(pair, 2 * hi + lo)


@pytest.mark.parametrize("bmax", [4, 6, 8])
def test_code2_prime_closed_forms(bmax):
    """|q - code'| <= 2^(bmax-b-1); MSE over all codes = (4^d + 2) / 12 with d = bmax - b (0 at b = bmax); the value is
    the printed equation q_b 2^(bmax-b) + 2^(bmax-b-1)"""
    qs = np.arange(1 << bmax)
    for b in range(2, bmax + 1, 2):
        cp = np.array([oracle.code2_prime(int(q), b, bmax) for q in qs])
        d = bmax - b
        if d == 0:
            assert np.array_equal(cp, qs)
            continue
        assert np.array_equal(cp, (qs >> d) * (1 << d) + (1 << (d - 1)))
        assert np.abs(qs - cp).max() <= 1 << (d - 1)
        assert abs(np.mean((qs - cp) ** 2.0) - (4.0 ** d + 2) / 12) < 1e-9
    assert oracle.code2_prime(13, 0, bmax) == 0


@pytest.mark.parametrize("bmax", [4, 6, 8])
def test_vmm2_special_cases(bmax):
    K, N = 256, 48
    W = synth.make_weights(K, N, 0.02, 20 + bmax)
    x = synth.make_x(2, K, 21, "student_t")
    segs, s, z = oracle.pack2(W, bmax)
    q = np_codes_from_segs(segs, bmax).astype(np.float64)
    sf, zf = s.astype(np.float64).repeat(128, 0), z.astype(np.float64).repeat(128, 0)
    full = np.full((2, K), bmax, np.uint8)
    y = oracle.vmm2(x, segs, s, z, full, bmax)
    assert np.allclose(y, x.astype(np.float64) @ (sf * q + zf), rtol=1e-12, atol=1e-12)   # all-bmax = dense GEMV
    assert not oracle.vmm2(x, segs, s, z, np.zeros((2, K), np.uint8), bmax).any()          # all-0 = 0
    for k, b in [(0, bmax), (127, 2), (200, bmax - 2)]:                                    # one-hot = the printed row
        xo = np.zeros((1, K), np.float16)
        xo[0, k] = 1.0
        bits = np.zeros((1, K), np.uint8)
        bits[0, k] = b
        d = bmax - b
        qk = np_codes_from_segs(segs, bmax)[k]
        row = sf[k] * ((qk >> d) * 2.0 ** d + (2.0 ** (d - 1) if d else 0.0)) + zf[k]
        assert np.allclose(oracle.vmm2(xo, segs, s, z, bits, bmax)[0], row, rtol=1e-12, atol=1e-15)
        assert np.allclose(oracle.dequant2(segs, s, z, bmax, b)[k], row, rtol=1e-12, atol=1e-15)
    with pytest.raises(ValueError):
        oracle.vmm2(x, segs, s, z, np.full((2, K), 3, np.uint8), bmax)                     # odd widths do not exist


def test_vmm2_bmax8_equals_the_plane_store_on_even_widths():
    """two stores, two code paths, one definition: with b_max = 8 and even widths the results are identical"""
    K, N = 384, 64
    W = synth.make_weights(K, N, 0.02, 31)
    x = synth.make_x(3, K, 32, "student_t")
    counts = oracle.mix_to_counts(K, [0.1, 0, 0.2, 0, 0.3, 0, 0.15, 0, 0.25])
    bits = oracle.assign(x, counts)["bits"]
    y1 = oracle.vmm(x, *oracle.pack(W), bits)
    y2 = oracle.vmm2(x, *oracle.pack2(W, 8), bits, 8)
    assert np.array_equal(y1, y2)
