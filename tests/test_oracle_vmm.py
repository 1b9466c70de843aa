"""Pins for the oracle VMM (c.3): reductions to library routines, the printed equation, brute force."""
import itertools

import numpy as np
import pytest

import oracle
from paper_2606_23419_b200 import synth
from tests.helpers import np_unpack_codes, paper_w_hat, rel_l2


def _setup(K=256, N=64, seed=0, T=1, mix="4"):
    W = synth.make_weights(K, N, 0.02, seed)
    x = synth.make_x(T, K, seed, "normal", n_outliers=4)
    planes, s, z = oracle.pack(W)
    counts = oracle.mix_to_counts(K, synth.MIXES[mix])
    a = oracle.assign(x, counts)
    return W, x, planes, s, z, a


def test_all_8_bit_equals_dense_gemv_on_dequantised_weights():
    W, x, planes, s, z, _ = _setup()
    K = x.shape[1]
    q = np_unpack_codes(planes)
    w_hat = np.repeat(s.astype(np.float64), 128, 0) * q + np.repeat(z.astype(np.float64), 128, 0)
    ref = x.astype(np.float64) @ w_hat                                      # numpy matmul
    y = oracle.vmm(x, planes, s, z, np.full((1, K), 8, np.uint8))
    assert rel_l2(y, ref) < 1e-13
    # and 8-bit dequant is within s/2 of the fp16 weights -> close to the unquantised GEMV
    ref16 = x.astype(np.float64) @ W.astype(np.float64)
    assert rel_l2(y, ref16) < 2e-2


def test_all_0_bit_is_exactly_zero():
    _, x, planes, s, z, _ = _setup()
    y = oracle.vmm(x, planes, s, z, np.zeros((1, x.shape[1]), np.uint8))
    assert np.all(y == 0.0)
    assert np.all(oracle.vmm_planewise(x, planes, s, z, np.zeros((1, x.shape[1]), np.uint8)) == 0.0)


@pytest.mark.parametrize("b", range(0, 9))
def test_one_hot_returns_printed_reconstruction(b):
    """x = e_k returns row k of w_hat = s (q_b 2^(8-b) + 2^(8-b-1)) + z."""
    _, _, planes, s, z, _ = _setup(seed=3)
    K, N = 256, 64
    q8 = np_unpack_codes(planes)
    for k in (0, 127, 128, 255):
        x = np.zeros((1, K), np.float16)
        x[0, k] = 1.0
        bits = np.zeros((1, K), np.uint8)
        bits[0, k] = b
        y = oracle.vmm(x, planes, s, z, bits)
        g = k // 128
        expect = paper_w_hat(q8[k], s[g], z[g], b)
        assert np.allclose(y[0], expect, rtol=0, atol=1e-15)
    w = oracle.dequant(planes, s, z, b)
    assert np.allclose(w, paper_w_hat(q8, np.repeat(s, 128, 0), np.repeat(z, 128, 0), b), rtol=0, atol=1e-15)


def test_mixed_assignment_equals_numpy_formula_and_planewise():
    _, x, planes, s, z, a = _setup(K=384, N=96, seed=5)
    bits = a["bits"]
    q8 = np_unpack_codes(planes)
    S, Z = np.repeat(s, 128, 0), np.repeat(z, 128, 0)
    w_mixed = np.zeros(q8.shape)
    for b in range(9):
        sel = bits[0] == b
        w_mixed[sel] = paper_w_hat(q8[sel], S[sel], Z[sel], b)
    ref = x.astype(np.float64) @ w_mixed
    y1 = oracle.vmm(x, planes, s, z, bits)
    y2 = oracle.vmm_planewise(x, planes, s, z, bits)
    assert rel_l2(y1, ref) < 1e-13
    assert rel_l2(y2, y1) < 1e-12
    cols = np.array([0, 5, 31, 32, 95], np.int32)
    assert np.array_equal(oracle.vmm(x, planes, s, z, bits, cols=cols)[0], y1[0, cols])


def test_linearity_in_x():
    _, x, planes, s, z, a = _setup(seed=7)
    bits = a["bits"]
    x1, x2 = x.copy(), x.copy()
    x1[0, ::2] = 0
    x2[0, 1::2] = 0                                                          # disjoint support: x1 + x2 == x exactly
    y = oracle.vmm(x, planes, s, z, bits)
    y12 = oracle.vmm(x1, planes, s, z, bits) + oracle.vmm(x2, planes, s, z, bits)
    assert rel_l2(y12, y) < 1e-13
    x3 = (x.astype(np.float32) * 2).astype(np.float16)                       # exact doubling
    assert rel_l2(oracle.vmm(x3, planes, s, z, bits), 2 * y) < 1e-15


def test_bruteforce_all_assignments_tiny():
    """All 9^4 assignments on K=4, N=32, G=4: definition == plane-wise == numpy evaluation of PAPER.md:85."""
    rng = np.random.default_rng(0)
    K, N, G = 4, 32, 4
    W = (rng.standard_normal((K, N)) * 0.05).astype(np.float16)
    x = np.array([[1.5, -0.375, 2.25, -3.0]], np.float16)
    planes, s, z = oracle.pack(W, G=G)
    q8 = np_unpack_codes(planes)
    xd = x.astype(np.float64)[0]
    for combo in itertools.product(range(9), repeat=K):
        bits = np.array([combo], np.uint8)
        y1 = oracle.vmm(x, planes, s, z, bits, G=G)[0]
        y2 = oracle.vmm_planewise(x, planes, s, z, bits, G=G)[0]
        ref = np.zeros(N)
        for k, b in enumerate(combo):
            ref += xd[k] * paper_w_hat(q8[k], s[0], z[0], b)
        scale = np.abs(ref).max() + 1e-30
        assert np.max(np.abs(y1 - ref)) <= 1e-13 * scale + 1e-18
        assert np.max(np.abs(y2 - y1)) <= 1e-12 * scale + 1e-18


def test_truncation_bound_and_error_shrinks_with_bits():
    """|y_b - y_8| <= sum_{b_k>=1} |x_k| s 2^(7-b_k) + sum_{b_k=0} |x_k w8_kn|; aggregate error falls with bits."""
    _, x, planes, s, z, _ = _setup(K=512, N=64, seed=8)
    K = 512
    y8 = oracle.vmm(x, planes, s, z, np.full((1, K), 8, np.uint8))
    w8 = oracle.dequant(planes, s, z, 8)
    S = np.repeat(s.astype(np.float64), 128, 0)
    ax = np.abs(x.astype(np.float64))[0]
    errs = []
    for name in ["2", "3", "4", "5"]:
        bits = oracle.assign(x, oracle.mix_to_counts(K, synth.MIXES[name]))["bits"]
        yb = oracle.vmm(x, planes, s, z, bits)
        b = bits[0].astype(np.int64)
        bound = (ax[:, None] * S * np.where(b >= 1, 2.0 ** (7 - b), 0.0)[:, None]).sum(0) \
            + (ax[:, None] * np.abs(w8) * (b == 0)[:, None]).sum(0)
        assert np.all(np.abs(yb - y8)[0] <= bound * (1 + 1e-12) + 1e-15)
        errs.append(rel_l2(yb, y8))
    assert errs[0] > errs[1] > errs[2] > errs[3]
    # uniform widths: error non-increasing in b on aggregate
    e = [rel_l2(oracle.vmm(x, planes, s, z, np.full((1, K), b, np.uint8)), y8) for b in range(1, 9)]
    assert all(e[i] >= e[i + 1] for i in range(7)) and e[-1] == 0.0


def test_multi_token_equals_independent_tokens():
    _, x, planes, s, z, a = _setup(K=256, N=64, seed=9, T=4)
    y = oracle.vmm(x, planes, s, z, a["bits"])
    for t in range(4):
        yt = oracle.vmm(x[t:t + 1], planes, s, z, a["bits"][t:t + 1])
        assert np.array_equal(y[t], yt[0])
