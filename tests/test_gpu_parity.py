"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.
Bit-exact on planes / scales / zeros / bits / lists; y within 1e-3 relative L2 per token (north_star)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_23419_b200 import synth
from tests.helpers import expected_gsched, rel_l2

pytestmark = pytest.mark.gpu
TOL = 1e-3


@pytest.fixture(scope="module")
def gq():
    from paper_2606_23419_b200 import binding
    return binding


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _check_y(y, y_ref, what=""):
    """north_star: <= 1e-3 relative L2 per token.  On top of it an ELEMENT-WISE bound, so that a single wrong column
    cannot hide inside the norm: the fp16 x fp16 products are exact and only the fp32 summation order differs from the
    fp64 oracle, so every output is within ~sqrt(K) * 2^-24 of the scale of the sum (measured 1e-7): 1e-5 * max|y| + 1e-6."""
    y = np.asarray(y, np.float64)
    y_ref = np.asarray(y_ref, np.float64)
    if y.ndim == 1:
        y, y_ref = y[None], y_ref[None]
    for t in range(y.shape[0]):
        n = np.linalg.norm(y_ref[t])
        assert np.linalg.norm(y[t] - y_ref[t]) <= TOL * n + 1e-6, (what, t, rel_l2(y[t], y_ref[t]))
        bound = 1e-5 * np.abs(y_ref[t]).max() + 1e-6
        worst = np.abs(y[t] - y_ref[t]).max()
        assert worst <= bound, (what, t, worst, bound, int(np.abs(y[t] - y_ref[t]).argmax()))


def _pack_both(gq, W):
    ref = oracle.pack(W)
    out = gq.grinqh_pack(_dev(W))
    torch.cuda.synchronize()
    return ref, out


def _check_pack(ref, out):
    planes, s, z = ref
    assert np.array_equal(out.planes.cpu().numpy().view(np.uint32), planes)
    assert np.array_equal(out.scales.cpu().numpy().view(np.uint16), s.view(np.uint16))
    assert np.array_equal(out.zeros.cpu().numpy().view(np.uint16), z.view(np.uint16))


def _check_assign(ref, a, x):
    assert np.array_equal(a.gsched.cpu().numpy().view(np.uint32), expected_gsched(ref, x))
    assert np.array_equal(a.bits.cpu().numpy(), ref["bits"])
    assert np.array_equal(a.bits_union.cpu().numpy(), ref["bits_union"])
    assert np.array_equal(a.rows.cpu().numpy(), ref["rows"])
    assert np.array_equal(a.cnt_ge.cpu().numpy()[:10], ref["cnt_ge"])
    assert np.array_equal(a.grows.cpu().numpy(), ref["grows"])
    assert np.array_equal(a.gcnt_ge.cpu().numpy(), ref["gcnt_ge"])


@pytest.mark.parametrize("K,N,std,seed", [(256, 512, 0.02, 0), (384, 1056, 0.02, 1), (1024, 96, 0.015, 2),
                                          (128, 32, 1.0, 3)])
def test_pack_bit_exact(gq, K, N, std, seed):
    W = synth.make_weights(K, N, std, seed)
    ref, out = _pack_both(gq, W)
    _check_pack(ref, out)


def test_pack_edge_values(gq):
    """constant groups (s = 0), signed zeros, a subnormal scale, large dynamic range"""
    rng = np.random.default_rng(5)
    W = synth.make_weights(256, 64, 0.02, 7)
    W[:128, 0] = np.float16(0.25)
    W[:128, 1] = np.float16(-0.0)
    W[:128:2, 2] = np.float16(0.0)
    W[1:128:2, 2] = np.float16(-0.0)
    W[:128, 3] = (rng.integers(0, 40, 128) * 2.0 ** -24).astype(np.float16)      # subnormal range -> tiny scale
    W[128:, 4] = (rng.standard_normal(128) * 3000).astype(np.float16)
    W[128:, 5] = np.float16(65504.0) * np.where(rng.random(128) < 0.5, 1, -1).astype(np.float16)
    ref, out = _pack_both(gq, W)
    _check_pack(ref, out)


@pytest.mark.parametrize("T,K,mix,dist,seed", [
    (1, 256, "4", "normal", 0), (1, 4096, "2", "student_t", 1), (1, 12288, "3.25", "normal", 2),
    (2, 8192, "3", "student_t", 3), (4, 28672, "4", "student_t", 4), (1, 14336, "5", "normal", 5),
    (1, 4096, "8", "normal", 6), (1, 4096, "0", "normal", 7), (3, 1536, "4", "normal", 8)])
def test_assign_bit_exact(gq, T, K, mix, dist, seed):
    x = synth.make_x(T, K, seed, dist)
    counts = oracle.mix_to_counts(K, synth.MIXES[mix])
    assert gq.grinqh_mix_to_counts(K, synth.MIXES[mix]) == list(counts)
    ref = oracle.assign(x, counts)
    a = gq.grinqh_assign(_dev(x), counts)
    torch.cuda.synchronize()
    _check_assign(ref, a, x)


def test_assign_ties_and_degenerate_inputs(gq):
    K = 2048
    rng = np.random.default_rng(0)
    cases = []
    cases.append(np.full((1, K), 1.5, np.float16))                                  # all equal
    cases.append(np.zeros((1, K), np.float16))                                      # all zero
    x = rng.integers(-3, 4, (2, K)).astype(np.float16)                              # 4 distinct magnitudes
    x[0, 7] = np.float16(-0.0)
    cases.append(x)
    x = synth.make_x(1, K, 3)
    x[0, 100:600] = x[0, 99]                                                        # a tie run across a cut
    x[0, 17] = np.float16(np.inf)
    cases.append(x)
    frac_odd = [0.11, 0.09, 0.13, 0.07, 0.2, 0.1, 0.1, 0.05, 0.15]                  # all nine widths present
    for x in cases:
        for frac in (synth.MIXES["4"], synth.MIXES["2"], frac_odd):
            counts = oracle.mix_to_counts(K, frac)
            ref = oracle.assign(x, counts)
            a = gq.grinqh_assign(_dev(x), counts)
            torch.cuda.synchronize()
            _check_assign(ref, a, x)


def _run_vmm(gq, W, x, frac):
    K, N = W.shape
    counts = oracle.mix_to_counts(K, frac)
    planes, s, z = oracle.pack(W)
    ref_a = oracle.assign(x, counts)
    y_ref = oracle.vmm(x, planes, s, z, ref_a["bits"])
    xd = _dev(x)
    w = gq.grinqh_pack(_dev(W))
    a = gq.grinqh_assign(xd, counts)
    y = gq.grinqh_vmm(w, a)
    y_rank = gq.grinqh_vmm_rank(xd, counts, w)      # the assignment made inside the launch: the same bits
    torch.cuda.synchronize()
    assert np.array_equal(y.cpu().numpy(), y_rank.cpu().numpy())
    return y.cpu().numpy(), y_ref


def test_vmm_tiny_config(gq):
    """BASELINE.json configs[0]"""
    W, x, frac = synth.tiny_config(0)
    y, y_ref = _run_vmm(gq, W, x, frac)
    _check_y(y, y_ref)


@pytest.mark.parametrize("K,N,mix,T,dist,seed", [
    (512, 2080, "4", 1, "normal", 1),        # several column tiles + ragged tail (2080 = 2*1024 + 32)
    (1024, 1024, "2", 1, "student_t", 2),
    (1024, 1056, "3.25", 1, "normal", 3),
    (768, 4096, "5", 1, "student_t", 4),
    (512, 1024, "8", 1, "normal", 5),
    (512, 1024, "0", 1, "normal", 6),
    (512, 1536, "4", 2, "student_t", 7),
    (512, 1056, "4", 4, "student_t", 8),
    (256, 96, "3", 3, "normal", 9),
])
def test_vmm_matches_oracle(gq, K, N, mix, T, dist, seed):
    W = synth.make_weights(K, N, 0.02, seed)
    x = synth.make_x(T, K, seed, dist)
    y, y_ref = _run_vmm(gq, W, x, synth.MIXES[mix])
    if mix == "0":
        assert np.all(y == 0.0) and np.all(y_ref == 0.0)
        return
    _check_y(y, y_ref)


def test_vmm_all_nine_widths_and_small_x(gq):
    K, N = 1024, 1056
    W = synth.make_weights(K, N, 0.02, 21)
    frac = [0.11, 0.09, 0.13, 0.07, 0.2, 0.1, 0.1, 0.05, 0.15]
    for scale in (1.0, 1e-4):                       # tiny activations: subnormal halfs must not be flushed
        x = (synth.make_x(2, K, 22).astype(np.float32) * scale).astype(np.float16)
        y, y_ref = _run_vmm(gq, W, x, frac)
        _check_y(y, y_ref, scale)


def test_vmm_one_hot_and_determinism(gq):
    K, N = 256, 1056
    W = synth.make_weights(K, N, 0.02, 31)
    planes, s, z = oracle.pack(W)
    w = gq.grinqh_pack(_dev(W))
    for k, b in [(0, 8), (127, 4), (128, 2), (255, 1), (5, 7)]:
        x = np.zeros((1, K), np.float16)
        x[0, k] = 1.0
        counts = np.zeros(9, np.uint32)
        counts[b] = 1
        counts[0] = K - 1
        a = gq.grinqh_assign(_dev(x), counts)
        y = gq.grinqh_vmm(w, a).cpu().numpy()
        y_ref = oracle.dequant(planes, s, z, b)[k]
        assert np.allclose(y[0], y_ref, rtol=1e-6, atol=1e-9)
    x = synth.make_x(1, K, 32)
    counts = oracle.mix_to_counts(K, synth.MIXES["4"])
    xd = _dev(x)
    a = gq.grinqh_assign(xd, counts)
    y1 = gq.grinqh_vmm(w, a).cpu().numpy()
    y2 = gq.grinqh_vmm(w, a).cpu().numpy()
    assert np.array_equal(y1, y2)                   # deterministic split-K


FULL_SIZE = [
    # BASELINE.json configs[1] (Llama-3-8B layer) in the launch shapes bench.py times (q|k|v, o, gate|up, down) + one gate
    (4096, 6144, 1, "4", "normal", 0.02), (4096, 4096, 1, "4", "normal", 0.02), (4096, 28672, 1, "4", "normal", 0.02),
    (14336, 4096, 1, "4", "normal", 0.02), (4096, 14336, 1, "4", "normal", 0.02),
    # configs[2] (Qwen3-8B sweep): the shapes config 2 does not have, at other mixes
    (4096, 12288, 1, "2", "normal", 0.02), (12288, 4096, 1, "5", "normal", 0.02), (4096, 1024, 1, "3.25", "normal", 0.02),
    # configs[4] (Llama-3-70B), 1 / 2 / 4 tokens, heavy-tailed x
    (8192, 8192, 1, "3", "student_t", 0.015), (8192, 8192, 4, "4", "student_t", 0.015),
    (8192, 1024, 2, "4", "student_t", 0.015), (8192, 28672, 2, "2", "student_t", 0.015),
    (8192, 28672, 1, "4", "student_t", 0.015), (28672, 8192, 4, "3", "student_t", 0.015),
    (28672, 8192, 1, "4", "student_t", 0.015),
]


@pytest.mark.parametrize("K,N,T,mix,dist,std", FULL_SIZE)
def test_full_size_layer_sampled_columns(gq, K, N, T, mix, dist, std):
    """BASELINE.json configs 2, 3 and 5 at full size, in the launch configurations bench.py times; the oracle
    recomputes a sample of output columns one by one (columns are independent).  Three forms of the same product:
    rank assignment inside the launch (the bench headline), grinqh_assign + grinqh_vmm (bit-identical), and the
    threshold assignment inside the launch."""
    g = torch.Generator(device="cuda")
    g.manual_seed(1234 + K + N)
    Wd = (torch.randn((K, N), generator=g, device="cuda", dtype=torch.float32) * std).to(torch.float16)
    x = synth.make_x(T, K, 77, dist)
    counts = oracle.mix_to_counts(K, synth.MIXES[mix])
    xd = _dev(x)
    w = gq.grinqh_pack(Wd)
    a = gq.grinqh_assign(xd, counts)
    y = gq.grinqh_vmm(w, a)
    y_rank = gq.grinqh_vmm_rank(xd, counts, w)
    torch.cuda.synchronize()
    ref_a = oracle.assign(x, counts)
    _check_assign(ref_a, a, x)
    assert np.array_equal(y.cpu().numpy(), y_rank.cpu().numpy())
    cols = np.unique(np.concatenate([np.arange(0, 64), np.arange(N - 64, N),
                                     np.random.default_rng(0).integers(0, N, 160)])).astype(np.int32)
    blocks = np.unique(cols // 32)
    # pack only the 32-column blocks that contain sampled columns (the quantiser is per column)
    Wh = Wd[:, torch.from_numpy(np.concatenate([np.arange(b * 32, (b + 1) * 32) for b in blocks])).cuda()].cpu().numpy()
    planes, s, z = oracle.pack(np.ascontiguousarray(Wh))
    gp = w.planes[:, :, torch.from_numpy(blocks.astype(np.int64)).cuda()].cpu().numpy().view(np.uint32)
    assert np.array_equal(gp, planes)
    remap = {int(b): i for i, b in enumerate(blocks)}
    sub_cols = np.array([remap[int(c) // 32] * 32 + int(c) % 32 for c in cols], np.int32)
    y_ref = oracle.vmm(x, planes, s, z, ref_a["bits"], cols=sub_cols)
    _check_y(y_rank.cpu().numpy()[:, cols], y_ref, "rank")
    # the threshold form made inside the VMM launch, same shape
    theta = oracle.calibrate_thresholds(x, counts)
    y_t = gq.grinqh_vmm_thresholds(xd, theta, w)
    y_t_ref = oracle.vmm(x, planes, s, z, oracle.assign_thresholds(x, theta)["bits"], cols=sub_cols)
    _check_y(y_t.cpu().numpy()[:, cols], y_t_ref, "thresholds")


def test_pack_ramp_and_rounding_ties(gq):
    """grinqh_pack divides with a hand-rolled reciprocal sequence: send it an adversarial sweep, bit-exact against the
    oracle's IEEE divide + rint.  (i) ramp columns w = z + s * j with exactly representable s, z (every quotient an
    exact integer or an exact tie after the group's own scale); (ii) for scales from the subnormal range up to 2^8 and every code k, weights whose quotient (w - z) / s sits
    exactly on k + 1/2 (when representable) and one fp16 ulp either side of it: the rounding decision must be the
    oracle's IEEE divide + rint, bit for bit."""
    cols = []
    for e in range(-14, 3):                     # s = 2^e: ramps (codes 0..255 exactly; 2 x 128 rows)
        s_ = np.float32(2.0 ** e)
        for z_ in (np.float32(0.0), np.float32(-0.125), np.float32(3.0)):
            j = np.arange(256, dtype=np.float32)
            col = (z_ + s_ * j).astype(np.float16)
            if np.all(np.isfinite(col)) and float(col.max()) - float(col.min()) == 255.0 * float(s_):
                cols.append(col)
    rng = np.random.default_rng(11)
    for e in np.linspace(-24, 8, 65):           # tie neighbourhoods: group min 0, max 255 s, the rest around k + 1/2
        s_ = np.float16(2.0 ** e)
        if not np.isfinite(np.float32(s_) * 255) or float(s_) == 0.0:
            continue
        hi = np.float16(np.float32(s_) * np.float32(255.0))
        if not np.isfinite(hi):
            continue
        for rep in range(2):
            col = np.empty(256, np.float16)
            for half in range(2):
                k = rng.integers(0, 255, 126).astype(np.float32)
                mid = ((k + np.float32(0.5)) * np.float32(s_)).astype(np.float16)
                step = rng.integers(-1, 2, 126).astype(np.int16)           # -1, 0, +1 ulp around the tie
                near = (mid.view(np.int16) + step).view(np.float16)
                near = np.where(np.isfinite(near) & (near >= 0) & (near <= hi), near, mid)
                col[128 * half:128 * half + 126] = near
                col[128 * half + 126] = np.float16(0.0)
                col[128 * half + 127] = hi
            cols.append(col)
    n = (len(cols) + 31) // 32 * 32
    W = np.zeros((256, n), np.float16)
    for i, c in enumerate(cols):
        W[:, i] = c
    ref, out = _pack_both(gq, W)
    _check_pack(ref, out)


def test_decode_host_entry(gq):
    K, N = 1024, 2048
    W = synth.make_weights(K, N, 0.02, 41)
    x = synth.make_x(1, K, 42)
    counts = oracle.mix_to_counts(K, synth.MIXES["4"])
    planes, s, z = oracle.pack(W)
    y_ref = oracle.vmm(x, planes, s, z, oracle.assign(x, counts)["bits"])
    w = gq.grinqh_pack(_dev(W))
    xh = torch.from_numpy(x).pin_memory()
    yh = torch.empty((1, N), dtype=torch.float32).pin_memory()
    xd = torch.empty((1, K), dtype=torch.float16, device="cuda")
    yd = torch.empty((1, N), dtype=torch.float32, device="cuda")
    ws = gq.grinqh_vmm_workspace(1, K, N)
    gq.grinqh_decode_host(xh, counts, w, xd, yd, ws, yh)           # pinned y: the kernel writes host memory directly
    torch.cuda.synchronize()
    assert rel_l2(yh.numpy(), y_ref) <= TOL
    y_direct = yh.numpy().copy()
    yh.zero_()
    gq.grinqh_decode_host(xh, counts, w, xd, yd, ws, yh, force_copies=True)   # staged with cudaMemcpyAsync
    torch.cuda.synchronize()
    assert np.array_equal(yh.numpy(), y_direct)
    xp, yp = torch.from_numpy(x.copy()), torch.zeros((1, N), dtype=torch.float32)   # pageable host buffers
    gq.grinqh_decode_host(xp, counts, w, xd, yd, ws, yp)
    torch.cuda.synchronize()
    assert np.array_equal(yp.numpy(), y_direct)
    with pytest.raises(gq.GrinqhError):                             # a bad mix is rejected before anything is enqueued
        gq.grinqh_decode_host(xh, [K, 1, 0, 0, 0, 0, 0, 0, 0], w, xd, yd, ws, yh)


def test_fused_second_pass_matches_two_launches_and_workspace_is_reusable(gq):
    """grinqh_vmm (last CTA per tile reduces) == grinqh_vmm_main + grinqh_vmm_reduce bit for bit, repeatedly and
    across shapes sharing one workspace (the tickets must come back to zero after every launch)."""
    shapes = [(1, 1024, 2048), (2, 512, 4096 + 96), (1, 2048, 1024), (4, 256, 512)]
    ws = gq.grinqh_vmm_workspace(4, 2048, 4096 + 96)
    packed = {}
    for rep in range(3):
        for T, K, N in shapes:
            if (K, N) not in packed:
                packed[(K, N)] = gq.grinqh_pack(_dev(synth.make_weights(K, N, 0.02, K + N)))
            w = packed[(K, N)]
            x = synth.make_x(T, K, 100 + rep, "student_t")
            a = gq.grinqh_assign(_dev(x), oracle.mix_to_counts(K, synth.MIXES["4"]))
            y1 = gq.grinqh_vmm(w, a, workspace=ws).cpu().numpy()
            gq.grinqh_vmm_main(w, a, ws)
            y2 = torch.empty((T, N), dtype=torch.float32, device="cuda")
            gq.grinqh_vmm_reduce(T, K, N, y2, ws)
            assert np.array_equal(y1, y2.cpu().numpy())


@pytest.mark.parametrize("T,K,N,mix,seed", [(1, 128, 32, "4", 1), (4, 1024, 96, "2", 3), (3, 640, 1184, "5", 5),
                                            (1, 4096, 1024, "0", 6), (2, 256, 4096 + 32, "8", 7)])
def test_vmm_edge_shapes(gq, T, K, N, mix, seed):
    """smallest legal shape, ragged tiles (N % 128 != 0 -> 4-byte copy path), all-zero and all-8-bit mixes, T up to 4"""
    W = synth.make_weights(K, N, 0.02, seed)
    x = synth.make_x(T, K, seed, "student_t")
    y, y_ref = _run_vmm(gq, W, x, synth.MIXES[mix])
    if mix == "0":
        assert not y.any() and not y_ref.any()
    else:
        _check_y(y, y_ref)


@pytest.mark.parametrize("T,K,mix,dist,seed", [(1, 4096, "4", "normal", 0), (2, 8192, "3", "student_t", 1),
                                               (4, 1536, "2", "normal", 2), (1, 28672, "4", "student_t", 3)])
def test_assign_thresholds_and_calibration_bit_exact(gq, T, K, mix, dist, seed):
    """calibration on 8 synthetic vectors, threshold assignment of a
    fresh one; theta, widths, lists and schedule bit-exact against the oracle; the VMM consumes it unchanged."""
    counts = oracle.mix_to_counts(K, synth.MIXES[mix])
    xs = np.concatenate([synth.make_x(1, K, 100 + seed * 10 + s, dist) for s in range(8)], axis=0)
    theta_ref = oracle.calibrate_thresholds(xs, counts)
    theta = gq.grinqh_calibrate_thresholds(torch.from_numpy(xs), counts)
    assert list(theta_ref) == theta
    x = synth.make_x(T, K, 500 + seed, dist)
    ref = oracle.assign_thresholds(x, theta_ref)
    a = gq.grinqh_assign_thresholds(_dev(x), theta)
    torch.cuda.synchronize()
    _check_assign(ref, a, x)
    avg = ref["bits"].mean()
    assert abs(avg - synth.mix_avg_bits(synth.MIXES[mix])) < 0.5      # floats around the target (Fig. 6B)
    if K <= 8192:
        N = 1024
        W = synth.make_weights(K, N, 0.02, seed)
        planes, s, z = oracle.pack(W)
        y_ref = oracle.vmm(x, planes, s, z, ref["bits"])
        y = gq.grinqh_vmm(gq.grinqh_pack(_dev(W)), a).cpu().numpy()
        _check_y(y, y_ref)


def test_assign_thresholds_extremes(gq):
    K = 2048
    x = synth.make_x(2, K, 5)
    for theta in ([0] * 9, [0x8000] * 9, [0, 0, 0, 0x3C00, 0x3C00, 0x4400, 0x8000, 0x8000, 0x8000]):
        ref = oracle.assign_thresholds(x, np.array(theta, np.uint16))
        a = gq.grinqh_assign_thresholds(_dev(x), theta)
        torch.cuda.synchronize()
        _check_assign(ref, a, x)
    with pytest.raises(gq.GrinqhError):
        gq.grinqh_assign_thresholds(_dev(x), [0, 5, 4, 5, 5, 5, 5, 5, 5])


@pytest.mark.parametrize("T,K,N,mix,seed", [(1, 1024, 2048, "4", 0), (2, 2048, 1024 + 96, "3", 1), (4, 512, 4096, "2", 2),
                                            (1, 4096, 6144, "4", 3), (3, 384, 160, "5", 4)])
def test_vmm_thresholds_fused_equals_two_calls(gq, T, K, N, mix, seed):
    """grinqh_vmm_thresholds (assignment inside the VMM launch) == grinqh_assign_thresholds + grinqh_vmm bit for bit,
    and within tolerance of the oracle's threshold assignment + definitional VMM."""
    W = synth.make_weights(K, N, 0.02, seed)
    counts = oracle.mix_to_counts(K, synth.MIXES[mix])
    xs = np.concatenate([synth.make_x(1, K, 300 + seed * 10 + s, "student_t") for s in range(4)], axis=0)
    theta = oracle.calibrate_thresholds(xs, counts)
    x = synth.make_x(T, K, 900 + seed, "student_t")
    w = gq.grinqh_pack(_dev(W))
    xd = _dev(x)
    y_f = gq.grinqh_vmm_thresholds(xd, theta, w).cpu().numpy()
    a = gq.grinqh_assign_thresholds(xd, theta)
    y_2 = gq.grinqh_vmm(w, a).cpu().numpy()
    assert np.array_equal(y_f, y_2)
    planes, s, z = oracle.pack(W)
    y_ref = oracle.vmm(x, planes, s, z, oracle.assign_thresholds(x, theta)["bits"])
    _check_y(y_f, y_ref)


@pytest.mark.parametrize("K,N,std,seed", [(256, 512, 0.02, 0), (384, 1056, 0.02, 1), (128, 32, 1.0, 3), (1024, 4096, 0.015, 4)])
def test_unpack_is_the_correctly_rounded_full_precision_dequant(gq, K, N, std, seed):
    """SURVEY.md 8f3 (first half of the prefill path): planes -> fp16 W_hat, bit-exact against the oracle's
    fp64 dequantisation rounded once to fp16; and the dense product on it matches the all-8-bit VMM."""
    W = synth.make_weights(K, N, std, seed)
    W[:128, 0] = np.float16(0.25)                      # a constant group (s = 0)
    w = gq.grinqh_pack(_dev(W))
    Wh = gq.grinqh_unpack(w)
    torch.cuda.synchronize()
    planes, s, z = oracle.pack(W)
    ref = oracle.dequant(planes, s, z, 8).astype(np.float16)
    assert np.array_equal(Wh.cpu().numpy().view(np.uint16), ref.view(np.uint16))
    x = synth.make_x(3, K, seed + 50)
    y_dense = (torch.from_numpy(x).cuda().float() @ Wh.float()).cpu().numpy()   # prefill-style dense product
    y_ref = x.astype(np.float64) @ oracle.dequant(planes, s, z, 8)
    assert rel_l2(y_dense, y_ref) <= 2e-3              # fp16 W_hat: rounding of the weights themselves (2^-11 relative)


def test_fuzz_random_shapes_mixes_and_ties(gq):
    """Randomised sweep (fixed seed): any widths 0..8 with arbitrary counts, 1..4 tokens, ragged N, inputs with many
    tied magnitudes; rank and threshold forms, two-call and fused VMM.  Integer outputs bit-exact, y within tolerance."""
    rng = np.random.default_rng(20261104)
    for case in range(36):
        T = int(rng.integers(1, 5))
        K = 128 * int(rng.integers(1, 17))
        N = 32 * int(rng.integers(1, 41))
        cuts = np.sort(rng.integers(0, K + 1, 8))
        counts = np.diff(np.concatenate([[0], cuts, [K]])).astype(np.uint32)
        rng.shuffle(counts)
        kind = case % 3
        if kind == 0:
            x = synth.make_x(T, K, 1000 + case, "student_t")
        elif kind == 1:                                   # few distinct magnitudes: every cut splits a tie run
            x = (rng.integers(-6, 7, (T, K)) * 0.25).astype(np.float16)
        else:                                             # mostly zeros and a heavy tail
            x = (rng.standard_t(2.0, (T, K)) * (rng.random((T, K)) < 0.3)).astype(np.float16)
        W = synth.make_weights(K, N, 0.02, 2000 + case)
        planes, s, z = oracle.pack(W)
        w = gq.grinqh_pack(_dev(W))
        xd = _dev(x)
        ref = oracle.assign(x, counts)
        a = gq.grinqh_assign(xd, counts)
        torch.cuda.synchronize()
        _check_assign(ref, a, x)
        y = gq.grinqh_vmm(w, a).cpu().numpy()
        y_r = gq.grinqh_vmm_rank(xd, counts, w).cpu().numpy()
        assert np.array_equal(y, y_r), (case, T, K, N, list(counts))
        y_ref = oracle.vmm(x, planes, s, z, ref["bits"])
        _check_y(y, y_ref, (case, T, K, N, list(counts)))
        theta = np.sort(rng.integers(0, 0x4800, 9)).astype(np.uint16)
        theta[rng.integers(1, 9):] = 0x8000 if case % 4 == 0 else theta[-1]
        theta = np.sort(theta)
        ref_t = oracle.assign_thresholds(x, theta)
        a_t = gq.grinqh_assign_thresholds(xd, theta)
        torch.cuda.synchronize()
        _check_assign(ref_t, a_t, x)
        y2 = gq.grinqh_vmm(w, a_t).cpu().numpy()
        y3 = gq.grinqh_vmm_thresholds(xd, theta, w).cpu().numpy()
        assert np.array_equal(y2, y3), (case, T, K, N)
        y_ref_t = oracle.vmm(x, planes, s, z, ref_t["bits"])
        _check_y(y2, y_ref_t, (case, T, K, N))


def _carve(nbytes, dtype, shape):
    """A tensor of `shape` inside a larger device buffer with 4 KB of canary bytes (0x7F) on both sides."""
    pad = 4096
    buf = torch.full((pad + nbytes + pad,), 0x7F, dtype=torch.uint8, device="cuda")
    view = buf[pad:pad + nbytes].view(dtype).view(shape)
    return buf, view


def _canaries_intact(buf, nbytes):
    pad = 4096
    return bool((buf[:pad] == 0x7F).all().item()) and bool((buf[pad + nbytes:] == 0x7F).all().item())


@pytest.mark.parametrize("T,K,N,mix", [(1, 512, 2080, "4"), (2, 384, 1056, "3"), (4, 256, 96, "5"), (1, 1024, 4096 + 128, "2"),
                                       (3, 640, 1184, "4")])
def test_no_write_outside_the_outputs(gq, T, K, N, mix):
    """compute-sanitizer is closed on this pool (profiles/r02_sanitizer.md): every buffer a kernel of the library writes
    is carved out of a larger allocation with canaries on both sides; after all forms they are intact."""
    W = synth.make_weights(K, N, 0.02, 3 * K + N)
    x = synth.make_x(T, K, K + T, "student_t")
    counts = oracle.mix_to_counts(K, synth.MIXES[mix])
    ref_p = oracle.pack(W)
    ref_a = oracle.assign(x, counts)
    y_ref = oracle.vmm(x, *ref_p, ref_a["bits"])
    bufs = []

    def carve(nbytes, dtype, shape):
        b, v = _carve(nbytes, dtype, shape)
        bufs.append((b, nbytes))
        return v

    w = gq.Packed.__new__(gq.Packed)
    w.K, w.N = K, N
    w.planes = carve(8 * K * N // 8, torch.int32, (8, K, N // 32))
    w.scales = carve(K // 128 * N * 2, torch.float16, (K // 128, N))
    w.zeros = carve(K // 128 * N * 2, torch.float16, (K // 128, N))
    gq.grinqh_pack(_dev(W), w)
    a = gq.Assignment.__new__(gq.Assignment)
    a.T, a.K = T, K
    a.bits = carve(T * K, torch.uint8, (T, K))
    a.bits_union = carve(K, torch.uint8, (K,))
    a.rows = carve(4 * K, torch.int32, (K,))
    a.cnt_ge = carve(64, torch.int32, (16,))
    a.grows = carve(K, torch.uint8, (K,))
    a.gcnt_ge = carve(K // 128 * 16, torch.uint8, (K // 128, 16))
    a.gsched = carve(4 * T * K, torch.int32, (T, K))
    xd = _dev(x)
    gq.grinqh_assign(xd, counts, a)
    nws = gq.grinqh_vmm_workspace_bytes(T, K, N)
    ws = carve(nws, torch.uint8, (nws,))
    ws.zero_()
    ys = [carve(4 * T * N, torch.float32, (T, N)) for _ in range(3)]
    gq.grinqh_vmm(w, a, ys[0], ws)
    gq.grinqh_vmm_rank(xd, counts, w, ys[1], ws)
    theta = oracle.calibrate_thresholds(x, counts)
    gq.grinqh_vmm_thresholds(xd, theta, w, ys[2], ws)
    Wh = carve(2 * K * N, torch.float16, (K, N))
    gq.grinqh_unpack(w, Wh)
    torch.cuda.synchronize()
    for b, n in bufs:
        assert _canaries_intact(b, n)
    _check_pack(ref_p, w)
    _check_assign(ref_a, a, x)
    _check_y(ys[0].cpu().numpy(), y_ref)
    assert np.array_equal(ys[0].cpu().numpy(), ys[1].cpu().numpy())
    _check_y(ys[2].cpu().numpy(), oracle.vmm(x, *ref_p, oracle.assign_thresholds(x, theta)["bits"]))


def test_repeatability_under_reuse(gq):
    """One workspace, shapes and forms alternating, 25 rounds: every y bit-identical to the first round's (a race in the
    ring / list / ticket protocols would change a bit sooner or later) and element-wise equal to the oracle's."""
    cases = []
    ws = gq.grinqh_vmm_workspace(4, 2048, 6144)
    for T, K, N, mix in [(1, 2048, 6144, "4"), (2, 1024, 2080, "3"), (4, 512, 1056, "2"), (1, 1536, 4096, "5")]:
        W = synth.make_weights(K, N, 0.02, K + N)
        x = synth.make_x(T, K, 9 + T, "student_t")
        counts = oracle.mix_to_counts(K, synth.MIXES[mix])
        y_ref = oracle.vmm(x, *oracle.pack(W), oracle.assign(x, counts)["bits"])
        cases.append((gq.grinqh_pack(_dev(W)), _dev(x), counts, y_ref))
    first = {}
    for rnd in range(25):
        for i, (w, xd, counts, y_ref) in enumerate(cases):
            if (rnd + i) % 2:
                y = gq.grinqh_vmm_rank(xd, counts, w, workspace=ws).cpu().numpy()
            else:
                y = gq.grinqh_vmm(w, gq.grinqh_assign(xd, counts), workspace=ws).cpu().numpy()
            if i not in first:
                _check_y(y, y_ref)
                first[i] = y
            assert np.array_equal(y, first[i]), (rnd, i)


# ---- the paper's 2-bit-segment store, b_max in {4, 6, 8}
SEG2_MIXES = {4: [0.125, 0, 0.375, 0, 0.5, 0, 0, 0, 0], 6: [0.125, 0, 0.25, 0, 0.375, 0, 0.25, 0, 0],
              8: [0.125, 0, 0.25, 0, 0.25, 0, 0.125, 0, 0.25]}


@pytest.mark.parametrize("bmax", [4, 6, 8])
@pytest.mark.parametrize("K,N,seed", [(256, 512, 0), (384, 1184, 1), (128, 32, 2)])
def test_pack_seg2_bit_exact(gq, bmax, K, N, seed):
    W = synth.make_weights(K, N, 0.02, seed)
    W[:128, 0] = np.float16(0.25)                       # constant group
    W[:128, 1] = np.float16(-0.0)
    segs, s, z = oracle.pack2(W, bmax)
    out = gq.grinqh_pack_seg2(_dev(W), bmax)
    torch.cuda.synchronize()
    assert np.array_equal(out.segs.cpu().numpy().view(np.uint32), segs)
    assert np.array_equal(out.scales.cpu().numpy().view(np.uint16), s.view(np.uint16))
    assert np.array_equal(out.zeros.cpu().numpy().view(np.uint16), z.view(np.uint16))


@pytest.mark.parametrize("bmax", [4, 6, 8])
@pytest.mark.parametrize("K,N,dist,seed", [(256, 512, "normal", 0), (1024, 2176, "student_t", 1), (2048, 4096, "normal", 2),
                                           (512, 128, "student_t", 3)])
def test_vmm_rank_seg2_matches_oracle(gq, bmax, K, N, dist, seed):
    """rank assignment (widths 0, 2, .., b_max) + selective SEGMENT fetch + reconstruction with the store's own b_max"""
    W = synth.make_weights(K, N, 0.02, 40 + seed)
    x = synth.make_x(1, K, 50 + seed, dist)
    counts = oracle.mix_to_counts(K, SEG2_MIXES[bmax])
    segs, s, z = oracle.pack2(W, bmax)
    bits = oracle.assign(x, counts)["bits"]
    y_ref = oracle.vmm2(x, segs, s, z, bits, bmax)
    w = gq.grinqh_pack_seg2(_dev(W), bmax)
    y = gq.grinqh_vmm_rank_seg2(_dev(x), counts, w).cpu().numpy()
    _check_y(y, y_ref, bmax)
    if bmax == 8:       # the same weights in the 1-bit plane store give the same y up to the summation order
        y_planes = gq.grinqh_vmm_rank(_dev(x), counts, gq.grinqh_pack(_dev(W))).cpu().numpy()
        _check_y(y, y_planes.astype(np.float64), "planes")
    with pytest.raises(gq.GrinqhError):
        gq.grinqh_vmm_rank_seg2(_dev(x), oracle.mix_to_counts(K, synth.MIXES["4"] if bmax < 8 else
                                                             [0.5, 0.5, 0, 0, 0, 0, 0, 0, 0]), w)


def test_vmm_rank_seg2_full_size_sampled_columns(gq):
    """4096 x 28672 (gate|up) over the b_max = 8 segment store, avg-4 mix, oracle on sampled columns"""
    K, N, bmax = 4096, 28672, 8
    g = torch.Generator(device="cuda")
    g.manual_seed(99)
    Wd = (torch.randn((K, N), generator=g, device="cuda", dtype=torch.float32) * 0.02).to(torch.float16)
    x = synth.make_x(1, K, 78, "normal")
    counts = oracle.mix_to_counts(K, synth.MIXES["4"])
    w = gq.grinqh_pack_seg2(Wd, bmax)
    y = gq.grinqh_vmm_rank_seg2(_dev(x), counts, w).cpu().numpy()
    cols = np.unique(np.concatenate([np.arange(0, 32), np.arange(N - 32, N),
                                     np.random.default_rng(1).integers(0, N, 96)])).astype(np.int32)
    blocks = np.unique(cols // 16)
    Wh = Wd[:, torch.from_numpy(np.concatenate([np.arange(b * 16, (b + 1) * 16) for b in blocks])).cuda()].cpu().numpy()
    segs, s, z = oracle.pack2(np.ascontiguousarray(Wh), bmax)
    gs = w.segs[:, :, torch.from_numpy(blocks.astype(np.int64)).cuda()].cpu().numpy().view(np.uint32)
    assert np.array_equal(gs, segs)
    remap = {int(b): i for i, b in enumerate(blocks)}
    sub_cols = np.array([remap[int(c) // 16] * 16 + int(c) % 16 for c in cols], np.int32)
    y_ref = oracle.vmm2(x, segs, s, z, oracle.assign(x, counts)["bits"], bmax, cols=sub_cols)
    _check_y(y[:, cols], y_ref)


@pytest.mark.parametrize("M,K,N,seed", [(128, 128, 256, 0), (200, 512, 512, 2), (300, 2048, 768, 3), (1, 256, 256, 4),
                                        (515, 1024, 1024, 5)])
def test_prefill_gemm_fused_unpack_on_tensor_cores(gq, M, K, N, seed):
    """Y = X . W_hat at b_max = 8 in one tcgen05 launch, the unpack fused into the
    operand staging.  Oracle: x @ dequant(planes, s, z, 8) in fp64.  The kernel multiplies fp16 X by W_hat rounded once
    to fp16 (relative 2^-11 per weight), accumulates in fp32 and rounds Y to fp16 (2^-11 per output): the relative L2
    bound is 1e-3 and no element may be off by more than 2^-9 of the largest |y| of its row set."""
    W = synth.make_weights(K, N, 0.02, seed)
    W[:128, 0] = np.float16(0.25)                      # a constant group (s = 0)
    rng = np.random.default_rng(seed + 900)
    X = rng.standard_normal((M, K)).astype(np.float16)
    X[0, :] = 0                                        # an all-zero token
    planes, s, z = oracle.pack(W)
    ref = X.astype(np.float64) @ oracle.dequant(planes, s, z, 8)
    w = gq.grinqh_pack(_dev(W))
    Y = torch.full((M, N), float("nan"), dtype=torch.float16, device="cuda")
    gq.grinqh_prefill_gemm(_dev(X), w, Y)
    torch.cuda.synchronize()
    y = Y.cpu().numpy().astype(np.float64)
    assert np.isfinite(y).all()
    assert rel_l2(y, ref) <= 1e-3
    assert np.abs(y - ref).max() <= 2.0 ** -9 * np.abs(ref).max()
    assert not y[0].any()
    # and it is the product on exactly the matrix grinqh_unpack writes: same inputs, fp32 accumulation on both sides
    y_dense = (torch.from_numpy(X).cuda().float() @ gq.grinqh_unpack(w).float()).cpu().numpy()
    assert np.abs(y - y_dense).max() <= 2.0 ** -9 * np.abs(ref).max()


def test_prefill_gemm_full_size_sampled(gq):
    """The shape bench.py --prefill times (3000 tokens x 4096 x 14336, the paper's 3000:1 benchmark):
    sampled rows x sampled columns recomputed by the oracle in fp64 (columns are independent: only the 32-column blocks
    that contain sampled columns are packed on the host)."""
    M, K, N = 3000, 4096, 14336
    g = torch.Generator(device="cuda")
    g.manual_seed(4242)
    Wd = (torch.randn((K, N), generator=g, device="cuda", dtype=torch.float32) * 0.02).to(torch.float16)
    Xd = torch.randn((M, K), generator=g, device="cuda", dtype=torch.float32).to(torch.float16)
    w = gq.grinqh_pack(Wd)
    Y = gq.grinqh_prefill_gemm(Xd, w)
    torch.cuda.synchronize()
    rng = np.random.default_rng(7)
    cols = np.unique(np.concatenate([np.arange(0, 32), np.arange(N - 32, N), rng.integers(0, N, 96)])).astype(np.int64)
    rows = np.unique(np.concatenate([[0, 127, 128, 255, 256, 2943, 2944, 2999], rng.integers(0, M, 24)])).astype(np.int64)
    blocks = np.unique(cols // 32)
    Wh = Wd[:, torch.from_numpy(np.concatenate([np.arange(b * 32, (b + 1) * 32) for b in blocks])).cuda()].cpu().numpy()
    planes, s, z = oracle.pack(np.ascontiguousarray(Wh))
    assert np.array_equal(w.planes[:, :, torch.from_numpy(blocks).cuda()].cpu().numpy().view(np.uint32), planes)
    remap = {int(b): i for i, b in enumerate(blocks)}
    sub = np.array([remap[int(c) // 32] * 32 + int(c) % 32 for c in cols])
    ref = Xd[torch.from_numpy(rows).cuda()].cpu().numpy().astype(np.float64) @ oracle.dequant(planes, s, z, 8)[:, sub]
    y = Y[torch.from_numpy(rows).cuda()][:, torch.from_numpy(cols).cuda()].cpu().numpy().astype(np.float64)
    assert rel_l2(y, ref) <= 1e-3
    assert np.abs(y - ref).max() <= 2.0 ** -9 * np.abs(ref).max()


def test_prefill_gemm_rejects_unsupported_shapes(gq):
    w = gq.grinqh_pack(_dev(synth.make_weights(128, 128, 0.02, 0)))   # N % 256 != 0
    X = torch.zeros((4, 128), dtype=torch.float16, device="cuda")
    with pytest.raises(gq.GrinqhError):
        gq.grinqh_prefill_gemm(X, w)


def test_second_device_when_present(gq):
    """the kernels' shared-memory attribute and the static scratch address are per device.  With two or more
    GPUs the same calls on device 1 must work and return device 0's bits (skipped on a one-GPU box)."""
    if torch.cuda.device_count() < 2:
        pytest.skip("one GPU")
    T, K, N = 2, 1024, 2080
    W = synth.make_weights(K, N, 0.02, 3)
    x = synth.make_x(T, K, 3, "student_t")
    counts = gq.grinqh_mix_to_counts(K, synth.MIXES["4"])
    ys = []
    for d in (0, 1):
        with torch.cuda.device(d):
            dev = torch.device("cuda", d)
            w = gq.grinqh_pack(torch.from_numpy(W).to(dev))
            xd = torch.from_numpy(x).to(dev)
            y = gq.grinqh_vmm_rank(xd, counts, w)
            y2 = torch.empty_like(y)
            gq.grinqh_vmm_rank_static(xd, counts, w, y2)
            a = gq.grinqh_assign(xd, counts)
            y3 = gq.grinqh_vmm(w, a)
            torch.cuda.synchronize(dev)
            assert torch.equal(y, y2) and torch.equal(y, y3)
            ys.append(y.cpu().numpy())
    assert np.array_equal(ys[0], ys[1])
