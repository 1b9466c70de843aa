"""grinqh_vmm_rank_static (include/grinqh.h): the allocation-free form of grinqh_vmm_rank, its scratch in the library's
static device array.  Collected last on purpose (the run uses pytest -x)."""
import numpy as np
import pytest
import torch

from paper_2606_23419_b200 import binding as gq
from paper_2606_23419_b200 import synth

pytestmark = pytest.mark.gpu


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _close(y, y_ref):
    # the element-wise bound of tests/test_gpu_parity.py (_check_y)
    tol = 1e-5 * float(np.abs(y_ref).max()) + 1e-6
    return float(np.abs(y - y_ref).max()) <= tol


def test_static_scratch_matches_workspace_path_on_two_calls_in_a_row():
    torch.cuda.set_device(0)
    # two different shapes and inputs back to back: the second call finds the first one's partials and tickets in the array
    cases = [(1, 4096, 4096, "4", 11), (2, 1024, 2080, "3", 12)]
    packed, xs, cnts, refs = [], [], [], []
    for (T, K, N, mix, seed) in cases:
        w = gq.grinqh_pack(_dev(synth.make_weights(K, N, 0.02, seed)))
        x = _dev(synth.make_x(T, K, seed, "student_t"))
        counts = gq.grinqh_mix_to_counts(K, synth.MIXES[mix])
        assert gq.grinqh_vmm_workspace_bytes(T, K, N) <= gq.grinqh_static_scratch_bytes()
        packed.append(w), xs.append(x), cnts.append(counts)
        refs.append(gq.grinqh_vmm_rank(x, counts, w).cpu().numpy())  # the existing path, its own workspace
    ys = [torch.full((T, N), float("nan"), dtype=torch.float32, device="cuda") for (T, K, N, _, _) in cases]
    torch.cuda.synchronize()
    for rep in range(2):  # ... and the same pair again: four calls on one stream, none of them allocating in the library
        for i in range(len(cases)):
            gq.grinqh_vmm_rank_static(xs[i], cnts[i], packed[i], ys[i])
        torch.cuda.synchronize()
        for i in range(len(cases)):
            y = ys[i].cpu().numpy()
            assert np.isfinite(y).all()
            assert _close(y, refs[i]), (rep, cases[i], float(np.abs(y - refs[i]).max()))
            assert np.array_equal(y, refs[i])  # same launch, same plan: the same bits
            ys[i].fill_(float("nan"))


def test_static_scratch_rejects_shapes_beyond_the_limit():
    torch.cuda.set_device(0)
    T, K, N = 4, 128, 1 << 18  # 4 x 262144 fp32 partials = 4 MiB + tickets > the array
    assert gq.grinqh_vmm_workspace_bytes(T, K, N) > gq.grinqh_static_scratch_bytes()
    w = gq.Packed(K, N, "cuda")  # contents irrelevant: nothing is enqueued
    x = torch.zeros((T, K), dtype=torch.float16, device="cuda")
    y = torch.zeros((T, N), dtype=torch.float32, device="cuda")
    counts = gq.grinqh_mix_to_counts(K, synth.MIXES["4"])
    with pytest.raises(gq.GrinqhError, match="static"):
        gq.grinqh_vmm_rank_static(x, counts, w, y)
