"""CPU-only checks of the CUDA library's host side: it loads, exports every symbol include/grinqh.h
declares, validates arguments without touching a GPU, and its bit-gather network (plain C++) is right."""
import ctypes as C
import os
import re
import subprocess

import numpy as np
import pytest

import oracle
from paper_2606_23419_b200 import build as gq_build
from paper_2606_23419_b200 import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    return C.CDLL(gq_build.build())


def test_library_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "grinqh.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(grinqh_[a-z0-9_]+)\s*\(", hdr))
    assert {"grinqh_pack", "grinqh_assign", "grinqh_vmm"} <= declared
    for name in sorted(declared):
        assert hasattr(lib, name), f"{name} declared in grinqh.h but not exported"
    from paper_2606_23419_b200 import binding
    assert set(binding.EXPORTS) == declared


def test_mix_to_counts_closed_forms(lib):
    """The product's own copy pinned directly (not through the oracle's): the config mixes are multiples of 1/32 and the
    config K multiples of 256, so counts = frac * K exactly; an arbitrary mix always sums to K, is monotone in the
    cumulative shares, and is within one row of frac * K per width boundary."""
    lib.grinqh_mix_to_counts.argtypes = [C.c_int, C.c_void_p, C.c_void_p]
    for K in (256, 4096, 12288, 14336, 8192, 28672):
        for name, frac in synth.MIXES.items():
            f = (C.c_double * 9)(*frac)
            c = (C.c_uint32 * 9)()
            assert lib.grinqh_mix_to_counts(K, f, c) == 0
            assert list(c) == [int(round(p * K)) for p in frac] and all(abs(p * K - round(p * K)) < 1e-9 for p in frac)
    rng = np.random.default_rng(1)
    for _ in range(50):
        K = 128 * int(rng.integers(1, 257))
        frac = rng.dirichlet(np.ones(9))
        f = (C.c_double * 9)(*frac)
        c = (C.c_uint32 * 9)()
        assert lib.grinqh_mix_to_counts(K, f, c) == 0
        assert sum(c) == K
        cum_c = np.cumsum(list(c)[::-1])[:-1]              # rows with width >= w, w = 8..1
        cum_f = np.cumsum(frac[::-1])[:-1] * K
        assert np.all(np.abs(cum_c - cum_f) <= 0.5 + 1e-6)  # C_w = floor(F_w K + 1/2)


def test_mix_to_counts_matches_oracle_and_rejects(lib):
    lib.grinqh_mix_to_counts.argtypes = [C.c_int, C.c_void_p, C.c_void_p]
    rng = np.random.default_rng(0)
    for K in (256, 4096, 12288, 14336, 28672):
        for name, frac in synth.MIXES.items():
            f = (C.c_double * 9)(*frac)
            c = (C.c_uint32 * 9)()
            assert lib.grinqh_mix_to_counts(K, f, c) == 0
            assert list(c) == list(oracle.mix_to_counts(K, frac))
        for _ in range(20):
            frac = rng.dirichlet(np.ones(9))
            f = (C.c_double * 9)(*frac)
            c = (C.c_uint32 * 9)()
            assert lib.grinqh_mix_to_counts(K, f, c) == 0
            assert list(c) == list(oracle.mix_to_counts(K, frac)) and sum(c) == K
    bad = (C.c_double * 9)(*([0.5] * 9))
    c = (C.c_uint32 * 9)()
    assert lib.grinqh_mix_to_counts(256, bad, c) == -4


def test_argument_validation_without_gpu(lib):
    lib.grinqh_status_string.restype = C.c_char_p
    assert lib.grinqh_status_string(0) == b"ok"
    assert lib.grinqh_version() >= 100
    vp = C.c_void_p
    lib.grinqh_pack.argtypes = [vp, C.c_int, C.c_int, C.c_int, vp, vp, vp, vp]
    assert lib.grinqh_pack(None, 128, 32, 128, None, None, None, None) == -1          # NULL
    assert lib.grinqh_pack(16, 100, 32, 128, 16, 16, 16, None) == -2                  # K % 128
    assert lib.grinqh_pack(16, 128, 40, 128, 16, 16, 16, None) == -2                  # N % 32
    assert lib.grinqh_pack(16, 128, 32, 64, 16, 16, 16, None) == -2                   # group
    assert lib.grinqh_pack(8, 128, 32, 128, 16, 16, 16, None) == -3                   # alignment
    lib.grinqh_assign.argtypes = [vp, C.c_int, C.c_int, vp] + [vp] * 7 + [vp, C.c_size_t, vp]
    counts = (C.c_uint32 * 9)(1, 0, 0, 0, 0, 0, 0, 0, 100)
    assert lib.grinqh_assign(16, 1, 128, counts, 16, 16, 16, 16, 16, 16, 16, None, 0, None) == -4   # sum != K
    assert lib.grinqh_assign(16, 5, 128, counts, 16, 16, 16, 16, 16, 16, 16, None, 0, None) == -2   # T
    lib.grinqh_vmm_workspace_bytes.restype = C.c_size_t
    lib.grinqh_vmm_workspace_bytes.argtypes = [C.c_int] * 3
    assert lib.grinqh_vmm_workspace_bytes(1, 4096, 4096) > 0
    assert lib.grinqh_vmm_workspace_bytes(1, 4000, 4096) == 0
    assert lib.grinqh_vmm_workspace_bytes(1, 32768, 4096) > 0 and lib.grinqh_vmm_workspace_bytes(1, 32768 + 128, 4096) == 0
    lib.grinqh_vmm.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int] + [vp] * 5 + [vp, vp, C.c_size_t, vp]
    assert lib.grinqh_vmm(1, 128, 32, 128, 16, 16, 16, 16, 16, 16, 16, 0, None) == -5  # workspace
    lib.grinqh_vmm_rank.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, vp] + [vp] * 3 + [vp, vp, C.c_size_t, vp]
    big = 1 << 30
    assert lib.grinqh_vmm_rank(16, 1, 128, 32, 128, counts, 16, 16, 16, 16, 16, big, None) == -4   # sum(counts) != K
    assert lib.grinqh_vmm_rank(16, 1, 128, 32, 128, None, 16, 16, 16, 16, 16, big, None) == -1     # NULL counts
    lib.grinqh_decode_host.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, vp] + [vp] * 3 + [vp, vp, vp,
                                                                                                  C.c_size_t, vp, C.c_int, vp]
    # every argument is validated before anything is enqueued (no GPU is touched here)
    assert lib.grinqh_decode_host(16, 1, 128, 32, 128, counts, 16, 16, 16, 16, 16, 16, big, 16, 0, None) == -4
    assert lib.grinqh_decode_host(16, 1, 128, 32, 128, counts, 16, 16, 16, 16, 16, 16, 0, 16, 0, None) == -5
    assert lib.grinqh_decode_host(16, 1, 128, 40, 128, counts, 16, 16, 16, 16, 16, 16, big, 16, 0, None) == -2


def test_gather_network_on_host(tmp_path):
    exe = tmp_path / "gather_check"
    subprocess.check_call(["g++", "-O2", "-std=c++17", "-o", str(exe),
                           os.path.join(ROOT, "tests", "host", "gather_check.cpp")])
    out = subprocess.run([str(exe)], capture_output=True, text=True)
    assert out.returncode == 0 and "OK" in out.stdout, out.stdout
