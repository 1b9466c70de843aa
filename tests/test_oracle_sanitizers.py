"""The oracle built with AddressSanitizer + UndefinedBehaviorSanitizer and driven through every entry point on the
tiny config and a ragged multi-token case (sanitizers on the oracle).  Runs in a subprocess: the
sanitizer runtime has to be loaded before Python's allocator."""
import os
import subprocess
import sys
import textwrap

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_oracle_under_asan_ubsan(tmp_path):
    so = tmp_path / "liborc_san.so"
    src = os.path.join(ROOT, "oracle", "grinqh_oracle.cpp")
    subprocess.check_call(["g++", "-std=c++17", "-O1", "-g", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
                           "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-o", str(so), src])
    asan = subprocess.run(["g++", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.exists(asan):
        pytest.skip("libasan.so not found")
    driver = textwrap.dedent(f"""
        import sys, numpy as np
        sys.path.insert(0, {ROOT!r})
        import oracle.build as ob
        ob.build = lambda force=False: {str(so)!r}       # the sanitizer build instead of the plain one
        import oracle
        oracle._build = ob.build
        from paper_2606_23419_b200 import synth
        W, x, frac = synth.tiny_config(0)
        counts = oracle.mix_to_counts(W.shape[0], frac)
        planes, s, z = oracle.pack(W)
        a = oracle.assign(x, counts)
        y = oracle.vmm(x, planes, s, z, a["bits"])
        y2 = oracle.vmm_planewise(x, planes, s, z, a["bits"])
        assert np.allclose(y, y2, rtol=1e-12, atol=1e-12)
        oracle.dequant(planes, s, z, 3)
        x4 = synth.make_x(4, 384, 5, "student_t")
        W4 = synth.make_weights(384, 96, 0.02, 6)
        p4 = oracle.pack(W4)
        a4 = oracle.assign(x4, oracle.mix_to_counts(384, [0.11, 0.09, 0.13, 0.07, 0.2, 0.1, 0.1, 0.05, 0.15]))
        oracle.vmm(x4, *p4, a4["bits"], cols=np.array([0, 5, 95], np.int32))
        th = oracle.calibrate_thresholds(x4, oracle.mix_to_counts(384, frac))
        oracle.assign_thresholds(x4, th)
        print("SANITIZED OK")
    """)
    env = dict(os.environ, LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0:abort_on_error=1", UBSAN_OPTIONS="halt_on_error=1")
    out = subprocess.run([sys.executable, "-c", driver], capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0 and "SANITIZED OK" in out.stdout, out.stdout[-2000:] + out.stderr[-4000:]
