"""N > 1 is "replicas only": no data-path collective.  What there is to test on the CPU is the host
logic of the launch contract: max-over-ranks timing over gloo (world_size 2), and the reference arm under torchrun
(rank 0 alone works and prints one JSON line; the other rank exits 0 without output)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
r = dist.get_rank()
out = bench.max_over_ranks([10.0 + r, 5.0 - r, 7.0])
assert out == [11.0, 5.0, 7.0], out
dist.barrier()
dist.destroy_process_group()
open(os.path.join({out!r}, "rank%d.ok" % r), "w").write("ok")
"""


def _torchrun(args, port, timeout):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port)] + args
    return subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=timeout)


def test_max_over_ranks_gloo_world2(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(_WORKER.format(root=ROOT, out=str(tmp_path)))
    out = _torchrun([str(w)], 29731, 300)
    assert out.returncode == 0, out.stderr[-2000:]
    assert (tmp_path / "rank0.ok").exists() and (tmp_path / "rank1.ok").exists()  # (stdout of the ranks interleaves)


def test_reference_arm_under_torchrun_prints_one_line():
    out = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"], 29732, 600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["higher_is_better"] is False
