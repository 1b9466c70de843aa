#!/usr/bin/env python
"""bench.py — GRINQH decode hot path on B200 (contract: see the task prompt / DESIGN.md "Measurement").

Workload (N = 1): BASELINE.json configs[1] — one Llama-3-8B-shaped layer, batch 1, avg 4 bits:
7 projections (q,k,v,o,gate,up,down), 4 distinct input vectors (q/k/v and gate/up share one).
A "step" = one pass of the per-step hot path over one layer: 4 x grinqh_vmm_rank — the rank assignment of the input
vector, the selective plane fetch and the deterministic split-K second pass all inside ONE launch per input vector
(q|k|v and gate|up concatenated along N).  The same step as 4 x grinqh_assign + 4 x grinqh_vmm ("two_kernel_form"),
with one launch per projection ("per_projection") and with the paper's threshold assignment are reported beside it.  grinqh_pack is offline (once per weight) and reported separately under "pack".
The timed loop rotates over LAYERS distinct packed layers (> L2) so every step streams from HBM.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--mix 4] [--layers 4]

`--impl reference` times the CPU oracle (kind "oracle") on a bounded column sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "us per decode step of one Llama-3-8B-shaped layer (4 rank assignments + the 7 projections as bit-planar VMMs), batch 1"


def _committed_traffic(mix):
    """dram__bytes_read.sum + dram__bytes_write.sum of the step's launches from the committed ncu capture
    (profiles/r02_traffic.json, written from an `ncu --set full` run of this command; it names the commit it was
    taken on).  None when no capture of this mix is committed: the value is never made up."""
    p = os.path.join(ROOT, "profiles", "r02_traffic.json")
    try:
        d = json.load(open(p))
        return d["bytes_per_step"].get(mix), d.get("captured_on")
    except Exception:
        return None, None
UNIT = "us"


def _args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="native", choices=["native", "reference"])
    ap.add_argument("--mix", default="4")
    ap.add_argument("--layers", type=int, default=4, help="distinct packed layers the timed loop rotates over")
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", action="store_true", help="configs 3 and 5: per-VMM latency vs average bits (not the contract line)")
    ap.add_argument("--prefill", action="store_true", help="f3: fused tcgen05 prefill GEMM against grinqh_unpack + dense library GEMM")
    ap.add_argument("--decode-step", action="store_true", help="config 4: 32-layer decode step in one CUDA graph")
    ap.add_argument("--no-split", action="store_true", help="skip the one-launch-per-projection variant")
    ap.add_argument("--seg2", action="store_true", help="f2: 2-bit-segment store against the 1-bit plane store (A/B)")
    return ap.parse_args()


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def _tensor_peak():
    """Dense 16-bit tensor peak for a kernel timed alone (burst figure of MEASURED_PEAKS.json; fp16 = bf16 rate)."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["bf16_tflops"]), "measured (MEASURED_PEAKS.json bf16_tflops, burst)"
        except Exception:
            pass
    return 2250.0, "fallback (nominal dense bf16 2.25 PFLOP/s)"


def alg_bytes(K, N, T, sum_bits):
    """Algorithmic bytes of one VMM: fetched planes + fp16 s,z + x + y + lists."""
    return (N // 8) * sum_bits + 4 * (K // 128) * N + 2 * T * K + 4 * T * N + 5 * K


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML during the timed region."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz, self._stop_evt = index, [], set(), None, threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            pass

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.004)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=1.0)
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


# ------------------------------------------------------------------------------------------ reference arm
class OracleLayerSample:
    """CPU oracle on a bounded sample of the layer step: for each of the 7 projections the first
    `cols_per_proj` output columns (all K rows) + the 4 assignments.  Packing the sample is offline
    (not timed).  run() returns the seconds one sampled step took; `fraction` scales it to the full layer."""

    def __init__(self, mix_name: str, seed: int, cols_per_proj: int = 1 << 30):
        import oracle
        from paper_2606_23419_b200 import synth
        self.oracle, self.synth = oracle, synth
        self.frac = synth.MIXES[mix_name]
        self.xs = {name: synth.make_x(1, K, seed + i, "normal")
                   for i, (name, K) in enumerate(synth.LLAMA3_8B_INPUT_DIMS.items())}
        self.packed, full_w, samp_w = {}, 0, 0
        for i, (name, K, N) in enumerate(synth.LLAMA3_8B_LAYER):
            n = min(N, cols_per_proj)
            self.packed[name] = oracle.pack(synth.make_weights(K, n, 0.02, seed + 100 + i))
            full_w += K * N
            samp_w += K * n
        self.fraction = samp_w / full_w
        if samp_w == full_w:
            self.desc = ("oracle assign x4 + oracle vmm (fp64, 1 thread) on the FULL layer step: all output columns of "
                         f"the 7 projections ({full_w / 1e6:.1f}M weights), no scaling")
        else:
            self.desc = (f"oracle assign x4 + oracle vmm (fp64, 1 thread) on the first {cols_per_proj} output columns of "
                         f"each of the 7 projections ({samp_w / 1e6:.2f}M of {full_w / 1e6:.1f}M weights), "
                         f"time scaled by the weight ratio")

    def run(self) -> float:
        oracle, synth = self.oracle, self.synth
        t0 = time.perf_counter()
        assigns = {}
        for name, K in synth.LLAMA3_8B_INPUT_DIMS.items():
            assigns[name] = oracle.assign(self.xs[name], oracle.mix_to_counts(K, self.frac))
        for name, K, N in synth.LLAMA3_8B_LAYER:
            inp = synth.LLAMA3_8B_INPUTS[name]
            planes, s, z = self.packed[name]
            oracle.vmm(self.xs[inp], planes, s, z, assigns[inp]["bits"])
        return time.perf_counter() - t0


WORKLOAD = ("llama3-8b-layer (BASELINE.json configs[1]): 4096->4096 x2 (q,o), 4096->1024 x2 (k,v), "
            "4096->14336 x2 (gate,up), 14336->4096 (down); batch 1; per-step rank assignment")


def run_reference(args):
    """The oracle as it stands on the host cores.  A full layer step takes ~4 s on one core: when steps + warmup of
    them fit in ~150 s every step IS the full step (no scaling); otherwise each step is the first `cols` output
    columns of every projection and the time is scaled by the weight ratio (said in the line)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2606_23419_b200 import synth
    n = max(1, args.steps + args.warmup)
    rows = sum(K for _, K, _ in synth.LLAMA3_8B_LAYER)
    if n * 4.5 <= 150.0:
        sample = OracleLayerSample(args.mix, args.seed)
    else:
        budget = 120.0 / n                                # about 25 ns per weight
        cols = max(32, min(1024, int(budget / (rows * 32 * 25e-9)) * 32))
        sample = OracleLayerSample(args.mix, args.seed, cols)
    times = []
    for i in range(args.warmup + args.steps):
        t = sample.run()
        if i >= args.warmup:
            times.append(t)
    sec = sum(times) / len(times)
    us = 1e6 * sec / sample.fraction
    line = {
        "impl": "reference", "metric": METRIC, "value": us, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": us / 1e3, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "avg_bits": synth.mix_avg_bits(synth.MIXES[args.mix]), "mix": args.mix},
        "cpu_baseline": {"value": us, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample.desc,
                         "sample_fraction": sample.fraction, "seconds_per_timed_step_as_run": sec},
        "e2e": {"value": us, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def max_over_ranks(values, device=None):
    """Replicas only: the ranks share nothing on the data path; the job's time is the slowest rank's."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in values]
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.tolist()]


# ------------------------------------------------------------------------------------------ native arm
def run_native(args):
    import numpy as np
    import torch

    from paper_2606_23419_b200 import binding as gq
    from paper_2606_23419_b200 import synth

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    frac = synth.MIXES[args.mix]
    avg_bits = synth.mix_avg_bits(frac)
    L = args.layers
    T = 1
    fused = synth.LLAMA3_8B_LAYER_FUSED          # (name, K, N, input): the launches of the timed step
    split = [(n, K, N, synth.LLAMA3_8B_INPUTS[n]) for n, K, N in synth.LLAMA3_8B_LAYER]
    in_dims = synth.LLAMA3_8B_INPUT_DIMS
    counts = {K: gq.grinqh_mix_to_counts(K, frac) for K in set(in_dims.values())}

    # ---- offline: generate + pack L distinct layers (grinqh_pack timed on its own)
    gen = torch.Generator(device=dev)
    gen.manual_seed(args.seed + 1000 * rank)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    pack_ms, pack_bytes = 0.0, 0

    def make_packed(shapes, timed):
        nonlocal pack_ms, pack_bytes
        d = {}
        for name, K, N, _ in shapes:
            W = (torch.randn((K, N), generator=gen, device=dev, dtype=torch.float32) * 0.02).to(torch.float16)
            out = gq.Packed(K, N, dev)
            gq.grinqh_pack(W, out)
            if timed:  # second launch on the same buffers (the first one pays the lazy module load)
                torch.cuda.synchronize()
                e0.record()
                gq.grinqh_pack(W, out)
                e1.record()
                torch.cuda.synchronize()
                pack_ms += e0.elapsed_time(e1)
                pack_bytes += K * N * 3 + (K // 128) * N * 4
            d[name] = out
            del W
        return d

    packed = [make_packed(fused, True) for _ in range(L)]
    packed_split = [make_packed(split, False) for _ in range(L)] if not args.no_split else None

    # ---- per-step inputs: fresh activations per layer copy (N(0,1), 1% channels x20)
    x_host = [{n: torch.from_numpy(synth.make_x(T, K, args.seed + 10 * l + i + 1000 * rank, "normal")).pin_memory()
               for i, (n, K) in enumerate(in_dims.items())} for l in range(L)]
    x_dev = [{n: v.to(dev) for n, v in xl.items()} for xl in x_host]
    assigns = [{n: gq.Assignment(T, K, dev) for n, K in in_dims.items()} for _ in range(L)]
    all_shapes = list(fused) + split
    y_dev = [{name: torch.empty((T, N), dtype=torch.float32, device=dev) for name, K, N, _ in all_shapes} for _ in range(L)]
    y_host = [{name: torch.empty((T, N), dtype=torch.float32).pin_memory() for name, K, N, _ in fused} for _ in range(L)]
    _, Kw, Nw, _ = max(all_shapes, key=lambda s: gq.grinqh_vmm_workspace_bytes(T, s[1], s[2]))
    ws = gq.grinqh_vmm_workspace(T, Kw, Nw, dev)
    x_stage = {n: torch.empty((T, K), dtype=torch.float16, device=dev) for n, K in in_dims.items()}

    def step_device(l):          # the timed step: the rank assignment inside the VMM launch, 4 launches
        for name, K, N, inp in fused:
            gq.grinqh_vmm_rank(x_dev[l][inp], counts[K], packed[l][name], y_dev[l][name], ws)

    def step_two_kernel(l):      # the same step as 4 x grinqh_assign + 4 x grinqh_vmm (round 1's form)
        for name, K, N, inp in fused:
            gq.grinqh_assign(x_dev[l][inp], counts[K], assigns[l][inp])
            gq.grinqh_vmm(packed[l][name], assigns[l][inp], y_dev[l][name], ws)

    def step_split(l):           # one launch per projection: 7 x grinqh_vmm_rank
        for name, K, N, inp in split:
            gq.grinqh_vmm_rank(x_dev[l][inp], counts[K], packed_split[l][name], y_dev[l][name], ws)

    # threshold form: thetas calibrated offline on 8 synthetic vectors per input
    thetas = {n: gq.grinqh_calibrate_thresholds(
        torch.from_numpy(np.concatenate([synth.make_x(1, K, 7000 + 10 * i + s, "normal") for s in range(8)], axis=0)),
        counts[K]) for i, (n, K) in enumerate(in_dims.items())}

    def step_thresholds_fused(l):  # the paper's threshold assignment made inside the VMM launch: 4 launches per step
        for name, K, N, inp in fused:
            gq.grinqh_vmm_thresholds(x_dev[l][inp], thetas[inp], packed[l][name], y_dev[l][name], ws)

    def step_sched_only(l):      # the VMM launches alone, on schedules already made by grinqh_assign
        for name, K, N, inp in fused:
            gq.grinqh_vmm(packed[l][name], assigns[l][inp], y_dev[l][name], ws)

    def step_host(l, force_copies=False):
        for name, K, N, inp in fused:
            gq.grinqh_decode_host(x_host[l][inp], counts[K], packed[l][name], x_stage[inp], y_dev[l][name], ws,
                                  y_host[l][name], force_copies=force_copies)

    stream = torch.cuda.Stream(device=dev)
    with torch.cuda.stream(stream):
        for l in range(L):          # eager warm-up
            step_device(l)
            step_two_kernel(l)
            step_host(l)
            if packed_split:
                step_split(l)
        stream.synchronize()

        def capture(fn):
            graphs = []
            for l in range(L):
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=stream):
                    fn(l)
                graphs.append(g)
            return graphs

        def barrier():
            if world > 1:
                import torch.distributed as dist
                dist.barrier()
            torch.cuda.synchronize()

        def timed(graphs, steps, sync_each=False):
            for i in range(3):
                graphs[i % L].replay()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            barrier()
            a.record(stream)
            for i in range(steps):
                graphs[i % L].replay()
                if sync_each:
                    stream.synchronize()
            b.record(stream)
            barrier()
            return a.elapsed_time(b) * 1e3 / steps   # us per step

        g_dev = capture(step_device)
        for i in range(max(args.warmup, 3)):
            g_dev[i % L].replay()
        sampler = ClockSampler(local)
        sampler.start()
        us_step = timed(g_dev, args.steps)
        clocks = sampler.stop()
        us_host = timed(capture(step_host), args.steps, sync_each=True)
        n_c = max(50, args.steps // 4)
        us_hostc = timed(capture(lambda l: step_host(l, True)), n_c, sync_each=True)
        us_two = timed(capture(step_two_kernel), args.steps)
        us_sched = timed(capture(step_sched_only), args.steps)
        step_thresholds_fused(0)
        stream.synchronize()
        us_thrf = timed(capture(step_thresholds_fused), args.steps)
        us_split = timed(capture(step_split), args.steps) if packed_split else 0.0
        for l in range(L):       # the rank-form assignments (byte accounting below)
            for n, K in in_dims.items():
                gq.grinqh_assign(x_dev[l][n], counts[K], assigns[l][n])
        stream.synchronize()

    us_step, us_host, us_hostc, us_two, us_sched, us_thrf, us_split = max_over_ranks(
        [us_step, us_host, us_hostc, us_two, us_sched, us_thrf, us_split], dev)

    # ---- algorithmic bytes of the VMM launches of one step (measured widths; SURVEY.md 8d / DESIGN.md)
    step_bytes, plane_bytes = 0, 0
    per_vmm = []
    for name, K, N, inp in fused:
        sb = int(assigns[0][inp].bits_union.sum().item())
        b = alg_bytes(K, N, T, sb)
        step_bytes += b
        plane_bytes += (N // 8) * sb
        per_vmm.append({"launch": name, "K": K, "N": N, "alg_bytes": b})
    peak, peak_src = _peaks()
    achieved = step_bytes / (us_step * 1e-6) / 1e9  # GB/s over the launches of a step (assignment included)
    traffic, traffic_on = _committed_traffic(args.mix)

    h2d = sum(T * K * 2 for K in in_dims.values())
    d2h = sum(T * N * 4 for _, _, N, _ in fused)
    weights = sum(K * N for _, K, N, _ in fused)
    line = {
        "metric": METRIC, "value": us_step, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": us_step / 1e3, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": WORKLOAD,
                   "launches": "4 x grinqh_vmm_rank per step: the rank assignment (one shared-memory histogram select per "
                               "CTA), the selective plane fetch and the deterministic split-K second pass in ONE launch per "
                               "input vector; q|k|v and gate|up are concatenated along N (same input vector, per-column "
                               "quantiser)",
                   "avg_bits": avg_bits, "mix": args.mix, "group": 128, "tokens": T,
                   "l2": f"timed loop rotates over {L} distinct packed layers "
                         f"({L * weights / 1e6:.0f} MB of planes > 126 MB L2); one CUDA graph per layer",
                   "replicas": ("replicas only (no data-path collective): value = slowest rank's us per step"
                                if world > 1 else "single GPU")},
        "clocks": clocks,
        "e2e": {"value": us_host, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "how": "grinqh_decode_host per launch, stream sync per step: x is copied from the pinned HOST buffer with "
                       "cudaMemcpyAsync, the VMM's second pass writes y into the pinned HOST buffer (host-mapped access); "
                       "the bytes cross PCIe inside the timed region every step",
                "value_with_y_copy_nodes": us_hostc},
        "gpu_launches": args.steps * len(fused),
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": traffic,
                     "traffic_source": (f"dram__bytes_read.sum + dram__bytes_write.sum of the step's launches, committed "
                                        f"ncu --set full capture (profiles/r02_traffic.json, taken on {traffic_on})"
                                        if traffic else "no committed capture for this mix"),
                     "kernel": f"items::vmm_items_kernel<1, 16, true> in rank mode, grinqh_vmm_rank ({len(fused)} launches per step = the whole step)",
                     "alg_bytes_per_step": step_bytes, "plane_bytes_per_step": plane_bytes,
                     "us_per_step_vmm_on_ready_schedules": us_sched,
                     "frac_vmm_on_ready_schedules": step_bytes / (us_sched * 1e-6) / 1e9 / peak,
                     "peak_source": peak_src},
        "pack": {"GBps": pack_bytes / (pack_ms * 1e-3) / 1e9, "ms_per_layer": pack_ms / L},
        "per_vmm": per_vmm,
        "steps_per_s_total": world / (us_step * 1e-6),
        "two_kernel_form": {"value": us_two, "unit": UNIT,
                            "what": "the same step as 4 x grinqh_assign + 4 x grinqh_vmm (8 launches)"},
        "threshold_assignment_fused": {"value": us_thrf, "unit": UNIT,
                                       "what": "the paper's threshold assignment (PAPER.md:61-65, thetas calibrated on 8 "
                                               "synthetic vectors) made inside the VMM launch (grinqh_vmm_thresholds)"},
    }
    if us_split:
        line["per_projection"] = {"value": us_split, "unit": UNIT,
                                  "what": "same step with one grinqh_vmm_rank launch per projection (7 launches)"}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        sample = OracleLayerSample(args.mix, args.seed)   # the full layer step, as it stands, on one host core
        t = min(sample.run() for _ in range(2))
        line["cpu_baseline"] = {"value": 1e6 * t / sample.fraction, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": sample.desc}
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------ sweep (not the contract line)
def run_sweep(args):
    """BASELINE.json configs 3 and 5: us per VMM and per assign vs average bits, per shape and token count.
    One JSON line per case on stdout (prefixed "SWEEP "), a linear fit t = a + c * bits per (shape, T)."""
    import math

    import torch

    from paper_2606_23419_b200 import binding as gq
    from paper_2606_23419_b200 import synth

    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    peak, _ = _peaks()
    gen = torch.Generator(device=dev)
    gen.manual_seed(args.seed)
    cases = [("qwen3-8b", K, N, 0.02, "normal", (1,)) for K, N in synth.QWEN3_8B_SHAPES]
    cases += [("llama3-70b", K, N, 0.015, "student_t", (1, 2, 4)) for K, N in synth.LLAMA3_70B_SHAPES]
    mixes = ["2", "3", "3.25", "4", "5", "8"]
    stream = torch.cuda.Stream(device=dev)

    def time_graph(fn, n_inner, reps=20):
        with torch.cuda.stream(stream):
            fn()
            stream.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=stream):
                fn()
            for _ in range(3):
                g.replay()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            stream.synchronize()
            a.record(stream)
            for _ in range(reps):
                g.replay()
            b.record(stream)
            stream.synchronize()
        return a.elapsed_time(b) * 1e3 / (reps * n_inner)

    for model, K, N, std, dist, Ts in cases:
        copies = int(math.ceil(300e6 / (K * N))) + 1          # > 2 x L2 of 8-bit codes, rotated
        packed = []
        for c in range(copies):
            W = (torch.randn((K, N), generator=gen, device=dev, dtype=torch.float32) * std).to(torch.float16)
            packed.append(gq.grinqh_pack(W))
            del W
        for T in Ts:
            ws = gq.grinqh_vmm_workspace(T, K, N, dev)
            x = torch.from_numpy(synth.make_x(T, K, args.seed + 7, dist)).to(dev)
            y = torch.empty((T, N), dtype=torch.float32, device=dev)
            pts = []
            for mix in mixes:
                counts = gq.grinqh_mix_to_counts(K, synth.MIXES[mix])
                a = gq.Assignment(T, K, dev)
                gq.grinqh_assign(x, counts, a)
                torch.cuda.synchronize()
                union_bits = float(a.bits_union.sum().item()) / K
                us_vmm = time_graph(lambda: [gq.grinqh_vmm_rank(x, counts, w, y, ws) for w in packed], copies)
                us_sched = time_graph(lambda: [gq.grinqh_vmm(w, a, y, ws) for w in packed], copies)
                us_asg = time_graph(lambda: [gq.grinqh_assign(x, counts, a) for _ in range(8)], 8)
                ab = alg_bytes(K, N, T, int(a.bits_union.sum().item()))
                rec = {"model": model, "K": K, "N": N, "T": T, "mix": mix,
                       "avg_bits_per_token": synth.mix_avg_bits(synth.MIXES[mix]), "union_bits": union_bits,
                       "us_vmm_rank": us_vmm, "us_vmm_on_ready_schedule": us_sched, "us_assign": us_asg,
                       "alg_MB": ab / 1e6, "GBps": ab / us_vmm / 1e3, "frac_of_measured_hbm": ab / us_vmm / 1e3 / peak}
                pts.append((union_bits, us_vmm))
                print("SWEEP " + json.dumps(rec), flush=True)
            n = len(pts)
            mx, my = sum(p[0] for p in pts) / n, sum(p[1] for p in pts) / n
            c = sum((p[0] - mx) * (p[1] - my) for p in pts) / sum((p[0] - mx) ** 2 for p in pts)
            a0 = my - c * mx
            ss_res = sum((p[1] - (a0 + c * p[0])) ** 2 for p in pts)
            ss_tot = sum((p[1] - my) ** 2 for p in pts)
            print("SWEEP " + json.dumps({"model": model, "K": K, "N": N, "T": T, "fit": "us_vmm_rank = a + c * union_bits",
                                         "a_us": a0, "c_us_per_bit": c, "r2": 1 - ss_res / ss_tot}), flush=True)
        del packed
        torch.cuda.empty_cache()


# ------------------------------------------------------------------------------------------ 32-layer decode step
def run_decode_step(args):
    """BASELINE.json configs[3]: all linear layers of a 32-layer Llama-3-8B-shaped model (6.98 G weights packed to
    bit planes, ~7 GB), fresh heavy-tailed activations per layer, per-layer rank assignment, ONE CUDA graph of
    32 x (4 assigns + 4 VMM launches).  One JSON line per mix, prefixed "DECODE "."""
    import torch

    from paper_2606_23419_b200 import binding as gq
    from paper_2606_23419_b200 import synth

    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    peak, _ = _peaks()
    gen = torch.Generator(device=dev)
    gen.manual_seed(args.seed)
    import numpy as np
    NL, T = 32, 1
    fused = synth.LLAMA3_8B_LAYER_FUSED
    in_dims = synth.LLAMA3_8B_INPUT_DIMS
    packed = []
    for l in range(NL):
        d = {}
        for name, K, N, _ in fused:
            W = (torch.randn((K, N), generator=gen, device=dev, dtype=torch.float32) * 0.02).to(torch.float16)
            d[name] = gq.grinqh_pack(W)
            del W
        packed.append(d)
    xs = [{n: torch.from_numpy(synth.make_x(T, K, args.seed + 17 * l + i, "student_t")).to(dev)
           for i, (n, K) in enumerate(in_dims.items())} for l in range(NL)]
    assigns = [{n: gq.Assignment(T, K, dev) for n, K in in_dims.items()} for _ in range(NL)]
    ys = [{name: torch.empty((T, N), dtype=torch.float32, device=dev) for name, K, N, _ in fused} for _ in range(NL)]
    _, Kw, Nw, _ = max(fused, key=lambda s: gq.grinqh_vmm_workspace_bytes(T, s[1], s[2]))
    ws = gq.grinqh_vmm_workspace(T, Kw, Nw, dev)
    stream = torch.cuda.Stream(device=dev)
    for mix in ("2", "3", "4", "8"):
        counts = {K: gq.grinqh_mix_to_counts(K, synth.MIXES[mix]) for K in set(in_dims.values())}

        def step():            # 128 launches: the rank assignment inside every VMM launch
            for l in range(NL):
                for name, K, N, inp in fused:
                    gq.grinqh_vmm_rank(xs[l][inp], counts[K], packed[l][name], ys[l][name], ws)

        for l in range(NL):    # (the assignments themselves, for the byte accounting below)
            for n_, K_ in in_dims.items():
                gq.grinqh_assign(xs[l][n_], counts[K_], assigns[l][n_])

        with torch.cuda.stream(stream):
            step()
            stream.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=stream):
                step()
            for _ in range(3):
                g.replay()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            stream.synchronize()
            reps = 20
            a.record(stream)
            for _ in range(reps):
                g.replay()
            b.record(stream)
            stream.synchronize()
        us = a.elapsed_time(b) * 1e3 / reps
        # the same decode step with the paper's threshold assignment made inside the VMM launches (128 launches)
        thetas = {n: gq.grinqh_calibrate_thresholds(
            torch.from_numpy(np.concatenate([synth.make_x(1, K, 9000 + 10 * i + s_, "student_t") for s_ in range(8)])),
            counts[K]) for i, (n, K) in enumerate(in_dims.items())}

        def step_thr():
            for l in range(NL):
                for name, K, N, inp in fused:
                    gq.grinqh_vmm_thresholds(xs[l][inp], thetas[inp], packed[l][name], ys[l][name], ws)

        with torch.cuda.stream(stream):
            step_thr()
            stream.synchronize()
            g2 = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g2, stream=stream):
                step_thr()
            for _ in range(3):
                g2.replay()
            a2, b2 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            stream.synchronize()
            a2.record(stream)
            for _ in range(reps):
                g2.replay()
            b2.record(stream)
            stream.synchronize()
        us_thr = a2.elapsed_time(b2) * 1e3 / reps
        nbytes = sum(alg_bytes(K, N, T, int(assigns[l][inp].bits_union.sum().item()))
                     for l in range(NL) for name, K, N, inp in fused)
        print("DECODE " + json.dumps({"workload": "32-layer llama3-8b-shaped decode step, 128 grinqh_vmm_rank launches in one CUDA graph",
                                      "mix": mix, "avg_bits": synth.mix_avg_bits(synth.MIXES[mix]), "us_per_decode_step": us,
                                      "us_per_decode_step_thresholds_fused": us_thr,
                                      "alg_GB": nbytes / 1e9, "GBps": nbytes / us / 1e3,
                                      "frac_of_measured_hbm": nbytes / us / 1e3 / peak}), flush=True)


# ------------------------------------------------------------------------------------------ prefill half (f3)
def run_prefill(args):
    """SURVEY.md 8f3 / PAPER.md:101: unpack at b_max (grinqh_unpack), then a dense library GEMM on the result.
    One JSON line per shape, prefixed "PREFILL "."""
    import torch

    from paper_2606_23419_b200 import binding as gq

    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    peak, _ = _peaks()
    gen = torch.Generator(device=dev)
    gen.manual_seed(args.seed)
    tokens = 3000                                       # the paper's 3000:1 prefill benchmark
    for K, N in [(4096, 14336), (14336, 4096), (8192, 28672)]:
        W = (torch.randn((K, N), generator=gen, device=dev) * 0.02).half()
        w = gq.grinqh_pack(W)
        out = torch.empty_like(W)
        X = torch.randn((tokens, K), device=dev, dtype=torch.float16)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

        def timed(fn, reps):
            for _ in range(3):
                fn()
            torch.cuda.synchronize()
            a.record()
            for _ in range(reps):
                fn()
            b.record()
            torch.cuda.synchronize()
            return a.elapsed_time(b) * 1e3 / reps

        us_unpack = timed(lambda: gq.grinqh_unpack(w, out), 20)
        us_gemm = timed(lambda: torch.matmul(X, out), 10)
        Y = torch.empty((tokens, N), device=dev, dtype=torch.float16)
        us_fused = timed(lambda: gq.grinqh_prefill_gemm(X, w, Y), 10)   # f3: unpack fused into the tcgen05 GEMM
        same = bool(torch.equal(Y, torch.matmul(X, out)))
        tf_peak, tf_src = _tensor_peak()
        flops = 2 * tokens * K * N
        print("PREFILL " + json.dumps({"K": K, "N": N, "tokens": tokens, "us_unpack": us_unpack,
                                       "unpack_GBps": K * N * 3 / us_unpack / 1e3,
                                       "unpack_frac_of_measured_hbm": K * N * 3 / us_unpack / 1e3 / peak,
                                       "us_dense_gemm_fp16_torch": us_gemm,
                                       "gemm_TFLOPs": flops / us_gemm / 1e6,
                                       "unpack_over_gemm": us_unpack / us_gemm,
                                       "us_fused_prefill_gemm": us_fused,
                                       "fused_TFLOPs": flops / us_fused / 1e6,
                                       "fused_over_unpack_plus_gemm": us_fused / (us_unpack + us_gemm),
                                       "fused_equals_library_path_bitwise": same,
                                       "roofline": {"bound": "tensor", "achieved": flops / us_fused / 1e6, "peak": tf_peak,
                                                    "unit": "TFLOP/s", "frac": flops / us_fused / 1e6 / tf_peak,
                                                    "peak_source": tf_src, "kernel": "prefill_kernel (tcgen05, fp16 dense)"}}),
              flush=True)
        del Y
        del W, w, out, X


# ------------------------------------------------------------------------------------------ f2: 2-bit segments A/B
def run_seg2(args):
    """SURVEY.md 8f2 / PAPER.md:79-81, :442: the same weights in the paper's 2-bit-segment store (b_max = 8) and in the
    1-bit plane store, rank assignment inside the launch, per mix.  One JSON line per case, prefixed "SEG2 "."""
    import math

    import torch

    from paper_2606_23419_b200 import binding as gq
    from paper_2606_23419_b200 import synth

    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    peak, _ = _peaks()
    gen = torch.Generator(device=dev)
    gen.manual_seed(args.seed)
    stream = torch.cuda.Stream(device=dev)

    def time_graph(fn, n_inner, reps=20):
        with torch.cuda.stream(stream):
            fn()
            stream.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=stream):
                fn()
            for _ in range(3):
                g.replay()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            stream.synchronize()
            a.record(stream)
            for _ in range(reps):
                g.replay()
            b.record(stream)
            stream.synchronize()
        return a.elapsed_time(b) * 1e3 / (reps * n_inner)

    for K, N in [(4096, 28672), (8192, 28672), (14336, 4096)]:
        copies = int(math.ceil(300e6 / (K * N))) + 1          # > 2 x L2 of 8-bit codes, rotated
        planes, segs = [], []
        for c in range(copies):
            W = (torch.randn((K, N), generator=gen, device=dev, dtype=torch.float32) * 0.02).to(torch.float16)
            planes.append(gq.grinqh_pack(W))
            segs.append(gq.grinqh_pack_seg2(W, 8))
            del W
        ws = gq.grinqh_vmm_workspace(1, K, N, dev)
        x = torch.from_numpy(synth.make_x(1, K, args.seed + 7, "normal")).to(dev)
        y = torch.empty((1, N), dtype=torch.float32, device=dev)
        for mix in ["2", "3", "4", "5", "8"]:
            counts = gq.grinqh_mix_to_counts(K, synth.MIXES[mix])
            bits = sum(w * c for w, c in enumerate(counts))
            ab = alg_bytes(K, N, 1, bits)
            us_p = time_graph(lambda: [gq.grinqh_vmm_rank(x, counts, w, y, ws) for w in planes], copies)
            us_s = time_graph(lambda: [gq.grinqh_vmm_rank_seg2(x, counts, w, y, ws) for w in segs], copies)
            print("SEG2 " + json.dumps({"K": K, "N": N, "mix": mix, "avg_bits": bits / K, "alg_MB": ab / 1e6,
                                        "us_planes": us_p, "us_seg2": us_s, "seg2_over_planes": us_s / us_p,
                                        "frac_planes": ab / us_p / 1e3 / peak, "frac_seg2": ab / us_s / 1e3 / peak}),
                  flush=True)
        del planes, segs
        torch.cuda.empty_cache()


def main():
    args = _args()
    if args.seg2:
        run_seg2(args)
    elif args.prefill:
        run_prefill(args)
    elif args.decode_step:
        run_decode_step(args)
    elif args.sweep:
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_native(args)


if __name__ == "__main__":
    main()
