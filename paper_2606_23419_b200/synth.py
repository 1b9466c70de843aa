"""Seeded synthetic inputs for the GRINQH decode hot path.

This module serves BOTH the CUDA path's tests/bench and the CPU oracle's tests.  It holds none of the
method's arithmetic: only random tensors with the shapes, value distributions and structure of the
paper's workloads (BASELINE.json configs; recipe in DESIGN.md "Input recipe"), and the named level
mixes (precision distributions P) as plain fractions.  numpy only.
"""
from __future__ import annotations

import numpy as np

# ---------------------------------------------------------------------------------------------
# Level mixes: frac[w] = share of input channels at w bits (w = 0..8).  BASELINE.json configs use
# levels {8, 4, 2, 0}.  "3.25" is BASELINE.json's "avg 3" mix verbatim (it averages 3.25 bits,
# DESIGN.md reading #15); "3" is an exact-3 mix over the same levels.
# ---------------------------------------------------------------------------------------------


def _mix(d):
    f = [0.0] * 9
    for w, p in d.items():
        f[w] = float(p)
    return tuple(f)


MIXES = {
    "2": _mix({8: 1 / 32, 4: 6 / 32, 2: 16 / 32, 0: 9 / 32}),
    "3": _mix({8: 4 / 32, 4: 8 / 32, 2: 16 / 32, 0: 4 / 32}),
    "3.25": _mix({8: 0.125, 4: 0.375, 2: 0.375, 0: 0.125}),
    "4": _mix({8: 0.25, 4: 0.375, 2: 0.25, 0: 0.125}),
    "5": _mix({8: 14 / 32, 4: 10 / 32, 2: 4 / 32, 0: 4 / 32}),
    "8": _mix({8: 1.0}),
    "0": _mix({0: 1.0}),
}


def mix_avg_bits(frac) -> float:
    return float(sum(w * p for w, p in enumerate(frac)))


# Layer shapes (K = d_in, N = d_out) of BASELINE.json configs 2, 3, 5.
LLAMA3_8B_LAYER = (
    ("q", 4096, 4096), ("k", 4096, 1024), ("v", 4096, 1024), ("o", 4096, 4096),
    ("gate", 4096, 14336), ("up", 4096, 14336), ("down", 14336, 4096),
)
# which input vector each projection consumes: q/k/v share one, gate/up share one (reading #13)
LLAMA3_8B_INPUTS = {"q": "attn_in", "k": "attn_in", "v": "attn_in", "o": "o_in",
                    "gate": "mlp_in", "up": "mlp_in", "down": "down_in"}
LLAMA3_8B_INPUT_DIMS = {"attn_in": 4096, "o_in": 4096, "mlp_in": 4096, "down_in": 14336}
# launch plan of the same layer with same-input projections concatenated along N (the quantiser is per column, so
# packing [W_q | W_k | W_v] equals concatenating the three packs): 4 VMM launches instead of 7
LLAMA3_8B_LAYER_FUSED = (
    ("qkv", 4096, 4096 + 1024 + 1024, "attn_in"), ("o", 4096, 4096, "o_in"),
    ("gate_up", 4096, 2 * 14336, "mlp_in"), ("down", 14336, 4096, "down_in"),
)
QWEN3_8B_SHAPES = ((4096, 4096), (4096, 1024), (4096, 12288), (12288, 4096))
LLAMA3_70B_SHAPES = ((8192, 8192), (8192, 1024), (8192, 28672), (28672, 8192))


def make_weights(K: int, N: int, std: float = 0.02, seed: int = 0) -> np.ndarray:
    """W [K, N] fp16 ~ N(0, std)."""
    rng = np.random.default_rng([seed, K, N, 0x57])
    return (rng.standard_normal((K, N), dtype=np.float32) * np.float32(std)).astype(np.float16)


def make_x(T: int, K: int, seed: int = 0, dist: str = "normal", outlier_frac: float = 0.01,
           n_outliers: int | None = None, outlier_scale: float = 20.0) -> np.ndarray:
    """x [T, K] fp16.  dist = "normal" (N(0,1)) or "student_t" (nu = 4, heavy-tailed).
    A fixed set of outlier channels (same indices for every token, config 5) is multiplied by
    outlier_scale: n_outliers channels if given, else round(outlier_frac * K)."""
    rng = np.random.default_rng([seed, T, K, 0x58])
    if dist == "normal":
        x = rng.standard_normal((T, K), dtype=np.float32)
    elif dist == "student_t":
        x = rng.standard_t(4.0, size=(T, K)).astype(np.float32)
    else:
        raise ValueError(dist)
    n_out = int(round(outlier_frac * K)) if n_outliers is None else int(n_outliers)
    if n_out > 0:
        ch = rng.choice(K, size=n_out, replace=False)
        x[:, ch] *= np.float32(outlier_scale)
    x = np.clip(x, -60000.0, 60000.0)  # generators never emit non-finite fp16
    return x.astype(np.float16)


def tiny_config(seed: int = 0):
    """BASELINE.json configs[0]: x [1,256] ~N(0,1) with 4 outlier channels x20; W [256,512] ~N(0,0.02);
    level mix avg 4."""
    W = make_weights(256, 512, 0.02, seed)
    x = make_x(1, 256, seed, "normal", n_outliers=4)
    return W, x, MIXES["4"]
