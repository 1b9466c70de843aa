"""Independent numpy helpers for the oracle pins (no oracle code, no CUDA code)."""
import numpy as np


def np_unpack_codes(planes: np.ndarray, upto: int = 8) -> np.ndarray:
    """Codes re-assembled with numpy from the first `upto` planes: plane j carries code bit (7 - j),
    column n sits at bit (n & 31) of word n >> 5 (include/grinqh.h)."""
    _, K, words = planes.shape
    N = words * 32
    n = np.arange(N)
    q = np.zeros((K, N), dtype=np.int64)
    for j in range(upto):
        bit = (planes[j][:, n >> 5] >> (n & 31).astype(np.uint32)) & 1
        q |= bit.astype(np.int64) << (7 - j)
    return q


def paper_w_hat(q8: np.ndarray, s: np.ndarray, z: np.ndarray, b: int) -> np.ndarray:
    """The printed reconstruction: w = s * (q_b * 2^(bmax-b) + phi) + z with
    phi = 2^(bmax-b-1), q_b = top b bits of the 8-bit code; readings #5 (phi_8 = 0) and #7 (b = 0 -> 0)."""
    s = s.astype(np.float64)
    z = z.astype(np.float64)
    if b == 0:
        return np.zeros_like(s * q8)
    q_b = q8 >> (8 - b)
    phi = 0.0 if b == 8 else 2.0 ** (8 - b - 1)
    return s * (q_b * 2.0 ** (8 - b) + phi) + z


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    d = np.linalg.norm(a - b)
    n = np.linalg.norm(b)
    return d / n if n > 0 else d


def expected_gsched(ref: dict, x: np.ndarray, G: int = 128) -> np.ndarray:
    """include/grinqh.h `gsched`: a pure re-indexing of the oracle's assignment outputs and of x.
    entry [t][G g + i]: r = grows[G g + i], k = G g + r ->
    r | bits[t][k] << 8 | bits_union[k] << 12 | fp16 pattern of x[t][k] << 16."""
    xb = np.ascontiguousarray(x).view(np.uint16).reshape(ref["bits"].shape).astype(np.uint32)
    T, K = xb.shape
    r = ref["grows"].astype(np.uint32)
    k = (np.arange(K, dtype=np.uint32) // G) * G + r
    out = np.empty((T, K), dtype=np.uint32)
    for t in range(T):
        out[t] = r | (ref["bits"][t][k].astype(np.uint32) << 8) | (ref["bits_union"][k].astype(np.uint32) << 12) \
            | (xb[t][k] << 16)
    return out
