"""CPU oracle for the GRINQH decode hot path — TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this package.  It never imports paper_2606_23419_b200 and shares no code with it.
Thin ctypes marshalling over oracle/grinqh_oracle.cpp (numpy arrays in, numpy arrays out).
"""
import ctypes as C

import numpy as np

from .build import build as _build

GCNT_STRIDE = 16

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.orc_half_to_float.restype = C.c_float
        _lib.orc_half_to_float.argtypes = [C.c_uint16]
        _lib.orc_float_to_half.restype = C.c_uint16
        _lib.orc_float_to_half.argtypes = [C.c_float]
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _u16(a):
    """fp16 array (or raw uint16 patterns) -> contiguous uint16 view."""
    a = np.ascontiguousarray(a)
    if a.dtype == np.float16:
        return a.view(np.uint16)
    assert a.dtype == np.uint16, a.dtype
    return a


def half_to_float(h: int) -> float:
    return float(lib().orc_half_to_float(int(h)))


def float_to_half(f: float) -> int:
    return int(lib().orc_float_to_half(C.c_float(f)))


def code_prime(q: int, b: int) -> int:
    return int(lib().orc_code_prime(int(q), int(b)))


def mix_to_counts(K: int, frac) -> np.ndarray:
    frac = np.ascontiguousarray(frac, dtype=np.float64)
    assert frac.shape == (9,)
    counts = np.zeros(9, dtype=np.uint32)
    rc = lib().orc_mix_to_counts(int(K), _p(frac), _p(counts))
    if rc:
        raise ValueError(f"orc_mix_to_counts failed: {rc}")
    return counts


def pack(W, G: int = 128):
    """W [K, N] fp16 -> planes [8, K, N/32] u32, scales [K/G, N] fp16, zeros [K/G, N] fp16."""
    Wb = _u16(W)
    K, N = Wb.shape
    planes = np.zeros((8, K, N // 32), dtype=np.uint32)
    scales = np.zeros((K // G, N), dtype=np.uint16)
    zeros = np.zeros((K // G, N), dtype=np.uint16)
    rc = lib().orc_pack(_p(Wb), K, N, G, _p(planes), _p(scales), _p(zeros))
    if rc:
        raise ValueError(f"orc_pack failed: {rc}")
    return planes, scales.view(np.float16), zeros.view(np.float16)


def codes(planes) -> np.ndarray:
    planes = np.ascontiguousarray(planes, dtype=np.uint32)
    _, K, words = planes.shape
    q = np.zeros((K, words * 32), dtype=np.uint8)
    lib().orc_codes(_p(planes), K, words * 32, _p(q))
    return q


def rank_bruteforce(x) -> np.ndarray:
    xb = _u16(x).reshape(-1)
    r = np.zeros(xb.shape[0], dtype=np.int32)
    lib().orc_rank_bruteforce(_p(xb), xb.shape[0], _p(r))
    return r


def assign(x, counts, G: int = 128):
    """x [T, K] fp16 -> dict(bits [T,K] u8, bits_union [K] u8, rows [K] i32, cnt_ge [10] i32,
    grows [K] u8, gcnt_ge [K/G, 16] u8)."""
    xb = _u16(x)
    if xb.ndim == 1:
        xb = xb[None, :]
    T, K = xb.shape
    counts = np.ascontiguousarray(counts, dtype=np.uint32)
    out = dict(
        bits=np.zeros((T, K), dtype=np.uint8),
        bits_union=np.zeros(K, dtype=np.uint8),
        rows=np.zeros(K, dtype=np.int32),
        cnt_ge=np.zeros(10, dtype=np.int32),
        grows=np.zeros(K, dtype=np.uint8),
        gcnt_ge=np.zeros((K // G, GCNT_STRIDE), dtype=np.uint8),
    )
    rc = lib().orc_assign(_p(xb), T, K, G, _p(counts), _p(out["bits"]), _p(out["bits_union"]), _p(out["rows"]),
                          _p(out["cnt_ge"]), _p(out["grows"]), _p(out["gcnt_ge"]), GCNT_STRIDE)
    if rc:
        raise ValueError(f"orc_assign failed: {rc}")
    return out


def assign_thresholds(x, theta, G: int = 128):
    """Threshold form.  theta: 9 fp16 magnitude patterns (uint16), theta[w] = smallest magnitude
    that still gets >= w bits (0x8000 = unreachable), theta[0] ignored.  Same outputs as assign()."""
    xb = _u16(x)
    if xb.ndim == 1:
        xb = xb[None, :]
    T, K = xb.shape
    theta = np.ascontiguousarray(theta, dtype=np.uint16)
    assert theta.shape == (9,)
    out = dict(
        bits=np.zeros((T, K), dtype=np.uint8),
        bits_union=np.zeros(K, dtype=np.uint8),
        rows=np.zeros(K, dtype=np.int32),
        cnt_ge=np.zeros(10, dtype=np.int32),
        grows=np.zeros(K, dtype=np.uint8),
        gcnt_ge=np.zeros((K // G, GCNT_STRIDE), dtype=np.uint8),
    )
    rc = lib().orc_assign_thresholds(_p(xb), T, K, G, _p(theta), _p(out["bits"]), _p(out["bits_union"]),
                                     _p(out["rows"]), _p(out["cnt_ge"]), _p(out["grows"]), _p(out["gcnt_ge"]),
                                     GCNT_STRIDE)
    if rc:
        raise ValueError(f"orc_assign_thresholds failed: {rc}")
    return out


def calibrate_thresholds(xs, counts) -> np.ndarray:
    """xs [S, K] fp16 calibration vectors -> theta [9] uint16 (Eq. 2: mean split magnitudes)."""
    xb = _u16(xs)
    S, K = xb.shape
    counts = np.ascontiguousarray(counts, dtype=np.uint32)
    theta = np.zeros(9, dtype=np.uint16)
    rc = lib().orc_calibrate_thresholds(_p(xb), S, K, _p(counts), _p(theta))
    if rc:
        raise ValueError(f"orc_calibrate_thresholds failed: {rc}")
    return theta


def _vmm_args(x, planes, scales, zeros, bits):
    xb = _u16(x)
    if xb.ndim == 1:
        xb = xb[None, :]
    T, K = xb.shape
    planes = np.ascontiguousarray(planes, dtype=np.uint32)
    N = planes.shape[2] * 32
    sb, zb = _u16(scales), _u16(zeros)
    bits = np.ascontiguousarray(bits, dtype=np.uint8).reshape(T, K)
    return xb, T, K, N, planes, sb, zb, bits


def vmm(x, planes, scales, zeros, bits, G: int = 128, cols=None) -> np.ndarray:
    """Definitional fp64 VMM.  cols: optional int32 column subset."""
    xb, T, K, N, planes, sb, zb, bits = _vmm_args(x, planes, scales, zeros, bits)
    if cols is None:
        y = np.zeros((T, N), dtype=np.float64)
        rc = lib().orc_vmm(_p(xb), T, K, N, G, _p(planes), _p(sb), _p(zb), _p(bits), _p(y))
    else:
        cols = np.ascontiguousarray(cols, dtype=np.int32)
        y = np.zeros((T, cols.shape[0]), dtype=np.float64)
        rc = lib().orc_vmm_cols(_p(xb), T, K, N, G, _p(planes), _p(sb), _p(zb), _p(bits), _p(cols),
                                int(cols.shape[0]), _p(y))
    if rc:
        raise ValueError(f"orc_vmm failed: {rc}")
    return y


def vmm_planewise(x, planes, scales, zeros, bits, G: int = 128) -> np.ndarray:
    xb, T, K, N, planes, sb, zb, bits = _vmm_args(x, planes, scales, zeros, bits)
    y = np.zeros((T, N), dtype=np.float64)
    rc = lib().orc_vmm_planewise(_p(xb), T, K, N, G, _p(planes), _p(sb), _p(zb), _p(bits), _p(y))
    if rc:
        raise ValueError(f"orc_vmm_planewise failed: {rc}")
    return y


def dequant(planes, scales, zeros, b: int, G: int = 128) -> np.ndarray:
    planes = np.ascontiguousarray(planes, dtype=np.uint32)
    _, K, words = planes.shape
    N = words * 32
    w = np.zeros((K, N), dtype=np.float64)
    lib().orc_dequant(_p(planes), _p(_u16(scales)), _p(_u16(zeros)), K, N, G, int(b), _p(w))
    return w


# ---- 2-bit-segment store, bmax in {4, 6, 8}
def code2_prime(q: int, b: int, bmax: int) -> int:
    return int(lib().orc_code2_prime(int(q), int(b), int(bmax)))


def pack2(W, bmax: int, G: int = 128):
    """W [K, N] fp16 -> segs [bmax/2, K, N/16] uint32, scales / zeros [K/G, N] fp16."""
    W = np.ascontiguousarray(W)
    K, N = W.shape
    segs = np.zeros((bmax // 2, K, N // 16), dtype=np.uint32)
    s = np.zeros((K // G, N), dtype=np.float16)
    z = np.zeros((K // G, N), dtype=np.float16)
    rc = lib().orc_pack2(_p(_u16(W)), K, N, G, int(bmax), _p(segs), _p(s.view(np.uint16)), _p(z.view(np.uint16)))
    if rc:
        raise ValueError(f"orc_pack2 failed: {rc}")
    return segs, s, z


def codes2(segs, bmax: int) -> np.ndarray:
    _, K, words = segs.shape
    q = np.zeros((K, words * 16), dtype=np.uint8)
    lib().orc_codes2(_p(np.ascontiguousarray(segs)), K, words * 16, int(bmax), _p(q))
    return q


def vmm2(x, segs, scales, zeros, bits, bmax: int, G: int = 128, cols=None) -> np.ndarray:
    x = np.ascontiguousarray(x)
    T, K = x.shape
    N = segs.shape[2] * 16
    bits = np.ascontiguousarray(bits, dtype=np.uint8)
    if cols is None:
        ncols, cp = N, None
    else:
        cols = np.ascontiguousarray(cols, dtype=np.int32)
        ncols, cp = len(cols), _p(cols)
    y = np.zeros((T, ncols), dtype=np.float64)
    rc = lib().orc_vmm2_cols(_p(_u16(x)), T, K, N, G, int(bmax), _p(np.ascontiguousarray(segs)),
                             _p(_u16(scales)), _p(_u16(zeros)), _p(bits), cp, ncols, _p(y))
    if rc:
        raise ValueError(f"orc_vmm2_cols failed: {rc}")
    return y


def dequant2(segs, scales, zeros, bmax: int, b: int, G: int = 128) -> np.ndarray:
    _, K, words = segs.shape
    w = np.zeros((K, words * 16), dtype=np.float64)
    rc = lib().orc_dequant2(_p(np.ascontiguousarray(segs)), _p(_u16(scales)), _p(_u16(zeros)), K, words * 16, G,
                            int(bmax), int(b), _p(w))
    if rc:
        raise ValueError(f"orc_dequant2 failed: {rc}")
    return w
