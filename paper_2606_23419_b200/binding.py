"""Thin Python binding over the C ABI in include/grinqh.h (argument marshalling only).

Every step of the path runs inside csrc/libgrinqh.so; torch is used for device memory and streams.
There is no CPU fallback: if the shared library is missing the import raises.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "csrc", "libgrinqh.so")

GROUP = 128
GCNT_STRIDE = 16
MAX_T = 4
MAX_K = 32768

if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} is missing: build it with `python -m paper_2606_23419_b200.build` "
        "(or __graft_entry__.build()).  There is no CPU fallback for the GRINQH path.")

_lib = C.CDLL(LIB_PATH)

_vp, _i, _sz = C.c_void_p, C.c_int, C.c_size_t
_lib.grinqh_status_string.restype = C.c_char_p
_lib.grinqh_status_string.argtypes = [_i]
_lib.grinqh_version.restype = _i
_lib.grinqh_mix_to_counts.restype = _i
_lib.grinqh_mix_to_counts.argtypes = [_i, _vp, _vp]
_lib.grinqh_pack.restype = _i
_lib.grinqh_pack.argtypes = [_vp, _i, _i, _i, _vp, _vp, _vp, _vp]
_lib.grinqh_unpack.restype = _i
_lib.grinqh_unpack.argtypes = [_vp, _vp, _vp, _i, _i, _i, _vp, _vp]
_lib.grinqh_assign_workspace_bytes.restype = _sz
_lib.grinqh_assign_workspace_bytes.argtypes = [_i, _i]
_lib.grinqh_assign.restype = _i
_lib.grinqh_assign.argtypes = [_vp, _i, _i, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _sz, _vp]
_lib.grinqh_assign_thresholds.restype = _i
_lib.grinqh_assign_thresholds.argtypes = [_vp, _i, _i, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp]
_lib.grinqh_calibrate_thresholds.restype = _i
_lib.grinqh_calibrate_thresholds.argtypes = [_vp, _i, _i, _vp, _vp]
_lib.grinqh_vmm_workspace_bytes.restype = _sz
_lib.grinqh_vmm_workspace_bytes.argtypes = [_i, _i, _i]
_lib.grinqh_vmm_workspace_init.restype = _i
_lib.grinqh_vmm_workspace_init.argtypes = [_vp, _sz, _vp]
_VMM_COMMON = [_i, _i, _i, _i, _vp, _vp, _vp, _vp, _vp]
_lib.grinqh_vmm.restype = _i
_lib.grinqh_vmm.argtypes = _VMM_COMMON + [_vp, _vp, _sz, _vp]
_lib.grinqh_vmm_thresholds.restype = _i
_lib.grinqh_vmm_thresholds.argtypes = [_vp, _i, _i, _i, _i, _vp, _vp, _vp, _vp, _vp, _vp, _sz, _vp]
_lib.grinqh_vmm_rank.restype = _i
_lib.grinqh_vmm_rank.argtypes = [_vp, _i, _i, _i, _i, _vp, _vp, _vp, _vp, _vp, _vp, _sz, _vp]
_lib.grinqh_vmm_rank_static.restype = _i
_lib.grinqh_vmm_rank_static.argtypes = [_vp, _i, _i, _i, _i, _vp, _vp, _vp, _vp, _vp, _vp]
_lib.grinqh_prefill_gemm.restype = _i
_lib.grinqh_prefill_gemm.argtypes = [_vp, _i, _i, _i, _i, _vp, _vp, _vp, _vp, _vp]
_lib.grinqh_static_scratch_bytes.restype = _sz
_lib.grinqh_static_scratch_bytes.argtypes = []
_lib.grinqh_pack_seg2.restype = _i
_lib.grinqh_pack_seg2.argtypes = [_vp, _i, _i, _i, _i, _vp, _vp, _vp, _vp]
_lib.grinqh_vmm_rank_seg2.restype = _i
_lib.grinqh_vmm_rank_seg2.argtypes = [_vp, _i, _i, _i, _i, _i, _vp, _vp, _vp, _vp, _vp, _vp, _sz, _vp]
_lib.grinqh_vmm_main.restype = _i
_lib.grinqh_vmm_main.argtypes = _VMM_COMMON + [_vp, _sz, _vp]
_lib.grinqh_vmm_reduce.restype = _i
_lib.grinqh_vmm_reduce.argtypes = [_i, _i, _i, _vp, _vp, _sz, _vp]
_lib.grinqh_decode_host.restype = _i
_lib.grinqh_decode_host.argtypes = [_vp, _i, _i, _i, _i, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _sz, _vp, _i, _vp]

EXPORTS = ("grinqh_status_string", "grinqh_version", "grinqh_mix_to_counts", "grinqh_pack", "grinqh_unpack",
           "grinqh_assign_workspace_bytes", "grinqh_assign", "grinqh_assign_thresholds",
           "grinqh_calibrate_thresholds", "grinqh_vmm_workspace_bytes",
           "grinqh_vmm_workspace_init", "grinqh_vmm", "grinqh_vmm_thresholds", "grinqh_vmm_rank",
           "grinqh_vmm_main", "grinqh_vmm_reduce", "grinqh_decode_host", "grinqh_pack_seg2", "grinqh_vmm_rank_seg2",
           "grinqh_static_scratch_bytes", "grinqh_vmm_rank_static", "grinqh_prefill_gemm")


class GrinqhError(RuntimeError):
    pass


def _check(rc: int, what: str):
    if rc != 0:
        raise GrinqhError(f"{what}: {_lib.grinqh_status_string(rc).decode()} ({rc})")


def _stream(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return stream.cuda_stream


def _dev(t: torch.Tensor, dtype, name: str) -> int:
    if not (t.is_cuda and t.is_contiguous() and t.dtype == dtype):
        raise GrinqhError(f"{name}: need a contiguous CUDA tensor of {dtype}, got {t.dtype} on {t.device}")
    return t.data_ptr()


def grinqh_version() -> int:
    return int(_lib.grinqh_version())


def grinqh_status_string(rc: int) -> str:
    return _lib.grinqh_status_string(int(rc)).decode()


def grinqh_mix_to_counts(K: int, frac) -> list[int]:
    f = (C.c_double * 9)(*[float(v) for v in frac])
    c = (C.c_uint32 * 9)()
    _check(_lib.grinqh_mix_to_counts(int(K), f, c), "grinqh_mix_to_counts")
    return [int(v) for v in c]


def _counts(counts):
    return (C.c_uint32 * 9)(*[int(v) for v in counts])


class Packed:
    """Device-resident packed weight: planes [8, K, N/32] int32 (bit patterns), scales/zeros [K/128, N] fp16."""

    def __init__(self, K: int, N: int, device="cuda"):
        self.K, self.N = K, N
        self.planes = torch.empty((8, K, N // 32), dtype=torch.int32, device=device)
        self.scales = torch.empty((K // GROUP, N), dtype=torch.float16, device=device)
        self.zeros = torch.empty((K // GROUP, N), dtype=torch.float16, device=device)


def grinqh_pack(W: torch.Tensor, out: Packed | None = None, stream=None) -> Packed:
    K, N = W.shape
    out = out or Packed(K, N, W.device)
    _check(_lib.grinqh_pack(_dev(W, torch.float16, "W"), K, N, GROUP, out.planes.data_ptr(),
                            out.scales.data_ptr(), out.zeros.data_ptr(), _stream(stream)), "grinqh_pack")
    return out


def grinqh_unpack(w: Packed, out: torch.Tensor | None = None, stream=None) -> torch.Tensor:
    """Full-precision dequantised weights [K, N] fp16 (prefill path: unpack at b_max, then a dense GEMM)."""
    if out is None:
        out = torch.empty((w.K, w.N), dtype=torch.float16, device=w.planes.device)
    _check(_lib.grinqh_unpack(w.planes.data_ptr(), w.scales.data_ptr(), w.zeros.data_ptr(), w.K, w.N, GROUP,
                              _dev(out, torch.float16, "W"), _stream(stream)), "grinqh_unpack")
    return out


class Assignment:
    """Device buffers written by grinqh_assign for one [T, K] input."""

    def __init__(self, T: int, K: int, device="cuda"):
        self.T, self.K = T, K
        self.bits = torch.empty((T, K), dtype=torch.uint8, device=device)
        self.bits_union = torch.empty((K,), dtype=torch.uint8, device=device)
        self.rows = torch.empty((K,), dtype=torch.int32, device=device)
        self.cnt_ge = torch.empty((16,), dtype=torch.int32, device=device)  # 10 used; padded for alignment
        self.grows = torch.empty((K,), dtype=torch.uint8, device=device)
        self.gcnt_ge = torch.empty((K // GROUP, GCNT_STRIDE), dtype=torch.uint8, device=device)
        self.gsched = torch.empty((T, K), dtype=torch.int32, device=device)  # uint32 bit patterns


def grinqh_assign(x: torch.Tensor, counts, out: Assignment | None = None, stream=None) -> Assignment:
    T, K = x.shape
    out = out or Assignment(T, K, x.device)
    _check(_lib.grinqh_assign(_dev(x, torch.float16, "x"), T, K, _counts(counts), out.bits.data_ptr(),
                              out.bits_union.data_ptr(), out.rows.data_ptr(), out.cnt_ge.data_ptr(),
                              out.grows.data_ptr(), out.gcnt_ge.data_ptr(), out.gsched.data_ptr(), None, 0,
                              _stream(stream)),
           "grinqh_assign")
    return out


def grinqh_assign_thresholds(x: torch.Tensor, theta, out: Assignment | None = None, stream=None) -> Assignment:
    """Threshold form of the assignment; theta: 9 uint16 fp16-magnitude patterns (theta[0] unused)."""
    T, K = x.shape
    out = out or Assignment(T, K, x.device)
    th = (C.c_uint16 * 9)(*[int(v) for v in theta])
    _check(_lib.grinqh_assign_thresholds(_dev(x, torch.float16, "x"), T, K, th, out.bits.data_ptr(),
                                         out.bits_union.data_ptr(), out.rows.data_ptr(), out.cnt_ge.data_ptr(),
                                         out.grows.data_ptr(), out.gcnt_ge.data_ptr(), out.gsched.data_ptr(),
                                         _stream(stream)), "grinqh_assign_thresholds")
    return out


def grinqh_calibrate_thresholds(xs_host: torch.Tensor, counts) -> list[int]:
    """HOST xs [S, K] fp16 calibration vectors -> theta [9] uint16 patterns."""
    if xs_host.is_cuda or xs_host.dtype != torch.float16 or not xs_host.is_contiguous():
        raise GrinqhError("grinqh_calibrate_thresholds takes a contiguous HOST fp16 tensor [S, K]")
    S, K = xs_host.shape
    th = (C.c_uint16 * 9)()
    _check(_lib.grinqh_calibrate_thresholds(xs_host.data_ptr(), S, K, _counts(counts), th),
           "grinqh_calibrate_thresholds")
    return [int(v) for v in th]


def grinqh_vmm_workspace_bytes(T: int, K: int, N: int) -> int:
    return int(_lib.grinqh_vmm_workspace_bytes(T, K, N))


def _vmm_common(w: Packed, a: Assignment):
    if a.K != w.K:
        raise GrinqhError(f"assignment is for K={a.K}, weight has K={w.K}")
    return [a.T, a.K, w.N, GROUP, w.planes.data_ptr(), w.scales.data_ptr(), w.zeros.data_ptr(),
            a.gsched.data_ptr(), a.gcnt_ge.data_ptr()]


def grinqh_vmm_workspace(T: int, K: int, N: int, device="cuda", stream=None) -> torch.Tensor:
    """A workspace for shapes up to (T, K, N), tickets cleared (grinqh_vmm_workspace_init)."""
    ws = torch.empty((grinqh_vmm_workspace_bytes(T, K, N),), dtype=torch.uint8, device=device)
    _check(_lib.grinqh_vmm_workspace_init(ws.data_ptr(), ws.numel(), _stream(stream)), "grinqh_vmm_workspace_init")
    return ws


def _ws(T, K, N, workspace, device):
    if workspace is None:
        workspace = grinqh_vmm_workspace(T, K, N, device)
    return workspace, workspace.numel() * workspace.element_size()


def grinqh_vmm(w: Packed, a: Assignment, y: torch.Tensor | None = None,
               workspace: torch.Tensor | None = None, stream=None) -> torch.Tensor:
    """y [T, N] fp32 = x . W over the planes the assignment `a` (made from x) selects."""
    T, K = a.T, a.K
    dev = w.planes.device
    if y is None:
        y = torch.empty((T, w.N), dtype=torch.float32, device=dev)
    workspace, nbytes = _ws(T, K, w.N, workspace, dev)
    _check(_lib.grinqh_vmm(*_vmm_common(w, a), _dev(y, torch.float32, "y"), workspace.data_ptr(), nbytes,
                           _stream(stream)), "grinqh_vmm")
    return y


def grinqh_vmm_thresholds(x: torch.Tensor, theta, w: Packed, y: torch.Tensor | None = None,
                          workspace: torch.Tensor | None = None, stream=None) -> torch.Tensor:
    """y [T, N] = x . W with the threshold assignment made inside the VMM launch (no assignment kernel)."""
    T, K = x.shape
    if y is None:
        y = torch.empty((T, w.N), dtype=torch.float32, device=x.device)
    workspace, nbytes = _ws(T, K, w.N, workspace, x.device)
    th = (C.c_uint16 * 9)(*[int(v) for v in theta])
    _check(_lib.grinqh_vmm_thresholds(_dev(x, torch.float16, "x"), T, K, w.N, GROUP, th, w.planes.data_ptr(),
                                      w.scales.data_ptr(), w.zeros.data_ptr(), _dev(y, torch.float32, "y"),
                                      workspace.data_ptr(), nbytes, _stream(stream)), "grinqh_vmm_thresholds")
    return y


def grinqh_vmm_rank(x: torch.Tensor, counts, w: Packed, y: torch.Tensor | None = None,
                    workspace: torch.Tensor | None = None, stream=None) -> torch.Tensor:
    """y [T, N] = x . W with the rank assignment made inside the VMM launch (no assignment kernel)."""
    T, K = x.shape
    if y is None:
        y = torch.empty((T, w.N), dtype=torch.float32, device=x.device)
    workspace, nbytes = _ws(T, K, w.N, workspace, x.device)
    _check(_lib.grinqh_vmm_rank(_dev(x, torch.float16, "x"), T, K, w.N, GROUP, _counts(counts), w.planes.data_ptr(),
                                w.scales.data_ptr(), w.zeros.data_ptr(), _dev(y, torch.float32, "y"),
                                workspace.data_ptr(), nbytes, _stream(stream)), "grinqh_vmm_rank")
    return y


def grinqh_static_scratch_bytes() -> int:
    return int(_lib.grinqh_static_scratch_bytes())


def grinqh_vmm_rank_static(x: torch.Tensor, counts, w: Packed, y: torch.Tensor, stream=None) -> torch.Tensor:
    """grinqh_vmm_rank with the library's static device scratch: allocates nothing, so y is the caller's.

    Shapes whose workspace exceeds grinqh_static_scratch_bytes() raise; calls that overlap on the GPU race on the array.
    """
    T, K = x.shape
    _check(_lib.grinqh_vmm_rank_static(_dev(x, torch.float16, "x"), T, K, w.N, GROUP, _counts(counts),
                                       w.planes.data_ptr(), w.scales.data_ptr(), w.zeros.data_ptr(),
                                       _dev(y, torch.float32, "y"), _stream(stream)), "grinqh_vmm_rank_static")
    return y


def grinqh_prefill_gemm(X: torch.Tensor, w: Packed, Y: torch.Tensor | None = None, stream=None) -> torch.Tensor:
    """Y [M, N] fp16 = X [M, K] fp16 . W_hat (b_max = 8), the unpack fused into a tcgen05 GEMM (prefill path)."""
    M, K = X.shape
    if K != w.K:
        raise GrinqhError(f"X has K={K}, weight has K={w.K}")
    if Y is None:
        Y = torch.empty((M, w.N), dtype=torch.float16, device=X.device)
    _check(_lib.grinqh_prefill_gemm(_dev(X, torch.float16, "X"), M, K, w.N, GROUP, w.planes.data_ptr(),
                                    w.scales.data_ptr(), w.zeros.data_ptr(), _dev(Y, torch.float16, "Y"),
                                    _stream(stream)), "grinqh_prefill_gemm")
    return Y


class PackedSeg2:
    """Device-resident 2-bit-segment store: segs [bmax/2, K, N/16] int32 (bit patterns), scales/zeros [K/128, N] fp16."""

    def __init__(self, K: int, N: int, bmax: int, device="cuda"):
        self.K, self.N, self.bmax = K, N, bmax
        self.segs = torch.empty((bmax // 2, K, N // 16), dtype=torch.int32, device=device)
        self.scales = torch.empty((K // GROUP, N), dtype=torch.float16, device=device)
        self.zeros = torch.empty((K // GROUP, N), dtype=torch.float16, device=device)


def grinqh_pack_seg2(W: torch.Tensor, bmax: int, out: PackedSeg2 | None = None, stream=None) -> PackedSeg2:
    K, N = W.shape
    out = out or PackedSeg2(K, N, bmax, W.device)
    _check(_lib.grinqh_pack_seg2(_dev(W, torch.float16, "W"), K, N, GROUP, int(bmax), out.segs.data_ptr(),
                                 out.scales.data_ptr(), out.zeros.data_ptr(), _stream(stream)), "grinqh_pack_seg2")
    return out


def grinqh_vmm_rank_seg2(x: torch.Tensor, counts, w: PackedSeg2, y: torch.Tensor | None = None,
                         workspace: torch.Tensor | None = None, stream=None) -> torch.Tensor:
    """y [1, N] = x . W over the 2-bit-segment store, rank assignment inside the launch (widths 0, 2, .., bmax)."""
    T, K = x.shape
    if y is None:
        y = torch.empty((T, w.N), dtype=torch.float32, device=x.device)
    workspace, nbytes = _ws(T, K, w.N, workspace, x.device)
    _check(_lib.grinqh_vmm_rank_seg2(_dev(x, torch.float16, "x"), T, K, w.N, GROUP, w.bmax, _counts(counts),
                                     w.segs.data_ptr(), w.scales.data_ptr(), w.zeros.data_ptr(),
                                     _dev(y, torch.float32, "y"), workspace.data_ptr(), nbytes, _stream(stream)),
           "grinqh_vmm_rank_seg2")
    return y


def grinqh_vmm_main(w: Packed, a: Assignment, workspace: torch.Tensor, stream=None):
    _check(_lib.grinqh_vmm_main(*_vmm_common(w, a), workspace.data_ptr(),
                                workspace.numel() * workspace.element_size(), _stream(stream)), "grinqh_vmm_main")


def grinqh_vmm_reduce(T: int, K: int, N: int, y: torch.Tensor, workspace: torch.Tensor, stream=None):
    _check(_lib.grinqh_vmm_reduce(T, K, N, _dev(y, torch.float32, "y"), workspace.data_ptr(),
                                  workspace.numel() * workspace.element_size(), _stream(stream)),
           "grinqh_vmm_reduce")


def grinqh_decode_host(x_host: torch.Tensor, counts, w: Packed, x_dev: torch.Tensor, y_dev: torch.Tensor,
                       workspace: torch.Tensor, y_host: torch.Tensor, force_copies: bool = False, stream=None):
    """HOST x [T, K] fp16 -> HOST y [T, N] fp32 (rank assignment inside the VMM launch); weights stay on the device.
    Enqueue only."""
    T, K = x_host.shape
    if x_host.is_cuda or y_host.is_cuda:
        raise GrinqhError("grinqh_decode_host takes HOST x and y")
    _check(_lib.grinqh_decode_host(
        x_host.data_ptr(), T, K, w.N, GROUP, _counts(counts), w.planes.data_ptr(), w.scales.data_ptr(),
        w.zeros.data_ptr(), x_dev.data_ptr(), y_dev.data_ptr(), workspace.data_ptr(),
        workspace.numel() * workspace.element_size(), y_host.data_ptr(), 2 if force_copies else 0, _stream(stream)),
        "grinqh_decode_host")
