"""Thin Python binding of the C ABI in include/afno.h (argument marshalling only).

Every step of the layer runs in the kernels of libafno_b200.so; PyTorch is used here only
for device memory (`tensor.data_ptr()`) and streams.  There is no CPU fallback: if the
library has not been built the first call raises.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libafno_b200.so")

AFNO_OK, AFNO_ERR_INVALID_ARG, AFNO_ERR_UNSUPPORTED, AFNO_ERR_WORKSPACE, AFNO_ERR_CUDA = range(5)
AFNO_F32, AFNO_BF16 = 0, 1
FLAG_NO_RESIDUAL, FLAG_ACCUM_GRADS, FLAG_FORCE_FP32_MATH, FLAG_EXPORT_MASKS = 1, 2, 4, 8
FLAG_SAVE_CONTEXT, FLAG_USE_CONTEXT = 16, 32

# every symbol include/afno.h declares (tests check that the library exports all of them)
EXPORTS = [
    "afno_version", "afno_status_string", "afno_last_error", "afno_spectral_path",
    "afno_spectral_workspace_bytes", "afno_spectral_mask_bytes", "afno_plan_warmup",
    "afno_spectral_fwd", "afno_spectral_bwd", "afno_spectral_host_arena_bytes",
    "afno_spectral_fwd_host", "afno_spectral_bwd_host", "afno_spectral_step_host", "afno_last_launch_count",
    "afno_profile_start", "afno_profile_stop", "afno_plan_destroy_all", "afno_block_wgrad_static",
]
STATIC_SCRATCH_BYTES = 16 << 20   # AFNO_STATIC_SCRATCH_BYTES


class AfnoDesc(ctypes.Structure):
    _fields_ = [
        ("B", ctypes.c_int32), ("H", ctypes.c_int32), ("W", ctypes.c_int32), ("C", ctypes.c_int32),
        ("num_blocks", ctypes.c_int32), ("hidden_factor", ctypes.c_int32),
        ("lam", ctypes.c_float), ("kept_fraction", ctypes.c_float),
        ("dtype", ctypes.c_int32), ("flags", ctypes.c_uint32),
    ]


class AfnoError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"afno status {status}: {message}")
        self.status = status


_lib = None


def lib():
    """Loads libafno_b200.so (built by paper_2208_05419_b200.build); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(
                f"{LIB_PATH} not found: build it with `python -m paper_2208_05419_b200.build` "
                "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, sz, dp = ctypes.c_void_p, ctypes.c_size_t, ctypes.POINTER(AfnoDesc)
        L.afno_version.restype = ctypes.c_int
        L.afno_status_string.restype = ctypes.c_char_p
        L.afno_status_string.argtypes = [ctypes.c_int]
        L.afno_last_error.restype = ctypes.c_char_p
        L.afno_spectral_path.restype = ctypes.c_char_p
        L.afno_spectral_path.argtypes = [dp]
        L.afno_spectral_workspace_bytes.restype = sz
        L.afno_spectral_workspace_bytes.argtypes = [dp, ctypes.c_int]
        L.afno_spectral_mask_bytes.restype = ctypes.c_int
        L.afno_spectral_mask_bytes.argtypes = [dp] + [ctypes.POINTER(sz)] * 3
        L.afno_plan_warmup.restype = ctypes.c_int
        L.afno_plan_warmup.argtypes = [dp]
        L.afno_spectral_fwd.restype = ctypes.c_int
        L.afno_spectral_fwd.argtypes = [dp] + [vp] * 7 + [sz, vp]
        L.afno_spectral_bwd.restype = ctypes.c_int
        L.afno_spectral_bwd.argtypes = [dp] + [vp] * 12 + [sz, vp]
        L.afno_spectral_host_arena_bytes.restype = sz
        L.afno_spectral_host_arena_bytes.argtypes = [dp, ctypes.c_int]
        L.afno_spectral_fwd_host.restype = ctypes.c_int
        L.afno_spectral_fwd_host.argtypes = [dp] + [vp] * 7 + [sz, vp]
        L.afno_spectral_bwd_host.restype = ctypes.c_int
        L.afno_spectral_bwd_host.argtypes = [dp] + [vp] * 12 + [sz, vp]
        L.afno_spectral_step_host.restype = ctypes.c_int
        L.afno_spectral_step_host.argtypes = [dp] + [vp] * 13 + [sz, vp]
        L.afno_last_launch_count.restype = ctypes.c_int
        L.afno_plan_destroy_all.restype = ctypes.c_int
        L.afno_profile_start.restype = ctypes.c_int
        L.afno_profile_stop.restype = ctypes.c_int
        L.afno_profile_stop.argtypes = [ctypes.c_char_p, sz]
        L.afno_block_wgrad_static.restype = ctypes.c_int
        L.afno_block_wgrad_static.argtypes = [vp, ctypes.c_int32, vp, ctypes.c_int32, ctypes.c_int64, ctypes.c_int32,
                                              ctypes.c_int32, ctypes.c_int32, vp, vp, ctypes.c_uint32, vp]
        _lib = L
    return _lib


def _check(rc: int):
    if rc != AFNO_OK:
        raise AfnoError(rc, (lib().afno_last_error() or b"").decode())


@dataclass
class Desc:
    B: int
    H: int
    W: int
    C: int
    num_blocks: int
    hidden_factor: int = 1
    lam: float = 0.01
    kept_fraction: float = 1.0
    dtype: int = AFNO_BF16
    flags: int = 0

    def c(self) -> AfnoDesc:
        return AfnoDesc(self.B, self.H, self.W, self.C, self.num_blocks, self.hidden_factor,
                        self.lam, self.kept_fraction, self.dtype, self.flags)

    @property
    def Wh(self):
        return self.W // 2 + 1

    @property
    def bs(self):
        return self.C // self.num_blocks

    @property
    def hid(self):
        return self.bs * self.hidden_factor


def _ptr(t):
    """Device (or host) address of a torch tensor / numpy array / int."""
    if t is None:
        return None
    if isinstance(t, int):
        return ctypes.c_void_p(t)
    if hasattr(t, "data_ptr"):
        return ctypes.c_void_p(t.data_ptr())
    return ctypes.c_void_p(t.ctypes.data)


def _stream_handle(stream):
    if stream is None:
        import torch
        return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return ctypes.c_void_p(stream)
    return ctypes.c_void_p(stream.cuda_stream)


def afno_version() -> int:
    return lib().afno_version()


def afno_spectral_path(d: Desc):
    cd = d.c()
    p = lib().afno_spectral_path(ctypes.byref(cd))
    return p.decode() if p else None


def afno_spectral_workspace_bytes(d: Desc, for_backward: bool) -> int:
    cd = d.c()
    return int(lib().afno_spectral_workspace_bytes(ctypes.byref(cd), int(for_backward)))


def afno_spectral_host_arena_bytes(d: Desc, for_backward) -> int:
    cd = d.c()
    return int(lib().afno_spectral_host_arena_bytes(ctypes.byref(cd), int(for_backward)))


def afno_spectral_mask_bytes(d: Desc):
    cd = d.c()
    a, b, c = ctypes.c_size_t(), ctypes.c_size_t(), ctypes.c_size_t()
    _check(lib().afno_spectral_mask_bytes(ctypes.byref(cd), ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)))
    return a.value, b.value, c.value


def afno_plan_warmup(d: Desc):
    cd = d.c()
    _check(lib().afno_plan_warmup(ctypes.byref(cd)))


def afno_plan_destroy_all():
    _check(lib().afno_plan_destroy_all())


def afno_last_launch_count() -> int:
    return int(lib().afno_last_launch_count())


def afno_profile_start():
    _check(lib().afno_profile_start())


def afno_profile_stop() -> dict:
    """{kernel name: (launches, total_ms)} for the launches since afno_profile_start()."""
    buf = ctypes.create_string_buffer(1 << 16)
    _check(lib().afno_profile_stop(buf, len(buf)))
    out = {}
    for line in buf.value.decode().splitlines():
        name, n, ms = line.split()
        out[name] = (int(n), float(ms))
    return out


def _ws_bytes(ws):
    return ws.numel() * ws.element_size()


def afno_spectral_fwd(d: Desc, x, w1, b1, w2, b2, y, workspace, stream=None):
    cd = d.c()
    _check(lib().afno_spectral_fwd(ctypes.byref(cd), _ptr(x), _ptr(w1), _ptr(b1), _ptr(w2), _ptr(b2),
                                   _ptr(y), _ptr(workspace), _ws_bytes(workspace), _stream_handle(stream)))


def afno_spectral_bwd(d: Desc, x, dy, w1, b1, w2, b2, dx, dw1, db1, dw2, db2, workspace, stream=None):
    cd = d.c()
    _check(lib().afno_spectral_bwd(ctypes.byref(cd), _ptr(x), _ptr(dy), _ptr(w1), _ptr(b1), _ptr(w2),
                                   _ptr(b2), _ptr(dx), _ptr(dw1), _ptr(db1), _ptr(dw2), _ptr(db2),
                                   _ptr(workspace), _ws_bytes(workspace), _stream_handle(stream)))


def afno_spectral_fwd_host(d: Desc, x, w1, b1, w2, b2, y, arena, stream=None):
    """x, w*, b*, y: HOST tensors/arrays (pinned recommended); arena: device tensor."""
    cd = d.c()
    _check(lib().afno_spectral_fwd_host(ctypes.byref(cd), _ptr(x), _ptr(w1), _ptr(b1), _ptr(w2), _ptr(b2),
                                        _ptr(y), _ptr(arena), _ws_bytes(arena), _stream_handle(stream)))


def afno_spectral_bwd_host(d: Desc, x, dy, w1, b1, w2, b2, dx, dw1, db1, dw2, db2, arena, stream=None):
    """x may be None: x is then the one the preceding afno_spectral_fwd_host left in `arena`."""
    cd = d.c()
    _check(lib().afno_spectral_bwd_host(ctypes.byref(cd), _ptr(x), _ptr(dy), _ptr(w1), _ptr(b1), _ptr(w2),
                                        _ptr(b2), _ptr(dx), _ptr(dw1), _ptr(db1), _ptr(dw2), _ptr(db2),
                                        _ptr(arena), _ws_bytes(arena), _stream_handle(stream)))


def afno_spectral_step_host(d: Desc, x, dy, w1, b1, w2, b2, y, dx, dw1, db1, dw2, db2, arena, stream=None):
    """One training step from HOST tensors/arrays (pinned recommended); arena: device tensor of
    afno_spectral_host_arena_bytes(d, 2) bytes."""
    cd = d.c()
    _check(lib().afno_spectral_step_host(ctypes.byref(cd), _ptr(x), _ptr(dy), _ptr(w1), _ptr(b1), _ptr(w2), _ptr(b2),
                                         _ptr(y), _ptr(dx), _ptr(dw1), _ptr(db1), _ptr(dw2), _ptr(db2),
                                         _ptr(arena), _ws_bytes(arena), _stream_handle(stream)))


def afno_block_wgrad_static(a, g, M: int, num_blocks: int, K: int, N: int, dw, db, flags: int = 0, stream=None,
                            lda: int | None = None, ldg: int | None = None):
    """dw[j][i][o] = sum_m conj(a[m][j*K+i]) g[m][j*N+o], db[j][o] = sum_m g[m][j*N+o] for callers that may not allocate
    device memory: the kernels' scratch is the library's static device array (include/afno.h has the contract: size
    limit, first-call set-up, no overlapping calls).  a, g: device tensors of complex fp32 rows ([M][lda] / [M][ldg],
    strides in complex elements, default num_blocks*K / num_blocks*N); dw, db: fp32 device tensors."""
    _check(lib().afno_block_wgrad_static(_ptr(a), num_blocks * K if lda is None else lda, _ptr(g),
                                         num_blocks * N if ldg is None else ldg, M, num_blocks, K, N, _ptr(dw), _ptr(db),
                                         flags, _stream_handle(stream)))
