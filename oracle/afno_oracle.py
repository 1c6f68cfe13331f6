"""ctypes front end of the fp64 CPU oracle (oracle/afno_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports nothing from
paper_2208_05419_b200 and shares no code with the CUDA path.

All arrays are numpy float64, C-contiguous, layouts as in afno_oracle.h.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "afno_oracle.c")
_HDR = os.path.join(_HERE, "afno_oracle.h")
_LIB = os.path.join(_HERE, "libafno_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C99 + OpenMP).  Returns the .so path."""
    stale = (
        force
        or not os.path.exists(_LIB)
        or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    )
    if stale:
        cmd = ["gcc", "-std=c99", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


class _Desc(ctypes.Structure):
    _fields_ = [
        ("B", ctypes.c_int32), ("H", ctypes.c_int32), ("W", ctypes.c_int32), ("C", ctypes.c_int32),
        ("num_blocks", ctypes.c_int32), ("hidden_factor", ctypes.c_int32),
        ("lam", ctypes.c_double), ("kept_fraction", ctypes.c_double),
        ("no_residual", ctypes.c_int32), ("naive_dft", ctypes.c_int32),
    ]


class _Dump(ctypes.Structure):
    _fields_ = [("xhat", ctypes.c_void_p), ("p1", ctypes.c_void_p),
                ("p2", ctypes.c_void_p), ("z", ctypes.c_void_p)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        vp = ctypes.c_void_p
        L.afno_oracle_fwd.argtypes = [ctypes.POINTER(_Desc)] + [vp] * 6 + [ctypes.POINTER(_Dump)]
        L.afno_oracle_fwd.restype = ctypes.c_int
        L.afno_oracle_fwd_dense.argtypes = [ctypes.POINTER(_Desc)] + [vp] * 6
        L.afno_oracle_fwd_dense.restype = ctypes.c_int
        L.afno_oracle_bwd.argtypes = [ctypes.POINTER(_Desc)] + [vp] * 13 + [ctypes.POINTER(_Dump)]
        L.afno_oracle_bwd.restype = ctypes.c_int
        L.afno_oracle_rfft2.argtypes = [ctypes.c_int, ctypes.c_int, vp, vp, ctypes.c_int]
        L.afno_oracle_irfft2.argtypes = [ctypes.c_int, ctypes.c_int, vp, vp, ctypes.c_int]
        L.afno_oracle_dft1.argtypes = [ctypes.c_int, vp, vp, ctypes.c_int, ctypes.c_int]
        L.afno_oracle_kept.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                       ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_int)]
        L.afno_oracle_num_threads.restype = ctypes.c_int
        _lib = L
    return _lib


@dataclass
class Config:
    B: int
    H: int
    W: int
    C: int
    num_blocks: int
    hidden_factor: int = 1
    lam: float = 0.01
    kept_fraction: float = 1.0
    no_residual: bool = False
    naive_dft: bool = False

    @property
    def Wh(self):
        return self.W // 2 + 1

    @property
    def bs(self):
        return self.C // self.num_blocks

    @property
    def hid(self):
        return self.bs * self.hidden_factor

    def desc(self) -> _Desc:
        return _Desc(self.B, self.H, self.W, self.C, self.num_blocks, self.hidden_factor,
                     float(self.lam), float(self.kept_fraction), int(self.no_residual),
                     int(self.naive_dft))


def _f64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        assert a.shape == tuple(shape), (a.shape, shape)
    return a


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def num_threads() -> int:
    return int(lib().afno_oracle_num_threads())


def kept(H: int, W: int, f: float):
    kh, kw = ctypes.c_int(), ctypes.c_int()
    lib().afno_oracle_kept(H, W, float(f), ctypes.byref(kh), ctypes.byref(kw))
    return kh.value, kw.value


def rfft2(x: np.ndarray, naive: bool = False) -> np.ndarray:
    """x [H][W] real -> complex [H][Wh], ortho."""
    x = _f64(x)
    H, W = x.shape
    X = np.empty((H, W // 2 + 1, 2), dtype=np.float64)
    lib().afno_oracle_rfft2(H, W, _p(x), _p(X), int(naive))
    return X[..., 0] + 1j * X[..., 1]


def irfft2(Z: np.ndarray, W: int, naive: bool = False) -> np.ndarray:
    """Z complex [H][Wh] -> real [H][W], ortho, reading A4."""
    Z = np.ascontiguousarray(Z, dtype=np.complex128)
    H, Wh = Z.shape
    assert Wh == W // 2 + 1
    s = np.empty((H, W), dtype=np.float64)
    lib().afno_oracle_irfft2(H, W, _p(Z.view(np.float64)), _p(s), int(naive))
    return s


def dft1(a: np.ndarray, sign: int = -1, naive: bool = False) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.complex128)
    out = np.empty_like(a)
    lib().afno_oracle_dft1(a.shape[0], _p(a.view(np.float64)), _p(out.view(np.float64)), sign,
                           int(naive))
    return out


def _alloc_dump(cfg: Config, want: bool):
    if not want:
        return None, None
    M = (cfg.B, cfg.H, cfg.Wh)
    arrs = {
        "xhat": np.zeros(M + (cfg.C,), dtype=np.complex128),
        "p1": np.zeros(M + (cfg.num_blocks * cfg.hid,), dtype=np.complex128),
        "p2": np.zeros(M + (cfg.C,), dtype=np.complex128),
        "z": np.zeros(M + (cfg.C,), dtype=np.complex128),
    }
    d = _Dump(*[arrs[k].ctypes.data for k in ("xhat", "p1", "p2", "z")])
    return arrs, d


def _check_params(cfg: Config, w1, b1, w2, b2):
    nb, bs, hid = cfg.num_blocks, cfg.bs, cfg.hid
    return (_f64(w1, (nb, bs, hid, 2)), _f64(b1, (nb, hid, 2)),
            _f64(w2, (nb, hid, bs, 2)), _f64(b2, (nb, bs, 2)))


def forward(cfg: Config, x, w1, b1, w2, b2, dump: bool = False):
    """Returns y [B,H,W,C] (and a dict of intermediates when dump=True)."""
    x = _f64(x, (cfg.B, cfg.H, cfg.W, cfg.C))
    w1, b1, w2, b2 = _check_params(cfg, w1, b1, w2, b2)
    y = np.empty_like(x)
    arrs, d = _alloc_dump(cfg, dump)
    desc = cfg.desc()
    rc = lib().afno_oracle_fwd(ctypes.byref(desc), _p(x), _p(w1), _p(b1), _p(w2), _p(b2), _p(y),
                               ctypes.byref(d) if d is not None else None)
    if rc != 0:
        raise ValueError("afno_oracle_fwd: invalid descriptor or argument")
    return (y, arrs) if dump else y


def forward_dense(cfg: Config, x, w1d, b1, w2d, b2):
    x = _f64(x, (cfg.B, cfg.H, cfg.W, cfg.C))
    CH = cfg.num_blocks * cfg.hid
    w1d = _f64(w1d, (cfg.C, CH, 2))
    w2d = _f64(w2d, (CH, cfg.C, 2))
    b1 = _f64(b1, (cfg.num_blocks, cfg.hid, 2))
    b2 = _f64(b2, (cfg.num_blocks, cfg.bs, 2))
    y = np.empty_like(x)
    desc = cfg.desc()
    rc = lib().afno_oracle_fwd_dense(ctypes.byref(desc), _p(x), _p(w1d), _p(b1), _p(w2d), _p(b2),
                                     _p(y))
    if rc != 0:
        raise ValueError("afno_oracle_fwd_dense: invalid descriptor or argument")
    return y


def backward(cfg: Config, x, dy, w1, b1, w2, b2, mask1=None, mask2=None, dump: bool = False):
    """Returns dict(dx, dw1, db1, dw2, db2[, dump]).

    mask1 [B,H,Wh,nb*hid,2] / mask2 [B,H,Wh,C,2] uint8 override the oracle's own masks
    (mask-consistent comparison, S3 P-bwd)."""
    x = _f64(x, (cfg.B, cfg.H, cfg.W, cfg.C))
    dy = _f64(dy, x.shape)
    w1, b1, w2, b2 = _check_params(cfg, w1, b1, w2, b2)
    dx = np.empty_like(x)
    dw1, db1, dw2, db2 = (np.empty_like(a) for a in (w1, b1, w2, b2))
    if mask1 is not None:
        mask1 = np.ascontiguousarray(mask1, dtype=np.uint8)
        assert mask1.shape == (cfg.B, cfg.H, cfg.Wh, cfg.num_blocks * cfg.hid, 2)
    if mask2 is not None:
        mask2 = np.ascontiguousarray(mask2, dtype=np.uint8)
        assert mask2.shape == (cfg.B, cfg.H, cfg.Wh, cfg.C, 2)
    arrs, d = _alloc_dump(cfg, dump)
    desc = cfg.desc()
    rc = lib().afno_oracle_bwd(ctypes.byref(desc), _p(x), _p(dy), _p(w1), _p(b1), _p(w2), _p(b2),
                               _p(dx), _p(dw1), _p(db1), _p(dw2), _p(db2), _p(mask1), _p(mask2),
                               ctypes.byref(d) if d is not None else None)
    if rc != 0:
        raise ValueError("afno_oracle_bwd: invalid descriptor or argument")
    out = dict(dx=dx, dw1=dw1, db1=db1, dw2=dw2, db2=db2)
    if dump:
        out["dump"] = arrs
    return out
