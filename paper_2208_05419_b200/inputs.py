"""Seeded synthetic inputs for the AFNO spectral layer (S4, input recipe).

This module serves BOTH the CUDA path's tests/bench and the oracle's tests.  It holds
none of the method's arithmetic (no transform, no MLP, no activation): only random
draws, the synthetic field recipe and the bf16 quantisation of generated inputs.

The fields stand in for ERA5-derived token activations (SIV-B): ERA5, the
HDF5 files and trained embeddings are not available and are not needed.

Seeds follow SURVEY.md S8(d): seed = 220805419 + 1000*config + stream,
stream: 0 x, 1 w1, 2 b1, 3 w2, 4 b2, 5 dY.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

BASE_SEED = 220805419
STREAM_X, STREAM_W1, STREAM_B1, STREAM_W2, STREAM_B2, STREAM_DY = range(6)


def seed_for(config: int, stream: int) -> int:
    return BASE_SEED + 1000 * config + stream


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def bf16_round(a: np.ndarray) -> np.ndarray:
    """Round float32 values to the nearest bfloat16 (ties to even); returns float32."""
    a = np.ascontiguousarray(a, dtype=np.float32)
    u = a.view(np.uint32).astype(np.uint64)
    bias = ((u >> 16) & 1) + 0x7FFF
    r = ((u + bias) >> 16) << 16
    return r.astype(np.uint32).view(np.float32).reshape(a.shape)


def bf16_bits(a: np.ndarray) -> np.ndarray:
    """float32 values that are already bf16-representable -> uint16 bit patterns."""
    a = np.ascontiguousarray(a, dtype=np.float32)
    return (a.view(np.uint32) >> 16).astype(np.uint16).reshape(a.shape)


def bf16_from_bits(u: np.ndarray) -> np.ndarray:
    u = np.ascontiguousarray(u, dtype=np.uint16)
    return (u.astype(np.uint32) << 16).view(np.float32).reshape(u.shape)


def gaussian(seed: int, shape, scale: float = 1.0) -> np.ndarray:
    return (scale * _rng(seed).standard_normal(size=shape)).astype(np.float32)


def weights(config: int, num_blocks: int, bs: int, hidden_factor: int = 1, scale: float = 0.02):
    """(w1 [nb,bs,hid,2], b1 [nb,hid,2], w2 [nb,hid,bs,2], b2 [nb,bs,2]) fp32,
    re and im each scale*N(0,1) (BASELINE.json configs)."""
    hid = bs * hidden_factor
    w1 = gaussian(seed_for(config, STREAM_W1), (num_blocks, bs, hid, 2), scale)
    b1 = gaussian(seed_for(config, STREAM_B1), (num_blocks, hid, 2), scale)
    w2 = gaussian(seed_for(config, STREAM_W2), (num_blocks, hid, bs, 2), scale)
    b2 = gaussian(seed_for(config, STREAM_B2), (num_blocks, bs, 2), scale)
    return w1, b1, w2, b2


def field(seed: int, B: int, H: int, W: int, C: int, n_terms: int = 6, noise: float = 0.1):
    """FourCastNet-shaped synthetic activations [B,H,W,C] float32.

    Per (b, channel) plane: n_terms random low-wavenumber sinusoids
    a*cos(2 pi (kh h/H + kw w/W) + phi) with integer kh ~ U{-4..4}, kw ~ U{0..8},
    (kh,kw) != (0,0), a ~ U(0.5,1.5)/(1+sqrt(kh^2+kw^2)), phi ~ U[0,2pi); plus
    noise*N(0,1) per token; minus the plane mean, divided by the plane's population std.
    """
    rng = _rng(seed)
    P = B * C
    kh = rng.integers(-4, 5, size=(P, n_terms))
    kw = rng.integers(0, 9, size=(P, n_terms))
    zero = (kh == 0) & (kw == 0)
    kw = np.where(zero, 1, kw)
    amp = rng.uniform(0.5, 1.5, size=(P, n_terms)) / (1.0 + np.sqrt(kh * kh + kw * kw))
    phi = rng.uniform(0.0, 2.0 * np.pi, size=(P, n_terms))
    h = np.arange(H, dtype=np.float64)
    w = np.arange(W, dtype=np.float64)
    # a cos(th_h + th_w + phi) = Re( a e^{i phi} e^{i th_h} e^{i th_w} ): an outer product
    eh = np.exp(2j * np.pi * kh[:, :, None] * h[None, None, :] / H)          # [P,T,H]
    ew = np.exp(2j * np.pi * kw[:, :, None] * w[None, None, :] / W)          # [P,T,W]
    ca = amp * np.exp(1j * phi)                                               # [P,T]
    out = np.empty((B, H, W, C), dtype=np.float32)
    chunk = 64
    for p0 in range(0, P, chunk):
        p1 = min(P, p0 + chunk)
        planes = np.einsum("pt,pth,ptw->phw", ca[p0:p1], eh[p0:p1], ew[p0:p1]).real
        planes = planes + noise * rng.standard_normal(size=planes.shape)
        planes -= planes.mean(axis=(1, 2), keepdims=True)
        planes /= planes.std(axis=(1, 2), keepdims=True)
        for p in range(p0, p1):
            out[p // C, :, :, p % C] = planes[p - p0]
    return out


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json config (index = position in BASELINE.json:configs)."""
    index: int
    name: str
    B: int
    H: int
    W: int
    C: int
    num_blocks: int
    hidden_factor: int
    lam: float
    kept_fraction: float
    dtype: str          # "f32" or "bf16": dtype of x, y, dy, dx
    backward: bool
    gaussian_x: bool    # configs[0] uses x ~ N(0,1); the others the field recipe


WORKLOADS = {
    "tiny": Workload(0, "tiny 8x16x16 fp32 fwd", 1, 8, 16, 16, 2, 1, 0.01, 1.0, "f32", False, True),
    "fcn_b1": Workload(1, "90x180x768 bf16 fwd B=1", 1, 90, 180, 768, 8, 1, 0.01, 1.0, "bf16", False, False),
    "fcn_b8": Workload(2, "90x180x768 bf16 fwd B=8", 8, 90, 180, 768, 8, 1, 0.01, 1.0, "bf16", False, False),
    "fcn_b8_half": Workload(2, "90x180x768 bf16 fwd B=8 kept 0.5", 8, 90, 180, 768, 8, 1, 0.01, 0.5, "bf16", False, False),
    "hires_b2": Workload(3, "180x360x768 bf16 fwd B=2", 2, 180, 360, 768, 8, 1, 0.01, 1.0, "bf16", False, False),
    # the paper's channel structure ("the 1024 channels are mixed using a block-diagonal MLP", 32 blocks
    # of 32) on the 90x180 token grid of the configs; SURVEY.md S8(f) item 1
    "paper_ch_b2": Workload(5, "90x180x1024 (32 blocks of 32) bf16 fwd+bwd B=2", 2, 90, 180, 1024, 32, 1, 0.01, 1.0, "bf16", True, False),
    # the paper's own layer shape (PAPER.md:112 p = 4 -> 180x360 tokens; :115, :138 1,024 channels in 32 blocks of 32)
    "paper_shape_b1": Workload(5, "180x360x1024 (32 blocks of 32) bf16 fwd B=1", 1, 180, 360, 1024, 32, 1, 0.01, 1.0, "bf16", False, False),
    "fcn_b4_bwd": Workload(4, "90x180x768 bf16 fwd+bwd B=4", 4, 90, 180, 768, 8, 1, 0.01, 1.0, "bf16", True, False),
    "sub_bwd_nb2": Workload(4, "16x32x64 fp32 fwd+bwd nb=2", 2, 16, 32, 64, 2, 1, 0.01, 1.0, "f32", True, False),
    "sub_bwd_nb8": Workload(4, "16x32x64 fp32 fwd+bwd nb=8", 2, 16, 32, 64, 8, 1, 0.01, 1.0, "f32", True, False),
}


def make_inputs(wl: Workload, B: int | None = None):
    """dict(x, dy, w1, b1, w2, b2) float32 arrays for a workload.  For bf16 workloads x and
    dy are already rounded to bf16-representable values (reading A16): the oracle is fed
    exactly these values, the GPU their bf16 bit patterns."""
    B = wl.B if B is None else B
    bs = wl.C // wl.num_blocks
    if wl.gaussian_x:
        x = gaussian(seed_for(wl.index, STREAM_X), (B, wl.H, wl.W, wl.C))
    else:
        x = field(seed_for(wl.index, STREAM_X), B, wl.H, wl.W, wl.C)
    dy = gaussian(seed_for(wl.index, STREAM_DY), (B, wl.H, wl.W, wl.C))
    if wl.dtype == "bf16":
        x, dy = bf16_round(x), bf16_round(dy)
    w1, b1, w2, b2 = weights(wl.index, wl.num_blocks, bs, wl.hidden_factor)
    return dict(x=x, dy=dy, w1=w1, b1=b1, w2=w2, b2=b2)
