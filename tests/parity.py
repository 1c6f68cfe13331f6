"""Helpers for the GPU-vs-oracle parity tests (test infrastructure).

The GPU side goes through the C ABI (paper_2208_05419_b200.binding); the oracle side
through oracle/afno_oracle.py.  The two never see each other's outputs as inputs, except
for the exported activation masks used for the mask-consistent backward comparison
(S3, P-bwd).
"""
from __future__ import annotations

import numpy as np

from paper_2208_05419_b200 import binding, inputs


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    den = np.linalg.norm(b.ravel())
    return float(np.linalg.norm((a - b).ravel()) / (den if den > 0 else 1.0))


def max_abs(a, b):
    return float(np.abs(np.asarray(a, dtype=np.float64) - np.asarray(b, dtype=np.float64)).max())


def _torch():
    import torch
    return torch


def to_device_act(a: np.ndarray, bf16: bool):
    torch = _torch()
    t = torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()
    return t.to(torch.bfloat16) if bf16 else t


def from_device_act(t):
    return t.float().cpu().numpy()


class GpuLayer:
    """Holds device buffers for one descriptor and calls the C ABI."""

    def __init__(self, desc: binding.Desc):
        torch = _torch()
        self.desc = desc
        self.bf16 = desc.dtype == binding.AFNO_BF16
        self.ws_fwd = torch.empty(max(16, binding.afno_spectral_workspace_bytes(desc, False)),
                                  dtype=torch.uint8, device="cuda")
        binding.afno_plan_warmup(desc)

    def params(self, w1, b1, w2, b2):
        torch = _torch()
        return [torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda() for a in (w1, b1, w2, b2)]

    def forward(self, x, w1, b1, w2, b2, flags=None):
        torch = _torch()
        d = self.desc if flags is None else binding.Desc(**{**self.desc.__dict__, "flags": flags})
        tx = to_device_act(x, self.bf16)
        ty = torch.empty_like(tx)
        p = self.params(w1, b1, w2, b2)
        binding.afno_spectral_fwd(d, tx, *p, ty, self.ws_fwd)
        torch.cuda.synchronize()
        return from_device_act(ty)

    def backward(self, x, dy, w1, b1, w2, b2, flags=None, export_masks=True):
        torch = _torch()
        fl = self.desc.flags if flags is None else flags
        if export_masks:
            fl |= binding.FLAG_EXPORT_MASKS
        d = binding.Desc(**{**self.desc.__dict__, "flags": fl})
        ws = torch.empty(binding.afno_spectral_workspace_bytes(d, True), dtype=torch.uint8, device="cuda")
        tx, tdy = to_device_act(x, self.bf16), to_device_act(dy, self.bf16)
        tdx = torch.empty_like(tx)
        p = self.params(w1, b1, w2, b2)
        g = [torch.zeros_like(t) for t in p]
        binding.afno_spectral_bwd(d, tx, tdy, *p, tdx, *g, ws)
        torch.cuda.synchronize()
        out = dict(dx=from_device_act(tdx), dw1=g[0].cpu().numpy(), db1=g[1].cpu().numpy(),
                   dw2=g[2].cpu().numpy(), db2=g[3].cpu().numpy())
        if export_masks:
            m1b, m2off, m2b = binding.afno_spectral_mask_bytes(d)
            host = ws[:m2off + m2b].cpu().numpy()
            out["mask1"] = host[:m1b].reshape(d.B, d.H, d.Wh, d.num_blocks * d.hid, 2).copy()
            out["mask2"] = host[m2off:m2off + m2b].reshape(d.B, d.H, d.Wh, d.C, 2).copy()
        return out


def desc_for(wl: inputs.Workload, B=None, flags=0, kept_fraction=None, lam=None, dtype=None):
    dt = wl.dtype if dtype is None else dtype
    return binding.Desc(B=wl.B if B is None else B, H=wl.H, W=wl.W, C=wl.C, num_blocks=wl.num_blocks,
                        hidden_factor=wl.hidden_factor, lam=wl.lam if lam is None else lam,
                        kept_fraction=wl.kept_fraction if kept_fraction is None else kept_fraction,
                        dtype=binding.AFNO_BF16 if dt == "bf16" else binding.AFNO_F32, flags=flags)


def oracle_cfg(oracle, d: binding.Desc, no_residual=False, naive=False):
    # the oracle receives the float32-rounded lambda / kept fraction the GPU received
    return oracle.Config(d.B, d.H, d.W, d.C, d.num_blocks, hidden_factor=d.hidden_factor,
                         lam=float(np.float32(d.lam)), kept_fraction=float(np.float32(d.kept_fraction)),
                         no_residual=no_residual, naive_dft=naive)


def preactivation_scales(cfg, dump, w1, b1, w2, b2):
    """Per-(mode, block) magnitude scale of the two pre-activations (S3, P-bwd (ii)).

    |P1[m,j,o] - b1| <= ||Xh[m,j,:]||_2 * ||W1[j,:,o]||_2 (Cauchy-Schwarz), so a kernel whose
    operands carry a relative error eps perturbs P1 by at most ~eps * that product.  A DFT is
    only NORMWISE accurate (||dXh|| <= eps ||x|| over the plane, not component by component),
    so the row norm gets the plane's rms row norm added as an absolute floor; the same holds
    for P2 with O1 and W2.  Returned arrays broadcast over the features of a block."""
    nb, bs, hid = cfg.num_blocks, cfg.bs, cfg.hid
    cw1 = w1[..., 0] + 1j * w1[..., 1]
    cw2 = w2[..., 0] + 1j * w2[..., 1]
    w1n = np.sqrt((np.abs(cw1) ** 2).sum(axis=1)).max(axis=1)          # [nb]
    w2n = np.sqrt((np.abs(cw2) ** 2).sum(axis=1)).max(axis=1)
    b1n = np.abs(b1[..., 0] + 1j * b1[..., 1]).max(axis=1)
    b2n = np.abs(b2[..., 0] + 1j * b2[..., 1]).max(axis=1)
    xh = dump["xhat"]
    xn = np.sqrt((np.abs(xh.reshape(xh.shape[:3] + (nb, bs))) ** 2).sum(-1))       # [B,H,Wh,nb]
    p1 = dump["p1"]
    o1 = np.maximum(p1.real, 0) + 1j * np.maximum(p1.imag, 0)
    on = np.sqrt((np.abs(o1.reshape(o1.shape[:3] + (nb, hid))) ** 2).sum(-1))
    xfloor = np.sqrt((xn ** 2).mean(axis=(1, 2), keepdims=True))                    # [B,1,1,nb]
    ofloor = np.sqrt((on ** 2).mean(axis=(1, 2), keepdims=True))
    s1 = np.repeat((xn + xfloor) * w1n + b1n, hid, axis=-1)                         # [B,H,Wh,nb*hid]
    s2 = np.repeat((on + ofloor) * w2n + b2n, bs, axis=-1)                          # [B,H,Wh,C]
    return s1, s2


def kept_modes(cfg):
    """Boolean [H, Wh]: the kept set of DESIGN.md S3 readings A7 / A8 (restated from the definition)."""
    f = float(np.float32(cfg.kept_fraction))
    hh, wh = cfg.H // 2 + 1, cfg.W // 2 + 1
    Kh = max(1, min(hh, int(np.floor(f * hh))))
    Kw = max(1, min(wh, int(np.floor(f * wh))))
    r = np.arange(cfg.H)
    kappa = np.where(r <= cfg.H // 2, r, cfg.H - r)
    return (kappa < Kh)[:, None] & (np.arange(wh) < Kw)[None, :]


def mask_flip_report(oracle_dump, gpu_mask1, gpu_mask2, lam, tau1, tau2, kept=None):
    """Fraction of flipped masks and whether every flip is justified: the oracle's fp64
    pre-activation lies within tau of the threshold (S3 P-bwd (ii)).  tau1 / tau2 are
    arrays broadcastable to the masks' shapes without the trailing (re, im) axis.  Only KEPT modes
    count (`kept`: boolean [H, Wh]): outside the kept set Z = 0 exactly (reading A9), no gradient
    passes, and the masks are not defined (a kernel may leave them unset)."""
    p1, p2 = oracle_dump["p1"], oracle_dump["p2"]
    z = oracle_dump["z"]
    o1 = np.stack([p1.real > 0, p1.imag > 0], -1)
    o2 = np.stack([z.real != 0, z.imag != 0], -1)
    f1 = o1 != gpu_mask1.astype(bool)
    f2 = o2 != gpu_mask2.astype(bool)
    if kept is not None:
        k = np.asarray(kept, dtype=bool)[None, :, :, None, None]
        f1 = f1 & k
        f2 = f2 & k
        norm = float(k.mean())
    else:
        norm = 1.0
    d1 = np.abs(np.stack([p1.real, p1.imag], -1)) / np.asarray(tau1)[..., None]
    d2 = np.abs(np.abs(np.stack([p2.real, p2.imag], -1)) - lam) / np.asarray(tau2)[..., None]
    worst1 = float(d1[f1].max()) if f1.any() else 0.0
    worst2 = float(d2[f2].max()) if f2.any() else 0.0
    return dict(flip1=float(f1.mean()) / norm, flip2=float(f2.mean()) / norm, worst1=worst1, worst2=worst2,
                justified=(worst1 <= 1.0 and worst2 <= 1.0))
