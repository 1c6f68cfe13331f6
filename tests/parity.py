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


# Standard deviation of the relative error of one bf16 rounding (uniform within half an ulp, ulp = 2^-8 of
# the leading bit), of an fp32 path operand (a generous 16 ulp for the depth of the FFT), and the multiple of
# the 1-sigma error model a flipped mask may sit away from its threshold (S3, P-bwd (ii)).
U_BF16 = 2.0 ** -9 / np.sqrt(3.0)
U_F32 = 16.0 * 2.0 ** -24
TAU_K = 6.0
LEAK = 0.1


def preactivation_scales(cfg, dump, w1, b1, w2, b2, bf16=True):
    """1-sigma error model of the two pre-activations, per (mode, output feature) (S3, P-bwd (ii)).

    Every operand of the path is rounded once to bf16 (relative error of standard deviation u) and products
    are accumulated in fp32, so errors add in quadrature.  Per complex component:
      * spectrum: the two transform stages are GEMMs against rounded DFT matrices with a rounded
        intermediate, so the error of Xh[r,kw,c] has a part u |Xh[r,kw,c]| (its own rounding), a part
        ~ u * rms_r |Xh[:,kw,c]| (the H transform against a rounded matrix spreads column kw's energy over
        its rows: a DFT is normwise, not componentwise, accurate), a part ~ u * rms_kw |Xh[r,:,c]| (the same
        for the W transform: its error is a random combination of the field's rows, so after the H transform
        it sits in the rows r where the field has energy, at every kw), a plane-wide floor, and a leak term: the
        rounding errors of a DFT matrix are not random, a strong line leaks coherently into the bins harmonically
        related to it, so LEAK times the largest line of the column and of the row enters whole.  With the second
        rounding of Xh (as the bf16 operand of layer 1) folded in, the code below uses
            var_X = u^2 (2 |Xh|^2 + 2 colms[kw,c] + 2 rowms[r,c] + planems[c] + LEAK (colmax[kw,c] + rowmax[r,c]))
      * P1[o] = sum_i Xh[i] W1[i,o] + b1:  var_1[o] = sum_i |W1[i,o]|^2 var_X[i]
      * O1 = relu(P1), rounded once when stored and once as the operand of layer 2:
                                           var_O[i] = var_1[i] + 2 u^2 |O1[i]|^2
      * P2[o] = sum_i O1[i] W2[i,o] + b2:  var_2[o] = sum_i |W2[i,o]|^2 var_O[i]
    The constants are hand-set, not fitted: TAU_K = 6 sigma, LEAK = 0.1, and for the fp32 path u = 16 ulp (U_F32, the
    depth of the FFT); the worst flip observed on the bf16 path sits at 0.81 of the allowed distance.
    Returns sigma1 [B,H,Wh,nb*hid], sigma2 [B,H,Wh,C] (per real component: half the complex variance); a
    flipped mask is justified when the oracle's pre-activation lies within TAU_K sigma of its threshold."""
    nb, bs, hid = cfg.num_blocks, cfg.bs, cfg.hid
    u2 = (U_BF16 if bf16 else U_F32) ** 2
    a1 = (w1[..., 0] ** 2 + w1[..., 1] ** 2)                           # [nb, bs, hid]  |W1[j,i,o]|^2
    a2 = (w2[..., 0] ** 2 + w2[..., 1] ** 2)                           # [nb, hid, bs]
    xh = dump["xhat"]
    x2 = np.abs(xh) ** 2                                               # [B,H,Wh,C]
    colms = x2.mean(axis=1, keepdims=True)                             # [B,1,Wh,C]
    planems = x2.mean(axis=(1, 2), keepdims=True)                      # [B,1,1,C]  = mean x^2 of the plane (Parseval)
    rowms = x2.mean(axis=2, keepdims=True)                             # [B,H,1,C]
    # The rounding errors of a DFT matrix are not random: the leak of a strong spectral line into the bins
    # harmonically related to it (same column, rows a multiple of H/5 apart, ...) adds up coherently to
    # ~ u |line| instead of u |line| / sqrt(H): the largest line of the column and of the row enter whole.
    colmax = x2.max(axis=1, keepdims=True)
    rowmax = x2.max(axis=2, keepdims=True)
    var_x = u2 * (2.0 * x2 + 2.0 * colms + 2.0 * rowms + planems + LEAK * (colmax + rowmax))
    shp = x2.shape[:3]
    var_1 = np.einsum("mji,jio->mjo", var_x.reshape(-1, nb, bs), a1).reshape(shp + (nb * hid,))
    p1 = dump["p1"]
    o2 = np.maximum(p1.real, 0) ** 2 + np.maximum(p1.imag, 0) ** 2     # |O1|^2
    var_o = var_1 + 2.0 * u2 * o2
    var_2 = np.einsum("mji,jio->mjo", var_o.reshape(-1, nb, hid), a2).reshape(shp + (nb * bs,))
    return np.sqrt(0.5 * var_1), np.sqrt(0.5 * var_2)


def tile_rel_l2(a, b, block: int, slab: bool = False):
    """Relative L2 error per tile of an activation-shaped tensor [B,H,W,C]: one tile = (b, h, channel block)
    (what one CTA iteration of the W-direction kernels produces), or with slab=True one (b, block) slab
    (what the 91 mode tiles of one block and sample feed).  Returns the array of per-tile errors."""
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    B, H, W, C = b.shape
    e = ((a - b) ** 2).reshape(B, H, W, C // block, block).sum(axis=(2, 4))         # [B,H,nb]
    n = (b ** 2).reshape(B, H, W, C // block, block).sum(axis=(2, 4))
    if slab:
        e, n = e.sum(axis=1), n.sum(axis=1)
    return np.sqrt(e / np.where(n > 0, n, 1.0))


def block_rel_l2(a, b):
    """Relative L2 error per channel block of a parameter-shaped tensor [nb, ...]."""
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    ax = tuple(range(1, b.ndim))
    n = np.sqrt((b ** 2).sum(axis=ax))
    return np.sqrt(((a - b) ** 2).sum(axis=ax)) / np.where(n > 0, n, 1.0)


MAXABS_K = 16.0
PLANE_K = 0.125


def gate_activation(got, ref, tol, block, label=""):
    """The parity gate of an activation tensor: rel-L2 over the whole tensor, over every (b, h, block) tile
    and every (b, block) slab at `tol`, and an elementwise max-abs gate
        |got - ref| <= tol * (MAXABS_K * rms(ref) + |ref| + PLANE_K * max over the element's (b, channel) plane of |ref|)
    (a stated multiple of the rms error the tolerance allows; the tolerance relative to the element itself;
    and a term relative to the largest element of the plane: the branch s has one spike per plane at token
    (0, 0), the image of the bias, 100-300x the plane's rms, and a transform computed against rounded DFT
    matrices is normwise accurate, i.e. it leaks ~1 unit roundoff of that spike (measured 0.1 %) into the
    tokens harmonically related to it).
    Returns a dict of the measured figures; raises AssertionError naming the worst tile."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    assert np.isfinite(got).all(), (label, "non-finite output")
    whole = rel_l2(got, ref)
    tiles = tile_rel_l2(got, ref, block)
    slabs = tile_rel_l2(got, ref, block, slab=True)
    rms = float(np.sqrt((ref ** 2).mean()))
    ma = max_abs(got, ref)
    plane_max = np.abs(ref).max(axis=(1, 2), keepdims=True)
    elem = float((np.abs(got - ref) / (tol * (MAXABS_K * rms + np.abs(ref) + PLANE_K * plane_max) + 1e-300)).max())
    rep = dict(rel_l2=whole, tile_max=float(tiles.max()), slab_max=float(slabs.max()), max_abs=ma,
               max_abs_gate=elem)
    assert whole <= tol, (label, "rel_l2", whole)
    assert tiles.max() <= tol, (label, "tile (b,h,block)", np.unravel_index(tiles.argmax(), tiles.shape), float(tiles.max()))
    assert slabs.max() <= tol, (label, "slab (b,block)", np.unravel_index(slabs.argmax(), slabs.shape), float(slabs.max()))
    assert elem <= 1.0, (label, "max_abs", ma, "elementwise |err| / (tol (K rms + |ref| + max|plane| / 8))", elem, "rms(ref)", rms)
    return rep


def gate_param(got, ref, tol, label=""):
    """Parameter gradients: rel-L2 over the whole tensor and per channel block."""
    assert np.isfinite(np.asarray(got)).all(), (label, "non-finite gradient")
    whole = rel_l2(got, ref)
    blocks = block_rel_l2(got, ref)
    assert whole <= tol, (label, "rel_l2", whole)
    assert blocks.max() <= tol, (label, "block", int(blocks.argmax()), float(blocks.max()))
    return dict(rel_l2=whole, block_max=float(blocks.max()), max_abs=max_abs(got, ref))


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
