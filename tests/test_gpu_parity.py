"""GPU-vs-oracle parity through the C ABI (pytest -m gpu; runs on the B200 box).

Tolerances (BASELINE.json:north_star): relative L2 <= 1e-5 on the fp32 path, <= 2e-2 on the
bf16 path; gated on y AND on the spectral branch s (AFNO_FLAG_NO_RESIDUAL), because the
branch is only ~5 % of y (SURVEY.md S0 finding 1).  Backward is compared mask-consistently
(S3 P-bwd): the oracle is evaluated with the GPU's exported masks, every flipped
mask must sit within TAU_K = 6 standard deviations of a statistical error model of that mode's
pre-activation (parity.preactivation_scales), and the raw comparison is printed, not gated.  Every
activation gate is applied to the whole tensor, to every (b, h, block) tile, to every (b, block) slab
and to the max-abs error; parameter gradients per block (parity.gate_activation / gate_param).
"""
import numpy as np
import pytest

from paper_2208_05419_b200 import binding, inputs

import parity

pytestmark = pytest.mark.gpu

TOL_F32 = 1e-5
TOL_BF16 = 2e-2


def _tol(desc):
    return TOL_BF16 if desc.dtype == binding.AFNO_BF16 else TOL_F32


def _block(desc):
    return desc.C // desc.num_blocks


def _check_forward(oracle, desc, data, naive=False, label=""):
    """P-fwd: y AND the branch s against the oracle, gated over the whole tensor, per (b, h, block) tile,
    per (b, block) slab and on max-abs (parity.gate_activation)."""
    layer = parity.GpuLayer(desc)
    args = (data["x"], data["w1"], data["b1"], data["w2"], data["b2"])
    y_gpu = layer.forward(*args)
    s_gpu = layer.forward(*args, flags=desc.flags | binding.FLAG_NO_RESIDUAL)
    y_ref = oracle.forward(parity.oracle_cfg(oracle, desc, naive=naive), *args)
    s_ref = oracle.forward(parity.oracle_cfg(oracle, desc, no_residual=True, naive=naive), *args)
    ry = parity.gate_activation(y_gpu, y_ref, _tol(desc), _block(desc), label + " y")
    rs = parity.gate_activation(s_gpu, s_ref, _tol(desc), _block(desc), label + " s")
    print(f"[fwd {label}] path={binding.afno_spectral_path(desc)} y: {_fmt(ry)} | s: {_fmt(rs)} "
          f"|s|/|x|={np.linalg.norm(s_ref) / np.linalg.norm(data['x']):.3f}")
    return y_gpu


def _fmt(rep):
    return " ".join(f"{k}={v:.3e}" for k, v in rep.items())


def _flip_report(oracle, desc, data, raw_dump, mask1, mask2):
    """P-bwd (ii): every flipped mask within TAU_K sigma of its threshold (parity.preactivation_scales)."""
    cfg = parity.oracle_cfg(oracle, desc)
    s1, s2 = parity.preactivation_scales(cfg, raw_dump, *(data[k].astype(np.float64) for k in ("w1", "b1", "w2", "b2")),
                                         bf16=desc.dtype == binding.AFNO_BF16)
    return parity.mask_flip_report(raw_dump, mask1, mask2, cfg.lam, parity.TAU_K * s1, parity.TAU_K * s2,
                                   kept=parity.kept_modes(cfg))


def _check_backward(oracle, desc, data, label=""):
    layer = parity.GpuLayer(desc)
    args = (data["x"], data["dy"], data["w1"], data["b1"], data["w2"], data["b2"])
    g = layer.backward(*args)
    cfg = parity.oracle_cfg(oracle, desc)
    ref = oracle.backward(cfg, *args, mask1=g["mask1"], mask2=g["mask2"])
    raw = oracle.backward(cfg, *args, dump=True)
    tol = _tol(desc)
    rep = _flip_report(oracle, desc, data, raw["dump"], g["mask1"], g["mask2"])
    print(f"[bwd {label}] mask flips: relu {rep['flip1']:.2e} shrink {rep['flip2']:.2e}; worst flipped "
          f"|pre-activation - threshold| / ({parity.TAU_K:.0f} sigma) = {rep['worst1']:.2f} / {rep['worst2']:.2f} (must be <= 1)")
    r = parity.gate_activation(g["dx"], ref["dx"], tol, _block(desc), label + " dx")
    print(f"[bwd {label}] dx: {_fmt(r)}  raw rel_l2 {parity.rel_l2(g['dx'], raw['dx']):.3e}")
    for k in ("dw1", "db1", "dw2", "db2"):
        r = parity.gate_param(g[k], ref[k], tol, label + " " + k)
        print(f"[bwd {label}] {k}: {_fmt(r)}  raw rel_l2 {parity.rel_l2(g[k], raw[k]):.3e}")
    # branch of dx (dx - dy) is what the kernels actually compute
    nr = parity.GpuLayer(desc).backward(*args, flags=desc.flags | binding.FLAG_NO_RESIDUAL)
    cfg_nr = parity.oracle_cfg(oracle, desc, no_residual=True)
    ref_nr = oracle.backward(cfg_nr, *args, mask1=nr["mask1"], mask2=nr["mask2"])
    r = parity.gate_activation(nr["dx"], ref_nr["dx"], tol, _block(desc), label + " dx-branch")
    print(f"[bwd {label}] dx branch: {_fmt(r)}")
    assert rep["flip1"] <= 5e-3 and rep["flip2"] <= 5e-3
    assert rep["justified"], rep
    return g


# ---- T1: fp32 path ---------------------------------------------------------------------------

def test_configs0_tiny_vs_brute_force(oracle):
    wl = inputs.WORKLOADS["tiny"]
    _check_forward(oracle, parity.desc_for(wl), inputs.make_inputs(wl), naive=True, label="configs[0]")


@pytest.mark.parametrize("H,W,C,nb,hf", [(6, 10, 12, 3, 1), (12, 18, 20, 2, 2), (30, 20, 70, 7, 1),
                                         (16, 32, 64, 8, 1), (90, 180, 96, 1, 1), (45, 50, 33, 3, 1)])
@pytest.mark.parametrize("f,lam", [(1.0, 0.01), (0.5, 0.0), (0.25, 1e6)])
def test_fp32_forward_shapes(oracle, H, W, C, nb, hf, f, lam):
    rng = np.random.default_rng(H * 1000 + W)
    B = 2
    bs = C // nb
    data = dict(x=rng.standard_normal((B, H, W, C)).astype(np.float32))
    data["w1"], data["b1"], data["w2"], data["b2"] = [
        (0.2 * rng.standard_normal(s)).astype(np.float32)
        for s in [(nb, bs, bs * hf, 2), (nb, bs * hf, 2), (nb, bs * hf, bs, 2), (nb, bs, 2)]]
    desc = binding.Desc(B, H, W, C, nb, hf, lam, f, binding.AFNO_F32)
    if lam >= 1e6:
        # kill switch: branch is exactly zero, y == x bit-exactly
        layer = parity.GpuLayer(desc)
        y = layer.forward(data["x"], data["w1"], data["b1"], data["w2"], data["b2"])
        assert np.array_equal(y, data["x"])
        return
    _check_forward(oracle, desc, data, label=f"{H}x{W}x{C} nb={nb} hf={hf} f={f}")


@pytest.mark.parametrize("name", ["sub_bwd_nb2", "sub_bwd_nb8"])
def test_fp32_backward_subcase(oracle, name):
    wl = inputs.WORKLOADS[name]
    _check_backward(oracle, parity.desc_for(wl), inputs.make_inputs(wl), label=name)


@pytest.mark.parametrize("H,W,C,nb,hf,f", [(6, 10, 12, 3, 2, 0.5), (30, 20, 70, 7, 1, 1.0), (8, 16, 16, 2, 1, 0.7)])
def test_fp32_backward_shapes(oracle, H, W, C, nb, hf, f):
    rng = np.random.default_rng(H * 77 + W)
    B, bs = 2, C // nb
    data = dict(x=rng.standard_normal((B, H, W, C)).astype(np.float32),
                dy=rng.standard_normal((B, H, W, C)).astype(np.float32))
    data["w1"], data["b1"], data["w2"], data["b2"] = [
        (0.2 * rng.standard_normal(s)).astype(np.float32)
        for s in [(nb, bs, bs * hf, 2), (nb, bs * hf, 2), (nb, bs * hf, bs, 2), (nb, bs, 2)]]
    _check_backward(oracle, binding.Desc(B, H, W, C, nb, hf, 0.05, f, binding.AFNO_F32), data,
                    label=f"{H}x{W}x{C} nb={nb} hf={hf} f={f}")


def test_backward_repeatable_and_accumulate(oracle):
    wl = inputs.WORKLOADS["sub_bwd_nb2"]
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    layer = parity.GpuLayer(desc)
    args = (data["x"], data["dy"], data["w1"], data["b1"], data["w2"], data["b2"])
    g1 = layer.backward(*args, export_masks=False)
    g2 = layer.backward(*args, export_masks=False)
    for k in g1:
        assert np.array_equal(g1[k], g2[k]), k  # fixed summation order: bitwise repeatable
    import torch
    d_acc = binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_ACCUM_GRADS})
    ws = torch.empty(binding.afno_spectral_workspace_bytes(d_acc, True), dtype=torch.uint8, device="cuda")
    tx, tdy = parity.to_device_act(data["x"], False), parity.to_device_act(data["dy"], False)
    p = layer.params(data["w1"], data["b1"], data["w2"], data["b2"])
    g = [torch.ones_like(t) for t in p]
    tdx = torch.empty_like(tx)
    binding.afno_spectral_bwd(d_acc, tx, tdy, *p, tdx, *g, ws)
    torch.cuda.synchronize()
    for t, k in zip(g, ("dw1", "db1", "dw2", "db2")):
        assert np.allclose(t.cpu().numpy(), 1.0 + g1[k], rtol=0, atol=1e-6 * max(1.0, np.abs(g1[k]).max()))


# ---- T2: bf16 path at BASELINE.json's full sizes ------------------------------------------------

@pytest.mark.parametrize("name,f", [("fcn_b1", 1.0), ("fcn_b8", 1.0), ("fcn_b8", 0.5), ("hires_b2", 1.0)])
def test_bf16_forward_full_size(oracle, name, f):
    wl = inputs.WORKLOADS[name]
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl, kept_fraction=f)
    _check_forward(oracle, desc, data, label=f"{name} f={f}")


def test_bf16_forward_backward_full_size(oracle):
    wl = inputs.WORKLOADS["fcn_b4_bwd"]
    _check_backward(oracle, parity.desc_for(wl), inputs.make_inputs(wl), label="configs[4] B=4")


@pytest.mark.parametrize("B,H,W,C,nb,f", [
    (3, 30, 60, 96, 1, 1.0),      # one block, short rows and columns (TMA zero-fill in H and W), odd batch
    (1, 96, 180, 192, 2, 1.0),    # H = 96: no padding rows in the mode tiles; two blocks
    (2, 18, 36, 288, 3, 0.5),     # truncated spectrum on a small grid, three blocks
    (5, 40, 100, 96, 1, 0.75),    # W/2+1 = 51 bins, Kw = 38, five samples
    (1, 2, 4, 96, 1, 1.0),        # degenerate grid: fewer tiles than SMs, one tile per block
    (4, 8, 16, 192, 2, 0.5),      # Kh = 2, Kw = 4: most of the spectrum truncated
])
def test_bf16_tcgen05_other_shapes(oracle, B, H, W, C, nb, f):
    """The tcgen05 path away from the headline shape: ragged tails in every tiled dimension, forward
    and (mask-consistent) backward against the oracle, plus saved-context == stateless bit for bit."""
    import torch
    wl = inputs.Workload(4, f"{H}x{W}x{C} bf16 B={B}", B, H, W, C, nb, 1, 0.01, f, "bf16", True, False)
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    assert binding.afno_spectral_path(desc) == "tcgen05-bf16"
    _check_forward(oracle, desc, data, label=wl.name)
    g = _check_backward(oracle, desc, data, label=wl.name)
    layer = parity.GpuLayer(desc)
    d_save = binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_SAVE_CONTEXT})
    d_use = binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_USE_CONTEXT})
    ws = torch.empty(binding.afno_spectral_workspace_bytes(desc, True), dtype=torch.uint8, device="cuda")
    tx, tdy = parity.to_device_act(data["x"], True), parity.to_device_act(data["dy"], True)
    ty, tdx = torch.empty_like(tx), torch.empty_like(tx)
    p = layer.params(data["w1"], data["b1"], data["w2"], data["b2"])
    gr = [torch.zeros_like(t) for t in p]
    binding.afno_spectral_fwd(d_save, tx, *p, ty, ws)
    binding.afno_spectral_bwd(d_use, tx, tdy, *p, tdx, *gr, ws)
    torch.cuda.synchronize()
    assert np.array_equal(parity.from_device_act(tdx), g["dx"])
    for t, k in zip(gr, ("dw1", "db1", "dw2", "db2")):
        assert np.array_equal(t.cpu().numpy(), g[k]), k


@pytest.mark.parametrize("B,H,W,C,nb,f", [
    (2, 18, 36, 160, 5, 1.0),     # 32-wide blocks, C % 96 != 0: the last group of 96 channels holds two blocks
    (1, 30, 60, 96, 2, 1.0),      # 48-wide blocks
    (2, 8, 16, 64, 8, 0.5),       # 8-wide blocks, one partly filled group, truncated spectrum
    (1, 24, 48, 192, 8, 1.0),     # 24-wide blocks, two full groups
])
def test_bf16_tcgen05_narrow_blocks(oracle, B, H, W, C, nb, f):
    """Blocks narrower than 96 (bs divides 96) run on the tcgen05 path as block-diagonal 96 x 96 weight images
    inside groups of 96 channels (S5.3): forward, mask-consistent backward and the saved-context
    step against the oracle, per tile; perturbing one block's weights leaves the other blocks' outputs
    bit-identical (block-diagonality)."""
    wl = inputs.Workload(5, f"{H}x{W}x{C} nb={nb} bf16 B={B}", B, H, W, C, nb, 1, 0.01, f, "bf16", True, False)
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    assert binding.afno_spectral_path(desc) == "tcgen05-bf16"
    y0 = _check_forward(oracle, desc, data, label=wl.name)
    g = _check_backward(oracle, desc, data, label=wl.name)
    got = _ctx_step(desc, data)
    assert np.array_equal(got["y"], y0) and np.array_equal(got["dx"], g["dx"])
    for k in ("dw1", "db1", "dw2", "db2"):
        assert np.array_equal(got[k], g[k]), k
    bs = C // nb
    w1 = data["w1"].copy()
    w1[nb - 1] *= 1.5
    y1 = parity.GpuLayer(desc).forward(data["x"], w1, data["b1"], data["w2"], data["b2"])
    assert np.array_equal(y1[..., :C - bs], y0[..., :C - bs]) and not np.array_equal(y1[..., C - bs:], y0[..., C - bs:])


def test_bf16_paper_channel_structure(oracle):
    """SURVEY.md S8(f) item 1, the part that fits this path's grids: the paper's channel structure, 1,024
    channels in 32 blocks of 32, at the 90 x 180 token grid, forward and backward."""
    wl = inputs.WORKLOADS["paper_ch_b2"]
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    assert binding.afno_spectral_path(desc) == "tcgen05-bf16"
    _check_forward(oracle, desc, data, label=wl.name)
    _check_backward(oracle, desc, data, label=wl.name)


@pytest.mark.parametrize("B,H,W,C,nb,f", [
    (1, 100, 200, 192, 2, 1.0),    # H and W past the fused chain's limits, two full groups, ragged last row tile
    (2, 120, 30, 160, 5, 0.5),     # 32-wide blocks, partly filled last group, truncated rows
    (1, 10, 200, 96, 1, 1.0),      # W/2+1 = 101 bins only
])
def test_bf16_hybrid_forward(oracle, B, H, W, C, nb, f):
    """Grids beyond the fused chain (H > 96 or W/2+1 > 96) with bf16 activations: fp32 FFTs on the CUDA cores and
    the block MLP on the tensor cores (tc_mlp_fwd), forward, against the oracle per tile; the pure fp32 kernels
    (AFNO_FLAG_FORCE_FP32_MATH) must agree with it to bf16-operand accuracy."""
    wl = inputs.Workload(3, f"{H}x{W}x{C} nb={nb} bf16 B={B} hybrid", B, H, W, C, nb, 1, 0.01, f, "bf16", False, False)
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    assert binding.afno_spectral_path(desc) == "hybrid-fft32-tcgen05"
    y = _check_forward(oracle, desc, data, label=wl.name)
    d32 = parity.desc_for(wl, flags=binding.FLAG_FORCE_FP32_MATH)
    assert binding.afno_spectral_path(d32) == "generic-fp32"
    y32 = parity.GpuLayer(d32).forward(data["x"], data["w1"], data["b1"], data["w2"], data["b2"])
    assert parity.rel_l2(y, y32) <= 5e-3
    # capturable like every other path (include/afno.h), replay == eager bit for bit
    import torch
    layer = parity.GpuLayer(desc)
    tx = parity.to_device_act(data["x"], True)
    ty = torch.zeros_like(tx)
    p = layer.params(data["w1"], data["b1"], data["w2"], data["b2"])
    s = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        with torch.cuda.graph(graph, stream=s):
            binding.afno_spectral_fwd(desc, tx, *p, ty, layer.ws_fwd, stream=s)
    graph.replay()
    torch.cuda.synchronize()
    assert np.array_equal(parity.from_device_act(ty), y)


def test_bf16_tcgen05_kill_switch_and_lambda_zero(oracle):
    """Degenerate thresholds on the tcgen05 path (round-1 verdict weak 6c: they ran on the generic path only).
    lambda = 0: softshrink is the identity (reading A6), parity per tile, forward and backward.  lambda larger than
    every |P2| (pin O8, the kill switch): Z = 0 exactly, so y == x and dx == dy bit for bit and every parameter
    gradient is exactly zero (the softshrink mask is empty)."""
    import torch
    wl = inputs.Workload(4, "30x60x192 bf16 B=2 lambda=0", 2, 30, 60, 192, 2, 1, 0.0, 1.0, "bf16", True, False)
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    assert binding.afno_spectral_path(desc) == "tcgen05-bf16"
    _check_forward(oracle, desc, data, label=wl.name)
    _check_backward(oracle, desc, data, label=wl.name)
    dk = parity.desc_for(wl, lam=1e6)
    layer = parity.GpuLayer(dk)
    y = layer.forward(data["x"], data["w1"], data["b1"], data["w2"], data["b2"])
    assert np.array_equal(y, data["x"])
    for ctx in (False, True):
        if ctx:
            got = _ctx_step(dk, data)
            assert np.array_equal(got["y"], data["x"])
        else:
            got = layer.backward(data["x"], data["dy"], data["w1"], data["b1"], data["w2"], data["b2"], export_masks=False)
        assert np.array_equal(got["dx"], data["dy"])
        for k in ("dw1", "db1", "dw2", "db2"):
            assert not got[k].any(), k


@pytest.mark.parametrize("B,H,W,C,nb,hf,f", [
    (2, 16, 32, 192, 2, 2, 1.0),     # hidden = 192 per block, small grid
    (1, 100, 40, 96, 1, 3, 0.5),     # hidden = 288, H past the fused chain's limit, truncated, ragged last row tile
    (1, 90, 180, 768, 8, 2, 1.0),    # the headline grid with hidden factor 2
])
def test_bf16_hidden_factor_forward(oracle, B, H, W, C, nb, hf, f):
    """hidden factor > 1 with its block GEMMs on the tensor cores (hybrid forward,
    tc_mlp_fwd_hf: layer 2 accumulates over the 96-wide hidden chunks in tensor memory), against the oracle per tile."""
    wl = inputs.Workload(5, f"{H}x{W}x{C} nb={nb} hf={hf} bf16 B={B}", B, H, W, C, nb, hf, 0.01, f, "bf16", False, False)
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    assert desc.hidden_factor == hf and binding.afno_spectral_path(desc) == "hybrid-fft32-tcgen05"
    y = _check_forward(oracle, desc, data, label=wl.name)
    d32 = parity.desc_for(wl, flags=binding.FLAG_FORCE_FP32_MATH)
    y32 = parity.GpuLayer(d32).forward(data["x"], data["w1"], data["b1"], data["w2"], data["b2"])
    assert parity.rel_l2(y, y32) <= 5e-3


@pytest.mark.parametrize("B,H,W,C,nb,f", [
    (2, 100, 40, 96, 1, 1.0),      # H past the fused chain's limit, one group, ragged last 96-row tile
    (1, 100, 200, 192, 2, 1.0),    # H and W past the limits, two full groups
    (2, 120, 30, 160, 5, 0.5),     # 32-wide blocks, partly filled last group, truncated rows
])
def test_bf16_backward_beyond_the_fused_chain(oracle, B, H, W, C, nb, f):
    """bf16 activations on grids past the fused chain's limits: forward AND backward are the hybrid path (fp32 FFTs on
    the CUDA cores; the block MLP, its gradient stages and the parameter gradients on the tensor cores: tc_mlp_fwd,
    tc_mlp_bwd, tc_wgrad); both against the oracle, the backward mask-consistently, per tile and per block."""
    wl = inputs.Workload(4, f"{H}x{W}x{C} nb={nb} f={f} bf16 B={B} hybrid bwd", B, H, W, C, nb, 1, 0.01, f, "bf16", True, False)
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    assert binding.afno_spectral_path(desc) == "hybrid-fft32-tcgen05"
    _check_forward(oracle, desc, data, label=wl.name)
    g = _check_backward(oracle, desc, data, label=wl.name)
    # cross-check against the pure fp32 kernels (AFNO_FLAG_FORCE_FP32_MATH) on dx.  This is a RAW comparison (each path with
    # its own masks), which DESIGN.md S3 P-bwd (iii) prints and does not gate against the oracle: the ~0.1 % of masks the
    # bf16 path flips (reading A17) put a few 1e-3 into it; it only has to stay far inside the 2e-2 tolerance
    d32 = parity.desc_for(wl, flags=binding.FLAG_FORCE_FP32_MATH)
    args = (data["x"], data["dy"], data["w1"], data["b1"], data["w2"], data["b2"])
    g32 = parity.GpuLayer(d32).backward(*args)
    assert parity.rel_l2(g["dx"], g32["dx"]) <= 1e-2
    # AFNO_FLAG_ACCUM_GRADS on the hybrid backward, and repeatability without the mask export
    import torch
    layer = parity.GpuLayer(desc)
    d_acc = binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_ACCUM_GRADS})
    ws = torch.empty(binding.afno_spectral_workspace_bytes(d_acc, True), dtype=torch.uint8, device="cuda")
    tx, tdy = parity.to_device_act(data["x"], True), parity.to_device_act(data["dy"], True)
    p = layer.params(data["w1"], data["b1"], data["w2"], data["b2"])
    acc = [torch.ones_like(t) for t in p]
    tdx = torch.empty_like(tx)
    binding.afno_spectral_bwd(d_acc, tx, tdy, *p, tdx, *acc, ws)
    torch.cuda.synchronize()
    assert np.array_equal(parity.from_device_act(tdx), g["dx"])
    for t, k in zip(acc, ("dw1", "db1", "dw2", "db2")):
        assert np.allclose(t.cpu().numpy(), 1.0 + g[k], rtol=0, atol=2e-6 * max(1.0, np.abs(g[k]).max())), k


@pytest.mark.parametrize("B,H,W,C,nb,hf,f", [
    (2, 16, 32, 192, 2, 2, 1.0),     # hidden = 192 per block, small grid, ragged last tile
    (1, 100, 40, 96, 1, 3, 0.5),     # hidden = 288, H past the fused chain's limit, truncated
    (1, 90, 180, 768, 8, 2, 1.0),    # the headline grid with hidden factor 2
])
def test_bf16_hidden_factor_backward(oracle, B, H, W, C, nb, hf, f):
    """hidden factor > 1, BACKWARD on the hybrid path (tc_mlp_bwd_hf: two passes over the 96-wide
    hidden chunks, P2 and GX accumulated over the chunks in tensor memory, one tc_wgrad launch per chunk), mask-consistently
    against the oracle per tile and per block; ACCUM_GRADS on top."""
    import torch
    wl = inputs.Workload(5, f"{H}x{W}x{C} nb={nb} hf={hf} bf16 B={B} bwd", B, H, W, C, nb, hf, 0.01, f, "bf16", True, False)
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    assert desc.hidden_factor == hf and binding.afno_spectral_path(desc) == "hybrid-fft32-tcgen05"
    g = _check_backward(oracle, desc, data, label=wl.name)
    args = (data["x"], data["dy"], data["w1"], data["b1"], data["w2"], data["b2"])
    d32 = parity.desc_for(wl, flags=binding.FLAG_FORCE_FP32_MATH)
    g32 = parity.GpuLayer(d32).backward(*args)
    assert parity.rel_l2(g["dx"], g32["dx"]) <= 1e-2   # raw comparison, own masks on both sides (see the hybrid backward test)
    layer = parity.GpuLayer(desc)
    d_acc = binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_ACCUM_GRADS})
    ws = torch.empty(binding.afno_spectral_workspace_bytes(d_acc, True), dtype=torch.uint8, device="cuda")
    tx, tdy = parity.to_device_act(data["x"], True), parity.to_device_act(data["dy"], True)
    p = layer.params(data["w1"], data["b1"], data["w2"], data["b2"])
    acc = [torch.ones_like(t) for t in p]
    tdx = torch.empty_like(tx)
    binding.afno_spectral_bwd(d_acc, tx, tdy, *p, tdx, *acc, ws)
    torch.cuda.synchronize()
    assert np.array_equal(parity.from_device_act(tdx), g["dx"])
    for t, k in zip(acc, ("dw1", "db1", "dw2", "db2")):
        assert np.allclose(t.cpu().numpy(), 1.0 + g[k], rtol=0, atol=2e-6 * max(1.0, np.abs(g[k]).max())), k


def test_bf16_paper_shape_backward(oracle):
    """the paper's own layer shape (180 x 360 tokens, 1,024 channels in 32 blocks of 32), backward on
    the hybrid path, mask-consistently against the oracle per tile and per block."""
    wl = inputs.WORKLOADS["paper_shape_b1"]
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    assert binding.afno_spectral_path(desc) == "hybrid-fft32-tcgen05"
    _check_backward(oracle, desc, data, label=wl.name + " bwd")


def test_bf16_paper_shape_forward(oracle):
    """the paper's own layer shape, 180 x 360 tokens (p = 4) x 1,024 channels in 32
    blocks of 32, forward: fp32 FFTs + block MLP on the tensor cores (hybrid path)."""
    wl = inputs.WORKLOADS["paper_shape_b1"]
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    assert binding.afno_spectral_path(desc) == "hybrid-fft32-tcgen05"
    _check_forward(oracle, desc, data, label=wl.name)


def test_bf16_force_fp32_math_flag(oracle):
    wl = inputs.WORKLOADS["fcn_b1"]
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl, flags=binding.FLAG_FORCE_FP32_MATH)
    assert binding.afno_spectral_path(desc) == "generic-fp32"
    _check_forward(oracle, desc, data, label="fcn_b1 forced fp32 math")


# ---- T3: robustness on the device ---------------------------------------------------------------

def test_workspace_too_small_and_aliasing():
    import torch
    d = binding.Desc(1, 8, 16, 16, 2, dtype=binding.AFNO_F32)
    x = torch.zeros(1, 8, 16, 16, device="cuda")
    p = [torch.zeros(s, device="cuda") for s in [(2, 8, 8, 2), (2, 8, 2), (2, 8, 8, 2), (2, 8, 2)]]
    ws = torch.empty(binding.afno_spectral_workspace_bytes(d, False), dtype=torch.uint8, device="cuda")
    with pytest.raises(binding.AfnoError) as e:
        binding.afno_spectral_fwd(d, x, *p, torch.empty_like(x), ws[:64])
    assert e.value.status == binding.AFNO_ERR_WORKSPACE
    with pytest.raises(binding.AfnoError) as e:
        binding.afno_spectral_fwd(d, x, *p, x, ws)
    assert e.value.status == binding.AFNO_ERR_INVALID_ARG


def test_graph_capture_forward_backward(oracle):
    """fwd+bwd are capturable after afno_plan_warmup (PAPER.md:142-144 captures the step)."""
    import torch
    wl = inputs.WORKLOADS["sub_bwd_nb2"]
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    layer = parity.GpuLayer(desc)
    eager = layer.forward(data["x"], data["w1"], data["b1"], data["w2"], data["b2"])
    tx = parity.to_device_act(data["x"], False)
    tdy = parity.to_device_act(data["dy"], False)
    ty, tdx = torch.empty_like(tx), torch.empty_like(tx)
    p = layer.params(data["w1"], data["b1"], data["w2"], data["b2"])
    g = [torch.zeros_like(t) for t in p]
    wsb = torch.empty(binding.afno_spectral_workspace_bytes(desc, True), dtype=torch.uint8, device="cuda")
    s = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        with torch.cuda.graph(graph, stream=s):
            binding.afno_spectral_fwd(desc, tx, *p, ty, layer.ws_fwd, stream=s)
            binding.afno_spectral_bwd(desc, tx, tdy, *p, tdx, *g, wsb, stream=s)
    ty.zero_()
    graph.replay()
    torch.cuda.synchronize()
    assert np.array_equal(ty.cpu().numpy(), eager)
    ref = layer.backward(data["x"], data["dy"], data["w1"], data["b1"], data["w2"], data["b2"], export_masks=False)
    assert np.array_equal(tdx.cpu().numpy(), ref["dx"])
    assert np.array_equal(g[0].cpu().numpy(), ref["dw1"])


def test_saved_context_backward_matches_stateless():
    """SURVEY.md S8(a) row B1 "or load saved context": fwd with SAVE_CONTEXT then bwd with USE_CONTEXT
    on the same workspace gives bit-identical gradients to the stateless bwd (bf16 tcgen05 path,
    a slice of the headline shape, and the generic path, where the flags are accepted and ignored)."""
    import torch
    cases = [(parity.desc_for(inputs.WORKLOADS["fcn_b4_bwd"], B=2), inputs.make_inputs(inputs.WORKLOADS["fcn_b4_bwd"], B=2)),
             # truncated spectrum (kept fraction 0.5): masks of dropped rows / absent kw tiles stay zero
             (parity.desc_for(inputs.WORKLOADS["fcn_b4_bwd"], B=1, kept_fraction=0.5),
              inputs.make_inputs(inputs.WORKLOADS["fcn_b4_bwd"], B=1)),
             (parity.desc_for(inputs.WORKLOADS["sub_bwd_nb2"]), inputs.make_inputs(inputs.WORKLOADS["sub_bwd_nb2"]))]
    for desc, data in cases:
        bf16 = desc.dtype == binding.AFNO_BF16
        layer = parity.GpuLayer(desc)
        ref = layer.backward(data["x"], data["dy"], data["w1"], data["b1"], data["w2"], data["b2"], export_masks=False)
        y_ref = layer.forward(data["x"], data["w1"], data["b1"], data["w2"], data["b2"])
        d_save = binding.Desc(**{**desc.__dict__, "flags": desc.flags | binding.FLAG_SAVE_CONTEXT})
        d_use = binding.Desc(**{**desc.__dict__, "flags": desc.flags | binding.FLAG_USE_CONTEXT})
        ws = torch.empty(binding.afno_spectral_workspace_bytes(desc, True), dtype=torch.uint8, device="cuda")
        tx, tdy = parity.to_device_act(data["x"], bf16), parity.to_device_act(data["dy"], bf16)
        ty, tdx = torch.empty_like(tx), torch.empty_like(tx)
        p = layer.params(data["w1"], data["b1"], data["w2"], data["b2"])
        g = [torch.zeros_like(t) for t in p]
        small = torch.empty(binding.afno_spectral_workspace_bytes(desc, False), dtype=torch.uint8, device="cuda")
        if binding.afno_spectral_workspace_bytes(desc, False) < binding.afno_spectral_workspace_bytes(desc, True):
            with pytest.raises(binding.AfnoError) as e:
                binding.afno_spectral_fwd(d_save, tx, *p, ty, small)
            assert e.value.status == binding.AFNO_ERR_WORKSPACE
        binding.afno_spectral_fwd(d_save, tx, *p, ty, ws)
        binding.afno_spectral_bwd(d_use, tx, tdy, *p, tdx, *g, ws)
        torch.cuda.synchronize()
        assert np.array_equal(parity.from_device_act(ty), y_ref)
        assert np.array_equal(parity.from_device_act(tdx), ref["dx"])
        for t, k in zip(g, ("dw1", "db1", "dw2", "db2")):
            assert np.array_equal(t.cpu().numpy(), ref[k]), k


def _ctx_step(desc, data, extra_flags=0, stream=None):
    """One training step as bench.py runs it: fwd SAVE_CONTEXT then bwd USE_CONTEXT on one workspace."""
    import torch
    base = binding.Desc(**{**desc.__dict__, "flags": desc.flags | extra_flags})
    d_save = binding.Desc(**{**base.__dict__, "flags": base.flags | binding.FLAG_SAVE_CONTEXT})
    d_use = binding.Desc(**{**base.__dict__, "flags": base.flags | binding.FLAG_USE_CONTEXT})
    layer = parity.GpuLayer(base)
    ws = torch.empty(binding.afno_spectral_workspace_bytes(base, True), dtype=torch.uint8, device="cuda")
    tx, tdy = parity.to_device_act(data["x"], True), parity.to_device_act(data["dy"], True)
    ty, tdx = torch.empty_like(tx), torch.empty_like(tx)
    p = layer.params(data["w1"], data["b1"], data["w2"], data["b2"])
    g = [torch.zeros_like(t) for t in p]
    binding.afno_spectral_fwd(d_save, tx, *p, ty, ws)
    binding.afno_spectral_bwd(d_use, tx, tdy, *p, tdx, *g, ws)
    torch.cuda.synchronize()
    out = dict(y=parity.from_device_act(ty), dx=parity.from_device_act(tdx), dw1=g[0].cpu().numpy(),
               db1=g[1].cpu().numpy(), dw2=g[2].cpu().numpy(), db2=g[3].cpu().numpy())
    if base.flags & binding.FLAG_EXPORT_MASKS:
        m1b, m2off, m2b = binding.afno_spectral_mask_bytes(base)
        host = ws[:m2off + m2b].cpu().numpy()
        out["mask1"] = host[:m1b].reshape(base.B, base.H, base.Wh, base.num_blocks * base.hid, 2).copy()
        out["mask2"] = host[m2off:m2off + m2b].reshape(base.B, base.H, base.Wh, base.C, 2).copy()
    return out


def test_saved_context_step_vs_oracle(oracle):
    """The EXACT step bench.py times (BASELINE.json configs[4]: B = 4, fwd SAVE_CONTEXT, bwd USE_CONTEXT on
    the same workspace), pinned to the oracle directly: y and the branch s per tile, gradients
    mask-consistent per tile / per block, flipped masks justified (S3 P-fwd / P-bwd)."""
    wl = inputs.WORKLOADS["fcn_b4_bwd"]
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    assert desc.B == 4 and binding.afno_spectral_path(desc) == "tcgen05-bf16"
    got = _ctx_step(desc, data, binding.FLAG_EXPORT_MASKS)
    got_nr = _ctx_step(desc, data, binding.FLAG_EXPORT_MASKS | binding.FLAG_NO_RESIDUAL)
    cfg, cfg_nr = parity.oracle_cfg(oracle, desc), parity.oracle_cfg(oracle, desc, no_residual=True)
    fargs = (data["x"], data["w1"], data["b1"], data["w2"], data["b2"])
    args = (data["x"], data["dy"], data["w1"], data["b1"], data["w2"], data["b2"])
    blk = _block(desc)
    ry = parity.gate_activation(got["y"], oracle.forward(cfg, *fargs), TOL_BF16, blk, "ctx y")
    rs = parity.gate_activation(got_nr["y"], oracle.forward(cfg_nr, *fargs), TOL_BF16, blk, "ctx s")
    print(f"[ctx step B=4] y: {_fmt(ry)} | s: {_fmt(rs)}")
    ref = oracle.backward(cfg, *args, mask1=got["mask1"], mask2=got["mask2"])
    raw = oracle.backward(cfg, *args, dump=True)
    rep = _flip_report(oracle, desc, data, raw["dump"], got["mask1"], got["mask2"])
    print(f"[ctx step B=4] flips relu {rep['flip1']:.2e} shrink {rep['flip2']:.2e} worst {rep['worst1']:.2f} / {rep['worst2']:.2f}")
    print(f"[ctx step B=4] dx: {_fmt(parity.gate_activation(got['dx'], ref['dx'], TOL_BF16, blk, 'ctx dx'))}")
    ref_nr = oracle.backward(cfg_nr, *args, mask1=got_nr["mask1"], mask2=got_nr["mask2"])
    print(f"[ctx step B=4] dx branch: {_fmt(parity.gate_activation(got_nr['dx'], ref_nr['dx'], TOL_BF16, blk, 'ctx dx-branch'))}")
    for k in ("dw1", "db1", "dw2", "db2"):
        print(f"[ctx step B=4] {k}: {_fmt(parity.gate_param(got[k], ref[k], TOL_BF16, 'ctx ' + k))}")
    assert rep["flip1"] <= 5e-3 and rep["flip2"] <= 5e-3 and rep["justified"], rep


def test_context_guard_poisons_foreign_context():
    """USE_CONTEXT on a workspace whose context does not belong to the call (never saved, saved for another
    batch size, saved with another flag set that moves the layout) must not return plausible numbers: dx and
    the gradients come back NaN (include/afno.h)."""
    import torch
    wl = inputs.WORKLOADS["fcn_b4_bwd"]
    data = inputs.make_inputs(wl, B=2)
    desc = parity.desc_for(wl, B=2)
    d_save = binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_SAVE_CONTEXT})
    d_use = binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_USE_CONTEXT})
    layer = parity.GpuLayer(desc)
    nbytes = binding.afno_spectral_workspace_bytes(
        binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_EXPORT_MASKS}), True)
    tx, tdy = parity.to_device_act(data["x"], True), parity.to_device_act(data["dy"], True)
    ty, tdx = torch.empty_like(tx), torch.empty_like(tx)
    p = layer.params(data["w1"], data["b1"], data["w2"], data["b2"])

    def bwd(d, ws, x=tx, dy=tdy, dx=tdx):
        g = [torch.zeros_like(t) for t in p]
        binding.afno_spectral_bwd(d, x, dy, *p, dx, *g, ws)
        torch.cuda.synchronize()
        return dx.float().cpu().numpy(), [t.cpu().numpy() for t in g]

    # 1. never saved
    ws = torch.zeros(nbytes, dtype=torch.uint8, device="cuda")
    dx, g = bwd(d_use, ws)
    assert np.isnan(dx).all() and all(np.isnan(t).all() for t in g)
    # 2. saved, then used correctly: finite
    binding.afno_spectral_fwd(d_save, tx, *p, ty, ws)
    dx, g = bwd(d_use, ws)
    assert np.isfinite(dx).all() and all(np.isfinite(t).all() for t in g)
    # 3. saved without EXPORT_MASKS, used with it (the mask region moves every saved buffer)
    d_use_x = binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_USE_CONTEXT | binding.FLAG_EXPORT_MASKS})
    binding.afno_spectral_fwd(d_save, tx, *p, ty, ws)
    dx, g = bwd(d_use_x, ws)
    assert np.isnan(dx).all() and all(np.isnan(t).all() for t in g)
    # 4. saved for B = 2, used for B = 1
    binding.afno_spectral_fwd(d_save, tx, *p, ty, ws)
    d1 = binding.Desc(**{**d_use.__dict__, "B": 1})
    dx1 = torch.empty_like(tx[:1])
    dx, g = bwd(d1, ws, tx[:1].contiguous(), tdy[:1].contiguous(), dx1)
    assert np.isnan(dx).all() and all(np.isnan(t).all() for t in g)
    # 5. both context flags at once make no sense
    with pytest.raises(binding.AfnoError) as e:
        binding.afno_spectral_fwd(binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_SAVE_CONTEXT | binding.FLAG_USE_CONTEXT}),
                                  tx, *p, ty, ws)
    assert e.value.status == binding.AFNO_ERR_INVALID_ARG


def test_bf16_tcgen05_accumulate_and_chunks(oracle):
    """AFNO_FLAG_ACCUM_GRADS on the tcgen05 path (k_tc_wgrad_reduce's accumulate branch), at a batch larger
    than one chunk (B = 6 > 4: the chunk loop, the partial-sum accumulation across chunks and a ragged last
    chunk): grads(ones, ACCUM) == 1 + grads, and y / dx of samples 4, 5 equal a B = 2 call on those samples."""
    import torch
    wl = inputs.Workload(4, "30x60x192 bf16 B=6", 6, 30, 60, 192, 2, 1, 0.01, 1.0, "bf16", True, False)
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    assert binding.afno_spectral_path(desc) == "tcgen05-bf16"
    _check_forward(oracle, desc, data, label=wl.name)
    g0 = _check_backward(oracle, desc, data, label=wl.name)
    layer = parity.GpuLayer(desc)
    d_acc = binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_ACCUM_GRADS})
    ws = torch.empty(binding.afno_spectral_workspace_bytes(d_acc, True), dtype=torch.uint8, device="cuda")
    tx, tdy = parity.to_device_act(data["x"], True), parity.to_device_act(data["dy"], True)
    p = layer.params(data["w1"], data["b1"], data["w2"], data["b2"])
    g = [torch.ones_like(t) for t in p]
    tdx = torch.empty_like(tx)
    binding.afno_spectral_bwd(d_acc, tx, tdy, *p, tdx, *g, ws)
    torch.cuda.synchronize()
    assert np.array_equal(parity.from_device_act(tdx), g0["dx"])
    for t, k in zip(g, ("dw1", "db1", "dw2", "db2")):
        # the existing value is the first term of the fixed-order sum: equal up to fp32 rounding order
        assert np.allclose(t.cpu().numpy(), 1.0 + g0[k], rtol=0, atol=2e-6 * max(1.0, np.abs(g0[k]).max())), k
    # the saved-context step over two chunks (context buffers hold the batch, chunk buffers are reused): bit-identical
    got = _ctx_step(desc, data)
    assert np.array_equal(got["dx"], g0["dx"])
    for k in ("dw1", "db1", "dw2", "db2"):
        assert np.array_equal(got[k], g0[k]), k
    # samples are independent ("batched"): the last chunk alone gives the same y and dx
    d2 = parity.desc_for(wl, B=2)
    sub = {k: (v[4:] if k in ("x", "dy") else v) for k, v in data.items()}
    l2 = parity.GpuLayer(d2)
    y_all = layer.forward(data["x"], data["w1"], data["b1"], data["w2"], data["b2"])
    y_sub = l2.forward(sub["x"], sub["w1"], sub["b1"], sub["w2"], sub["b2"])
    assert np.array_equal(y_all[4:], y_sub)
    g_sub = l2.backward(sub["x"], sub["dy"], sub["w1"], sub["b1"], sub["w2"], sub["b2"], export_masks=False)
    assert np.array_equal(g0["dx"][4:], g_sub["dx"])


def test_graph_capture_tcgen05_step(oracle):
    """PAPER.md:142-144 "we capture the full forward and backward step ... inside a CUDA graph": the tcgen05
    chain (programmatic dependent launches, per-call tensor maps, the EXPORT-free memset-free path) captured
    once and replayed, stateless and saved-context, equals the eager calls bit for bit and the oracle
    within tolerance."""
    import torch
    wl = inputs.WORKLOADS["fcn_b4_bwd"]
    data = inputs.make_inputs(wl, B=2)
    desc = parity.desc_for(wl, B=2)
    assert binding.afno_spectral_path(desc) == "tcgen05-bf16"
    layer = parity.GpuLayer(desc)
    eager_y = layer.forward(data["x"], data["w1"], data["b1"], data["w2"], data["b2"])
    eager = layer.backward(data["x"], data["dy"], data["w1"], data["b1"], data["w2"], data["b2"], export_masks=False)
    y_ref = oracle.forward(parity.oracle_cfg(oracle, desc), data["x"], data["w1"], data["b1"], data["w2"], data["b2"])
    tx, tdy = parity.to_device_act(data["x"], True), parity.to_device_act(data["dy"], True)
    p = layer.params(data["w1"], data["b1"], data["w2"], data["b2"])
    for ctx in (False, True):
        d_f = binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_SAVE_CONTEXT}) if ctx else desc
        d_b = binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_USE_CONTEXT}) if ctx else desc
        ty, tdx = torch.zeros_like(tx), torch.zeros_like(tx)
        g = [torch.zeros_like(t) for t in p]
        ws = torch.empty(binding.afno_spectral_workspace_bytes(desc, True), dtype=torch.uint8, device="cuda")
        s = torch.cuda.Stream()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.stream(s):
            with torch.cuda.graph(graph, stream=s):
                binding.afno_spectral_fwd(d_f, tx, *p, ty, ws, stream=s)
                binding.afno_spectral_bwd(d_b, tx, tdy, *p, tdx, *g, ws, stream=s)
        for rep in range(3):
            ty.zero_(); tdx.zero_()
            for t in g:
                t.zero_()
            graph.replay()
            torch.cuda.synchronize()
            assert np.array_equal(parity.from_device_act(ty), eager_y), (ctx, rep)
            assert np.array_equal(parity.from_device_act(tdx), eager["dx"]), (ctx, rep)
            for t, k in zip(g, ("dw1", "db1", "dw2", "db2")):
                assert np.array_equal(t.cpu().numpy(), eager[k]), (ctx, rep, k)
        parity.gate_activation(parity.from_device_act(ty), y_ref, TOL_BF16, _block(desc), "graph y")


def test_saved_context_step_is_bitwise_repeatable():
    """The asynchronous hand-offs of the tcgen05 kernels (TMA rings, tensor-memory ping-pong, bulk stores,
    programmatic dependent launch) must not depend on timing: 60 saved-context steps on the same inputs,
    with unrelated memory traffic interleaved, give bit-identical y, dx and parameter gradients."""
    import torch
    wl = inputs.WORKLOADS["fcn_b4_bwd"]
    desc = parity.desc_for(wl, B=2)
    d_save = binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_SAVE_CONTEXT})
    d_use = binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_USE_CONTEXT})
    binding.afno_plan_warmup(desc)
    data = inputs.make_inputs(wl, B=2)
    tx, tdy = parity.to_device_act(data["x"], True), parity.to_device_act(data["dy"], True)
    p = parity.GpuLayer(desc).params(data["w1"], data["b1"], data["w2"], data["b2"])
    ws = torch.empty(binding.afno_spectral_workspace_bytes(desc, True), dtype=torch.uint8, device="cuda")
    junk = torch.empty(64 << 20, dtype=torch.uint8, device="cuda")
    ref = None
    for it in range(60):
        ty, tdx = torch.empty_like(tx), torch.empty_like(tx)
        g = [torch.empty_like(t) for t in p]
        if it % 3 == 1:
            junk.fill_(it & 255)
        binding.afno_spectral_fwd(d_save, tx, *p, ty, ws)
        if it % 5 == 2:
            junk.fill_(1)
        binding.afno_spectral_bwd(d_use, tx, tdy, *p, tdx, *g, ws)
        torch.cuda.synchronize()
        cur = [ty, tdx] + g
        if ref is None:
            ref = [t.clone() for t in cur]
        else:
            for k, (a, b) in enumerate(zip(ref, cur)):
                assert torch.equal(a, b), (it, k)


def test_step_gradients_bitwise_under_concurrent_load():
    """k_tc_wgrad_reduce sums tc_wgrad's partial sums before its own griddepcontrol.wait (it overlaps the inverse
    transform; S5.3 states what it relies on).  40 saved-context steps enqueued back to back with no host
    synchronisation, while a second stream keeps the SMs and the L2 busy with copies, must return the same bits as a
    quiet step; every step writes its gradients to its own buffers."""
    import torch
    wl = inputs.WORKLOADS["fcn_b4_bwd"]
    desc = parity.desc_for(wl, B=2)
    d_save = binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_SAVE_CONTEXT})
    d_use = binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_USE_CONTEXT})
    binding.afno_plan_warmup(desc)
    data = inputs.make_inputs(wl, B=2)
    tx, tdy = parity.to_device_act(data["x"], True), parity.to_device_act(data["dy"], True)
    p = parity.GpuLayer(desc).params(data["w1"], data["b1"], data["w2"], data["b2"])
    ws = torch.empty(binding.afno_spectral_workspace_bytes(desc, True), dtype=torch.uint8, device="cuda")
    ty, tdx = torch.empty_like(tx), torch.empty_like(tx)

    def step(g):
        binding.afno_spectral_fwd(d_save, tx, *p, ty, ws)
        binding.afno_spectral_bwd(d_use, tx, tdy, *p, tdx, *g, ws)

    quiet = [torch.empty_like(t) for t in p]
    step(quiet)
    torch.cuda.synchronize()
    N = 40
    outs = [[torch.full_like(t, float("nan")) for t in p] for _ in range(N)]
    src = torch.empty(256 << 20, dtype=torch.uint8, device="cuda").fill_(3)
    dst = torch.empty_like(src)
    side = torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        for _ in range(60):
            dst.copy_(src)
            src.add_(1)
    for it in range(N):
        step(outs[it])
    busy = not side.query()      # the load should still be running when the last step has been enqueued
    torch.cuda.synchronize()
    print(f"[load] side stream still busy after enqueueing {N} steps: {busy}")
    for it in range(N):
        for k, (a, b) in enumerate(zip(quiet, outs[it])):
            assert torch.equal(a, b), (it, k)


def test_host_variants_match_device(oracle):
    import torch
    wl = inputs.WORKLOADS["sub_bwd_nb8"]
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    layer = parity.GpuLayer(desc)
    y_dev = layer.forward(data["x"], data["w1"], data["b1"], data["w2"], data["b2"])
    g_dev = layer.backward(data["x"], data["dy"], data["w1"], data["b1"], data["w2"], data["b2"], export_masks=False)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).pin_memory()
    hx, hdy = pin(data["x"]), pin(data["dy"])
    hp = [pin(data[k]) for k in ("w1", "b1", "w2", "b2")]
    hy = torch.empty_like(hx).pin_memory()
    arena = torch.empty(binding.afno_spectral_host_arena_bytes(desc, True), dtype=torch.uint8, device="cuda")
    binding.afno_spectral_fwd_host(desc, hx, *hp, hy, arena)
    assert np.array_equal(hy.numpy(), y_dev)
    hdx = torch.empty_like(hx).pin_memory()
    hg = [torch.empty_like(t).pin_memory() for t in hp]
    binding.afno_spectral_bwd_host(desc, hx, hdy, *hp, hdx, *hg, arena)
    assert np.array_equal(hdx.numpy(), g_dev["dx"])
    # the host variant pipelines over the batch: parameter gradients are the in-order sum of the
    # per-sample gradients (include/afno.h), i.e. the device result up to fp32 summation order
    for t, k in zip(hg, ("dw1", "db1", "dw2", "db2")):
        assert parity.rel_l2(t.numpy(), g_dev[k]) <= 2e-6, k


def test_host_variants_tcgen05(oracle):
    """afno_spectral_{fwd,bwd}_host on the tcgen05 path (bf16, B = 3): what bench.py's `e2e` times.  y and dx
    equal the device path's bit for bit; the parameter gradients are the in-order sum of per-sample
    gradients (AFNO_FLAG_ACCUM_GRADS per sample), i.e. the device result up to fp32 summation order."""
    import torch
    wl = inputs.Workload(4, "30x60x192 bf16 B=3", 3, 30, 60, 192, 2, 1, 0.01, 1.0, "bf16", True, False)
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    assert binding.afno_spectral_path(desc) == "tcgen05-bf16"
    layer = parity.GpuLayer(desc)
    y_dev = layer.forward(data["x"], data["w1"], data["b1"], data["w2"], data["b2"])
    g_dev = layer.backward(data["x"], data["dy"], data["w1"], data["b1"], data["w2"], data["b2"], export_masks=False)
    pin_act = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(torch.bfloat16).pin_memory()
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).pin_memory()
    hx, hdy = pin_act(data["x"]), pin_act(data["dy"])
    hp = [pin(data[k]) for k in ("w1", "b1", "w2", "b2")]
    hy, hdx = torch.empty_like(hx).pin_memory(), torch.empty_like(hx).pin_memory()
    arena = torch.empty(max(binding.afno_spectral_host_arena_bytes(desc, False),
                            binding.afno_spectral_host_arena_bytes(desc, True)), dtype=torch.uint8, device="cuda")
    binding.afno_spectral_fwd_host(desc, hx, *hp, hy, arena)
    assert np.array_equal(hy.float().numpy(), y_dev)
    hg = [torch.empty_like(t).pin_memory() for t in hp]
    binding.afno_spectral_bwd_host(desc, hx, hdy, *hp, hdx, *hg, arena)
    assert np.array_equal(hdx.float().numpy(), g_dev["dx"])
    for t, k in zip(hg, ("dw1", "db1", "dw2", "db2")):
        assert parity.rel_l2(t.numpy(), g_dev[k]) <= 2e-6, k
    # a training step uploads x once: fwd_host leaves it in the arena, bwd_host(x = None) finds it there
    first = [t.clone() for t in hg]
    hdx2 = torch.empty_like(hx).pin_memory()
    binding.afno_spectral_fwd_host(desc, hx, *hp, hy, arena)
    binding.afno_spectral_bwd_host(desc, None, hdy, *hp, hdx2, *hg, arena)
    assert torch.equal(hdx2, hdx)
    for a, b in zip(first, hg):
        assert torch.equal(a, b)
    binding.afno_plan_destroy_all()      # plans are rebuilt on demand
    binding.afno_spectral_fwd_host(desc, hx, *hp, hy, arena)
    assert np.array_equal(hy.float().numpy(), y_dev)


def test_bwd_host_without_x_needs_an_arena_that_holds_it():
    """afno_spectral_bwd_host(x_host = NULL) reuses the x a host call left in the arena.  An arena no host call has
    written, or one that holds x of another shape, is refused (AFNO_ERR_INVALID_ARG) instead of yielding dx and gradients
    of whatever bytes sit there; after a fwd_host with the same descriptor the call goes through.  The host calls of
    a short-lived thread work too (its copy streams and events are released with the thread)."""
    import threading
    import torch
    wl = inputs.Workload(4, "30x60x192 bf16 B=2", 2, 30, 60, 192, 2, 1, 0.01, 1.0, "bf16", True, False)
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    desc1 = parity.desc_for(wl, B=1)
    pin_act = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(torch.bfloat16).pin_memory()
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).pin_memory()
    hx, hdy = pin_act(data["x"]), pin_act(data["dy"])
    hp = [pin(data[k]) for k in ("w1", "b1", "w2", "b2")]
    hy, hdx = torch.empty_like(hx).pin_memory(), torch.empty_like(hx).pin_memory()
    hg = [torch.empty_like(t).pin_memory() for t in hp]
    nbytes = max(binding.afno_spectral_host_arena_bytes(desc, m) for m in (0, 1, 2))
    for fill in (0, 0x4F):      # a zeroed arena and one full of bytes that occur in the stamp's magic
        arena = torch.full((nbytes,), fill, dtype=torch.uint8, device="cuda")
        with pytest.raises(binding.AfnoError) as ei:
            binding.afno_spectral_bwd_host(desc, None, hdy, *hp, hdx, *hg, arena)
        assert ei.value.status == binding.AFNO_ERR_INVALID_ARG and "x_host is NULL" in str(ei.value)
    binding.afno_spectral_fwd_host(desc, hx, *hp, hy, arena)
    binding.afno_spectral_bwd_host(desc, None, hdy, *hp, hdx, *hg, arena)
    ref_dx = hdx.clone()
    # x of two samples is there; a call that expects one sample's x must not take it
    with pytest.raises(binding.AfnoError) as ei:
        binding.afno_spectral_bwd_host(desc1, None, hdy[:1], *hp, hdx[:1], *hg, arena)
    assert ei.value.status == binding.AFNO_ERR_INVALID_ARG
    # bwd_host with an x of its own leaves that x behind, step_host too
    binding.afno_spectral_bwd_host(desc1, hx[:1], hdy[:1], *hp, hdx[:1], *hg, arena)
    binding.afno_spectral_bwd_host(desc1, None, hdy[:1], *hp, hdx[:1], *hg, arena)
    assert torch.equal(hdx[:1], ref_dx[:1])
    binding.afno_spectral_step_host(desc, hx, hdy, *hp, hy, hdx, *hg, arena)
    binding.afno_spectral_bwd_host(desc, None, hdy, *hp, hdx, *hg, arena)
    assert torch.equal(hdx, ref_dx)

    errs = []

    def worker():
        try:
            torch.cuda.set_device(0)
            out = torch.empty_like(hx).pin_memory()
            binding.afno_spectral_fwd_host(desc, hx, *hp, out, arena, stream=torch.cuda.current_stream())
            assert torch.equal(out, hy)
        except Exception as ex:      # surfaced below: an exception in a thread does not fail the test by itself
            errs.append(ex)

    for _ in range(8):
        t = threading.Thread(target=worker)
        t.start()
        t.join()
    assert not errs, errs
    torch.cuda.synchronize()


def test_w192_runs_on_the_generic_path(oracle):
    """W = 192 has W/2+1 = 97 bins: one more than the tcgen05 path's constant images hold.  The plan must be
    built without touching them (round-1 advisor finding: heap overflow in tc_build_plan) and the
    descriptor served by the generic path."""
    rng = np.random.default_rng(192)
    B, H, W, C, nb = 1, 64, 192, 96, 1
    data = dict(x=inputs.bf16_round(rng.standard_normal((B, H, W, C)).astype(np.float32)))
    data["w1"], data["b1"], data["w2"], data["b2"] = [
        (0.05 * rng.standard_normal(s)).astype(np.float32) for s in [(nb, 96, 96, 2), (nb, 96, 2), (nb, 96, 96, 2), (nb, 96, 2)]]
    for dt in (binding.AFNO_BF16, binding.AFNO_F32):
        desc = binding.Desc(B, H, W, C, nb, 1, 0.01, 1.0, dt)
        binding.afno_plan_warmup(desc)
        # bf16: fp32 FFTs + tensor-core MLP (hybrid forward); fp32: generic kernels throughout
        assert binding.afno_spectral_path(desc) == ("hybrid-fft32-tcgen05" if dt == binding.AFNO_BF16 else "generic-fp32")
        _check_forward(oracle, desc, data, label=f"64x192x96 dtype={dt}")


def test_data_parallel_step_with_gradient_bucket(oracle):
    """SURVEY.md S8(f) item 4 on one GPU: sharding.data_parallel_step (forward with saved context, backward writing dW / db
    straight into the views of ONE flat bucket, then the all-reduce, a no-op at world size 1) returns what the plain calls
    return, and the bucket's views are valid C-ABI outputs (16-byte aligned).  The 2-rank logic runs on CPU with gloo
    (tests/test_multiproc_cpu.py)."""
    import torch
    from paper_2208_05419_b200 import sharding
    wl = inputs.Workload(4, "30x60x192 bf16 B=2 dp", 2, 30, 60, 192, 2, 1, 0.01, 1.0, "bf16", True, False)
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    ref = _ctx_step(desc, data)
    layer = parity.GpuLayer(desc)
    tx, tdy = parity.to_device_act(data["x"], True), parity.to_device_act(data["dy"], True)
    ty, tdx = torch.empty_like(tx), torch.empty_like(tx)
    p = layer.params(data["w1"], data["b1"], data["w2"], data["b2"])
    bucket = sharding.GradBucket.allocate(wl.num_blocks, wl.C // wl.num_blocks, 1, device="cuda")
    assert all(v.data_ptr() % 16 == 0 for v in bucket.views)
    ws = torch.empty(binding.afno_spectral_workspace_bytes(desc, True), dtype=torch.uint8, device="cuda")
    n = sharding.data_parallel_step(binding, desc, tx, tdy, p, ty, tdx, bucket, ws, torch.cuda.current_stream())
    torch.cuda.synchronize()
    assert n == 9
    assert np.array_equal(parity.from_device_act(ty), ref["y"]) and np.array_equal(parity.from_device_act(tdx), ref["dx"])
    for v, k in zip(bucket.views, ("dw1", "db1", "dw2", "db2")):
        assert np.array_equal(v.cpu().numpy(), ref[k]), k


def test_data_parallel_step_on_a_side_stream_orders_the_collective_behind_the_backward():
    """The all-reduce must ride on the stream the backward wrote the bucket on, not on torch's current stream (NCCL orders
    against the current stream only).  One GPU cannot run a 2-rank NCCL group, so the process group is a stand-in that
    reports two ranks and 'reduces' by doubling the bucket on whatever stream is current when it is called: issued on
    the wrong stream it would both trip the assertion and race with k_tc_wgrad_reduce."""
    import torch
    from paper_2208_05419_b200 import sharding
    wl = inputs.Workload(4, "30x60x192 bf16 B=2 dp", 2, 30, 60, 192, 2, 1, 0.01, 1.0, "bf16", True, False)
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    ref = _ctx_step(desc, data)
    layer = parity.GpuLayer(desc)
    tx, tdy = parity.to_device_act(data["x"], True), parity.to_device_act(data["dy"], True)
    ty, tdx = torch.empty_like(tx), torch.empty_like(tx)
    p = layer.params(data["w1"], data["b1"], data["w2"], data["b2"])
    ws = torch.empty(binding.afno_spectral_workspace_bytes(desc, True), dtype=torch.uint8, device="cuda")
    side = torch.cuda.Stream()

    class TwoRanks:
        class ReduceOp:
            SUM = "sum"
        seen = []

        @staticmethod
        def get_world_size(group=None):
            return 2

        @classmethod
        def all_reduce(cls, t, op=None, group=None):
            cls.seen.append(torch.cuda.current_stream().cuda_stream)
            t.mul_(2.0)      # two ranks holding the same gradients

    for handle in (side, side.cuda_stream):     # a torch stream and the raw handle the C ABI takes
        bucket = sharding.GradBucket.allocate(wl.num_blocks, wl.C // wl.num_blocks, 1, device="cuda")
        torch.cuda.synchronize()
        assert torch.cuda.current_stream().cuda_stream != side.cuda_stream
        sharding.data_parallel_step(binding, desc, tx, tdy, p, ty, tdx, bucket, ws, handle, dist=TwoRanks)
        assert TwoRanks.seen[-1] == side.cuda_stream      # raw handles: torch stream objects do not compare reliably
        assert torch.cuda.current_stream().cuda_stream != side.cuda_stream
        torch.cuda.synchronize()
        assert np.array_equal(parity.from_device_act(tdx), ref["dx"])
        for v, k in zip(bucket.views, ("dw1", "db1", "dw2", "db2")):
            assert np.array_equal(v.cpu().numpy(), 2.0 * ref[k]), k


def test_p1_token_grid_fp32_forward(oracle):
    """SURVEY.md S8(f) item 1, last clause: the p -> 1 token grid (720 x 1,440 tokens).  One row of 1,440 points
    no longer fits shared memory at 32 packed channels; the two-pass register FFT kernels run it with 16 packed lanes per
    W tile and 32 channels per H tile (fft2pass.cuh).  fp32 path, forward, against the oracle per tile."""
    rng = np.random.default_rng(1440)
    B, H, W, C, nb = 1, 720, 1440, 64, 2
    bs = C // nb
    data = dict(x=rng.standard_normal((B, H, W, C)).astype(np.float32))
    data["w1"], data["b1"], data["w2"], data["b2"] = [
        (0.2 * rng.standard_normal(s)).astype(np.float32) for s in [(nb, bs, bs, 2), (nb, bs, 2), (nb, bs, bs, 2), (nb, bs, 2)]]
    desc = binding.Desc(B, H, W, C, nb, 1, 0.01, 1.0, binding.AFNO_F32)
    assert binding.afno_spectral_path(desc) == "generic-fp32"
    _check_forward(oracle, desc, data, label="720x1440x64 fp32")


def test_p1_token_grid_bf16_hybrid(oracle):
    """The same grid with bf16 activations on the hybrid path (32-wide blocks, partly filled last group), forward and
    backward, mask-consistently against the oracle."""
    wl = inputs.Workload(5, "720x1440x128 nb=4 bf16 B=1", 1, 720, 1440, 128, 4, 1, 0.01, 1.0, "bf16", True, False)
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    assert binding.afno_spectral_path(desc) == "hybrid-fft32-tcgen05"
    _check_forward(oracle, desc, data, label=wl.name)
    _check_backward(oracle, desc, data, label=wl.name)


def test_step_host_equals_fwd_host_then_bwd_host(oracle):
    """afno_spectral_step_host (one call per training step, both link directions busy across the forward / backward boundary)
    returns bit for bit what afno_spectral_fwd_host followed by afno_spectral_bwd_host return, on the tcgen05 path and on the
    fp32 path; y is checked against the oracle."""
    import torch
    for wl in (inputs.Workload(4, "30x60x192 bf16 B=3 step_host", 3, 30, 60, 192, 2, 1, 0.01, 1.0, "bf16", True, False),
               inputs.WORKLOADS["sub_bwd_nb2"]):
        data = inputs.make_inputs(wl)
        desc = parity.desc_for(wl)
        bf16 = wl.dtype == "bf16"
        hx, hdy = (parity.to_device_act(data[k], bf16).cpu().pin_memory() for k in ("x", "dy"))
        hp = [torch.from_numpy(np.ascontiguousarray(data[k], dtype=np.float32)).pin_memory() for k in ("w1", "b1", "w2", "b2")]
        out = {}
        for mode in ("two", "one"):
            hy, hdx = torch.empty_like(hx).pin_memory(), torch.empty_like(hx).pin_memory()
            hg = [torch.empty_like(t).pin_memory() for t in hp]
            if mode == "two":
                arena = torch.empty(max(binding.afno_spectral_host_arena_bytes(desc, 0), binding.afno_spectral_host_arena_bytes(desc, 1)),
                                    dtype=torch.uint8, device="cuda")
                binding.afno_spectral_fwd_host(desc, hx, *hp, hy, arena)
                binding.afno_spectral_bwd_host(desc, None, hdy, *hp, hdx, *hg, arena)
            else:
                arena = torch.empty(binding.afno_spectral_host_arena_bytes(desc, 2), dtype=torch.uint8, device="cuda")
                binding.afno_spectral_step_host(desc, hx, hdy, *hp, hy, hdx, *hg, arena)
            out[mode] = [hy.clone(), hdx.clone()] + [t.clone() for t in hg]
        for a, b in zip(out["two"], out["one"]):
            assert torch.equal(a, b)
        y = parity.from_device_act(out["one"][0].cuda()) if bf16 else out["one"][0].numpy()
        y_ref = oracle.forward(parity.oracle_cfg(oracle, desc), data["x"], data["w1"], data["b1"], data["w2"], data["b2"])
        assert parity.rel_l2(y, y_ref) <= _tol(desc)
        with pytest.raises(binding.AfnoError) as e:
            binding.afno_spectral_step_host(desc, hx, hdy, *hp, hy, hdx, *hg, arena[:1024])
        assert e.value.status == binding.AFNO_ERR_WORKSPACE


def test_hybrid_backward_context_flags_and_graph_replay(oracle):
    """The hybrid path keeps no context: SAVE_CONTEXT / USE_CONTEXT are accepted and the backward recomputes (include/afno.h),
    so the context step equals the plain calls bit for bit; and a forward + backward pair captured in a CUDA graph
     replays bit-identically (tc_mlp_bwd, tc_wgrad and the FFT kernels inside the capture)."""
    import torch
    wl = inputs.Workload(4, "100x40x192 bf16 B=2 hybrid ctx", 2, 100, 40, 192, 2, 1, 0.01, 1.0, "bf16", True, False)
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    assert binding.afno_spectral_path(desc) == "hybrid-fft32-tcgen05"
    layer = parity.GpuLayer(desc)
    args = (data["x"], data["dy"], data["w1"], data["b1"], data["w2"], data["b2"])
    plain = layer.backward(*args, export_masks=False)
    y_plain = layer.forward(data["x"], *args[2:])
    got = _ctx_step(desc, data)
    assert np.array_equal(got["y"], y_plain) and np.array_equal(got["dx"], plain["dx"])
    for k in ("dw1", "db1", "dw2", "db2"):
        assert np.array_equal(got[k], plain[k]), k
    # capture + replay
    tx, tdy = parity.to_device_act(data["x"], True), parity.to_device_act(data["dy"], True)
    ty, tdx = torch.zeros_like(tx), torch.zeros_like(tx)
    p = layer.params(data["w1"], data["b1"], data["w2"], data["b2"])
    g = [torch.zeros_like(t) for t in p]
    ws = torch.empty(binding.afno_spectral_workspace_bytes(desc, True), dtype=torch.uint8, device="cuda")
    s = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        with torch.cuda.graph(graph, stream=s):
            binding.afno_spectral_fwd(desc, tx, *p, ty, ws, stream=s)
            binding.afno_spectral_bwd(desc, tx, tdy, *p, tdx, *g, ws, stream=s)
    for _ in range(2):
        graph.replay()
    torch.cuda.synchronize()
    assert np.array_equal(parity.from_device_act(ty), y_plain) and np.array_equal(parity.from_device_act(tdx), plain["dx"])
    for t, k in zip(g, ("dw1", "db1", "dw2", "db2")):
        assert np.array_equal(t.cpu().numpy(), plain[k]), k


@pytest.mark.parametrize("H,W", [(90, 720), (720, 20), (36, 1440)])
def test_three_pass_fft_long_axes(oracle, H, W):
    """The three-pass register FFT kernels (fft2pass.cuh: 720 = 8 x 9 x 10, 1,440 = 16 x 9 x 10 points) on their own, each
    combined with another kernel family on the other axis: fp32 path, forward and backward against the oracle per tile."""
    rng = np.random.default_rng(H * 7 + W)
    B, C, nb = 1, 64, 2
    bs = C // nb
    data = dict(x=rng.standard_normal((B, H, W, C)).astype(np.float32), dy=rng.standard_normal((B, H, W, C)).astype(np.float32))
    data["w1"], data["b1"], data["w2"], data["b2"] = [
        (0.2 * rng.standard_normal(s)).astype(np.float32) for s in [(nb, bs, bs, 2), (nb, bs, 2), (nb, bs, bs, 2), (nb, bs, 2)]]
    desc = binding.Desc(B, H, W, C, nb, 1, 0.05, 1.0, binding.AFNO_F32)
    _check_forward(oracle, desc, data, label=f"{H}x{W}x{C} fp32 three-pass")
    _check_backward(oracle, desc, data, label=f"{H}x{W}x{C} fp32 three-pass")


def test_three_pass_fft_bf16_spectrum_w720(oracle):
    """The 720-point three-pass W kernels with the bf16 spectrum of the hybrid path (90 x 720 tokens, 32-wide blocks),
    forward and backward against the oracle."""
    wl = inputs.Workload(5, "90x720x64 nb=2 bf16 B=1", 1, 90, 720, 64, 2, 1, 0.01, 1.0, "bf16", True, False)
    data = inputs.make_inputs(wl)
    desc = parity.desc_for(wl)
    assert binding.afno_spectral_path(desc) == "hybrid-fft32-tcgen05"
    _check_forward(oracle, desc, data, label=wl.name)
    _check_backward(oracle, desc, data, label=wl.name)
