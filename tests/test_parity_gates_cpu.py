"""CPU tests of the parity GATES themselves (tests/parity.py): they must bite.

* the flip-justification tolerance tau = TAU_K sigma (statistical error model of the bf16 path) leaves only a
  small fraction of all masks "justifiable" on the headline workload (a tau that covers most masks cannot
  fail: round-1 verdict, What's weak 1);
* the error model is pinned to something other than itself: a numpy emulation of the path's roundings
  (every GEMM operand rounded to bf16, fp32 results) against the fp64 oracle;
* the per-tile gates fail on one corrupted tile that the whole-tensor rel-L2 gate lets through.
"""
import numpy as np
import pytest

from paper_2208_05419_b200 import inputs

import parity


@pytest.fixture(scope="module")
def headline_b1(oracle):
    wl = inputs.WORKLOADS["fcn_b4_bwd"]
    d = inputs.make_inputs(wl, B=1)
    cfg = oracle.Config(1, wl.H, wl.W, wl.C, wl.num_blocks, lam=float(np.float32(wl.lam)), kept_fraction=1.0)
    y, dump = oracle.forward(cfg, d["x"], d["w1"], d["b1"], d["w2"], d["b2"], dump=True)
    s1, s2 = parity.preactivation_scales(cfg, dump, *(d[k].astype(np.float64) for k in ("w1", "b1", "w2", "b2")))
    return wl, d, cfg, y, dump, s1, s2


def test_tau_covers_only_a_small_fraction_of_masks(headline_b1):
    wl, d, cfg, y, dump, s1, s2 = headline_b1
    p1, p2 = dump["p1"], dump["p2"]
    near1 = (np.abs(np.stack([p1.real, p1.imag], -1)) <= parity.TAU_K * s1[..., None]).mean()
    near2 = (np.abs(np.abs(np.stack([p2.real, p2.imag], -1)) - cfg.lam) <= parity.TAU_K * s2[..., None]).mean()
    print(f"fraction of masks within tau of their threshold: relu {near1:.4f} softshrink {near2:.4f}")
    assert near1 <= 0.10 and near2 <= 0.10


def _emulate_bf16_path(wl, d):
    """The tcgen05 path's roundings restated in numpy: bf16 DFT matrices, bf16 intermediates, bf16 weights,
    wide accumulation (S3 reading A15).  Returns the complex pre-activations P1, P2 [1,H,Wh,C]."""
    r = lambda a: inputs.bf16_round(np.asarray(a, dtype=np.float32)).astype(np.float64)
    H, W, C, nb = wl.H, wl.W, wl.C, wl.num_blocks
    bs, Wh = C // nb, W // 2 + 1
    x = d["x"].astype(np.float64)[0]
    ang = 2 * np.pi * ((np.arange(Wh)[:, None] * np.arange(W)[None, :]) % W) / W
    Fc, Fs = r(np.cos(ang) / np.sqrt(W)), r(-np.sin(ang) / np.sqrt(W))
    A1r, A1i = r(np.einsum("kw,hwc->hkc", Fc, x)), r(np.einsum("kw,hwc->hkc", Fs, x))
    angh = 2 * np.pi * ((np.arange(H)[:, None] * np.arange(H)[None, :]) % H) / H
    Ch, Sh = r(np.cos(angh) / np.sqrt(H)), r(np.sin(angh) / np.sqrt(H))
    Xr = r(np.einsum("rh,hkc->rkc", Ch, A1r) + np.einsum("rh,hkc->rkc", Sh, A1i))
    Xi = r(np.einsum("rh,hkc->rkc", Ch, A1i) - np.einsum("rh,hkc->rkc", Sh, A1r))
    X = (Xr + 1j * Xi).reshape(H, Wh, nb, bs)
    w1, w2 = r(d["w1"]), r(d["w2"])
    b1, b2 = d["b1"].astype(np.float64), d["b2"].astype(np.float64)
    P1 = np.einsum("rkji,jio->rkjo", X, w1[..., 0] + 1j * w1[..., 1]) + (b1[..., 0] + 1j * b1[..., 1])
    O1 = r(np.maximum(P1.real, 0)) + 1j * r(np.maximum(P1.imag, 0))
    P2 = np.einsum("rkji,jio->rkjo", O1, w2[..., 0] + 1j * w2[..., 1]) + (b2[..., 0] + 1j * b2[..., 1])
    return P1.reshape(1, H, Wh, C), P2.reshape(1, H, Wh, C)


def test_error_model_against_emulated_bf16_path(headline_b1):
    """sigma of parity.preactivation_scales against measured errors of an emulated bf16 pipeline: the errors
    are of the modelled size (std of error / sigma between 0.3 and 1.5), no error exceeds 1.5 TAU_K sigma,
    and every mask the emulation flips is justified under tau = TAU_K sigma."""
    wl, d, cfg, y, dump, s1, s2 = headline_b1
    P1, P2 = _emulate_bf16_path(wl, d)
    for name, P, ref, sg in (("P1", P1, dump["p1"], s1), ("P2", P2, dump["p2"], s2)):
        e = np.concatenate([((P.real - ref.real) / sg).ravel(), ((P.imag - ref.imag) / sg).ravel()])
        print(f"{name}: error / sigma std {e.std():.3f} p99.9 {np.quantile(np.abs(e), 0.999):.2f} max {np.abs(e).max():.2f}")
        assert 0.3 <= e.std() <= 1.5
        assert np.abs(e).max() <= 1.5 * parity.TAU_K
    m1 = np.stack([P1.real > 0, P1.imag > 0], -1)
    m2 = np.stack([np.abs(P2.real) > cfg.lam, np.abs(P2.imag) > cfg.lam], -1)
    rep = parity.mask_flip_report(dump, m1, m2, cfg.lam, parity.TAU_K * s1, parity.TAU_K * s2, kept=parity.kept_modes(cfg))
    print(rep)
    assert 0 < rep["flip1"] <= 5e-3 and 0 < rep["flip2"] <= 5e-3
    assert rep["justified"], rep


def test_unjustified_flips_are_caught(headline_b1):
    """A mask set that is wrong far from the thresholds (the masks of ANOTHER channel) fails gate (ii)."""
    wl, d, cfg, y, dump, s1, s2 = headline_b1
    p1, z = dump["p1"], dump["z"]
    m1 = np.stack([p1.real > 0, p1.imag > 0], -1)
    m2 = np.stack([z.real != 0, z.imag != 0], -1)
    ok = parity.mask_flip_report(dump, m1, m2, cfg.lam, parity.TAU_K * s1, parity.TAU_K * s2, kept=parity.kept_modes(cfg))
    assert ok["justified"] and ok["flip1"] == 0 and ok["flip2"] == 0
    bad1 = m1.copy()
    bad1[0, 7, 13, 100] = ~bad1[0, 7, 13, 100]        # one mode tile's worth is enough: flip one channel's pair
    far = np.abs(p1.real[0, 7, 13, 100]) > parity.TAU_K * s1[0, 7, 13, 100] or \
        np.abs(p1.imag[0, 7, 13, 100]) > parity.TAU_K * s1[0, 7, 13, 100]
    rep = parity.mask_flip_report(dump, bad1, m2, cfg.lam, parity.TAU_K * s1, parity.TAU_K * s2, kept=parity.kept_modes(cfg))
    assert far and not rep["justified"], rep
    bad2 = np.roll(m2, 1, axis=3)                      # masks shifted by one channel
    rep = parity.mask_flip_report(dump, m1, bad2, cfg.lam, parity.TAU_K * s1, parity.TAU_K * s2, kept=parity.kept_modes(cfg))
    assert not rep["justified"] and rep["flip2"] > 5e-3


def test_one_corrupted_tile_fails_the_tile_gate_not_the_whole_tensor_gate(headline_b1):
    """A fault copied into ONE (b, h, block) tile of y (that tile halved, i.e. 50 % wrong) moves the
    whole-tensor rel-L2 by only ~0.5 sqrt(1/720) (at B = 4, 2,880 tiles, even a 100 % wrong tile stays under
    2e-2): the round-1 gate passes it, the per-tile gate does not.  The same for one (b, kw, block) mode
    tile of the branch s dropped from the spectrum."""
    wl, d, cfg, y, dump, s1, s2 = headline_b1
    tol, blk = 2e-2, wl.C // wl.num_blocks
    rng = np.random.default_rng(1)
    good = y * (1.0 + 1.5e-3 * rng.standard_normal(y.shape))        # bf16-sized honest error
    parity.gate_activation(good, y, tol, blk, "honest")
    bad = good.copy()
    bad[0, 41, :, 3 * blk:4 * blk] *= 0.5
    assert parity.rel_l2(bad, y) <= tol                              # the old gate is blind to it
    with pytest.raises(AssertionError) as e:
        parity.gate_activation(bad, y, tol, blk, "one dead tile")
    assert "tile (b,h,block)" in str(e.value)
    # branch: drop one kw column of one block from the spectrum Z before the inverse transform
    from oracle import afno_oracle
    z = dump["z"][0, :, :, 2 * blk:3 * blk]                        # block 2: [H, Wh, 96]
    inv = lambda zz: np.stack([afno_oracle.irfft2(zz[:, :, c], wl.W) for c in range(blk)], -1)[None]
    s_ref = inv(z)
    zb = z.copy()
    zb[:, 20, :] = 0.0                                               # the (b, kw = 20, block 2) mode tile is lost
    s_bad = inv(zb)
    whole = parity.rel_l2(s_bad, s_ref) / np.sqrt(wl.num_blocks)     # its weight in the whole tensor (8 blocks)
    slabs = parity.tile_rel_l2(s_bad, s_ref, blk, slab=True)
    print(f"dropped mode tile: whole-tensor rel_l2 ~{whole:.3e}, its slab {slabs.max():.3e}")
    assert whole <= tol < slabs.max()
    with pytest.raises(AssertionError):
        parity.gate_activation(s_bad, s_ref, tol, blk, "one dead mode tile")
    # a single element off by more than MAXABS_K * tol * rms
    spike = good.copy()
    spike[0, 3, 7, 11] += 1.0
    assert parity.rel_l2(spike, y) <= tol and parity.tile_rel_l2(spike, y, blk).max() <= tol
    with pytest.raises(AssertionError) as e:
        parity.gate_activation(spike, y, tol, blk, "spike")
    assert "max_abs" in str(e.value)
