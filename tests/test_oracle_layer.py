"""Pins O5-O10, O12-O14 for the oracle's forward and backward (S3).  CPU only."""
import numpy as np
import pytest

from paper_2208_05419_b200 import inputs


def _identity_params(nb, bs):
    w = np.zeros((nb, bs, bs, 2))
    for j in range(nb):
        w[j, np.arange(bs), np.arange(bs), 0] = 1.0
    b = np.zeros((nb, bs, 2))
    return w, b, w.copy(), b.copy()


def _random_params(seed, nb, bs, hf=1, scale=0.02):
    rng = np.random.default_rng(seed)
    hid = bs * hf
    return (scale * rng.standard_normal((nb, bs, hid, 2)), scale * rng.standard_normal((nb, hid, 2)),
            scale * rng.standard_normal((nb, hid, bs, 2)), scale * rng.standard_normal((nb, bs, 2)))


def _plane(H, W, C, fn):
    h = np.arange(H)[:, None]
    w = np.arange(W)[None, :]
    return np.repeat(fn(h, w)[None, :, :, None], C, axis=3)


def _cplx(a):
    return a[..., 0] + 1j * a[..., 1]


def numpy_forward(cfg, x, w1, b1, w2, b2):
    """Third restatement with numpy.fft + einsum (test-only, O13)."""
    B, H, W, C = x.shape
    nb, bs, hid = cfg.num_blocks, cfg.bs, cfg.hid
    X = np.fft.rfft2(x, axes=(1, 2), norm="ortho").reshape(B, H, W // 2 + 1, nb, bs)
    P1 = np.einsum("bhwji,jio->bhwjo", X, _cplx(w1)) + _cplx(b1)
    O1 = np.maximum(P1.real, 0) + 1j * np.maximum(P1.imag, 0)
    P2 = np.einsum("bhwji,jio->bhwjo", O1, _cplx(w2)) + _cplx(b2)
    sh = lambda v: np.sign(v) * np.maximum(np.abs(v) - cfg.lam, 0)
    Z = (sh(P2.real) + 1j * sh(P2.imag)).reshape(B, H, W // 2 + 1, C)
    Kh = int(max(1, min(H // 2 + 1, np.floor(cfg.kept_fraction * (H // 2 + 1)))))
    Kw = int(max(1, min(W // 2 + 1, np.floor(cfg.kept_fraction * (W // 2 + 1)))))
    r = np.arange(H)
    kap = np.abs(np.where(r <= H // 2, r, r - H))
    keep = (kap[:, None] < Kh) & (np.arange(W // 2 + 1)[None, :] < Kw)
    Z = Z * keep[None, :, :, None]
    s = np.fft.irfft2(Z, s=(H, W), axes=(1, 2), norm="ortho")
    return s if cfg.no_residual else x + s


@pytest.mark.parametrize("naive", [True, False])
def test_O5_identity_mlp_cos_sin(oracle, naive):
    H, W, C, nb = 8, 16, 4, 2
    cfg = oracle.Config(1, H, W, C, nb, lam=0.0, naive_dft=naive)
    p = _identity_params(nb, C // nb)
    ang = lambda h, w: 2 * np.pi * (2 * h / H + 3 * w / W)
    xc = _plane(H, W, C, lambda h, w: np.cos(ang(h, w)))
    xs = _plane(H, W, C, lambda h, w: np.sin(ang(h, w)))
    # cos -> +real bin survives ReLU: y = 2x;  sin -> -i bin is clipped: y = x;  -sin -> y = 2x
    assert np.abs(oracle.forward(cfg, xc, *p) - 2 * xc).max() < 1e-12
    assert np.abs(oracle.forward(cfg, xs, *p) - xs).max() < 1e-12
    assert np.abs(oracle.forward(cfg, -xs, *p) - 2 * (-xs)).max() < 1e-12


def test_O6_constant_input_closed_form(oracle):
    # DC bin = c0 sqrt(HW) ("ortho"), passes ReLU, shrunk by lambda: y = 2 c0 - lambda/sqrt(HW)
    H, W, C, nb, c0, lam = 6, 10, 4, 2, 0.7, 0.01
    cfg = oracle.Config(1, H, W, C, nb, lam=lam)
    x = np.full((1, H, W, C), c0)
    y = oracle.forward(cfg, x, *_identity_params(nb, C // nb))
    assert np.abs(y - (2 * c0 - lam / np.sqrt(H * W))).max() < 1e-13


def test_O7_truncation_box(oracle):
    H, W, C, nb = 8, 16, 4, 2
    cfg = oracle.Config(1, H, W, C, nb, lam=0.0, kept_fraction=0.5)  # Kh = 2, Kw = 4
    p = _identity_params(nb, C // nb)
    cases = {(1, 3): 2.0, (-1, 3): 2.0, (2, 3): 1.0, (1, 4): 1.0, (0, 0): 2.0, (-2, 1): 1.0}
    for (k0, l0), gain in cases.items():
        x = _plane(H, W, C, lambda h, w: np.cos(2 * np.pi * (k0 * h / H + l0 * w / W)))
        y = oracle.forward(cfg, x, *p)
        assert np.abs(y - gain * x).max() < 1e-12, (k0, l0)


def test_O8_kill_switch(oracle):
    H, W, C, nb = 8, 16, 16, 2
    x = np.random.default_rng(5).standard_normal((1, H, W, C))
    w1, b1, w2, b2 = _random_params(6, nb, C // nb)
    cfg = oracle.Config(1, H, W, C, nb, lam=0.01)
    y = oracle.forward(cfg, x, w1, b1, np.zeros_like(w2), np.zeros_like(b2))
    assert np.array_equal(y, x)
    cfg_big = oracle.Config(1, H, W, C, nb, lam=1e6)
    assert np.array_equal(oracle.forward(cfg_big, x, w1, b1, w2, b2), x)


@pytest.mark.parametrize("hf", [1, 2])
def test_O9_block_dense_equivalence_and_block_independence(oracle, hf):
    H, W, C, nb = 8, 16, 16, 4
    bs, hid = C // nb, (C // nb) * hf
    rng = np.random.default_rng(9)
    x = rng.standard_normal((2, H, W, C))
    w1, b1, w2, b2 = _random_params(10, nb, bs, hf, scale=0.3)
    cfg = oracle.Config(2, H, W, C, nb, hidden_factor=hf, lam=0.01)
    y = oracle.forward(cfg, x, w1, b1, w2, b2)
    w1d = np.zeros((C, nb * hid, 2))
    w2d = np.zeros((nb * hid, C, 2))
    for j in range(nb):
        w1d[j * bs:(j + 1) * bs, j * hid:(j + 1) * hid] = w1[j]
        w2d[j * hid:(j + 1) * hid, j * bs:(j + 1) * bs] = w2[j]
    yd = oracle.forward_dense(cfg, x, w1d, b1, w2d, b2)
    assert np.abs(y - yd).max() < 1e-13
    # perturbing block 1's input channels leaves the other blocks' branch bit-identical
    x2 = x.copy()
    x2[..., bs:2 * bs] += rng.standard_normal((2, H, W, bs))
    y2 = oracle.forward(cfg, x2, w1, b1, w2, b2)
    other = np.r_[0:bs, 2 * bs:C]
    assert np.array_equal(y2[..., other], y[..., other])
    assert not np.array_equal(y2[..., bs:2 * bs], y[..., bs:2 * bs])


def test_O10_batch_independence(oracle):
    H, W, C, nb = 6, 10, 8, 2
    rng = np.random.default_rng(12)
    x = rng.standard_normal((3, H, W, C))
    p = _random_params(13, nb, C // nb, scale=0.3)
    y = oracle.forward(oracle.Config(3, H, W, C, nb), x, *p)
    y1 = oracle.forward(oracle.Config(1, H, W, C, nb), x[1:2], *p)
    assert np.array_equal(y[1:2], y1)


@pytest.mark.parametrize("H,W,C,nb,hf,f,naive", [
    (8, 16, 16, 2, 1, 1.0, True), (8, 16, 16, 2, 1, 1.0, False), (6, 10, 12, 3, 2, 0.5, False),
    (9, 15, 8, 2, 1, 0.7, False), (16, 32, 64, 8, 1, 1.0, False), (16, 32, 64, 2, 1, 0.5, False)])
def test_O13_forward_vs_numpy_restatement(oracle, H, W, C, nb, hf, f, naive):
    rng = np.random.default_rng(H * W + C)
    x = rng.standard_normal((2, H, W, C))
    p = _random_params(14, nb, C // nb, hf, scale=0.2)
    for no_res in (False, True):
        cfg = oracle.Config(2, H, W, C, nb, hidden_factor=hf, lam=0.05,
                            kept_fraction=float(np.float32(f)), no_residual=no_res, naive_dft=naive)
        y = oracle.forward(cfg, x, *p)
        assert np.abs(y - numpy_forward(cfg, x, *p)).max() < 1e-12


def test_O14_affine_regime_is_two_matrix_products(oracle):
    # lambda = 0 and b1 large enough that ReLU never clips: layer is affine (orientation A11)
    H, W, C, nb = 8, 16, 8, 2
    bs = C // nb
    rng = np.random.default_rng(15)
    x = 0.1 * rng.standard_normal((1, H, W, C))
    w1, b1, w2, b2 = _random_params(16, nb, bs, scale=0.3)
    b1 = b1 + 100.0
    cfg = oracle.Config(1, H, W, C, nb, lam=0.0, no_residual=True)
    s = oracle.forward(cfg, x, w1, b1, w2, b2)
    X = np.fft.rfft2(x, axes=(1, 2), norm="ortho")
    Z = np.empty_like(X)
    for j in range(nb):
        A = X[..., j * bs:(j + 1) * bs]
        Z[..., j * bs:(j + 1) * bs] = (A @ _cplx(w1[j]) + _cplx(b1[j])) @ _cplx(w2[j]) + _cplx(b2[j])
    ref = np.fft.irfft2(Z, s=(H, W), axes=(1, 2), norm="ortho")
    assert np.abs(s - ref).max() < 1e-10


def test_configs0_golden_regression(oracle):
    """tests/golden/configs0_oracle.txt is written by tests/golden/make_golden.py, which calls
    only oracle/: a regression pin that the committed oracle has not drifted."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "configs0_oracle.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    wl = inputs.WORKLOADS["tiny"]
    d = inputs.make_inputs(wl)
    cfg = oracle.Config(wl.B, wl.H, wl.W, wl.C, wl.num_blocks, lam=float(np.float32(wl.lam)),
                        naive_dft=True)
    y = oracle.forward(cfg, d["x"], d["w1"], d["b1"], d["w2"], d["b2"])
    for h, w, c, val in rows:
        assert abs(y[0, int(h), int(w), int(c)] - float(val)) < 1e-13


# ----------------------------------------------------------------------------------------
# Backward
# ----------------------------------------------------------------------------------------

def _loss_and_masks(oracle, cfg, x, dy, p):
    y, dump = oracle.forward(cfg, x, *p, dump=True)
    m1 = np.stack([dump["p1"].real > 0, dump["p1"].imag > 0], -1)
    m2 = np.stack([np.abs(dump["p2"].real) > cfg.lam, np.abs(dump["p2"].imag) > cfg.lam], -1)
    return (dy * y).sum(), m1, m2


@pytest.mark.parametrize("H,W,C,nb,hf,f", [(8, 16, 16, 2, 1, 1.0), (6, 10, 12, 3, 2, 0.5),
                                            (16, 32, 64, 2, 1, 1.0), (16, 32, 64, 8, 1, 0.5)])
def test_O12_finite_differences(oracle, H, W, C, nb, hf, f):
    """L = sum(dY (.) y); central differences along random directions in x and every
    parameter agree with <grad, direction> when no mask changes between +-eps."""
    B = 2
    rng = np.random.default_rng(100 + H + C + nb)
    x = rng.standard_normal((B, H, W, C))
    dy = rng.standard_normal((B, H, W, C))
    p = list(_random_params(101, nb, C // nb, hf, scale=0.25))
    cfg = oracle.Config(B, H, W, C, nb, hidden_factor=hf, lam=0.05, kept_fraction=f)
    g = oracle.backward(cfg, x, dy, *p)
    grads = [g["dx"], g["dw1"], g["db1"], g["dw2"], g["db2"]]
    args = [x] + p
    eps = 1e-6
    checked = 0
    for which in range(5):
        for trial in range(6):
            dirn = rng.standard_normal(args[which].shape)
            plus = [a.copy() for a in args]
            minus = [a.copy() for a in args]
            plus[which] = plus[which] + eps * dirn
            minus[which] = minus[which] - eps * dirn
            Lp, m1p, m2p = _loss_and_masks(oracle, cfg, plus[0], dy, plus[1:])
            Lm, m1m, m2m = _loss_and_masks(oracle, cfg, minus[0], dy, minus[1:])
            if not (np.array_equal(m1p, m1m) and np.array_equal(m2p, m2m)):
                continue  # a kink was crossed: redraw the direction
            fd = (Lp - Lm) / (2 * eps)
            an = (grads[which] * dirn).sum()
            assert abs(fd - an) <= 2e-7 * max(1.0, abs(an)), (which, fd, an)
            checked += 1
            break
        else:
            pytest.fail("no mask-stable direction found")
    assert checked == 5


@pytest.mark.parametrize("H,W,C,nb,hf,f", [(8, 16, 16, 2, 1, 1.0), (9, 15, 8, 2, 2, 0.6),
                                            (16, 32, 64, 8, 1, 1.0)])
def test_O13_backward_vs_torch_autograd(oracle, H, W, C, nb, hf, f):
    torch = pytest.importorskip("torch")
    B = 2
    rng = np.random.default_rng(200 + H)
    x = rng.standard_normal((B, H, W, C))
    dy = rng.standard_normal((B, H, W, C))
    p = _random_params(201, nb, C // nb, hf, scale=0.25)
    f = float(np.float32(f))
    cfg = oracle.Config(B, H, W, C, nb, hidden_factor=hf, lam=0.05, kept_fraction=f)
    g = oracle.backward(cfg, x, dy, *p)

    tx = torch.tensor(x, dtype=torch.float64, requires_grad=True)
    tp = [torch.tensor(a, dtype=torch.float64, requires_grad=True) for a in p]
    bs, hid = cfg.bs, cfg.hid
    X = torch.fft.rfft2(tx, dim=(1, 2), norm="ortho").reshape(B, H, W // 2 + 1, nb, bs)
    P1 = torch.einsum("bhwji,jio->bhwjo", X, torch.view_as_complex(tp[0])) + torch.view_as_complex(tp[1])
    O1 = torch.view_as_complex(torch.relu(torch.view_as_real(P1)))
    P2 = torch.einsum("bhwji,jio->bhwjo", O1, torch.view_as_complex(tp[2])) + torch.view_as_complex(tp[3])
    Z = torch.view_as_complex(torch.nn.functional.softshrink(torch.view_as_real(P2), lambd=0.05))
    Kh, Kw = oracle.kept(H, W, f)
    r = np.arange(H)
    kap = np.abs(np.where(r <= H // 2, r, r - H))
    keep = torch.tensor((kap[:, None] < Kh) & (np.arange(W // 2 + 1)[None, :] < Kw))
    Z = Z.reshape(B, H, W // 2 + 1, C) * keep[None, :, :, None]
    y = tx + torch.fft.irfft2(Z, s=(H, W), dim=(1, 2), norm="ortho")
    (y * torch.tensor(dy)).sum().backward()
    for name, t in zip(("dx", "dw1", "db1", "dw2", "db2"), [tx] + tp):
        ref = t.grad.numpy()
        assert np.abs(g[name] - ref).max() <= 1e-11 * max(1.0, np.abs(ref).max()), name


def test_backward_mask_override_and_no_residual(oracle):
    H, W, C, nb = 8, 16, 16, 2
    B = 1
    rng = np.random.default_rng(300)
    x = rng.standard_normal((B, H, W, C))
    dy = rng.standard_normal((B, H, W, C))
    p = _random_params(301, nb, C // nb, scale=0.25)
    cfg = oracle.Config(B, H, W, C, nb, lam=0.05)
    g = oracle.backward(cfg, x, dy, *p, dump=True)
    d = g["dump"]
    m1 = np.stack([d["p1"].real > 0, d["p1"].imag > 0], -1).astype(np.uint8)
    m2 = np.stack([np.abs(d["p2"].real) > 0.05, np.abs(d["p2"].imag) > 0.05], -1).astype(np.uint8)
    g2 = oracle.backward(cfg, x, dy, *p, mask1=m1, mask2=m2)
    for k in ("dx", "dw1", "db1", "dw2", "db2"):
        assert np.array_equal(g[k], g2[k])
    # all-zero masks: no gradient reaches the parameters, dx = dy
    g0 = oracle.backward(cfg, x, dy, *p, mask1=np.zeros_like(m1), mask2=np.zeros_like(m2))
    assert np.array_equal(g0["dx"], dy)
    assert not g0["dw1"].any() and not g0["dw2"].any() and not g0["db2"].any()
    # branch-only variant differs from the full one by exactly dy
    cfg_nr = oracle.Config(B, H, W, C, nb, lam=0.05, no_residual=True)
    gn = oracle.backward(cfg_nr, x, dy, *p)
    assert np.abs(gn["dx"] + dy - g["dx"]).max() < 1e-13
