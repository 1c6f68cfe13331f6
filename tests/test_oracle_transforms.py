"""Pins O1-O4, O11 for the oracle's transforms (S3).  CPU only.

Each pin checks the oracle against something other than itself: the literal O(N^2)
definition, numpy.fft (a library routine the special case reduces to), closed forms
and algebraic identities.
"""
import numpy as np
import pytest

SHAPES = [(8, 16), (6, 10), (9, 15), (16, 32), (12, 18), (30, 20), (5, 7)]


def _rng(seed):
    return np.random.default_rng(seed)


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 12, 15, 16, 30, 45, 90, 180, 22])
def test_dft1_fast_equals_definition_and_numpy(oracle, n):
    a = _rng(n).standard_normal(n) + 1j * _rng(n + 1).standard_normal(n)
    for sign in (-1, +1):
        slow = oracle.dft1(a, sign, naive=True)
        fast = oracle.dft1(a, sign, naive=False)
        ref = np.fft.fft(a) if sign < 0 else np.fft.ifft(a) * n
        assert np.abs(fast - slow).max() <= 1e-12 * max(1.0, np.abs(slow).max())
        assert np.abs(slow - ref).max() <= 1e-12 * max(1.0, np.abs(ref).max())


@pytest.mark.parametrize("H,W", SHAPES)
def test_O1_rfft2_fast_equals_brute_force(oracle, H, W):
    x = _rng(H * 100 + W).standard_normal((H, W))
    brute = oracle.rfft2(x, naive=True)
    fast = oracle.rfft2(x, naive=False)
    assert np.abs(brute - fast).max() <= 1e-12


def test_O1_brute_force_is_the_written_definition(oracle):
    # retype definition 1 with explicit python loops on a tiny grid
    H, W = 4, 6
    x = _rng(7).standard_normal((H, W))
    X = oracle.rfft2(x, naive=True)
    for r in range(H):
        for c in range(W // 2 + 1):
            acc = 0.0
            for h in range(H):
                for w in range(W):
                    acc += x[h, w] * np.exp(-2j * np.pi * (r * h / H + c * w / W))
            assert abs(X[r, c] - acc / np.sqrt(H * W)) < 1e-13


def test_O1_full_grid_one_channel(oracle):
    H, W = 90, 180
    x = _rng(3).standard_normal((H, W))
    brute = oracle.rfft2(x, naive=True)
    fast = oracle.rfft2(x, naive=False)
    assert np.abs(brute - fast).max() <= 1e-12
    assert np.abs(fast - np.fft.rfft2(x, norm="ortho")).max() <= 1e-12


@pytest.mark.parametrize("H,W", SHAPES)
def test_O13_library_restatement(oracle, H, W):
    x = _rng(11).standard_normal((H, W))
    assert np.abs(oracle.rfft2(x) - np.fft.rfft2(x, norm="ortho")).max() <= 1e-13
    Z = _rng(12).standard_normal((H, W // 2 + 1)) + 1j * _rng(13).standard_normal((H, W // 2 + 1))
    ref = np.fft.irfft2(Z, s=(H, W), norm="ortho")  # non-Hermitian input: reading A4
    assert np.abs(oracle.irfft2(Z, W, naive=True) - ref).max() <= 1e-13
    assert np.abs(oracle.irfft2(Z, W, naive=False) - ref).max() <= 1e-13


@pytest.mark.parametrize("H,W", SHAPES)
def test_O2_round_trip(oracle, H, W):
    x = _rng(21).standard_normal((H, W))
    for naive in (True, False):
        back = oracle.irfft2(oracle.rfft2(x, naive), W, naive)
        assert np.abs(back - x).max() <= 1e-13


@pytest.mark.parametrize("H,W", SHAPES)
def test_O3_parseval(oracle, H, W):
    x = _rng(31).standard_normal((H, W))
    X = oracle.rfft2(x)
    alpha = np.full(W // 2 + 1, 2.0)
    alpha[0] = 1.0
    if W % 2 == 0:
        alpha[W // 2] = 1.0
    assert abs((x ** 2).sum() - (alpha[None, :] * np.abs(X) ** 2).sum()) <= 1e-11 * (x ** 2).sum()


@pytest.mark.parametrize("H,W,k0,l0", [(8, 16, 1, 3), (8, 16, -1, 3), (90, 180, 7, 11), (6, 10, 2, 4),
                                        (16, 32, 0, 5)])
def test_O4_single_cosine_maps_to_single_mode(oracle, H, W, k0, l0):
    h = np.arange(H)[:, None]
    w = np.arange(W)[None, :]
    x = np.cos(2 * np.pi * (k0 * h / H + l0 * w / W))
    X = oracle.rfft2(x)
    expect = np.zeros_like(X)
    expect[k0 % H, l0] = np.sqrt(H * W) / 2  # real, positive
    assert np.abs(X - expect).max() <= 1e-11


def test_O4_cosine_on_dc_column_gives_two_bins(oracle):
    H, W, k0 = 8, 16, 3
    x = np.cos(2 * np.pi * k0 * np.arange(H)[:, None] / H) * np.ones((1, W))
    X = oracle.rfft2(x)
    expect = np.zeros_like(X)
    expect[k0, 0] = expect[H - k0, 0] = np.sqrt(H * W) / 2
    assert np.abs(X - expect).max() <= 1e-12


def test_O5_sine_sign_convention(oracle):
    # forward kernel is exp(-i...): sin -> -i sqrt(HW)/2 at (k0, l0)   (reading A2)
    H, W, k0, l0 = 8, 16, 2, 5
    h = np.arange(H)[:, None]
    w = np.arange(W)[None, :]
    X = oracle.rfft2(np.sin(2 * np.pi * (k0 * h / H + l0 * w / W)))
    expect = np.zeros_like(X)
    expect[k0, l0] = -1j * np.sqrt(H * W) / 2
    assert np.abs(X - expect).max() <= 1e-12


@pytest.mark.parametrize("H,W", SHAPES)
def test_O11_dot_product_adjoint_identities(oracle, H, W):
    Wh = W // 2 + 1
    alpha = np.full(Wh, 2.0)
    alpha[0] = 1.0
    if W % 2 == 0:
        alpha[W // 2] = 1.0
    rng = _rng(41)
    dy = rng.standard_normal((H, W))
    Z = rng.standard_normal((H, Wh)) + 1j * rng.standard_normal((H, Wh))
    x = rng.standard_normal((H, W))
    g = rng.standard_normal((H, Wh)) + 1j * rng.standard_normal((H, Wh))
    real_inner = lambda a, b: (a.real * b.real + a.imag * b.imag).sum()
    # <dy, irfft2(Z)> = <alpha (.) rfft2(dy), Z>_R
    lhs = (dy * oracle.irfft2(Z, W)).sum()
    rhs = real_inner(alpha[None, :] * oracle.rfft2(dy), Z)
    assert abs(lhs - rhs) <= 1e-12 * max(1.0, abs(lhs))
    # <g, rfft2(x)>_R = <irfft2(g / alpha), x>
    lhs = real_inner(g, oracle.rfft2(x))
    rhs = (oracle.irfft2(g / alpha[None, :], W) * x).sum()
    assert abs(lhs - rhs) <= 1e-12 * max(1.0, abs(lhs))


def test_kept_set_reading_A7_A8(oracle):
    assert oracle.kept(90, 180, 1.0) == (46, 91)     # every mode
    assert oracle.kept(90, 180, 0.5) == (23, 45)     # |kappa| <= 22 -> 45 rows, 45 columns
    assert oracle.kept(8, 16, 0.5) == (2, 4)
    assert oracle.kept(180, 360, 1.0) == (91, 181)
    assert oracle.kept(8, 16, 1e-6) == (1, 1)        # clamped to >= 1
