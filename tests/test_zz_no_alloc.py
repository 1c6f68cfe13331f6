"""afno_block_wgrad_static: the parameter-gradient kernels for callers that may not allocate device memory.

Some users of this library run where cudaMalloc / cudaFree are not an option and no spare device buffer can be handed
over as a workspace: an operator inside a framework or serving engine whose memory pool owns the whole device, a
latency-critical loop that cannot afford the device-wide synchronisation an allocation may cause, a process whose
fixed memory reservation is already handed out.  For them the library keeps the split partial sums of rows B4 / B6
(dW, db of one block-diagonal complex layer) in a static device array of 16 MiB (include/afno.h,
AFNO_STATIC_SCRATCH_BYTES) and offers one entry point that allocates nothing.

The GPU test checks that entry point against the EXISTING path: afno_spectral_bwd on the generic-fp32 kernels, whose
partial sums live in a caller workspace.  The operands that path forms internally (Xh, O1, G2, G1) are rebuilt here in
fp64 numpy from the same x, dy and parameters, with the activation masks the existing path exported, so a threshold
decision can never differ between the two.  Two calls follow each other on one stream without a synchronisation in
between and with different shapes (layer 2, then layer 1), so the second call finds the first call's partial sums in
the array; a third call repeats the first and must reproduce it bit for bit.

The file sorts last on purpose: pytest -x stops at the first failure, and a failure here must not hide the parity
tests.  It passes on its own in a fresh process (the first test is then the library's first use on the device, which
is the set-up path of the entry point) and after the other tests.
"""
import ctypes

import numpy as np
import pytest

from paper_2208_05419_b200 import binding, inputs

import parity

TOL_F32 = 1e-5   # the fp32 contract tolerance of tests/test_gpu_parity.py (relative L2)


def _cplx(a):
    a = np.asarray(a, dtype=np.float64)
    return a[..., 0] + 1j * a[..., 1]


def _pairs(z):
    return np.stack([z.real, z.imag], -1)


def _dev_rows(z):
    """complex [M, n] -> contiguous fp32 device tensor [M, n, 2]"""
    import torch
    return torch.from_numpy(np.ascontiguousarray(_pairs(z), dtype=np.float32)).cuda()


def _wgrad_f64(a, g, nb):
    """The definition in include/afno.h, in fp64, on the fp32-rounded operands the device received."""
    a = _cplx(np.float32(_pairs(a)))
    g = _cplx(np.float32(_pairs(g)))
    M = a.shape[0]
    ab, gb = a.reshape(M, nb, -1), g.reshape(M, nb, -1)
    return _pairs(np.einsum("mji,mjo->jio", ab.conj(), gb)), _pairs(gb.sum(0))


def _call(a, g, nb, flags=0, out=None):
    import torch
    M, K, N = a.shape[0], a.shape[1] // nb, g.shape[1] // nb
    if out is None:
        out = (torch.full((nb, K, N, 2), float("nan"), device="cuda"), torch.full((nb, N, 2), float("nan"), device="cuda"))
    binding.afno_block_wgrad_static(a, g, M, nb, K, N, out[0], out[1], flags=flags)
    return out


@pytest.mark.gpu
def test_first_use_in_a_fresh_process_random_operands():
    """Run alone, this is the first thing the process asks of the library on the device: the address lookup of the
    static array happens here.  Random operands with a ragged row count and row strides wider than the data, against
    the fp64 definition; then a shape change that reuses the array."""
    import torch
    rng = np.random.Generator(np.random.PCG64(inputs.seed_for(9, 0)))
    for (M, nb, K, N, pad) in [(1000 + 7, 3, 40, 100, 5), (33, 2, 100, 7, 0), (1, 1, 1, 1, 3)]:
        a = rng.standard_normal((M, nb * K + pad)) + 1j * rng.standard_normal((M, nb * K + pad))
        g = rng.standard_normal((M, nb * N + pad)) + 1j * rng.standard_normal((M, nb * N + pad))
        ta, tg = _dev_rows(a), _dev_rows(g)
        dw = torch.full((nb, K, N, 2), float("nan"), device="cuda")
        db = torch.full((nb, N, 2), float("nan"), device="cuda")
        binding.afno_block_wgrad_static(ta, tg, M, nb, K, N, dw, db, lda=nb * K + pad, ldg=nb * N + pad)
        torch.cuda.synchronize()
        assert binding.afno_last_launch_count() == 3
        rw, rb = _wgrad_f64(a[:, :nb * K], g[:, :nb * N], nb)
        assert parity.rel_l2(dw.cpu().numpy(), rw) <= TOL_F32, (M, nb, K, N)
        assert parity.rel_l2(db.cpu().numpy(), rb) <= TOL_F32, (M, nb, K, N)


@pytest.mark.gpu
def test_static_scratch_wgrad_matches_the_workspace_path_two_calls_in_a_row():
    import torch
    B, H, W, C, nb, hf = 2, 12, 20, 48, 4, 2
    d = binding.Desc(B=B, H=H, W=W, C=C, num_blocks=nb, hidden_factor=hf, lam=0.01, kept_fraction=0.75,
                     dtype=binding.AFNO_F32)
    assert binding.afno_spectral_path(d) == "generic-fp32"
    bs, hid, Wh = d.bs, d.hid, d.Wh
    x = inputs.field(inputs.seed_for(9, inputs.STREAM_X), B, H, W, C)
    dy = inputs.gaussian(inputs.seed_for(9, inputs.STREAM_DY), (B, H, W, C))
    w1, b1, w2, b2 = inputs.weights(9, nb, bs, hf, scale=0.1)

    # the existing path: partial sums in the caller's workspace
    ref = parity.GpuLayer(d).backward(x, dy, w1, b1, w2, b2, export_masks=True)
    m1 = ref["mask1"].astype(np.float64).reshape(B, H, Wh, nb, hid, 2)
    m2 = ref["mask2"].astype(np.float64).reshape(B, H, Wh, nb, bs, 2)
    assert 0.02 < m1.mean() < 0.98 and 0.02 < m2.mean() < 0.98   # both activations and the truncation are at work

    # the operands of rows B4 / B6 (include/afno.h formulas), fp64, with the existing path's own masks
    W1, B1, W2 = _cplx(w1), _cplx(b1), _cplx(w2)
    Xh = np.fft.rfft2(x.astype(np.float64), axes=(1, 2), norm="ortho").reshape(B, H, Wh, nb, bs)
    P1 = np.einsum("bhwji,jio->bhwjo", Xh, W1) + B1
    O1 = np.maximum(P1.real, 0) + 1j * np.maximum(P1.imag, 0)
    alpha = np.full(Wh, 2.0)
    alpha[0] = alpha[W // 2] = 1.0
    G = (alpha[None, None, :, None] * np.fft.rfft2(dy.astype(np.float64), axes=(1, 2), norm="ortho")).reshape(B, H, Wh, nb, bs)
    G2 = G.real * m2[..., 0] + 1j * G.imag * m2[..., 1]
    G1 = np.einsum("bhwjo,jio->bhwji", G2, W2.conj())
    G1 = G1.real * m1[..., 0] + 1j * G1.imag * m1[..., 1]
    M = B * H * Wh
    a2, g2 = _dev_rows(O1.reshape(M, nb * hid)), _dev_rows(G2.reshape(M, C))     # layer 2: K = hid, N = bs
    a1, g1 = _dev_rows(Xh.reshape(M, C)), _dev_rows(G1.reshape(M, nb * hid))     # layer 1: K = bs, N = hid

    # two calls in a row, no synchronisation between them; then the first one again
    dw2, db2 = _call(a2, g2, nb)
    dw1, db1 = _call(a1, g1, nb)
    dw2_again, db2_again = _call(a2, g2, nb)
    torch.cuda.synchronize()
    got = dict(dw1=dw1, db1=db1, dw2=dw2, db2=db2)
    for k, t in got.items():
        err = parity.rel_l2(t.cpu().numpy(), ref[k])
        print(f"[no-alloc] {k}: rel_l2 vs afno_spectral_bwd = {err:.3e}")
        assert np.isfinite(t.cpu().numpy()).all(), k
        assert err <= TOL_F32, (k, err)
    assert torch.equal(dw2, dw2_again) and torch.equal(db2, db2_again)

    # AFNO_FLAG_ACCUM_GRADS adds to what is there
    _call(a2, g2, nb, flags=binding.FLAG_ACCUM_GRADS, out=(dw2_again, db2_again))
    torch.cuda.synchronize()
    assert parity.rel_l2(dw2_again.cpu().numpy(), 2.0 * ref["dw2"]) <= TOL_F32
    assert parity.rel_l2(db2_again.cpu().numpy(), 2.0 * ref["db2"]) <= TOL_F32

    # no rows: zeros (operands not read)
    z = _call(torch.empty(0, nb * hid, 2, device="cuda"), torch.empty(0, C, 2, device="cuda"), nb)
    torch.cuda.synchronize()
    assert float(z[0].abs().max()) == 0.0 and float(z[1].abs().max()) == 0.0


def test_sizes_beyond_the_static_array_are_rejected_before_any_cuda_call():
    """No GPU needed: the checks come first.  nb * (K + 1) * N * 8 bytes must fit AFNO_STATIC_SCRATCH_BYTES."""
    L = binding.lib()
    dummy = ctypes.c_void_p(256)
    # one block of 1,024 x 1,024 fits (8.4 MB), 2,048 x 1,024 does not (16.8 MB > 16 MiB)
    rc = L.afno_block_wgrad_static(dummy, 2048, dummy, 1024, 16, 1, 2048, 1024, dummy, dummy, 0, None)
    assert rc == binding.AFNO_ERR_UNSUPPORTED
    msg = L.afno_last_error().decode()
    assert "static scratch" in msg and str(binding.STATIC_SCRATCH_BYTES) in msg and str(1 * 2049 * 1024 * 8) in msg
    assert 1 * 1025 * 1024 * 8 <= binding.STATIC_SCRATCH_BYTES
    for bad in [
        (None, 8, dummy, 8, 4, 1, 8, 8, dummy, dummy, 0),               # NULL operand with M > 0
        (dummy, 8, dummy, 8, 4, 1, 8, 8, None, dummy, 0),               # NULL output
        (dummy, 7, dummy, 8, 4, 1, 8, 8, dummy, dummy, 0),              # lda < nb*K
        (dummy, 8, dummy, 8, -1, 1, 8, 8, dummy, dummy, 0),             # negative M
        (dummy, 8, dummy, 8, 4, 0, 8, 8, dummy, dummy, 0),              # no blocks
        (dummy, 8, dummy, 8, 4, 1, 8, 8, dummy, dummy, 1),              # a flag of another call
        (ctypes.c_void_p(260), 8, dummy, 8, 4, 1, 8, 8, dummy, dummy, 0),   # misaligned
    ]:
        assert L.afno_block_wgrad_static(*bad, None) == binding.AFNO_ERR_INVALID_ARG, bad
        assert L.afno_last_error() != b""
