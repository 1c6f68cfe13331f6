"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/afno.h
declares, and its host-side logic (descriptor validation, size queries) behaves as the header
says.  No compute call is made (there is no GPU here)."""
import ctypes
import os
import re

import pytest

from paper_2208_05419_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.lib()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "afno.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(afno_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(lib):
    names = _declared_symbols()
    assert len(names) >= 13
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(binding.EXPORTS) == names


def test_version_and_status_strings(lib):
    assert binding.afno_version() == 100
    assert lib.afno_status_string(0) == b"ok"
    assert lib.afno_status_string(3) == b"workspace too small"


@pytest.mark.parametrize("kw,status", [
    (dict(B=0), binding.AFNO_ERR_INVALID_ARG),
    (dict(C=770), binding.AFNO_ERR_INVALID_ARG),          # C % num_blocks != 0
    (dict(hidden_factor=0), binding.AFNO_ERR_INVALID_ARG),
    (dict(lam=-0.1), binding.AFNO_ERR_INVALID_ARG),
    (dict(lam=float("nan")), binding.AFNO_ERR_INVALID_ARG),
    (dict(kept_fraction=0.0), binding.AFNO_ERR_INVALID_ARG),
    (dict(kept_fraction=1.5), binding.AFNO_ERR_INVALID_ARG),
    (dict(dtype=7), binding.AFNO_ERR_INVALID_ARG),
    (dict(flags=1 << 20), binding.AFNO_ERR_INVALID_ARG),
    (dict(W=181), binding.AFNO_ERR_UNSUPPORTED),           # odd W
    (dict(H=14), binding.AFNO_ERR_UNSUPPORTED),            # prime factor 7
    (dict(W=2 * 11), binding.AFNO_ERR_UNSUPPORTED),
])
def test_descriptor_validation(lib, kw, status):
    base = dict(B=1, H=90, W=180, C=768, num_blocks=8)
    d = binding.Desc(**{**base, **kw})
    cd = d.c()
    assert lib.afno_plan_warmup(ctypes.byref(cd)) == status   # fails before any CUDA call
    assert lib.afno_last_error() != b""
    assert binding.afno_spectral_workspace_bytes(d, False) == 0
    assert binding.afno_spectral_path(d) is None


def test_null_pointers_rejected_before_any_cuda_call(lib):
    d = binding.Desc(1, 8, 16, 16, 2, dtype=binding.AFNO_F32).c()
    rc = lib.afno_spectral_fwd(ctypes.byref(d), None, None, None, None, None, None, None, 0, None)
    assert rc == binding.AFNO_ERR_INVALID_ARG
    rc = lib.afno_spectral_fwd(None, None, None, None, None, None, None, None, 0, None)
    assert rc == binding.AFNO_ERR_INVALID_ARG


def test_size_queries(lib):
    d = binding.Desc(4, 90, 180, 768, 8)
    fwd = binding.afno_spectral_workspace_bytes(d, False)
    bwd = binding.afno_spectral_workspace_bytes(d, True)
    assert 0 < fwd < bwd
    m1, off2, m2 = binding.afno_spectral_mask_bytes(d)
    assert m1 == 4 * 90 * 91 * 768 * 2 and m2 == m1 and off2 % 256 == 0 and off2 >= m1
    dm = binding.Desc(4, 90, 180, 768, 8, flags=binding.FLAG_EXPORT_MASKS)
    assert binding.afno_spectral_workspace_bytes(dm, True) >= bwd + m1 + m2
    assert binding.afno_spectral_host_arena_bytes(d, True) > bwd
    # truncation shrinks the stored spectra
    dh = binding.Desc(4, 90, 180, 768, 8, kept_fraction=0.5)
    assert binding.afno_spectral_workspace_bytes(dh, False) < fwd


def test_missing_library_fails_loudly(monkeypatch):
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", "/nonexistent/libafno_b200.so")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.lib()
