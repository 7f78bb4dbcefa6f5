"""CPU-side checks of the C-ABI library: it builds, loads without a GPU, exports every symbol that
include/amp.h declares, and fails loudly (no CPU fallback) when no device is present."""
import ctypes as C
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "amp.h")


def header_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(amp_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2007_14931_b200 import build
    return build.build()


def test_header_declares_the_north_star_calls():
    syms = header_symbols()
    for need in ("amp_model_create", "amp_load_events", "amp_load_norm", "amp_set_params", "amp_nll"):
        assert need in syms


def test_library_exports_every_declared_symbol(libpath):
    out = subprocess.run(["nm", "-D", "--defined-only", libpath], capture_output=True, text=True, check=True).stdout
    exported = set(re.findall(r" T (amp_[a-z0-9_]+)", out))
    for s in header_symbols():
        assert s in exported, f"{s} declared in amp.h but not exported"


def test_binding_covers_header(libpath):
    from paper_2007_14931_b200 import binding
    assert sorted(binding.SYMBOLS) == header_symbols()
    L = binding.lib()
    for s in binding.SYMBOLS:
        assert hasattr(L, s)
    assert b"sm_100a" in L.amp_version()
    assert L.amp_status_string(3) == b"AMP_ERR_DOMAIN"
    assert L.amp_cache_column_name(0) == b"m2" and L.amp_cache_column_name(99) is None


def test_sass_is_sm_100a(libpath):
    out = subprocess.run(["cuobjdump", "-lelf", libpath], capture_output=True, text=True)
    if out.returncode != 0:
        pytest.skip("cuobjdump unavailable")
    assert "sm_100a" in out.stdout


def test_argument_validation_without_device(libpath):
    from paper_2007_14931_b200 import binding as B
    L = B.lib()
    h = C.c_void_p()
    dec = B.amp_decay(5279.65, 3096.9, 493.677, 139.570)
    res = (B.amp_resonance * 1)(B.amp_resonance(B.AMP_KSTAR, 7, 895.55, 47.3, 1.6e-3))     # J out of range
    assert L.amp_model_create(C.byref(dec), res, 1, C.byref(h)) == B.AMP_ERR_INVALID
    res = (B.amp_resonance * 1)(B.amp_resonance(B.AMP_KSTAR, 1, 2500.0, 47.3, 1.6e-3))     # pole above m_B - m_psi
    assert L.amp_model_create(C.byref(dec), res, 1, C.byref(h)) == B.AMP_ERR_DOMAIN
    assert L.amp_model_create(None, res, 1, C.byref(h)) == B.AMP_ERR_INVALID
    assert L.amp_num_couplings(None) == -1
    assert L.amp_nll(None, None, None) == B.AMP_ERR_INVALID


def test_no_cpu_fallback(libpath):
    """Without a CUDA device model creation must fail with AMP_ERR_CUDA — the product never computes on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    from paper_2007_14931_b200 import binding as B
    with pytest.raises(B.AmpError) as e:
        B.Model((5279.65, 3096.9, 493.677, 139.570), [(B.AMP_KSTAR, 1, 895.55, 47.3, 1.6e-3)])
    assert e.value.status == B.AMP_ERR_CUDA


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2007_14931_b200")
    for dirpath, _dirs, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "liboracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2007_14931_b200" not in text.replace("paper_2007_14931_b200/csrc", ""), f
