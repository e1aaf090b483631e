"""CPU checks of the C-ABI library: it builds for sm_100a, loads, and exports every symbol include/sph.h declares.
No compute calls are made here (there is no GPU on the build box)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "sph.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sph_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = _declared_symbols()
    for need in ("sph_build_cells", "sph_neighbors", "sph_density", "sph_rhs", "sph_rhs_vjp", "sph_rk_step"):
        assert need in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2507_21684_b200 import build
    path = build.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    for name in _declared_symbols():
        assert hasattr(lib, name), f"{name} declared in include/sph.h but not exported"
    lib.sph_strerror.restype = ctypes.c_char_p
    assert lib.sph_strerror(0) == b"ok"
    assert b"no CPU fallback" in lib.sph_strerror(-5)


def test_binding_lists_the_same_symbols():
    from paper_2507_21684_b200 import binding
    assert sorted(binding.EXPORTS) == _declared_symbols()


def test_product_does_not_touch_the_oracle():
    """The CUDA package must not import, read or link anything under oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_2507_21684_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "liboracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2507_21684_b200" not in txt.replace("paper_2507_21684_b200/csrc/", ""), f
            assert "libsph_b200" not in txt, f


def test_no_cuda_device_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2507_21684_b200 import binding
    with pytest.raises(RuntimeError):
        binding.Sph(0)
