"""CPU-side checks of the boundary: libgf.so builds, loads and exports every symbol that
include/gf.h declares; without a CUDA device the product path fails loudly (no CPU fallback)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_1212_5221_b200 import build
    return build.build()


def declared_functions():
    text = open(os.path.join(ROOT, "include", "gf.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gf_[a-z_0-9]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = declared_functions()
    for n in ("gf_create", "gf_set_links", "gf_sweep", "gf_run", "gf_reunitarize", "gf_get_links",
              "gf_get_gauge_transform"):
        assert n in names


def test_library_exports_every_declared_symbol(libpath):
    lib = ctypes.CDLL(libpath)
    for n in declared_functions():
        assert hasattr(lib, n), n


def test_binding_mirrors_the_header(libpath):
    from paper_1212_5221_b200 import gf
    assert sorted(gf.EXPORTS) == declared_functions()
    for n in gf.EXPORTS:
        assert callable(getattr(gf, n)), n
    assert "sm_100a" in gf.gf_version()


def test_fails_loudly_without_a_gpu(libpath):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_1212_5221_b200 import gf
    with pytest.raises(gf.GfError) as e:
        gf.gf_create(4, 4, 4, 4, gf.GF_DP)
    assert e.value.code == gf.GF_ECUDA


def test_bad_extents_rejected_before_touching_the_device(libpath):
    lib = ctypes.CDLL(libpath)
    h = ctypes.c_void_p()
    assert lib.gf_create(ctypes.byref(h), 3, 4, 4, 4, 1, 18, 0, None) == -1
    assert lib.gf_create(ctypes.byref(h), 4, 4, 4, 4, 1, 17, 0, None) == -1
    assert lib.gf_create(None, 4, 4, 4, 4, 1, 18, 0, None) == -1


def test_sass_is_sm100a_and_uses_async_copies(libpath):
    import shutil
    import subprocess
    if not shutil.which("cuobjdump"):
        pytest.skip("cuobjdump not available")
    out = subprocess.run(["cuobjdump", "-lelf", libpath], capture_output=True, text=True).stdout
    assert "sm_100a" in out
