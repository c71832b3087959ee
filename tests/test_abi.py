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


def _sass_opcodes(obj, kernel):
    """{opcode: count} of one kernel of an object file (cuobjdump -sass -fun)."""
    import subprocess
    out = subprocess.run(["cuobjdump", "-sass", "-fun", kernel, obj], capture_output=True, text=True).stdout
    ops = {}
    for line in out.splitlines():
        m = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P[0-9T]+\s+)?([A-Z0-9_.]+)", line)
        if m:
            ops[m.group(1)] = ops.get(m.group(1), 0) + 1
    return ops


def test_sass_is_sm100a_and_uses_async_copies(libpath):
    """What DESIGN.md §6.1 says about the half-sweep kernel, read off its SASS: sm_100a code; the gather is cp.async
    (LDGSTS) with 16-byte accesses, one per chunk of the 2d links; nothing spills to local memory in the
    overrelaxation instantiations; programmatic dependent launch is there (griddepcontrol.launch_dependents = PREEXIT,
    griddepcontrol.wait = ACQBULK); results leave with 16-byte stores.  (profiles/r02_sass_census.md keeps the counts.)"""
    import shutil
    import subprocess
    if not shutil.which("cuobjdump"):
        pytest.skip("cuobjdump not available")
    out = subprocess.run(["cuobjdump", "-lelf", libpath], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    build_dir = os.path.join(os.path.dirname(libpath), "build")
    # Landau overrelaxation, no tracked transform, no fused partials: <R, A, RECON, GAUGE = 0, STOCH = 0, TRACK = 0, RED = 0>
    cases = {"sweep_dp18.o": ("_ZN2gf12sweep_kernelIddLi18ELi0ELb0ELb0ELb0EEEvNS_9SweepArgsE", 8 * 9),
             "sweep_dp12.o": ("_ZN2gf12sweep_kernelIddLi12ELi0ELb0ELb0ELb0EEEvNS_9SweepArgsE", 8 * 6),
             "sweep_sp12.o": ("_ZN2gf12sweep_kernelIffLi12ELi0ELb0ELb0ELb0EEEvNS_9SweepArgsE", 8 * 3),
             "sweep_mp12.o": ("_ZN2gf12sweep_kernelIfdLi12ELi0ELb0ELb0ELb0EEEvNS_9SweepArgsE", 8 * 3)}
    for obj, (kern, n_chunks) in cases.items():
        ops = _sass_opcodes(os.path.join(build_dir, obj), kern)
        assert ops, (obj, "kernel not found")
        ldgsts = sum(n for o, n in ops.items() if o.startswith("LDGSTS"))
        assert ldgsts == n_chunks and ops.get("LDGSTS.E.BYPASS.128", 0) == n_chunks, (obj, ldgsts)
        assert not any(o.startswith(("LDL", "STL")) for o in ops), (obj, [o for o in ops if o.startswith(("LDL", "STL"))])
        assert ops.get("PREEXIT", 0) == 1 and ops.get("ACQBULK", 0) == 1, obj
        assert any(o.startswith("STG.E.128") for o in ops), obj
        assert not any(o.startswith(("HMMA", "UTC", "HGMMA")) for o in ops)      # no tensor-core path: a 3x3 stencil
