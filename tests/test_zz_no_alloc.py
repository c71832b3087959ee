"""gf_unitarity_noalloc (include/gf.h): the unitarity measure of Eq. (33) for callers that cannot allocate.

gf_unitarity needs a context — a second copy of the configuration on the GPU — and takes and frees scratch memory with
cudaMalloc / cudaFree on every call.  A lattice code whose fields already fill the GPU, code inside a memory pool with a
fixed budget, or a check that must not stall other streams (cudaFree waits for the device) cannot use it.
gf_unitarity_noalloc reads the caller's own device buffer, writes the caller's two result doubles, and keeps its partial
sums in a fixed 2 MiB array of the library that all calls share.

What is checked here, against the existing path (a context + gf_unitarity) and within the tolerance
test_unitarity_measure_matches_numpy uses (1e-12, plus 1e-6 for float links):
  * two calls in a row that share the array: a buffer spanning several CTAs with a ragged tail, then a smaller one
    (the first call's partial sums stay behind in the array and must not leak), then the first again, bit for bit;
  * float and double buffers;
  * sizes beyond the stated maximum and other bad arguments are refused with a message, before the device is touched
    (this part needs no GPU).

The file sorts last on purpose: `pytest -x` stops at the first failure, and this test should never hide another one.
It makes no assumption about what ran before it in the process (the first call on a device looks up the array's
address itself), so it passes alone and after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest

from paper_1212_5221_b200 import inputs

SP, DP = 0, 1


def _off_group_links(dims, seed, dtype):
    """[t,x,y,z,mu,3,3,2] reals: SU(3) links pushed off the group link by link, so that |1 - det U| ~ 3e-3."""
    rng = np.random.default_rng(seed)
    U = inputs.make_config(*dims, 0.5, seed, seed + 1)
    U = U * (1 + 1e-3 * rng.standard_normal(U.shape[:-2] + (1, 1)))
    return inputs.as_real(U, dtype)


@pytest.mark.gpu
@pytest.mark.parametrize("prec", [DP, SP])
def test_noalloc_equals_the_context_path_on_consecutive_calls(prec):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1212_5221_b200 import gf
    dt = np.float64 if prec == DP else np.float32
    tol = 1e-12 + 1e-6 * (prec == SP)
    cases = [(6, 6, 6, 8), (4, 6, 4, 4)]          # 6912 links = 3 CTAs + a tail of 768; then 1536 links < one CTA
    host = [_off_group_links(d, 31 + k, dt) for k, d in enumerate(cases)]

    # the existing path: a context per lattice, gf_unitarity
    want = []
    for d, L in zip(cases, host):
        with gf.GaugeFixer(*d, precision=prec) as fx:
            fx.set_links(L)
            avg, mx = fx.unitarity()
        want.append((avg[0], mx[0]))
        assert mx[0] > 1e-4                       # the measurement is not trivially zero

    # the caller's side of the new entry point: its buffers exist before the calls, the calls create nothing
    dev = [torch.from_numpy(L).cuda() for L in host]
    res = [torch.full((2,), -1.0, dtype=torch.float64, device="cuda") for _ in range(3)]
    torch.cuda.synchronize()
    mem0 = torch.cuda.memory_allocated()
    gf.gf_unitarity_noalloc(dev[0], res[0])       # large
    gf.gf_unitarity_noalloc(dev[1], res[1])       # small, right behind it on the same stream, same scratch array
    gf.gf_unitarity_noalloc(dev[0], res[2])       # large again
    torch.cuda.synchronize()
    got = [r.cpu().numpy() for r in res]
    for k, (a, m) in enumerate(want):
        assert abs(got[k][0] - a) <= tol and abs(got[k][1] - m) <= tol, (k, got[k], a, m)
    assert got[2][0] == got[0][0] and got[2][1] == got[0][1]          # fixed summation order: bit for bit
    assert torch.cuda.memory_allocated() == mem0
    # after the first call on this device (which may load the kernels) further calls leave free memory untouched
    free1 = torch.cuda.mem_get_info()[0]
    gf.gf_unitarity_noalloc(dev[1], res[1])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free1

    # an empty buffer is a valid input: both numbers 0
    gf.gf_unitarity_noalloc(dev[0][:0], res[1])
    torch.cuda.synchronize()
    assert res[1].cpu().tolist() == [0.0, 0.0]


def test_noalloc_refuses_what_it_cannot_hold():
    """Argument checks come before any CUDA call, so they can be exercised without a GPU; the pointers are never read."""
    from paper_1212_5221_b200 import gf
    lib, fake = gf._lib, ctypes.c_void_p(4096)
    err = ctypes.create_string_buffer(512)
    nmax = gf.GF_UNITARITY_NOALLOC_MAX_LINKS
    assert nmax == 4 * 64 * 64 * 64 * 256         # the paper's largest lattice still fits
    assert lib.gf_unitarity_noalloc(fake, 8, nmax + 1, fake, None, err, 512) == gf.GF_EINVAL
    msg = err.value.decode()
    assert "GF_UNITARITY_NOALLOC_MAX_LINKS" in msg and str(nmax + 1) in msg and str(nmax) in msg
    assert lib.gf_unitarity_noalloc(fake, 2, 10, fake, None, err, 512) == gf.GF_EINVAL and b"elem_bytes" in err.value
    assert lib.gf_unitarity_noalloc(fake, 8, -1, fake, None, err, 512) == gf.GF_EINVAL
    assert lib.gf_unitarity_noalloc(fake, 8, 10, None, None, err, 512) == gf.GF_EINVAL and b"result_device" in err.value
    assert lib.gf_unitarity_noalloc(None, 8, 10, fake, None, err, 512) == gf.GF_EINVAL
    assert lib.gf_unitarity_noalloc(ctypes.c_void_p(4104), 8, 10, fake, None, err, 512) == gf.GF_EINVAL and b"aligned" in err.value
    assert lib.gf_unitarity_noalloc(fake, 8, nmax + 1, fake, None, None, 0) == gf.GF_EINVAL      # no message buffer: still refused


def test_noalloc_object_references_no_allocating_runtime_call():
    """The translation unit of the entry point, read with nm: the only CUDA runtime calls it can reach are the device
    query, the symbol-address lookup, kernel launches and error strings — no cudaMalloc*, cudaFree*, cudaHostAlloc,
    no memcpy (which may stage through driver memory), no stream or event creation."""
    import os
    import shutil
    import subprocess
    from paper_1212_5221_b200 import build
    build.build()
    obj = os.path.join(build.OBJ, "unitarity_noalloc.o")
    if not shutil.which("nm") or not os.path.exists(obj):
        pytest.skip("nm or the object file is not available")
    out = subprocess.run(["nm", "-u", obj], capture_output=True, text=True, check=True).stdout
    cuda_calls = sorted(w for w in out.split() if w.startswith("cuda"))
    assert cuda_calls == ["cudaGetDevice", "cudaGetErrorString", "cudaGetLastError", "cudaGetSymbolAddress",
                          "cudaLaunchKernel"], cuda_calls
