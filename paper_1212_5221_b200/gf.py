"""Thin Python binding of libgf.so (include/gf.h): argument marshalling only.

Every function has the name and the argument order of the C entry point it forwards to; all
arithmetic of the method runs in the CUDA kernels behind the ABI.  Buffers may be NumPy arrays
(host), CPU torch tensors (host, pinned or not) or CUDA torch tensors (device); PyTorch is used for
device memory and streams only.  The library is loaded at import and the import fails loudly if
``libgf.so`` has not been built (``python -m paper_1212_5221_b200.build``): there is no fallback.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgf.so")

if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1212_5221_b200.build` "
                      "(nvcc, sm_100a). There is no CPU fallback.")
_lib = ctypes.CDLL(LIB_PATH)

# constants of include/gf.h
GF_OK, GF_NOT_CONVERGED, GF_EINVAL, GF_ENOMEM, GF_ECUDA, GF_ESTATE = 0, 1, -1, -2, -3, -4
GF_SP, GF_DP, GF_MP = 0, 1, 2
GF_LANDAU, GF_COULOMB, GF_MAG = 0, 1, 2
GF_OR, GF_SR, GF_SA, GF_MICRO = 0, 1, 2, 3
GF_FLAG_TRACK_TRANSFORM = 1
GF_FLAG_FREEZE_SLICES = 2
GF_FLAG_SU2 = 4
GF_FLAG_LAGGED_STOP = 8
GF_UNITARITY_NOALLOC_MAX_LINKS = 1 << 28

EXPORTS = ["gf_create", "gf_num_colors", "gf_create_batch", "gf_num_copies", "gf_set_links_copy", "gf_get_links_copy",
           "gf_get_gauge_transform_copy", "gf_measure_batch", "gf_measure_mag_eq16", "gf_run_batch", "gf_fix", "gf_random_gauge", "gf_wilson_heatbath", "gf_plaquette", "gf_unitarity", "gf_unitarity_noalloc", "gf_destroy", "gf_set_links", "gf_get_links", "gf_get_gauge_transform", "gf_sweep",
           "gf_half_sweep", "gf_measure", "gf_run", "gf_get_slice_sweeps", "gf_anneal", "gf_reunitarize", "gf_coulomb_finalize",
           "gf_sync", "gf_kernel_timing", "gf_kernel_time_ms", "gf_launch_count", "gf_device_bytes", "gf_volume", "gf_last_error", "gf_version",
           "gf_create_shard", "gf_shard_attach", "gf_shard_export", "gf_shard_attach_ipc", "gf_shard_set_comm", "gf_shard_info",
           "gf_debug_set_fused", "gf_debug_set_pdl", "gf_debug_set_block"]


class gf_result(ctypes.Structure):
    _fields_ = [("sweeps", ctypes.c_int), ("F", ctypes.c_double), ("theta", ctypes.c_double)]


class gf_fix_params(ctypes.Structure):
    _fields_ = [("gauge", ctypes.c_int), ("seed", ctypes.c_uint64), ("sa_steps", ctypes.c_int),
                ("sa_T_hi", ctypes.c_double), ("sa_T_lo", ctypes.c_double), ("sa_micro", ctypes.c_int),
                ("sr_max_sweeps", ctypes.c_int), ("sr_p", ctypes.c_double), ("or_omega", ctypes.c_double),
                ("or_max_sweeps", ctypes.c_int), ("eps", ctypes.c_double), ("check_every", ctypes.c_int),
                ("reunit_every", ctypes.c_int)]


class gf_shard_handle(ctypes.Structure):
    _fields_ = [("links", ctypes.c_ubyte * 64), ("gtot", ctypes.c_ubyte * 64), ("gapplied", ctypes.c_ubyte * 64),
                ("t0", ctypes.c_int), ("Nt_local", ctypes.c_int), ("has_transform", ctypes.c_int),
                ("Nx", ctypes.c_int), ("Ny", ctypes.c_int), ("Nz", ctypes.c_int), ("Nt_global", ctypes.c_int),
                ("precision", ctypes.c_int), ("recon", ctypes.c_int)]


GF_BARRIER_FN = ctypes.CFUNCTYPE(None, ctypes.c_void_p)
GF_ALLREDUCE_FN = ctypes.CFUNCTYPE(None, ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.c_int)


class gf_comm(ctypes.Structure):
    _fields_ = [("barrier", GF_BARRIER_FN), ("allreduce_sum", GF_ALLREDUCE_FN), ("user", ctypes.c_void_p)]


_vp, _ci, _cd, _u64, _u32 = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_uint64, ctypes.c_uint32
_lib.gf_create_shard.argtypes = [ctypes.POINTER(_vp), _ci, _ci, _ci, _ci, _ci, _ci, _ci, _ci, ctypes.c_uint, _vp]
_lib.gf_shard_attach.argtypes = [_vp, _vp, _vp]
_lib.gf_shard_export.argtypes = [_vp, ctypes.POINTER(gf_shard_handle)]
_lib.gf_shard_attach_ipc.argtypes = [_vp, ctypes.POINTER(gf_shard_handle), ctypes.POINTER(gf_shard_handle)]
_lib.gf_shard_set_comm.argtypes = [_vp, ctypes.POINTER(gf_comm)]
_lib.gf_shard_info.argtypes = [_vp, ctypes.POINTER(_ci), ctypes.POINTER(_ci), ctypes.POINTER(_ci)]
_lib.gf_create_batch.argtypes = [ctypes.POINTER(_vp), _ci, _ci, _ci, _ci, _ci, _ci, _ci, ctypes.c_uint, _vp]
_lib.gf_num_copies.argtypes = [_vp]
_lib.gf_num_colors.argtypes = [_vp]
_lib.gf_set_links_copy.argtypes = [_vp, _ci, _vp, _ci, _ci]
_lib.gf_get_links_copy.argtypes = [_vp, _ci, _vp, _ci, _ci]
_lib.gf_get_gauge_transform_copy.argtypes = [_vp, _ci, _vp, _ci, _ci]
_lib.gf_measure_batch.argtypes = [_vp, _ci, _vp, _vp, _vp]
_lib.gf_measure_mag_eq16.argtypes = [_vp, _vp]
_lib.gf_run_batch.argtypes = [_vp, _ci, _ci, _cd, _u64, _u32, _ci, _cd, _ci, _ci, _vp, _vp]
_lib.gf_fix.argtypes = [_vp, ctypes.POINTER(gf_fix_params), _vp]
_lib.gf_random_gauge.argtypes = [_vp, _u64]
_lib.gf_wilson_heatbath.argtypes = [_vp, _cd, _u64, _u32, _ci]
_lib.gf_plaquette.argtypes = [_vp, _vp]
_lib.gf_unitarity.argtypes = [_vp, _vp, _vp]
_lib.gf_unitarity_noalloc.argtypes = [_vp, _ci, ctypes.c_int64, _vp, _vp, ctypes.c_char_p, _ci]
_lib.gf_create.argtypes = [ctypes.POINTER(_vp), _ci, _ci, _ci, _ci, _ci, _ci, ctypes.c_uint, _vp]
_lib.gf_destroy.argtypes = [_vp]
_lib.gf_set_links.argtypes = [_vp, _vp, _ci, _ci]
_lib.gf_get_links.argtypes = [_vp, _vp, _ci, _ci]
_lib.gf_get_gauge_transform.argtypes = [_vp, _vp, _ci, _ci]
_lib.gf_sweep.argtypes = [_vp, _ci, _ci, _cd, _u64, _u32]
_lib.gf_half_sweep.argtypes = [_vp, _ci, _ci, _cd, _u64, _u32, _ci]
_lib.gf_measure.argtypes = [_vp, _ci, ctypes.POINTER(_cd), ctypes.POINTER(_cd), _vp]
_lib.gf_run.argtypes = [_vp, _ci, _ci, _cd, _u64, _u32, _ci, _cd, _ci, _ci, ctypes.POINTER(gf_result), _vp]
_lib.gf_get_slice_sweeps.argtypes = [_vp, _vp]
_lib.gf_anneal.argtypes = [_vp, _ci, _cd, _cd, _ci, _ci, _u64, _u32, ctypes.POINTER(_u32)]
_lib.gf_reunitarize.argtypes = [_vp]
_lib.gf_coulomb_finalize.argtypes = [_vp]
_lib.gf_sync.argtypes = [_vp]
_lib.gf_kernel_timing.argtypes = [_vp, _ci]
_lib.gf_kernel_time_ms.argtypes = [_vp, ctypes.POINTER(_cd), ctypes.POINTER(_ci), _ci]
_lib.gf_launch_count.argtypes = [_vp, ctypes.POINTER(ctypes.c_int64), _ci]
_lib.gf_device_bytes.argtypes = [_vp]
_lib.gf_device_bytes.restype = ctypes.c_int64
_lib.gf_volume.argtypes = [_vp]
_lib.gf_volume.restype = ctypes.c_int64
_lib.gf_last_error.argtypes = [_vp]
_lib.gf_last_error.restype = ctypes.c_char_p
_lib.gf_version.restype = ctypes.c_char_p
_lib.gf_debug_set_block.argtypes = [_vp, _ci]
_lib.gf_debug_set_fused.argtypes = [_vp, _ci]
_lib.gf_debug_set_pdl.argtypes = [_vp, _ci]


class GfError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libgf error {code}: {msg}")
        self.code = code


def _check(ctx, rc, ok=(GF_OK,)):
    if rc not in ok:
        msg = _lib.gf_last_error(ctx).decode() if ctx else "invalid arguments or no CUDA device"
        raise GfError(rc, msg)
    return rc


def _buffer(a):
    """(pointer, elem_bytes, is_device, n_elements) of a NumPy array or torch tensor."""
    if isinstance(a, np.ndarray):
        if not a.flags.c_contiguous:
            raise ValueError("array must be C-contiguous")
        if a.dtype not in (np.float32, np.float64):
            raise TypeError(a.dtype)
        return a.ctypes.data, a.dtype.itemsize, 0, a.size
    import torch
    if isinstance(a, torch.Tensor):
        if not a.is_contiguous():
            raise ValueError("tensor must be contiguous")
        if a.dtype not in (torch.float32, torch.float64):
            raise TypeError(a.dtype)
        return a.data_ptr(), a.element_size(), 1 if a.is_cuda else 0, a.numel()
    raise TypeError(type(a))


def gf_version() -> str:
    return _lib.gf_version().decode()


def _stream_handle(cuda_stream):
    if cuda_stream is None:
        try:
            import torch
            cuda_stream = torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else 0
        except ImportError:
            cuda_stream = 0
    elif hasattr(cuda_stream, "cuda_stream"):
        cuda_stream = cuda_stream.cuda_stream
    return cuda_stream


def gf_create(Nx, Ny, Nz, Nt, precision, recon=18, flags=0, cuda_stream=None):
    """-> opaque context handle.  cuda_stream: None (torch's current stream if torch has CUDA,
    else the default stream), an int cudaStream_t, or a torch.cuda.Stream."""
    h = _vp()
    rc = _lib.gf_create(ctypes.byref(h), Nx, Ny, Nz, Nt, precision, recon, flags, _vp(_stream_handle(cuda_stream)))
    _check(None, rc)
    return h


def gf_create_batch(Nx, Ny, Nz, Nt, n_copies, precision, recon=18, flags=0, cuda_stream=None):
    h = _vp()
    rc = _lib.gf_create_batch(ctypes.byref(h), Nx, Ny, Nz, Nt, n_copies, precision, recon, flags,
                              _vp(_stream_handle(cuda_stream)))
    _check(None, rc)
    return h


def gf_create_shard(Nx, Ny, Nz, Nt_local, t0, Nt_global, precision, recon=18, flags=0, cuda_stream=None):
    """-> context holding the time-slices [t0, t0 + Nt_local) of an Nx*Ny*Nz*Nt_global lattice (gf.h, "t-shards")."""
    h = _vp()
    rc = _lib.gf_create_shard(ctypes.byref(h), Nx, Ny, Nz, Nt_local, t0, Nt_global, precision, recon, flags,
                              _vp(_stream_handle(cuda_stream)))
    _check(None, rc)
    return h


def gf_shard_attach(ctx, below, above):
    return _check(ctx, _lib.gf_shard_attach(ctx, below, above))


def gf_shard_export(ctx) -> gf_shard_handle:
    h = gf_shard_handle()
    _check(ctx, _lib.gf_shard_export(ctx, ctypes.byref(h)))
    return h


def gf_shard_attach_ipc(ctx, below: gf_shard_handle, above: gf_shard_handle):
    return _check(ctx, _lib.gf_shard_attach_ipc(ctx, ctypes.byref(below), ctypes.byref(above)))


def gf_shard_set_comm(ctx, comm):
    """comm: a gf_comm (the caller keeps it, and the callables it was built from, alive) or None."""
    return _check(ctx, _lib.gf_shard_set_comm(ctx, ctypes.byref(comm) if comm is not None else None))


def gf_shard_info(ctx):
    """-> (t0, Nt_local, Nt_global)"""
    a, b, c = _ci(), _ci(), _ci()
    _check(ctx, _lib.gf_shard_info(ctx, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)))
    return a.value, b.value, c.value


def gf_num_copies(ctx):
    return int(_lib.gf_num_copies(ctx))


def gf_num_colors(ctx):
    return int(_lib.gf_num_colors(ctx))


def gf_destroy(ctx):
    return _lib.gf_destroy(ctx)


def _sized(ctx, n, per_site, what):
    """per_site is given for SU(3) (72 reals of links, 18 of a transform); SU(2) matrices hold 8 reals."""
    if gf_num_colors(ctx) == 2:
        per_site = per_site * 8 // 18
    want = gf_volume(ctx) * per_site
    if n != want:
        raise ValueError(f"{what}: buffer holds {n} reals, the context's lattice needs {want}")


def gf_set_links(ctx, links):
    p, eb, dev, n = _buffer(links)
    _sized(ctx, n, 72, "gf_set_links")
    return _check(ctx, _lib.gf_set_links(ctx, _vp(p), eb, dev))


def gf_get_links(ctx, out):
    p, eb, dev, n = _buffer(out)
    _sized(ctx, n, 72, "gf_get_links")
    return _check(ctx, _lib.gf_get_links(ctx, _vp(p), eb, dev))


def gf_get_gauge_transform(ctx, out):
    p, eb, dev, n = _buffer(out)
    _sized(ctx, n, 18, "gf_get_gauge_transform")
    return _check(ctx, _lib.gf_get_gauge_transform(ctx, _vp(p), eb, dev))


def gf_set_links_copy(ctx, copy, links):
    p, eb, dev, n = _buffer(links)
    _sized(ctx, n, 72, "gf_set_links_copy")
    return _check(ctx, _lib.gf_set_links_copy(ctx, copy, _vp(p), eb, dev))


def gf_get_links_copy(ctx, copy, out):
    p, eb, dev, n = _buffer(out)
    _sized(ctx, n, 72, "gf_get_links_copy")
    return _check(ctx, _lib.gf_get_links_copy(ctx, copy, _vp(p), eb, dev))


def gf_get_gauge_transform_copy(ctx, copy, out):
    p, eb, dev, n = _buffer(out)
    _sized(ctx, n, 18, "gf_get_gauge_transform_copy")
    return _check(ctx, _lib.gf_get_gauge_transform_copy(ctx, copy, _vp(p), eb, dev))


def gf_measure_batch(ctx, gauge, Nt=None):
    """-> (F[n_copies], theta[n_copies]) or, with Nt given (any true value), (F, theta, theta_slice[n_copies, Nt_global]).
    The library writes Nt_global entries per copy — on a t-shard more than the shard's own slices — so the buffer is
    sized from gf_shard_info, never from the caller's number."""
    B = gf_num_copies(ctx)
    F, th = np.zeros(B), np.zeros(B)
    if Nt:
        Nt = gf_shard_info(ctx)[2]
    ts = np.zeros((B, Nt)) if Nt else None
    _check(ctx, _lib.gf_measure_batch(ctx, gauge, _vp(F.ctypes.data), _vp(th.ctypes.data),
                                      _vp(ts.ctypes.data) if Nt else None))
    return (F, th, ts) if Nt else (F, th)


def gf_measure_mag_eq16(ctx):
    """-> theta[n_copies] of Eq. (16) as printed (sum over the subgroups inside the modulus); gf.h."""
    th = np.zeros(gf_num_copies(ctx))
    _check(ctx, _lib.gf_measure_mag_eq16(ctx, _vp(th.ctypes.data)))
    return th


def gf_run_batch(ctx, gauge, algo, param, seed=0, first_sweep_index=0, max_sweeps=1000, eps=1e-12, check_every=1,
                 reunit_every=0, history=False):
    """-> list of dict(sweeps, F, theta, converged[, history]) per copy."""
    B = gf_num_copies(ctx)
    res = (gf_result * B)()
    nchk = max_sweeps // check_every + 1
    hist = np.zeros((nchk, B, 3)) if history else None
    rc = _lib.gf_run_batch(ctx, gauge, algo, float(param), seed, first_sweep_index, max_sweeps, float(eps),
                           check_every, reunit_every, ctypes.cast(res, _vp), _vp(hist.ctypes.data) if history else None)
    _check(ctx, rc, ok=(GF_OK, GF_NOT_CONVERGED))
    out = []
    for c in range(B):
        d = {"sweeps": res[c].sweeps, "F": res[c].F, "theta": res[c].theta, "converged": res[c].theta < eps}
        if history:
            n = int(np.count_nonzero(hist[:, c, 0]))
            d["history"] = hist[:n, c]
        out.append(d)
    return out


def gf_fix(ctx, gauge, seed=0, sa_steps=0, sa_T_hi=1.0, sa_T_lo=0.01, sa_micro=3, sr_max_sweeps=0, sr_p=0.5,
           or_omega=1.7, or_max_sweeps=1000, eps=1e-12, check_every=1, reunit_every=0):
    """SA -> SR -> OR pipeline.  -> list of dict(sweeps, F, theta, converged) per copy."""
    B = gf_num_copies(ctx)
    p = gf_fix_params(gauge, seed, sa_steps, float(sa_T_hi), float(sa_T_lo), sa_micro, sr_max_sweeps, float(sr_p),
                      float(or_omega), or_max_sweeps, float(eps), check_every, reunit_every)
    res = (gf_result * B)()
    rc = _lib.gf_fix(ctx, ctypes.byref(p), ctypes.cast(res, _vp))
    _check(ctx, rc, ok=(GF_OK, GF_NOT_CONVERGED))
    return [{"sweeps": res[c].sweeps, "F": res[c].F, "theta": res[c].theta, "converged": res[c].theta < eps}
            for c in range(B)]


def gf_random_gauge(ctx, seed):
    return _check(ctx, _lib.gf_random_gauge(ctx, seed))


def gf_wilson_heatbath(ctx, beta, seed, first_sweep_index=0, n_sweeps=1):
    return _check(ctx, _lib.gf_wilson_heatbath(ctx, float(beta), seed, first_sweep_index, n_sweeps))


def gf_plaquette(ctx):
    """-> array[n_copies] of <Re tr U_P> / 3."""
    out = np.zeros(gf_num_copies(ctx))
    _check(ctx, _lib.gf_plaquette(ctx, _vp(out.ctypes.data)))
    return out


def gf_unitarity(ctx):
    """-> (avg[n_copies], max[n_copies]) of |1 - det U| (Eq. (33))."""
    B = gf_num_copies(ctx)
    a, m = np.zeros(B), np.zeros(B)
    _check(ctx, _lib.gf_unitarity(ctx, _vp(a.ctypes.data), _vp(m.ctypes.data)))
    return a, m


def gf_unitarity_noalloc(links, result, cuda_stream=None):
    """Eq. (33) on a buffer the caller already has on the GPU, for callers that must not allocate (gf.h,
    gf_unitarity_noalloc: no context, no cudaMalloc / cudaFree inside; scratch is a fixed 2 MiB array of the library).

    links: CUDA tensor, float32 or float64, contiguous, 18 reals per link (any leading shape; numel / 18 links, at most
    GF_UNITARITY_NOALLOC_MAX_LINKS).  result: the caller's CUDA float64 tensor with at least 2 elements; it receives
    (average, maximum) of |1 - det U| once the work enqueued on the stream has run — this wrapper creates no tensor
    and does not synchronise.  Calls on one device must not overlap on the GPU (they share the scratch array); the first
    call on a device should come before any stream capture.  Returns `result`."""
    import torch
    if not (isinstance(links, torch.Tensor) and links.is_cuda and isinstance(result, torch.Tensor) and result.is_cuda):
        raise TypeError("gf_unitarity_noalloc: links and result must be CUDA tensors (device memory owned by the caller)")
    if result.dtype != torch.float64 or result.numel() < 2 or not result.is_contiguous():
        raise TypeError("gf_unitarity_noalloc: result must be a contiguous float64 tensor with at least 2 elements")
    ptr, eb, _, n = _buffer(links)
    if n % 18:
        raise ValueError("gf_unitarity_noalloc: links must hold 18 reals per link")
    err = ctypes.create_string_buffer(512)
    rc = _lib.gf_unitarity_noalloc(_vp(ptr), eb, n // 18, _vp(result.data_ptr()), _vp(_stream_handle(cuda_stream)), err, 512)
    if rc != GF_OK:
        raise GfError(rc, err.value.decode())
    return result


def gf_sweep(ctx, gauge, algo, param, seed=0, sweep_index=0):
    return _check(ctx, _lib.gf_sweep(ctx, gauge, algo, float(param), seed, sweep_index))


def gf_half_sweep(ctx, gauge, algo, param, seed, sweep_index, parity):
    return _check(ctx, _lib.gf_half_sweep(ctx, gauge, algo, float(param), seed, sweep_index, parity))


def gf_measure(ctx, gauge, Nt=None):
    """-> (F, theta) or, with Nt given (any true value), (F, theta, theta_slice[Nt_global]); the buffer is sized from
    gf_shard_info (a t-shard reports every slice of the whole lattice)."""
    F, th = _cd(), _cd()
    if Nt:
        Nt = gf_shard_info(ctx)[2]
    ts = np.zeros(Nt) if Nt else None
    _check(ctx, _lib.gf_measure(ctx, gauge, ctypes.byref(F), ctypes.byref(th), _vp(ts.ctypes.data) if Nt else None))
    return (F.value, th.value, ts) if Nt else (F.value, th.value)


def gf_run(ctx, gauge, algo, param, seed=0, first_sweep_index=0, max_sweeps=1000, eps=1e-12, check_every=1,
           reunit_every=0, history=False):
    """-> dict(sweeps, F, theta, converged[, history = array of (sweep, F, theta)])."""
    res = gf_result()
    hist = np.zeros((max_sweeps // check_every + 1, 3)) if history else None
    rc = _lib.gf_run(ctx, gauge, algo, float(param), seed, first_sweep_index, max_sweeps, float(eps), check_every,
                     reunit_every, ctypes.byref(res), _vp(hist.ctypes.data) if history else None)
    _check(ctx, rc, ok=(GF_OK, GF_NOT_CONVERGED))
    out = {"sweeps": res.sweeps, "F": res.F, "theta": res.theta, "converged": rc == GF_OK}
    if history:
        n = int(np.count_nonzero(hist[:, 0]))
        out["history"] = hist[:n]
    return out


def gf_get_slice_sweeps(ctx, Nt=None):
    """-> int32[n_copies * Nt_global] (the size comes from gf_shard_info; Nt is accepted for older callers and ignored)."""
    out = np.zeros(gf_shard_info(ctx)[2] * gf_num_copies(ctx), dtype=np.int32)
    _check(ctx, _lib.gf_get_slice_sweeps(ctx, _vp(out.ctypes.data)))
    return out


def gf_anneal(ctx, gauge, T_hi, T_lo, n_steps, n_micro, seed, first_sweep_index=0):
    nxt = _u32()
    _check(ctx, _lib.gf_anneal(ctx, gauge, float(T_hi), float(T_lo), n_steps, n_micro, seed, first_sweep_index,
                               ctypes.byref(nxt)))
    return nxt.value


def gf_reunitarize(ctx):
    return _check(ctx, _lib.gf_reunitarize(ctx))


def gf_coulomb_finalize(ctx):
    return _check(ctx, _lib.gf_coulomb_finalize(ctx))


def gf_sync(ctx):
    return _check(ctx, _lib.gf_sync(ctx))


def gf_kernel_timing(ctx, enable):
    return _check(ctx, _lib.gf_kernel_timing(ctx, 1 if enable else 0))


def gf_kernel_time_ms(ctx, reset=True):
    ms, n = _cd(), _ci()
    _check(ctx, _lib.gf_kernel_time_ms(ctx, ctypes.byref(ms), ctypes.byref(n), 1 if reset else 0))
    return ms.value, n.value


def gf_launch_count(ctx, reset=True):
    n = ctypes.c_int64()
    _check(ctx, _lib.gf_launch_count(ctx, ctypes.byref(n), 1 if reset else 0))
    return n.value


def gf_volume(ctx):
    return int(_lib.gf_volume(ctx))


def gf_device_bytes(ctx):
    return int(_lib.gf_device_bytes(ctx))


def gf_last_error(ctx) -> str:
    return _lib.gf_last_error(ctx).decode()


def gf_debug_set_fused(ctx, fused):
    return _check(ctx, _lib.gf_debug_set_fused(ctx, 1 if fused else 0))


def gf_debug_set_pdl(ctx, pdl):
    return _check(ctx, _lib.gf_debug_set_pdl(ctx, 1 if pdl else 0))


def gf_debug_set_block(ctx, block):
    return _check(ctx, _lib.gf_debug_set_block(ctx, block))


class GaugeFixer:
    """Context manager around one gf_ctx.  Methods forward to the C entry points of the same name."""

    def __init__(self, Nx, Ny, Nz, Nt, precision=GF_DP, recon=18, track_transform=False, cuda_stream=None,
                 freeze_slices=False, n_copies=1, su2=False, shard=None, lagged_stop=False):
        """shard = (t0, Nt_global): the context holds the slices [t0, t0 + Nt) of an Nx*Ny*Nz*Nt_global lattice
        (gf_create_shard); buffers of set_links / get_links / get_gauge_transform then are the shard's own slab."""
        self.dims = (Nx, Ny, Nz, Nt)
        self.precision, self.recon, self.n_copies = precision, recon, n_copies
        self.nc = 2 if su2 else 3
        flags = ((GF_FLAG_TRACK_TRANSFORM if track_transform else 0) | (GF_FLAG_FREEZE_SLICES if freeze_slices else 0)
                 | (GF_FLAG_SU2 if su2 else 0) | (GF_FLAG_LAGGED_STOP if lagged_stop else 0))
        self.Nt_global = Nt
        self._comm = None
        if shard is None:
            self.ctx = gf_create_batch(Nx, Ny, Nz, Nt, n_copies, precision, recon, flags, cuda_stream)
        else:
            t0, self.Nt_global = shard
            self.ctx = gf_create_shard(Nx, Ny, Nz, Nt, t0, self.Nt_global, precision, recon, flags, cuda_stream)

    def attach(self, below, above):
        """below / above: the GaugeFixer shards (of this process) that hold the slices below and above this one."""
        return gf_shard_attach(self.ctx, below.ctx, above.ctx)

    def set_comm(self, comm):
        self._comm = comm          # keeps the callbacks alive
        return gf_shard_set_comm(self.ctx, comm)

    def close(self):
        if self.ctx is not None:
            gf_destroy(self.ctx)
            self.ctx = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def shape(self):
        Nx, Ny, Nz, Nt = self.dims
        return (Nt, Nx, Ny, Nz, 4, self.nc, self.nc, 2)

    def set_links(self, links):
        return gf_set_links(self.ctx, links)

    def get_links(self, out=None, dtype=np.float64):
        if out is None:
            out = np.empty(self.shape, dtype=dtype)
        gf_get_links(self.ctx, out)
        return out

    def get_gauge_transform(self, out=None, dtype=np.float64):
        if out is None:
            out = np.empty(self.shape[:4] + self.shape[-3:], dtype=dtype)
        gf_get_gauge_transform(self.ctx, out)
        return out

    def sweep(self, gauge, algo, param, seed=0, sweep_index=0):
        return gf_sweep(self.ctx, gauge, algo, param, seed, sweep_index)

    def half_sweep(self, gauge, algo, param, seed, sweep_index, parity):
        return gf_half_sweep(self.ctx, gauge, algo, param, seed, sweep_index, parity)

    def measure(self, gauge, slices=False):
        return gf_measure(self.ctx, gauge, self.Nt_global if slices else None)

    def run(self, gauge, algo, param, **kw):
        return gf_run(self.ctx, gauge, algo, param, **kw)

    def slice_sweeps(self):
        return gf_get_slice_sweeps(self.ctx, self.Nt_global)

    def anneal(self, gauge, T_hi, T_lo, n_steps, n_micro, seed, first_sweep_index=0):
        return gf_anneal(self.ctx, gauge, T_hi, T_lo, n_steps, n_micro, seed, first_sweep_index)

    def reunitarize(self):
        return gf_reunitarize(self.ctx)

    def coulomb_finalize(self):
        return gf_coulomb_finalize(self.ctx)

    def sync(self):
        return gf_sync(self.ctx)

    # ---- batched gauge copies (gf_create_batch) ----
    def set_links_copy(self, copy, links):
        return gf_set_links_copy(self.ctx, copy, links)

    def get_links_copy(self, copy, out=None, dtype=np.float64):
        if out is None:
            out = np.empty(self.shape, dtype=dtype)
        gf_get_links_copy(self.ctx, copy, out)
        return out

    def get_gauge_transform_copy(self, copy, out=None, dtype=np.float64):
        if out is None:
            out = np.empty(self.shape[:4] + self.shape[-3:], dtype=dtype)
        gf_get_gauge_transform_copy(self.ctx, copy, out)
        return out

    def measure_mag_eq16(self):
        return gf_measure_mag_eq16(self.ctx)

    def measure_batch(self, gauge, slices=False):
        return gf_measure_batch(self.ctx, gauge, self.Nt_global if slices else None)

    def run_batch(self, gauge, algo, param, **kw):
        return gf_run_batch(self.ctx, gauge, algo, param, **kw)

    def fix(self, gauge, **kw):
        return gf_fix(self.ctx, gauge, **kw)

    def random_gauge(self, seed):
        return gf_random_gauge(self.ctx, seed)

    def wilson_heatbath(self, beta, seed, first_sweep_index=0, n_sweeps=1):
        return gf_wilson_heatbath(self.ctx, beta, seed, first_sweep_index, n_sweeps)

    def plaquette(self):
        return gf_plaquette(self.ctx)

    def unitarity(self):
        return gf_unitarity(self.ctx)
