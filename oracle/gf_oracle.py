"""ctypes front end of the CPU ORACLE (oracle/gf_oracle.cpp) — TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this module.  It shares nothing with the CUDA path
(``paper_1212_5221_b200/csrc``) and never imports the package's binding.

All link arrays are the paper's StandardPattern:
``links[t, x, y, z, mu, i, j, (re, im)]`` float32 or float64, C-contiguous, modified in place.
The run loops below (``run``, ``anneal``) are Alg. 1's outer ``while`` and the
simulated-annealing schedule of PAPER.md:243 / 556 written out in plain Python.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gf_oracle.cpp")
_LIB = os.path.join(_HERE, "libgf_oracle.so")

LANDAU, COULOMB, MAG = 0, 1, 2
OR, SR, SA, MICRO = 0, 1, 2, 3


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (-O2, OpenMP).  Building the checker is not using it."""
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(os.path.join(_HERE, "gf_oracle_su2.hpp")),
                 os.path.getmtime(os.path.join(_HERE, "gf_oracle_wilson.hpp")))
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        cmd = ["g++", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c++17",
               "-ffp-contract=off", "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        vp, ci, cd, u64, u32, i64 = (ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_uint64,
                                     ctypes.c_uint32, ctypes.c_int64)
        L.gfo_sweep_d.argtypes = [vp, vp, ci, ci, ci, cd, u64, u32, vp]
        L.gfo_sweep_f.argtypes = [vp, vp, ci, ci, ci, cd, u64, u32, ci, vp]
        L.gfo_measure_d.argtypes = [vp, vp, ci, vp, vp, vp]
        L.gfo_measure_f.argtypes = [vp, vp, ci, vp, vp, vp]
        L.gfo_reunitarize_d.argtypes = [vp, i64]
        L.gfo_reunitarize_f.argtypes = [vp, i64]
        L.gfo_reunitarize_d.restype = None
        L.gfo_reunitarize_f.restype = None
        L.gfo_coulomb_finalize_d.argtypes = [vp, vp, vp]
        L.gfo_coulomb_finalize_f.argtypes = [vp, vp, vp]
        L.gfo_site_update_d.argtypes = [vp, vp, ci, ci, ci, cd, u64, u32, u32, vp]
        L.gfo_site_update_d.restype = None
        L.gfo_site_update_f.argtypes = [vp, vp, ci, ci, ci, cd, u64, u32, u32, ci, vp]
        L.gfo_site_update_f.restype = None
        L.gfo_philox4x32_10.argtypes = [vp, vp, vp]
        L.gfo_philox4x32_10.restype = None
        L.gfo_draw.argtypes = [u64, u32, u32, ci, ci, u32, vp, vp]
        L.gfo_draw.restype = None
        L.gfo_local_quaternion_d.argtypes = [vp, vp, ci, ci, ci, vp]
        L.gfo_local_quaternion_d.restype = None
        L.gfo_local_mag_def_d.argtypes = [vp, vp, ci, ci, ci, vp]
        L.gfo_local_mag_def_d.restype = None
        L.gfo_rule_or_d.argtypes = [vp, cd, vp]
        L.gfo_rule_or_d.restype = None
        L.gfo_rule_micro_d.argtypes = [vp, vp]
        L.gfo_rule_micro_d.restype = None
        L.gfo_rule_heatbath_landau.argtypes = [vp, cd, u64, u32, u32, ci, vp]
        L.gfo_rule_heatbath_landau.restype = None
        L.gfo_rule_heatbath_mag.argtypes = [cd, cd, cd, cd, u64, u32, u32, ci, vp]
        L.gfo_rule_heatbath_mag.restype = None
        L.gfo_apply_subgroup_d.argtypes = [vp, vp, ci, ci, ci]
        L.gfo_apply_subgroup_d.restype = None
        L.gfo_num_threads.restype = ci
        # input generator (gf_oracle_wilson.hpp)
        L.gfo_wilson_heatbath_d.argtypes = [vp, vp, cd, u64, u32]
        L.gfo_wilson_heatbath_f.argtypes = [vp, vp, cd, u64, u32]
        L.gfo_plaquette_d.argtypes = [vp, vp]
        L.gfo_plaquette_d.restype = cd
        L.gfo_plaquette_f.argtypes = [vp, vp]
        L.gfo_plaquette_f.restype = cd
        L.gfo2_wilson_heatbath_d.argtypes = [vp, vp, cd, u64, u32]
        L.gfo2_wilson_heatbath_f.argtypes = [vp, vp, cd, u64, u32]
        L.gfo2_plaquette_d.argtypes = [vp, vp]
        L.gfo2_plaquette_d.restype = cd
        L.gfo2_plaquette_f.argtypes = [vp, vp]
        L.gfo2_plaquette_f.restype = cd
        L.gfo_staple_d.argtypes = [vp, vp, ci, ci, ci, ci, ci, vp]
        L.gfo_staple_d.restype = None
        # N_c = 2 (gf_oracle_su2.hpp)
        L.gfo2_sweep_d.argtypes = [vp, vp, ci, ci, ci, cd, u64, u32, vp]
        L.gfo2_sweep_f.argtypes = [vp, vp, ci, ci, ci, cd, u64, u32, ci, vp]
        L.gfo2_measure_d.argtypes = [vp, vp, ci, vp, vp, vp]
        L.gfo2_measure_f.argtypes = [vp, vp, ci, vp, vp, vp]
        L.gfo2_reunitarize_d.argtypes = [vp, i64]
        L.gfo2_reunitarize_f.argtypes = [vp, i64]
        L.gfo2_reunitarize_d.restype = None
        L.gfo2_reunitarize_f.restype = None
        L.gfo2_coulomb_finalize_d.argtypes = [vp, vp, vp]
        L.gfo2_coulomb_finalize_f.argtypes = [vp, vp, vp]
        L.gfo2_site_update_d.argtypes = [vp, vp, ci, ci, ci, cd, u64, u32, u32]
        L.gfo2_site_update_d.restype = None
        L.gfo2_haar_field_d.argtypes = [vp, vp, u64]
        L.gfo2_haar_field_d.restype = None
        L.gfo_haar_field_d.argtypes = [vp, vp, u64]
        L.gfo_haar_field_d.restype = None
        _lib = L
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def _dims(links: np.ndarray) -> np.ndarray:
    assert links.ndim == 8 and links.shape[4:] in ((4, 3, 3, 2), (4, 2, 2, 2)), links.shape
    assert links.flags.c_contiguous
    return np.array(links.shape[:4], dtype=np.int32)


def nc_of(a: np.ndarray) -> int:
    """Gauge group of a links / transform array: N_c = 3 ([...,3,3,2]) or 2 ([...,2,2,2])."""
    return int(a.shape[-2])


def num_threads() -> int:
    return int(lib().gfo_num_threads())


def _check_gtot(links, gtot):
    if gtot is None:
        return None
    assert gtot.dtype == links.dtype and gtot.flags.c_contiguous
    assert gtot.shape == links.shape[:4] + links.shape[-3:]
    return _p(gtot)


def sweep(links: np.ndarray, gauge: int, algo: int, param: float, seed: int = 0, sweep_index: int = 0,
          mixed: bool = False, gtot: np.ndarray | None = None, parity_mask: int = 3) -> None:
    """One sweep of Alg. 1 (even half-sweep then odd), in place.  float32 links: Step 1 in
    float (SP) or, with ``mixed``, in double (MP).  float64 links: DP."""
    d = _dims(links)
    g = _check_gtot(links, gtot)
    su2 = nc_of(links) == 2
    if links.dtype == np.float64:
        fn = lib().gfo2_sweep_d if su2 else lib().gfo_sweep_d
        rc = fn(_p(links), _p(d), parity_mask, gauge, algo, float(param), seed, sweep_index, g)
    elif links.dtype == np.float32:
        fn = lib().gfo2_sweep_f if su2 else lib().gfo_sweep_f
        rc = fn(_p(links), _p(d), parity_mask, gauge, algo, float(param), seed, sweep_index, 1 if mixed else 0, g)
    else:
        raise TypeError(links.dtype)
    if rc != 0:
        raise ValueError("oracle sweep: invalid arguments (extents must be even and >= 2)")


def measure(links: np.ndarray, gauge: int):
    """F and theta (Eqs. 4, 7, 11; R11).  Returns dict with F, theta, theta_literal,
    theta_slice[Nt], F_slice[Nt]."""
    d = _dims(links)
    out = np.zeros(3)
    ths = np.zeros(int(d[0]))
    fs = np.zeros(int(d[0]))
    if nc_of(links) == 2:
        fn = lib().gfo2_measure_d if links.dtype == np.float64 else lib().gfo2_measure_f
    else:
        fn = lib().gfo_measure_d if links.dtype == np.float64 else lib().gfo_measure_f
    rc = fn(_p(links), _p(d), gauge, _p(out), _p(ths), _p(fs))
    if rc != 0:
        raise ValueError("oracle measure: invalid arguments")
    third = "F_eq8" if nc_of(links) == 2 else "theta_literal"      # N_c = 2: F of Eq. (8) (MAG)
    return {"F": float(out[0]), "theta": float(out[1]), third: float(out[2]), "theta_slice": ths, "F_slice": fs}


def reunitarize(mats: np.ndarray) -> None:
    """Gram-Schmidt reprojection of every [...,3,3,2] matrix in place (R20)."""
    assert mats.flags.c_contiguous and mats.shape[-3:] in ((3, 3, 2), (2, 2, 2))
    if nc_of(mats) == 2:
        (lib().gfo2_reunitarize_d if mats.dtype == np.float64 else lib().gfo2_reunitarize_f)(_p(mats), mats.size // 8)
        return
    n = mats.size // 18
    if mats.dtype == np.float64:
        lib().gfo_reunitarize_d(_p(mats), n)
    else:
        lib().gfo_reunitarize_f(_p(mats), n)


def coulomb_finalize(links: np.ndarray, gtot: np.ndarray) -> None:
    """U_0(x,t) <- G(x,t) U_0(x,t) G(x,t+1)^dagger."""
    d = _dims(links)
    g = _check_gtot(links, gtot)
    if nc_of(links) == 2:
        fn = lib().gfo2_coulomb_finalize_d if links.dtype == np.float64 else lib().gfo2_coulomb_finalize_f
    else:
        fn = lib().gfo_coulomb_finalize_d if links.dtype == np.float64 else lib().gfo_coulomb_finalize_f
    if fn(_p(links), g, _p(d)) != 0:
        raise ValueError("oracle coulomb_finalize: invalid arguments")


def identity_transform(links: np.ndarray) -> np.ndarray:
    g = np.zeros(links.shape[:4] + links.shape[-3:], dtype=links.dtype)
    for i in range(nc_of(links)):
        g[..., i, i, 0] = 1
    return g


def stop_value(m: dict, gauge: int) -> float:
    """Coulomb stops on max_t theta_t (each slice is its own problem); else theta."""
    return float(m["theta_slice"].max()) if gauge == COULOMB else m["theta"]


def run(links: np.ndarray, gauge: int, algo: int, param: float, seed: int = 0, max_sweeps: int = 1000,
        eps: float = 1e-12, check_every: int = 1, reunit_every: int = 0, mixed: bool = False,
        gtot: np.ndarray | None = None, first_sweep_index: int = 0, lagged_stop: bool = False):
    """Alg. 1's outer loop: sweep until theta < eps (checked every `check_every` sweeps) or
    max_sweeps; reproject every `reunit_every` sweeps.  Returns
    (sweeps, F, theta, history[(sweep, F, theta)], converged).
    lagged_stop (the reading of include/gf.h GF_FLAG_LAGGED_STOP, not Alg. 1's): a run that converges at a check
    before max_sweeps applies the even half-sweep of the next sweep before it returns; F, theta returned are those
    of the links returned, the history entry that of the check."""
    hist = []
    m = None
    s = 0
    conv = False
    while s < max_sweeps:
        sweep(links, gauge, algo, param, seed, first_sweep_index + s, mixed, gtot)
        s += 1
        if reunit_every and s % reunit_every == 0:
            reunitarize(links)
            if gtot is not None:
                reunitarize(gtot)
        if s % check_every == 0 or s == max_sweeps:
            m = measure(links, gauge)
            th = stop_value(m, gauge)
            hist.append((s, m["F"], th))
            if th < eps:
                conv = True
                if lagged_stop and s < max_sweeps:
                    sweep(links, gauge, algo, param, seed, first_sweep_index + s, mixed, gtot, parity_mask=1)
                    m = measure(links, gauge)
                break
    if m is None:
        m = measure(links, gauge)
    return s, m["F"], stop_value(m, gauge), hist, conv


def run_coulomb_freeze(links: np.ndarray, algo: int, param: float, seed: int = 0, max_sweeps: int = 1000,
                       eps: float = 1e-12, check_every: int = 1, reunit_every: int = 0, mixed: bool = False,
                       gtot: np.ndarray | None = None, first_sweep_index: int = 0):
    """Coulomb gauge with every time-slice treated as the independent problem it is (PAPER.md:76,
    376 "one slice at a time"): slice t stops being swept at the first check at which its own
    theta_t < eps (R21b).  Written the slow, obvious way: sweep everything, then put the
    spatial links (and the tracked transform) of the already-stopped slices back.  Reprojection, when
    asked for, is applied to every link of every slice.  Returns
    (sweeps, F, max_t theta_t, history[(sweep, F, max_t theta_t)], converged, slice_sweeps[Nt])."""
    Nt = links.shape[0]
    frozen = np.zeros(Nt, dtype=bool)
    slice_sweeps = np.zeros(Nt, dtype=np.int64)
    hist = []
    m = None
    s = 0
    conv = False
    while s < max_sweeps:
        keep = links[frozen].copy()
        keep_g = gtot[frozen].copy() if gtot is not None else None
        sweep(links, COULOMB, algo, param, seed, first_sweep_index + s, mixed, gtot)
        links[frozen] = keep
        if gtot is not None:
            gtot[frozen] = keep_g
        s += 1
        if reunit_every and s % reunit_every == 0:
            reunitarize(links)
            if gtot is not None:
                reunitarize(gtot)
        if s % check_every == 0 or s == max_sweeps:
            m = measure(links, COULOMB)
            newly = (~frozen) & (m["theta_slice"] < eps)
            slice_sweeps[newly] = s
            frozen |= newly
            hist.append((s, m["F"], float(m["theta_slice"].max())))
            if frozen.all():
                conv = True
                break
    if m is None:
        m = measure(links, COULOMB)
    slice_sweeps[~frozen] = s
    return s, m["F"], float(m["theta_slice"].max()), hist, conv, slice_sweeps


def temperature(k: int, n_steps: int, T_hi: float, T_lo: float) -> float:
    """Linear schedule (BASELINE.json config 3; R17)."""
    if n_steps <= 1:
        return T_hi
    return T_hi - k * (T_hi - T_lo) / (n_steps - 1)


def anneal(links: np.ndarray, gauge: int, T_hi: float, T_lo: float, n_steps: int, n_micro: int, seed: int,
           first_sweep_index: int = 0, mixed: bool = False, gtot: np.ndarray | None = None) -> int:
    """Simulated annealing: n_steps heatbath sweeps, each followed by
    n_micro microcanonical sweeps.  Every sweep consumes one sweep index.  Returns the next index."""
    idx = first_sweep_index
    for k in range(n_steps):
        T = temperature(k, n_steps, T_hi, T_lo)
        sweep(links, gauge, SA, T, seed, idx, mixed, gtot)
        idx += 1
        for _ in range(n_micro):
            sweep(links, gauge, MICRO, 0.0, seed, idx, mixed, gtot)
            idx += 1
    return idx


def haar_field(dims_txyz, seed: int, nc: int = 3) -> np.ndarray:
    """h[t,x,y,z,nc,nc,2] (float64), Haar on SU(nc) from Philox normals (R27)."""
    d = np.array(dims_txyz, dtype=np.int32)
    h = np.zeros(tuple(int(v) for v in d) + (nc, nc, 2))
    (lib().gfo2_haar_field_d if nc == 2 else lib().gfo_haar_field_d)(_p(h), _p(d), seed)
    return h


def gauge_transform(links: np.ndarray, h: np.ndarray) -> None:
    """Eq. (1), in place: U_mu(x) <- h(x) U_mu(x) h(x+mu)^dagger (computed in double)."""
    U = links[..., 0].astype(np.float64) + 1j * links[..., 1].astype(np.float64)
    H = h[..., 0].astype(np.float64) + 1j * h[..., 1].astype(np.float64)
    for mu in range(4):
        Hf = np.roll(H, -1, axis=mu)                      # h(x + mu)
        U[..., mu, :, :] = np.einsum("...ab,...bc,...dc->...ad", H, U[..., mu, :, :], Hf.conj())
    links[..., 0] = U.real
    links[..., 1] = U.imag


def random_gauge(links: np.ndarray, seed: int, gtot: np.ndarray | None = None) -> None:
    """A random start on the gauge orbit: Haar h(x), Eq. (1); g(x) <- h(x) g(x)."""
    h = haar_field(links.shape[:4], seed, nc_of(links)).astype(links.dtype)
    gauge_transform(links, h)
    if gtot is not None:
        H = h[..., 0].astype(np.float64) + 1j * h[..., 1].astype(np.float64)
        G = gtot[..., 0].astype(np.float64) + 1j * gtot[..., 1].astype(np.float64)
        G = np.einsum("...ab,...bc->...ac", H, G)
        gtot[..., 0] = G.real
        gtot[..., 1] = G.imag


def fix(links: np.ndarray, gauge: int, seed: int = 0, sa_steps: int = 0, sa_T_hi: float = 1.0, sa_T_lo: float = 0.01,
        sa_micro: int = 3, sr_max_sweeps: int = 0, sr_p: float = 0.5, or_omega: float = 1.7, or_max_sweeps: int = 1000,
        eps: float = 1e-12, check_every: int = 1, reunit_every: int = 0, mixed: bool = False,
        gtot: np.ndarray | None = None):
    """The production recipe of PAPER.md:556 / 580-582: simulated annealing (with microcanonical sweeps),
    then at most sr_max_sweeps stochastic-relaxation sweeps, then overrelaxation until theta < eps.  A stage
    of length 0 is left out; a stage is not entered once theta < eps was reached.  Sweep indices run on from
    stage to stage; reprojection every reunit_every sweeps of each stage.
    Returns (total sweeps, F, theta, converged)."""
    idx = 0
    total = 0
    conv = False
    m = None
    if sa_steps > 0:
        done = 0
        for k in range(sa_steps):
            T = temperature(k, sa_steps, sa_T_hi, sa_T_lo)
            for algo, par in [(SA, T)] + [(MICRO, 0.0)] * sa_micro:
                sweep(links, gauge, algo, par, seed, idx, mixed, gtot)
                idx += 1
                done += 1
                if reunit_every and done % reunit_every == 0:
                    reunitarize(links)
                    if gtot is not None:
                        reunitarize(gtot)
        total += idx
    if sr_max_sweeps > 0:
        s, F, th, _, conv = run(links, gauge, SR, sr_p, seed, sr_max_sweeps, eps, check_every, reunit_every, mixed,
                                gtot, idx)
        total += s
        m = (F, th)
    if or_max_sweeps > 0 and not conv:
        s, F, th, _, conv = run(links, gauge, OR, or_omega, seed, or_max_sweeps, eps, check_every, reunit_every,
                                mixed, gtot, idx)
        total += s
        m = (F, th)
    if m is None:
        mm = measure(links, gauge)
        m = (mm["F"], stop_value(mm, gauge))
        conv = m[1] < eps
    return total, m[0], m[1], conv


def wilson_heatbath(links: np.ndarray, beta: float, seed: int, sweep_index: int = 0) -> None:
    """One Cabibbo-Marinari heatbath sweep of the Wilson action at coupling beta (SU(3)), in place
    (gf_oracle_wilson.hpp): the input generator standing in for the paper's beta = 5.7 ensemble."""
    d = _dims(links)
    if nc_of(links) == 2:
        fn = lib().gfo2_wilson_heatbath_d if links.dtype == np.float64 else lib().gfo2_wilson_heatbath_f
    else:
        fn = lib().gfo_wilson_heatbath_d if links.dtype == np.float64 else lib().gfo_wilson_heatbath_f
    if fn(_p(links), _p(d), float(beta), seed, sweep_index) != 0:
        raise ValueError("oracle wilson_heatbath: invalid arguments")


def plaquette(links: np.ndarray) -> float:
    """<Re tr U_P> / N_c over all 6 V plaquettes."""
    d = _dims(links)
    if nc_of(links) == 2:
        return float((lib().gfo2_plaquette_d if links.dtype == np.float64 else lib().gfo2_plaquette_f)(_p(links), _p(d)))
    return float((lib().gfo_plaquette_d if links.dtype == np.float64 else lib().gfo_plaquette_f)(_p(links), _p(d)))


def staple(links: np.ndarray, t: int, x: int, y: int, z: int, mu: int) -> np.ndarray:
    d = _dims(links)
    out = np.zeros((3, 3, 2))
    lib().gfo_staple_d(_p(links), _p(d), t, x, y, z, mu, _p(out))
    return out


def site_update(up: np.ndarray, dn: np.ndarray, gauge: int, algo: int, param: float, seed: int = 0,
                site_index: int = 0, sweep_index: int = 0, mixed: bool = False):
    """Update of one site from its gathered links up[m]=U_mu(x), dn[m]=U_mu(x-mu), shape [nd,3,3,2]."""
    nd = up.shape[0]
    assert up.shape[1:] in ((3, 3, 2), (2, 2, 2)) and dn.shape == up.shape and up.flags.c_contiguous and dn.flags.c_contiguous
    if nc_of(up) == 2:
        assert up.dtype == np.float64
        lib().gfo2_site_update_d(_p(up), _p(dn), nd, gauge, algo, float(param), seed, site_index, sweep_index)
    elif up.dtype == np.float64:
        lib().gfo_site_update_d(_p(up), _p(dn), nd, gauge, algo, float(param), seed, site_index, sweep_index, None)
    else:
        lib().gfo_site_update_f(_p(up), _p(dn), nd, gauge, algo, float(param), seed, site_index, sweep_index,
                                1 if mixed else 0, None)


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().gfo_philox4x32_10(_p(c), _p(k), _p(out))
    return out


def draw(seed: int, site: int, sweep: int, sub: int, purpose: int, trial: int):
    out = np.zeros(4, dtype=np.uint32)
    uni = np.zeros(4)
    lib().gfo_draw(seed, site, sweep, sub, purpose, trial, _p(out), _p(uni))
    return out, uni


def local_quaternion(up, dn, i, j) -> np.ndarray:
    a = np.zeros(4)
    lib().gfo_local_quaternion_d(_p(up), _p(dn), up.shape[0], i, j, _p(a))
    return a


def local_mag_def(up, dn, i, j) -> np.ndarray:
    a = np.zeros(3)
    lib().gfo_local_mag_def_d(_p(up), _p(dn), up.shape[0], i, j, _p(a))
    return a


def rule_or(a, omega) -> np.ndarray:
    a = np.asarray(a, dtype=np.float64).copy()
    g = np.zeros(4)
    lib().gfo_rule_or_d(_p(a), float(omega), _p(g))
    return g


def rule_micro(a) -> np.ndarray:
    a = np.asarray(a, dtype=np.float64).copy()
    g = np.zeros(4)
    lib().gfo_rule_micro_d(_p(a), _p(g))
    return g


def rule_heatbath_landau(a, T, seed, site, sweep, sub) -> np.ndarray:
    a = np.asarray(a, dtype=np.float64).copy()
    g = np.zeros(4)
    lib().gfo_rule_heatbath_landau(_p(a), float(T), seed, site, sweep, sub, _p(g))
    return g


def rule_heatbath_mag(D, E, F, T, seed, site, sweep, sub) -> np.ndarray:
    g = np.zeros(4)
    lib().gfo_rule_heatbath_mag(float(D), float(E), float(F), float(T), seed, site, sweep, sub, _p(g))
    return g


def apply_subgroup(mat: np.ndarray, g, i: int, j: int, right_dagger: bool = False) -> np.ndarray:
    m = np.ascontiguousarray(mat, dtype=np.float64).copy()
    g = np.asarray(g, dtype=np.float64).copy()
    lib().gfo_apply_subgroup_d(_p(m), _p(g), i, j, 1 if right_dagger else 0)
    return m
