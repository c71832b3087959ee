"""Sequences of calls on a context that tracks g(x) (GF_FLAG_TRACK_TRANSFORM) in which Coulomb sweeps follow
operations that have ALREADY rotated the temporal links: gf_random_gauge and Landau / MAG sweeps act on all four
directions (Eq. (1)), Coulomb sweeps on the spatial links only, and the finalisation
U_0(x,t) <- g(x,t) U_0(x,t) g(x,t+1)^dagger must then apply only what the Coulomb sweeps added.
gf.h documents these sequences (implicit finalisation on gf_get_links and on Landau/MAG calls after Coulomb).

The oracle side is the obviously correct composition: it tracks the Coulomb part g_C of the transform in a field
of its own, finalises with g_C alone and multiplies the pieces afterwards.  Two checks per case:
  (1) the links returned equal the oracle's, and the returned g(x) equals the oracle's product;
  (2) Eq. (1) end to end: links_out == g(x) links_in g(x+mu)^dagger with the returned g — the property that
      the accumulated transform exists for (gf_get_gauge_transform, gf.h).
"""
import numpy as np
import pytest

from paper_1212_5221_b200 import inputs

pytestmark = pytest.mark.gpu

LANDAU, COULOMB, MAG = 0, 1, 2
OR, SR, SA, MICRO = 0, 1, 2, 3
SP, DP, MP = 0, 1, 2


@pytest.fixture(scope="module")
def gf():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1212_5221_b200 import gf as _gf
    return _gf


def config(dims_xyzt, su2, seed):
    Nx, Ny, Nz, Nt = dims_xyzt
    mk = inputs.make_config_su2 if su2 else inputs.make_config
    return inputs.as_real(mk(Nx, Ny, Nz, Nt, 0.4, seed, seed + 1))


def cmul(a, b):
    """matrix product of two [..., n, n, 2] real-pair fields"""
    A = a[..., 0] + 1j * a[..., 1]
    B = b[..., 0] + 1j * b[..., 1]
    C = np.einsum("...ab,...bc->...ac", A, B)
    out = np.empty_like(a)
    out[..., 0], out[..., 1] = C.real, C.imag
    return out


def check_eq1(oracle, L_in, L_out, g, tol):
    want = L_in.copy()
    oracle.gauge_transform(want, g)
    assert np.abs(want - L_out).max() <= tol


@pytest.mark.parametrize("su2", [False, True])
@pytest.mark.parametrize("B", [1, 2])
def test_random_gauge_then_coulomb_run(gf, oracle, su2, B):
    dims = (4, 6, 4, 6)
    L = config(dims, su2, 710)
    n_sw = 10
    with gf.GaugeFixer(*dims, precision=DP, n_copies=B, track_transform=True, su2=su2) as fx:
        fx.set_links(L)
        fx.random_gauge(41)
        res = fx.run_batch(COULOMB, OR, 1.7, max_sweeps=n_sw, eps=1e-30, check_every=5)
        assert all(r["sweeps"] == n_sw for r in res)
        for c in range(B):
            ref = L.copy()
            h = oracle.identity_transform(ref)
            oracle.random_gauge(ref, 41 + c, h)           # all four directions rotated by h
            gC = oracle.identity_transform(ref)
            oracle.run(ref, COULOMB, OR, 1.7, max_sweeps=n_sw, eps=1e-30, check_every=5, gtot=gC)
            oracle.coulomb_finalize(ref, gC)              # only the Coulomb part goes onto U_0
            got = fx.get_links_copy(c)
            g = fx.get_gauge_transform_copy(c)
            assert np.abs(got - ref).max() <= 1e-11
            assert np.abs(g - cmul(gC, h)).max() <= 1e-11
            check_eq1(oracle, L, got, g, 1e-11)


@pytest.mark.parametrize("su2", [False, True])
@pytest.mark.parametrize("first", [LANDAU, MAG])
def test_landau_or_mag_sweeps_then_coulomb_run_then_get(gf, oracle, su2, first):
    dims = (4, 4, 6, 4)
    L = config(dims, su2, 720)
    with gf.GaugeFixer(*dims, precision=DP, track_transform=True, su2=su2) as fx:
        fx.set_links(L)
        ref = L.copy()
        g1 = oracle.identity_transform(ref)
        for k in range(2):
            fx.sweep(first, OR, 1.6)
            oracle.sweep(ref, first, OR, 1.6, gtot=g1)
        r = fx.run(COULOMB, OR, 1.7, max_sweeps=8, eps=1e-30, check_every=4)
        assert r["sweeps"] == 8
        gC = oracle.identity_transform(ref)
        oracle.run(ref, COULOMB, OR, 1.7, max_sweeps=8, eps=1e-30, check_every=4, gtot=gC)
        oracle.coulomb_finalize(ref, gC)
        got = fx.get_links()
        g = fx.get_gauge_transform()
        assert np.abs(got - ref).max() <= 1e-11
        assert np.abs(g - cmul(gC, g1)).max() <= 1e-11
        check_eq1(oracle, L, got, g, 1e-11)


@pytest.mark.parametrize("prec,recon,tol", [(DP, 12, 1e-11), (SP, 18, 2e-5)])
def test_coulomb_landau_coulomb_interleaved(gf, oracle, prec, recon, tol):
    # Coulomb sweeps (finalised implicitly by the Landau sweep that follows), Landau sweeps, Coulomb sweeps again
    # (finalised implicitly by gf_get_links): two snapshots of g(x), the second on a non-trivial transform
    dims = (4, 4, 4, 6)
    dt = np.float64 if prec == DP else np.float32
    L = config(dims, False, 730).astype(dt)
    with gf.GaugeFixer(*dims, precision=prec, recon=recon, track_transform=True) as fx:
        fx.set_links(L)
        ref = L.copy()
        gA = oracle.identity_transform(ref)
        for k in range(2):
            fx.sweep(COULOMB, OR, 1.5)
            oracle.sweep(ref, COULOMB, OR, 1.5, gtot=gA)
        oracle.coulomb_finalize(ref, gA)
        gB = oracle.identity_transform(ref)
        fx.sweep(LANDAU, OR, 1.7)
        oracle.sweep(ref, LANDAU, OR, 1.7, gtot=gB)
        gC = oracle.identity_transform(ref)
        for k in range(2):
            fx.sweep(COULOMB, SR, 0.5, seed=3, sweep_index=k)
            oracle.sweep(ref, COULOMB, SR, 0.5, 3, k, gtot=gC)
        oracle.coulomb_finalize(ref, gC)
        got = fx.get_links(dtype=dt)
        g = fx.get_gauge_transform(dtype=dt)
        assert np.abs(got.astype(np.float64) - ref).max() <= tol
        gref = cmul(gC.astype(np.float64), cmul(gB.astype(np.float64), gA.astype(np.float64)))
        assert np.abs(g.astype(np.float64) - gref).max() <= tol
        check_eq1(oracle, L.astype(np.float64), got.astype(np.float64), g.astype(np.float64), tol)


def test_batch_copy_replaced_between_coulomb_runs(gf, oracle):
    # B > 1: one copy receives new links while the others carry an accumulated transform; the next Coulomb run
    # must finalise every copy with its own increment
    dims = (4, 4, 4, 4)
    B = 3
    Ls = [config(dims, False, 740 + 10 * c) for c in range(B)]
    Lnew = config(dims, False, 790)
    with gf.GaugeFixer(*dims, precision=DP, n_copies=B, track_transform=True) as fx:
        for c in range(B):
            fx.set_links_copy(c, Ls[c])
        fx.run_batch(COULOMB, OR, 1.7, max_sweeps=4, eps=1e-30, check_every=4)
        fx.set_links_copy(1, Lnew)
        fx.run_batch(COULOMB, OR, 1.7, max_sweeps=3, eps=1e-30, check_every=3)
        for c in range(B):
            src = Lnew if c == 1 else Ls[c]
            ref = src.copy()
            g = oracle.identity_transform(ref)
            if c != 1:
                oracle.run(ref, COULOMB, OR, 1.7, max_sweeps=4, eps=1e-30, check_every=4, gtot=g)
            oracle.run(ref, COULOMB, OR, 1.7, max_sweeps=3, eps=1e-30, check_every=3, gtot=g)
            oracle.coulomb_finalize(ref, g)       # Coulomb only: one finalisation with the whole g is the definition
            got = fx.get_links_copy(c)
            gg = fx.get_gauge_transform_copy(c)
            assert np.abs(got - ref).max() <= 1e-11
            assert np.abs(gg - g).max() <= 1e-11
            check_eq1(oracle, src, got, gg, 1e-11)
