"""GPU parity for the gauge group SU(2) (GF_FLAG_SU2): the quaternion kernels of
csrc/sweep_su2.cuh / aux_su2.cuh through the C ABI against the N_c = 2 oracle (oracle/gf_oracle_su2.hpp,
2x2 complex matrices), element by element on identical seeded inputs, BASELINE.json's tolerances:
one sweep per link <= 1e-12 (DP) / 5e-5 (SP, MP), annealing <= 1e-11 (DP), full runs F to 1e-10 / 1e-5.
"""
import numpy as np
import pytest

from paper_1212_5221_b200 import inputs

pytestmark = pytest.mark.gpu

LANDAU, COULOMB, MAG = 0, 1, 2
OR, SR, SA, MICRO = 0, 1, 2, 3
SP, DP, MP = 0, 1, 2
TOL = {DP: 1e-12, SP: 5e-5, MP: 5e-5}


@pytest.fixture(scope="module")
def gf():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1212_5221_b200 import gf as _gf
    return _gf


def make(dims_xyzt, eps=0.5, seed=900, dtype=np.float64):
    Nx, Ny, Nz, Nt = dims_xyzt
    return inputs.as_real(inputs.make_config_su2(Nx, Ny, Nz, Nt, eps, seed, seed + 1), dtype)


def dt_of(prec):
    return np.float64 if prec == DP else np.float32


@pytest.mark.parametrize("prec", [DP, SP])
def test_layout_roundtrip(gf, prec):
    dims = (6, 4, 8, 4)
    L = make(dims, dtype=dt_of(prec))
    with gf.GaugeFixer(*dims, precision=prec, su2=True) as fx:
        assert gf.gf_num_colors(fx.ctx) == 2
        fx.set_links(L)
        got = fx.get_links(dtype=dt_of(prec))
        with pytest.raises(ValueError):
            fx.set_links(np.zeros((4, 6, 4, 8, 4, 3, 3, 2)))       # SU(3)-shaped buffer
    # first row bit exact; second row rebuilt as (-conj b, conj a)
    assert np.array_equal(got[..., 0, :, :], L[..., 0, :, :])
    assert np.abs(got - L).max() <= (1e-15 if prec == DP else 2e-7)


CASES = [(LANDAU, OR, 1.7), (LANDAU, OR, 1.0), (COULOMB, OR, 1.7), (MAG, OR, 1.7), (LANDAU, MICRO, 0.0),
         (MAG, MICRO, 0.0), (COULOMB, SR, 0.5), (MAG, SR, 0.5), (LANDAU, SA, 1.2), (COULOMB, SA, 0.3), (MAG, SA, 0.8)]


@pytest.mark.parametrize("prec", [DP, SP, MP])
@pytest.mark.parametrize("gauge,algo,param", CASES)
def test_one_sweep_per_link(gf, oracle, prec, gauge, algo, param):
    dims = (6, 4, 10, 6)          # Vsh = 120 per slice: ragged against the 128-thread CTA
    dt = dt_of(prec)
    L = make(dims, seed=910 + gauge, dtype=dt)
    ref = L.copy()
    g = oracle.identity_transform(ref)
    oracle.sweep(ref, gauge, algo, param, seed=77, sweep_index=3, mixed=(prec == MP), gtot=g)
    if gauge == COULOMB:
        oracle.coulomb_finalize(ref, g)
    with gf.GaugeFixer(*dims, precision=prec, su2=True, track_transform=True) as fx:
        fx.set_links(L)
        fx.sweep(gauge, algo, param, seed=77, sweep_index=3)
        got = fx.get_links(dtype=dt)
        gg = fx.get_gauge_transform(dtype=dt)
    tol = TOL[prec] * (10 if (algo == SA and prec == DP) else 1)
    for diff in (np.abs(got.astype(np.float64) - ref), np.abs(gg.astype(np.float64) - g)):
        assert diff.max() <= tol, diff.max()


@pytest.mark.parametrize("prec", [DP, SP])
@pytest.mark.parametrize("gauge", [LANDAU, COULOMB, MAG])
def test_measure_and_reunitarize(gf, oracle, prec, gauge):
    dims = (4, 6, 4, 6)
    dt = dt_of(prec)
    L = make(dims, seed=930, dtype=dt)
    L *= dt(1.0 + 3e-3)               # off the group: reprojection has something to do
    m = oracle.measure(L, gauge)
    ref = L.copy()
    oracle.reunitarize(ref)
    with gf.GaugeFixer(*dims, precision=prec, su2=True) as fx:
        fx.set_links(L)
        F, th, ths = fx.measure(gauge, slices=True)
        fx.reunitarize()
        got = fx.get_links(dtype=dt)
    rel = 1e-12 if prec == DP else 1e-5
    # the oracle measures all 8 stored reals, the device the first row: the same on (scaled) SU(2) links
    assert F == pytest.approx(m["F"], rel=rel, abs=rel)
    assert th == pytest.approx(m["theta"], rel=max(rel, 1e-10))
    np.testing.assert_allclose(ths, m["theta_slice"], rtol=max(rel, 1e-10))
    assert np.abs(got.astype(np.float64) - ref).max() <= (1e-15 if prec == DP else 2e-7)


@pytest.mark.parametrize("gauge,prec,eps_stop", [(LANDAU, DP, 1e-12), (MAG, DP, 1e-12), (COULOMB, DP, 1e-12),
                                                (LANDAU, SP, 1e-9), (COULOMB, MP, 1e-9)])
def test_full_run(gf, oracle, gauge, prec, eps_stop):
    dims = (8, 8, 8, 8)
    dt = dt_of(prec)
    L = make(dims, seed=940 + gauge, dtype=dt)
    ref = L.copy()
    reunit = 0 if prec == DP else 50
    s, F, th, hist, conv = oracle.run(ref, gauge, OR, 1.7, max_sweeps=5000, eps=eps_stop, check_every=2,
                                      reunit_every=reunit, mixed=(prec == MP))
    with gf.GaugeFixer(*dims, precision=prec, su2=True, track_transform=True) as fx:
        fx.set_links(L)
        r = fx.run(gauge, OR, 1.7, max_sweeps=5000, eps=eps_stop, check_every=2, reunit_every=reunit, history=True)
        got = fx.get_links(dtype=dt)
        g = fx.get_gauge_transform()
    assert conv and r["converged"] and r["theta"] < eps_stop
    if prec == DP:
        assert abs(r["sweeps"] - s) <= 2 and abs(r["F"] - F) <= 1e-10
        n = min(len(hist), len(r["history"]))
        np.testing.assert_allclose(r["history"][:n, 1], [h[1] for h in hist][:n], atol=1e-10)
        if r["sweeps"] == s:
            assert abs(r["theta"] - th) <= 0.1 * th
        gc = inputs.as_complex(g)
        want = inputs.gauge_transform(inputs.as_complex(L), gc)
        assert np.abs(inputs.as_complex(got) - want).max() < 1e-10
    else:
        assert abs(r["F"] - F) <= 1e-5 and abs(r["sweeps"] - s) <= 0.1 * s + 10


def test_batch_fix_and_random_gauge(gf, oracle):
    dims = (4, 4, 4, 4)
    B = 3
    L = make(dims, eps=0.4, seed=950)
    kw = dict(seed=21, sa_steps=3, sa_T_hi=0.05, sa_T_lo=0.01, sa_micro=1, sr_max_sweeps=6, sr_p=0.3,
              or_omega=1.7, or_max_sweeps=3000, eps=1e-12, check_every=1)
    with gf.GaugeFixer(*dims, precision=DP, su2=True, n_copies=B, track_transform=True) as fx:
        fx.set_links(L)
        fx.random_gauge(5)
        starts = []
        for c in range(B):
            ref = L.copy()
            g = oracle.identity_transform(ref)
            oracle.random_gauge(ref, 5 + c, g)
            assert np.abs(fx.get_links_copy(c) - ref).max() <= 1e-12
            assert np.abs(fx.get_gauge_transform_copy(c) - g).max() <= 1e-12
            starts.append(ref)
        res = fx.fix(LANDAU, **kw)
        for c in range(B):
            kwo = dict(kw)
            kwo["seed"] = 21 + c
            tot, F, th, conv = oracle.fix(starts[c], LANDAU, **kwo)
            assert conv and res[c]["converged"] and res[c]["theta"] < 1e-12
            assert abs(res[c]["F"] - F) <= 1e-9 and abs(res[c]["sweeps"] - tot) <= 3
            # links of copy c = input transformed by the accumulated g (random start and all sweeps)
            gc = inputs.as_complex(fx.get_gauge_transform_copy(c))
            want = inputs.gauge_transform(inputs.as_complex(L), gc)
            assert np.abs(inputs.as_complex(fx.get_links_copy(c)) - want).max() < 1e-10


@pytest.mark.parametrize("prec", [DP, SP])
def test_large_lattice_tiled(gf, oracle, prec):
    # 32^3 x 64 in the launch configuration bench.py times: a sweep of the periodic tiling of an 8^4 lattice
    # is the tiling of the swept 8^4 lattice
    import torch
    dims = (32, 32, 32, 64)
    dt = dt_of(prec)
    tile = make((8, 8, 8, 8), seed=960, dtype=dt)
    ref = tile.copy()
    oracle.sweep(ref, LANDAU, OR, 1.7)
    m = oracle.measure(ref, LANDAU)
    dev = torch.device("cuda", 0)
    src = torch.from_numpy(tile).to(dev).repeat(8, 4, 4, 4, 1, 1, 1, 1).contiguous()
    with gf.GaugeFixer(*dims, precision=prec, su2=True) as fx:
        fx.set_links(src)
        fx.sweep(LANDAU, OR, 1.7)
        F, th = fx.measure(LANDAU)
        out = torch.empty_like(src)
        gf.gf_get_links(fx.ctx, out)
    want = torch.from_numpy(ref).to(dev).repeat(8, 4, 4, 4, 1, 1, 1, 1)
    assert (out.to(torch.float64) - want.to(torch.float64)).abs().max().item() <= TOL[prec]
    rel = 1e-12 if prec == DP else 2e-6
    assert F == pytest.approx(m["F"], rel=rel, abs=rel) and th == pytest.approx(m["theta"], rel=10 * rel)


def test_unitarity_and_bad_arguments_on_su2_contexts(gf):
    dims = (4, 4, 4, 4)
    L = make(dims)
    with gf.GaugeFixer(*dims, precision=DP, su2=True) as fx:
        fx.set_links(L)
        avg, mx = fx.unitarity()                       # Eq. (33) with det U = |u|^2
        assert mx[0] < 1e-15
        fx.set_links(L * 1.001)
        avg, mx = fx.unitarity()
        assert abs(avg[0] - (1.001 ** 2 - 1)) < 1e-12 and abs(mx[0] - (1.001 ** 2 - 1)) < 1e-12
        fx.set_links(L)
        for kw in (dict(check_every=0), dict(sa_steps=-1), dict(or_omega=2.5), dict(sa_steps=2, sa_T_lo=0.0)):
            with pytest.raises(gf.GfError) as e:
                fx.fix(LANDAU, **kw)
            assert e.value.code == gf.GF_EINVAL
        with pytest.raises(gf.GfError):
            fx.sweep(LANDAU, OR, 2.0)


def test_three_dimensional_lattices_are_coulomb_slices(gf, oracle):
    # d = 3 ("3+1 dimensional" in the paper's abstract): a stack of N_t independent three-dimensional SU(2)
    # lattices is fixed to the 3-d Landau gauge by GF_COULOMB, one lattice per time-slice; with
    # GF_FLAG_FREEZE_SLICES every lattice stops on its own theta
    dims = (6, 6, 6, 4)
    L = make(dims, eps=0.4, seed=970)
    with gf.GaugeFixer(*dims, precision=DP, su2=True, freeze_slices=True) as fx:
        fx.set_links(L)
        r = fx.run(COULOMB, OR, 1.6, max_sweeps=4000, eps=1e-12, check_every=2)
        sw = fx.slice_sweeps()
        F, th, ths = fx.measure(COULOMB, slices=True)
    ref = L.copy()
    s, Fo, tho, hist, conv, sl = oracle.run_coulomb_freeze(ref, OR, 1.6, max_sweeps=4000, eps=1e-12, check_every=2)
    assert conv and r["converged"] and ths.max() < 1e-12
    assert np.all(np.abs(sw - sl) <= 2) and abs(r["F"] - Fo) <= 1e-10
    assert len(set(sw.tolist())) > 1


@pytest.mark.parametrize("prec,beta", [(DP, 2.4), (DP, 0.5), (SP, 2.4)])
def test_wilson_heatbath_and_plaquette(gf, oracle, prec, beta):
    # the input generator on SU(2) links: draws identical to the oracle's, per link <= 1e-11 per sweep in DP
    dims = (4, 6, 4, 6)
    B = 2
    dt = dt_of(prec)
    L = make(dims, eps=0.4, seed=980, dtype=dt)
    with gf.GaugeFixer(*dims, precision=prec, su2=True, n_copies=B) as fx:
        fx.set_links(L)
        assert abs(fx.plaquette()[0] - oracle.plaquette(L)) <= (1e-13 if prec == DP else 2e-7)
        fx.wilson_heatbath(beta, seed=41, first_sweep_index=2, n_sweeps=2)
        P = fx.plaquette()
        for c in range(B):
            ref = L.copy()
            oracle.wilson_heatbath(ref, beta, 41 + c, 2)
            oracle.wilson_heatbath(ref, beta, 41 + c, 3)
            diff = np.abs(fx.get_links_copy(c, dtype=dt).astype(np.float64) - ref)
            assert diff.max() <= (1e-10 if prec == DP else 5e-5), diff.max()
            assert abs(P[c] - oracle.plaquette(ref)) <= (1e-10 if prec == DP else 1e-4)


def test_thermalised_su2_lattice_is_fixed_and_keeps_its_plaquette(gf):
    # 16^4 at beta = 2.4 from a cold start (lattice literature: <P> = 0.630; not a number of the paper), then Landau
    dims = (16, 16, 16, 16)
    cold = inputs.as_real(np.broadcast_to(np.eye(2, dtype=np.complex128), (16, 16, 16, 16, 4, 2, 2)).copy())
    with gf.GaugeFixer(*dims, precision=DP, su2=True) as fx:
        fx.set_links(cold)
        fx.wilson_heatbath(2.4, seed=3, n_sweeps=200)
        vals = []
        for k in range(10):
            fx.wilson_heatbath(2.4, seed=3, first_sweep_index=200 + 5 * k, n_sweeps=5)
            vals.append(fx.plaquette()[0])
        assert abs(np.mean(vals) - 0.630) < 0.004, np.mean(vals)
        P0 = fx.plaquette()[0]
        r = fx.run(LANDAU, OR, 1.7, max_sweeps=20000, eps=1e-12, check_every=10)
        assert r["converged"] and 0.8 < r["F"] < 0.95
        assert abs(fx.plaquette()[0] - P0) < 1e-12
