"""GF_FLAG_LAGGED_STOP (include/gf.h, gf_run): the stopping decision of a check is taken half a sweep later from the
even half-sweep's own partial sums, at no extra traffic; the run stops at the sweep Alg. 1 stops at, with one more even
half-sweep applied.  Against the oracle's mirror of that reading (oracle.run(..., lagged_stop=True))."""
import numpy as np
import pytest

from paper_1212_5221_b200 import inputs

pytestmark = pytest.mark.gpu

LANDAU, COULOMB, MAG = 0, 1, 2
OR = 0
SP, DP, MP = 0, 1, 2


@pytest.fixture(scope="module")
def gf():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1212_5221_b200 import gf as _gf
    return _gf


@pytest.mark.parametrize("gauge,check_every", [(LANDAU, 1), (LANDAU, 4), (MAG, 1), (COULOMB, 2)])
def test_lagged_stop_matches_the_oracle_and_the_plain_stopping_sweep(gf, oracle, gauge, check_every):
    dims = (8, 6, 4, 8)
    L = inputs.as_real(inputs.make_config(*dims, 0.4, 501, 502))
    eps = 1e-11
    ref = L.copy()
    g = oracle.identity_transform(ref)
    s_o, F_o, th_o, hist_o, conv_o = oracle.run(ref, gauge, OR, 1.7, max_sweeps=3000, eps=eps, check_every=check_every, gtot=g,
                                                lagged_stop=True)
    if gauge == COULOMB:
        oracle.coulomb_finalize(ref, g)
    out = {}
    for lagged in (True, False):
        with gf.GaugeFixer(*dims, precision=DP, track_transform=True, lagged_stop=lagged) as fx:
            fx.set_links(L)
            gf.gf_launch_count(fx.ctx, reset=True)
            r = fx.run(gauge, OR, 1.7, max_sweeps=3000, eps=eps, check_every=check_every, history=True)
            out[lagged] = (r, fx.get_links(), gf.gf_launch_count(fx.ctx, reset=True))
    r, got, n_lag = out[True]
    r0, _, n_plain = out[False]
    assert conv_o and r["converged"] and r0["converged"]
    assert r["sweeps"] == s_o == r0["sweeps"]                       # the stopping sweep is Alg. 1's
    assert abs(r["F"] - F_o) <= 1e-10 and r["theta"] < eps and abs(r["theta"] - th_o) <= 0.1 * th_o
    assert np.abs(got - ref).max() <= 1e-9
    h = r["history"]
    assert len(h) == len(hist_o) and np.array_equal(h[:, 0], [x[0] for x in hist_o])
    assert np.abs(h[:, 1] - [x[1] for x in hist_o]).max() <= 1e-10
    assert np.all(np.abs(h[:, 2] - [x[2] for x in hist_o]) <= 1e-6 * np.array([x[2] for x in hist_o]) + 1e-18)
    assert n_lag < n_plain                                            # no stand-alone reductions but the final one


def test_lagged_stop_at_max_sweeps_and_mp(gf, oracle):
    dims = (4, 4, 4, 4)
    L = inputs.as_real(inputs.make_config(*dims, 0.4, 511, 512), np.float32)
    ref = L.copy()
    s_o, F_o, th_o, _, conv_o = oracle.run(ref, LANDAU, OR, 1.7, max_sweeps=400, eps=1e-9, mixed=True, lagged_stop=True)
    with gf.GaugeFixer(*dims, precision=MP, lagged_stop=True) as fx:
        fx.set_links(L)
        r = fx.run(LANDAU, OR, 1.7, max_sweeps=400, eps=1e-9)
        assert conv_o and r["converged"] and abs(r["sweeps"] - s_o) <= 1 and abs(r["F"] - F_o) <= 1e-5
        fx.set_links(L)
        r = fx.run(LANDAU, OR, 1.7, max_sweeps=7, eps=1e-9)       # not converged: exactly 7 sweeps, nothing more
        ref7 = L.copy()
        for k in range(7):
            oracle.sweep(ref7, LANDAU, OR, 1.7, 0, k, True)
        assert not r["converged"] and r["sweeps"] == 7
        assert np.abs(fx.get_links(dtype=np.float32).astype(np.float64) - ref7).max() <= 5e-5


def test_lagged_stop_is_ignored_on_sp_contexts(gf):
    """on GF_SP the fused sums are float sums with ~1e-12 of noise in theta, so a lagged decision near eps
    could contradict the exact reduction after the links have moved on.  The flag therefore does nothing on SP: the run
    is the plain one bit for bit (sweeps, F, theta, history, links), converged means theta of the RETURNED links < eps,
    and no extra half-sweep has been applied."""
    dims = (8, 6, 4, 8)
    L = inputs.as_real(inputs.make_config(*dims, 0.4, 521, 522), np.float32)
    for eps in (1e-9, 3e-11):             # the second sits inside the noise band of the fused float sums
        out = {}
        for lagged in (True, False):
            with gf.GaugeFixer(*dims, precision=SP, lagged_stop=lagged) as fx:
                fx.set_links(L)
                r = fx.run(LANDAU, OR, 1.7, max_sweeps=600, eps=eps, check_every=1, reunit_every=50, history=True)
                F, th = fx.measure(LANDAU)
                out[lagged] = (r, fx.get_links(dtype=np.float32), F, th)
        r, links, F, th = out[True]
        r0, links0, F0, th0 = out[False]
        assert r["sweeps"] == r0["sweeps"] and r["F"] == r0["F"] and r["theta"] == r0["theta"] and r["converged"] == r0["converged"]
        assert np.array_equal(r["history"], r0["history"]) and np.array_equal(links, links0)
        assert th == r["theta"] and F == r["F"]                    # what the run reports is the state it returns
        if r["converged"]:
            assert th < eps
