"""Pins of the oracle's input generator (oracle/gf_oracle_wilson.hpp): the
Cabibbo-Marinari heatbath of the Wilson action and the plaquette, against what the mathematics fixes:
  * the plaquette against an independent NumPy evaluation (tests/helpers.py);
  * the staple sum: Re tr[U A] summed over a link's 6 plaquettes equals the sum of those plaquettes;
  * strong coupling: <P> = beta/18 + beta^2/216 + O(beta^3) (SU(3) character expansion);
  * weak coupling: 1 - <P> -> (N_c^2 - 1)/(4 beta/ (2 N_c)) ... = 2/beta for SU(3) in four dimensions;
  * beta -> infinity: the update maximises Re tr[U A] subgroup by subgroup, so the mean plaquette rises
    monotonically and no link's local action term decreases;
  * links stay in SU(3); different seeds / sweep indices give different configurations, same ones the same.
"""
import numpy as np
import pytest

from paper_1212_5221_b200 import inputs
from tests.helpers import dag, plaquettes


def cold(dims_txyz):
    U = np.broadcast_to(np.eye(3, dtype=np.complex128), tuple(dims_txyz) + (4, 3, 3)).copy()
    return inputs.as_real(U)


def test_plaquette_matches_numpy(oracle):
    U = inputs.make_config(4, 6, 4, 4, 0.5, 3, 4)
    assert abs(oracle.plaquette(inputs.as_real(U)) - plaquettes(U).mean()) < 1e-14
    assert abs(oracle.plaquette(cold((4, 4, 4, 4))) - 1.0) < 1e-15


def test_staple_sum_is_the_sum_of_the_links_plaquettes(oracle):
    U = inputs.make_config(4, 4, 4, 4, 0.5, 5, 6)
    L = inputs.as_real(U)
    t, x, y, z, mu = 1, 3, 0, 2, 2
    A = inputs.as_complex(oracle.staple(L, t, x, y, z, mu))
    got = np.trace(U[t, x, y, z, mu] @ A).real
    # the 6 plaquettes through the link, written out with np.roll'ed fields
    want = 0.0
    c = (t, x, y, z)
    for nu in range(4):
        if nu == mu:
            continue
        Umu, Unu = U[..., mu, :, :], U[..., nu, :, :]
        P = Umu @ np.roll(Unu, -1, axis=mu) @ dag(np.roll(Umu, -1, axis=nu)) @ dag(Unu)      # plaquette at x
        want += np.trace(P[c]).real
        cm = list(c)
        cm[nu] = (cm[nu] - 1) % U.shape[nu]
        want += np.trace(P[tuple(cm)]).real                                                  # plaquette at x - nu
    assert abs(got - want) < 1e-13


def test_links_stay_in_su3_and_draws_are_keyed(oracle):
    L = inputs.as_real(inputs.make_config(4, 4, 4, 4, 0.3, 7, 8))
    a, b, c = L.copy(), L.copy(), L.copy()
    oracle.wilson_heatbath(a, 5.7, seed=1, sweep_index=0)
    oracle.wilson_heatbath(b, 5.7, seed=1, sweep_index=0)
    oracle.wilson_heatbath(c, 5.7, seed=1, sweep_index=1)
    assert np.array_equal(a, b) and np.abs(a - c).max() > 1e-2
    V = inputs.as_complex(a)
    assert np.abs(V @ dag(V) - np.eye(3)).max() < 1e-13 and np.abs(np.linalg.det(V) - 1).max() < 1e-13


def test_strong_coupling_plaquette(oracle):
    beta = 0.6
    L = inputs.as_real(inputs.make_config(4, 4, 4, 4, 3.0, 9, 10))     # a rough start
    vals = []
    for s in range(45):
        oracle.wilson_heatbath(L, beta, seed=11, sweep_index=s)
        if s >= 5:
            vals.append(oracle.plaquette(L))
    want = beta / 18 + beta ** 2 / 216
    assert abs(np.mean(vals) - want) < 0.004, (np.mean(vals), want)


def test_weak_coupling_plaquette(oracle):
    beta = 40.0
    L = cold((4, 4, 4, 4))
    vals = []
    for s in range(40):
        oracle.wilson_heatbath(L, beta, seed=13, sweep_index=s)
        if s >= 15:
            vals.append(oracle.plaquette(L))
    # 1 - <P> = 2/beta (1 + O(1/beta)); on 4^4 the zero modes take a few per cent off
    assert 0.85 * 2 / beta < 1 - np.mean(vals) < 1.1 * 2 / beta, 1 - np.mean(vals)


def test_infinite_beta_is_a_monotone_cooling(oracle):
    L = inputs.as_real(inputs.make_config(4, 4, 4, 4, 0.8, 15, 16))
    P = [oracle.plaquette(L)]
    for s in range(6):
        oracle.wilson_heatbath(L, 1e9, seed=17, sweep_index=s)
        P.append(oracle.plaquette(L))
    assert np.all(np.diff(P) > 0) and P[-1] > P[0] + 0.2


# ---- gauge group SU(2): <P> = beta/4 + O(beta^3) at strong coupling, 1 - <P> -> 3/(4 beta) at weak coupling ----
def cold2(dims_txyz):
    U = np.broadcast_to(np.eye(2, dtype=np.complex128), tuple(dims_txyz) + (4, 2, 2)).copy()
    return inputs.as_real(U)


def test_su2_plaquette_matches_numpy(oracle):
    U = inputs.make_config_su2(4, 6, 4, 4, 0.5, 3, 4)
    assert abs(oracle.plaquette(inputs.as_real(U)) - plaquettes(U).mean() * 3 / 2) < 1e-14      # helper divides by 3
    assert abs(oracle.plaquette(cold2((4, 4, 4, 4))) - 1.0) < 1e-15


def test_su2_strong_and_weak_coupling(oracle):
    L = inputs.as_real(inputs.make_config_su2(4, 4, 4, 4, 3.0, 9, 10))
    vals = []
    for s in range(45):
        oracle.wilson_heatbath(L, 0.4, seed=11, sweep_index=s)
        if s >= 5:
            vals.append(oracle.plaquette(L))
    assert abs(np.mean(vals) - 0.4 / 4) < 0.005, np.mean(vals)
    L = cold2((4, 4, 4, 4))
    vals = []
    for s in range(40):
        oracle.wilson_heatbath(L, 30.0, seed=13, sweep_index=s)
        if s >= 15:
            vals.append(oracle.plaquette(L))
    assert 0.85 * 3 / (4 * 30.0) < 1 - np.mean(vals) < 1.1 * 3 / (4 * 30.0), 1 - np.mean(vals)
    V = inputs.as_complex(L)
    assert np.abs(V @ dag(V) - np.eye(2)).max() < 1e-13 and np.abs(np.linalg.det(V) - 1).max() < 1e-13
