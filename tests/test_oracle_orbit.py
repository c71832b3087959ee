"""Pins of the oracle's random start on the gauge orbit (R27) and of the
SA -> SR -> OR recipe, against what the mathematics fixes:
  Haar measure on SU(3): h unitary, det h = 1, E|h_ij|^2 = 1/3, E tr h = 0, E|tr h|^2 = 1,
  E (tr h)^3 = 1 (the epsilon-tensor invariant: 0 on U(3), 1 on SU(3)), E|tr h|^4 = 2;
  Eq. (1): every plaquette is unchanged by a gauge transformation; each link is h(x) U h(x+mu)^dag;
  the recipe is the composition of its (separately pinned) stages.
"""
import numpy as np
import pytest

from paper_1212_5221_b200 import inputs
from tests.helpers import plaquettes

LANDAU, COULOMB, MAG = 0, 1, 2
OR, SR, SA, MICRO = 0, 1, 2, 3


def cplx(a):
    return a[..., 0] + 1j * a[..., 1]


def test_haar_field_is_special_unitary(oracle):
    H = cplx(oracle.haar_field((4, 4, 6, 4), 12))
    eye = np.eye(3)
    assert np.abs(H @ np.conj(np.swapaxes(H, -1, -2)) - eye).max() < 1e-14
    assert np.abs(np.linalg.det(H) - 1).max() < 1e-14


def test_haar_field_moments(oracle):
    H = cplx(oracle.haar_field((16, 8, 8, 8), 2024)).reshape(-1, 3, 3)     # 8192 samples
    n = H.shape[0]
    tr = np.trace(H, axis1=-2, axis2=-1)
    se = 1.0 / np.sqrt(n)
    assert np.abs((np.abs(H) ** 2).mean(axis=0) - 1 / 3).max() < 5 * 0.25 * se      # var |h_ij|^2 < 1/16
    assert abs(tr.mean()) < 5 * se
    assert abs((np.abs(tr) ** 2).mean() - 1.0) < 5 * 1.0 * se                     # var |tr|^2 = 2 - 1
    assert abs((tr ** 3).mean() - 1.0) < 5 * np.sqrt(6.0) * se                     # E|tr|^6 = 6 on SU(3)
    assert abs((np.abs(tr) ** 4).mean() - 2.0) < 0.25
    # rows are exchangeable and there is no preferred phase: E h_ij = 0, E h_ij h_kl = 0
    assert np.abs(H.mean(axis=0)).max() < 5 * se
    assert abs((H[:, 0, 0] * H[:, 1, 1]).mean()) < 5 * se


def test_haar_field_depends_on_seed_and_site_only(oracle):
    a = oracle.haar_field((4, 4, 4, 4), 5)
    b = oracle.haar_field((4, 4, 4, 4), 5)
    c = oracle.haar_field((4, 4, 4, 4), 6)
    assert np.array_equal(a, b) and np.abs(a - c).max() > 0.1
    # counter = lexicographic site index: the first 4*4*4*2 sites of a longer lattice are the same field
    d = oracle.haar_field((4, 4, 4, 4), 5).reshape(-1, 18)
    e = oracle.haar_field((8, 4, 4, 4), 5).reshape(-1, 18)
    assert np.array_equal(d, e[:d.shape[0]])


def test_gauge_transform_is_eq1(oracle):
    dims = (4, 4, 6, 4)     # t, x, y, z
    U = inputs.make_config(dims[1], dims[2], dims[3], dims[0], 0.5, 31, 32)
    L = inputs.as_real(U)
    h = oracle.haar_field(dims, 9)
    H = cplx(h)
    oracle.gauge_transform(L, h)
    V = inputs.as_complex(L)
    # one link written out: U_2(x) at x = (1,2,5,3) -> h(x) U h(x + y_hat)^dagger, periodic in y
    t, x, y, z = 1, 2, 5, 3
    want = H[t, x, y, z] @ U[t, x, y, z, 2] @ np.conj(H[t, x, 0, z]).T
    assert np.abs(V[t, x, y, z, 2] - want).max() < 1e-14
    assert np.abs(plaquettes(V) - plaquettes(U)).max() < 1e-13
    assert abs(oracle.measure(L, LANDAU)["F"] - oracle.measure(inputs.as_real(U), LANDAU)["F"]) > 1e-3


def test_random_gauge_tracks_the_transform(oracle):
    dims = (4, 4, 4, 6)
    U = inputs.make_config(dims[1], dims[2], dims[3], dims[0], 0.4, 41, 42)
    L = inputs.as_real(U)
    g = oracle.identity_transform(L)
    oracle.random_gauge(L, 3, g)
    oracle.random_gauge(L, 4, g)       # g accumulates: g <- h g
    want = inputs.gauge_transform(U, cplx(g))
    assert np.abs(inputs.as_complex(L) - want).max() < 1e-13


def test_fix_is_the_composition_of_its_stages(oracle):
    U = inputs.config_k(0)
    kw = dict(seed=8, sa_steps=5, sa_T_hi=0.7, sa_T_lo=0.05, sa_micro=2, sr_max_sweeps=15, sr_p=0.4,
              or_omega=1.7, or_max_sweeps=2000, eps=1e-12, check_every=2)
    A = inputs.as_real(U)
    tot, F, th, conv = oracle.fix(A, LANDAU, **kw)
    B = inputs.as_real(U)
    nxt = oracle.anneal(B, LANDAU, 0.7, 0.05, 5, 2, 8)
    s2, F2, th2, _, c2 = oracle.run(B, LANDAU, SR, 0.4, 8, 15, 1e-12, 2, first_sweep_index=nxt)
    s3 = 0
    if not c2:
        s3, F2, th2, _, c2 = oracle.run(B, LANDAU, OR, 1.7, 8, 2000, 1e-12, 2, first_sweep_index=nxt)
    assert conv and c2 and tot == nxt + s2 + s3 and F == F2 and th == th2
    assert np.array_equal(A, B)
    assert th < 1e-12
    # the result is on the orbit of the input and has a larger functional
    assert np.abs(plaquettes(inputs.as_complex(A)) - plaquettes(U)).max() < 1e-12
    assert F > oracle.measure(inputs.as_real(U), LANDAU)["F"] + 0.1


def test_fix_without_annealing_is_run(oracle):
    U = inputs.config_k(0)
    A, B = inputs.as_real(U), inputs.as_real(U)
    tot, F, th, conv = oracle.fix(A, MAG, or_omega=1.6, or_max_sweeps=3000, eps=1e-11)
    s, F2, th2, _, c2 = oracle.run(B, MAG, OR, 1.6, max_sweeps=3000, eps=1e-11)
    assert (tot, F, th, conv) == (s, F2, th2, c2) and np.array_equal(A, B)


def test_annealing_only_reports_the_measured_state(oracle):
    U = inputs.config_k(0)
    A, B = inputs.as_real(U), inputs.as_real(U)
    tot, F, th, conv = oracle.fix(A, LANDAU, seed=3, sa_steps=4, sa_T_hi=0.5, sa_T_lo=0.1, sa_micro=1, or_max_sweeps=0)
    nxt = oracle.anneal(B, LANDAU, 0.5, 0.1, 4, 1, 3)
    m = oracle.measure(B, LANDAU)
    assert tot == nxt == 8 and not conv and F == m["F"] and th == m["theta"] and np.array_equal(A, B)
