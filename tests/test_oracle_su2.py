"""Pins of the N_c = 2 oracle (oracle/gf_oracle_su2.hpp) against what the paper
and the mathematics fix, independent of the oracle's own formulas:
  * Step 1 is the maximiser of the local functional: brute force over a dense grid of SU(2)
    (Eq. (18)/(20) PAPER.md:150-159 for Landau/Coulomb, Eq. (21)/(11) PAPER.md:102, 170 for MAG);
  * Eq. (8) == 2 Eq. (11) - 1 on SU(2) links;
  * closed forms on an Abelian field U = exp(i phi sigma_3): F = mean cos phi, Delta = (div phi) sigma_3,
    theta = mean (div phi)^2 (Eqs. (4), (6), (7) with N_c = 2); F_MAG = 1, theta_MAG = 0;
  * every sweep is a gauge transformation (plaquettes, unitarity, det), F is monotone at omega = 1,
    a microcanonical sweep leaves F unchanged, a pure gauge fixes to F = 1;
  * theta_MAG (Eq. (13)) vanishes exactly where a relaxation sweep changes nothing;
  * a Coulomb time-slice is a stand-alone 3-d problem.
"""
import numpy as np
import pytest

from paper_1212_5221_b200 import inputs
from tests.helpers import dag, gather_site, local_landau, local_mag, plaquettes, su2_grid_full

LANDAU, COULOMB, MAG = 0, 1, 2
OR, SR, SA, MICRO = 0, 1, 2, 3


def su2_mat(g):
    g = np.asarray(g, dtype=np.float64)
    m = np.empty(g.shape[:-1] + (2, 2), dtype=np.complex128)
    m[..., 0, 0] = g[..., 0] + 1j * g[..., 3]
    m[..., 0, 1] = g[..., 2] + 1j * g[..., 1]
    m[..., 1, 0] = -g[..., 2] + 1j * g[..., 1]
    m[..., 1, 1] = g[..., 0] - 1j * g[..., 3]
    return m


def config(dims_txyz=(4, 4, 4, 4), eps=0.5, seed=11):
    Nt, Nx, Ny, Nz = dims_txyz
    return inputs.make_config_su2(Nx, Ny, Nz, Nt, eps, seed, seed + 1)


@pytest.mark.parametrize("gauge", [LANDAU, COULOMB, MAG])
def test_step1_is_the_brute_force_maximiser(oracle, gauge):
    U = config(seed=21 + gauge)
    dirs = (1, 2, 3) if gauge == COULOMB else (0, 1, 2, 3)
    grid = su2_grid_full(36)
    G = su2_mat(grid)
    f_loc = local_mag if gauge == MAG else local_landau
    for (t, x, y, z) in [(0, 0, 0, 0), (1, 3, 2, 0), (3, 3, 3, 3)]:
        up, dn = gather_site(U, t, x, y, z, dirs)
        brute = f_loc(G, up, dn).max()
        u, d = inputs.as_real(up), inputs.as_real(dn)
        oracle.site_update(u, d, gauge, OR, 1.0)
        eye = np.eye(2)[None]
        after = f_loc(eye, inputs.as_complex(u), inputs.as_complex(d))[0]
        before = f_loc(eye, up, dn)[0]
        assert after >= brute - 1e-9                      # nothing on the grid beats the closed form
        assert after <= brute + 2e-2 * abs(brute)         # and the grid comes close to it
        assert after >= before - 1e-12
        # after the update the identity is the local maximiser: no grid point improves on it
        assert f_loc(G, inputs.as_complex(u), inputs.as_complex(d)).max() <= after + 1e-9


def test_eq8_is_twice_eq11_minus_one(oracle):
    L = inputs.as_real(config(seed=31))
    m = oracle.measure(L, MAG)
    assert abs(m["F_eq8"] - (2 * m["F"] - 1)) < 1e-14
    # Eq. (11) written out: mean over links of (|U_00|^2 + |U_11|^2) / N_c
    U = inputs.as_complex(L)
    want = (np.abs(U[..., 0, 0]) ** 2 + np.abs(U[..., 1, 1]) ** 2).mean() / 2
    assert abs(m["F"] - want) < 1e-14


def test_abelian_field_closed_forms(oracle):
    rng = np.random.default_rng(5)
    dims = (4, 6, 4, 4)
    phi = rng.uniform(-1, 1, size=dims + (4,))
    U = np.zeros(dims + (4, 2, 2), dtype=np.complex128)
    U[..., 0, 0] = np.exp(1j * phi)
    U[..., 1, 1] = np.exp(-1j * phi)
    L = inputs.as_real(U)
    m = oracle.measure(L, LANDAU)
    assert abs(m["F"] - np.cos(phi).mean()) < 1e-14
    # A_mu = sin(phi_mu) sigma_3; Delta = sum_mu [sin phi_mu(x) - sin phi_mu(x - mu)] sigma_3; tr Delta^2 = 2 d^2
    sp = np.sin(phi)
    div = sum(sp[..., mu] - np.roll(sp[..., mu], 1, axis=mu) for mu in range(4))
    assert abs(m["theta"] - (div ** 2).mean()) < 1e-13
    mc = oracle.measure(L, COULOMB)
    div3 = sum(sp[..., mu] - np.roll(sp[..., mu], 1, axis=mu) for mu in range(1, 4))
    np.testing.assert_allclose(mc["theta_slice"], (div3 ** 2).mean(axis=(1, 2, 3)), atol=1e-13)
    assert abs(mc["F"] - np.cos(phi[..., 1:]).mean()) < 1e-14
    mm = oracle.measure(L, MAG)
    assert abs(mm["F"] - 1.0) < 1e-14 and mm["theta"] < 1e-28 and abs(mm["F_eq8"] - 1.0) < 1e-14
    # diagonal links are a fixed point of the MAG relaxation
    before = L.copy()
    oracle.sweep(L, MAG, OR, 1.0)
    assert np.abs(L - before).max() < 1e-14


@pytest.mark.parametrize("gauge,algo,param", [(LANDAU, OR, 1.7), (COULOMB, OR, 1.0), (MAG, OR, 1.7), (LANDAU, SA, 0.9),
                                              (MAG, SA, 0.7), (COULOMB, SR, 0.5), (MAG, MICRO, 0.0)])
def test_sweep_is_a_gauge_transformation(oracle, gauge, algo, param):
    U = config((4, 4, 6, 4), seed=41)
    L = inputs.as_real(U)
    g = oracle.identity_transform(L)
    oracle.sweep(L, gauge, algo, param, seed=9, sweep_index=2, gtot=g)
    if gauge == COULOMB:
        oracle.coulomb_finalize(L, g)
    V = inputs.as_complex(L)
    assert np.abs(plaquettes(V) - plaquettes(U)).max() < 1e-13
    assert np.abs(V @ dag(V) - np.eye(2)).max() < 1e-13 and np.abs(np.linalg.det(V) - 1).max() < 1e-13
    assert np.abs(V - inputs.gauge_transform(U, inputs.as_complex(g))).max() < 1e-13
    assert np.abs(V - U).max() > 1e-3


@pytest.mark.parametrize("gauge", [LANDAU, COULOMB, MAG])
def test_monotone_relaxation_micro_invariance_and_convergence(oracle, gauge):
    L = inputs.as_real(config(seed=51, eps=0.4))
    F = [oracle.measure(L, gauge)["F"]]
    for s in range(25):
        oracle.sweep(L, gauge, OR, 1.0)
        F.append(oracle.measure(L, gauge)["F"])
    assert np.all(np.diff(F) > -1e-14) and F[-1] > F[0] + 0.05
    oracle.sweep(L, gauge, MICRO, 0.0)
    assert abs(oracle.measure(L, gauge)["F"] - F[-1]) < 1e-13
    s, Ff, th, hist, conv = oracle.run(L, gauge, OR, 1.6, max_sweeps=5000, eps=1e-13)
    assert conv and th < 1e-13 and Ff >= F[-1] - 1e-12
    # at the stationary point a relaxation sweep is the identity (theta = 0 iff stationary)
    before = L.copy()
    oracle.sweep(L, gauge, OR, 1.0)
    assert np.abs(L - before).max() < 1e-5


def test_pure_gauge_fixes_to_one(oracle):
    dims = (4, 4, 4, 4)
    h = inputs.haar_su2(dims, np.random.default_rng(3))
    unit = np.broadcast_to(np.eye(2, dtype=np.complex128), dims + (4, 2, 2)).copy()
    L = inputs.as_real(inputs.gauge_transform(unit, h))
    s, F, th, hist, conv = oracle.run(L, LANDAU, OR, 1.7, max_sweeps=2000, eps=1e-14)
    assert conv and abs(F - 1.0) < 1e-12


def test_theta_mag_nonzero_off_the_stationary_point_and_scales(oracle):
    L = inputs.as_real(config(seed=61))
    m = oracle.measure(L, MAG)
    assert m["theta"] > 1e-3
    # Eq. (12)/(13) written out for one site from the matrices
    U = inputs.as_complex(L)
    s3 = np.diag([1.0, -1.0])
    up, dn = gather_site(U, 2, 1, 3, 0)
    X = sum(u @ s3 @ dag(u) for u in up) + sum(dag(w) @ s3 @ w for w in dn)
    tot = 0.0
    for t in range(4):
        for x in range(4):
            for y in range(4):
                for z in range(4):
                    a, b = gather_site(U, t, x, y, z)
                    Xs = sum(u @ s3 @ dag(u) for u in a) + sum(dag(w) @ s3 @ w for w in b)
                    tot += abs(Xs[0, 1]) ** 2
    assert abs(m["theta"] - tot / (2 * 256)) < 1e-13
    assert abs(X[0, 0] + X[1, 1]) < 1e-13                 # X is traceless Hermitian


def test_coulomb_slice_is_a_standalone_problem(oracle):
    U = config((4, 4, 4, 6), seed=71)
    L = inputs.as_real(U)
    oracle.sweep(L, COULOMB, OR, 1.5)
    m = oracle.measure(L, COULOMB)
    for t in (0, 3):
        # the same slice as a lattice of temporal extent 2 whose two slices are copies of it
        S = np.ascontiguousarray(np.stack([inputs.as_real(U)[t], inputs.as_real(U)[t]]))
        oracle.sweep(S, COULOMB, OR, 1.5)
        assert np.array_equal(S[0][..., 1:, :, :, :], L[t][..., 1:, :, :, :])
        assert abs(oracle.measure(S, COULOMB)["theta_slice"][0] - m["theta_slice"][t]) < 1e-15


def test_haar_su2_moments(oracle):
    h = oracle.haar_field((16, 8, 8, 8), 77, nc=2)
    H = inputs.as_complex(h).reshape(-1, 2, 2)
    n = H.shape[0]
    assert np.abs(H @ dag(H) - np.eye(2)).max() < 1e-14 and np.abs(np.linalg.det(H) - 1).max() < 1e-14
    tr = np.trace(H, axis1=-2, axis2=-1).real               # = 2 q0, q uniform on S^3
    se = 1 / np.sqrt(n)
    assert abs(tr.mean()) < 5 * se                           # E q0 = 0, var(2 q0) = 1
    assert abs((tr ** 2).mean() - 1.0) < 5 * se              # E (tr h)^2 = 1 (one singlet in 2 x 2)
    assert abs((tr ** 4).mean() - 2.0) < 10 * se             # E (tr h)^4 = 2 (Catalan number)
    assert np.abs((np.abs(H) ** 2).mean(axis=0) - 0.5).max() < 5 * se


def test_mixed_precision_and_float_paths_follow_double(oracle):
    U = config(seed=81)
    Ld, Lf, Lm = inputs.as_real(U), inputs.as_real(U, np.float32), inputs.as_real(U, np.float32)
    for s in range(3):
        oracle.sweep(Ld, LANDAU, OR, 1.7)
        oracle.sweep(Lf, LANDAU, OR, 1.7)
        oracle.sweep(Lm, LANDAU, OR, 1.7, mixed=True)
    assert np.abs(Lf - Ld).max() < 5e-5 and np.abs(Lm - Ld).max() < 5e-5
    oracle.reunitarize(Lf)
    V = inputs.as_complex(Lf)
    assert np.abs(V @ dag(V) - np.eye(2)).max() < 3e-7
