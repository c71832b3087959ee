"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Each test names the passage of /root/reference/PAPER.md (or the DESIGN.md reading) it pins.
Nothing here re-types the oracle's formulas: expected values come from closed forms, gauge
invariants, brute force over dense SU(2) grids, analytic densities, or published known answers.
"""
import os

import numpy as np
import pytest
from scipy import special

from paper_1212_5221_b200 import inputs
from tests import helpers as H

LANDAU, COULOMB, MAG = 0, 1, 2
OR, SR, SA, MICRO = 0, 1, 2, 3
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def small_config(seed=11, dims=(4, 4, 4, 4), eps=0.5):
    return inputs.make_config(dims[0], dims[1], dims[2], dims[3], eps, seed, seed + 1)


# ------------------------------------------------------------------------------------------
# Philox (PAPER.md:249 fn. 2): published known answers
# ------------------------------------------------------------------------------------------
def test_philox_known_answers(oracle):
    n = 0
    for line in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(t, 16) for t in line.split()]
        got = oracle.philox4x32_10(w[0:4], w[4:6])
        assert [int(v) for v in got] == w[6:10]
        n += 1
    assert n == 3


def test_philox_uniform_mapping_and_keying(oracle):
    # (u32 + 0.5) * 2^-32 in (0,1) (R19); counter = (site, sweep, sub | purpose<<8, trial)
    words, uni = oracle.draw(seed=(7 << 32) | 5, site=123, sweep=9, sub=2, purpose=1, trial=4)
    ref = oracle.philox4x32_10([123, 9, 2 | (1 << 8), 4], [5, 7])
    assert list(words) == list(ref)
    assert np.all(uni == (words.astype(np.float64) + 0.5) / 2.0 ** 32)
    assert np.all((uni > 0) & (uni < 1))
    # statistical sanity: mean 1/2, variance 1/12 over many counters
    u = np.array([oracle.draw(1234, s, 0, 0, 0, 0)[1] for s in range(4000)]).ravel()
    assert abs(u.mean() - 0.5) < 0.01 and abs(u.var() - 1 / 12) < 0.005


# ------------------------------------------------------------------------------------------
# F and theta: closed forms (Eqs. 4, 6, 7, 11)
# ------------------------------------------------------------------------------------------
def test_measure_closed_form_abelian_field(oracle):
    # U_mu(x) = diag(e^{i phi}, e^{-i phi}, 1): A_mu = diag(sin phi, -sin phi, 0) is already traceless,
    # Delta(x) = sum_mu (sin phi_mu(x) - sin phi_mu(x-mu)) diag(1,-1,0), tr[Delta Delta^dag] = 2 (...)^2.
    rng = np.random.default_rng(5)
    dims = (4, 6, 2, 8)
    phi = rng.uniform(-1.0, 1.0, size=dims + (4,))
    U = np.zeros(dims + (4, 3, 3), dtype=np.complex128)
    U[..., 0, 0] = np.exp(1j * phi)
    U[..., 1, 1] = np.exp(-1j * phi)
    U[..., 2, 2] = 1
    V = np.prod(dims)
    s = np.sin(phi)
    for gauge, dirs in ((LANDAU, (0, 1, 2, 3)), (COULOMB, (1, 2, 3))):
        div = sum(s[..., mu] - np.roll(s[..., mu], 1, axis=mu) for mu in dirs)
        theta = 2.0 * (div ** 2).sum() / (3 * V)
        F = sum((2 * np.cos(phi[..., mu]) + 1).sum() for mu in dirs) / (3 * len(dirs) * V)
        m = oracle.measure(inputs.as_real(U), gauge)
        assert m["F"] == pytest.approx(F, rel=1e-14)
        assert m["theta"] == pytest.approx(theta, rel=1e-13)
        Vs = V / dims[0]
        th_t = 2.0 * (div ** 2).sum(axis=(1, 2, 3)) / (3 * Vs)
        np.testing.assert_allclose(m["theta_slice"], th_t, rtol=1e-13)
    # MAG: diagonal links maximise Eq. (11): F = 1, theta = 0
    m = oracle.measure(inputs.as_real(U), MAG)
    assert m["F"] == pytest.approx(1.0, abs=1e-15) and m["theta"] < 1e-30


def test_measure_trace_part_removed(oracle):
    # A is the *traceless* anti-Hermitian part (R8): a centre-like phase e^{i a} on every
    # link in one direction gives (U - U^dag)/2i = sin(a) 1, whose traceless part vanishes -> theta = 0
    dims = (2, 2, 2, 2)
    rng = np.random.default_rng(1)
    a = rng.uniform(-0.5, 0.5, size=dims + (4,))
    U = np.exp(1j * a)[..., None, None] * np.eye(3)
    m = oracle.measure(inputs.as_real(U), LANDAU)
    assert m["theta"] < 1e-30
    assert m["F"] == pytest.approx(np.cos(a).mean(), rel=1e-14)


def test_mag_functional_closed_form(oracle):
    # links = SU(2) rotation by angle w in the (0,1) block: sum_i |U_ii|^2 = 2 cos^2 w + 1
    dims = (2, 2, 2, 2)
    rng = np.random.default_rng(2)
    w = rng.uniform(0, np.pi, size=dims + (4,))
    g = np.stack([np.cos(w), np.zeros_like(w), np.sin(w), np.zeros_like(w)], -1)
    U = H.embed_su2(g, 0, 1)
    m = oracle.measure(inputs.as_real(U), MAG)
    assert m["F"] == pytest.approx(((2 * np.cos(w) ** 2 + 1).mean()) / 3.0, rel=1e-14)


# ------------------------------------------------------------------------------------------
# Step 1 by brute force on one site (Eq. 20; Eq. 29; Fig. A.10)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("sub", [(0, 1), (0, 2), (1, 2)])
def test_step1_landau_bruteforce(oracle, sub):
    U = small_config(21)
    up, dn = H.gather_site(U, 1, 2, 3, 0)
    i, j = sub
    a = oracle.local_quaternion(H.to_real(up), H.to_real(dn), i, j)
    g = oracle.rule_or(a, 1.0)
    assert abs(np.dot(g, g) - 1) < 1e-14
    f_star = H.local_landau(H.embed_su2(g, i, j), up, dn)
    grid = H.su2_grid_full(48)
    f_grid = H.local_landau(H.embed_su2(grid, i, j), up, dn)
    assert f_star >= f_grid.max() - 1e-12          # nothing on the grid beats the closed form
    assert f_star - f_grid.max() < 5e-3 * abs(f_star)   # and the grid comes close to it
    # the value of the maximum: f = K_kk-term + |a|   (|a| un-halved, Fig. A.10 restored signs)
    K = up.sum(0) + H.dag(dn).sum(0)
    k = 3 - i - j
    assert f_star == pytest.approx(K[k, k].real + np.linalg.norm(a), rel=1e-13)
    # stationarity: small rotations about the maximiser only decrease f
    for axis in range(1, 4):
        for sgn in (-1, 1):
            d = np.zeros(4); d[0] = np.cos(1e-3); d[axis] = sgn * np.sin(1e-3)
            gm = H.embed_su2(d, i, j) @ H.embed_su2(g, i, j)
            assert H.local_landau(gm, up, dn) < f_star


@pytest.mark.parametrize("sub", [(0, 1), (0, 2), (1, 2)])
def test_step1_mag_bruteforce(oracle, sub):
    U = small_config(22)
    up, dn = H.gather_site(U, 3, 0, 1, 2)
    i, j = sub
    D, E, F = oracle.local_mag_def(H.to_real(up), H.to_real(dn), i, j)
    lam = np.sqrt(D * D + E * E + F * F)
    # quadratic form reproduces Eq. (11) on g3 = 0 (Eqs. 24-25 generalised): f = c + g^T A g
    rng = np.random.default_rng(0)
    v = rng.standard_normal((200, 3)); v /= np.linalg.norm(v, axis=1, keepdims=True)
    g = np.concatenate([v, np.zeros((200, 1))], axis=1)
    f = H.local_mag(H.embed_su2(g, i, j), up, dn)
    A = np.array([[D, E, F], [E, -D, 0], [F, 0, -D]])
    quad = np.einsum("na,ab,nb->n", v, A, v)
    const = f - quad
    assert np.ptp(const) < 1e-12
    # closed-form maximum (Eq. 29) beats a dense grid over *all* of SU(2), g3 != 0 included
    a = np.array([D + lam, -E, -F, 0.0])
    gs = oracle.rule_or(a, 1.0)
    np.testing.assert_allclose(gs, np.array([D + lam, E, F, 0]) / np.linalg.norm([D + lam, E, F]), atol=1e-14)
    f_star = H.local_mag(H.embed_su2(gs, i, j), up, dn)
    assert f_star == pytest.approx(const.mean() + lam, rel=1e-13)
    f_grid = H.local_mag(H.embed_su2(H.su2_grid_full(40), i, j), up, dn)
    assert f_star >= f_grid.max() - 1e-12
    assert f_star - f_grid.max() < 5e-3 * abs(f_star)


def test_eq26_factor_two_reading(oracle):
    # DESIGN.md R12b: with D as printed in Eq. (26) (half of ours) Eq. (29) is not the maximiser.
    U = small_config(23)
    up, dn = H.gather_site(U, 0, 0, 0, 0)
    D, E, F = oracle.local_mag_def(H.to_real(up), H.to_real(dn), 0, 1)
    def fval(Dx):
        lam = np.sqrt(Dx * Dx + E * E + F * F)
        g = np.array([Dx + lam, E, F, 0.0]); g /= np.linalg.norm(g)
        return H.local_mag(H.embed_su2(g, 0, 1), up, dn)
    assert fval(D) > fval(D / 2) + 1e-6


def test_or_rule_limits(oracle):
    # Fig. A.11: omega=1 -> Eq. (20); small angles: rotation angle scales by omega
    rng = np.random.default_rng(3)
    a = rng.standard_normal(4)
    g1 = oracle.rule_or(a, 1.0)
    np.testing.assert_allclose(g1, np.array([a[0], -a[1], -a[2], -a[3]]) / np.linalg.norm(a), atol=1e-15)
    a = np.array([1.0, 1e-4, -2e-4, 0.5e-4])
    for om in (1.3, 1.7, 1.95):
        g = oracle.rule_or(a, om)
        assert abs(np.dot(g, g) - 1) < 1e-14
        np.testing.assert_allclose(g[1:], -om * a[1:], rtol=1e-6)   # tan(phi') ~ omega * phi
    # unit norm for any omega, any a
    for _ in range(20):
        a = rng.standard_normal(4) * 10
        g = oracle.rule_or(a, 1.7)
        assert abs(np.dot(g, g) - 1) < 1e-14


def test_micro_is_exact_square(oracle):
    # PAPER.md:222-224 + DESIGN.md R4: g^2 of the maximiser, via the 2x2 matrices of Eq. (22)
    rng = np.random.default_rng(4)
    a = rng.standard_normal(4)
    g1 = oracle.rule_or(a, 1.0)
    g2 = oracle.rule_micro(a)
    m1 = H.embed_su2(g1, 0, 1)
    np.testing.assert_allclose(H.embed_su2(g2, 0, 1), m1 @ m1, atol=1e-15)


def test_apply_subgroup_matches_eq1(oracle):
    # Step 2 (Fig. A.9 caption): U <- g~ U and U <- U g~^dag with g~ of Eq. (22)
    rng = np.random.default_rng(6)
    M = rng.standard_normal((3, 3)) + 1j * rng.standard_normal((3, 3))
    g = rng.standard_normal(4); g /= np.linalg.norm(g)
    for (i, j) in ((0, 1), (0, 2), (1, 2)):
        gm = H.embed_su2(g, i, j)
        np.testing.assert_allclose(H.cplx(oracle.apply_subgroup(H.to_real(M), g, i, j)), gm @ M, atol=1e-15)
        np.testing.assert_allclose(H.cplx(oracle.apply_subgroup(H.to_real(M), g, i, j, True)), M @ H.dag(gm), atol=1e-15)
        assert abs(np.linalg.det(gm) - 1) < 1e-15


# ------------------------------------------------------------------------------------------
# Whole-sweep invariants (PAPER.md:23-27 gauge invariance; 416-422 unitarity; 430 monotone F)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gauge", [LANDAU, COULOMB, MAG])
@pytest.mark.parametrize("algo,param", [(OR, 1.7), (OR, 1.0), (SR, 0.5), (SA, 0.8), (MICRO, 0.0)])
def test_sweep_is_a_gauge_transformation(oracle, gauge, algo, param):
    U0 = small_config(31, dims=(4, 6, 4, 2))
    L = inputs.as_real(U0)
    G = oracle.identity_transform(L)
    P0 = H.plaquettes(U0)
    for s in range(3):
        oracle.sweep(L, gauge, algo, param, seed=99, sweep_index=s, gtot=G)
    U1 = H.cplx(L)
    # plaquette invariance to 1e-12 (BASELINE.json north_star); during Coulomb sweeps only the
    # spatial plaquettes (orientations 3..5), the temporal links follow in the finalisation step
    psel = slice(3, 6) if gauge == COULOMB else slice(0, 6)
    assert np.abs(H.plaquettes(U1) - P0)[psel].max() < 1e-12
    # unitarity and det = 1 after every sweep (Eq. 33)
    assert np.abs(U1 @ H.dag(U1) - np.eye(3)).max() < 1e-12
    assert np.abs(np.linalg.det(U1) - 1).max() < 1e-12
    # the accumulated g(x) reproduces the links through Eq. (1): U^g = g(x) U g(x+mu)^dag
    g = H.cplx(G)
    assert np.abs(g @ H.dag(g) - np.eye(3)).max() < 1e-12
    msel = slice(1, 4) if gauge == COULOMB else slice(0, 4)
    np.testing.assert_allclose(U1[..., msel, :, :], inputs.gauge_transform(U0, g)[..., msel, :, :], atol=1e-12)
    if gauge == COULOMB:   # temporal links untouched during Coulomb sweeps
        assert np.array_equal(U1[..., 0, :, :], U0[..., 0, :, :])


@pytest.mark.parametrize("gauge", [LANDAU, COULOMB, MAG])
def test_relaxation_monotone_F(oracle, gauge):
    L = inputs.as_real(small_config(32))
    F_prev = oracle.measure(L, gauge)["F"]
    for s in range(25):
        oracle.sweep(L, gauge, OR, 1.0)
        F = oracle.measure(L, gauge)["F"]
        assert F >= F_prev - 1e-15
        F_prev = F
    # each half sweep alone is monotone too
    for p in (1, 2, 1, 2):
        oracle.sweep(L, gauge, OR, 1.0, parity_mask=p)
        F = oracle.measure(L, gauge)["F"]
        assert F >= F_prev - 1e-15
        F_prev = F


@pytest.mark.parametrize("gauge", [LANDAU, COULOMB, MAG])
def test_micro_sweep_preserves_F(oracle, gauge):
    # microcanonical steps leave the functional invariant (exact g^2, R4/R13)
    L = inputs.as_real(small_config(33))
    F0 = oracle.measure(L, gauge)["F"]
    for s in range(5):
        oracle.sweep(L, gauge, MICRO, 0.0)
        assert abs(oracle.measure(L, gauge)["F"] - F0) < 1e-13
    assert np.abs(H.cplx(L) - small_config(33)).max() > 0.1   # but the links do move


def test_pure_gauge_fixes_to_unit_links(oracle):
    # BASELINE.json: U_mu(x) = h(x) h(x+mu)^dag must fix to F = 1, theta -> 0
    for omega, nmax in ((1.0, 200), (1.7, 400)):
        L = inputs.as_real(inputs.pure_gauge((4, 4, 4, 4), 7))
        s, F, th, hist, conv = oracle.run(L, LANDAU, OR, omega, max_sweeps=nmax, eps=1e-14)
        assert conv and abs(F - 1) < 1e-13 and th < 1e-14
        U = H.cplx(L)
        # all links equal one constant centre-free matrix? No: F=1 forces U = 1 exactly
        assert np.abs(U - np.eye(3)).max() < 1e-6
    L = inputs.as_real(inputs.pure_gauge((4, 4, 4, 4), 8))
    s, F, th, hist, conv = oracle.run(L, COULOMB, OR, 1.0, max_sweeps=300, eps=1e-14)
    assert conv and abs(F - 1) < 1e-13
    L = inputs.as_real(inputs.pure_gauge((4, 4, 4, 4), 9))
    s, F, th, hist, conv = oracle.run(L, MAG, OR, 1.0, max_sweeps=3000, eps=1e-14)
    assert conv and abs(F - 1) < 1e-12


def test_config0_converges_like_the_survey_says(oracle):
    # BASELINE.json config 0 (4^4, eps=0.3, omega=1.7, theta<1e-12 within 2000 sweeps).
    L = inputs.as_real(inputs.config_k(0))
    m0 = oracle.measure(L, LANDAU)
    assert abs(m0["F"]) < 0.05 and 2.0 < m0["theta"] < 5.0      # Haar-transformed start
    s, F, th, hist, conv = oracle.run(L, LANDAU, OR, 1.7, max_sweeps=2000, eps=1e-12)
    assert conv and s < 200 and 0.93 < F < 0.98
    Fs = [h[1] for h in hist]
    assert all(b >= a - 1e-14 for a, b in zip(Fs, Fs[1:]))      # monotone here
    # relaxation (omega=1) reaches the same Gribov copy on this small lattice
    L1 = inputs.as_real(inputs.config_k(0))
    s1, F1, th1, _, conv1 = oracle.run(L1, LANDAU, OR, 1.0, max_sweeps=2000, eps=1e-12)
    assert conv1


def test_theta_zero_iff_stationary_mag(oracle):
    # DESIGN.md R11: stopping theta = sum_s |X^s_12|^2 vanishes exactly when OR stalls
    L = inputs.as_real(small_config(35))
    s, F, th, hist, conv = oracle.run(L, MAG, OR, 1.7, max_sweeps=4000, eps=1e-13)
    assert conv
    before = L.copy()
    oracle.sweep(L, MAG, OR, 1.0)
    assert np.abs(L - before).max() < 1e-5
    m = oracle.measure(L, MAG)
    assert m["theta_literal"] <= 3 * m["theta"] + 1e-30


def _x_mag(U, sigma):
    """X(x) = sum_mu [ U_mu(x) sigma U_mu(x)^dag + U_mu(x-mu)^dag sigma U_mu(x-mu) ] of Eq. (12) at
    every site, from the complex links U[t,x,y,z,mu,n,n]; sigma a diagonal matrix.  Returns [t,x,y,z,n,n]."""
    X = 0
    for mu in range(4):
        W = U[..., mu, :, :]
        Wd = np.roll(W, 1, axis=mu)                      # U_mu(x - mu)
        X = X + W @ sigma @ H.dag(W) + H.dag(Wd) @ sigma @ Wd
    return X


def test_theta_mag_su3_from_eq12_matrices(oracle):
    # Eqs. (12), (13), (16) in the reading R11: for the subgroup s = (i,j) sigma_3 is the 3x3
    # matrix diag(+1 at i, -1 at j); X^s(x) is Eq. (12) with it, its (i,j) element the quantity whose modulus
    # squared enters theta.  Stopping theta = sum_x sum_s |X^s_ij|^2 / (N_c V); the literal Eq. (16) puts the sum
    # over s inside the modulus.  Everything below is NumPy matrix algebra on a rough random field: a wrong
    # prefactor, a dropped subgroup, a dropped up/down term or a transposed link fails it.
    dims = (4, 4, 4, 6)
    U = small_config(36, dims=dims, eps=0.6)
    V = int(np.prod(dims))
    tot = 0.0
    lit = 0
    for (i, j) in ((0, 1), (0, 2), (1, 2)):
        sig = np.zeros((3, 3))
        sig[i, i], sig[j, j] = 1.0, -1.0
        X = _x_mag(U, sig)
        assert np.abs(X - H.dag(X)).max() < 1e-13 and np.abs(np.trace(X, axis1=-2, axis2=-1)).max() < 1e-13
        tot += (np.abs(X[..., i, j]) ** 2).sum()
        lit = lit + X[..., i, j]
    m = oracle.measure(inputs.as_real(U), MAG)
    assert m["theta"] > 1e-2                              # far from stationary: a non-trivial expected value
    assert m["theta"] == pytest.approx(tot / (3 * V), rel=1e-13)
    assert m["theta_literal"] == pytest.approx((np.abs(lit) ** 2).sum() / (3 * V), rel=1e-13)
    # the per-slice values are the same sums restricted to a slice (V -> Nx Ny Nz)
    th_t = 0
    for (i, j) in ((0, 1), (0, 2), (1, 2)):
        sig = np.zeros((3, 3))
        sig[i, i], sig[j, j] = 1.0, -1.0
        th_t = th_t + (np.abs(_x_mag(U, sig)[..., i, j]) ** 2).sum(axis=(1, 2, 3))
    assert np.allclose(m["theta_slice"], th_t / (3 * V / U.shape[0]), rtol=1e-13, atol=0)


def test_theta_mag_su3_reduces_to_su2_on_embedded_links(oracle):
    # links that are SU(2) matrices in the (0,1) block of the 3x3 identity: the subgroups (0,2) and (1,2) see
    # diagonal blocks (X^s_ij = 0) and the (0,1) subgroup sees the SU(2) problem, so the N_c = 3 value is the
    # N_c = 2 oracle's theta (pinned by Eq. (12)/(13) in tests/test_oracle_su2.py) times 2/3; F of Eq. (11):
    # 3 F_3 = 2 F_2 + 1 per link
    dims = (4, 4, 4, 4)
    u = inputs.make_config_su2(*dims, 0.5, 81, 82)
    U = np.zeros(dims + (4, 3, 3), dtype=np.complex128)
    U[..., :2, :2] = u
    U[..., 2, 2] = 1.0
    m3 = oracle.measure(inputs.as_real(U), MAG)
    m2 = oracle.measure(inputs.as_real(u), MAG)
    assert m2["theta"] > 1e-3
    assert m3["theta"] == pytest.approx(2.0 * m2["theta"] / 3.0, rel=1e-13)
    assert m3["theta_literal"] == pytest.approx(m3["theta"], rel=1e-13)
    assert m3["F"] == pytest.approx((2.0 * m2["F"] + 1.0) / 3.0, rel=1e-13)


# ------------------------------------------------------------------------------------------
# Coulomb: time-slices are independent problems (R21/R22)
# ------------------------------------------------------------------------------------------
def test_coulomb_slices_independent(oracle):
    U = small_config(41, dims=(4, 4, 4, 4))
    V = small_config(42, dims=(4, 4, 4, 4))
    mix = V.copy()
    mix[2] = U[2]                      # same slice t=2, everything else different
    A, B = inputs.as_real(U), inputs.as_real(mix)
    for s in range(3):
        oracle.sweep(A, COULOMB, OR, 1.7)
        oracle.sweep(B, COULOMB, OR, 1.7)
    assert np.array_equal(A[2][..., 1:, :, :, :], B[2][..., 1:, :, :, :])
    mA, mB = oracle.measure(A, COULOMB), oracle.measure(B, COULOMB)
    assert mA["theta_slice"][2] == mB["theta_slice"][2]


def test_coulomb_freeze_is_one_standalone_run_per_slice(oracle):
    # the paper fixes one slice at a time.  The frozen run of the whole lattice must give,
    # in slice t, bit for bit what the plain run loop gives on a lattice made of slice t alone (all its
    # slices then converge at the same check), with the same sweep count; slices stop at different sweeps.
    U = small_config(44, dims=(4, 4, 4, 4), eps=0.6)
    L = inputs.as_real(U)
    G = oracle.identity_transform(L)
    s, F, th, hist, conv, ss = oracle.run_coulomb_freeze(L, OR, 1.7, max_sweeps=2000, eps=1e-12, check_every=3,
                                                         gtot=G)
    assert conv and th < 1e-12 and s == ss.max() and len(set(ss.tolist())) > 1
    for t in range(4):
        one = inputs.as_real(np.stack([U[t], U[t]]))
        g1 = oracle.identity_transform(one)
        s1, F1, th1, h1, c1 = oracle.run(one, COULOMB, OR, 1.7, max_sweeps=2000, eps=1e-12, check_every=3, gtot=g1)
        assert c1 and s1 == ss[t]
        assert np.array_equal(one[0][..., 1:, :, :, :], L[t][..., 1:, :, :, :])
        assert np.array_equal(g1[0], G[t])
    # temporal links untouched until finalisation; afterwards the whole field is a gauge transform of U
    assert np.array_equal(L[..., 0, :, :, :], inputs.as_real(U)[..., 0, :, :, :])
    oracle.coulomb_finalize(L, G)
    np.testing.assert_allclose(H.plaquettes(H.cplx(L)), H.plaquettes(U), atol=1e-12)


def test_coulomb_finalize_keeps_all_plaquettes(oracle):
    U0 = small_config(43)
    L = inputs.as_real(U0)
    G = oracle.identity_transform(L)
    s, F, th, hist, conv = oracle.run(L, COULOMB, OR, 1.7, max_sweeps=500, eps=1e-12, gtot=G)
    assert conv and max(h[2] for h in hist[-1:]) < 1e-12
    # before finalisation the temporal plaquettes are broken (spatial links rotated, U_0 not)
    assert np.abs(H.plaquettes(H.cplx(L)) - H.plaquettes(U0)).max() > 1e-3
    oracle.coulomb_finalize(L, G)
    np.testing.assert_allclose(H.plaquettes(H.cplx(L)), H.plaquettes(U0), atol=1e-12)
    np.testing.assert_allclose(H.cplx(L), inputs.gauge_transform(U0, H.cplx(G)), atol=1e-12)
    # Coulomb gauge condition per slice: theta_t all below eps
    assert oracle.measure(L, COULOMB)["theta_slice"].max() < 1e-12


# ------------------------------------------------------------------------------------------
# Heatbath (Eq. 30; R14/R15) and stochastic relaxation
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("alpha", [0.5, 1.5, 3.0, 8.0, 60.0])
def test_heatbath_landau_distribution(oracle, alpha):
    # u0 = g . g_hat has density sqrt(1-u0^2) exp(alpha u0): mean I2(alpha)/I1(alpha),
    # second moment 1 - 3 I2/(alpha I1); the direction of the rest is uniform.
    rng = np.random.default_rng(8)
    a = rng.standard_normal(4); a *= 2.0 / np.linalg.norm(a)
    T = np.linalg.norm(a) / alpha
    ghat = np.array([a[0], -a[1], -a[2], -a[3]]) / np.linalg.norm(a)
    n = 6000
    gs = np.array([oracle.rule_heatbath_landau(a, T, 4321, site, 3, 1) for site in range(n)])
    np.testing.assert_allclose((gs ** 2).sum(1), 1.0, atol=1e-13)
    u0 = gs @ ghat
    r = special.ive(2, alpha) / special.ive(1, alpha)
    var = (1 - 3 * r / alpha) - r * r
    assert abs(u0.mean() - r) < 5 * np.sqrt(var / n) + 1e-4
    assert abs((u0 ** 2).mean() - (1 - 3 * r / alpha)) < 0.02
    # components orthogonal to g_hat average to zero (uniform direction)
    perp = gs - np.outer(u0, ghat)
    assert np.abs(perp.mean(0)).max() < 5 * np.sqrt((1 - (u0 ** 2).mean()) / 3 / n) + 1e-3


def test_heatbath_zero_temperature_is_relaxation(oracle):
    # (over)relaxation = simulated annealing at T -> 0
    rng = np.random.default_rng(9)
    a = rng.standard_normal(4)
    g = oracle.rule_heatbath_landau(a, 1e-9, 1, 2, 3, 0)
    np.testing.assert_allclose(g, oracle.rule_or(a, 1.0), atol=1e-4)
    D, E, F = 0.3, -0.2, 0.5
    lam = np.sqrt(D * D + E * E + F * F)
    g = oracle.rule_heatbath_mag(D, E, F, 1e-9, 1, 2, 3, 0)
    ref = np.array([D + lam, E, F, 0.0]); ref /= np.linalg.norm(ref)
    np.testing.assert_allclose(g, ref, atol=1e-4)


@pytest.mark.parametrize("kappa", [0.3, 2.0, 15.0])
def test_heatbath_mag_distribution(oracle, kappa):
    # phi ~ exp(phi.X/T) uniformly on S^2: <cos gamma> = coth(k) - 1/k (Langevin), k = lambda/T
    D, E, F = 0.4, 0.7, -0.3
    lam = np.sqrt(D * D + E * E + F * F)
    T = lam / kappa
    n = 6000
    gs = np.array([oracle.rule_heatbath_mag(D, E, F, T, 77, site, 0, 2) for site in range(n)])
    assert np.all(gs[:, 3] == 0) and np.all(gs[:, 0] >= 0)
    np.testing.assert_allclose((gs ** 2).sum(1), 1.0, atol=1e-13)
    # local functional difference f(g) - const = g^T A g = phi . X
    val = D * (gs[:, 0] ** 2 - gs[:, 1] ** 2 - gs[:, 2] ** 2) + 2 * gs[:, 0] * (gs[:, 1] * E + gs[:, 2] * F)
    cosg = val / lam
    lang = 1 / np.tanh(kappa) - 1 / kappa
    var = 1 - 2 * lang / kappa - lang ** 2
    assert abs(cosg.mean() - lang) < 5 * np.sqrt(var / n) + 1e-4
    # azimuth about X is uniform: the part of phi orthogonal to X averages to zero
    phi = np.stack([2 * gs[:, 0] * gs[:, 1], 2 * gs[:, 0] * gs[:, 2], gs[:, 0] ** 2 - gs[:, 1] ** 2 - gs[:, 2] ** 2], 1)
    X = np.array([E, F, D]) / lam
    perp = phi - np.outer(phi @ X, X)
    assert np.abs(perp.mean(0)).max() < 0.05


def test_metropolis_chain_agrees_with_heatbath(oracle):
    # Eq. (30): a Metropolis chain on one SU(2) variable with f = g.a' has the
    # heatbath's stationary law.  Compare <f> from an independent NumPy chain with the oracle.
    rng = np.random.default_rng(10)
    a = np.array([1.2, -0.4, 0.7, 0.3]); T = 0.9
    ap = np.array([a[0], -a[1], -a[2], -a[3]])
    g = np.array([1.0, 0, 0, 0]); acc = []
    for it in range(60000):
        prop = g + 0.7 * rng.standard_normal(4); prop /= np.linalg.norm(prop)
        df = (prop - g) @ ap
        if df >= 0 or rng.random() < np.exp(df / T):
            g = prop
        if it > 2000:
            acc.append(g @ ap)
    hb = np.array([oracle.rule_heatbath_landau(a, T, 5, s, 0, 0) @ ap for s in range(6000)])
    assert abs(np.mean(acc) - hb.mean()) < 0.03 * np.linalg.norm(a)


def test_stochastic_relaxation_probability(oracle):
    U = small_config(51)
    base = inputs.as_real(U)
    relax, micro = base.copy(), base.copy()
    oracle.sweep(relax, LANDAU, OR, 1.0, parity_mask=1)
    oracle.sweep(micro, LANDAU, MICRO, 0.0, parity_mask=1)
    for p, ref in ((0.0, relax), (1.0, micro)):
        L = base.copy()
        oracle.sweep(L, LANDAU, SR, p, seed=3, sweep_index=0, parity_mask=1)
        assert np.array_equal(L, ref)
    # the draw decides: u < p -> micro (first subgroup decides whether the up-link rows 0,1 match)
    L = base.copy()
    oracle.sweep(L, LANDAU, SR, 0.3, seed=3, sweep_index=0, parity_mask=1)
    n_micro = n_tot = 0
    dims = base.shape[:4]
    for t in range(dims[0]):
        for x in range(dims[1]):
            for y in range(dims[2]):
                for z in range(dims[3]):
                    if (t + x + y + z) & 1:
                        continue
                    site = ((t * dims[1] + x) * dims[2] + y) * dims[3] + z
                    us = [oracle.draw(3, site, 0, s, 0, 0)[1][0] for s in range(3)]
                    n_tot += 3
                    n_micro += sum(u < 0.3 for u in us)
                    if all(u >= 0.3 for u in us):
                        assert np.array_equal(L[t, x, y, z], relax[t, x, y, z])
                    if all(u < 0.3 for u in us):
                        assert np.array_equal(L[t, x, y, z], micro[t, x, y, z])
    assert abs(n_micro / n_tot - 0.3) < 0.08
    # different sweep index -> different decisions (counter-based keying, R19)
    L2 = base.copy()
    oracle.sweep(L2, LANDAU, SR, 0.3, seed=3, sweep_index=1, parity_mask=1)
    assert not np.array_equal(L, L2)


def test_annealing_schedule_and_reproducibility(oracle):
    assert oracle.temperature(0, 2000, 1.45, 0.01) == 1.45
    assert oracle.temperature(1999, 2000, 1.45, 0.01) == pytest.approx(0.01, abs=1e-15)
    U = small_config(52)
    A, B = inputs.as_real(U), inputs.as_real(U)
    ia = oracle.anneal(A, MAG, 1.45, 0.01, 6, 3, seed=1234)
    ib = oracle.anneal(B, MAG, 1.45, 0.01, 6, 3, seed=1234)
    assert ia == ib == 24 and np.array_equal(A, B)          # stateless RNG: bit-reproducible
    C = inputs.as_real(U)
    oracle.anneal(C, MAG, 1.45, 0.01, 6, 3, seed=1235)
    assert not np.array_equal(A, C)
    # annealing to low T then OR improves F over the hot start
    F0 = oracle.measure(inputs.as_real(U), MAG)["F"]
    assert oracle.measure(A, MAG)["F"] > F0


# ------------------------------------------------------------------------------------------
# Reprojection and precision policy (R20/R23)
# ------------------------------------------------------------------------------------------
def test_reunitarize(oracle):
    rng = np.random.default_rng(12)
    U = inputs.haar_su3((50,), rng)
    R = inputs.as_real(U)
    R2 = R.copy()
    oracle.reunitarize(R2)
    np.testing.assert_allclose(R2, R, atol=5e-16)           # SU(3) is a fixed point
    noisy = R + 1e-3 * rng.standard_normal(R.shape)
    oracle.reunitarize(noisy)
    W = H.cplx(noisy)
    assert np.abs(W @ H.dag(W) - np.eye(3)).max() < 1e-15
    assert np.abs(np.linalg.det(W) - 1).max() < 1e-15
    assert np.abs(W - U).max() < 1e-2
    again = noisy.copy()
    oracle.reunitarize(again)
    np.testing.assert_allclose(again, noisy, atol=5e-16)    # idempotent
    # third row = (u x v)^*
    np.testing.assert_allclose(W[:, 2], np.conj(np.cross(W[:, 0], W[:, 1])), atol=1e-15)
    f = (R + 1e-3 * rng.standard_normal(R.shape)).astype(np.float32)
    oracle.reunitarize(f)
    Wf = H.cplx(f)
    assert np.abs(Wf @ H.dag(Wf) - np.eye(3)).max() < 5e-7


def test_precision_modes_agree_with_dp(oracle):
    # SP with reprojection every 100 and MP stay within 2e-5 of the DP functional
    U = inputs.make_config(4, 4, 4, 8, 0.5, 61, 62)
    D = inputs.as_real(U)
    sD, FD, thD, _, convD = oracle.run(D, LANDAU, OR, 1.7, max_sweeps=3000, eps=1e-12)
    assert convD
    S = inputs.as_real(U, np.float32)
    sS, FS, thS, _, _ = oracle.run(S, LANDAU, OR, 1.7, max_sweeps=sD, eps=0.0, check_every=sD, reunit_every=100)
    M = inputs.as_real(U, np.float32)
    sM, FM, thM, _, _ = oracle.run(M, LANDAU, OR, 1.7, max_sweeps=sD, eps=0.0, check_every=sD, reunit_every=100, mixed=True)
    assert abs(FS - FD) < 2e-5 and abs(FM - FD) < 2e-5
    assert thS < 1e-9 and thM < 1e-9
    # one sweep: SP and MP links within float rounding of DP
    D1, S1, M1 = inputs.as_real(U), inputs.as_real(U, np.float32), inputs.as_real(U, np.float32)
    oracle.sweep(D1, LANDAU, OR, 1.7); oracle.sweep(S1, LANDAU, OR, 1.7); oracle.sweep(M1, LANDAU, OR, 1.7, mixed=True)
    assert np.abs(S1 - D1).max() < 2e-5 and np.abs(M1 - D1).max() < 2e-5


def test_invalid_extents_rejected(oracle):
    L = np.zeros((3, 4, 4, 4, 4, 3, 3, 2))
    with pytest.raises(ValueError):
        oracle.sweep(L, LANDAU, OR, 1.7)


def test_lagged_stop_reading_is_the_plain_run_plus_one_even_half_sweep(oracle):
    # include/gf.h GF_FLAG_LAGGED_STOP: same checks, same stopping sweep, same history; the links returned have received
    # the even half-sweep of the next sweep (a gauge transformation: plaquettes unchanged, Eq. (1))
    from paper_1212_5221_b200 import inputs
    L0 = inputs.as_real(inputs.make_config(4, 4, 4, 4, 0.4, 91, 92))
    a, b = L0.copy(), L0.copy()
    sa, Fa, tha, ha, ca = oracle.run(a, oracle.LANDAU, oracle.OR, 1.7, max_sweeps=500, eps=1e-10, check_every=3)
    sb, Fb, thb, hb, cb = oracle.run(b, oracle.LANDAU, oracle.OR, 1.7, max_sweeps=500, eps=1e-10, check_every=3, lagged_stop=True)
    assert ca and cb and sa == sb and ha == hb
    oracle.sweep(a, oracle.LANDAU, oracle.OR, 1.7, 0, sa, parity_mask=1)
    assert np.array_equal(a, b)
    m = oracle.measure(b, oracle.LANDAU)
    assert Fb == m["F"] and thb == m["theta"] and Fb >= Fa - 1e-15
    # a run that exhausts max_sweeps is not touched
    c, d = L0.copy(), L0.copy()
    assert oracle.run(c, oracle.LANDAU, oracle.OR, 1.7, max_sweeps=6, eps=1e-10)[:3] == \
        oracle.run(d, oracle.LANDAU, oracle.OR, 1.7, max_sweeps=6, eps=1e-10, lagged_stop=True)[:3]
    assert np.array_equal(c, d)


def test_config3_copy_spread_fixture_is_the_oracles(oracle):
    """tests/golden/config3_copy_spread.txt is written by tests/golden/make_config3_copy_spread.py from the oracle alone;
    two of its 32 random sequences are replayed here (PAPER.md:243, 556 schedule; R25).  On this 6^4 lattice
    every sequence ends in the same maximum of the maximally Abelian functional, which is what lets the GPU parity test
    ask for F to 1e-10 after a chaotic annealing trajectory."""
    from tests.helpers import golden_values
    from paper_1212_5221_b200 import inputs
    sp = golden_values("config3_copy_spread.txt")
    assert sp["n_seeds"] == 32 and sp["F_final_max"] - sp["F_final_min"] < 1e-11 and 5e-4 < sp["F_after_anneal_sigma"] < 2e-3
    L = inputs.as_real(inputs.make_config(6, 6, 6, 6, 0.5, 350, 351))
    for k in (0, 17):
        ref = L.copy()
        nxt = oracle.anneal(ref, 2, 1.45, 0.01, 12, 3, seed=1234 + k)
        Fa = oracle.measure(ref, 2)["F"]
        s, F, th, hist, conv = oracle.run(ref, 2, 0, 1.7, max_sweeps=8000, eps=1e-12, first_sweep_index=nxt)
        assert conv and abs(F - sp["F_final_mean"]) < 1e-11
        assert abs(Fa - sp["F_after_anneal_mean"]) < 4 * sp["F_after_anneal_sigma"]
