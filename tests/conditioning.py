"""First-order rounding-error bound for one heatbath HALF-sweep in single precision (tests only).

The SP path forms the neighbourhood sums of a site (K(x) of Eq. (19), resp. D, E, F of Eqs. (26)-(28),
PAPER.md:200-206) in float, with a different association order on the CPU oracle and on the GPU, so the input of
Step 1 differs by a few float ulps of the 2d summed links.  The heatbath turns that into a difference of the drawn
g(x) amplified by the inverse of the local field: the direction conj(a)/|a| of Eq. (20) has the
condition number 1/|a|; for MAG the sampling frame about X = (E, F, D) (R15) is conditioned by
1/lambda (Eq. (29)), its azimuth by 1/sqrt(E^2 + F^2), and the map from the drawn point of S^2
to g by 1/g_0.  BASELINE.json's 5e-5 holds wherever
those numbers are O(1); a rare site with a weak local field exceeds it on both paths legitimately.

`half_sweep_error_bound` replays the oracle's site updates of one half-sweep in double on the float links (oracle
calls only), takes c(x) = min over the three subgroups of the conditioning number, and bounds the difference of
every link the site x rotates, and of g(x), by

    C eps (1 + S / c(x)),      eps = 2^-23,  S = 2d unit-size links in the sum,  one constant C for all sites.

Both paths start the half-sweep from the same float links, so nothing compounds.
"""
import numpy as np

LANDAU, COULOMB, MAG = 0, 1, 2
SUBS = ((0, 1), (0, 2), (1, 2))
EPS_F = 2.0 ** -23


def _gather(L, t, x, y, z, dirs):
    up = np.ascontiguousarray(np.stack([L[t, x, y, z, mu] for mu in dirs]))
    dn = []
    for mu in dirs:
        c = [t, x, y, z]
        c[mu] = (c[mu] - 1) % L.shape[mu]
        dn.append(L[c[0], c[1], c[2], c[3], mu])
    return up, np.ascontiguousarray(np.stack(dn))


def site_conditioning(oracle, Lpre, txyz, gauge, T, seed, sweep_index):
    """min over the Cabibbo-Marinari subgroups of the local field that conditions the heatbath at this site, the
    subgroups updated one after the other as in Alg. 1.  Lpre: float64 links before the
    half-sweep that updates the site."""
    t, x, y, z = txyz
    Nt, Nx, Ny, Nz = Lpre.shape[:4]
    dirs = (1, 2, 3) if gauge == COULOMB else (0, 1, 2, 3)
    up, dn = _gather(Lpre, t, x, y, z, dirs)
    sidx = ((t * Nx + x) * Ny + y) * Nz + z
    return gathered_conditioning(oracle, up, dn, gauge, T, seed, sidx, sweep_index)


def gathered_conditioning(oracle, up, dn, gauge, T, seed, sidx, sweep_index):
    """site_conditioning for a site given by its gathered links up[mu] = U_mu(x), dn[mu] = U_mu(x - mu) (float64,
    modified in place) and its lexicographic index sidx in the whole lattice (the Philox counter)."""
    dirs = range(up.shape[0])
    c = np.inf
    for s, (i, j) in enumerate(SUBS):
        if gauge == MAG:
            D, E, F = oracle.local_mag_def(up, dn, i, j)
            g = oracle.rule_heatbath_mag(D, E, F, T, seed, sidx, sweep_index, s)
            # the drawn point phi of S^2 is turned into g by g0 = sqrt((1 + phi_3)/2), (g1, g2) = (phi_1, phi_2)/(2 g0)
            # (R15): a further factor 1/g0 where the draw lands near the south pole
            c = min(c, min(np.sqrt(D * D + E * E + F * F), np.hypot(E, F)) * max(abs(g[0]), 1e-300))
        else:
            a = oracle.local_quaternion(up, dn, i, j)
            c = min(c, float(np.linalg.norm(a)))
            g = oracle.rule_heatbath_landau(a, T, seed, sidx, sweep_index, s)
        for m in range(len(dirs)):
            up[m] = oracle.apply_subgroup(up[m], g, i, j, False)
            dn[m] = oracle.apply_subgroup(dn[m], g, i, j, True)
    return c


def half_sweep_error_bound(oracle, L32, gauge, T, seed, sweep_index, parity, C=4.0):
    """-> (bound[t,x,y,z,mu] for every link, bound_g[t,x,y,z] (0 at sites of the other parity), c[t,x,y,z] (inf at
    sites of the other parity)) for one SP heatbath half-sweep of `parity` from the float links L32
    (StandardPattern).  Landau / MAG only (4-d colouring)."""
    assert gauge in (LANDAU, MAG) and L32.dtype == np.float32
    pre = L32.astype(np.float64)
    dims = L32.shape[:4]
    S = 8.0
    c = np.full(dims, np.inf)
    for idx in np.ndindex(*dims):
        if (sum(idx) & 1) == parity:
            c[idx] = site_conditioning(oracle, pre, idx, gauge, T, seed, sweep_index)
    bg = np.where(np.isfinite(c), C * EPS_F * (1.0 + S / c), 0.0)
    active = np.isfinite(c)
    bl = np.zeros(dims + (4,))
    for mu in range(4):      # link (x, mu) has the end points x and x + mu, exactly one of them of the active parity
        bl[..., mu] = np.where(active, bg, np.roll(bg, -1, axis=mu))
    return bl, bg, c
