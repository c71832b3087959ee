"""NumPy helpers for the tests: observables and brute-force evaluators written directly from
the paper's definitions, independent of both oracle/ and the CUDA path."""
import numpy as np


def dag(m):
    return np.conj(np.swapaxes(m, -1, -2))


def cplx(reals):
    r = np.asarray(reals, dtype=np.float64)
    return r[..., 0] + 1j * r[..., 1]


def plaquettes(U):
    """Re tr of all 6 plaquette orientations at every site, U complex [t,x,y,z,mu,3,3];
    gauge invariant under Eq. (1).  Returns array [6, t,x,y,z]."""
    out = []
    for mu in range(4):
        for nu in range(mu + 1, 4):
            Umu, Unu = U[..., mu, :, :], U[..., nu, :, :]
            Unu_xmu = np.roll(Unu, -1, axis=mu)
            Umu_xnu = np.roll(Umu, -1, axis=nu)
            P = Umu @ Unu_xmu @ dag(Umu_xnu) @ dag(Unu)
            out.append(np.real(np.trace(P, axis1=-2, axis2=-1)) / 3.0)
    return np.array(out)


def embed_su2(g, i, j):
    """SU(2) element (g0,g1,g2,g3) in the Cayley-Klein form of Eq. (22), embedded
    in rows/columns (i,j) of a 3x3 identity."""
    g = np.asarray(g, dtype=np.float64)
    m = np.zeros(g.shape[:-1] + (3, 3), dtype=np.complex128)
    for k in range(3):
        m[..., k, k] = 1
    m[..., i, i] = g[..., 0] + 1j * g[..., 3]
    m[..., i, j] = g[..., 2] + 1j * g[..., 1]
    m[..., j, i] = -g[..., 2] + 1j * g[..., 1]
    m[..., j, j] = g[..., 0] - 1j * g[..., 3]
    return m


def local_landau(gm, up, dn):
    """sum_mu Re tr[g U_mu(x)] + Re tr[U_mu(x-mu) g^dag]  (Eqs. 4, 5, 18 at one site);
    gm [...,3,3], up/dn [nd,3,3] complex."""
    K = up.sum(axis=0) + dag(dn).sum(axis=0)   # Eq. (19) with neighbours' g = 1
    return np.real(np.trace(gm @ K, axis1=-2, axis2=-1))


def local_mag(gm, up, dn):
    """sum_mu sum_i |(g U_mu(x))_ii|^2 + |(U_mu(x-mu) g^dag)_ii|^2  (Eq. 11 at one site)."""
    tot = 0.0
    for m in range(up.shape[0]):
        a = gm @ up[m]
        b = dn[m] @ dag(gm)
        tot = tot + (np.abs(np.diagonal(a, axis1=-2, axis2=-1)) ** 2).sum(-1)
        tot = tot + (np.abs(np.diagonal(b, axis1=-2, axis2=-1)) ** 2).sum(-1)
    return tot


def su2_grid_full(n):
    """Dense grid on S^3 (all of SU(2)): Hopf-like angles, ~n^3 points."""
    chi = np.linspace(0, np.pi / 2, n)
    p1 = np.linspace(0, 2 * np.pi, 2 * n, endpoint=False)
    p2 = np.linspace(0, 2 * np.pi, 2 * n, endpoint=False)
    C, A, B = np.meshgrid(chi, p1, p2, indexing="ij")
    g = np.stack([np.cos(C) * np.cos(A), np.sin(C) * np.cos(B), np.sin(C) * np.sin(B), np.cos(C) * np.sin(A)], -1)
    return g.reshape(-1, 4)


def gather_site(U, t, x, y, z, dirs=(0, 1, 2, 3)):
    """up[m] = U_mu(x), dn[m] = U_mu(x - mu) from complex U[t,x,y,z,mu,3,3] (periodic)."""
    up = np.array([U[t, x, y, z, mu] for mu in dirs])
    c = [t, x, y, z]
    dn = []
    for mu in dirs:
        cc = list(c)
        cc[mu] = (cc[mu] - 1) % U.shape[mu]
        dn.append(U[cc[0], cc[1], cc[2], cc[3], mu])
    return up, np.array(dn)


def to_real(c, dtype=np.float64):
    out = np.empty(c.shape + (2,), dtype=dtype)
    out[..., 0] = c.real
    out[..., 1] = c.imag
    return out


def paper_values():
    """The numbers printed in the paper that tests compare against (tests/golden/paper_printed_values.txt)."""
    import os
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_printed_values.txt")) as fh:
        for line in fh:
            line = line.split("#")[0].split()
            if len(line) == 2:
                out[line[0]] = float(line[1])
    return out


def golden_values(name):
    """key -> float of a `key value` fixture under tests/golden/ (lines starting with # are comments)."""
    import os
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", name)) as fh:
        for line in fh:
            line = line.split("#")[0].split()
            if len(line) == 2:
                out[line[0]] = float(line[1])
    return out
