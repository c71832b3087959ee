"""Seeded synthetic SU(3) lattices (input recipe of DESIGN.md §4, BASELINE.json `configs`).

This module holds *no* arithmetic of the gauge-fixing method: it only manufactures inputs.
Both the CPU oracle's tests and the CUDA path's tests/bench draw from it, so that the two
sides see bit-identical inputs.

Layout of every array returned here is the paper's *StandardPattern*
(Sec. 4.2.1): ``links[t, x, y, z, mu, i, j]`` complex, ``mu = 0`` temporal,
``mu = 1, 2, 3`` = x, y, z.  ``as_real`` views it as ``[..., i, j, (re, im)]``.

Recipe (BASELINE.json configs 0-4): ``U = exp(i * eps * sum_a r_a lambda_a / 2)`` with
``r_a ~ N(0, 1)`` and the Gell-Mann matrices ``lambda_a``, projected back onto SU(3);
then a Haar-random gauge transformation ``h(x)`` is applied at every site,
``U_mu(x) <- h(x) U_mu(x) h(x + mu)^dagger`` (Eq. 1).
"""
from __future__ import annotations

import numpy as np

# Gell-Mann matrices lambda_1..lambda_8 (generators of SU(3), Eq. 10).
_GM = np.zeros((8, 3, 3), dtype=np.complex128)
_GM[0, 0, 1] = _GM[0, 1, 0] = 1
_GM[1, 0, 1] = -1j
_GM[1, 1, 0] = 1j
_GM[2, 0, 0] = 1
_GM[2, 1, 1] = -1
_GM[3, 0, 2] = _GM[3, 2, 0] = 1
_GM[4, 0, 2] = -1j
_GM[4, 2, 0] = 1j
_GM[5, 1, 2] = _GM[5, 2, 1] = 1
_GM[6, 1, 2] = -1j
_GM[6, 2, 1] = 1j
_GM[7, 0, 0] = _GM[7, 1, 1] = 1 / np.sqrt(3)
_GM[7, 2, 2] = -2 / np.sqrt(3)


def gell_mann() -> np.ndarray:
    return _GM.copy()


def _dag(m: np.ndarray) -> np.ndarray:
    return np.conj(np.swapaxes(m, -1, -2))


def project_su3(m: np.ndarray) -> np.ndarray:
    """Nearest special-unitary matrix (polar factor via SVD, then remove the det phase)."""
    u, _, vh = np.linalg.svd(m)
    w = u @ vh
    det = np.linalg.det(w)
    return w * np.exp(-1j * np.angle(det) / 3.0)[..., None, None]


def random_algebra_links(shape, eps: float, rng: np.random.Generator) -> np.ndarray:
    """exp(i eps sum_a r_a lambda_a/2), r_a ~ N(0,1); `shape` = leading (batch) shape."""
    r = rng.standard_normal(tuple(shape) + (8,))
    herm = np.einsum("...a,aij->...ij", r, _GM) * (0.5 * eps)
    w, v = np.linalg.eigh(herm)
    u = (v * np.exp(1j * w)[..., None, :]) @ _dag(v)
    return project_su3(u)


def haar_su3(shape, rng: np.random.Generator) -> np.ndarray:
    """Haar-distributed SU(3): QR of a complex Ginibre matrix with the phases of diag(R)
    moved into Q (Haar on U(3)), then the determinant phase divided out."""
    shape = tuple(shape)
    z = rng.standard_normal(shape + (3, 3)) + 1j * rng.standard_normal(shape + (3, 3))
    q, r = np.linalg.qr(z)
    d = np.diagonal(r, axis1=-2, axis2=-1)
    q = q * (d / np.abs(d))[..., None, :]
    det = np.linalg.det(q)
    return q * np.exp(-1j * np.angle(det) / 3.0)[..., None, None]


def gauge_transform(links: np.ndarray, h: np.ndarray) -> np.ndarray:
    """U_mu(x) <- h(x) U_mu(x) h(x+mu)^dagger, periodic (Eq. 1).  Axis mu of the
    site array is axis mu of `links`/`h` (0=t, 1=x, 2=y, 3=z)."""
    out = np.empty_like(links)
    for mu in range(4):
        hf = np.roll(h, -1, axis=mu)
        out[..., mu, :, :] = h @ links[..., mu, :, :] @ _dag(hf)
    return out


def pure_gauge(dims_txyz, seed: int) -> np.ndarray:
    """U_mu(x) = h(x) h(x+mu)^dagger with Haar h: a gauge copy of the trivial vacuum."""
    rng = np.random.default_rng(seed)
    h = haar_su3(tuple(dims_txyz), rng)
    unit = np.broadcast_to(np.eye(3, dtype=np.complex128), tuple(dims_txyz) + (4, 3, 3)).copy()
    return gauge_transform(unit, h)


def make_config(Nx: int, Ny: int, Nz: int, Nt: int, eps: float, seed_links: int,
                seed_gauge: int | None = None) -> np.ndarray:
    """Synthetic lattice of BASELINE.json's configs: complex128 [Nt,Nx,Ny,Nz,4,3,3]."""
    dims = (Nt, Nx, Ny, Nz)
    rng = np.random.default_rng(seed_links)
    links = random_algebra_links(dims + (4,), eps, rng)
    if seed_gauge is not None:
        h = haar_su3(dims, np.random.default_rng(seed_gauge))
        links = gauge_transform(links, h)
    return links


def config_k(k: int, dims_xyzt=None) -> np.ndarray:
    """Config k of BASELINE.json (seeds 1000+k / 2000+k)."""
    table = {0: ((4, 4, 4, 4), 0.3), 1: ((16, 16, 16, 16), 0.5), 2: ((32, 32, 32, 64), 0.6),
             3: ((24, 24, 24, 24), 0.5), 4: ((64, 64, 64, 256), 0.5)}
    d, eps = table[k]
    if dims_xyzt is not None:
        d = tuple(dims_xyzt)
    return make_config(d[0], d[1], d[2], d[3], eps, 1000 + k, 2000 + k)


_PAULI = np.array([[[0, 1], [1, 0]], [[0, -1j], [1j, 0]], [[1, 0], [0, -1]]], dtype=np.complex128)


def su2_from_quaternion(q: np.ndarray) -> np.ndarray:
    """q[...,4] on S^3 -> q0 1 + i (q1 s1 + q2 s2 + q3 s3), the parametrisation of PAPER.md:124 Eq. (15)."""
    out = np.einsum("...a,aij->...ij", q[..., 1:], _PAULI) * 1j
    out[..., 0, 0] += q[..., 0]
    out[..., 1, 1] += q[..., 0]
    return out


def random_algebra_links_su2(shape, eps: float, rng: np.random.Generator) -> np.ndarray:
    """exp(i eps sum_a r_a sigma_a/2), r_a ~ N(0,1): the N_c = 2 analogue of random_algebra_links."""
    r = rng.standard_normal(tuple(shape) + (3,)) * (0.5 * eps)
    n = np.linalg.norm(r, axis=-1, keepdims=True)
    q = np.concatenate([np.cos(n), np.sin(n) * r / np.where(n > 0, n, 1.0)], axis=-1)
    return su2_from_quaternion(q)


def haar_su2(shape, rng: np.random.Generator) -> np.ndarray:
    """Haar-distributed SU(2): a uniform point of S^3."""
    q = rng.standard_normal(tuple(shape) + (4,))
    return su2_from_quaternion(q / np.linalg.norm(q, axis=-1, keepdims=True))


def make_config_su2(Nx: int, Ny: int, Nz: int, Nt: int, eps: float, seed_links: int,
                    seed_gauge: int | None = None) -> np.ndarray:
    """Synthetic SU(2) lattice, the recipe of make_config with Pauli matrices: complex128 [Nt,Nx,Ny,Nz,4,2,2]."""
    dims = (Nt, Nx, Ny, Nz)
    links = random_algebra_links_su2(dims + (4,), eps, np.random.default_rng(seed_links))
    if seed_gauge is not None:
        links = gauge_transform(links, haar_su2(dims, np.random.default_rng(seed_gauge)))
    return links


def as_real(links: np.ndarray, dtype=np.float64) -> np.ndarray:
    """complex [...,3,3] -> real [...,3,3,2] (re, im) contiguous, StandardPattern order."""
    out = np.empty(links.shape + (2,), dtype=dtype)
    out[..., 0] = links.real
    out[..., 1] = links.imag
    return out


def as_complex(reals: np.ndarray) -> np.ndarray:
    r = np.asarray(reals, dtype=np.float64)
    return r[..., 0] + 1j * r[..., 1]


def tile_lattice(links: np.ndarray, reps_txyz) -> np.ndarray:
    """Periodic tiling of a lattice (a tiled gauge field is again a gauge field)."""
    return np.tile(links, tuple(reps_txyz) + (1, 1, 1))
