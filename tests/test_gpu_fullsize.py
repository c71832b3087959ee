"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times
(64^3 x 256 and 32^3 x 64, default CTA shapes, links set from a device pointer).

Two kinds of check that the oracle can afford at 67 M sites:

* periodic tiling — a sweep is local and deterministic, so sweeping the periodic tiling of a 16^4
  lattice must give the tiling of the swept 16^4 lattice: the oracle sweeps the tile (milliseconds)
  and EVERY link of the full lattice is compared element by element;
* sampled sites on a NON-periodic lattice (the tiling times a site-dependent diagonal gauge
  transformation, so that a wrong wrap-around or an overflowing offset cannot hide behind the
  period): the oracle updates a few thousand sampled sites one by one from their gathered links
  (gfo_site_update) and the corresponding outputs of one GPU half-sweep are compared.

torch is used here for device memory and for comparing/gathering on the device only.
"""
import numpy as np
import pytest

from paper_1212_5221_b200 import inputs

pytestmark = pytest.mark.gpu

LANDAU, COULOMB, MAG = 0, 1, 2
OR = 0
SP, DP, MP = 0, 1, 2
TILE = (16, 16, 16, 16)
TOL = {DP: 1e-12, SP: 5e-5, MP: 5e-5}


@pytest.fixture(scope="module")
def gf():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1212_5221_b200 import gf as _gf
    return _gf


@pytest.fixture(scope="module")
def tile():
    return inputs.as_real(inputs.make_config(*TILE, 0.5, 1004, 2004))     # the tile bench.py uses


def reps(dims_xyzt):
    Nx, Ny, Nz, Nt = dims_xyzt
    return (Nt // TILE[3], Nx // TILE[0], Ny // TILE[1], Nz // TILE[2])


def max_diff_against_tiling(torch, out_dev, ref_tile_dev, r):
    """max |out - tiling(ref_tile)| computed block by block on the device."""
    tt = ref_tile_dev.shape[0]
    block = ref_tile_dev.repeat(1, r[1], r[2], r[3], 1, 1, 1, 1)
    worst = 0.0
    for k in range(r[0]):
        d = (out_dev[k * tt:(k + 1) * tt].to(torch.float64) - block).abs().max().item()
        worst = max(worst, d)
    return worst


@pytest.mark.parametrize("dims,prec,recon,gauge", [
    ((64, 64, 64, 256), DP, 18, LANDAU),      # bench.py headline
    ((64, 64, 64, 256), SP, 12, LANDAU),      # bench.py variant
    ((64, 64, 64, 256), SP, 18, LANDAU),
    ((64, 64, 64, 256), DP, 12, LANDAU),
    ((64, 64, 64, 256), MP, 12, LANDAU),
    ((32, 32, 32, 64), SP, 12, COULOMB),      # BASELINE.json configs[2]
    ((32, 32, 32, 64), DP, 18, MAG),
])
def test_full_size_sweep_equals_tiled_oracle(gf, oracle, tile, dims, prec, recon, gauge):
    import torch
    dt = np.float64 if prec == DP else np.float32
    tdt = torch.float64 if prec == DP else torch.float32
    ref = tile.astype(dt)
    oracle.sweep(ref, gauge, OR, 1.7, mixed=(prec == MP))
    m = oracle.measure(ref, gauge)
    r = reps(dims)
    dev = torch.device("cuda", 0)
    src = torch.from_numpy(tile.astype(dt)).to(dev).repeat(*r, 1, 1, 1, 1).contiguous()
    with gf.GaugeFixer(*dims, precision=prec, recon=recon) as fx:
        fx.set_links(src)
        del src
        fx.sweep(gauge, OR, 1.7)
        F, th = fx.measure(gauge)
        out = torch.empty((dims[3], dims[0], dims[1], dims[2], 4, 3, 3, 2), dtype=tdt, device=dev)
        gf.gf_get_links(fx.ctx, out)
    worst = max_diff_against_tiling(torch, out, torch.from_numpy(ref).to(dev).to(torch.float64), r)
    assert worst <= TOL[prec], worst
    # F and theta are intensive: the tiled lattice has the tile's values
    rel = 1e-12 if prec == DP else 2e-6
    assert F == pytest.approx(m["F"], rel=rel, abs=rel)
    assert th == pytest.approx(m["theta"], rel=10 * rel)


def phase_field(torch, dims_xyzt, dev):
    """Site-dependent diagonal SU(3) element diag(e^{i a}, e^{i b}, e^{-i(a+b)}), not periodic in any
    sub-extent: input manufacture only (a gauge transformation, Eq. (1))."""
    Nx, Ny, Nz, Nt = dims_xyzt
    t = torch.arange(Nt, device=dev, dtype=torch.float64).view(Nt, 1, 1, 1)
    x = torch.arange(Nx, device=dev, dtype=torch.float64).view(1, Nx, 1, 1)
    y = torch.arange(Ny, device=dev, dtype=torch.float64).view(1, 1, Ny, 1)
    z = torch.arange(Nz, device=dev, dtype=torch.float64).view(1, 1, 1, Nz)
    a = torch.sin(0.7310 * t + 1.1930 * x - 0.4170 * y + 0.9050 * z + 0.003 * t * x) * 2.0
    b = torch.cos(0.2930 * t - 0.8110 * x + 1.3070 * y + 0.5530 * z - 0.002 * y * z) * 2.0
    ph = torch.stack([a, b, -(a + b)], dim=-1)
    return torch.polar(torch.ones_like(ph), ph)                   # complex128 [Nt,Nx,Ny,Nz,3]


def nonperiodic_lattice(torch, tile, dims_xyzt, dev):
    r = reps(dims_xyzt)
    U = torch.view_as_complex(torch.from_numpy(tile).to(dev).repeat(*r, 1, 1, 1, 1).contiguous())
    P = phase_field(torch, dims_xyzt, dev)
    for mu in range(4):
        Pf = torch.roll(P, -1, dims=mu)
        U[..., mu, :, :] *= P[..., :, None] * Pf.conj()[..., None, :]
        del Pf
    return torch.view_as_real(U)                                   # [Nt,Nx,Ny,Nz,4,3,3,2] f64


def sample_sites(dims_xyzt, parity, n, rng):
    Nx, Ny, Nz, Nt = dims_xyzt
    ext = np.array([Nt, Nx, Ny, Nz])
    s = rng.integers(0, ext, size=(n, 4))
    # force a good share onto the lattice boundary in each direction (wrap-around neighbours)
    for k in range(n // 2):
        d = k % 4
        s[k, d] = 0 if (k // 4) % 2 == 0 else ext[d] - 1
    fix = (s.sum(axis=1) & 1) != parity
    s[fix, 3] ^= 1                                                 # flip z's low bit (extents are even)
    return s


@pytest.mark.parametrize("dims,prec,recon", [((64, 64, 64, 256), DP, 18), ((64, 64, 64, 256), SP, 12),
                                             ((32, 32, 32, 64), DP, 12)])
def test_full_size_sampled_sites_nonperiodic(gf, oracle, tile, dims, prec, recon):
    import torch
    dev = torch.device("cuda", 0)
    dt = np.float64 if prec == DP else np.float32
    tdt = torch.float64 if prec == DP else torch.float32
    src = nonperiodic_lattice(torch, tile, dims, dev).to(tdt)
    ext = [dims[3], dims[0], dims[1], dims[2]]
    rng = np.random.default_rng(77)
    with gf.GaugeFixer(*dims, precision=prec, recon=recon) as fx:
        out = torch.empty_like(src)
        for parity in (0, 1):
            fx.set_links(src)
            fx.half_sweep(LANDAU, OR, 1.7, 0, 0, parity)
            gf.gf_get_links(fx.ctx, out)
            s = sample_sites(dims, parity, 3000, rng)
            st = torch.from_numpy(s).to(dev)
            mu = torch.arange(4, device=dev)
            dn = st[:, None, :].repeat(1, 4, 1)
            for d in range(4):
                dn[:, d, d] = (dn[:, d, d] - 1) % ext[d]
            gather_up = lambda A: A[st[:, 0, None], st[:, 1, None], st[:, 2, None], st[:, 3, None], mu[None, :]]
            gather_dn = lambda A: A[dn[..., 0], dn[..., 1], dn[..., 2], dn[..., 3], mu[None, :]]
            up_in, dn_in = gather_up(src).cpu().numpy(), gather_dn(src).cpu().numpy()
            up_out, dn_out = gather_up(out).cpu().numpy(), gather_dn(out).cpu().numpy()
            worst = 0.0
            for k in range(s.shape[0]):
                u, d_ = np.ascontiguousarray(up_in[k]), np.ascontiguousarray(dn_in[k])
                oracle.site_update(u, d_, LANDAU, OR, 1.7)
                worst = max(worst, float(np.abs(u.astype(np.float64) - up_out[k]).max()),
                            float(np.abs(d_.astype(np.float64) - dn_out[k]).max()))
            assert worst <= TOL[prec], (parity, worst)
            # sites of the other parity are untouched by this half-sweep except through these links:
            # a link not adjacent to any active site does not exist (every link has one end of each
            # parity), so instead check global invariants: unitarity of a random sample of outputs
            W = up_out[..., 0] + 1j * up_out[..., 1]
            uni = np.abs(W @ np.conj(np.swapaxes(W, -1, -2)) - np.eye(3)).max()
            assert uni < (1e-12 if prec == DP else 2e-5)
