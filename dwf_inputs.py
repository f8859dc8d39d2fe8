"""Seeded synthetic input generators shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no gamma matrices, no stencil, no operator):
it only draws random numbers and shapes them into the canonical arrays of DESIGN.md §3
(SURVEY.md App. A.1):

    gauge  : complex128 [mu=4][t][z][y][x][3][3]      mu = 0,1,2,3 <-> x,y,z,t ; element U_mu(x)_{ab}
    spinor : complex128 [nrhs][Ls][t][z][y][x][4][3]  spin, colour innermost

They stand in for the paper's RBC-UKQCD configurations, which are not
available; recipe = BASELINE.json configs[*] and SURVEY.md §8(c) R15/R16/R17:
  * SU(3) link: 3x3 complex Gaussian, rows 0,1 Gram-Schmidt orthonormalised in order, row 2 =
    conj(row0 x row1)  (the unique det=+1 unitary completion).
  * spinor: Re, Im independent N(0,1).
  * fp32 runs: round ONCE to fp32; the rounded data is the input to both sides.
"""
from __future__ import annotations

import numpy as np

__all__ = [
    "su3_from_gaussian", "gauge_random", "gauge_unit", "su3_site_field", "spinor_gaussian",
    "round_to_precision", "site_parity", "keep_parity", "point_source",
]


def su3_from_gaussian(g: np.ndarray) -> np.ndarray:
    """Map complex Gaussian matrices [...,3,3] to SU(3) (R15)."""
    r0 = g[..., 0, :]
    r1 = g[..., 1, :]
    r0 = r0 / np.sqrt(np.sum(np.abs(r0) ** 2, axis=-1, keepdims=True))
    proj = np.sum(np.conj(r0) * r1, axis=-1, keepdims=True)  # <r0, r1>
    r1 = r1 - r0 * proj
    r1 = r1 / np.sqrt(np.sum(np.abs(r1) ** 2, axis=-1, keepdims=True))
    r2 = np.conj(np.cross(r0, r1))
    return np.stack([r0, r1, r2], axis=-2)


def _gauss_complex(rng: np.random.Generator, shape) -> np.ndarray:
    a = rng.standard_normal(shape + (2,))
    return a[..., 0] + 1j * a[..., 1]


def gauge_random(L, seed: int) -> np.ndarray:
    """Random SU(3) gauge field, canonical [4][t][z][y][x][3][3] complex128. L = (Lx,Ly,Lz,Lt)."""
    Lx, Ly, Lz, Lt = (int(v) for v in L)
    rng = np.random.default_rng(seed)
    g = _gauss_complex(rng, (4, Lt, Lz, Ly, Lx, 3, 3))
    return np.ascontiguousarray(su3_from_gaussian(g))


def gauge_unit(L) -> np.ndarray:
    Lx, Ly, Lz, Lt = (int(v) for v in L)
    U = np.zeros((4, Lt, Lz, Ly, Lx, 3, 3), dtype=np.complex128)
    U[..., 0, 0] = U[..., 1, 1] = U[..., 2, 2] = 1.0
    return U


def su3_site_field(L, seed: int) -> np.ndarray:
    """One random SU(3) matrix per 4D site, [t][z][y][x][3][3] (used as a gauge transformation g(x))."""
    Lx, Ly, Lz, Lt = (int(v) for v in L)
    rng = np.random.default_rng(seed)
    return np.ascontiguousarray(su3_from_gaussian(_gauss_complex(rng, (Lt, Lz, Ly, Lx, 3, 3))))


def spinor_gaussian(L, Ls: int, nrhs: int, seed: int) -> np.ndarray:
    """nrhs Gaussian 5D spinor fields, canonical [nrhs][Ls][t][z][y][x][4][3] complex128.

    Field r is drawn from its own stream seed + 100*r so that the first k fields
    of a larger batch are the same fields whatever the batch size.
    """
    Lx, Ly, Lz, Lt = (int(v) for v in L)
    out = np.empty((nrhs, Ls, Lt, Lz, Ly, Lx, 4, 3), dtype=np.complex128)
    for r in range(nrhs):
        rng = np.random.default_rng(seed + 100 * r)
        out[r] = _gauss_complex(rng, (Ls, Lt, Lz, Ly, Lx, 4, 3))
    return out


def round_to_precision(a: np.ndarray, precision: str) -> np.ndarray:
    """R17: fp32 runs round the fp64-generated data once; result returned as complex128 again."""
    if precision in ("f64", "fp64"):
        return a
    if precision in ("f32", "fp32"):
        return a.astype(np.complex64).astype(np.complex128)
    raise ValueError(precision)


def site_parity(L) -> np.ndarray:
    """(x+y+z+t) mod 2 as an int array [t][z][y][x]."""
    Lx, Ly, Lz, Lt = (int(v) for v in L)
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    return (x + y + z + t) & 1


def keep_parity(psi: np.ndarray, L, parity: int) -> np.ndarray:
    """Zero the sites of the other 4D parity (canonical half field = full array, other half zero)."""
    mask = (site_parity(L) == parity)
    return psi * mask[None, None, :, :, :, :, None, None]


def point_source(L, Ls: int, site, s: int, spin: int, colour: int) -> np.ndarray:
    Lx, Ly, Lz, Lt = (int(v) for v in L)
    psi = np.zeros((1, Ls, Lt, Lz, Ly, Lx, 4, 3), dtype=np.complex128)
    x, y, z, t = site
    psi[0, s, t, z, y, x, spin, colour] = 1.0
    return psi


# ---- device-side generation for lattices too big to draw on the host (configs[4]) -------------------
def su3_from_gaussian_torch(g):
    """Same recipe as su3_from_gaussian (R15) on a torch complex tensor [...,3,3] (any device)."""
    import torch
    r0 = g[..., 0, :]
    r1 = g[..., 1, :]
    r0 = r0 / torch.sqrt(torch.sum(r0.abs() ** 2, dim=-1, keepdim=True))
    proj = torch.sum(torch.conj(r0) * r1, dim=-1, keepdim=True)
    r1 = r1 - r0 * proj
    r1 = r1 / torch.sqrt(torch.sum(r1.abs() ** 2, dim=-1, keepdim=True))
    r2 = torch.conj(torch.linalg.cross(r0, r1))
    return torch.stack([r0, r1, r2], dim=-2)


def gauge_random_torch(L, seed: int, device, dtype):
    """Random SU(3) gauge field drawn on `device` with torch's seeded generator, one direction at a time."""
    import torch
    Lx, Ly, Lz, Lt = (int(v) for v in L)
    gen_ = torch.Generator(device=device); gen_.manual_seed(seed)
    rdt = torch.float32 if dtype == torch.complex64 else torch.float64
    U = torch.empty((4, Lt, Lz, Ly, Lx, 3, 3), dtype=dtype, device=device)
    for mu in range(4):
        g = torch.view_as_complex(torch.randn((Lt, Lz, Ly, Lx, 3, 3, 2), generator=gen_, device=device, dtype=rdt))
        U[mu] = su3_from_gaussian_torch(g)
    return U


def spinor_gaussian_torch(L, Ls: int, nrhs: int, seed: int, device, dtype):
    """Gaussian spinor fields drawn on `device`: canonical [nrhs][Ls][t][z][y][x][4][3]."""
    import torch
    Lx, Ly, Lz, Lt = (int(v) for v in L)
    gen_ = torch.Generator(device=device); gen_.manual_seed(seed)
    rdt = torch.float32 if dtype == torch.complex64 else torch.float64
    out = torch.empty((nrhs, Ls, Lt, Lz, Ly, Lx, 4, 3), dtype=dtype, device=device)
    for r in range(nrhs):
        for s in range(Ls):
            out[r, s] = torch.view_as_complex(torch.randn((Lt, Lz, Ly, Lx, 4, 3, 2), generator=gen_, device=device, dtype=rdt))
    return out
