"""Small numpy helpers for the tests (no method arithmetic from either implementation)."""
from __future__ import annotations

import numpy as np


def c(a: np.ndarray) -> np.ndarray:
    """float64[...,2] -> complex128[...]"""
    return a[..., 0] + 1j * a[..., 1]


def f(a: np.ndarray) -> np.ndarray:
    """complex128[...] -> float64[...,2]"""
    return np.ascontiguousarray(np.stack([a.real, a.imag], axis=-1))


def rel_l2(a: np.ndarray, b: np.ndarray) -> float:
    """||a-b||_2 / ||b||_2"""
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def dense_from_operator(apply, nsite: int) -> np.ndarray:
    """Dense complex matrix of a linear map on float64[nsite,3,2] vectors, column by column."""
    n = nsite * 3
    m = np.empty((n, n), dtype=np.complex128)
    e = np.zeros((nsite, 3, 2))
    for j in range(n):
        e.reshape(n, 2)[j, 0] = 1.0
        m[:, j] = c(apply(e)).reshape(n)
        e.reshape(n, 2)[j, 0] = 0.0
    return m


def coords(dims) -> np.ndarray:
    """int[V,4]: (x,y,z,t) of every canonical address l = ((t*Nz+z)*Ny+y)*Nx+x."""
    nx, ny, nz, nt = dims
    l = np.arange(nx * ny * nz * nt)
    x = l % nx
    y = (l // nx) % ny
    z = (l // (nx * ny)) % nz
    t = l // (nx * ny * nz)
    return np.stack([x, y, z, t], axis=1)


def address(dims, x, y, z, t):
    nx, ny, nz, nt = dims
    return ((t * nz + z) * ny + y) * nx + x


def free_spectrum_even(dims, mass: float) -> np.ndarray:
    """Closed form for U = 1 (BASELINE.json north_star):
    eigenvalues of (M^dag M)_ee are m^2 + sum_mu sin^2 p_mu with p_{x,y,z} = 2 pi n/N and
    antiperiodic p_t = 2 pi (n + 1/2)/Nt.  The V momenta pair up as (p, p + (pi,pi,pi,pi))
    with equal values; the even sublattice carries one of each pair, times 3 colours."""
    nx, ny, nz, nt = dims
    px = 2 * np.pi * np.arange(nx) / nx
    py = 2 * np.pi * np.arange(ny) / ny
    pz = 2 * np.pi * np.arange(nz) / nz
    pt = 2 * np.pi * (np.arange(nt) + 0.5) / nt
    s = (np.sin(px)[:, None, None, None] ** 2 + np.sin(py)[None, :, None, None] ** 2
         + np.sin(pz)[None, None, :, None] ** 2 + np.sin(pt)[None, None, None, :] ** 2)
    vals = np.sort(mass ** 2 + s.ravel())
    assert np.allclose(vals[0::2], vals[1::2], atol=1e-13)
    return np.sort(np.repeat(vals[0::2], 3))
