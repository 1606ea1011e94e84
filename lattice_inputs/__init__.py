"""Seeded synthetic inputs for the staggered Dslash / multishift-CG hot path.

This module is the ONLY code shared by the CPU oracle's tests and the CUDA
path's tests/bench.  It holds none of the method's arithmetic (no Dslash, no
M^dag M, no CG): it only draws SU(3) links, Gaussian sources, shifts and
residues, in the *canonical* exchange layout:

  site address  l = ((t*Nz + z)*Ny + y)*Nx + x      (made 0-based)
  links         float64[V, 4, 3, 3, 2]  = [l][mu][row][col][re,im]   (72 V doubles)
  parity vector float64[V/2, 3, 2]      = [j][colour][re,im], j enumerating the
                sites of one parity in increasing l                  (6 V doubles full)

The five configurations are the ones BASELINE.json lists;
they stand in for the paper's thermalised beta=5.6 ensembles,
which do not exist in this container.

RNG recipe: numpy.random.default_rng([seed, stream, chunk]),
PCG64; seed = config number; stream 0 = links, 1 = source, 2 = residues;
chunk = t-slice index, so every t-slice is generated independently.
"""
from __future__ import annotations

import dataclasses
import hashlib

import numpy as np

STREAM_LINKS, STREAM_SOURCE, STREAM_RESIDUES = 0, 1, 2


@dataclasses.dataclass(frozen=True)
class Config:
    """One BASELINE.json workload."""

    number: int
    dims: tuple  # (Nx, Ny, Nz, Nt)
    mass: float
    links: str  # "random" | "near_identity"
    eps: float  # near-identity step (0 for random)
    nshift: int
    shift_lo: float
    shift_hi: float
    residues: str  # "harmonic" 1/(k+1) | "ones" | "uniform" in [0.1, 1]
    tol: float
    parity: int = 0  # all configs solve on the even parity

    @property
    def seed(self) -> int:
        return self.number

    @property
    def volume(self) -> int:
        nx, ny, nz, nt = self.dims
        return nx * ny * nz * nt

    @property
    def name(self) -> str:
        nx, ny, nz, nt = self.dims
        return f"cfg{self.number}_{nx}x{ny}x{nz}x{nt}"


# BASELINE.json "configs" (1-based numbering as in SURVEY.md 8(d)).  Where
# BASELINE.json leaves a value open the SURVEY.md 8(d) reading is used:
# cfg 3 shifts in [1e-5, 2] and residues 1.0; cfg 5 residues 1.0.
CONFIGS = {
    1: Config(1, (4, 4, 4, 4), 0.1, "random", 0.0, 8, 1e-4, 1.0, "harmonic", 1e-10),
    2: Config(2, (8, 8, 8, 4), 0.05, "near_identity", 0.3, 12, 1e-5, 2.0, "ones", 1e-10),
    3: Config(3, (32, 32, 32, 8), 0.02, "near_identity", 0.2, 12, 1e-5, 2.0, "ones", 1e-10),
    4: Config(4, (48, 48, 48, 12), 0.01, "near_identity", 0.2, 16, 1e-6, 4.0, "uniform", 1e-12),
    5: Config(5, (64, 64, 64, 16), 0.005, "random", 0.0, 16, 1e-6, 4.0, "ones", 1e-10),
}


def _slice_sites(dims) -> int:
    nx, ny, nz, _ = dims
    return nx * ny * nz


def _project_su3(m: np.ndarray) -> np.ndarray:
    """Row Gram-Schmidt + conjugate cross product: complex (N,3,3) -> SU(3).

    row1 = m1/|m1|; row2 = m2 - <row1,m2> row1, normalised; row3 = conj(row1 x row2)
    (BASELINE.json config 1).  det = 1 by construction.
    """
    r1 = m[:, 0, :]
    r1 = r1 / np.linalg.norm(r1, axis=1, keepdims=True)
    r2 = m[:, 1, :]
    r2 = r2 - np.sum(np.conj(r1) * r2, axis=1, keepdims=True) * r1
    r2 = r2 / np.linalg.norm(r2, axis=1, keepdims=True)
    r3 = np.conj(np.cross(r1, r2))
    return np.stack([r1, r2, r3], axis=1)


def _complex_gauss(rng: np.random.Generator, shape) -> np.ndarray:
    """Entries N(0,1) + i N(0,1)."""
    re = rng.standard_normal(shape)
    im = rng.standard_normal(shape)
    return re + 1j * im


def _links_slice_random(rng: np.random.Generator, n: int) -> np.ndarray:
    return _project_su3(_complex_gauss(rng, (n, 3, 3)))


def _links_slice_near_identity(rng: np.random.Generator, n: int, eps: float) -> np.ndarray:
    """U = exp(i eps H), H traceless Hermitian Gaussian, projected back to SU(3)."""
    g = _complex_gauss(rng, (n, 3, 3)) / np.sqrt(2.0)
    h = 0.5 * (g + np.conj(np.swapaxes(g, 1, 2)))
    tr = np.trace(h, axis1=1, axis2=2) / 3.0
    h = h - tr[:, None, None] * np.eye(3)[None]
    w, q = np.linalg.eigh(h)
    u = (q * np.exp(1j * eps * w)[:, None, :]) @ np.conj(np.swapaxes(q, 1, 2))
    return _project_su3(u)


def unit_links(dims) -> np.ndarray:
    """Free field U = 1 in canonical layout (used by closed-form pins)."""
    nx, ny, nz, nt = dims
    v = nx * ny * nz * nt
    u = np.zeros((v, 4, 3, 3, 2), dtype=np.float64)
    for c in range(3):
        u[:, :, c, c, 0] = 1.0
    return u


def make_links(dims, kind: str, seed: int, eps: float = 0.0) -> np.ndarray:
    """Canonical gauge field float64[V,4,3,3,2], generated t-slice by t-slice."""
    nt = dims[3]
    n3 = _slice_sites(dims)
    out = np.empty((nt * n3, 4, 3, 3, 2), dtype=np.float64)
    for t in range(nt):
        rng = np.random.default_rng([seed, STREAM_LINKS, t])
        if kind == "random":
            u = _links_slice_random(rng, n3 * 4)
        elif kind == "near_identity":
            u = _links_slice_near_identity(rng, n3 * 4, eps)
        else:
            raise ValueError(f"unknown link kind {kind!r}")
        blk = out[t * n3:(t + 1) * n3].reshape(n3 * 4, 3, 3, 2)
        blk[..., 0] = u.real
        blk[..., 1] = u.imag
    return out


def random_su3_field(dims, seed: int, stream: int = 7) -> np.ndarray:
    """One random SU(3) matrix per site, complex128[V,3,3] (gauge-transform tests)."""
    nt = dims[3]
    n3 = _slice_sites(dims)
    out = np.empty((nt * n3, 3, 3), dtype=np.complex128)
    for t in range(nt):
        rng = np.random.default_rng([seed, stream, t])
        out[t * n3:(t + 1) * n3] = _links_slice_random(rng, n3)
    return out


def site_parity(dims) -> np.ndarray:
    """int8[V]: (x+y+z+t) mod 2 for every canonical address l."""
    nx, ny, nz, nt = dims
    x = np.arange(nx)[None, None, None, :]
    y = np.arange(ny)[None, None, :, None]
    z = np.arange(nz)[None, :, None, None]
    t = np.arange(nt)[:, None, None, None]
    return ((x + y + z + t) & 1).astype(np.int8).reshape(-1)


def make_full_vector(dims, seed: int, stream: int = STREAM_SOURCE) -> np.ndarray:
    """Complex Gaussian on every site, float64[V,3,2]."""
    nt = dims[3]
    n3 = _slice_sites(dims)
    out = np.empty((nt * n3, 3, 2), dtype=np.float64)
    for t in range(nt):
        rng = np.random.default_rng([seed, stream, t])
        out[t * n3:(t + 1) * n3, :, 0] = rng.standard_normal((n3, 3))
        out[t * n3:(t + 1) * n3, :, 1] = rng.standard_normal((n3, 3))
    return out


def make_source(dims, seed: int, parity: int = 0, stream: int = STREAM_SOURCE) -> np.ndarray:
    """Complex Gaussian source on the sites of one parity, float64[V/2,3,2]."""
    full = make_full_vector(dims, seed, stream)
    return np.ascontiguousarray(full[site_parity(dims) == parity])


def make_shifts(cfg: Config) -> np.ndarray:
    """sigma_k log-spaced in [shift_lo, shift_hi] (numpy.logspace)."""
    return np.logspace(np.log10(cfg.shift_lo), np.log10(cfg.shift_hi), cfg.nshift)


def make_residues(cfg: Config) -> np.ndarray:
    if cfg.residues == "harmonic":
        return 1.0 / (np.arange(cfg.nshift) + 1.0)
    if cfg.residues == "ones":
        return np.ones(cfg.nshift)
    if cfg.residues == "uniform":
        rng = np.random.default_rng([cfg.seed, STREAM_RESIDUES, 0])
        return rng.uniform(0.1, 1.0, cfg.nshift)
    raise ValueError(cfg.residues)


def make_config_inputs(number: int, dims=None):
    """(cfg, links, source, shifts, residues) for BASELINE.json config `number`.

    `dims` overrides the lattice extents (same recipe on a smaller lattice, used
    by tests that need the config's distribution but not its size).
    """
    cfg = CONFIGS[number]
    if dims is not None:
        cfg = dataclasses.replace(cfg, dims=tuple(dims))
    links = make_links(cfg.dims, cfg.links, cfg.seed, cfg.eps)
    src = make_source(cfg.dims, cfg.seed, cfg.parity)
    return cfg, links, src, make_shifts(cfg), make_residues(cfg)


def links_as_complex(links: np.ndarray) -> np.ndarray:
    """float64[V,4,3,3,2] -> complex128[V,4,3,3] (copy)."""
    return links[..., 0] + 1j * links[..., 1]


def su3_defects(links: np.ndarray):
    """(max |U U^dag - 1|, max |det U - 1|) over all links: generator self-check."""
    u = links_as_complex(links).reshape(-1, 3, 3)
    uu = u @ np.conj(np.swapaxes(u, 1, 2)) - np.eye(3)[None]
    return float(np.abs(uu).max()), float(np.abs(np.linalg.det(u) - 1.0).max())


def sha256(a: np.ndarray) -> str:
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()
