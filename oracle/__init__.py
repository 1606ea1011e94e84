"""CPU oracle (TEST INFRASTRUCTURE, not the product).

ctypes front end of `staggered_oracle.c`: a plain fp64 C/OpenMP restatement of
the staggered D_oe/D_eo, (M^dag M)_ee and the multishift CG of arXiv:1710.09178
(SURVEY.md 8(c)).  Only tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / `--impl reference` legs may import this package;
`paper_1710_09178_b200` never does, and this package never imports it.

All arrays are numpy float64 in the canonical layout documented in
staggered_oracle.c (links [V,4,3,3,2]; parity vectors [V/2,3,2]).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "staggered_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

_c_double_p = ctypes.POINTER(ctypes.c_double)
_c_int_p = ctypes.POINTER(ctypes.c_int)


def build(force: bool = False) -> str:
    """Compile staggered_oracle.c with gcc (-O2 -fopenmp) into oracle/liboracle.so."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    tmp = _LIB + f".{os.getpid()}.tmp"
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-o", tmp, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = ctypes.CDLL(build())
    vp = ctypes.c_void_p
    lib.orc_create.restype = vp
    lib.orc_create.argtypes = [_c_int_p, _c_double_p]
    lib.orc_destroy.argtypes = [vp]
    lib.orc_threads.restype = ctypes.c_int
    lib.orc_set_threads.argtypes = [ctypes.c_int]
    lib.orc_D_full.argtypes = [vp, _c_double_p, _c_double_p]
    lib.orc_dslash.argtypes = [vp, ctypes.c_int, _c_double_p, _c_double_p]
    lib.orc_mdagm.argtypes = [vp, ctypes.c_double, ctypes.c_int, _c_double_p, _c_double_p]
    lib.orc_cg.restype = ctypes.c_int
    lib.orc_cg.argtypes = [vp, ctypes.c_double, ctypes.c_int, ctypes.c_double, _c_double_p,
                           _c_double_p, ctypes.c_double, ctypes.c_int, _c_int_p, _c_double_p]
    lib.orc_multishift_cg.restype = ctypes.c_int
    lib.orc_multishift_cg.argtypes = [vp, ctypes.c_double, ctypes.c_int, _c_double_p, ctypes.c_int,
                                      _c_double_p, _c_double_p, ctypes.c_double, ctypes.c_int,
                                      ctypes.c_double, _c_double_p, _c_double_p, _c_int_p,
                                      _c_double_p]
    lib.orc_polish.restype = ctypes.c_double
    lib.orc_polish.argtypes = [vp, ctypes.c_double, ctypes.c_int, ctypes.c_double, _c_double_p,
                               _c_double_p, ctypes.c_int, ctypes.c_int]
    _lib = lib
    return lib


def threads() -> int:
    """OpenMP threads the oracle will use."""
    return int(_load().orc_threads())


def set_threads(n: int) -> None:
    _load().orc_set_threads(int(n))


def _p(a: np.ndarray):
    return a.ctypes.data_as(_c_double_p)


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


FREEZE_FACTOR = 0.1  # f of SURVEY.md C13


class Lattice:
    """Gauge field + lattice geometry the oracle's operators act with."""

    def __init__(self, dims, links: np.ndarray):
        self.dims = tuple(int(d) for d in dims)
        self.volume = int(np.prod(self.dims))
        self.links = _f64(links)
        if self.links.size != self.volume * 72:
            raise ValueError("links must hold 72*V doubles (PAPER.md:43)")
        self._lib = _load()
        cd = (ctypes.c_int * 4)(*self.dims)
        self._h = self._lib.orc_create(cd, _p(self.links))
        if not self._h:
            raise MemoryError("orc_create failed")

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h:
            self._lib.orc_destroy(h)

    @property
    def half_shape(self):
        return (self.volume // 2, 3, 2)

    def D_full(self, psi: np.ndarray) -> np.ndarray:
        """(D psi) on the full lattice; psi float64[V,3,2]."""
        psi = _f64(psi)
        out = np.empty_like(psi)
        self._lib.orc_D_full(self._h, _p(psi), _p(out))
        return out

    def dslash(self, out_parity: int, v: np.ndarray) -> np.ndarray:
        """D_{out_parity,other} v ; v lives on parity 1-out_parity."""
        v = _f64(v)
        out = np.empty(self.half_shape)
        self._lib.orc_dslash(self._h, int(out_parity), _p(v), _p(out))
        return out

    def mdagm(self, mass: float, parity: int, v: np.ndarray) -> np.ndarray:
        """(M^dag M)_pp v = m^2 v - D_pq D_qp v."""
        v = _f64(v)
        out = np.empty(self.half_shape)
        self._lib.orc_mdagm(self._h, float(mass), int(parity), _p(v), _p(out))
        return out

    def cg(self, mass, parity, sigma, b, tol, max_iter=100000, x0=None):
        """Single-shift CG on (M^dag M + sigma). Returns (x, iterations, true_res, status)."""
        b = _f64(b)
        x = np.zeros(self.half_shape) if x0 is None else _f64(x0).copy()
        it = ctypes.c_int(0)
        tr = ctypes.c_double(0.0)
        st = self._lib.orc_cg(self._h, float(mass), int(parity), float(sigma), _p(b), _p(x),
                              float(tol), int(max_iter), ctypes.byref(it), ctypes.byref(tr))
        return x, it.value, tr.value, st

    def multishift_cg(self, mass, parity, b, shifts, residues, tol, max_iter=100000,
                      freeze_factor=FREEZE_FACTOR, want_x=True):
        """SURVEY.md 8(c.2). Returns dict(x, y, iterations, true_res, status)."""
        b = _f64(b)
        shifts = _f64(shifts)
        residues = _f64(residues)
        n = shifts.size
        x = np.empty((n,) + self.half_shape) if want_x else None
        y = np.empty(self.half_shape)
        tr = np.empty(n)
        it = ctypes.c_int(0)
        st = self._lib.orc_multishift_cg(
            self._h, float(mass), int(parity), _p(b), n, _p(shifts), _p(residues), float(tol),
            int(max_iter), float(freeze_factor), _p(x) if want_x else None, _p(y),
            ctypes.byref(it), _p(tr))
        return dict(x=x, y=y, iterations=it.value, true_res=tr, status=st)

    def polish(self, mass, parity, sigma, b, x, max_rounds=6, max_iter=100000) -> float:
        """Defect-correct x in place towards the fp64 floor (C16); returns true residual."""
        b = _f64(b)
        assert x.dtype == np.float64 and x.flags.c_contiguous
        return float(self._lib.orc_polish(self._h, float(mass), int(parity), float(sigma), _p(b),
                                          _p(x), int(max_rounds), int(max_iter)))

    def solve_exact(self, mass, parity, b, shifts, residues, tol, max_iter=100000):
        """The oracle's stand-in for the exact x_k: multishift CG at
        tol_oracle = min(tol*1e-3, 1e-13), then each shift polished to the floor.
        Returns dict(x, y, true_res, iterations)."""
        shifts = _f64(shifts)
        residues = _f64(residues)
        tol_o = min(tol * 1e-3, 1e-13)
        out = self.multishift_cg(mass, parity, b, shifts, residues, tol_o, max_iter)
        x = out["x"]
        tr = np.empty(shifts.size)
        for k in range(shifts.size):
            tr[k] = self.polish(mass, parity, shifts[k], b, x[k], max_iter=max_iter)
        y = np.tensordot(residues, x, axes=(0, 0))
        return dict(x=x, y=y, true_res=tr, iterations=out["iterations"])


# ---------------------------------------------------------------------------------------------
# NEXT-1: two-row link storage.  PAPER.md:168: "one often stores and moves only
# two rows (or columns) of the (3 x 3) complex link matrix and recovers the third by
# orthogonalization.  This is often known as data compression."  For U in SU(3) the rows are
# orthonormal and det U = 1, which fixes the third row uniquely: row_2 = conj(row_0 x row_1)
# (the complex cross product).  The definition is written out below with plain numpy; the
# operator itself is unchanged, so the oracle for the compressed Dslash is Lattice(...) built on
# reconstruct_links_2row(compress_links_2row(U)).
# Pins (tests/test_oracle_compression.py): hand-written SU(3) matrices (diagonal phases, a cyclic
# permutation, a real rotation), det/unitarity of the result for arbitrary orthonormal rows,
# identity with the input on the seeded SU(3) generators.

def compress_links_2row(links: np.ndarray) -> np.ndarray:
    """float64[V,4,3,3,2] -> float64[V,4,2,3,2]: rows 0 and 1 of every link, bit for bit."""
    links = _f64(links)
    v = links.size // 72
    return np.ascontiguousarray(links.reshape(v, 4, 3, 3, 2)[:, :, :2])


def reconstruct_links_2row(rows: np.ndarray) -> np.ndarray:
    """float64[V,4,2,3,2] -> float64[V,4,3,3,2] with row_2 = conj(row_0 x row_1), i.e.
    row_2[c] = conj(row_0[c+1] row_1[c+2] - row_0[c+2] row_1[c+1]), indices mod 3."""
    rows = _f64(rows)
    a = rows[:, :, 0, :, 0] + 1j * rows[:, :, 0, :, 1]      # row 0: complex[V,4,3]
    b = rows[:, :, 1, :, 0] + 1j * rows[:, :, 1, :, 1]      # row 1
    third = np.empty_like(a)
    for c in range(3):
        c1, c2 = (c + 1) % 3, (c + 2) % 3
        third[:, :, c] = np.conj(a[:, :, c1] * b[:, :, c2] - a[:, :, c2] * b[:, :, c1])
    out = np.empty(rows.shape[:2] + (3, 3, 2))
    out[:, :, :2] = rows
    out[:, :, 2, :, 0] = third.real
    out[:, :, 2, :, 1] = third.imag
    return out
