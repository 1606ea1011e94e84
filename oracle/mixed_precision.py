"""CPU oracle (TEST INFRASTRUCTURE, not the product) for SURVEY.md 8(f) NEXT-3: the mixed-precision
variant of the multishift solve.

PAPER.md:168: "Mixed precision routines are often used to boost performance ... led to convergence
problems for the multi-shift conjugate gradient [25].  We therefore use fully double precision
routines."  The paper does not print a mixed-precision algorithm; the one restated here is the usual
way round the problem it names (reading N3): the shifted systems share one Krylov space only
while all residuals stay collinear, which a low-precision operator with fp64 corrections destroys, so

  stage 1   the paper's solver as it stands (fp64 multishift CG) down to a LOOSE
            tolerance switch_tol >= tol;
  stage 2   every shift on its own, by defect correction (iterative refinement):
                r   = b - (A + sigma_k) x_k          recomputed with the fp64 operator A
                stop when ||r|| <= tol ||b||
                e  ~= (A32 + sigma_k)^-1 r           plain CG, x0 = 0, to ||r_in|| <= tau ||r||, with the
                                                     INNER operator A32 = M^dag M built on the links
                                                     rounded to fp32 (arithmetic stays fp64)
                x_k += e
            tau = max(tol ||b|| / (2 ||r||), inner_floor): one round if the inner operator allows it,
            never asked for more than inner_floor = 1e-2 per round beyond that, because the round
            cannot gain more than ~ kappa_k * 2^-24 anyway.

The fixed point of stage 2 is the solution of the fp64 system (the outer residual uses A), whatever
A32 is, as long as the rounds contract; only the number of rounds depends on the rounding.

Everything is written with the primitives of oracle.Lattice (mdagm, cg, multishift_cg), which are
pinned in tests/test_oracle_*.py; this file adds no operator arithmetic of its own.  Pins
(tests/test_oracle_mixed.py): the result against numpy.linalg.solve on 4^4 (<= 1e-9), the recomputed
fp64 residual <= tol for every shift, the inner operator differing from A at the fp32 level (1e-8 ..
1e-6, not 0), stage 2 doing work (stage-1 residual above tol), and the fixed point being independent
of the inner operator (a deliberately worse inner field still lands on the same x).
"""
from __future__ import annotations

import numpy as np

from . import Lattice

INNER_FLOOR = 1e-2      # largest reduction asked of one inner solve
MAX_ROUNDS = 60


def round_links_fp32(links: np.ndarray) -> np.ndarray:
    """The inner field: every link entry rounded to fp32 (round to nearest even), kept as float64."""
    return np.ascontiguousarray(links, dtype=np.float64).astype(np.float32).astype(np.float64)


def mixed_precision_multishift(dims, links, mass, parity, b, shifts, residues, tol, switch_tol=1e-5,
                               inner_links=None, inner_floor=INNER_FLOOR, max_iter=100000):
    """Returns dict(x, y, true_res, stage1_iterations, inner_iterations[k], rounds[k], stage1_res[k]).
    inner_links: the field of the inner operator (default: round_links_fp32(links))."""
    outer = Lattice(dims, links)
    inner = Lattice(dims, round_links_fp32(links) if inner_links is None else inner_links)
    shifts = np.ascontiguousarray(shifts, dtype=np.float64)
    residues = np.ascontiguousarray(residues, dtype=np.float64)
    nb = np.linalg.norm(b)
    # stage 1: the fp64 multishift CG of SURVEY.md 8(c.2), loose
    s1 = outer.multishift_cg(mass, parity, b, shifts, residues, max(tol, switch_tol), max_iter)
    x = s1["x"]
    n = shifts.size
    rounds = np.zeros(n, dtype=int)
    inner_its = np.zeros(n, dtype=int)
    true_res = np.empty(n)
    stage1_res = np.empty(n)
    # stage 2: defect correction, one shift at a time
    for k in range(n):
        for rnd in range(MAX_ROUNDS + 1):
            r = b - (outer.mdagm(mass, parity, x[k]) + shifts[k] * x[k])      # fp64 operator
            nr = np.linalg.norm(r)
            if rnd == 0:
                stage1_res[k] = nr / nb if nb > 0 else 0.0
            true_res[k] = nr / nb if nb > 0 else 0.0
            if nr <= tol * nb or rnd == MAX_ROUNDS:
                break
            tau = max(0.5 * tol * nb / nr, inner_floor)
            e, its, _, _ = inner.cg(mass, parity, shifts[k], r, tau, max_iter)   # fp32-rounded links
            x[k] += e
            rounds[k] += 1
            inner_its[k] += its
    y = np.tensordot(residues, x, axes=(0, 0))
    return dict(x=x, y=y, true_res=true_res, stage1_iterations=s1["iterations"], inner_iterations=inner_its,
                rounds=rounds, stage1_res=stage1_res)
