"""Pins for the oracle's CG and multishift CG.

The operator itself is pinned in test_oracle_dslash.py; here the solver is pinned to
LAPACK dense solves, to eq. 8 of the paper through an eigendecomposition, and to
independent single-shift CGs (the checks BASELINE.json north_star lists).
"""
import numpy as np
import pytest

import lattice_inputs as li
import oracle
from helpers import c, dense_from_operator, f, rel_l2


def _setup(dims, kind, mass, seed, eps=0.3):
    u = li.make_links(dims, kind, seed, eps)
    lat = oracle.Lattice(dims, u)
    b = li.make_source(dims, seed, 0)
    a = dense_from_operator(lambda v: lat.mdagm(mass, 0, v), lat.volume // 2)
    return lat, b, a


@pytest.mark.parametrize("dims,kind,mass", [((2, 2, 2, 2), "random", 0.1),
                                            ((4, 4, 4, 4), "random", 0.1),
                                            ((4, 4, 4, 4), "near_identity", 0.05)])
def test_multishift_vs_dense_solve(dims, kind, mass):
    """x_k = (A + sigma_k)^-1 b against numpy.linalg.solve; true residuals recomputed densely."""
    lat, b, a = _setup(dims, kind, mass, seed=1)
    shifts = np.logspace(-4, 0, 8)
    res = 1.0 / (np.arange(8) + 1.0)
    tol = 1e-10
    bc = c(b).ravel()
    out = lat.multishift_cg(mass, 0, b, shifts, res, tol)
    assert out["status"] == 0
    exact = lat.solve_exact(mass, 0, b, shifts, res, tol)
    n = a.shape[0]
    y_dense = np.zeros(n, dtype=complex)
    for k, s in enumerate(shifts):
        xd = np.linalg.solve(a + s * np.eye(n), bc)
        y_dense += res[k] * xd
        # requested tolerance: converged, recomputed residual honest, error within 1e-9 (C17)
        xk = c(out["x"][k]).ravel()
        r_dense = np.linalg.norm(bc - (a + s * np.eye(n)) @ xk) / np.linalg.norm(bc)
        assert abs(out["true_res"][k] - r_dense) < 1e-13
        assert out["true_res"][k] <= 1.5 * tol
        assert rel_l2(xk, xd) < 1e-9
        # polished oracle stands for the exact solution (C16)
        assert rel_l2(c(exact["x"][k]).ravel(), xd) < 2e-13
        assert exact["true_res"][k] < 1e-13
    assert rel_l2(c(exact["y"]).ravel(), y_dense) < 2e-13
    assert rel_l2(c(out["y"]).ravel(), y_dense) < 1e-9


def test_eq8_identity_via_eigh():
    """PAPER.md:133 eq. 8 as a matrix identity: sum_k c_k (A+sigma_k)^-1 b =
    Q diag(sum_k c_k/(lambda_i+sigma_k)) Q^dag b."""
    lat, b, a = _setup((4, 4, 4, 4), "random", 0.1, seed=2)
    shifts = np.logspace(-3, 0.5, 6)
    res = np.array([0.7, -0.2, 1.3, 0.05, 2.0, 0.4])
    lam, q = np.linalg.eigh(a)
    weights = (res[None, :] / (lam[:, None] + shifts[None, :])).sum(axis=1)
    y_ref = q @ (weights * (q.conj().T @ c(b).ravel()))
    exact = lat.solve_exact(0.1, 0, b, shifts, res, 1e-10)
    assert rel_l2(c(exact["y"]).ravel(), y_ref) < 5e-13


def test_multishift_equals_separate_single_shift_cgs():
    """The north_star check: one multishift solve == N separate single-shift CGs."""
    dims, mass = (4, 4, 4, 4), 0.1
    cfg, u, b, shifts, res = li.make_config_inputs(1)
    lat = oracle.Lattice(dims, u)
    tol = 1e-12
    out = lat.multishift_cg(mass, 0, b, shifts, res, tol)
    for k, s in enumerate(shifts):
        xs, its, tr, st = lat.cg(mass, 0, s, b, tol)
        assert st == 0 and tr < 1.5 * tol
        assert its <= out["iterations"]          # shifted systems converge no slower than the base
        assert rel_l2(out["x"][k], xs) < 1e-10


def test_single_shift_cg_vs_dense():
    lat, b, a = _setup((4, 4, 4, 4), "random", 0.1, seed=4)
    x, its, tr, st = lat.cg(0.1, 0, 0.0, b, 1e-13)
    xd = np.linalg.solve(a, c(b).ravel())
    assert st == 0 and rel_l2(c(x).ravel(), xd) < 1e-11


def test_shift_order_and_zero_shift():
    """Unsorted shifts (sigma = 0 allowed, C12) come back in the caller's order."""
    cfg, u, b, _, _ = li.make_config_inputs(1)
    lat = oracle.Lattice(cfg.dims, u)
    shifts = np.array([0.3, 0.0, 1.0, 1e-3])
    res = np.array([1.0, 2.0, 3.0, 4.0])
    perm = np.argsort(shifts)
    o1 = lat.multishift_cg(cfg.mass, 0, b, shifts, res, 1e-11)
    o2 = lat.multishift_cg(cfg.mass, 0, b, shifts[perm], res[perm], 1e-11)
    assert o1["iterations"] == o2["iterations"]
    assert np.array_equal(o1["x"][perm], o2["x"])
    assert np.array_equal(o1["true_res"][perm], o2["true_res"])
    assert rel_l2(o1["y"], o2["y"]) < 1e-15
    x0, _, _, _ = lat.cg(cfg.mass, 0, 0.0, b, 1e-11)
    assert rel_l2(o1["x"][1], x0) < 1e-9


def test_freezing_keeps_large_shifts_finite():
    """C13: 16 shifts up to 4 at light mass; without freezing zeta_k underflows to 0/0.
    With f = 0.1 every shift stays finite and meets the residual bound."""
    dims, mass = (4, 4, 4, 4), 0.005
    u = li.make_links(dims, "random", seed=5)
    lat = oracle.Lattice(dims, u)
    b = li.make_source(dims, 5, 0)
    shifts = np.logspace(-6, np.log10(4.0), 16)
    tol = 1e-10
    out = lat.multishift_cg(mass, 0, b, shifts, np.ones(16), tol)
    assert out["status"] == 0
    assert np.isfinite(out["x"]).all() and np.isfinite(out["y"]).all()
    assert (out["true_res"] <= 1.5 * tol).all()
    assert out["iterations"] > 300


def test_max_iter_reports_not_converged():
    cfg, u, b, shifts, res = li.make_config_inputs(1)
    lat = oracle.Lattice(cfg.dims, u)
    out = lat.multishift_cg(cfg.mass, 0, b, shifts, res, 1e-10, max_iter=5)
    assert out["status"] == 1 and out["iterations"] == 5
    assert (out["true_res"] > 1e-10).any()


def test_config2_iteration_count_is_modest():
    """Near-identity links are well conditioned: tens of iterations."""
    cfg, u, b, shifts, res = li.make_config_inputs(2)
    lat = oracle.Lattice(cfg.dims, u)
    out = lat.multishift_cg(cfg.mass, 0, b, shifts, res, cfg.tol)
    assert out["status"] == 0 and 20 < out["iterations"] < 400
    assert (out["true_res"] <= 1.5 * cfg.tol).all()


def test_polished_oracle_equals_lapack_on_config_2_itself():
    """Config 2 (8^3 x 4, near-identity links, m = 0.05, 12 shifts down to 1e-5) is small enough for LAPACK:
    the 3072 x 3072 matrix of (M^dag M)_ee is assembled column by column from the oracle's operator and every
    shifted system solved densely.  Pins the polished oracle (C16) and the multishift recurrences at one of
    the BASELINE.json configurations themselves, not only on 2^4 and 4^4."""
    cfg, links, b, shifts, res = li.make_config_inputs(2)
    lat = oracle.Lattice(cfg.dims, links)
    a = dense_from_operator(lambda v: lat.mdagm(cfg.mass, 0, v), lat.volume // 2)
    assert np.abs(a - a.conj().T).max() < 1e-14                       # Hermitian
    bc = c(b).ravel()
    n = a.shape[0]
    exact = lat.solve_exact(cfg.mass, 0, b, shifts, res, cfg.tol)
    out = lat.multishift_cg(cfg.mass, 0, b, shifts, res, cfg.tol)
    y = np.zeros(n, dtype=complex)
    for k in (0, 3, 7, 11):
        xd = np.linalg.solve(a + shifts[k] * np.eye(n), bc)
        assert rel_l2(c(exact["x"][k]).ravel(), xd) < 1e-12, k
        assert rel_l2(c(out["x"][k]).ravel(), xd) < 1e-9, k
    lam = np.linalg.eigvalsh(a)
    assert lam.min() > cfg.mass ** 2 and lam.max() < cfg.mass ** 2 + 16.0   # m^2 <= spectrum <= m^2 + 16 (C1)
