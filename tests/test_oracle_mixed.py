"""Pins for oracle/mixed_precision.py: the mixed-precision
variant must land on the solution of the fp64 systems, whatever its inner operator is."""
import numpy as np
import pytest

import lattice_inputs as li
import oracle
from oracle import mixed_precision as mp
from helpers import c, dense_from_operator, rel_l2


def _dense(dims, links, mass):
    lat = oracle.Lattice(dims, links)
    return lat, dense_from_operator(lambda v: lat.mdagm(mass, 0, v), lat.volume // 2)


@pytest.mark.parametrize("kind,mass,nshift,lo", [("random", 0.1, 8, 1e-4), ("near_identity", 0.05, 5, 1e-5),
                                                  ("random", 0.01, 6, 1e-5)])
def test_mixed_precision_lands_on_the_dense_solution(kind, mass, nshift, lo):
    dims, tol = (4, 4, 4, 4), 1e-10
    links = li.make_links(dims, kind, 1, 0.3)
    b = li.make_source(dims, 1, 0)
    shifts = np.logspace(np.log10(lo), 0, nshift)
    res = 1.0 / (np.arange(nshift) + 1.0)
    lat, a = _dense(dims, links, mass)
    out = mp.mixed_precision_multishift(dims, links, mass, 0, b, shifts, res, tol, switch_tol=1e-4)
    bc = c(b).ravel()
    n = a.shape[0]
    y = np.zeros(n, dtype=complex)
    for k, s in enumerate(shifts):
        xd = np.linalg.solve(a + s * np.eye(n), bc)
        y += res[k] * xd
        xk = c(out["x"][k]).ravel()
        assert rel_l2(xk, xd) <= 1e-9, (k, rel_l2(xk, xd))
        r_dense = np.linalg.norm(bc - (a + s * np.eye(n)) @ xk) / np.linalg.norm(bc)
        assert r_dense <= tol * (1 + 1e-6) and abs(out["true_res"][k] - r_dense) <= 1e-13
    assert rel_l2(c(out["y"]).ravel(), y) <= 1e-9
    # stage 1 stopped early (on the base system's residual), stage 2 did the rest, at least for the base shift
    assert out["stage1_res"][0] > tol and out["rounds"][0] >= 1 and out["inner_iterations"][0] > 0
    assert (out["stage1_res"] <= 1.5e-4).all()
    full = lat.multishift_cg(mass, 0, b, shifts, res, tol, want_x=False)["iterations"]
    assert out["stage1_iterations"] < full


def test_inner_operator_is_the_fp32_rounded_field():
    dims, mass = (4, 4, 4, 4), 0.1
    links = li.make_links(dims, "random", 3)
    l32 = mp.round_links_fp32(links)
    assert l32.dtype == np.float64 and np.array_equal(l32, l32.astype(np.float32).astype(np.float64))
    assert 1e-9 < np.abs(l32 - links).max() <= 2.0 ** -25          # |entries| <= 1: half an fp32 ulp
    v = li.make_source(dims, 4, 0)
    a64 = oracle.Lattice(dims, links).mdagm(mass, 0, v)
    a32 = oracle.Lattice(dims, l32).mdagm(mass, 0, v)
    assert 1e-9 < rel_l2(a32, a64) < 1e-6


def test_fixed_point_does_not_depend_on_the_inner_operator():
    """The outer residual is formed with the fp64 operator, so an inner field that is wrong by 1e-3
    (not 6e-8) only costs more rounds."""
    dims, mass, tol = (4, 4, 4, 4), 0.1, 1e-10
    links = li.make_links(dims, "random", 5)
    b = li.make_source(dims, 5, 0)
    shifts, res = np.array([1e-3, 0.1, 1.0]), np.ones(3)
    rng = np.random.default_rng(7)
    bad = links + 1e-3 * rng.standard_normal(links.shape)
    good = mp.mixed_precision_multishift(dims, links, mass, 0, b, shifts, res, tol, switch_tol=1e-3)
    worse = mp.mixed_precision_multishift(dims, links, mass, 0, b, shifts, res, tol, switch_tol=1e-3,
                                          inner_links=bad)
    exact = oracle.Lattice(dims, links).solve_exact(mass, 0, b, shifts, res, tol)
    for k in range(3):
        assert rel_l2(good["x"][k], exact["x"][k]) <= 1e-9 and rel_l2(worse["x"][k], exact["x"][k]) <= 1e-9
    assert worse["rounds"].sum() > good["rounds"].sum()
    assert (good["true_res"] <= tol).all() and (worse["true_res"] <= tol).all()


def test_switch_at_the_target_is_the_plain_solver():
    dims, mass, tol = (4, 4, 4, 4), 0.1, 1e-10
    cfg, links, b, shifts, res = li.make_config_inputs(1)
    out = mp.mixed_precision_multishift(dims, links, mass, 0, b, shifts, res, tol, switch_tol=tol)
    ref = oracle.Lattice(dims, links).multishift_cg(mass, 0, b, shifts, res, tol)
    assert out["stage1_iterations"] == ref["iterations"]
    # shifts already below tol after stage 1 are untouched; the others get a (small) correction
    for k in range(len(shifts)):
        if out["rounds"][k] == 0:
            assert np.array_equal(out["x"][k], ref["x"][k])
    assert (out["true_res"] <= tol).all()
