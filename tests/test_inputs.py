"""Seeded input generators: SU(3) validity, determinism, layout."""
import numpy as np
import pytest

import lattice_inputs as li


@pytest.mark.parametrize("kind,eps", [("random", 0.0), ("near_identity", 0.3)])
def test_links_are_su3(kind, eps):
    u = li.make_links((4, 4, 4, 4), kind, seed=1, eps=eps)
    assert u.shape == (256, 4, 3, 3, 2) and u.dtype == np.float64
    unit, det = li.su3_defects(u)
    assert unit < 1e-14 and det < 1e-14


def test_near_identity_is_near_identity_and_random_is_not():
    near = li.links_as_complex(li.make_links((4, 4, 4, 4), "near_identity", 2, 0.2))
    rnd = li.links_as_complex(li.make_links((4, 4, 4, 4), "random", 2))
    assert np.abs(near - np.eye(3)).max() < 1.0
    assert np.mean(np.abs(np.trace(near, axis1=2, axis2=3)) / 3) > 0.9
    assert np.mean(np.abs(np.trace(rnd, axis1=2, axis2=3)) / 3) < 0.5


def test_deterministic_and_slice_independent():
    a = li.make_links((4, 4, 4, 4), "random", 1)
    b = li.make_links((4, 4, 4, 4), "random", 1)
    assert li.sha256(a) == li.sha256(b)
    # t-slice chunks: a lattice with more t-slices starts with the same slices
    c8 = li.make_links((4, 4, 4, 8), "random", 1)
    assert np.array_equal(c8[:256], a)
    assert li.sha256(li.make_links((4, 4, 4, 4), "random", 2)) != li.sha256(a)


def test_parity_and_source_layout():
    dims = (4, 2, 6, 4)
    par = li.site_parity(dims)
    assert par.sum() * 2 == par.size
    nx = dims[0]
    # with Nx even every (2k, 2k+1) pair of addresses holds one site of each parity
    assert np.array_equal(par[0::2] + par[1::2], np.ones(par.size // 2, dtype=par.dtype))
    full = li.make_full_vector(dims, 3)
    src = li.make_source(dims, 3, 0)
    assert np.array_equal(src, full[par == 0])
    assert src.shape == (par.size // 2, 3, 2)


def test_configs_match_baseline_json():
    c = li.CONFIGS
    assert [c[i].dims for i in range(1, 6)] == [(4, 4, 4, 4), (8, 8, 8, 4), (32, 32, 32, 8),
                                                (48, 48, 48, 12), (64, 64, 64, 16)]
    assert [c[i].mass for i in range(1, 6)] == [0.1, 0.05, 0.02, 0.01, 0.005]
    assert [c[i].nshift for i in range(1, 6)] == [8, 12, 12, 16, 16]
    assert [c[i].tol for i in range(1, 6)] == [1e-10, 1e-10, 1e-10, 1e-12, 1e-10]
    s = li.make_shifts(c[4])
    assert np.isclose(s[0], 1e-6) and np.isclose(s[-1], 4.0) and np.all(np.diff(np.log(s)) > 0)
    assert np.allclose(li.make_residues(c[1]), 1 / np.arange(1, 9))
    r = li.make_residues(c[4])
    assert r.min() >= 0.1 and r.max() <= 1.0 and np.array_equal(r, li.make_residues(c[4]))
