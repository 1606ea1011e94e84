"""Pins for the oracle's D, D_oe/D_eo and M^dag M.

Each test pins the oracle to something other than itself: a closed form, an
invariant, hand-derived matrix elements, or brute force through a different
route.  A dropped 1/2, a wrong sign/phase/boundary, a transposed or misplaced
link each fail at least one of them.
"""
import os

import numpy as np
import pytest

import lattice_inputs as li
import oracle
from helpers import address, c, coords, dense_from_operator, f, free_spectrum_even, rel_l2

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "dslash_matrix_elements.txt")


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 4, 4, 4), (4, 4, 2, 6), (2, 4, 6, 2)])
def test_free_field_spectrum(dims):
    """U = 1: spec (M^dag M)_ee = { m^2 + sum_mu sin^2 p_mu }, antiperiodic p_t (north_star)."""
    mass = 0.1
    lat = oracle.Lattice(dims, li.unit_links(dims))
    nh = lat.volume // 2
    a = dense_from_operator(lambda v: lat.mdagm(mass, 0, v), nh)
    assert np.abs(a - a.conj().T).max() < 1e-14
    ev = np.linalg.eigvalsh(a)
    expect = free_spectrum_even(dims, mass)
    assert np.abs(ev - expect).max() < 2e-13
    # antiperiodic, not periodic, in t: the smallest eigenvalue is m^2 + sin^2(pi/Nt), not m^2
    assert abs(ev[0] - (mass ** 2 + np.sin(np.pi / dims[3]) ** 2)) < 2e-13


def test_free_field_all_ones_on_2to4():
    """2^4, U = 1: every momentum has sin^2 p = 0 in x,y,z and 1 in t, so M^dag M = (1+m^2) 1 (C8)."""
    dims, mass = (2, 2, 2, 2), 0.3
    lat = oracle.Lattice(dims, li.unit_links(dims))
    a = dense_from_operator(lambda v: lat.mdagm(mass, 0, v), lat.volume // 2)
    assert np.abs(a - (1 + mass ** 2) * np.eye(a.shape[0])).max() < 1e-14


@pytest.mark.parametrize("dims,n", [((4, 4, 4, 4), (1, 0, 3, 2)), ((4, 6, 2, 8), (3, 5, 1, 6))])
def test_plane_wave(dims, n):
    """U = 1, psi = e^{ip.x} v on the full lattice: D^2 psi = -(sum_mu sin^2 p_mu) psi."""
    lat = oracle.Lattice(dims, li.unit_links(dims))
    xyzt = coords(dims)
    p = np.array([2 * np.pi * n[0] / dims[0], 2 * np.pi * n[1] / dims[1],
                  2 * np.pi * n[2] / dims[2], 2 * np.pi * (n[3] + 0.5) / dims[3]])
    v = np.array([0.3 - 1.1j, 2.0 + 0.5j, -0.7j])
    psi = np.exp(1j * xyzt @ p)[:, None] * v[None, :]
    d2 = c(lat.D_full(lat.D_full(f(psi))))
    assert rel_l2(d2, -(np.sin(p) ** 2).sum() * psi) < 1e-14


@pytest.mark.parametrize("kind,dims", [("random", (4, 4, 4, 4)), ("random", (2, 2, 2, 2)),
                                       ("near_identity", (4, 6, 2, 4))])
def test_anti_hermiticity(kind, dims):
    """<chi, D psi> = -<D chi, psi>  (PAPER.md:114 as read in SURVEY.md C3)."""
    u = li.make_links(dims, kind, seed=11, eps=0.3)
    lat = oracle.Lattice(dims, u)
    chi = c(li.make_full_vector(dims, 21))
    psi = c(li.make_full_vector(dims, 22))
    lhs = np.vdot(chi, c(lat.D_full(f(psi))))
    rhs = -np.vdot(c(lat.D_full(f(chi))), psi)
    assert abs(lhs - rhs) < 1e-12 * abs(lhs)
    # half-lattice form: <chi_o, D_oe psi_e> = -conj <psi_e, D_eo chi_o>
    par = li.site_parity(dims)
    chi_o, psi_e = f(chi[par == 1]), f(psi[par == 0])
    lhs = np.vdot(c(chi_o), c(lat.dslash(1, psi_e)))
    rhs = -np.conj(np.vdot(c(psi_e), c(lat.dslash(0, chi_o))))
    assert abs(lhs - rhs) < 1e-12 * abs(lhs)


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 4, 2, 6)])
def test_D_connects_opposite_parities_only(dims):
    """D_ee = D_oo = 0 (block form PAPER.md:112) with parity = (x+y+z+t) mod 2 (C2)."""
    u = li.make_links(dims, "random", seed=3)
    lat = oracle.Lattice(dims, u)
    par = li.site_parity(dims)
    psi = c(li.make_full_vector(dims, 5))
    for p in (0, 1):
        only_p = psi * (par == p)[:, None]
        out = c(lat.D_full(f(only_p)))
        assert np.abs(out[par == p]).max() == 0.0
        assert np.abs(out[par != p]).max() > 0.1
        # and the half-lattice operator is exactly that restriction
        half = c(lat.dslash(1 - p, f(psi[par == p])))
        assert np.abs(half - out[par != p]).max() == 0.0


def _shift_field(a, dims, mu, step):
    """a[l] -> a[l + step*mu_hat] with periodic wrap; a has leading axis V."""
    nx, ny, nz, nt = dims
    g = a.reshape((nt, nz, ny, nx) + a.shape[1:])
    return np.roll(g, -step, axis=3 - mu).reshape(a.shape)


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 2, 2, 2), (4, 2, 6, 4)])
def test_gauge_covariance(dims):
    """D[U^g](g psi) = g D[U] psi with U^g_mu(x) = g(x) U_mu(x) g(x+mu)^dag (C7)."""
    u = li.links_as_complex(li.make_links(dims, "random", seed=9))
    g = li.random_su3_field(dims, seed=10)
    psi = c(li.make_full_vector(dims, 12))
    ug = np.empty_like(u)
    for mu in range(4):
        g_fwd = _shift_field(g, dims, mu, 1)
        ug[:, mu] = g @ u[:, mu] @ np.conj(np.swapaxes(g_fwd, 1, 2))
    lat = oracle.Lattice(dims, f(u))
    lat_g = oracle.Lattice(dims, f(ug))
    gpsi = np.einsum("lab,lb->la", g, psi)
    lhs = c(lat_g.D_full(f(gpsi)))
    rhs = np.einsum("lab,lb->la", g, c(lat.D_full(f(psi))))
    assert rel_l2(lhs, rhs) < 1e-14


def _golden_rows():
    rows = []
    with open(GOLDEN) as fh:
        for line in fh:
            line = line.split("#")[0].strip()
            if not line:
                continue
            t = line.split()
            rows.append((tuple(map(int, t[0:4])), tuple(map(int, t[4:8])), int(t[8]), t[9],
                         float(t[10])))
    return rows


def test_hand_derived_matrix_elements():
    """tests/golden/dslash_matrix_elements.txt: D(x,x') = c U_mu(x) or c U_mu(x')^dag, derived by hand."""
    dims = (4, 4, 4, 4)
    ulinks = li.make_links(dims, "random", seed=1)
    u = li.links_as_complex(ulinks)
    lat = oracle.Lattice(dims, ulinks)
    rows = _golden_rows()
    assert len(rows) >= 16
    for xo, xi, mu, kind, coeff in rows:
        lo, lin = address(dims, *xo), address(dims, *xi)
        block = coeff * (u[lo, mu] if kind == "F" else u[lin, mu].conj().T)
        for b in range(3):
            src = np.zeros((lat.volume, 3), dtype=complex)
            src[lin, b] = 1.0
            out = c(lat.D_full(f(src)))
            assert np.abs(out[lo] - block[:, b]).max() < 1e-15, (xo, xi, mu, kind)
            # a column of D has exactly 8 non-zero sites on 4^4
            assert (np.abs(out).max(axis=1) > 0).sum() == 8


def test_mdagm_is_ee_block_of_dense_MdagM():
    """(M^dag M)_ee = m^2 - D_eo D_oe equals the ee block of (m+D)^dag (m+D); off-diagonal blocks
    vanish; spec_ee = spec_oo; lambda_min >= m^2."""
    dims, mass = (4, 4, 4, 4), 0.1
    ulinks = li.make_links(dims, "random", seed=1)
    lat = oracle.Lattice(dims, ulinks)
    v = lat.volume
    d = dense_from_operator(lat.D_full, v)
    assert np.abs(d + d.conj().T).max() < 1e-15          # anti-Hermitian as a matrix
    m = mass * np.eye(3 * v) + d
    mm = m.conj().T @ m
    par3 = np.repeat(li.site_parity(dims), 3)
    ee = mm[np.ix_(par3 == 0, par3 == 0)]
    oo = mm[np.ix_(par3 == 1, par3 == 1)]
    eo = mm[np.ix_(par3 == 0, par3 == 1)]
    assert np.abs(eo).max() < 1e-15
    a_e = dense_from_operator(lambda x: lat.mdagm(mass, 0, x), v // 2)
    a_o = dense_from_operator(lambda x: lat.mdagm(mass, 1, x), v // 2)
    assert np.abs(a_e - ee).max() < 5e-15
    assert np.abs(a_o - oo).max() < 5e-15
    ev_e, ev_o = np.linalg.eigvalsh(a_e), np.linalg.eigvalsh(a_o)
    assert np.abs(ev_e - ev_o).max() < 1e-12
    assert ev_e[0] >= mass ** 2 - 1e-14
    assert ev_e[-1] < 8.0 + mass ** 2                      # paper: xmax > 32 in its 4x normalisation


def test_storage_sizes():
    """72 V doubles of links, 6 V doubles per full vector."""
    cfg, u, b, _, _ = li.make_config_inputs(1)
    assert u.size == 72 * cfg.volume
    assert b.size == 6 * cfg.volume // 2
    with pytest.raises(ValueError):
        oracle.Lattice(cfg.dims, u[:-1])
