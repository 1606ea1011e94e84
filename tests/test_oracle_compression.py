"""Pins for the oracle's two-row link reconstruction (NEXT-1): the third row of an
SU(3) matrix is conj(row_0 x row_1).  Checked against matrices written out by hand, against the
determinant / unitarity it must restore, and against the seeded SU(3) generators."""
import numpy as np

import lattice_inputs as li
import oracle
from helpers import c, f


def _as_links(mats):
    """list of complex 3x3 -> float64[V=len/4... padded to [n,4,3,3,2] with the same matrix per mu"""
    m = np.stack([np.stack([u] * 4) for u in mats])          # [n,4,3,3]
    return f(m)


def test_hand_written_su3_matrices():
    a, b = 0.37, -1.21
    diag = np.diag([np.exp(1j * a), np.exp(1j * b), np.exp(-1j * (a + b))])
    cyc = np.array([[0, 1, 0], [0, 0, 1], [1, 0, 0]], dtype=complex)          # det = +1
    th = 0.83
    rot = np.array([[np.cos(th), -np.sin(th), 0], [np.sin(th), np.cos(th), 0], [0, 0, 1]], dtype=complex)
    # rotation in the (1,2) plane times a phase pattern of determinant 1
    ph = np.diag([1j, 1j, -1.0])                                              # det = i*i*(-1) = 1
    mix = ph @ rot
    links = _as_links([diag, cyc, rot, mix])
    rec = oracle.reconstruct_links_2row(oracle.compress_links_2row(links))
    assert np.abs(rec - links).max() <= 1e-15
    # the expected third rows, typed out: diag -> (0,0,e^{-i(a+b)}); cyc -> (1,0,0); rot -> (0,0,1)
    third = c(rec)[:, 0, 2, :]
    assert np.allclose(third[0], [0, 0, np.exp(-1j * (a + b))], atol=1e-15)
    assert np.allclose(third[1], [1, 0, 0], atol=0)
    assert np.allclose(third[2], [0, 0, 1], atol=1e-16)
    assert np.allclose(third[3], [0, 0, -1], atol=1e-16)


def test_wrong_sign_or_missing_conjugate_would_fail():
    """A reconstruction without the conjugate, or with the cross product reversed, gives det != 1
    on a complex matrix: make sure the oracle's result has det = +1 and is unitary for arbitrary
    orthonormal complex rows (not taken from a generator that used the same formula)."""
    rng = np.random.default_rng(5)
    g = rng.normal(size=(64, 3, 3)) + 1j * rng.normal(size=(64, 3, 3))
    qmat, _ = np.linalg.qr(g)                     # unitary, det = arbitrary phase
    rows = np.zeros((16, 4, 2, 3, 2))
    rows[..., 0] = qmat[:, :2, :].real.reshape(16, 4, 2, 3)
    rows[..., 1] = qmat[:, :2, :].imag.reshape(16, 4, 2, 3)
    u = c(oracle.reconstruct_links_2row(rows)).reshape(64, 3, 3)
    eye = np.eye(3)
    assert max(np.abs(m @ m.conj().T - eye).max() for m in u) <= 1e-14
    assert max(abs(np.linalg.det(m) - 1.0) for m in u) <= 1e-14
    # and the two stored rows are returned untouched
    assert np.array_equal(u[:, :2, :], qmat[:, :2, :])


def test_identity_on_seeded_su3_fields():
    for kind, eps in (("random", 0.0), ("near_identity", 0.3)):
        links = li.make_links((4, 4, 2, 6), kind, 11, eps)
        rec = oracle.reconstruct_links_2row(oracle.compress_links_2row(links))
        assert np.abs(rec.reshape(-1) - links.reshape(-1)).max() <= 4e-15
        assert oracle.compress_links_2row(links).size == links.size * 2 // 3      # 48 V doubles


def test_dslash_on_reconstructed_links_equals_dslash():
    """The operator is unchanged: D[reconstruct(compress(U))] = D[U] to rounding."""
    dims = (4, 4, 4, 4)
    links = li.make_links(dims, "random", 3, 0.0)
    rec = oracle.reconstruct_links_2row(oracle.compress_links_2row(links))
    v = li.make_source(dims, 9, 0)
    a = oracle.Lattice(dims, links).dslash(1, v)
    b = oracle.Lattice(dims, rec).dslash(1, v)
    assert np.linalg.norm(a - b) / np.linalg.norm(a) <= 1e-15
