"""GPU parity: the CUDA library (through its C ABI) against the CPU oracle, element by element, on
the same seeded inputs.  Tolerances are BASELINE.json north_star's:
  Dslash / M^dag M   relative L2 error <= 1e-13
  multishift CG      recomputed true residual <= 1.5 tol for every shift;
                     ||x_k - x_k^oracle|| / ||x_k^oracle|| <= 1e-9 against the polished oracle (C16).
"""
import os

import numpy as np
import pytest

import lattice_inputs as li
import oracle
from helpers import rel_l2

pytestmark = pytest.mark.gpu

TOL_OP = 1e-13
TOL_X = 1e-9
E, O = 0, 1


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available()
    return torch


@pytest.fixture(scope="module")
def q():
    import paper_1710_09178_b200 as q
    q.load_library()          # fails loudly if the extension is missing: no fallback
    return q


class Rig:
    """One lattice: oracle + CUDA context fed the same canonical arrays."""

    def __init__(self, torch, q, dims, mass, links, link_rows=3, mixed=False):
        self.torch, self.q = torch, q
        self.dims, self.mass = dims, mass
        self.lat = oracle.Lattice(dims, links)
        self.ctx = q.Context(dims, mass)
        if link_rows != 3:
            self.ctx.set_option(q.QCD_OPT_LINK_ROWS, link_rows)
        if mixed:
            self.ctx.set_option(q.QCD_OPT_MIXED, 1)
        # QCD_TEST_DSLASH_KERNEL=1 [QCD_TEST_DSLASH_PERSIST=n] runs the WHOLE suite on the bulk-staged kernel
        if os.environ.get("QCD_TEST_DSLASH_KERNEL"):
            self.ctx.set_option(q.QCD_OPT_DSLASH_KERNEL, int(os.environ["QCD_TEST_DSLASH_KERNEL"]))
            self.ctx.set_option(q.QCD_OPT_DSLASH_PERSIST, int(os.environ.get("QCD_TEST_DSLASH_PERSIST", "0")))
        self.d_links = torch.from_numpy(links).cuda()
        self.ctx.load_gauge(self.d_links)
        self.nh = self.lat.volume // 2

    def to_internal(self, parity, canon: np.ndarray):
        d_c = self.torch.from_numpy(np.ascontiguousarray(canon)).cuda().reshape(-1)
        d_i = self.ctx.new_vector()
        self.ctx.pack(parity, d_c, d_i)
        return d_i

    def to_canonical(self, parity, d_i) -> np.ndarray:
        d_c = self.torch.empty(self.ctx.vector_doubles, dtype=self.torch.float64, device="cuda")
        self.ctx.unpack(parity, d_i, d_c)
        return d_c.cpu().numpy().reshape(self.nh, 3, 2)

    def dslash(self, out_parity, v):
        d_out = self.ctx.new_vector()
        self.ctx.dslash(out_parity, self.to_internal(1 - out_parity, v), d_out)
        return self.to_canonical(out_parity, d_out)

    def mdagm(self, parity, v):
        d_out = self.ctx.new_vector()
        self.ctx.mdagm(parity, self.to_internal(parity, v), d_out)
        return self.to_canonical(parity, d_out)

    def mdagm_internal(self, parity, d_in):
        d_out = self.ctx.new_vector()
        self.ctx.mdagm(parity, d_in, d_out)
        return self.to_canonical(parity, d_out)

    def solve(self, parity, b, shifts, residues, tol, max_iter=100000, own_x=True):
        n = len(shifts)
        d_x = self.ctx.new_vector(n) if own_x else None
        d_y = self.ctx.new_vector()
        st, it, tr = self.ctx.multishift_cg(parity, self.to_internal(parity, b), shifts, residues,
                                            tol, max_iter, d_x, d_y)
        x = None
        if own_x:
            x = np.stack([self.to_canonical(parity, d_x[k]) for k in range(n)])
        return dict(status=st, iterations=it, true_res=tr, x=x, y=self.to_canonical(parity, d_y))


def make_rig(torch, q, dims, kind, mass, seed, eps=0.3, link_rows=3):
    return Rig(torch, q, dims, mass, li.make_links(dims, kind, seed, eps), link_rows)


# ------------------------------------------------------------------ layout

def test_pack_unpack_roundtrip_bit_exact(torch, q):
    rig = make_rig(torch, q, (4, 6, 2, 8), "random", 0.1, 3)
    v = li.make_source(rig.dims, 3, 0)
    for par in (E, O):
        assert np.array_equal(rig.to_canonical(par, rig.to_internal(par, v)), v)


# ------------------------------------------------------------------ Dslash, M^dag M

SHAPES = [
    ((2, 2, 2, 2), "random"),          # extents of 2: x+mu == x-mu (C8)
    ((4, 4, 4, 4), "random"),          # config 1
    ((8, 8, 8, 4), "near_identity"),   # config 2
    ((4, 4, 2, 6), "random"),
    ((2, 4, 6, 2), "near_identity"),
    ((6, 2, 4, 8), "random"),
    ((12, 6, 10, 4), "random"),        # Vh = 1440: several blocks and a ragged tail
    ((10, 14, 6, 6), "near_identity"), # Vh = 2520, non power-of-two strides
]


@pytest.mark.parametrize("dims,kind", SHAPES)
def test_dslash_and_mdagm_match_oracle(torch, q, dims, kind):
    rig = make_rig(torch, q, dims, kind, 0.07, seed=sum(dims))
    ve = li.make_source(dims, 41, E)
    vo = li.make_source(dims, 42, O)
    assert rel_l2(rig.dslash(O, ve), rig.lat.dslash(O, ve)) <= TOL_OP    # D_oe
    assert rel_l2(rig.dslash(E, vo), rig.lat.dslash(E, vo)) <= TOL_OP    # D_eo
    assert rel_l2(rig.mdagm(E, ve), rig.lat.mdagm(0.07, E, ve)) <= TOL_OP
    assert rel_l2(rig.mdagm(O, vo), rig.lat.mdagm(0.07, O, vo)) <= TOL_OP


def test_dslash_free_field_eigenvalue_on_gpu(torch, q):
    """Property that holds at any size: U = 1, plane wave restricted to the even sites is an
    eigenvector of (M^dag M)_ee with eigenvalue m^2 + sum sin^2 p (north_star closed form)."""
    dims, mass = (8, 4, 6, 4), 0.3
    rig = Rig(torch, q, dims, mass, li.unit_links(dims))
    from helpers import coords
    xyzt = coords(dims)
    n = (3, 1, 2, 1)
    p = np.array([2 * np.pi * n[0] / dims[0], 2 * np.pi * n[1] / dims[1], 2 * np.pi * n[2] / dims[2],
                  2 * np.pi * (n[3] + 0.5) / dims[3]])
    psi = (np.exp(1j * xyzt @ p)[:, None] * np.array([1.0, 2j, -0.5])[None, :])[li.site_parity(dims) == 0]
    v = np.stack([psi.real, psi.imag], axis=-1)
    out = rig.mdagm(E, v)
    assert rel_l2(out, (mass ** 2 + (np.sin(p) ** 2).sum()) * v) < 1e-13


def test_set_mass_changes_mdagm(torch, q):
    rig = make_rig(torch, q, (4, 4, 4, 4), "random", 0.1, 1)
    v = li.make_source(rig.dims, 1, E)
    rig.ctx.set_mass(0.25)
    assert rel_l2(rig.mdagm(E, v), rig.lat.mdagm(0.25, E, v)) <= TOL_OP


# ------------------------------------------------------------------ two-row link storage (NEXT-1)

@pytest.mark.parametrize("dims,kind", SHAPES)
def test_two_row_dslash_and_mdagm_match_oracle(torch, q, dims, kind):
    """QCD_OPT_LINK_ROWS = 2: same operator, third row rebuilt in the kernel; the
    oracle is the plain definition on reconstruct_links_2row(compress_links_2row(U))."""
    links = li.make_links(dims, kind, sum(dims), 0.3)
    rec = oracle.reconstruct_links_2row(oracle.compress_links_2row(links))
    rig = Rig(torch, q, dims, 0.07, links, link_rows=2)
    lat2 = oracle.Lattice(dims, rec)
    ve = li.make_source(dims, 41, E)
    vo = li.make_source(dims, 42, O)
    for lat in (lat2, rig.lat):       # the reconstructed field and the original agree to rounding
        assert rel_l2(rig.dslash(O, ve), lat.dslash(O, ve)) <= TOL_OP
        assert rel_l2(rig.dslash(E, vo), lat.dslash(E, vo)) <= TOL_OP
        assert rel_l2(rig.mdagm(E, ve), lat.mdagm(0.07, E, ve)) <= TOL_OP
        assert rel_l2(rig.mdagm(O, vo), lat.mdagm(0.07, O, vo)) <= TOL_OP


def test_two_row_refuses_links_outside_su3(torch, q):
    """Two-row storage can only represent SU(3): a field whose third row is not conj(row0 x row1)
    (here: one link out of 4*V scaled by 1 + 1e-6) is refused at load, loudly, and leaves the
    context without a gauge field; the same field loads fine with three rows."""
    dims = (4, 6, 4, 4)
    links = li.make_links(dims, "random", 21)
    bad = links.reshape(-1, 4, 3, 3, 2).copy()
    bad[137, 2, 2] *= 1.0 + 1e-6
    bad = np.ascontiguousarray(bad.reshape(links.shape))
    rig = Rig(torch, q, dims, 0.1, links, link_rows=2)
    v = li.make_source(dims, 3, E)
    good = rig.dslash(O, v)
    with pytest.raises(q.QcdError, match="SU"):
        rig.ctx.load_gauge(torch.from_numpy(bad).cuda())
    with pytest.raises(q.QcdError, match="QCD_ESTATE"):
        rig.dslash(O, v)
    rig.ctx.load_gauge(rig.d_links)                       # a good field restores the context
    assert np.array_equal(rig.dslash(O, v), good)
    rig3 = Rig(torch, q, dims, 0.1, bad)                  # three-row storage takes any 3x3 matrices
    assert rel_l2(rig3.dslash(O, v), rig3.lat.dslash(O, v)) <= TOL_OP


def test_two_row_option_is_per_load_and_validated(torch, q):
    dims = (4, 4, 4, 4)
    links = li.make_links(dims, "random", 1)
    rig = Rig(torch, q, dims, 0.1, links)
    v = li.make_source(dims, 1, E)
    three = rig.dslash(O, v)
    rig.ctx.set_option(q.QCD_OPT_LINK_ROWS, 2)      # takes effect at the next load only
    assert np.array_equal(rig.dslash(O, v), three)
    rig.ctx.load_gauge(rig.d_links)
    two = rig.dslash(O, v)
    assert rel_l2(two, three) <= 1e-14
    rig.ctx.set_option(q.QCD_OPT_LINK_ROWS, 3)
    rig.ctx.load_gauge(rig.d_links)
    assert np.array_equal(rig.dslash(O, v), three)
    for bad in (1, 4, 0):
        with pytest.raises(q.QcdError, match="QCD_EINVAL"):
            rig.ctx.set_option(q.QCD_OPT_LINK_ROWS, bad)



# ------------------------------------------------------------------ bulk-copy staged Dslash (dslash_bulk.cu)

@pytest.mark.parametrize("dims,kind", SHAPES + [((16, 16, 16, 4), "random"), ((48, 6, 4, 4), "near_identity")])
def test_bulk_staged_dslash_matches_oracle_and_register_kernel(torch, q, dims, kind):
    """QCD_OPT_DSLASH_KERNEL = 1: links staged through shared memory by cp.async.bulk behind an mbarrier
    ring.  Same arithmetic in the same order: bit-identical to the register-staged kernel, one CTA per
    tile or persistent, both link layouts, any CTA order; and within 1e-13 of the oracle."""
    links = li.make_links(dims, kind, sum(dims), 0.3)
    ve, vo = li.make_source(dims, 41, E), li.make_source(dims, 42, O)
    for rows in (3, 2):
        rig = Rig(torch, q, dims, 0.07, links, link_rows=rows)
        rig.ctx.set_option(q.QCD_OPT_DSLASH_KERNEL, 0)
        ref = (rig.dslash(O, ve), rig.dslash(E, vo), rig.mdagm(E, ve), rig.mdagm(O, vo))
        assert rel_l2(ref[0], rig.lat.dslash(O, ve)) <= TOL_OP
        rig.ctx.set_option(q.QCD_OPT_DSLASH_KERNEL, 1)
        for persist, tg in ((0, 0), (1, 0), (3, 2), (2, 1), (8, 0)):
            rig.ctx.set_option(q.QCD_OPT_DSLASH_PERSIST, persist)
            rig.ctx.set_option(q.QCD_OPT_TGROUP, tg)
            out = (rig.dslash(O, ve), rig.dslash(E, vo), rig.mdagm(E, ve), rig.mdagm(O, vo))
            assert all(np.array_equal(a, b) for a, b in zip(out, ref)), (rows, persist, tg)
        assert rel_l2(out[1], rig.lat.dslash(E, vo)) <= TOL_OP
        assert rel_l2(out[3], rig.lat.mdagm(0.07, O, vo)) <= TOL_OP
        rig.ctx.close()


@pytest.mark.parametrize("persist", [0, 2])
def test_bulk_staged_kernel_in_the_solver(torch, q, persist):
    """The multishift CG on the bulk-staged kernel (fused <p,Ap> epilogue, dead iterations after
    convergence, graph replay, the device-side loop): against the polished oracle."""
    cfg, links, b, shifts, res = li.make_config_inputs(2)
    rig = Rig(torch, q, cfg.dims, cfg.mass, links)
    exact = rig.lat.solve_exact(cfg.mass, cfg.parity, b, shifts, res, cfg.tol)
    rig.ctx.set_option(q.QCD_OPT_DSLASH_KERNEL, 1)
    rig.ctx.set_option(q.QCD_OPT_DSLASH_PERSIST, persist)
    first = None
    for pdl, graph in ((1, 1), (0, 0), (1, 2), (1, 0)):
        rig.ctx.set_option(q.QCD_OPT_PDL, pdl)
        rig.ctx.set_option(q.QCD_OPT_CG_GRAPH, graph)
        out = rig.solve(cfg.parity, b, shifts, res, cfg.tol)
        check_solve(rig, cfg, b, shifts, res, out, exact)
        first = first or out
        assert out["iterations"] == first["iterations"] and np.array_equal(out["x"], first["x"])
    zero = rig.solve(E, np.zeros_like(b), shifts, res, cfg.tol)      # cg_init sets `done`: drain path
    assert zero["status"] == 0 and zero["iterations"] == 0 and not zero["x"].any()
    cut = rig.solve(E, b, shifts, res, cfg.tol, max_iter=5)
    assert cut["status"] == 4 and cut["iterations"] == 5


# ------------------------------------------------------------------ mixed precision (NEXT-3)

def test_fp32_link_operator_is_the_oracle_operator_on_the_rounded_field(torch, q):
    """QCD_OPT_OPERATOR_LINKS32: the inner operator of the mixed solver.  Links rounded to fp32, fp64
    arithmetic: equal (1e-13) to the oracle's plain definition on the rounded field, and different from
    the fp64 operator at the fp32 level."""
    from oracle import mixed_precision as mp
    dims, mass = (12, 6, 10, 4), 0.07
    links = li.make_links(dims, "random", 11)
    rig = Rig(torch, q, dims, mass, links, mixed=True)
    lat32 = oracle.Lattice(dims, mp.round_links_fp32(links))
    ve, vo = li.make_source(dims, 41, E), li.make_source(dims, 42, O)
    full = (rig.dslash(O, ve), rig.mdagm(E, ve))
    assert rel_l2(full[0], rig.lat.dslash(O, ve)) <= TOL_OP          # the fp64 path is untouched by the option
    rig.ctx.set_option(q.QCD_OPT_OPERATOR_LINKS32, 1)
    assert rel_l2(rig.dslash(O, ve), lat32.dslash(O, ve)) <= TOL_OP
    assert rel_l2(rig.dslash(E, vo), lat32.dslash(E, vo)) <= TOL_OP
    assert rel_l2(rig.mdagm(E, ve), lat32.mdagm(mass, E, ve)) <= TOL_OP
    assert rel_l2(rig.mdagm(O, vo), lat32.mdagm(mass, O, vo)) <= TOL_OP
    assert 1e-9 < rel_l2(rig.dslash(O, ve), full[0]) < 1e-6
    rig.ctx.set_option(q.QCD_OPT_OPERATOR_LINKS32, 0)
    assert np.array_equal(rig.dslash(O, ve), full[0])
    plain = Rig(torch, q, dims, mass, links)                          # no fp32 copy loaded: refused
    plain.ctx.set_option(q.QCD_OPT_OPERATOR_LINKS32, 1)
    with pytest.raises(q.QcdError, match="QCD_ESTATE"):
        plain.dslash(O, ve)


@pytest.mark.parametrize("number,switch", [(1, 4), (2, 5), (1, 10)])
def test_mixed_precision_solver_matches_the_oracle(torch, q, number, switch):
    """QCD_OPT_MIXED: fp64 multishift to 10^-switch, then per-shift defect correction with the fp32-link
    inner operator.  Same bars as the fp64 solver: recomputed fp64 residual <= 1.5 tol (here <= tol by
    construction), every x_k and y within 1e-9 of the polished oracle; and within 1e-9 of the oracle's
    own restatement of the mixed algorithm (oracle/mixed_precision.py)."""
    from oracle import mixed_precision as mp
    cfg, links, b, shifts, res = li.make_config_inputs(number)
    rig = Rig(torch, q, cfg.dims, cfg.mass, links, mixed=True)
    rig.ctx.set_option(q.QCD_OPT_MIXED_SWITCH_EXP, switch)
    out = rig.solve(cfg.parity, b, shifts, res, cfg.tol)
    exact = rig.lat.solve_exact(cfg.mass, cfg.parity, b, shifts, res, cfg.tol)
    check_solve(rig, cfg, b, shifts, res, out, exact)
    assert (out["true_res"] <= cfg.tol * (1 + 1e-9)).all()
    ref = mp.mixed_precision_multishift(cfg.dims, links, cfg.mass, cfg.parity, b, shifts, res, cfg.tol,
                                        switch_tol=10.0 ** -switch)
    for k in range(len(shifts)):
        assert rel_l2(out["x"][k], ref["x"][k]) <= TOL_X
    total_ref = ref["stage1_iterations"] + int(ref["inner_iterations"].sum())
    assert abs(out["iterations"] - total_ref) <= max(4, total_ref // 20), (out["iterations"], total_ref)
    # without an x buffer (library workspace, sorted order) and with unsorted shifts: same answers
    perm = np.argsort(-shifts)
    out2 = rig.solve(cfg.parity, b, shifts[perm], res[perm], cfg.tol, own_x=False)
    assert out2["status"] == 0 and rel_l2(out2["y"], exact["y"]) <= TOL_X
    assert (out2["true_res"] <= cfg.tol * (1 + 1e-9)).all()
    zero = rig.solve(E, np.zeros_like(b), shifts, res, cfg.tol)
    assert zero["status"] == 0 and not zero["x"].any() and not zero["true_res"].any()


def test_mixed_precision_light_mass(torch, q):
    """kappa ~ 3e5: one round of the fp32-link inner solve gains about two digits only; the refinement
    still lands on the fp64 solution."""
    dims, mass, tol = (4, 4, 4, 4), 0.005, 1e-10
    links = li.make_links(dims, "random", 5)
    b = li.make_source(dims, 5, E)
    shifts = np.logspace(-6, np.log10(4.0), 6)
    rig = Rig(torch, q, dims, mass, links, mixed=True)
    out = rig.solve(E, b, shifts, np.ones(6), tol)
    assert out["status"] == 0 and (out["true_res"] <= tol * (1 + 1e-9)).all()
    exact = rig.lat.solve_exact(mass, E, b, shifts, np.ones(6), tol)
    for k in range(6):
        assert rel_l2(out["x"][k], exact["x"][k]) <= TOL_X


# ------------------------------------------------------------------ t-slab decomposition (NEXT-4, first half)

@pytest.mark.parametrize("world,kernel", [(2, 0), (4, 0), (2, 1)])
def test_slab_decomposition_on_one_gpu(torch, q, world, kernel):
    """paper_1710_09178_b200/slab.py + qcd_dslash_range: every rank's slab, held with its two halo slices
    as a lattice of its own, computed one after the other on this one GPU (no kernel waits on another).
    Owned slices put together must EQUAL the single-context result bit for bit (same arithmetic per
    site), and agree with the oracle's global operator; M^dag M needs a second halo fill."""
    from paper_1710_09178_b200.slab import SlabPartition
    dims, mass = (8, 6, 4, 8), 0.07
    links = li.make_links(dims, "random", 3)
    ve = li.make_source(dims, 41, E)
    ref = Rig(torch, q, dims, mass, links)
    ref.ctx.set_option(q.QCD_OPT_DSLASH_KERNEL, kernel)
    want_d, want_a = ref.dslash(O, ve), ref.mdagm(E, ve)
    parts = [SlabPartition(dims, world, r) for r in range(world)]
    rigs = [Rig(torch, q, p.local_dims, mass, p.local_links(links)) for p in parts]
    for r in rigs:
        r.ctx.set_option(q.QCD_OPT_DSLASH_KERNEL, kernel)
    lp_e, lp_o = SlabPartition.local_parity(E), SlabPartition.local_parity(O)
    nt = dims[3]

    def apply(global_in, out_parity_local, src_global=None, coeff=0.0):
        """one slab-decomposed D: halos come from the global vector (what the exchange delivers)"""
        pieces = []
        for p, r in zip(parts, rigs):
            d_in = r.to_internal(1 - out_parity_local, p.local_vector(global_in))
            d_out = torch.full((r.ctx.vector_doubles,), np.nan, dtype=torch.float64, device="cuda")
            d_src = None if src_global is None else r.to_internal(out_parity_local, p.local_vector(src_global))
            r.ctx.dslash_range(out_parity_local, d_in, d_out, 1, p.nt_loc, d_src, coeff)
            out = r.to_canonical(out_parity_local, d_out)
            halo = out.reshape(p.nt_loc + 2, -1)[[0, -1]]
            assert np.isnan(halo).all()                       # halo slices of the output are not touched
            pieces.append(p.owned(out))
        return np.concatenate(pieces)

    got_d = apply(ve, lp_o)
    assert np.array_equal(got_d, want_d) and rel_l2(got_d, ref.lat.dslash(O, ve)) <= TOL_OP
    got_a = apply(got_d, lp_e, src_global=ve, coeff=mass * mass)          # m^2 v - D_eo (D_oe v)
    assert np.array_equal(got_a, want_a) and rel_l2(got_a, ref.lat.mdagm(mass, E, ve)) <= TOL_OP
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):
        rigs[0].ctx.dslash_range(0, rigs[0].ctx.new_vector(), rigs[0].ctx.new_vector(), 1, nt)


def test_dslash_range_writes_exactly_the_requested_slices(torch, q):
    """qcd_dslash_range (the building block of the slab decomposition): for any t-range the requested
    slices carry the bits of the full apply, with and without the fused epilogue, every other site of the
    output keeps what it held; both kernels, both link layouts, both parities."""
    dims, mass = (6, 4, 4, 10), 0.07
    links = li.make_links(dims, "random", 17)
    rng = np.random.default_rng(5)
    for rows in (3, 2):
        rig = Rig(torch, q, dims, mass, links, link_rows=rows)
        st = rig.nh // dims[3]                     # sites of one parity per t-slice
        for kernel in (0, 1):
            rig.ctx.set_option(q.QCD_OPT_DSLASH_KERNEL, kernel)
            for par in (O, E):
                v, w = li.make_source(dims, 3 + par, 1 - par), li.make_source(dims, 9 + par, par)
                full = rig.dslash(par, v)
                d_in, d_src = rig.to_internal(1 - par, v), rig.to_internal(par, w)
                for t0, nt in [(0, dims[3]), (0, 1), (dims[3] - 1, 1), (3, 4), tuple(int(x) for x in (rng.integers(0, 5), rng.integers(1, 6)))]:
                    for fused in (False, True):
                        d_out = torch.full((rig.ctx.vector_doubles,), 7.25, dtype=torch.float64, device="cuda")
                        rig.ctx.dslash_range(par, d_in, d_out, t0, nt, d_src if fused else None, 0.3)
                        out = rig.to_canonical(par, d_out).reshape(dims[3], st, 3, 2)
                        want = (0.3 * w - full if fused else full).reshape(dims[3], st, 3, 2)
                        assert np.array_equal(out[t0:t0 + nt], want[t0:t0 + nt]) or \
                            rel_l2(out[t0:t0 + nt], want[t0:t0 + nt]) <= 1e-15, (rows, kernel, par, t0, nt, fused)
                        mask = np.ones(dims[3], dtype=bool)
                        mask[t0:t0 + nt] = False
                        assert (out[mask] == 7.25).all(), (rows, kernel, par, t0, nt, fused)
        for bad in ((-1, 2), (0, 0), (9, 2)):
            with pytest.raises(q.QcdError, match="QCD_EINVAL"):
                rig.ctx.dslash_range(O, d_in, rig.ctx.new_vector(), bad[0], bad[1])
        rig.ctx.close()

# ------------------------------------------------------------------ multishift CG

def check_solve(rig, cfg, b, shifts, res, out, exact=None):
    assert out["status"] == 0
    assert np.isfinite(out["true_res"]).all()
    assert (out["true_res"] <= 1.5 * cfg.tol).all(), out["true_res"]
    for k, s in enumerate(shifts):
        # the library's own true residual agrees with one recomputed by the ORACLE's operator
        xk = out["x"][k]
        r = b - (rig.lat.mdagm(cfg.mass, cfg.parity, xk) + s * xk)
        tr = np.linalg.norm(r) / np.linalg.norm(b)
        assert abs(tr - out["true_res"][k]) <= 1e-3 * tr + 1e-15
        if exact is not None:
            assert rel_l2(xk, exact["x"][k]) <= TOL_X, (k, rel_l2(xk, exact["x"][k]))
    y_from_x = np.tensordot(res, out["x"], axes=(0, 0))
    assert rel_l2(out["y"], y_from_x) <= 1e-14
    if exact is not None:
        assert rel_l2(out["y"], exact["y"]) <= TOL_X


@pytest.mark.parametrize("number", [1, 2])
def test_multishift_cg_configs_1_2(torch, q, number):
    cfg, links, b, shifts, res = li.make_config_inputs(number)
    rig = Rig(torch, q, cfg.dims, cfg.mass, links)
    out = rig.solve(cfg.parity, b, shifts, res, cfg.tol)
    exact = rig.lat.solve_exact(cfg.mass, cfg.parity, b, shifts, res, cfg.tol)
    check_solve(rig, cfg, b, shifts, res, out, exact)
    ref = rig.lat.multishift_cg(cfg.mass, cfg.parity, b, shifts, res, cfg.tol, want_x=False)
    assert abs(out["iterations"] - ref["iterations"]) <= max(2, ref["iterations"] // 50)


@pytest.mark.parametrize("number", [1, 2])
def test_two_row_multishift_cg_configs_1_2(torch, q, number):
    cfg, links, b, shifts, res = li.make_config_inputs(number)
    rig = Rig(torch, q, cfg.dims, cfg.mass, links, link_rows=2)
    out = rig.solve(cfg.parity, b, shifts, res, cfg.tol)
    exact = rig.lat.solve_exact(cfg.mass, cfg.parity, b, shifts, res, cfg.tol)
    check_solve(rig, cfg, b, shifts, res, out, exact)


def test_config2_solutions_against_lapack_directly(torch, q):
    """Independent of the oracle's CG and polish: the matrix of (M^dag M)_ee on config 2 assembled column by
    column from the oracle's OPERATOR (pinned by closed forms), every shifted system solved by LAPACK, and
    the GPU's x_k compared with that."""
    from helpers import c as cplx, dense_from_operator
    cfg, links, b, shifts, res = li.make_config_inputs(2)
    rig = Rig(torch, q, cfg.dims, cfg.mass, links)
    out = rig.solve(cfg.parity, b, shifts, res, cfg.tol)
    a = dense_from_operator(lambda v: rig.lat.mdagm(cfg.mass, E, v), rig.nh)
    bc = cplx(b).ravel()
    y = np.zeros_like(bc)
    for k, s in enumerate(shifts):
        xd = np.linalg.solve(a + s * np.eye(a.shape[0]), bc)
        y += res[k] * xd
        assert rel_l2(cplx(out["x"][k]).ravel(), xd) <= TOL_X, k
    assert rel_l2(cplx(out["y"]).ravel(), y) <= TOL_X


def test_multishift_cg_is_deterministic(torch, q):
    cfg, links, b, shifts, res = li.make_config_inputs(2)
    rig = Rig(torch, q, cfg.dims, cfg.mass, links)
    o1 = rig.solve(cfg.parity, b, shifts, res, cfg.tol)
    o2 = rig.solve(cfg.parity, b, shifts, res, cfg.tol)
    assert o1["iterations"] == o2["iterations"]
    assert np.array_equal(o1["x"], o2["x"]) and np.array_equal(o1["y"], o2["y"])


def test_deferred_shift_updates_do_not_change_a_single_bit(torch, q):
    """QCD_OPT_CG_DEFER: x_k, p_k of the shifts k >= 1 are updated once per m iterations from the stored
    coefficients and a ring of residuals.  Same operations per element in the same order: every m,
    every way of enqueueing, the freezing of shifts inside a window, max_iter inside a window and the
    zero source give the bits of m = 1; and m = 1 matches the oracle."""
    cases = [li.make_config_inputs(2)[:5]]
    dims, mass = (4, 4, 4, 4), 0.005                      # light mass: shifts freeze one after the other
    cases.append((li.Config(0, dims, mass, "random", 0.0, 16, 1e-6, 4.0, "ones", 1e-10),
                  li.make_links(dims, "random", 5), li.make_source(dims, 5, E),
                  np.logspace(-6, np.log10(4.0), 16), np.linspace(0.5, 2.0, 16)))
    for cfg, links, b, shifts, res in cases:
        rig = Rig(torch, q, cfg.dims, cfg.mass, links)
        rig.ctx.set_option(q.QCD_OPT_CG_DEFER, 1)
        ref = rig.solve(E, b, shifts, res, cfg.tol)
        exact = rig.lat.solve_exact(cfg.mass, E, b, shifts, res, cfg.tol)
        check_solve(rig, cfg, b, shifts, res, ref, exact)
        cut_ref = rig.solve(E, b, shifts, res, cfg.tol, max_iter=13)
        for m, graph, batch in [(8, 1, 8), (2, 1, 8), (3, 0, 8), (5, 1, 3), (8, 2, 8), (4, 0, 1), (7, 1, 16), (8, 0, 5), (3, 2, 8)]:
            rig.ctx.set_option(q.QCD_OPT_CG_DEFER, m)
            rig.ctx.set_option(q.QCD_OPT_CG_GRAPH, graph)
            rig.ctx.set_option(q.QCD_OPT_CG_BATCH, batch)
            out = rig.solve(E, b, shifts, res, cfg.tol)
            assert out["status"] == 0 and out["iterations"] == ref["iterations"], (m, graph, batch)
            assert np.array_equal(out["x"], ref["x"]) and np.array_equal(out["y"], ref["y"]), (m, graph, batch)
            assert np.array_equal(out["true_res"], ref["true_res"])
            cut = rig.solve(E, b, shifts, res, cfg.tol, max_iter=13)
            assert cut["status"] == 4 and cut["iterations"] == 13 and np.array_equal(cut["x"], cut_ref["x"])
            zero = rig.solve(E, np.zeros_like(b), shifts, res, cfg.tol)
            assert zero["status"] == 0 and zero["iterations"] == 0 and not zero["x"].any()
            no_x = rig.solve(E, b, shifts, res, cfg.tol, own_x=False)
            assert np.array_equal(no_x["y"], ref["y"])
        # QCD_OPT_CG_FUSE: r-update and base-shift update as one cooperative kernel, same bits
        rig.ctx.set_option(q.QCD_OPT_CG_FUSE, 1)
        for m, graph, batch in [(8, 1, 8), (4, 0, 8), (8, 2, 8), (3, 1, 5)]:
            rig.ctx.set_option(q.QCD_OPT_CG_DEFER, m)
            rig.ctx.set_option(q.QCD_OPT_CG_GRAPH, graph)
            rig.ctx.set_option(q.QCD_OPT_CG_BATCH, batch)
            out = rig.solve(E, b, shifts, res, cfg.tol)
            assert out["status"] == 0 and out["iterations"] == ref["iterations"], (m, graph, batch)
            assert np.array_equal(out["x"], ref["x"]) and np.array_equal(out["y"], ref["y"]), (m, graph, batch)
            cut = rig.solve(E, b, shifts, res, cfg.tol, max_iter=13)
            assert cut["status"] == 4 and cut["iterations"] == 13 and np.array_equal(cut["x"], cut_ref["x"])
            zero = rig.solve(E, np.zeros_like(b), shifts, res, cfg.tol)
            assert zero["status"] == 0 and zero["iterations"] == 0 and not zero["x"].any()
        rig.ctx.set_option(q.QCD_OPT_CG_FUSE, 0)
        for bad in (0, 9):
            with pytest.raises(q.QcdError, match="QCD_EINVAL"):
                rig.ctx.set_option(q.QCD_OPT_CG_DEFER, bad)
        rig.ctx.close()


def test_execution_options_do_not_change_a_single_bit(torch, q):
    """QCD_OPT_PDL / QCD_OPT_CG_GRAPH / QCD_OPT_CG_BATCH only change how work is enqueued."""
    cfg, links, b, shifts, res = li.make_config_inputs(2)
    rig = Rig(torch, q, cfg.dims, cfg.mass, links)
    ref = rig.solve(E, b, shifts, res, cfg.tol)
    ref_d = rig.dslash(O, b)
    for pdl, graph, batch in [(0, 0, 16), (1, 0, 3), (0, 1, 1), (1, 1, 5), (1, 1, 64), (1, 2, 8), (0, 2, 8)]:
        rig.ctx.set_option(q.QCD_OPT_PDL, pdl)
        rig.ctx.set_option(q.QCD_OPT_CG_GRAPH, graph)
        rig.ctx.set_option(q.QCD_OPT_CG_BATCH, batch)
        out = rig.solve(E, b, shifts, res, cfg.tol)
        assert out["iterations"] == ref["iterations"] and out["status"] == 0
        assert np.array_equal(out["x"], ref["x"]) and np.array_equal(out["y"], ref["y"])
        assert np.array_equal(out["true_res"], ref["true_res"])
        assert np.array_equal(rig.dslash(O, b), ref_d)
    # device-side loop: max_iter and the zero source end the WHILE node too
    cut = rig.solve(E, b, shifts, res, cfg.tol, max_iter=7)
    assert cut["status"] == 4 and cut["iterations"] == 7
    zero = rig.solve(E, np.zeros_like(b), shifts, res, cfg.tol)
    assert zero["status"] == 0 and zero["iterations"] == 0 and not zero["x"].any()
    again = rig.solve(E, b, shifts, res, cfg.tol)
    assert np.array_equal(again["x"], ref["x"])
    with pytest.raises(q.QcdError):
        rig.ctx.set_option(q.QCD_OPT_CG_GRAPH, 3)
    with pytest.raises(q.QcdError):
        rig.ctx.set_option(q.QCD_OPT_CG_BATCH, 0)
    with pytest.raises(q.QcdError):
        rig.ctx.set_option(99, 1)


def test_cta_order_option_does_not_change_a_single_bit(torch, q):
    """QCD_OPT_TGROUP only permutes which CTA handles which 128-site chunk (3 ragged chunks per
    t-slice here); the CG reduction order is by blockIdx, so only Dslash/M^dag M must be bit-equal,
    the solve to rounding."""
    dims, mass = (12, 6, 10, 4), 0.07
    rig = make_rig(torch, q, dims, "random", mass, 9)
    ve, vo = li.make_source(dims, 1, E), li.make_source(dims, 2, O)
    ref = (rig.dslash(O, ve), rig.dslash(E, vo), rig.mdagm(E, ve))
    shifts, res = np.array([0.01, 0.3, 1.5]), np.ones(3)
    sref = rig.solve(E, ve, shifts, res, 1e-10)
    for g in (1, 2, 3, 100000, 0):
        rig.ctx.set_option(q.QCD_OPT_TGROUP, g)
        out = (rig.dslash(O, ve), rig.dslash(E, vo), rig.mdagm(E, ve))
        assert all(np.array_equal(a, b) for a, b in zip(out, ref))
        s = rig.solve(E, ve, shifts, res, 1e-10)
        assert s["status"] == 0 and rel_l2(s["x"], sref["x"]) <= 1e-12
    assert rel_l2(ref[0], rig.lat.dslash(O, ve)) <= TOL_OP
    # QCD_OPT_SWEEP_ALTERNATE: even-output launches walk the tiles backwards; same bits for the operators
    for kern in (0, 1):
        rig.ctx.set_option(q.QCD_OPT_DSLASH_KERNEL, kern)
        rig.ctx.set_option(q.QCD_OPT_SWEEP_ALTERNATE, 1)
        out = (rig.dslash(O, ve), rig.dslash(E, vo), rig.mdagm(E, ve))
        assert all(np.array_equal(a, b) for a, b in zip(out, ref))
        s = rig.solve(E, ve, shifts, res, 1e-10)
        assert s["status"] == 0 and rel_l2(s["x"], sref["x"]) <= 1e-12
        rig.ctx.set_option(q.QCD_OPT_SWEEP_ALTERNATE, 0)
    rig.ctx.set_option(q.QCD_OPT_DSLASH_KERNEL, 0)
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):
        rig.ctx.set_option(q.QCD_OPT_TGROUP, -1)
    # L2 persisting window: applies at the next load, results unchanged
    rig.ctx.set_option(q.QCD_OPT_TGROUP, 0)
    rig.ctx.set_option(q.QCD_OPT_L2_PERSIST_MB, 16)
    rig.ctx.load_gauge(rig.d_links)
    assert np.array_equal(rig.dslash(O, ve), ref[0]) and np.array_equal(rig.mdagm(E, ve), ref[2])
    s = rig.solve(E, ve, shifts, res, 1e-10)
    assert s["status"] == 0 and np.array_equal(s["x"], sref["x"])
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):
        rig.ctx.set_option(q.QCD_OPT_L2_PERSIST_MB, -1)


def test_multishift_cg_odd_parity_unsorted_shifts_zero_shift(torch, q):
    dims, mass = (4, 6, 4, 4), 0.08
    rig = make_rig(torch, q, dims, "random", mass, 7)
    b = li.make_source(dims, 7, O)
    shifts = np.array([0.5, 0.0, 2.0, 1e-3, 0.02])
    res = np.array([1.0, -2.0, 0.5, 3.0, 0.25])
    out = rig.solve(O, b, shifts, res, 1e-11)
    exact = rig.lat.solve_exact(mass, O, b, shifts, res, 1e-11)
    assert out["status"] == 0 and (out["true_res"] <= 1.5e-11).all()
    for k in range(len(shifts)):
        assert rel_l2(out["x"][k], exact["x"][k]) <= TOL_X
    assert rel_l2(out["y"], exact["y"]) <= TOL_X


def test_multishift_cg_without_x_buffer_and_single_shift(torch, q):
    cfg, links, b, shifts, res = li.make_config_inputs(1)
    rig = Rig(torch, q, cfg.dims, cfg.mass, links)
    with_x = rig.solve(E, b, shifts, res, cfg.tol)
    no_x = rig.solve(E, b, shifts, res, cfg.tol, own_x=False)
    assert np.array_equal(with_x["y"], no_x["y"]) and np.array_equal(with_x["true_res"], no_x["true_res"])
    one = rig.solve(E, b, shifts[:1], res[:1], cfg.tol)
    assert rel_l2(one["x"][0], with_x["x"][0]) <= 1e-9


def test_freezing_light_mass_16_shifts(torch, q):
    """C13 on the GPU: zeta_k of large shifts would underflow to 0/0 without freezing."""
    dims, mass = (4, 4, 4, 4), 0.005
    rig = make_rig(torch, q, dims, "random", mass, 5)
    b = li.make_source(dims, 5, E)
    shifts = np.logspace(-6, np.log10(4.0), 16)
    out = rig.solve(E, b, shifts, np.ones(16), 1e-10)
    assert out["status"] == 0 and out["iterations"] > 300
    assert np.isfinite(out["x"]).all() and (out["true_res"] <= 1.5e-10).all()
    exact = rig.lat.solve_exact(mass, E, b, shifts, np.ones(16), 1e-10)
    for k in range(16):
        assert rel_l2(out["x"][k], exact["x"][k]) <= TOL_X


def test_maximum_number_of_shifts(torch, q):
    """QCD_MAX_SHIFTS = 64 shifts in one solve (16 batches of the multi-RHS finish); 65 is refused."""
    dims, mass = (4, 4, 4, 6), 0.2
    rig = make_rig(torch, q, dims, "random", mass, 13)
    b = li.make_source(dims, 13, E)
    shifts = np.logspace(-3, 1, 64)[::-1].copy()          # descending: the library sorts
    res = np.linspace(0.5, 1.5, 64)
    out = rig.solve(E, b, shifts, res, 1e-10)
    assert out["status"] == 0 and (out["true_res"] <= 1.5e-10).all()
    for k in (0, 17, 40, 63):
        xs, _, tr, st = rig.lat.cg(mass, E, shifts[k], b, 1e-14, max_iter=5000)
        assert st == 0 and rel_l2(out["x"][k], xs) <= TOL_X
        r = b - (rig.lat.mdagm(mass, E, out["x"][k]) + shifts[k] * out["x"][k])
        tr = np.linalg.norm(r) / np.linalg.norm(b)
        assert abs(tr - out["true_res"][k]) <= 1e-3 * tr + 1e-15
    assert rel_l2(out["y"], np.tensordot(res, out["x"], axes=(0, 0))) <= 1e-14
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):
        rig.solve(E, b, np.ones(65), np.ones(65), 1e-10)


def test_dslash_inside_a_cuda_graph_replay_is_bit_identical(torch, q):
    """bench.py times graph replays of the Dslash on a side stream: same kernels, same bits."""
    dims = (12, 6, 10, 4)
    rig = make_rig(torch, q, dims, "near_identity", 0.07, 5)
    v = li.make_source(dims, 5, E)
    d_in, d_o, d_e = rig.to_internal(E, v), rig.ctx.new_vector(), rig.ctx.new_vector()
    rig.ctx.dslash(O, d_in, d_o)
    rig.ctx.dslash(E, d_o, d_e)
    ref_o, ref_e = rig.to_canonical(O, d_o), rig.to_canonical(E, d_e)
    d_o.zero_(); d_e.zero_()
    main = torch.cuda.current_stream()
    side = torch.cuda.Stream()
    side.wait_stream(main)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        rig.ctx.set_stream(side.cuda_stream)
        with torch.cuda.graph(g, stream=side):
            for _ in range(3):
                rig.ctx.dslash(O, d_in, d_o)
                rig.ctx.dslash(E, d_o, d_e)
    rig.ctx.set_stream(main.cuda_stream)
    main.wait_stream(side)
    d_o.zero_(); d_e.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert np.array_equal(rig.to_canonical(O, d_o), ref_o) and np.array_equal(rig.to_canonical(E, d_e), ref_e)
    assert rel_l2(ref_o, rig.lat.dslash(O, v)) <= TOL_OP


def test_max_iter_and_zero_source(torch, q):
    cfg, links, b, shifts, res = li.make_config_inputs(1)
    rig = Rig(torch, q, cfg.dims, cfg.mass, links)
    out = rig.solve(E, b, shifts, res, cfg.tol, max_iter=7)
    assert out["status"] == 4 and out["iterations"] == 7          # QCD_ENOTCONV, outputs still written
    ref = rig.lat.multishift_cg(cfg.mass, E, b, shifts, res, cfg.tol, max_iter=7)
    assert rel_l2(out["x"], ref["x"]) < 1e-12
    assert np.allclose(out["true_res"], ref["true_res"], rtol=1e-9)
    zero = rig.solve(E, np.zeros_like(b), shifts, res, cfg.tol)
    assert zero["status"] == 0 and zero["iterations"] == 0 and not zero["x"].any() and not zero["y"].any()


def test_error_codes(torch, q):
    ctx = q.Context((4, 4, 4, 4), 0.1)
    v, w = ctx.new_vector(), ctx.new_vector()
    with pytest.raises(q.QcdError, match="QCD_ESTATE"):
        ctx.dslash(E, v, w)
    ctx.load_gauge(torch.from_numpy(li.make_links((4, 4, 4, 4), "random", 1)).cuda())
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):
        ctx.dslash(E, v, v)
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):
        ctx.dslash(2, v, w)
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):
        ctx.multishift_cg(E, v, [-1.0], [1.0], 1e-10, 10)
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):
        ctx.multishift_cg(E, v, [1.0], [1.0], 0.0, 10)
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):
        q.Context((4, 4, 3, 4), 0.1)
    # overlapping ranges and misaligned device pointers are refused before anything is launched
    n = ctx.vector_doubles
    big = torch.zeros(4 * n + 2, dtype=torch.float64, device="cuda")
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):
        ctx.dslash(E, big[:n], big[n // 2: n // 2 + n])            # partial overlap
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):
        ctx.dslash(E, big[1:n + 1], w)                             # 8-byte aligned only
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):
        ctx.mdagm(E, v, big[n + 1:2 * n + 1])
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):
        ctx.pack(E, big[:n], big[n - 2:2 * n - 2])
    sh, rs = [0.1, 0.2], [1.0, 1.0]
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):            # the source inside the x buffer
        ctx.multishift_cg(E, big[n:2 * n], sh, rs, 1e-10, 10, big[:2 * n], None)
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):            # y == b
        ctx.multishift_cg(E, v, sh, rs, 1e-10, 10, None, v)
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):            # y inside x
        ctx.multishift_cg(E, v, sh, rs, 1e-10, 10, big[:2 * n], big[n:2 * n])
    with pytest.raises(ValueError):                                # binding: short x buffer
        ctx.multishift_cg(E, v, sh, rs, 1e-10, 10, big[:n], None)
    with pytest.raises(ValueError):
        ctx.multishift_cg(E, v, sh, [1.0], 1e-10, 10)
    with pytest.raises(ValueError):
        ctx.dslash(E, v[:-2], w)
    torch.cuda.synchronize()                                       # and the context is still healthy
    ctx.dslash(E, v, w)
    torch.cuda.synchronize()


def test_host_entry_points_equal_device_entry_points(torch, q):
    cfg, links, b, shifts, res = li.make_config_inputs(2)
    rig = Rig(torch, q, cfg.dims, cfg.mass, links)
    ctx2 = q.Context(cfg.dims, cfg.mass)
    ctx2.load_gauge_host(links)
    out = np.empty_like(b)
    ctx2.dslash_host(O, b, out)
    assert np.array_equal(out, rig.dslash(O, b))
    ctx2.mdagm_host(E, b, out)
    assert np.array_equal(out, rig.mdagm(E, b))
    hx = np.empty((len(shifts),) + b.shape)
    hy = np.empty_like(b)
    st, it, tr = ctx2.multishift_cg_host(E, b, shifts, res, cfg.tol, 10000, hx, hy)
    dev = rig.solve(E, b, shifts, res, cfg.tol)
    assert st == 0 and it == dev["iterations"]
    assert np.array_equal(hx, dev["x"]) and np.array_equal(hy, dev["y"])
    assert np.array_equal(tr, dev["true_res"])


# ------------------------------------------------------------------ (M^dag M)^(-1/2) phi  (NEXT-2)

@pytest.mark.parametrize("number,n", [(1, 10), (2, 12)])
def test_inv_sqrt_matches_oracle_and_dense_definition(torch, q, number, n):
    """qcd_inv_sqrt against (i) the oracle's eq. 8 with the ORACLE's coefficients and polished
    solves, (ii) the definition Q diag(lambda^-1/2) Q^dag phi through eigh (config 1 only)."""
    from oracle import rational as R
    from helpers import c as cplx, dense_from_operator
    cfg, links, b, _, _ = li.make_config_inputs(number)
    rig = Rig(torch, q, cfg.dims, cfg.mass, links)
    xmin, xmax = 0.9 * cfg.mass ** 2, 8.5      # the paper's xmax = 34 in its normalisation
    d_out = rig.ctx.new_vector()
    st, it, tr, delta = rig.ctx.inv_sqrt(E, rig.to_internal(E, b), n, xmin, xmax, 1e-11, 100000, d_out)
    got = rig.to_canonical(E, d_out)
    z = R.zolotarev_inv_sqrt(n, xmin, xmax)
    assert st == 0 and (tr <= 1.5e-11).all() and abs(delta - z["delta"]) <= 1e-6 * z["delta"]
    sol = rig.lat.solve_exact(cfg.mass, E, b, z["d"], z["c"], 1e-11)
    assert rel_l2(got, z["c0"] * b + sol["y"]) <= TOL_X
    if number == 1:
        a = dense_from_operator(lambda v: rig.lat.mdagm(cfg.mass, E, v), rig.nh)
        lam, qm = np.linalg.eigh(a)
        assert xmin < lam.min() and lam.max() < xmax
        phi = cplx(b).reshape(-1)
        exact = qm @ ((qm.conj().T @ phi) / np.sqrt(lam))
        err = np.linalg.norm(cplx(got).reshape(-1) - exact) / np.linalg.norm(exact)
        assert err <= 1.05 * delta + 1e-9
        # applying it twice inverts M^dag M:  A r(A)^2 phi = phi +- 2 delta
        d_2 = rig.ctx.new_vector()
        rig.ctx.inv_sqrt(E, d_out, n, xmin, xmax, 1e-11, 100000, d_2)
        back = rig.mdagm_internal(E, d_2)
        assert rel_l2(back, b) <= 2.2 * delta + 1e-8


def test_inv_sqrt_argument_errors(torch, q):
    rig = make_rig(torch, q, (4, 4, 4, 4), "random", 0.1, 1)
    v, w = rig.ctx.new_vector(), rig.ctx.new_vector()
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):
        rig.ctx.inv_sqrt(E, v, 0, 0.01, 5.0, 1e-10, 100, w)
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):
        rig.ctx.inv_sqrt(E, v, 4, 5.0, 0.01, 1e-10, 100, w)
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):
        rig.ctx.inv_sqrt(E, v, 4, 0.01, 5.0, 1e-10, 100, v)


def test_pipelined_host_dslash(torch, q):
    """qcd_dslash_host on vectors of 4.5 MB or more runs as a t-slab pipeline (upload / compute /
    download on three streams; 3 slabs of 4 t-slices here): same bits as the device entry point, and
    the oracle's operator."""
    dims = (32, 32, 16, 12)
    links = li.make_links(dims, "random", 17)
    for rows in (3, 2):
        rig = Rig(torch, q, dims, 0.05, links, link_rows=rows)
        for par in (O, E):
            v = li.make_source(dims, 3 + par, 1 - par)
            hin = torch.from_numpy(v).pin_memory().numpy()
            hout = torch.empty(v.shape, dtype=torch.float64).pin_memory().numpy()
            for _ in range(2):                      # second call reuses streams and events
                hout[:] = 0.0
                rig.ctx.dslash_host(par, hin, hout)
                assert np.array_equal(hout, rig.dslash(par, v))
            assert rel_l2(hout, rig.lat.dslash(par, v)) <= TOL_OP
        out = np.empty_like(v)                      # pageable host memory works too
        rig.ctx.dslash_host(par, v, out)
        assert np.array_equal(out, hout)


# ------------------------------------------------------------------ full-size configs 3, 4, 5

@pytest.mark.slow
def test_config3_full_size(torch, q):
    """32^3 x 8, the configuration the metric is quoted on: operators element by element, solve
    against the polished oracle."""
    cfg, links, b, shifts, res = li.make_config_inputs(3)
    rig = Rig(torch, q, cfg.dims, cfg.mass, links)
    vo = li.make_source(cfg.dims, 43, O)
    assert rel_l2(rig.dslash(O, b), rig.lat.dslash(O, b)) <= TOL_OP
    assert rel_l2(rig.dslash(E, vo), rig.lat.dslash(E, vo)) <= TOL_OP
    assert rel_l2(rig.mdagm(E, b), rig.lat.mdagm(cfg.mass, E, b)) <= TOL_OP
    out = rig.solve(E, b, shifts, res, cfg.tol)
    exact = rig.lat.solve_exact(cfg.mass, E, b, shifts, res, cfg.tol)
    check_solve(rig, cfg, b, shifts, res, out, exact)


@pytest.mark.slow
def test_config3_full_size_two_row(torch, q):
    cfg, links, b, shifts, res = li.make_config_inputs(3)
    rig = Rig(torch, q, cfg.dims, cfg.mass, links, link_rows=2)
    vo = li.make_source(cfg.dims, 43, O)
    assert rel_l2(rig.dslash(O, b), rig.lat.dslash(O, b)) <= TOL_OP
    assert rel_l2(rig.dslash(E, vo), rig.lat.dslash(E, vo)) <= TOL_OP
    assert rel_l2(rig.mdagm(E, b), rig.lat.mdagm(cfg.mass, E, b)) <= TOL_OP
    out = rig.solve(E, b, shifts, res, cfg.tol)
    assert out["status"] == 0 and (out["true_res"] <= 1.5 * cfg.tol).all()
    for k in (0, 11):
        xs, _, tr, st = rig.lat.cg(cfg.mass, E, shifts[k], b, 1e-14, max_iter=5000)
        assert st == 0 and rel_l2(out["x"][k], xs) <= TOL_X


@pytest.mark.slow
def test_config4_full_size(torch, q):
    """48^3 x 12, tol 1e-12: operators element by element; EVERY shift (the base shift included) and y
    against the polished oracle (about two minutes of oracle time on 16 cores)."""
    cfg, links, b, shifts, res = li.make_config_inputs(4)
    rig = Rig(torch, q, cfg.dims, cfg.mass, links)
    assert rel_l2(rig.dslash(O, b), rig.lat.dslash(O, b)) <= TOL_OP
    assert rel_l2(rig.mdagm(E, b), rig.lat.mdagm(cfg.mass, E, b)) <= TOL_OP
    out = rig.solve(E, b, shifts, res, cfg.tol)
    exact = rig.lat.solve_exact(cfg.mass, E, b, shifts, res, cfg.tol)
    check_solve(rig, cfg, b, shifts, res, out, exact)


def _golden_cfg5():
    """tests/golden/cfg5_samples_kNN.txt, written by tests/golden/make_cfg5_samples.py from the oracle
    alone: polished x_k at 2048 seeded sites, ||x_k||^2 and <w, x_k> for k = 0 (base shift), 5, 10, 15."""
    import os
    import sys
    gdir = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    sys.path.insert(0, gdir)
    import make_cfg5_samples as gen
    cfg = li.CONFIGS[5]
    gold = {}
    for k in (0, 5, 10, 15):
        path = gen.out_path(cfg, k)
        assert os.path.exists(path), f"{path} missing: run tests/golden/make_cfg5_samples.py"
        gold[k] = gen.read_shift(path)
    return gen, gold


@pytest.mark.slow
def test_config5_full_size(torch, q):
    """64^3 x 16, random SU(3), m = 0.005: thousands of iterations, kappa_0 ~ 2.6e5.  The
    full oracle solve takes hours on the host, so the oracle's polished solutions of the base shift and
    of shifts 5, 10, 15 are stored at 2048 seeded sites together with two global functionals
    (tests/golden/cfg5_samples_k*.txt, oracle-written).  Here: operators element by element; the four
    stored shifts site by site, in norm and in projection to 1e-9; the true residual of every shift
    recomputed by the oracle's operator; the largest shift against an in-test oracle CG on all sites."""
    cfg, links, b, shifts, res = li.make_config_inputs(5)
    gen, gold = _golden_cfg5()
    assert all(gold[k]["sigma"] == shifts[k] for k in gold)
    sites = gen.sample_sites(cfg)
    rig = Rig(torch, q, cfg.dims, cfg.mass, links)
    assert rel_l2(rig.dslash(O, b), rig.lat.dslash(O, b)) <= TOL_OP
    assert rel_l2(rig.mdagm(E, b), rig.lat.mdagm(cfg.mass, E, b)) <= TOL_OP
    out = rig.solve(E, b, shifts, res, cfg.tol)
    assert out["status"] == 0 and out["iterations"] > 1000
    assert (out["true_res"] <= 1.5 * cfg.tol).all(), out["true_res"]
    w = gen.projection_vector(cfg)
    wc = w[..., 0] + 1j * w[..., 1]
    wnorm = np.linalg.norm(wc)
    for k, g in gold.items():
        xk = out["x"][k]
        assert np.array_equal(g["sites"], sites)
        # element by element at the sampled sites, relative to the size of x_k there
        err = np.linalg.norm((xk[sites] - g["x"]).ravel()) / np.linalg.norm(g["x"].ravel())
        assert err <= TOL_X, (k, err)
        assert np.abs(xk[sites] - g["x"]).max() <= 20 * TOL_X * np.sqrt(g["norm2"] / xk.size), k
        # two functionals of ALL sites: the norm, and the projection on a seeded Gaussian vector
        n2 = float(np.sum(xk.astype(np.longdouble) ** 2))
        assert abs(n2 - g["norm2"]) <= 2 * TOL_X * g["norm2"], (k, n2, g["norm2"])
        proj = np.vdot(wc, xk[..., 0] + 1j * xk[..., 1])
        assert abs(proj - g["proj"]) <= TOL_X * wnorm * np.sqrt(g["norm2"]), (k, proj, g["proj"])
    for k in range(cfg.nshift):          # residual of every shift recomputed with the oracle's operator
        xk = out["x"][k]
        r = b - (rig.lat.mdagm(cfg.mass, E, xk) + shifts[k] * xk)
        tr = np.linalg.norm(r) / np.linalg.norm(b)
        assert tr <= 1.5 * cfg.tol and abs(tr - out["true_res"][k]) <= 1e-2 * tr, (k, tr)
    assert rel_l2(out["y"], np.tensordot(res, out["x"], axes=(0, 0))) <= 1e-14
    xs, _, tr, st = rig.lat.cg(cfg.mass, cfg.parity, shifts[15], b, 1e-14, max_iter=2000)
    assert st == 0 and tr < 1e-13 and rel_l2(out["x"][15], xs) <= TOL_X


@pytest.mark.slow
def test_config5_two_row_links_and_bulk_kernel(torch, q):
    """The options at the largest size: two-row link storage (NEXT-1) solves config 5 to the same stored
    oracle solutions (base shift included), and the bulk-staged Dslash (one CTA per tile and persistent)
    gives the bits of the register-staged one on the 2.4 GB field."""
    cfg, links, b, shifts, res = li.make_config_inputs(5)
    gen, gold = _golden_cfg5()
    sites = gen.sample_sites(cfg)
    rig = Rig(torch, q, cfg.dims, cfg.mass, links, link_rows=2)
    ref_o = rig.lat.dslash(O, b)
    assert rel_l2(rig.dslash(O, b), ref_o) <= TOL_OP
    out = rig.solve(E, b, shifts, res, cfg.tol)
    assert out["status"] == 0 and (out["true_res"] <= 1.5 * cfg.tol).all(), out["true_res"]
    for k, g in gold.items():
        xk = out["x"][k]
        err = np.linalg.norm((xk[sites] - g["x"]).ravel()) / np.linalg.norm(g["x"].ravel())
        assert err <= TOL_X, (k, err)
        n2 = float(np.sum(xk.astype(np.longdouble) ** 2))
        assert abs(n2 - g["norm2"]) <= 2 * TOL_X * g["norm2"], (k, n2, g["norm2"])
    rig.ctx.close()
    del out
    rig3 = Rig(torch, q, cfg.dims, cfg.mass, links)
    d3 = rig3.dslash(O, b)
    assert rel_l2(d3, ref_o) <= TOL_OP
    rig3.ctx.set_option(q.QCD_OPT_DSLASH_KERNEL, 1)
    for persist in (0, 3):
        rig3.ctx.set_option(q.QCD_OPT_DSLASH_PERSIST, persist)
        assert np.array_equal(rig3.dslash(O, b), d3), persist


# ------------------------------------------------------------------ (M^dag M)^(1/4) phi  (heat bath)

def test_fourth_root_matches_oracle_and_dense_definition(torch, q):
    """qcd_apply_pow with alpha = 1/4 on config 1: against eq. 8 with the ORACLE's Remez coefficients
    and polished solves, against Q diag(lambda^(1/4)) Q^dag phi, and A^(1/4) A^(1/4) A^(-1/2) = 1."""
    from fractions import Fraction
    from oracle import rational as R
    from helpers import c as cplx, dense_from_operator
    cfg, links, b, _, _ = li.make_config_inputs(1)
    rig = Rig(torch, q, cfg.dims, cfg.mass, links)
    n, xmin, xmax = 10, 0.9 * cfg.mass ** 2, 8.5
    d_phi, d_out = rig.to_internal(E, b), rig.ctx.new_vector()
    st, it, tr, delta = rig.ctx.apply_pow(E, d_phi, 1, 4, n, xmin, xmax, 1e-11, 100000, d_out)
    got = rig.to_canonical(E, d_out)
    z = R.minimax_pow(Fraction(1, 4), n, xmin, xmax)
    assert st == 0 and (tr <= 1.5e-11).all() and abs(delta / z["delta"] - 1) <= 1e-6
    sol = rig.lat.solve_exact(cfg.mass, E, b, z["d"], z["c"], 1e-11)
    assert rel_l2(got, z["c0"] * b + sol["y"]) <= TOL_X
    a = dense_from_operator(lambda v: rig.lat.mdagm(cfg.mass, E, v), rig.nh)
    lam, qm = np.linalg.eigh(a)
    phi = cplx(b).reshape(-1)
    exact = qm @ ((qm.conj().T @ phi) * lam ** 0.25)
    assert np.linalg.norm(cplx(got).reshape(-1) - exact) / np.linalg.norm(exact) <= 1.05 * delta + 1e-9
    # A^(1/4) A^(1/4) A^(-1/2) phi = phi
    d_2, d_3 = rig.ctx.new_vector(), rig.ctx.new_vector()
    rig.ctx.apply_pow(E, d_out, 1, 4, n, xmin, xmax, 1e-11, 100000, d_2)
    _, _, _, delta_is = rig.ctx.inv_sqrt(E, d_2, n, xmin, xmax, 1e-11, 100000, d_3)
    assert rel_l2(rig.to_canonical(E, d_3), b) <= 2.2 * delta + 1.1 * delta_is + 1e-8
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):
        rig.ctx.apply_pow(E, d_phi, 5, 4, n, xmin, xmax, 1e-11, 100, d_out)


@pytest.mark.parametrize("number,n", [(1, 10), (2, 12)])
def test_y_only_mode_gives_the_same_y_without_forming_x(torch, q, number, n):
    """QCD_OPT_Y_ONLY: qcd_inv_sqrt / qcd_apply_pow accumulate y += c_k alpha_k p_k in the iteration.
    Same y as the default path to rounding, same y as the oracle's eq. 8; the reported residuals are
    the recursion's estimates and must bracket the recomputed ones."""
    from fractions import Fraction
    from oracle import rational as R
    cfg, links, b, _, _ = li.make_config_inputs(number)
    rig = Rig(torch, q, cfg.dims, cfg.mass, links)
    xmin, xmax, tol = 0.9 * cfg.mass ** 2, 8.5, 1e-11
    d_phi, d_a, d_b = rig.to_internal(E, b), rig.ctx.new_vector(), rig.ctx.new_vector()
    for num, den in ((-1, 2), (1, 4)):
        rig.ctx.set_option(q.QCD_OPT_Y_ONLY, 0)
        st0, it0, tr0, delta0 = rig.ctx.apply_pow(E, d_phi, num, den, n, xmin, xmax, tol, 100000, d_a)
        rig.ctx.set_option(q.QCD_OPT_Y_ONLY, 1)
        l0 = rig.ctx.launch_count
        st1, it1, tr1, delta1 = rig.ctx.apply_pow(E, d_phi, num, den, n, xmin, xmax, tol, 100000, d_b)
        ya, yb = rig.to_canonical(E, d_a), rig.to_canonical(E, d_b)
        assert st0 == 0 and st1 == 0 and it0 == it1 and delta0 == delta1
        assert rel_l2(yb, ya) <= 1e-12
        z = (R.zolotarev_inv_sqrt(n, xmin, xmax) if (num, den) == (-1, 2)
             else R.minimax_pow(Fraction(num, den), n, xmin, xmax))
        sol = rig.lat.solve_exact(cfg.mass, E, b, z["d"], z["c"], tol)
        assert rel_l2(yb, z["c0"] * b + sol["y"]) <= TOL_X
        assert (tr1 <= 1.5 * tol).all() and (tr1 > 0).all()
        assert (tr0 <= 1.5 * tol).all()
        assert tr1[0] == pytest.approx(tr0[0], rel=0.05)          # base shift: recursion vs recomputed
        # deferred (default, once per 8 iterations) against undeferred y-only accumulation: another order of
        # the same sum
        for m in (1, 3):
            rig.ctx.set_option(q.QCD_OPT_CG_DEFER, m)
            d_c = rig.ctx.new_vector()
            st2, it2, tr2, _ = rig.ctx.apply_pow(E, d_phi, num, den, n, xmin, xmax, tol, 100000, d_c)
            assert st2 == 0 and it2 == it1 and rel_l2(rig.to_canonical(E, d_c), yb) <= 1e-12
            assert np.allclose(tr2, tr1, rtol=1e-9)
        rig.ctx.set_option(q.QCD_OPT_CG_DEFER, 8)
        # the fused cooperative BLAS-1 kernel (default) against the two-kernel path: same bits in the y-only form too
        rig.ctx.set_option(q.QCD_OPT_CG_FUSE, 0)
        d_c = rig.ctx.new_vector()
        st3, it3, tr3, _ = rig.ctx.apply_pow(E, d_phi, num, den, n, xmin, xmax, tol, 100000, d_c)
        assert st3 == 0 and it3 == it1 and np.array_equal(rig.to_canonical(E, d_c), yb) and np.array_equal(tr3, tr1)
        rig.ctx.set_option(q.QCD_OPT_CG_FUSE, 1)
    # the inv_sqrt entry point takes the same path; the zero source still works
    st, it, tr, _ = rig.ctx.inv_sqrt(E, torch.zeros_like(d_phi), n, xmin, xmax, tol, 100, d_b)
    assert st == 0 and it == 0 and not rig.to_canonical(E, d_b).any() and not tr.any()
    rig.ctx.set_option(q.QCD_OPT_Y_ONLY, 0)


def test_random_shapes_rows_and_cta_orders(torch, q):
    """A seeded sweep over lattice shapes (extents 2..16, odd half-extents, thin directions), both
    link layouts and three CTA orders: Dslash and M^dag M element by element, a 5-shift solve against
    independent single-shift oracle CGs."""
    rng = np.random.default_rng(2024)
    shapes = {(16, 2, 2, 2), (2, 16, 2, 2), (2, 2, 16, 2), (2, 2, 2, 16), (18, 14, 10, 6)}
    while len(shapes) < 14:
        d = tuple(int(2 * rng.integers(1, 9)) for _ in range(4))
        if np.prod(d) <= 12000:
            shapes.add(d)
    mass = 0.13
    shifts, res = np.array([0.7, 0.0, 0.05, 2.5, 0.3]), np.array([1.0, -0.5, 2.0, 0.25, 3.0])
    for dims in sorted(shapes):
        links = li.make_links(dims, "random", sum(dims))
        for rows in (3, 2):
            rig = Rig(torch, q, dims, mass, links, link_rows=rows)
            for tg in (0, 1, 2):
                rig.ctx.set_option(q.QCD_OPT_TGROUP, tg)
                for par in (O, E):
                    v, w = li.make_source(dims, 7 + par, 1 - par), li.make_source(dims, 9 + par, par)
                    assert rel_l2(rig.dslash(par, v), rig.lat.dslash(par, v)) <= TOL_OP, (dims, rows, tg, par)
                    assert rel_l2(rig.mdagm(par, w), rig.lat.mdagm(mass, par, w)) <= TOL_OP, (dims, rows, tg, par)
            b = li.make_source(dims, 3, E)
            out = rig.solve(E, b, shifts, res, 1e-11)
            assert out["status"] == 0 and (out["true_res"] <= 1.5e-11).all(), (dims, rows)
            for k in (1, 3):
                xs, _, _, st = rig.lat.cg(mass, E, shifts[k], b, 1e-14, max_iter=20000)
                assert st == 0 and rel_l2(out["x"][k], xs) <= TOL_X, (dims, rows, k)
            rig.ctx.close()
