"""tests/golden/make_cfg5_samples.py (oracle-only generator of the stored config-5 solutions): the same
recipe on 4^4 lands on numpy.linalg.solve, and the committed files belong to today's seeded inputs."""
import os
import re
import sys

import numpy as np
import pytest

import lattice_inputs as li
import oracle
from helpers import c as cplx, dense_from_operator

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
sys.path.insert(0, GOLDEN)
import make_cfg5_samples as gen  # noqa: E402


def test_generator_recipe_matches_dense_solve(tmp_path):
    dims = (4, 4, 4, 4)
    gen.main(["--dims", "4,4,4,4", "--shifts", "0,9", "--outdir", str(tmp_path)])
    cfg, links, b, shifts, _ = li.make_config_inputs(5, dims)
    lat = oracle.Lattice(dims, links)
    a = dense_from_operator(lambda v: lat.mdagm(cfg.mass, 0, v), lat.volume // 2)
    w = cplx(gen.projection_vector(cfg)).reshape(-1)
    for k in (0, 9):
        g = gen.read_shift(gen.out_path(cfg, k, str(tmp_path)))
        assert g["k"] == k and g["sigma"] == shifts[k]
        x = np.linalg.solve(a + shifts[k] * np.eye(a.shape[0]), cplx(b).reshape(-1))
        xs = x.reshape(-1, 3)[g["sites"]]
        assert np.array_equal(g["sites"], np.arange(lat.volume // 2))      # 128 < NSITES: all sites
        assert np.linalg.norm(cplx(g["x"]) - xs) <= 1e-10 * np.linalg.norm(xs)
        assert abs(g["norm2"] - np.vdot(x, x).real) <= 1e-10 * g["norm2"]
        assert abs(g["proj"] - np.vdot(w, x)) <= 1e-10 * np.linalg.norm(w) * np.linalg.norm(x)


def test_committed_cfg5_files_belong_to_the_seeded_inputs():
    cfg = li.CONFIGS[5]
    b = li.make_source(cfg.dims, cfg.seed, cfg.parity)
    shifts = li.make_shifts(cfg)
    sites = gen.sample_sites(cfg)
    want = {"sha256_source": li.sha256(b), "sha256_shifts": li.sha256(shifts), "sha256_sites": li.sha256(sites)}
    for k in (0, 5, 10, 15):
        path = gen.out_path(cfg, k)
        assert os.path.exists(path), path
        head = open(path).read(4096)
        for key, val in want.items():
            assert re.search(rf"# {key} = {val}\b", head), (path, key)
        g = gen.read_shift(path)
        assert g["sigma"] == shifts[k] and np.array_equal(g["sites"], sites)
        res = float(re.search(r"# true_res_polished = (\S+)", head).group(1))
        assert res < 1e-12          # far below the 1e-10 the GPU solve is asked for
        assert np.isfinite(g["x"]).all() and g["norm2"] > 0
