"""Writes tests/golden/cfg5_samples_kNN.txt: the ORACLE's polished solutions of BASELINE.json config 5
(64^3 x 16, random SU(3), m = 0.005, 16 shifts log-spaced in [1e-6, 4]) at sampled sites, so that the
GPU parity test can compare the base shift (kappa ~ 2.6e5) and three others element by
element without running the oracle for hours inside pytest ("cache the polished
solution").  Calls `oracle` and `lattice_inputs` ONLY; never run against the CUDA library.

    python tests/golden/make_cfg5_samples.py [--shifts 0,5,10,15] [--threads N] [--config 5] [--dims x,y,z,t]

Per shift k: x_k = single-shift oracle CG on (M^dag M + sigma_k) to 1e-13 of the
recursion residual, then defect-correction polish to the fp64 floor.  Stored per shift:
  * x_k at NSITES seeded-random even sites (index j into the canonical even-parity vector),
  * ||x_k||^2 and the projection <w, x_k> on a seeded Gaussian vector w (global quantities that see
    every site), the oracle's true residual, iteration count, wall time, host cores.
One file per shift, written when that shift is done (the base shift alone takes about an hour on 8
cores).  `--dims` runs the same recipe on a smaller lattice (used by the CPU test of this script).
"""
from __future__ import annotations

import argparse
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import lattice_inputs as li  # noqa: E402
import oracle  # noqa: E402

NSITES = 2048
SITE_STREAM = 99        # default_rng([seed, SITE_STREAM]) draws the sampled sites
PROJ_SEED_OFFSET = 50   # w = make_source(dims, seed + PROJ_SEED_OFFSET, parity)
CG_TOL = 1e-13


def sample_sites(cfg) -> np.ndarray:
    nh = cfg.volume // 2
    rng = np.random.default_rng([cfg.seed, SITE_STREAM])
    return np.sort(rng.choice(nh, size=min(NSITES, nh), replace=False))


def projection_vector(cfg) -> np.ndarray:
    return li.make_source(cfg.dims, cfg.seed + PROJ_SEED_OFFSET, cfg.parity)


def out_path(cfg, k: int, directory: str = HERE) -> str:
    return os.path.join(directory, f"cfg{cfg.number}_samples_k{k:02d}.txt")


def solve_shift(lat, cfg, b, sigma):
    t0 = time.time()
    x, it, tr_cg, st = lat.cg(cfg.mass, cfg.parity, sigma, b, CG_TOL, max_iter=200000)
    if st != 0:
        raise RuntimeError(f"oracle CG did not converge (sigma={sigma!r}, {it} iterations)")
    tr = lat.polish(cfg.mass, cfg.parity, sigma, b, x, max_iter=200000)
    return x, it, tr_cg, tr, time.time() - t0


def write_shift(path, cfg, k, sigma, sites, x, w, meta):
    xs = x[sites]
    wc = w[..., 0] + 1j * w[..., 1]
    xc = x[..., 0] + 1j * x[..., 1]
    proj = np.vdot(wc, xc)                      # <w, x> = sum conj(w) x
    norm2 = float(np.sum(x.astype(np.longdouble) ** 2))
    with open(path + ".tmp", "w") as fh:
        fh.write(f"# ORACLE-written (tests/golden/make_cfg5_samples.py; oracle/ + lattice_inputs/ only).\n"
                 f"# BASELINE.json config {cfg.number}, dims {cfg.dims}, mass {cfg.mass!r}, parity {cfg.parity}:\n"
                 f"# x_k = (M^dag M + sigma_k)^-1 b (PAPER.md:133 eq. 8, :136), single-shift CG to {CG_TOL:g} + polish (SURVEY.md C16).\n")
        for key, val in meta.items():
            fh.write(f"# {key} = {val}\n")
        fh.write(f"k {k}\nsigma {float(sigma)!r}\nnorm2 {norm2!r}\nproj {float(proj.real)!r} {float(proj.imag)!r}\n"
                 f"nsites {len(sites)}\n# j  re0 im0 re1 im1 re2 im2   (j = index into the canonical parity vector)\n")
        for j, row in zip(sites, xs.reshape(len(sites), 6)):
            fh.write(f"{int(j)} " + " ".join(repr(float(v)) for v in row) + "\n")
    os.replace(path + ".tmp", path)


def read_shift(path):
    """Parser used by the tests: dict(k, sigma, norm2, proj, sites int64[n], x float64[n,3,2])."""
    out, rows = {}, []
    with open(path) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            tok = line.split()
            if tok[0] == "k":
                out["k"] = int(tok[1])
            elif tok[0] == "sigma":
                out["sigma"] = float(tok[1])
            elif tok[0] == "norm2":
                out["norm2"] = float(tok[1])
            elif tok[0] == "proj":
                out["proj"] = complex(float(tok[1]), float(tok[2]))
            elif tok[0] == "nsites":
                out["nsites"] = int(tok[1])
            else:
                rows.append([float(t) for t in tok])
    a = np.array(rows)
    assert a.shape == (out["nsites"], 7)
    out["sites"] = a[:, 0].astype(np.int64)
    out["x"] = np.ascontiguousarray(a[:, 1:].reshape(-1, 3, 2))
    return out


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--shifts", default="0,5,10,15")
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--dims", default=None, help="override the lattice (testing the script itself)")
    ap.add_argument("--outdir", default=HERE)
    args = ap.parse_args(argv)
    if args.threads:
        oracle.set_threads(args.threads)
    dims = tuple(int(d) for d in args.dims.split(",")) if args.dims else None
    cfg, links, b, shifts, _ = li.make_config_inputs(args.config, dims)
    lat = oracle.Lattice(cfg.dims, links)
    sites = sample_sites(cfg)
    w = projection_vector(cfg)
    base = {"numpy": np.__version__, "oracle_threads": oracle.threads(), "host_cores": os.cpu_count(),
            "sha256_source": li.sha256(b), "sha256_shifts": li.sha256(shifts),
            "sha256_links": li.sha256(links), "sha256_sites": li.sha256(sites)}
    for k in (int(s) for s in args.shifts.split(",")):
        x, it, tr_cg, tr, secs = solve_shift(lat, cfg, b, shifts[k])
        meta = dict(base, cg_iterations=it, true_res_after_cg=repr(tr_cg), true_res_polished=repr(tr),
                    wall_seconds=f"{secs:.1f}")
        write_shift(out_path(cfg, k, args.outdir), cfg, k, shifts[k], sites, x, w, meta)
        print(f"k={k} sigma={shifts[k]:.3e} it={it} res_cg={tr_cg:.2e} res_polished={tr:.2e} {secs:.0f}s",
              flush=True)


if __name__ == "__main__":
    main()
