"""SURVEY.md 8(f) NEXT-4, first half: the t-slab decomposition (paper_1710_09178_b200/slab.py) --
index maps, parity flip, the antiperiodic seam carried by the data, and the halo exchange -- checked with
world_size 2 and 4 on the gloo backend against the oracle's full-lattice operator.  Every rank applies
the ORACLE's D to its own extended local lattice (on a GPU box that call is qcd_dslash_range, see
tests/test_gpu_parity.py::test_slab_decomposition_on_one_gpu), so what is tested here is exactly the
decomposition: owned slices of the local results, gathered, must EQUAL the global result bit for bit."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


_WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
sys.path.insert(0, os.path.join({root!r}, "tests"))
import numpy as np, torch
import torch.distributed as dist
import lattice_inputs as li
import oracle
from paper_1710_09178_b200.slab import SlabPartition

world = {world}
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=world)
rank = dist.get_rank()
dims, mass = {dims!r}, 0.07
links = li.make_links(dims, "random", 3)
ve, vo = li.make_source(dims, 41, 0), li.make_source(dims, 42, 1)
glob = oracle.Lattice(dims, links)
part = SlabPartition(dims, world, rank)
loc = oracle.Lattice(part.local_dims, part.local_links(links))
n = part.nt_loc

def with_halos(v_owned_full, internal):
    # a rank knows its OWNED slices only: halos zeroed, then filled by the exchange
    a = part.local_vector(v_owned_full).reshape(n + 2, part.slice_half, 3, 2).copy()
    a[0] = 0.0; a[-1] = 0.0
    if internal:      # [3][t][site][2], the library's internal layout
        t = torch.from_numpy(np.ascontiguousarray(a.transpose(2, 0, 1, 3)))
        part.exchange_halos(t, dist, internal=True)
        return np.ascontiguousarray(t.numpy().transpose(1, 2, 0, 3)).reshape(-1, 3, 2)
    t = torch.from_numpy(a.reshape(-1, 3, 2))
    part.exchange_halos(t, dist, internal=False)
    return t.numpy()

def gather(owned):
    parts = [torch.empty_like(torch.from_numpy(owned)) for _ in range(world)]
    dist.all_gather(parts, torch.from_numpy(np.ascontiguousarray(owned)))
    return np.concatenate([p.numpy() for p in parts])

res = {{}}
for internal in (False, True):
    tag = "int" if internal else "can"
    v_loc = with_halos(ve, internal)
    res["halo_" + tag] = bool(np.array_equal(v_loc, part.local_vector(ve)))
    # D_oe: global output parity 1 lives on local parity 0
    d_loc = loc.dslash(part.local_parity(1), v_loc)
    d_all = gather(part.owned(d_loc))
    res["D_oe_" + tag] = bool(np.array_equal(d_all, glob.dslash(1, ve)))
    # D_eo on an odd vector
    w_loc = with_halos(vo, internal)
    res["D_eo_" + tag] = bool(np.array_equal(gather(part.owned(loc.dslash(part.local_parity(0), w_loc))), glob.dslash(0, vo)))
    # M^dag M = m^2 - D_eo D_oe: second exchange on the intermediate vector (its halos were never computed)
    t_loc = with_halos(gather(part.owned(d_loc)), internal)
    a_loc = mass * mass * part.owned(v_loc) - part.owned(loc.dslash(part.local_parity(0), t_loc))
    res["MdagM_" + tag] = bool(np.array_equal(gather(a_loc), glob.mdagm(mass, 0, ve)))
# <v, A v>: local sums over the owned slices, one all-reduce (the CG's per-iteration scalar)
av = glob.mdagm(mass, 0, ve)
mine = torch.tensor([float(np.sum(part.owned(part.local_vector(ve)) * part.owned(part.local_vector(av))))], dtype=torch.float64)
dist.all_reduce(mine)
res["dot_rel"] = abs(mine.item() - float(np.sum(ve * av))) / abs(float(np.sum(ve * av)))
res["rank"] = rank
dist.barrier()
print(json.dumps(res))
dist.destroy_process_group()
"""


@pytest.mark.parametrize("world,dims", [(2, (4, 6, 4, 8)), (2, (4, 4, 2, 4)), (4, (6, 4, 4, 8))])
def test_slab_decomposition_equals_the_global_operator(tmp_path, world, dims):
    port = _free_port()
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT, port=port, world=world, dims=dims))
    env = dict(os.environ, OMP_NUM_THREADS="2")     # the ranks share the host: small OpenMP teams
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE,
                              stderr=subprocess.PIPE, text=True, env=env) for r in range(world)]
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=300)
        assert p.returncode == 0, e
        outs.append(json.loads(o.strip().splitlines()[-1]))
    assert sorted(o["rank"] for o in outs) == list(range(world))
    for o in outs:
        for key in ("halo", "D_oe", "D_eo", "MdagM"):
            for tag in ("can", "int"):
                assert o[f"{key}_{tag}"] is True, (key, tag, o)
        assert o["dot_rel"] < 1e-14


def test_partition_geometry_and_argument_checks():
    sys.path.insert(0, ROOT)
    from paper_1710_09178_b200.slab import SlabPartition
    p = SlabPartition((4, 4, 4, 8), 2, 1)
    assert p.local_dims == (4, 4, 4, 6) and p.t_lo == 4 and p.up == 0 and p.down == 0
    assert list(p.global_t()) == [3, 4, 5, 6, 7, 0]
    assert list(SlabPartition((4, 4, 4, 8), 2, 0).global_t()) == [7, 0, 1, 2, 3, 4]
    assert SlabPartition.local_parity(0) == 1 and SlabPartition.local_parity(1) == 0
    for dims, world in (((4, 4, 4, 6), 2), ((4, 4, 4, 8), 3), ((4, 4, 4, 8), 1), ((4, 4, 4, 4), 4)):
        with pytest.raises(ValueError):
            SlabPartition(dims, world, 0)
    # the seam: t-links of the global slice Nt-1 are negated, nothing else is touched
    links = np.random.default_rng(0).standard_normal((4 * 4 * 4 * 8, 4, 3, 3, 2))
    g = links.reshape(8, 64, 4, 3, 3, 2)
    l0 = SlabPartition((4, 4, 4, 8), 2, 0).local_links(links).reshape(6, 64, 4, 3, 3, 2)
    l1 = SlabPartition((4, 4, 4, 8), 2, 1).local_links(links).reshape(6, 64, 4, 3, 3, 2)
    assert np.array_equal(l0[0, :, 3], -g[7, :, 3]) and np.array_equal(l0[0, :, :3], g[7, :, :3])
    assert np.array_equal(l0[1:], g[[0, 1, 2, 3, 4]])
    assert np.array_equal(l1[4, :, 3], -g[7, :, 3]) and np.array_equal(l1[:4], g[[3, 4, 5, 6]]) and np.array_equal(l1[5], g[0])
