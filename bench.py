#!/usr/bin/env python
"""bench.py -- the measurement contract.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 3] [--impl ours|reference]

Metric (BASELINE.json): fp64 staggered Dslash algorithmic HBM GB/s at 32^3 x 8 (config 3), with the
multishift-CG seconds per solve reported beside it.

One STEP is one pass of the whole hot path over one batch of seeded
synthetic input already resident in HBM (a1, the gauge ingest, happens once before the timed region
on the device arm, and inside it on the e2e arm's first step only -- a gauge field serves thousands
of applies):
    A. PAIRS x (D_oe, D_eo) back to back, one CUDA graph          (a2, a3)   -> `value`
    B. PAIRS/2 x M^dag M                                           (a4)
    C. one multishift-CG solve incl. true residuals and y         (a5, a6)   -> cg.s_per_solve
After the timed region, once, on rank 0: the e2e leg (host buffers through the C ABI), (M^dag M)^(-1/2) phi and
(M^dag M)^(1/4) phi via eq. 8 (`inv_sqrt`, `fourth_root`; also with QCD_OPT_Y_ONLY), the two-row-link
variant of sections A and C (`two_row`), and the oracle on the host cores (`cpu_baseline`).
`value` = 624*V bytes x (Dslash launches of section A) / (CUDA-event time of section A), summed over
the K steps: the STEADY STATE of back-to-back applies, which is how the solver uses the kernel.  It is
an algorithmic rate, NOT a pure HBM rate: the 151 MB of links exceed the 126 MB L2, but the vectors
and part of the links are served by L2 (no flush is issued between launches), so about a fifth of
the algorithmic bytes never reach DRAM.  The line therefore also carries
  roofline.frac_dram   DRAM bytes per launch (ncu, steady state, profiles/*.json) / time / peak,
  dslash.cold_l2       the same launch after an L2 flush, timed inside a graph (flush time subtracted),
  streaming            config 5 (64^3 x 16, 2.4 GB of links): Dslash only, where L2 cannot help,
and `target_check` evaluates BASELINE.json's ">= 70 % of HBM peak at 32^3 x 8" against the cold figure.

N > 1: the path runs on one GPU with no sharding (BASELINE.json north_star; DESIGN.md "replicas
only"): every rank runs the same workload independently, no data-path collective; `value` is the
sum over ranks of algorithmic bytes divided by the slowest rank's time.

`--impl reference` times the CPU oracle as it stands on the host cores (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import lattice_inputs as li  # noqa: E402

METRIC = "staggered_dslash_fp64_algorithmic_GBps"
UNIT = "GB/s"
PAIRS = 50                      # (D_oe, D_eo) pairs per step in section A
FALLBACK_HBM_GBS = 6650.0       # /opt/skills/guides/B200_PROFILING.md fallback
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "r02_dslash_traffic.json")


def kernel_source_hash(kernel: int = 0) -> str:
    """SHA-256 over the sources of the Dslash kernel in question (0: register-staged, 1: bulk-staged): ties a
    stored ncu figure to the code it was taken from."""
    import hashlib
    h = hashlib.sha256()
    for name in (("dslash.cu", "dslash_site.cuh") if kernel == 0 else ("dslash_bulk.cu", "dslash_site.cuh")):
        with open(os.path.join(ROOT, "paper_1710_09178_b200", "csrc", name), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def traffic_entry(cfg_number: int, link_rows: int, kernel: int):
    """The stored ncu figures of one workload/kernel (dict, possibly empty) and a note on their origin; a
    capture taken from other kernel sources than today's is reported as stale."""
    try:
        with open(TRAFFIC_JSON) as fh:
            doc = json.load(fh)
    except Exception:
        return {}, "no profiles/r02_dslash_traffic.json"
    e = doc.get("entries", {}).get(f"cfg{cfg_number}_rows{link_rows}_kernel{kernel}")
    if not e:
        return {}, "no ncu capture for this workload/kernel in profiles/r02_dslash_traffic.json"
    note = f"ncu, {TRAFFIC_JSON[len(ROOT) + 1:]}"
    if e.get("source_hash") != kernel_source_hash(kernel):
        note += " (STALE: kernel sources changed since the capture)"
    return e, note


def load_traffic(cfg_number: int, link_rows: int, kernel: int):
    """DRAM read+write bytes per Dslash launch measured by ncu, written to profiles/r02_dslash_traffic.json
    by `bench.py --ncu-import` from the raw ncu page.  Returns (cold, warm, note)."""
    e, note = traffic_entry(cfg_number, link_rows, kernel)
    return e.get("cold_bytes_per_launch"), e.get("warm_bytes_per_launch"), note


def ncu_import(args):
    """bench.py --ncu-import RAW.csv [RAW2.csv ...] --ncu-key cfg3_rows3_kernel0 --ncu-mode cold|warm:
    reads `ncu -i X.ncu-rep --page raw --csv` output, averages dram__bytes_read.sum + dram__bytes_write.sum
    over the Dslash launches in it and stores the figure (with today's kernel-source hash)."""
    import csv
    tot, n, dur = 0.0, 0, 0.0
    for path in args.ncu_import:
        with open(path, newline="") as fh:
            rows = list(csv.reader(fh))
        hdr = rows[0]
        units = rows[1]
        ik = hdr.index("Kernel Name")
        ir, iw = hdr.index("dram__bytes_read.sum"), hdr.index("dram__bytes_write.sum")
        it = hdr.index("gpu__time_duration.sum")
        scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
        tscale = {"ns": 1e-9, "us": 1e-6, "usecond": 1e-6, "nsecond": 1e-9, "ms": 1e-3, "msecond": 1e-3}
        for r in rows[2:]:
            if len(r) <= max(ir, iw) or "dslash" not in r[ik]:
                continue
            tot += float(r[ir].replace(",", "")) * scale[units[ir]] + float(r[iw].replace(",", "")) * scale[units[iw]]
            dur += float(r[it].replace(",", "")) * tscale[units[it]]
            n += 1
    if n == 0:
        raise SystemExit("no Dslash launches in the ncu export")
    try:
        with open(TRAFFIC_JSON) as fh:
            doc = json.load(fh)
    except Exception:
        doc = {"what": "dram__bytes_read.sum + dram__bytes_write.sum per Dslash launch (ncu --set full); "
                       "cold = ncu's default cache flush before every replay, warm = --cache-control none "
                       "inside back-to-back applies; written by `python bench.py --ncu-import`",
               "entries": {}}
    e = doc["entries"].setdefault(args.ncu_key, {})
    e[f"{args.ncu_mode}_bytes_per_launch"] = tot / n
    e[f"{args.ncu_mode}_us_per_launch_under_ncu"] = 1e6 * dur / n
    e[f"{args.ncu_mode}_launches"] = n
    e["source_hash"] = kernel_source_hash(1 if args.ncu_key.endswith("kernel1") else 0)
    with open(TRAFFIC_JSON, "w") as fh:
        json.dump(doc, fh, indent=1, sort_keys=True)
        fh.write("\n")
    print(json.dumps({args.ncu_key: e}))


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def dslash_bytes(volume: int, link_rows: int = 3) -> int:
    """Algorithmic bytes of one single-parity Dslash apply: links 576V + in 24V + out 24V
    (DESIGN.md 'Algorithmic bytes'); two-row storage moves 384V of links."""
    return (624 if link_rows == 3 else 432) * volume


def dslash_flops(volume: int) -> int:
    return 285 * volume          # 570 flop per output site


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def max_over_ranks(values, dist=None, device="cpu"):
    """Element-wise MAX over all ranks of a list of floats (device timings).  `dist` is
    torch.distributed once initialised (nccl on the GPU box, gloo in the CPU tests) or None."""
    import torch
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def whole_job_rate(world: int, units_per_rank: float, slowest_seconds: float) -> float:
    """Replicas only: every rank processes `units_per_rank`; the job's rate is
    all ranks' units over the slowest rank's time."""
    return world * units_per_rank / slowest_seconds


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled every 50 ms during the timed region."""

    FIELDS = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index: int):
        self.proc = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(index), f"--query-gpu={self.FIELDS}",
                 "--format=csv,noheader,nounits", "-lms", "50"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except Exception:
            self.proc.kill()
            out = ""
        sm, mx, reasons = [], [], set()
        for line in out.splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for name, val in zip(self.NAMES, f[2:6]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                "samples": len(sm)}


def oracle_sample(cfg, links, b, shifts, res, dslash_seconds: float = 6.0, cg_seconds: float = 12.0):
    """Time the oracle as it stands on the host cores on a bounded sample of the workload: (D_oe, D_eo)
    pairs on the full lattice for about `dslash_seconds`, then the multishift CG at the requested tol
    for as many iterations as fit in about `cg_seconds` (the whole solve if it fits)."""
    import oracle
    lat = oracle.Lattice(cfg.dims, links)
    vo = lat.dslash(1, b)                       # warm-up, also the odd vector
    n_pairs = 0
    t0 = time.perf_counter()
    while True:
        vo = lat.dslash(1, b)
        ve = lat.dslash(0, vo)
        n_pairs += 1
        t_d = time.perf_counter() - t0
        if t_d >= dslash_seconds:
            break
    del ve
    # the same pair on ONE thread ("for Dslash only, also with 1 thread")
    nthreads = oracle.threads()
    oracle.set_threads(1)
    t0 = time.perf_counter()
    lat.dslash(0, lat.dslash(1, b))
    t_1 = (time.perf_counter() - t0) / 2
    oracle.set_threads(nthreads)
    gbps = 2 * n_pairs * dslash_bytes(cfg.volume) / t_d / 1e9
    t0 = time.perf_counter()
    probe = lat.multishift_cg(cfg.mass, cfg.parity, b, shifts, res, cfg.tol, max_iter=3, want_x=False)
    per_it = (time.perf_counter() - t0) / max(probe["iterations"], 1)
    iters = max(3, int(cg_seconds / per_it))
    t0 = time.perf_counter()
    out = lat.multishift_cg(cfg.mass, cfg.parity, b, shifts, res, cfg.tol, max_iter=iters, want_x=False)
    t_cg = time.perf_counter() - t0
    return dict(gbps=gbps, dslash_s=t_d / (2 * n_pairs), dslash_s_1thread=t_1, pairs=n_pairs,
                cg_s_per_iter=t_cg / max(out["iterations"], 1), cg_iters=out["iterations"],
                cg_converged=out["status"] == 0, cg_seconds=t_cg,
                cores=oracle.threads(), seconds=t_d + t_cg)


def run_reference(args, cfg, links, b, shifts, res):
    """--impl reference: the CPU oracle on the host cores; each step is a bounded sample."""
    import oracle
    lat = oracle.Lattice(cfg.dims, links)
    pairs = 2
    for _ in range(args.warmup):
        lat.dslash(0, lat.dslash(1, b))
    t0 = time.perf_counter()
    for _ in range(args.steps):
        for _ in range(pairs):
            lat.dslash(0, lat.dslash(1, b))
    t = time.perf_counter() - t0
    value = args.steps * pairs * 2 * dslash_bytes(cfg.volume) / t / 1e9
    t0 = time.perf_counter()
    cg = lat.multishift_cg(cfg.mass, cfg.parity, b, shifts, res, cfg.tol, max_iter=10, want_x=False)
    t_cg = (time.perf_counter() - t0) / max(cg["iterations"], 1)
    sample = (f"{pairs} x (D_oe, D_eo) per step on {cfg.name}, all of the lattice; CG: 10 iterations "
              f"of the {cfg.nshift}-shift solve")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": workload_config(cfg, args),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.threads(), "kind": "oracle",
                         "sample": sample, "cg_s_per_iteration": t_cg},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_config(cfg, args):
    nx, ny, nz, nt = cfg.dims
    return {"workload": f"config {cfg.number}: {nx}^3x{nt} staggered fp64, {cfg.links} SU(3) links"
                        f"{' eps=%g' % cfg.eps if cfg.eps else ''}, m={cfg.mass}, "
                        f"{cfg.nshift} shifts in [{cfg.shift_lo:g},{cfg.shift_hi:g}], tol={cfg.tol:g}",
            "dims": list(cfg.dims), "dslash_pairs_per_step": PAIRS, "mdagm_per_step": PAIRS // 2,
            "solves_per_step": 1,
            "l2": "no explicit flush: the links (576 V bytes: 151 MB at config 3) exceed the 126 MB L2, the "
                  "vectors do not; in the steady state of back-to-back applies L2 serves the vectors and part "
                  "of the links (D_oe and D_eo read the same links and walk them in opposite directions, the last "
                  "48 MB of each sweep are kept for the next: see roofline.frac_dram for the DRAM side); "
                  "dslash.cold_l2 is the same launch after a flush, `streaming` the 2.4 GB config-5 field",
            "parallelism": "replicas only" if args.gpus > 1 else "single GPU"}


def streaming_record(torch, q, args, peak, device_index):
    """Config 5 (64^3 x 16: 2.4 GB of links, 20x the L2), Dslash only: the clean streaming case
    (SURVEY.md 7 hard part 2, 8(d)).  20 graph-replayed (D_oe, D_eo) pairs, own clock sample."""
    cfg = li.CONFIGS[5]
    V = cfg.volume
    links = li.make_links(cfg.dims, cfg.links, cfg.seed, cfg.eps)
    b = li.make_source(cfg.dims, cfg.seed, cfg.parity)
    stream = torch.cuda.current_stream()
    ctx = q.Context(cfg.dims, cfg.mass, stream=stream.cuda_stream)
    if args.dslash_kernel >= 0:
        ctx.set_option(q.QCD_OPT_DSLASH_KERNEL, args.dslash_kernel)
    if args.dslash_persist >= 0:
        ctx.set_option(q.QCD_OPT_DSLASH_PERSIST, args.dslash_persist)
    ctx.load_gauge_host(links)
    del links
    d_b, d_o, d_e = ctx.new_vector(), ctx.new_vector(), ctx.new_vector()
    ctx.pack(0, torch.from_numpy(b).cuda().reshape(-1), d_b)
    pairs = 20
    g = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    side.wait_stream(stream)
    with torch.cuda.stream(side):
        ctx.set_stream(side.cuda_stream)
        ctx.dslash(1, d_b, d_o)
        ctx.dslash(0, d_o, d_e)
        side.synchronize()
        with torch.cuda.graph(g, stream=side):
            for _ in range(pairs):
                ctx.dslash(1, d_b, d_o)
                ctx.dslash(0, d_o, d_e)
    ctx.set_stream(stream.cuda_stream)
    stream.wait_stream(side)
    for _ in range(3):
        g.replay()
    torch.cuda.synchronize()
    sampler = ClockSampler(device_index)
    reps = 10
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        g.replay()
    e1.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    t = e0.elapsed_time(e1) * 1e-3 / (reps * 2 * pairs)
    cold, warm, src = load_traffic(5, 3, max(args.dslash_kernel, 0))
    ctx.close()
    gbps = dslash_bytes(V) / t / 1e9
    return {"workload": "config 5: 64^3x16 staggered fp64, random SU(3) links (2.4 GB), Dslash only",
            "us_per_apply": 1e6 * t, "GBps": gbps, "frac": gbps / peak, "pct_of_8000": 100 * gbps / 8000.0,
            "gflops": dslash_flops(V) / t / 1e9, "algorithmic_bytes_per_launch": dslash_bytes(V),
            "traffic": cold, "frac_dram": (cold / t / 1e9 / peak) if cold else None, "traffic_source": src,
            "launches": reps * 2 * pairs, "clocks": clocks,
            "l2": "links 19x the L2: every link byte comes from DRAM; only the 100 MB vectors can hit"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", type=int, default=3, help="BASELINE.json config number (1-5)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-solve", action="store_true", help="skip section C (profiling aid)")
    ap.add_argument("--no-pdl", action="store_true", help="QCD_OPT_PDL=0 (A/B aid)")
    ap.add_argument("--no-cg-graph", action="store_true", help="QCD_OPT_CG_GRAPH=0 (A/B aid)")
    ap.add_argument("--cg-graph", type=int, default=-1, help="QCD_OPT_CG_GRAPH value (-1 = library default)")
    ap.add_argument("--cg-batch", type=int, default=0, help="QCD_OPT_CG_BATCH (0 = library default)")
    ap.add_argument("--link-rows", type=int, default=3, choices=[2, 3],
                    help="QCD_OPT_LINK_ROWS for the whole run (default 3, the paper's uncompressed "
                         "storage; the default run also reports a two-row section)")
    ap.add_argument("--tgroup", type=int, default=0, help="QCD_OPT_TGROUP (0 = library default)")
    ap.add_argument("--no-two-row", action="store_true", help="skip the extra two-row section")
    ap.add_argument("--no-streaming", action="store_true", help="skip the config-5 Dslash streaming record")
    ap.add_argument("--no-extras", action="store_true", help="skip inv_sqrt / fourth_root / two-row / mixed sections")
    ap.add_argument("--dslash-kernel", type=int, default=-1, help="QCD_OPT_DSLASH_KERNEL (-1 = library default)")
    ap.add_argument("--dslash-persist", type=int, default=-1, help="QCD_OPT_DSLASH_PERSIST (-1 = library default)")
    ap.add_argument("--profile-dslash", type=int, default=0,
                    help="profiling aid for ncu: only load the field and launch this many (D_oe, D_eo) pairs")
    ap.add_argument("--ncu-import", nargs="+", default=None, help="raw ncu csv export(s) -> profiles/r02_dslash_traffic.json")
    ap.add_argument("--ncu-key", default="cfg3_rows3_kernel0")
    ap.add_argument("--ncu-mode", default="cold", choices=["cold", "warm"])
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    if args.ncu_import:
        ncu_import(args)
        return 0

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        if rank != 0:
            return 0
        cfg, links, b, shifts, res = li.make_config_inputs(args.workload)
        run_reference(args, cfg, links, b, shifts, res)
        return 0

    import torch
    import paper_1710_09178_b200 as q

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    cfg, links, b, shifts, res = li.make_config_inputs(args.workload)
    V = cfg.volume
    stream = torch.cuda.current_stream()
    ctx = q.Context(cfg.dims, cfg.mass, stream=stream.cuda_stream)
    if args.no_pdl:
        ctx.set_option(q.QCD_OPT_PDL, 0)
    if args.no_cg_graph:
        ctx.set_option(q.QCD_OPT_CG_GRAPH, 0)
    if args.cg_graph >= 0:
        ctx.set_option(q.QCD_OPT_CG_GRAPH, args.cg_graph)
    if args.cg_batch:
        ctx.set_option(q.QCD_OPT_CG_BATCH, args.cg_batch)
    ctx.set_option(q.QCD_OPT_LINK_ROWS, args.link_rows)
    if args.tgroup:
        ctx.set_option(q.QCD_OPT_TGROUP, args.tgroup)
    if args.dslash_kernel >= 0:
        ctx.set_option(q.QCD_OPT_DSLASH_KERNEL, args.dslash_kernel)
    if args.dslash_persist >= 0:
        ctx.set_option(q.QCD_OPT_DSLASH_PERSIST, args.dslash_persist)
    kernel_id = max(args.dslash_kernel, 0)
    d_links = torch.from_numpy(links).cuda()
    ctx.load_gauge(d_links)
    torch.cuda.synchronize()
    del d_links

    d_b, d_o, d_e, d_a = ctx.new_vector(), ctx.new_vector(), ctx.new_vector(), ctx.new_vector()
    ctx.pack(0, torch.from_numpy(b).cuda().reshape(-1), d_b)
    d_y = ctx.new_vector()

    if args.profile_dslash:              # ncu aid: nothing but Dslash launches after the load
        for _ in range(args.profile_dslash):
            ctx.dslash(1, d_b, d_o)
            ctx.dslash(0, d_o, d_e)
        torch.cuda.synchronize()
        ctx.close()
        return 0

    # sections A and B as CUDA graphs (launch gaps minimised; the kernels are ~25 us each)
    def capture(fn):
        g = torch.cuda.CUDAGraph()
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            ctx.set_stream(side.cuda_stream)
            fn()                                   # warm-up outside capture
            side.synchronize()
            with torch.cuda.graph(g, stream=side):
                fn()
        ctx.set_stream(stream.cuda_stream)
        torch.cuda.current_stream().wait_stream(side)
        return g

    def section_a():
        for _ in range(PAIRS):
            ctx.dslash(1, d_b, d_o)    # D_oe
            ctx.dslash(0, d_o, d_e)    # D_eo

    def section_b():
        for _ in range(PAIRS // 2):
            ctx.mdagm(0, d_b, d_a)

    graph_a, graph_b = capture(section_a), capture(section_b)
    launches_a, launches_b = 2 * PAIRS, 2 * (PAIRS // 2)

    def solve():
        return ctx.multishift_cg(cfg.parity, d_b, shifts, res, cfg.tol, 100000, None, d_y)

    ev = lambda: torch.cuda.Event(enable_timing=True)  # noqa: E731
    t_a = t_b = 0.0
    t_c = []
    iters = 0
    cg_launches = 0

    def step(timed: bool):
        nonlocal t_a, t_b, iters, cg_launches
        e0, e1, e2 = ev(), ev(), ev()
        e0.record()
        graph_a.replay()
        e1.record()
        graph_b.replay()
        e2.record()
        if not args.no_solve:
            l0 = ctx.launch_count
            torch.cuda.synchronize()           # sections A and B are asynchronous: drain them first
            w0 = time.perf_counter()
            st, it, tr = solve()
            w1 = time.perf_counter()
            assert st == 0 and tr.max() <= 1.5 * cfg.tol, (st, tr)
        torch.cuda.synchronize()
        if timed:
            t_a += e0.elapsed_time(e1) * 1e-3
            t_b += e1.elapsed_time(e2) * 1e-3
            if not args.no_solve:
                t_c.append(w1 - w0)
                iters = it
                cg_launches = ctx.launch_count - l0

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step(False)
    barrier()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    e_start, e_stop = ev(), ev()
    e_start.record()
    for _ in range(args.steps):
        step(True)
    e_stop.record()
    barrier()
    total_s = e_start.elapsed_time(e_stop) * 1e-3
    clocks = sampler.stop() if sampler else None

    # max over ranks of every timing
    total_s, t_a, t_b, t_c_sum = max_over_ranks([total_s, t_a, t_b, sum(t_c)], dist, "cuda")

    K = args.steps
    n = world
    R = args.link_rows
    bytes_a = K * launches_a * dslash_bytes(V, R)
    value = whole_job_rate(n, bytes_a, t_a) / 1e9
    per_launch_s = t_a / (K * launches_a)
    peak, peak_src = measured_peak()
    achieved = dslash_bytes(V, R) / per_launch_s / 1e9
    mdagm_bytes = 2 * dslash_bytes(V, R) + 24 * V
    traffic_cold, traffic_warm, traffic_src = load_traffic(cfg.number, R, kernel_id)
    mdagm_gbps = n * K * (PAIRS // 2) * mdagm_bytes / t_b / 1e9

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": n, "steps": K, "warmup": args.warmup,
        "ms_per_step": 1e3 * total_s / K, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "value_note": "L2-ASSISTED steady state of back-to-back applies: algorithmic bytes (624 V per apply) over time, "
                      "not DRAM bandwidth; DRAM side: roofline.frac_dram; every byte from DRAM: dslash.cold_l2 / "
                      "target_check (one launch behind a flushed L2) and streaming (64^3x16)",
        "config": workload_config(cfg, args),
        "dslash": {"us_per_apply": 1e6 * per_launch_s, "gflops": dslash_flops(V) / per_launch_s / 1e9,
                   "pct_of_8000": 100 * achieved / 8000.0, "pct_of_measured_peak": 100 * achieved / peak},
        "mdagm": {"us_per_apply": 1e6 * t_b / (K * (PAIRS // 2)), "GBps": mdagm_gbps, "algorithmic_bytes": mdagm_bytes},
        "roofline": {"bound": "hbm",
                     "kernel": ("dslash_bulk_kernel" if kernel_id == 1 else "dslash_kernel") + "<false,false> (one D_oe or D_eo apply)",
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "peak_source": peak_src,
                     "frac_note": "ALGORITHMIC bytes / time in the steady state of back-to-back applies: L2 serves the "
                                  "vectors and part of the links, so this is not a pure HBM fraction (frac_dram is); "
                                  "hbm_gbs is a copy (read+write) rate and the kernel is 96 % reads (read-only probe of "
                                  "the same pattern: DESIGN.md section 5)",
                     "algorithmic_bytes_per_launch": dslash_bytes(V, R), "link_rows": R,
                     "traffic": traffic_cold, "traffic_warm": traffic_warm,
                     "frac_dram": (traffic_warm / per_launch_s / 1e9 / peak) if traffic_warm else None,
                     "traffic_note": "traffic: dram__bytes_read+write per launch with ncu's cache flush (cold L2); "
                                     "traffic_warm: the same inside back-to-back applies (--cache-control none); "
                                     "frac_dram = traffic_warm / live launch time / peak; source: " + traffic_src},
        "gpu_launches": K * (launches_a + launches_b + cg_launches),
    }
    # the same apply with a COLD L2.  One graph holds 10 x (overwrite a 512 MB buffer, one Dslash), a second
    # one the 10 flushes alone; their difference / 10 is what an isolated launch behind a flushed L2 costs,
    # without the ~6 us a CUDA-event bracket around a single short kernel adds.  (Section A above is the
    # steady state of back-to-back applies, where L2 holds the vectors and part of the links.)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    NCOLD = 10

    def cold_with():
        for i in range(NCOLD):
            flush.fill_(i)
            ctx.dslash(1 - (i & 1), d_b if not (i & 1) else d_o, d_o if not (i & 1) else d_e)

    def cold_without():
        for i in range(NCOLD):
            flush.fill_(i)

    g_with, g_without = capture(cold_with), capture(cold_without)

    def time_graph(g, reps=7):
        ts = []
        for _ in range(reps):
            e0, e1 = ev(), ev()
            e0.record()
            g.replay()
            e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1) * 1e-3)
        return statistics.median(ts[2:])

    t_without = time_graph(g_without)
    cold_s = (time_graph(g_with) - t_without) / NCOLD
    # the same with QCD_OPT_SWEEP_ALTERNATE = 0 (one direction, every link streaming): the setting meant for an
    # isolated apply; the library default keeps the tail of each sweep in L2 for the NEXT apply
    ctx.set_option(q.QCD_OPT_SWEEP_ALTERNATE, 0)
    g_with0 = capture(cold_with)
    cold0_s = (time_graph(g_with0) - t_without) / NCOLD
    ctx.set_option(q.QCD_OPT_SWEEP_ALTERNATE, 1)
    del flush, g_with, g_with0, g_without

    def cold_record(sec, what):
        return {"us_per_apply": 1e6 * sec, "GBps": dslash_bytes(V, R) / sec / 1e9,
                "frac_of_peak": dslash_bytes(V, R) / sec / 1e9 / peak,
                "pct_of_8000": 100 * dslash_bytes(V, R) / sec / 1e9 / 8000.0, "what": what}

    line["dslash"]["cold_l2"] = cold_record(
        cold_s, "library default (alternating sweeps, 48 MB of links kept for the next apply): one launch behind a "
                "512 MB L2 flush = (graph of 10 x [flush, Dslash]) - (graph of 10 x [flush]), median of 5 replays "
                "each, / 10; no predecessor to overlap with")
    line["dslash"]["cold_l2"]["flush_us"] = 1e6 * t_without / NCOLD
    line["dslash"]["cold_l2_streaming"] = cold_record(
        cold0_s, "the same with QCD_OPT_SWEEP_ALTERNATE = 0: one direction, every link loaded evict-first")
    # The live figures above are differences of two graph timings and include the ~2 us between the end of the
    # flush kernel and the first CTA of the Dslash; the kernel's own duration behind a flushed L2 is what ncu
    # reports (gpu__time_duration, cache flushed before every replay), stored with the traffic figures.
    te, te_note = traffic_entry(cfg.number, R, kernel_id)
    ncu_cold_us = te.get("cold_us_per_launch_under_ncu") if "STALE" not in te_note else None
    ncu_pct = 100 * dslash_bytes(V, R) / (ncu_cold_us * 1e-6) / 1e9 / 8000.0 if ncu_cold_us else None
    live_best = max(line["dslash"]["cold_l2"]["pct_of_8000"], line["dslash"]["cold_l2_streaming"]["pct_of_8000"])
    line["target_check"] = {
        "target": "fp64 Dslash >= 70 % of B200 HBM peak (~8 TB/s) at 32^3 x 8 (BASELINE.json north_star)",
        "cold_l2_pct_of_8000": line["dslash"]["cold_l2"]["pct_of_8000"],
        "cold_l2_streaming_pct_of_8000": line["dslash"]["cold_l2_streaming"]["pct_of_8000"],
        "cold_l2_ncu_kernel_duration_us": ncu_cold_us, "cold_l2_ncu_pct_of_8000": ncu_pct, "ncu_source": te_note,
        "steady_state_pct_of_8000": line["dslash"]["pct_of_8000"],
        "evaluated_on": "the cold-L2 launch (every byte from DRAM): the kernel duration ncu measured for exactly these "
                        "kernel sources if a capture is stored, else the live graph-difference figure (which "
                        "includes the launch gap); the steady-state figure is L2-assisted and is not used",
        "met": (bool((ncu_pct if ncu_pct is not None else live_best) >= 70.0) if cfg.number == 3 else None)}

    if not args.no_solve:
        line["cg"] = {"s_per_solve": t_c_sum / K, "iterations": iters,
                      "us_per_iteration": 1e6 * (t_c_sum / K) / max(iters, 1), "nshift": cfg.nshift,
                      "tol": cfg.tol, "includes": "true residuals (a6) and y = sum c_k x_k",
                      "defer": "QCD_OPT_CG_DEFER = 8 (shifts k >= 1 updated once per 8 iterations, bit-identical)",
                      "timing": "host wall clock around the blocking C-ABI call"}
    if clocks is not None:
        line["clocks"] = clocks

    if rank == 0:
        # e2e: the same metric through the C ABI with HOST buffers (pinned), copies inside the region
        hb = torch.from_numpy(b).pin_memory().numpy()
        ho = torch.empty(b.shape, dtype=torch.float64).pin_memory().numpy()
        he = torch.empty(b.shape, dtype=torch.float64).pin_memory().numpy()
        hy = torch.empty(b.shape, dtype=torch.float64).pin_memory().numpy()
        for _ in range(max(args.warmup, 1)):
            ctx.dslash_host(1, hb, ho)
            ctx.dslash_host(0, ho, he)
        torch.cuda.synchronize()
        reps = max(K, 5)
        w0 = time.perf_counter()
        for _ in range(reps):
            ctx.dslash_host(1, hb, ho)
            ctx.dslash_host(0, ho, he)
        w = time.perf_counter() - w0
        e2e = {"value": reps * 2 * dslash_bytes(V, R) / w / 1e9, "unit": UNIT,
               "h2d_bytes_per_step": 2 * b.nbytes, "d2h_bytes_per_step": 2 * b.nbytes,
               "step": "qcd_dslash_host(D_oe) + qcd_dslash_host(D_eo), pinned host vectors, gauge resident",
               "us_per_apply": 1e6 * w / (2 * reps)}
        if not args.no_solve:
            ts = []
            for _ in range(4):          # the first call allocates the staging buffers: not timed
                w0 = time.perf_counter()
                st, it, tr = ctx.multishift_cg_host(cfg.parity, hb, shifts, res, cfg.tol, 100000, None, hy)
                ts.append(time.perf_counter() - w0)
            e2e["cg_s_per_solve"] = statistics.median(ts[1:])
            e2e["cg_h2d_bytes"] = b.nbytes
            e2e["cg_d2h_bytes"] = b.nbytes
        w0 = time.perf_counter()
        ctx.load_gauge_host(links)
        e2e["gauge_ingest_s"] = time.perf_counter() - w0
        e2e["gauge_h2d_bytes"] = links.nbytes
        line["e2e"] = e2e

        if not args.no_solve and not args.no_extras:
            # the same solve with the shift updates applied every iteration (round-1 behaviour), for the record
            ctx.set_option(q.QCD_OPT_CG_DEFER, 1)
            ts = []
            for _ in range(3):
                torch.cuda.synchronize()
                w0 = time.perf_counter()
                st, it, tr = solve()
                ts.append(time.perf_counter() - w0)
            line["cg"]["undeferred_s_per_solve"] = statistics.median(ts[1:])
            ctx.set_option(q.QCD_OPT_CG_DEFER, 8)

        if not args.no_solve and not args.no_extras:
            # the paper's step 2, (M^dag M)^(-1/2) phi via eq. 8
            xmin, xmax = 0.9 * cfg.mass ** 2, 8.5      # the paper's xmax = 34 in its normalisation
            ts = []
            for _ in range(3):
                torch.cuda.synchronize()
                w0 = time.perf_counter()
                st, it, tr, delta = ctx.inv_sqrt(cfg.parity, d_b, cfg.nshift, xmin, xmax, cfg.tol,
                                                 100000, d_y)
                ts.append(time.perf_counter() - w0)
                assert st == 0 and tr.max() <= 1.5 * cfg.tol, (st, tr)
            line["inv_sqrt"] = {"n": cfg.nshift, "xmin": xmin, "xmax": xmax, "delta": delta,
                                "iterations": it, "s_per_apply": statistics.median(ts[1:]),
                                "what": "qcd_inv_sqrt: Zolotarev coefficients + one multishift CG + "
                                        "fused c0*phi + sum c_k x_k"}

            # ... and the heat-bath power (M^dag M)^(1/4) (Remez coefficients, cached)
            ts = []
            for _ in range(3):
                torch.cuda.synchronize()
                w0 = time.perf_counter()
                st, it, tr, delta = ctx.apply_pow(cfg.parity, d_b, 1, 4, cfg.nshift, xmin, xmax, cfg.tol,
                                                  100000, d_y)
                ts.append(time.perf_counter() - w0)
                assert st == 0 and tr.max() <= 1.5 * cfg.tol, (st, tr)
            line["fourth_root"] = {"n": cfg.nshift, "delta": delta, "iterations": it,
                                   "s_per_apply": statistics.median(ts[1:]),
                                   "first_call_s": ts[0],
                                   "what": "qcd_apply_pow(1/4): Remez coefficients in binary128 on the "
                                           "first call, then one multishift CG + fused combine"}

            # QCD_OPT_Y_ONLY: the same two applications without forming the x_k
            ctx.set_option(q.QCD_OPT_Y_ONLY, 1)
            for key, fn in (("inv_sqrt", lambda: ctx.inv_sqrt(cfg.parity, d_b, cfg.nshift, xmin, xmax, cfg.tol, 100000, d_y)),
                            ("fourth_root", lambda: ctx.apply_pow(cfg.parity, d_b, 1, 4, cfg.nshift, xmin, xmax, cfg.tol, 100000, d_y))):
                ts = []
                for _ in range(3):
                    torch.cuda.synchronize()
                    w0 = time.perf_counter()
                    st, it, tr, delta = fn()
                    ts.append(time.perf_counter() - w0)
                    assert st == 0 and tr.max() <= 1.5 * cfg.tol, (st, tr)
                line[key]["y_only_s_per_apply"] = statistics.median(ts[1:])
            ctx.set_option(q.QCD_OPT_Y_ONLY, 0)

        if R == 3 and not args.no_two_row and not args.no_extras:
            # the same sections A and C with two-row link storage
            ctx.set_option(q.QCD_OPT_LINK_ROWS, 2)
            ctx.load_gauge_host(links)
            graph_a2 = capture(section_a)
            for _ in range(max(args.warmup, 1)):
                graph_a2.replay()
            torch.cuda.synchronize()
            e0, e1 = ev(), ev()
            e0.record()
            for _ in range(K):
                graph_a2.replay()
            e1.record()
            torch.cuda.synchronize()
            t2 = e0.elapsed_time(e1) * 1e-3 / (K * launches_a)
            two = {"link_rows": 2, "us_per_apply": 1e6 * t2,
                   "GBps_at_432V": dslash_bytes(V, 2) / t2 / 1e9,
                   "frac_of_peak": dslash_bytes(V, 2) / t2 / 1e9 / peak,
                   "gflops": (285 + 168) * V / t2 / 1e9,
                   "speedup_vs_three_row": per_launch_s / t2}
            if not args.no_solve:
                ts = []
                for _ in range(max(1, min(K, 3)) + 1):
                    torch.cuda.synchronize()
                    w0 = time.perf_counter()
                    st, it, tr = solve()
                    ts.append(time.perf_counter() - w0)
                    assert st == 0 and tr.max() <= 1.5 * cfg.tol, (st, tr)
                two["cg_s_per_solve"] = statistics.median(ts[1:])
                two["cg_iterations"] = it
            line["two_row"] = two
            ctx.set_option(q.QCD_OPT_LINK_ROWS, 3)

        if not args.no_solve and not args.no_extras and R == 3:
            # the mixed-precision form of the solve, against the fp64 solver
            ctx.set_option(q.QCD_OPT_MIXED, 1)
            ctx.load_gauge_host(links)
            mixed = {"what": "fp64 multishift to 10^-switch_exp, then per-shift defect correction with the "
                             "fp32-link inner operator (fp64 arithmetic); `iterations` = stage 1 + all inner",
                     "fp64_solver_s_per_solve": t_c_sum / K, "runs": []}
            for sw in (3, 5, 8):
                ctx.set_option(q.QCD_OPT_MIXED_SWITCH_EXP, sw)
                ts = []
                for _ in range(3):
                    torch.cuda.synchronize()
                    w0 = time.perf_counter()
                    st, it, tr = solve()
                    ts.append(time.perf_counter() - w0)
                    assert st == 0 and tr.max() <= 1.5 * cfg.tol, (st, tr)
                mixed["runs"].append({"switch_exp": sw, "s_per_solve": statistics.median(ts[1:]), "iterations": it,
                                      "max_true_res": float(tr.max())})
            ctx.set_option(q.QCD_OPT_OPERATOR_LINKS32, 1)     # the inner operator on its own
            g32 = capture(section_a)
            for _ in range(3):
                g32.replay()
            torch.cuda.synchronize()
            e0, e1 = ev(), ev()
            e0.record()
            for _ in range(max(K, 3)):
                g32.replay()
            e1.record()
            torch.cuda.synchronize()
            t32 = e0.elapsed_time(e1) * 1e-3 / (max(K, 3) * launches_a)
            mixed["fp32_link_dslash"] = {"us_per_apply": 1e6 * t32, "algorithmic_bytes": 336 * V,
                                         "GBps_at_336V": 336 * V / t32 / 1e9, "speedup_vs_fp64_links": per_launch_s / t32}
            ctx.set_option(q.QCD_OPT_OPERATOR_LINKS32, 0)
            ctx.set_option(q.QCD_OPT_MIXED, 0)
            line["mixed_precision"] = mixed
            del g32

        ctx.close()
        if cfg.number != 5 and not args.no_streaming:
            line["streaming"] = streaming_record(torch, q, args, peak, local_rank)

        if not args.no_cpu_baseline:
            smp = oracle_sample(cfg, links, b, shifts, res)
            line["cpu_baseline"] = {
                "value": smp["gbps"], "unit": UNIT, "cores": smp["cores"], "kind": "oracle",
                "sample": f"{smp['pairs']} x (D_oe, D_eo) on the full {cfg.name} lattice + {smp['cg_iters']} "
                          f"iterations of the {cfg.nshift}-shift CG"
                          f"{' (the whole solve)' if smp['cg_converged'] else ''} "
                          f"({smp['seconds']:.1f} s of host time)",
                "dslash_us_per_apply": 1e6 * smp["dslash_s"], "dslash_us_per_apply_1_thread": 1e6 * smp["dslash_s_1thread"],
                "cg_s_per_iteration": smp["cg_s_per_iter"],
                "cg_s_sampled": smp["cg_seconds"], "cg_converged_in_sample": smp["cg_converged"],
                "host_cpu_count": os.cpu_count()}
        print(json.dumps(line), flush=True)

    ctx.close()
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
