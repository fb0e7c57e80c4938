#!/usr/bin/env python
"""bench.py — zone-cycles/s of the fp64 GRMHD step on B200 (BASELINE.json metric), the HBM/ALU roofline
fraction of the dominant kernel, the end-to-end number through the C-ABI with host buffers, and the
CPU oracle timed beside it.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload cfg2|cfg2r|cfg1|cfg0|cfg3|cfg4b|cfg4|cfg4t|cfg4r|paper150]
                  [--shard S]

A "step" is one full pass of the hot path over the whole grid: hamr_step(1) = predictor + corrector
= one zone-cycle per zone.  Default workload: BASELINE.json configs[2], the 256x128x128
Kerr Fishbone-Moncrief torus (the config the metric is quoted on).  Inputs are seeded and synthetic
(paper_1912_10192_b200/inputs.py); the state (2.4 GB of fp64 arrays) is far larger than the 126 MB L2.
N > 1: BASELINE's north_star runs everything on one GPU ("replicas only"): every rank runs an independent
replica.  --shard runs ONE grid as x1 slabs instead: one slab per rank under torchrun.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "zone_cycles_per_sec"
UNIT = "zone-cycles/s"


def workload(name, n_override=None):
    from paper_1912_10192_b200 import inputs as I
    if name == "cfg2":
        # n_override: the reference arm's bounded sample (run_reference) only
        p = I.torus_params(n=n_override or (256, 128, 128), r_out=1000.0)
        return p, (lambda: I.fm_torus(p, seed=2)), "BASELINE cfg2: Kerr FM torus 256x128x128 fp64, a=0.9375, PPM+HLL+CT"
    if name == "cfg2r":
        # cfg 2 with the robust inversion path on: ninth conserved row, entropy inversion where
        # the energy inversion fails, drift-frame floors; runs on the generic kernels
        p = I.torus_params(n=n_override or (256, 128, 128), r_out=1000.0, entropy_backup=1, drift_floors=1)
        return p, (lambda: I.fm_torus(p, seed=2)), ("cfg2 with entropy advection + backup inversion and drift-frame floors "
                                                    "(NEXT-2): Kerr FM torus 256x128x128 fp64")
    if name == "cfg0":
        p = I.torus_params()
        return p, (lambda: I.fm_torus(p, seed=0)), "BASELINE cfg0: tiny Kerr FM torus 32x16x16"
    if name == "cfg1":
        p = I.minkowski_params(n=(128, 128, 128))
        return p, (lambda: I.minkowski_waves(p, seed=1)), "BASELINE cfg1: Minkowski periodic 128^3 linear waves"
    if name == "paper150":
        # the paper's own single-GPU benchmark shape (one 150^3 block, no AMR / SMR / LAT): context
        p = I.torus_params(n=(150, 150, 150), r_out=1000.0)
        return p, (lambda: I.fm_torus(p, seed=2)), "paper's single-GPU shape: one 150^3 Kerr-Schild block (FM torus data)"
    if name == "cfg3":
        p = I.tilted_disk_params()
        return p, (lambda: I.tilted_disk(p, seed=3)), ("BASELINE cfg3: tilted thin disk 512x256x256 fp64 (synthetic stand-in: "
                                                        "h/r=0.03, tilt 65 deg, toroidal field beta=10)")
    if name == "cfg4b":
        # the part of BASELINE cfg 4 that is built: cfg 2's torus (seed 4) on 16 x 16 x 128
        # blocks, phi-derefined by 2 / 4 within 15 / 5 degrees of the poles, LAT levels 1, 2, 4; no r-refinement
        p = I.torus_params(n=(256, 128, 128), r_out=1000.0, nb=(16, 16, 128), lat_max_level=2,
                           deref_theta_deg=(15.0, 5.0), deref_factor=(2, 4))
        return p, (lambda: I.fm_torus(p, seed=4)), ("BASELINE cfg4 without r-refinement: Kerr FM torus 256x128x128 in 16x16x128 "
                                                     "blocks, phi-derefinement 2x/4x, LAT levels 1/2/4")
    if name in ("cfg4", "cfg4t", "cfg4r"):
        # BASELINE cfg 4: base 256x128x128 in 16^3 blocks, phi-derefined 2x / 4x within 15 / 5
        # degrees of the poles, one x1 refinement level for r < 20 (1472 blocks, 6 029 312 zones), LAT levels 1, 2, 4;
        # torus data sampled per block, seed 4.  gen() returns the per-block data.
        # cfg4t: the same grid with the paper's own polar boundary (NEXT-1) instead of BASELINE's reflecting
        # one: the rows beyond the pole of every polar block come from the block half a turn away
        bc = {}
        if name == "cfg4t":
            bc = dict(bc_lo=(I.BC_OUTFLOW, I.BC_POLAR_TRANSMIT, I.BC_PERIODIC),
                      bc_hi=(I.BC_OUTFLOW, I.BC_POLAR_TRANSMIT, I.BC_PERIODIC))
        if name == "cfg4r":   # cfg 4 with the robust inversion path on (NEXT-2 on the whole feature set)
            bc = dict(entropy_backup=1, drift_floors=1)
        p = I.torus_params(n=(256, 128, 128), r_out=1000.0, nb=(16, 16, 16), lat_max_level=2, r_refine_max=20.0,
                           deref_theta_deg=(15.0, 5.0), deref_factor=(2, 4), **bc)
        return p, (lambda infos: I.fm_torus_blocks(p, infos, seed=4)), ("BASELINE cfg4: Kerr FM torus, base 256x128x128 in "
                   "16^3 blocks (1472), one x1 refinement level r<20, phi-derefinement 2x/4x, LAT levels 1/2/4"
                   + (", transmissive poles" if name == "cfg4t" else "")
                   + (", entropy backup + drift-frame floors (NEXT-2)" if name == "cfg4r" else ""))
    raise SystemExit(f"unknown workload {name}")


class ClockSampler:
    """samples nvidia-smi clocks / throttle reasons while the timed region runs"""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for nme, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# algorithmic doubles per unit of each kernel class: (reads, writes) per face / zone
ALG_RW = {"flux_x1": (9, 7), "flux_x2": (9, 7), "flux_x3": (9, 7),   # r: P5, 2 transverse Bc, Bf^d; w: F5, 2 EMFs
          # update: r src P5+Bc3 (+ base P5+Bc3 in the corrector), base Bf3, Ee3, F15; w P5, Bc3, Bf3
          "update_predictor": (8 + 3 + 3 + 15, 11), "update_corrector": (8 + 8 + 3 + 3 + 15, 11),
          "centre_emf": (6, 3), "edge_emf": (6 + 3 + 3, 3), "ghosts": (0, 0), "dt": (0, 0), "other": (0, 0)}

# DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of each kernel class and the FP64 thread
# instructions (dadd + dmul + dfma) the flux kernels execute per face, from the round's `ncu --set full` capture of
# this same command on cfg 2
NCU_TRAFFIC_SOURCE = "profiles/r2e_ncu_full_cfg2.md"
NCU_TRAFFIC = {"flux_x1": 539700000, "flux_x2": 523600000, "flux_x3": 499400000, "centre_emf": 294500000,
               "edge_emf": 534800000, "update_predictor": 1459300000, "update_corrector": 1822900000, "ghosts": 15600000}
FLUX_FP64_INST_PER_FACE = {"flux_x1": 324.7, "flux_x2": 321.2, "flux_x3": 313.7}
FLUX_FMA_FRACTION = 0.445          # the DFMA share of those (2 FLOP each), the rest DADD / DMUL (1 FLOP)
# every instruction the flux kernels send down the FP64 pipe per face (the arithmetic above plus the compares behind
# min / max / limiter switches), from the same capture: sm__pipe_fp64_cycles_active x cycles / 2 cycles per warp
# instruction x 592 schedulers x 32 threads / faces; and all warp-level instructions per face-warp
FLUX_FP64PIPE_INST_PER_FACE = {"flux_x1": 355.0, "flux_x2": 352.0, "flux_x3": 343.0}
FLUX_INST_PER_FACE = {"flux_x1": 777.0, "flux_x2": 786.0, "flux_x3": 709.0}
FP64_PEAK_TFLOPS_DERIVED = 148 * 64 * 2 * 1.965e9 / 1e12
PAPER_V100_150CUBED = 0.85e8   # ~0.85e8 zone-cycles/s, 1 V100, one 150^3 block


def alg_bytes(cls, n):
    """algorithmic bytes of one launch of kernel class `cls` on a monolithic n1 x n2 x n3 grid.  The flux kernels
    evaluate one row of faces per transverse zone row incl. one ghost row on either side (C-9 reads them); along a
    periodic x3 the two ghost columns are stored twice, not computed: reads count the computed faces,
    writes the stored ones."""
    n1, n2, n3 = n
    r, w = ALG_RW.get(cls, (0, 0))
    if cls == "flux_x1":
        return 8 * (n1 + 1) * (n2 + 2) * (r * n3 + w * (n3 + 2))
    if cls == "flux_x2":
        return 8 * (n1 + 2) * (n2 + 1) * (r * n3 + w * (n3 + 2))
    return 8 * (r + w) * units_per_launch(cls, n)


def units_per_launch(cls, n):
    n1, n2, n3 = n
    if cls == "flux_x1":
        return (n1 + 1) * (n2 + 2) * (n3 + 2)
    if cls == "flux_x2":
        return (n1 + 2) * (n2 + 1) * (n3 + 2)
    if cls == "flux_x3":
        return (n1 + 2) * (n2 + 2) * (n3 + 1)
    if cls == "centre_emf":
        return (n1 + 2) * (n2 + 2) * (n3 + 2)
    if cls == "edge_emf":
        return (n1 + 1) * (n2 + 1) * (n3 + 1)
    return n1 * n2 * n3


def replica_throughput(ms_local, units_per_rank, world, device):
    """Whole-job value of N independent replicas ("replicas only"): the timed region of
    every rank, the MAX over ranks (one scalar all-reduce of the TIMING, not a data-path collective), and
    world x units / that time.  Returns (value per second, max ms).  Covered on CPU by a world_size-2 gloo test."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_max = float(t.item())
    return world * units_per_rank / (ms_max * 1e-3), ms_max


def oracle_set(o, p, gen):
    """initial state into an oracle grid (block by block on a refined grid); returns the number of zones"""
    if p["r_refine_max"] > 0:
        infos = []
        for b in range(o.num_blocks()):
            d = o.block_info(b)
            infos.append((d["x_lo"], d["dx"], d["n"]))
        for b, (hb, fb) in enumerate(gen(infos)):
            assert o.set_block_prims(b, hb, fb) == 0
        assert o.commit() == 0
        return sum(int(np.prod(i[2])) for i in infos)
    hyd, bf = gen()
    assert o.set_prims(hyd, bf) == 0
    return int(np.prod(p["n"]))


def cpu_oracle_time(p, gen, steps, threads=0):
    """times the oracle as it stands on the host cores: `steps` full steps of the workload (threads = 0: all cores)"""
    from tests import _orc
    _orc.lib().orc_set_threads.argtypes = [__import__("ctypes").c_int]
    _orc.lib().orc_set_threads(int(threads))
    o = _orc.OrcGrid(p)
    nz = oracle_set(o, p, gen)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    cores = int(_orc.lib().orc_omp_threads())
    o.close()
    _orc.lib().orc_set_threads(0)
    nz = nz * 2 ** int(p["lat_max_level"])   # effective zone-cycles per (coarse) step
    return nz * steps / dt, dt, cores


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import __graft_entry__ as ge
    subprocess.check_call(["make", "-s", "-C", os.path.join(ROOT, "oracle")])
    p, gen, desc = workload(args.workload)
    from tests import _orc
    # a bounded sample when K is large: one calibration step of the whole grid is timed; if K + W such steps would
    # take more than ~4 minutes, the same torus is set up on fewer x1 zones (same r range) so that they do not
    o = _orc.OrcGrid(p)
    nz0 = oracle_set(o, p, gen)
    tc = time.perf_counter()
    o.step(1)
    tc = time.perf_counter() - tc
    shrunk = None
    if args.workload == "cfg2" and tc * (args.steps + args.warmup) > 240.0:  # resized to ~180 s: small grids run a little slower per zone
        n0 = max(32, int(p["n"][0] * 180.0 / (tc * (args.steps + args.warmup))) // 8 * 8)
        shrunk = (n0,) + tuple(p["n"][1:])
        o.close()
        p, gen, desc = workload(args.workload, n_override=shrunk)
        o = _orc.OrcGrid(p)
        nz0 = oracle_set(o, p, gen)
    for _ in range(args.warmup):
        o.step(1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.step(1)
    dt = time.perf_counter() - t0
    cores = int(_orc.lib().orc_omp_threads())
    nz = nz0 * 2 ** int(p["lat_max_level"])
    val = nz * args.steps / dt
    sample = f"{args.steps} full oracle steps of the whole {p['n'][0]}x{p['n'][1]}x{p['n'][2]} grid per timed step"
    if shrunk:
        sample = (f"{args.steps} oracle steps of the workload on {shrunk[0]}x{shrunk[1]}x{shrunk[2]} zones (x1 zone count reduced, "
                  f"same r range) so that the run ends within minutes")
    if shrunk:   # the label names the grid that actually ran
        desc = desc.replace("256x128x128", f"{shrunk[0]}x{shrunk[1]}x{shrunk[2]} (x1 zone count reduced from 256, same r range)")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": desc},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def run_sharded(args):
    """--shard: ONE grid as x1 slabs (paper_1912_10192_b200/shard.py).  Under torchrun every rank holds
    one slab on its GPU and reads its neighbours' ghost layers over NVLink (strong scaling: the grid is fixed); on one GPU
    (--shard S) the S slabs live in this process and the line carries the cost of slab stepping against the one-grid step."""
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    torch.cuda.set_device(local)
    torch.cuda.set_stream(torch.cuda.Stream())
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import __graft_entry__ as ge
    if rank == 0:
        ge.build()
    if world > 1:
        dist.barrier()
    from paper_1912_10192_b200 import hamr, shard
    p, gen, desc = workload(args.workload)
    if any(p["nb"]) or p["lat_max_level"] > 0:
        raise SystemExit("--shard needs a one-block workload (cfg2, cfg2r, cfg3, cfg1, cfg0, paper150)")
    nz = int(np.prod(p["n"]))
    hyd, bf = gen()
    steps = args.steps or 200
    warm = max(args.warmup, 3)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(obj, k):
        for _ in range(warm):
            obj.step_async(1)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(k):
            obj.step_async(1)
        e1.record()
        barrier()
        return e0.elapsed_time(e1)

    sampler = ClockSampler(local)
    one_ms = None
    if world > 1:
        mem = "symm"
        try:
            ds = shard.DistSlab(p, peer_memory="symm")
        except Exception as e:   # no symmetric-memory support on this box: CUDA IPC handles
            mem = f"ipc (symmetric memory unavailable: {type(e).__name__})"
            ds = shard.DistSlab(p, peer_memory="ipc")
        assert ds.set_prims(hyd, bf) == 0
        sampler.start()
        l0 = ds.slab.launch_count()
        ms = timed(ds, steps)
        launches = round((ds.slab.launch_count() - l0) * steps / (steps + warm))   # the timed steps' share
        clocks = sampler.stop()
        t = torch.tensor([ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
        parts, par = ds.ranges, f"{world} x1 slabs, one per GPU, ghost layers read over NVLink ({mem}); 2 all-reduces per step"
        divb = ds.slab.divb()
        ds.close()
    else:
        nslab = max(1, args.shard)
        ring = shard.LocalRing(p, nslab)
        assert ring.set_prims(hyd, bf) == 0
        sampler.start()
        l0 = ring.launch_count()
        ms = timed(ring, steps)
        launches = round((ring.launch_count() - l0) * steps / (steps + warm))      # the timed steps' share
        one = hamr.Grid(p, torch_arena=True)
        assert one.set_prims(hyd, bf) == 0
        one_ms = timed(one, steps)
        clocks = sampler.stop()
        parts, par = ring.ranges, f"{nslab} x1 slabs on 1 GPU in one process (neighbour arenas on the same device)"
        divb = ring.divb()
        ring.close()
        one.close()
    if rank == 0:
        line = {"metric": METRIC, "value": nz * steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": steps,
                "warmup": warm, "ms_per_step": ms / steps, "higher_is_better": True, "scaling": "strong",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": desc, "zones": nz, "parallelism": par, "slabs": [list(q) for q in parts]},
                "clocks": clocks, "gpu_launches": launches, "divb": divb}
        if one_ms is not None:
            line["one_grid"] = {"ms_per_step": one_ms / steps, "value": nz * steps / (one_ms * 1e-3),
                                "slab_cost": ms / one_ms,
                                "what": "the same workload as one grid (CUDA-graph replay of the step), timed right after"}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="hamr", choices=["hamr", "reference"])
    ap.add_argument("--workload", default="cfg2")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--e2e-grids", type=int, default=3, help="grids in flight in the end-to-end measurement")
    ap.add_argument("--shard", type=int, default=0,
                    help="run ONE grid as x1 slabs (NEXT-4): under torchrun one slab per rank; on one GPU this many slabs")
    args = ap.parse_args()
    if args.shard and args.impl != "reference":
        return run_sharded(args)
    if args.impl == "reference":
        if args.steps is None:
            args.steps = 5
        args.warmup = min(args.warmup, 1) if args.warmup else 0
        return run_reference(args)
    if args.steps is None:
        # BASELINE cfg 2 runs 200 steps (0.6 s on a B200: long enough for the clock sampler to see the load)
        args.steps = 200 if args.workload in ("cfg2", "cfg2r", "cfg1", "cfg0", "paper150") else 20
    args.warmup = max(args.warmup, 3)

    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    torch.cuda.set_device(local)
    # everything below runs on one non-default stream (torch's current stream from here on): the library captures its
    # step sequence as a CUDA graph, which the legacy default stream does not allow
    torch.cuda.set_stream(torch.cuda.Stream())
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    import __graft_entry__ as ge
    if rank == 0:
        ge.build()
    if world > 1:
        dist.barrier()
    from paper_1912_10192_b200 import hamr

    p, gen, desc = workload(args.workload)
    n = tuple(p["n"])
    nz = int(np.prod(n))
    blocky = any(p["nb"]) or p["lat_max_level"] > 0
    fin = 2 ** int(p["lat_max_level"])        # finest steps per hamr_step on a LAT grid
    g = hamr.Grid(p, torch_arena=True)        # device memory and stream from torch; all math in libhamr
    refined = p["r_refine_max"] > 0
    if refined:                               # a refined grid has no global zone array: block-by-block state
        infos = [g.block_info(b)[:3] for b in range(g.num_blocks())]
        bdata = gen(infos)
        nz = sum(int(np.prod(i[2])) for i in infos)
        for b, (hb, fb) in enumerate(bdata):
            assert g.set_block_prims(b, hb, fb) == 0
        assert g.commit() == 0
    else:
        hyd, bf = gen()
        hd = [torch.from_numpy(np.ascontiguousarray(h)).cuda() for h in hyd]
        bd = [torch.from_numpy(np.ascontiguousarray(b)).cuda() for b in bf]
        assert g.set_prims_dev(hd, bd) == 0
    g.sync()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident throughput ---------------------------------------------------------------
    # three passes under one clock sampler: (1) the headline, EXACTLY --steps steps with no instrumentation; (2) the
    # same steps with a CUDA event pair around every launch, for the per-kernel shares only; (3) a sustained pass of
    # >= 0.7 s so that the sampler (100 ms period) sees the load and the power cap, reported beside the headline
    for _ in range(args.warmup):
        g.step_async(1)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    l0 = g.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(args.steps):
        g.step_async(1)
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    launches = g.launch_count() - l0
    g.profile_begin()                          # per-kernel CUDA event pairs on the launching stream
    for _ in range(args.steps):
        g.step_async(1)
    barrier()
    prof = g.profile_end()
    ms_prof = sum(v[0] for v in prof.values())
    sus_steps = max(args.steps, int(0.7e3 / max(ms / args.steps, 1e-3)) + 1)
    barrier()
    ev0.record()
    for _ in range(sus_steps):
        g.step_async(1)
    ev1.record()
    barrier()
    ms_sus = ev0.elapsed_time(ev1)
    # FP64 pipe peak, measured: all-DFMA chains and the flux kernels' DFMA / DADD / DMUL blend
    fp64 = None
    if rank == 0:
        sec0, ins0 = hamr.bench_fp64(0, 20000, torch.cuda.current_stream().cuda_stream)
        sec1, ins1 = hamr.bench_fp64(1, 20000, torch.cuda.current_stream().cuda_stream)
        sec2, ins2 = hamr.bench_fp64(2, 20000, torch.cuda.current_stream().cuda_stream)
        fp64 = {"tflops_measured_dfma": 2.0 * ins0 / sec0 / 1e12, "ginstr_per_s_dfma": ins0 / sec0 / 1e9,
                "ginstr_per_s_flux_mix": ins1 / sec1 / 1e9, "tflops_flux_mix": (4.0 / 3.0) * ins1 / sec1 / 1e12,
                # FP64-pipe instruction rate when every 4 of them come with 5 select / integer instructions, as in
                # the flux kernels (~350 : ~420 per face): what the machine sustains on THAT blend
                "ginstr_per_s_flux_blend": ins2 / sec2 / 1e9,
                "tflops_derived": FP64_PEAK_TFLOPS_DERIVED,
                "how": "hamr_bench_fp64: 8 independent chains per thread, 64 warps per SM, 96 x 20000 instructions per thread"}
    clocks = sampler.stop()
    g.sync()
    # LAT: "effective" zone-cycles (zones x finest-level steps, the paper's convention)
    value, ms_max = replica_throughput(ms, nz * fin * args.steps, world, "cuda")
    sustained, _ = replica_throughput(ms_sus, nz * fin * sus_steps, world, "cuda")
    performed = None
    if blocky:
        lv = np.array(g.levels())
        performed = world * nz * float(np.mean(fin / 2.0 ** lv)) * args.steps / (ms_max * 1e-3)

    # ---- end to end through the C-ABI with HOST buffers (pinned): set_prims + step + get_prims -----
    # Two numbers.  "serial": one grid, call after call; PCIe carries the step's input, then the GPU steps, then PCIe
    # carries the result: nothing overlaps (each call needs the one before).  The headline `value`: SEVERAL grids in flight (--e2e-grids),
    # each driven by its own host thread through the same three calls on its own stream (the library has no global
    # state; ctypes releases the GIL), so one grid's result goes down the link while the other's input comes up (PCIe is
    # full duplex) and the kernels of one run under the copies of the other.  Every step of either grid still copies
    # all of its input from pinned host memory and all of its result back inside the timed region.
    import threading
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
    C = hamr.C
    L = hamr.lib()
    ng = max(1, args.e2e_grids)
    gx = [g] + [hamr.Grid(p) for _ in range(ng - 1)]   # the other grids: own device memory, own stream
    if refined:
        # every block in one call: the per-block arrays back to back (hamr_set_all_blocks / hamr_get_all_blocks)
        hh = [pin(np.stack([hb[c] for hb, fb in bdata])) for c in range(5)]
        bh = [pin(np.stack([fb[c] for hb, fb in bdata])) for c in range(3)]
        nbk = g.num_blocks()
        oshape = (nbk,) + tuple(infos[0][2])
        set_call, get_call = L.hamr_set_all_blocks, L.hamr_get_all_blocks
    else:
        hh = [pin(h) for h in hyd]
        bh = [pin(b) for b in bf]
        oshape = n
        set_call, get_call = L.hamr_set_prims, L.hamr_get_prims
    hp = (hamr.c_double_p * 5)(*[hamr._dp(h) for h in hh])
    bp = (hamr.c_double_p * 3)(*[hamr._dp(b) for b in bh])
    outs2 = [[torch.empty(oshape, dtype=torch.float64).pin_memory().numpy() for _ in range(8)] for _ in range(ng)]
    ops = [(hamr.c_double_p * 8)(*[hamr._dp(o) for o in oo]) for oo in outs2]
    outs = outs2[0]

    # one grid at a time per direction of the link: a grid that shares the link with two others gets its input three
    # times later, while one that has the link to itself starts stepping after a third of that time and frees the link
    # for the next (the copies of concurrent calls would otherwise interleave array by array)
    link_in, link_out = threading.Lock(), threading.Lock()

    def e2e_step(gh=None, op=None):
        gh = g.h if gh is None else gh
        op = ops[0] if op is None else op
        with link_in:
            if refined:
                rc = set_call(gh, hp, bp)
            else:   # the link is released as soon as the input has left the host, not when the first flux pass is done
                rc = L.hamr_set_prims_async(gh, hp, bp)
                rc |= L.hamr_wait_input(gh)
        if refined:
            rc |= L.hamr_step(gh, 1, None, None)
        else:   # the outbound link is taken when the result is ready to leave (gathered into the staging area), not before
            rc |= L.hamr_step_async(gh, 1)
            rc |= L.hamr_stage_output(gh)
            rc |= L.hamr_sync(gh)
        with link_out:
            rc |= get_call(gh, op)
        assert rc == 0, rc

    e2e_step()
    for q in range(1, ng):
        for _ in range(2):                      # the second call captures the grid's step graph (on this thread)
            e2e_step(gx[q].h, ops[q])
    barrier()
    t0 = time.perf_counter()
    ev0.record()
    for _ in range(args.e2e_steps):
        e2e_step()
    ev1.record()
    barrier()
    e2e_ms = max(ev0.elapsed_time(ev1), 1e3 * (time.perf_counter() - t0))
    e2e_serial, _ = replica_throughput(e2e_ms, nz * fin * args.e2e_steps, world, "cuda")

    def e2e_worker(gh, op):
        torch.cuda.set_device(local)            # the current device is per host thread
        for _ in range(args.e2e_steps):
            e2e_step(gh, op)
    th = [threading.Thread(target=e2e_worker, args=(gx[q].h, ops[q])) for q in range(ng)]
    barrier()
    t0 = time.perf_counter()
    for t_ in th:
        t_.start()
    for t_ in th:
        t_.join()                               # every call above has synchronised its own stream before returning
    e2e_ms2 = 1e3 * (time.perf_counter() - t0)
    barrier()
    e2e_val, _ = replica_throughput(e2e_ms2, nz * fin * ng * args.e2e_steps, world, "cuda")
    same_result = all(np.array_equal(a, b) for q in range(1, ng) for a, b in zip(outs2[0], outs2[q]))
    for q in range(1, ng):
        gx[q].close()
    h2d = sum(a.nbytes for a in hh) + sum(a.nbytes for a in bh)
    d2h = sum(a.nbytes for a in outs)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    nb_ws = C.c_size_t(0)
    L.hamr_workspace_bytes(C.byref(g._par), C.byref(nb_ws))
    ws_gb = nb_ws.value / 1e9
    # ---- roofline -----------------------------------------------------------------------------------------------
    # per kernel class from the instrumented pass; the object leads with the class that takes the largest share of the
    # step (the three fused reconstruct + HLL kernels count as one class: same code, one per direction)
    hbm_peak, peak_src = peaks()
    kern = {k: {"ms_total": v[0], "launches": v[1], "ms_avg": v[0] / v[1] if v[1] else 0.0,
                "share": v[0] / ms_prof if ms_prof else 0.0} for k, v in prof.items() if v[1]}
    for k, d in kern.items():
        # per-launch algorithmic bytes are defined for the monolithic launch shape only
        by = 0 if blocky else alg_bytes(k, n)
        d["alg_bytes"] = by
        d["gbs"] = by / (d["ms_avg"] * 1e-3) / 1e9 if d["ms_avg"] > 0 else 0.0
    classes = {"flux": [k for k in ("flux_x1", "flux_x2", "flux_x3") if k in kern],
               "update": [k for k in ("update_predictor", "update_corrector") if k in kern],
               "ct": [k for k in ("centre_emf", "edge_emf") if k in kern], "ghosts": [k for k in ("ghosts",) if k in kern]}
    cshare = {c: sum(kern[k]["share"] for k in ks) for c, ks in classes.items() if ks}
    dom = max(cshare, key=cshare.get)
    dk = classes[dom]
    dom_bytes = sum(kern[k]["alg_bytes"] * kern[k]["launches"] for k in dk)
    dom_ms = sum(kern[k]["ms_total"] for k in dk)
    dom_gbs = dom_bytes / (dom_ms * 1e-3) / 1e9 if dom_ms else 0.0
    traffic = None
    if args.workload == "cfg2" and all(k in NCU_TRAFFIC for k in dk):
        traffic = sum(NCU_TRAFFIC[k] for k in dk)          # the class's launches of one stage, like `achieved`
    flux_alu = None
    if classes["flux"] and not blocky and fp64:
        # faces the kernels COMPUTE on cfg 2 (the x3 ghost columns and the face at k = n3 are stored periodic images)
        nface = {"flux_x1": (n[0] + 1) * (n[1] + 2) * n[2], "flux_x2": (n[0] + 2) * (n[1] + 1) * n[2],
                 "flux_x3": (n[0] + 2) * (n[1] + 2) * n[2]}
        ins = sum(FLUX_FP64_INST_PER_FACE[k] * nface[k] * kern[k]["launches"] for k in classes["flux"])
        sec = sum(kern[k]["ms_total"] for k in classes["flux"]) * 1e-3
        flux_alu = {"bound": "alu", "kernels": "+".join(classes["flux"]), "achieved": ins / sec / 1e9,
                    "peak": fp64["ginstr_per_s_flux_mix"], "unit": "G thread-instructions/s (FP64 pipe)",
                    "frac": ins / sec / 1e9 / fp64["ginstr_per_s_flux_mix"],
                    "tflops": (1.0 + FLUX_FMA_FRACTION) * ins / sec / 1e12,
                    "fp64_inst_per_face": FLUX_FP64_INST_PER_FACE, "inst_source": NCU_TRAFFIC_SOURCE,
                    "note": "executed dadd + dmul + dfma thread instructions per face (ncu) x faces / CUDA-event time, "
                            "against the MEASURED issue rate of the same instruction blend (hamr_bench_fp64 mix 1)"}
        # The bound that holds for these kernels: of their ~800 instructions per face only half go down the FP64 pipe,
        # and the others (selects, integer, shared-memory loads) take issue slots from it.  hamr_bench_fp64 mix 2 runs
        # dependency-free chains with that blend (4 FP64-pipe : 5 other) on every scheduler; the flux kernels' FP64-pipe
        # instruction rate is measured against the rate that microbenchmark sustains
        pins = sum(FLUX_FP64PIPE_INST_PER_FACE[k] * nface[k] * kern[k]["launches"] for k in classes["flux"])
        flux_alu["blend"] = {"achieved": pins / sec / 1e9, "peak": fp64["ginstr_per_s_flux_blend"],
                             "unit": "G thread-instructions/s on the FP64 pipe (arithmetic + compares)",
                             "frac": pins / sec / 1e9 / fp64["ginstr_per_s_flux_blend"],
                             "fp64pipe_inst_per_face": FLUX_FP64PIPE_INST_PER_FACE, "inst_per_face": FLUX_INST_PER_FACE,
                             "per_kernel_frac": {k: FLUX_FP64PIPE_INST_PER_FACE[k] * nface[k] * kern[k]["launches"] /
                                                 (kern[k]["ms_total"] * 1e-3) / 1e9 / fp64["ginstr_per_s_flux_blend"]
                                                 for k in classes["flux"]},
                             "note": "FP64-pipe instruction rate of the flux kernels against the rate the same blend of "
                                     "FP64-pipe and other instructions sustains without dependencies (hamr_bench_fp64 "
                                     "mix 2: 4 FP64-pipe to 5 select / integer instructions; the kernels: ~350 to ~420)"}
    roof = {"bound": "hbm", "kernel": "+".join(dk), "achieved": dom_gbs, "peak": hbm_peak, "unit": "GB/s",
            "frac": dom_gbs / hbm_peak, "traffic": traffic, "traffic_source": NCU_TRAFFIC_SOURCE, "peak_source": peak_src,
            "share_of_step": cshare[dom], "class_shares": {c: round(v, 4) for c, v in cshare.items()},
            "fp64": fp64, "flux_alu": flux_alu,
            "whole_step": {"alg_bytes_per_zone_cycle_floor": 440,
                           "frac_of_hbm_at_floor": 440.0 * value / world / 1e9 / hbm_peak,
                           "alg_bytes_per_zone_cycle_pipeline": sum(d["alg_bytes"] * d["launches"] for d in kern.values()) / (nz * fin * args.steps),
                           "frac_of_hbm_pipeline": sum(d["alg_bytes"] * d["launches"] for d in kern.values()) / args.steps / (ms / args.steps * 1e-3) / 1e9 / hbm_peak},
            "kernels": {k: {"ms_avg": round(d["ms_avg"], 4), "share": round(d["share"], 4),
                            "gbs": round(d["gbs"], 1), "frac_of_hbm": round(d["gbs"] / hbm_peak, 4),
                            "launches": d["launches"]} for k, d in kern.items()}}

    cpu = None
    if not args.no_cpu_baseline:
        subprocess.check_call(["make", "-s", "-C", os.path.join(ROOT, "oracle")])
        steps_cpu = 3 if args.workload == "cfg2" else (1 if args.workload in ("cfg4b", "cfg4", "cfg4t", "cfg4r") else 2)
        v, secs, cores = cpu_oracle_time(p, gen, steps_cpu)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{steps_cpu} full {'coarse ' if fin > 1 else ''}steps of the same workload, all {nz} zones ({secs:.1f} s)"}
        if args.workload == "cfg2":
            # the oracle on ONE core as well, on the same torus at 64 x 32 x 32 zones (one core needs
            # about a minute for a step of the full grid)
            p1, gen1, _ = workload("cfg2", n_override=(64, 32, 32))
            v1, secs1, c1 = cpu_oracle_time(p1, gen1, 3, threads=1)
            cpu["single_thread"] = {"value": v1, "unit": UNIT, "cores": c1,
                                    "sample": f"3 steps of the same torus on 64x32x32 zones ({secs1:.1f} s)"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": (value / PAPER_V100_150CUBED if args.workload == "paper150" else None),
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": desc, "zones": nz, "blocks": g.num_blocks(), "finest_steps_per_step": fin,
                       "performed_zone_updates_per_sec": performed,
                       "parallelism": "replicas only" if world > 1 else "1 GPU",
                       "l2": f"state arrays ({ws_gb:.1f} GB workspace) far larger than the 126 MB L2; no flush needed",
                       "timing": "CUDA events on the launching (torch current) stream; the headline pass carries no "
                                 "per-kernel instrumentation (the kernel table comes from a second pass of the same steps)"},
            "clocks": clocks,
            "sustained": {"value": sustained, "unit": UNIT, "steps": sus_steps, "ms_per_step": ms_sus / sus_steps,
                          "what": "the same step repeated for >= 0.7 s right after the headline pass (power-capped clocks)"},
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": ng * args.e2e_steps, "grids_in_flight": ng, "results_identical": bool(same_result),
                    "what": ("hamr_set_all_blocks + hamr_step(1) + hamr_get_all_blocks" if refined else
                             "hamr_set_prims(host) + hamr_step(1) + hamr_get_prims(host)") + ", pinned buffers; several "
                            "grids in flight, one host thread and stream each (one grid's D2H overlaps another's H2D "
                            "and kernels); wall clock over all steps of all grids",
                    "serial": {"value": e2e_serial, "unit": UNIT, "steps": args.e2e_steps,
                               "what": "the same three calls on one grid, one after the other (nothing overlaps)"}},
            "gpu_launches": launches,
            "roofline": roof, "cpu_baseline": cpu}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
