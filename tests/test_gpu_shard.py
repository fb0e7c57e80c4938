"""NEXT-4 (include/hamr.h "x1 slabs over peer memory"): a grid cut into x1 slabs whose ghost fill reads the
neighbour slabs through device pointers.  On one GPU all slabs live in this process (shard.LocalRing: the kernels and
the neighbour reads of the multi-GPU job, the neighbour's arena being a pointer on the same device).

What is checked: (1) the slabs reproduce the ONE-grid result of the same library bit for bit — same geometry tables,
same per-face and per-zone arithmetic, interface faces advanced identically on both sides — for 2 and 3 slabs, ragged
thicknesses, an outflow x1 (Kerr torus) and a periodic x1 that closes the ring (Minkowski waves), also with the robust
inversion options and with phi-derefined polar rows; (2) parity of the slabs with the ORACLE at north_star's tolerances (the oracle knows nothing of
slabs: it steps the whole grid); (3) div B, also across the interfaces; (4) the call-order and argument checks of the
boundary; (5) cfg 2 at full size in two slabs, every zone, against the one-grid run."""
import ctypes as C

import numpy as np
import pytest

from paper_1912_10192_b200 import inputs as I
from tests._parity import parity_errors, rel_max

pytestmark = pytest.mark.gpu

TOL_1, TOL_10, TOL_DIVB = 1e-10, 1e-7, 1e-12


@pytest.fixture(scope="module")
def H():
    from paper_1912_10192_b200 import build, hamr
    build.build_lib()
    hamr.lib()
    return hamr


@pytest.fixture(scope="module")
def S(H):
    from paper_1912_10192_b200 import shard
    return shard


def _cases():
    c = {}
    p = I.torus_params()                                        # BASELINE cfg 0: outflow x1
    c["cfg0_torus_2"] = (p, lambda: I.fm_torus(p, seed=0), 2)
    c["cfg0_torus_3"] = (p, lambda: I.fm_torus(p, seed=0), [(0, 11), (11, 4), (15, 17)])   # ragged, one thin slab
    q = I.minkowski_params(n=(40, 24, 36))                      # periodic x1: the ring closes; generic kernels
    c["minkowski_ring_3"] = (q, lambda: I.minkowski_waves(q, seed=1, amp=1e-2, noise=1e-3), 3)
    s = I.minkowski_params(n=(32, 32, 32))                      # staged kernels (x3 a multiple of 32), two slabs: each
    c["cfg1_waves_2"] = (s, lambda: I.minkowski_waves(s, seed=1), 2)   # is the other's neighbour on BOTH sides
    r = I.torus_params(n=(24, 16, 8), recon=I.RECON_PLM)
    c["torus_plm_2"] = (r, lambda: I.fm_torus(r, seed=5), 2)
    e = dict(I.torus_params(n=(32, 16, 32)), entropy_backup=1, drift_floors=1)
    c["torus_robust_2"] = (e, lambda: I.fm_torus(e, seed=6), 2)
    d = I.torus_params(n=(32, 16, 16), deref_theta_deg=(30.0, 12.0), deref_factor=(2, 4))   # phi-derefined polar rows
    c["torus_deref_2"] = (d, lambda: I.fm_torus(d, seed=7), 2)
    return c


CASES = _cases()


def _same(a, b):
    return all(np.array_equal(x, y) for x, y in zip(a, b))


@pytest.mark.parametrize("name", list(CASES))
def test_slabs_reproduce_the_one_grid_result_bit_for_bit_and_match_the_oracle(H, S, orc, name):
    p, gen, parts = CASES[name]
    hyd, bf = gen()
    one = H.Grid(p, torch_arena=True)
    ring = S.LocalRing(p, parts)
    o = orc.OrcGrid(p)
    assert one.set_prims(hyd, bf) == 0 and ring.set_prims(hyd, bf) == 0 and o.set_prims(hyd, bf) == 0
    assert ring.dt == one.dt                                     # max over the slabs' Courant maxima (C-14)
    assert abs(ring.dt - o.dt) <= 1e-13 * o.dt
    one.step(1)
    ring.step(1)
    o.step(1)
    assert ring.t == one.t and ring.dt == one.dt
    P1, R1 = one.get_prims(), ring.get_prims()
    assert _same(P1, R1), [float(np.abs(a - b).max()) for a, b in zip(P1, R1)]
    assert _same(one.get_bface(), ring.get_bface())
    # the face two slabs share: both copies equal
    for a, b in zip(ring.slabs[:-1], ring.slabs[1:]):
        assert np.array_equal(a.get_bface()[0][-1], b.get_bface()[0][0])
    e1 = parity_errors(p, o.get_prims(), R1)
    assert max(e1.values()) <= TOL_1, (name, e1)
    for a, b in zip(o.get_bface(), ring.get_bface()):
        assert rel_max(a, b) <= TOL_1
    one.step(9)
    ring.step(9)
    o.step(9)
    assert ring.t == one.t
    assert _same(one.get_prims(), ring.get_prims()) and _same(one.get_bface(), ring.get_bface())
    e10 = parity_errors(p, o.get_prims(), ring.get_prims())
    assert max(e10.values()) <= TOL_10, (name, e10)
    assert ring.divb() <= TOL_DIVB
    assert ring.stats() == one.stats()
    # div B of the assembled field, interface zones included, with the no-grid diagnostic on the global arrays
    B = ring.get_bface()
    n, d = p["n"], [(p["xmax"][c] - p["xmin"][c]) / p["n"][c] for c in range(3)]
    if p["metric"] == I.METRIC_KS:
        d[0] = (np.log(p["xmax"][0]) - np.log(p["xmin"][0])) / n[0]
    div = sum(np.diff(B[c], axis=c) / d[c] for c in range(3))
    den = sum((np.abs(np.take(B[c], range(1, n[c] + 1), axis=c)) + np.abs(np.take(B[c], range(0, n[c]), axis=c))) / (2 * d[c])
              for c in range(3))
    if den.max() > 0:
        ok = den > 1e-12 * den.max()
        assert float(np.max(np.abs(div[ok]) / den[ok])) <= TOL_DIVB
    one.close()
    ring.close()


def test_one_slab_covering_the_grid_needs_no_neighbour_and_equals_the_grid(H, S):
    p = I.minkowski_params(n=(32, 32, 32))
    hyd, bf = I.minkowski_waves(p, seed=2)
    one = H.Grid(p, torch_arena=True)
    ring = S.LocalRing(p, 1)
    assert one.set_prims(hyd, bf) == 0 and ring.set_prims(hyd, bf) == 0
    one.step(3)
    ring.step(3)
    assert _same(one.get_prims(), ring.get_prims())
    one.close()
    ring.close()


def test_call_order_and_arguments_are_checked(H, S):
    L = H.lib()
    p = I.torus_params()
    par = H.pack_params(p)
    n = C.c_size_t(0)
    assert L.hamr_shard_workspace_bytes(C.byref(par), 0, 16, C.byref(n)) == H.OK and n.value > 0
    for lo, n1 in ((0, 2), (-1, 8), (20, 16), (0, 0)):                    # thinner than 3 zones / outside the grid
        assert L.hamr_shard_workspace_bytes(C.byref(par), lo, n1, C.byref(n)) == H.EINVAL, (lo, n1)
    blk = H.pack_params(dict(p, nb=(8, 8, 8)))
    assert L.hamr_shard_workspace_bytes(C.byref(blk), 0, 16, C.byref(n)) == H.EINVAL   # one-block grids only
    a, b = S.Slab(p, 0, 16), S.Slab(p, 16, 16)
    hyd, bf = I.fm_torus(p, seed=0)
    assert a.set_prims([a.local(h) for h in hyd], [a.local(x, d) for d, x in enumerate(bf)]) == 0
    assert L.hamr_shard_commit(a.h) == H.ESTATE                           # the high side has no neighbour yet
    assert L.hamr_shard_stage(a.h, 0) == H.ESTATE                         # not committed
    assert L.hamr_step(a.h, 1, None, None) == H.ESTATE                    # a slab does not step alone
    assert L.hamr_shard_attach(a.h, 1, C.c_void_p(b.arena_ptr), 12, 16) == H.EINVAL    # does not adjoin
    assert L.hamr_shard_attach(a.h, 0, C.c_void_p(b.arena_ptr), 16, 16) == H.EINVAL    # physical boundary side
    assert L.hamr_shard_attach(a.h, 1, C.c_void_p(b.arena_ptr + 8), 16, 16) == H.EINVAL  # misaligned
    assert L.hamr_shard_attach(a.h, 1, C.c_void_p(b.arena_ptr), 16, 16) == H.OK
    assert L.hamr_shard_attach(b.h, 0, C.c_void_p(a.arena_ptr), 0, 16) == H.OK
    assert b.set_prims([b.local(h) for h in hyd], [b.local(x, d) for d, x in enumerate(bf)]) == 0
    assert L.hamr_shard_commit(a.h) == H.OK and L.hamr_shard_commit(b.h) == H.OK
    assert L.hamr_shard_stage(a.h, 0) == H.ESTATE                         # the first dt has not been set
    assert L.hamr_shard_stage(a.h, 1) == H.ESTATE
    assert L.hamr_shard_stage(None, 0) == H.EINVAL and L.hamr_shard_stage(a.h, 2) == H.EINVAL
    g = H.Grid(p)
    assert L.hamr_shard_stage(g.h, 0) == H.EINVAL and L.hamr_shard_commit(g.h) == H.EINVAL   # not a slab
    g.close()
    a.close()
    b.close()


def test_headline_config_in_two_slabs_equals_the_one_grid_run_at_full_size(H, S):
    """BASELINE cfg 2 (256x128x128 Kerr torus), 2 slabs of 128: every zone after 1 and 3 steps."""
    p = I.torus_params(n=(256, 128, 128), r_out=1000.0)
    hyd, bf = I.fm_torus(p, seed=2)
    one = H.Grid(p, torch_arena=True)
    ring = S.LocalRing(p, 2)
    assert one.set_prims(hyd, bf) == 0 and ring.set_prims(hyd, bf) == 0
    for n in (1, 2):
        one.step(n)
        ring.step(n)
        assert ring.t == one.t and ring.dt == one.dt
        assert _same(one.get_prims(), ring.get_prims())
        assert _same(one.get_bface(), ring.get_bface())
    assert ring.divb() <= TOL_DIVB and ring.stats() == one.stats()
    one.close()
    ring.close()


def _rank_main(rank, world, port, out_dir, p, seed, nsteps):
    """one process of a 2-process job on ONE GPU: gloo for the reductions (through host memory), CUDA IPC for the
    neighbour arenas — the multi-process plumbing of shard.DistSlab with the kernels of the job; no kernel of one process
    waits on the other's (every ordering point is a host-side reduction after a stream synchronisation)"""
    import os
    import sys
    import torch
    import torch.distributed as dist
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    from paper_1912_10192_b200 import shard
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    hyd, bf = I.fm_torus(p, seed=seed)
    ds = shard.DistSlab(p, peer_memory="ipc")
    assert ds.set_prims(hyd, bf) == 0
    ds.step(nsteps)
    P, B = ds.slab.get_prims(), ds.slab.get_bface()
    np.savez(os.path.join(out_dir, f"rank{rank}.npz"), t=ds.slab.t, dt=ds.slab.dt, i_lo=ds.slab.i_lo,
             **{f"P{c}": P[c] for c in range(8)}, **{f"B{d}": B[d] for d in range(3)})
    ds.close()
    dist.destroy_process_group()


def test_two_processes_with_ipc_neighbour_arenas_reproduce_the_one_grid_run(H, S, tmp_path):
    import socket
    import torch.multiprocessing as mp
    p = I.torus_params()
    nsteps = 5
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, str(tmp_path), p, 0, nsteps)) for r in range(2)]
    for q in procs:
        q.start()
    for q in procs:
        q.join(timeout=300)
    hung = [q for q in procs if q.is_alive()]
    for q in hung:
        q.kill()
    assert not hung and all(q.exitcode == 0 for q in procs), [q.exitcode for q in procs]
    hyd, bf = I.fm_torus(p, seed=0)
    one = H.Grid(p, torch_arena=True)
    assert one.set_prims(hyd, bf) == 0
    one.step(nsteps)
    P, B = one.get_prims(), one.get_bface()
    for r in range(2):
        z = np.load(tmp_path / f"rank{r}.npz")
        lo = int(z["i_lo"])
        n1 = z["P0"].shape[0]
        assert float(z["t"]) == one.t and float(z["dt"]) == one.dt
        for c in range(8):
            assert np.array_equal(z[f"P{c}"], P[c][lo:lo + n1]), (r, c)
        assert np.array_equal(z["B0"], B[0][lo:lo + n1 + 1])
        for d in (1, 2):
            assert np.array_equal(z[f"B{d}"], B[d][lo:lo + n1])
    one.close()


def test_bench_shard_line():
    """`bench.py --shard 2` (the slab arm of the bench) prints one JSON line with the slab and the one-grid step"""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--shard", "2", "--workload", "cfg0", "--steps", "5"],
                       capture_output=True, text=True, timeout=600, cwd=root)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().split("\n")[-1])
    assert line["metric"] == "zone_cycles_per_sec" and line["scaling"] == "strong" and line["value"] > 0
    assert line["config"]["slabs"] == [[0, 16], [16, 16]] and line["gpu_launches"] > 0
    assert line["divb"] <= TOL_DIVB and line["one_grid"]["ms_per_step"] > 0


def _nccl_one_rank(port, out_path, mem):
    import os
    import sys
    import torch
    import torch.distributed as dist
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    from paper_1912_10192_b200 import hamr, shard
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(0)
    torch.cuda.set_stream(torch.cuda.Stream())
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    p = I.torus_params()
    hyd, bf = I.fm_torus(p, seed=0)
    one = hamr.Grid(p, torch_arena=True)
    assert one.set_prims(hyd, bf) == 0
    one.step(5)
    ds = shard.DistSlab(p, peer_memory=mem)
    assert ds.red.on_stream and ds.ranges == [(0, 32)]
    assert ds.set_prims(hyd, bf) == 0
    ds.step(5)
    same = all(np.array_equal(a, b) for a, b in zip(one.get_prims(), ds.slab.get_prims())) and ds.slab.t == one.t
    ds.close()
    dist.destroy_process_group()
    with open(out_path, "w") as f:
        f.write("same" if same else "different")


@pytest.mark.parametrize("mem", ["symm", "ipc"])
def test_dist_slab_on_a_one_rank_nccl_group(tmp_path, mem):
    """the torch.distributed plumbing of shard.DistSlab with the NCCL backend (all-reduces enqueued on the grid's stream)
    and both ways of mapping arenas (torch symmetric memory; CUDA IPC handles), on the one GPU there is: a group of ONE
    rank, whose slab covers the grid; the run equals the one-grid run bit for bit"""
    import socket
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    out = tmp_path / "r.txt"
    ctx = mp.get_context("spawn")
    q = ctx.Process(target=_nccl_one_rank, args=(port, str(out), mem))
    q.start()
    q.join(timeout=300)
    if q.is_alive():
        q.kill()
        raise AssertionError("the rank did not finish")
    assert q.exitcode == 0 and out.read_text() == "same"
