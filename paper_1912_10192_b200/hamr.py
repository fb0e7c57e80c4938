"""Thin ctypes binding of libhamr.so (include/hamr.h, include/hamr_debug.h).  Argument marshalling only: every step of the
hot path runs in the CUDA kernels behind the C-ABI.  There is no CPU fallback: if the library is
missing or fails to load, importing the binding's entry points raises.

Names mirror the C calls: hamr_grid_create -> Grid(...), hamr_set_prims -> Grid.set_prims,
hamr_step -> Grid.step, hamr_get_prims -> Grid.get_prims, hamr_divb -> Grid.divb, ...
PyTorch is used only for device memory and streams (Grid(..., torch_arena=True) places every
device array of the grid inside one torch CUDA tensor and issues all work on torch's current stream).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhamr.so")
_LIB = None

c_double_p = C.POINTER(C.c_double)

OK, EINVAL, ENOMEM, ECUDA, ESTATE, ENONFINITE = range(6)
_STATUS = {0: "HAMR_OK", 1: "HAMR_EINVAL", 2: "HAMR_ENOMEM", 3: "HAMR_ECUDA", 4: "HAMR_ESTATE",
           5: "HAMR_ENONFINITE"}

# every symbol include/hamr.h declares (checked by tests/test_abi.py against the header text)
SYMBOLS = ["hamr_grid_create", "hamr_workspace_bytes", "hamr_grid_create_in", "hamr_grid_destroy",
           "hamr_set_prims", "hamr_set_prims_dev", "hamr_set_prims_async", "hamr_wait_input", "hamr_stage_output", "hamr_step", "hamr_step_async", "hamr_sync",
           "hamr_get_prims", "hamr_get_prims_dev", "hamr_get_bface", "hamr_divb", "hamr_get_stats",
           "hamr_get_backup_count", "hamr_get_time", "hamr_set_dt", "hamr_last_error", "hamr_num_blocks", "hamr_block_info",
           "hamr_set_block_prims", "hamr_blocks_commit", "hamr_get_block_prims",
           "hamr_get_block_bface", "hamr_set_all_blocks", "hamr_get_all_blocks",
           "hamr_refine_radius", "hamr_regrid",
           "hamr_shard_workspace_bytes", "hamr_shard_create_in", "hamr_shard_attach", "hamr_shard_commit",
           "hamr_shard_stage", "hamr_shard_ctop_get_dev", "hamr_shard_ctop_set_dev",
           "hamr_noalloc_setup", "hamr_divb_noalloc", "hamr_noalloc_last_error"]
NOALLOC_MAX_ZONES = 16777216
# ... and include/hamr_debug.h (test hooks and diagnostics)
DEBUG_SYMBOLS = ["hamr_set_levels", "hamr_debug_emf", "hamr_get_face", "hamr_get_edge", "hamr_get_ctop", "hamr_totals",
                 "hamr_profile_begin", "hamr_profile_end", "hamr_profile_class_name", "hamr_launch_count",
                 "hamr_debug_geometry", "hamr_debug_prim2cons", "hamr_debug_con2prim", "hamr_debug_floors",
                 "hamr_debug_kappa", "hamr_debug_con2prim_entropy", "hamr_debug_floors_drift", "hamr_debug_con2prim_aitken",
                 "hamr_debug_aitken_count", "hamr_bench_fp64"]
NKCLASS = 10


class HamrError(RuntimeError):
    def __init__(self, code, msg=""):
        self.code = code
        super().__init__(f"{_STATUS.get(code, code)}: {msg}")


class Params(C.Structure):
    """hamr_params of include/hamr.h"""
    _fields_ = [("metric", C.c_int), ("recon", C.c_int), ("n", C.c_int * 3),
                ("bc_lo", C.c_int * 3), ("bc_hi", C.c_int * 3), ("nb", C.c_int * 3),
                ("n_deref", C.c_int), ("deref_factor", C.c_int * 4),
                ("lat_max_level", C.c_int), ("map", C.c_int),
                ("entropy_backup", C.c_int), ("drift_floors", C.c_int),
                ("a", C.c_double), ("xmin", C.c_double * 3), ("xmax", C.c_double * 3),
                ("gamma_ad", C.c_double), ("cour", C.c_double),
                ("rho_fl_coef", C.c_double), ("rho_fl_pow", C.c_double),
                ("u_fl_coef", C.c_double), ("u_fl_pow", C.c_double), ("gamma_max", C.c_double),
                ("deref_theta_deg", C.c_double * 4), ("r_refine_max", C.c_double)]


def lib():
    """Loads libhamr.so; raises if it has not been built (python -m paper_1912_10192_b200.build)."""
    global _LIB
    if _LIB is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python paper_1912_10192_b200/build.py` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp = C.c_void_p
        L.hamr_grid_create.argtypes = [C.POINTER(Params), C.POINTER(vp)]
        L.hamr_workspace_bytes.argtypes = [C.POINTER(Params), C.POINTER(C.c_size_t)]
        L.hamr_grid_create_in.argtypes = [C.POINTER(Params), vp, C.c_size_t, vp, C.POINTER(vp)]
        L.hamr_grid_destroy.argtypes = [vp]
        L.hamr_set_prims.argtypes = [vp, C.POINTER(c_double_p), C.POINTER(c_double_p)]
        L.hamr_set_prims_dev.argtypes = [vp, C.POINTER(c_double_p), C.POINTER(c_double_p)]
        L.hamr_set_prims_async.argtypes = [vp, C.POINTER(c_double_p), C.POINTER(c_double_p)]
        L.hamr_wait_input.argtypes = [vp]
        L.hamr_stage_output.argtypes = [vp]
        L.hamr_step.argtypes = [vp, C.c_int, c_double_p, c_double_p]
        L.hamr_step_async.argtypes = [vp, C.c_int]
        L.hamr_sync.argtypes = [vp]
        L.hamr_get_prims.argtypes = [vp, C.POINTER(c_double_p)]
        L.hamr_get_prims_dev.argtypes = [vp, C.POINTER(c_double_p)]
        L.hamr_get_bface.argtypes = [vp, C.POINTER(c_double_p)]
        L.hamr_divb.argtypes = [vp, c_double_p]
        L.hamr_get_stats.argtypes = [vp, C.POINTER(C.c_longlong)]
        L.hamr_get_backup_count.argtypes = [vp, C.POINTER(C.c_longlong)]
        L.hamr_get_time.argtypes = [vp, c_double_p, c_double_p]
        L.hamr_set_dt.argtypes = [vp, C.c_double]
        L.hamr_last_error.argtypes = [vp]
        L.hamr_last_error.restype = C.c_char_p
        L.hamr_num_blocks.argtypes = [vp]
        L.hamr_block_info.argtypes = [vp, C.c_int, c_double_p, c_double_p, C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.hamr_set_levels.argtypes = [vp, C.POINTER(C.c_int)]
        L.hamr_set_block_prims.argtypes = [vp, C.c_int, C.POINTER(c_double_p), C.POINTER(c_double_p)]
        L.hamr_blocks_commit.argtypes = [vp]
        L.hamr_set_all_blocks.argtypes = [vp, C.POINTER(c_double_p), C.POINTER(c_double_p)]
        L.hamr_get_all_blocks.argtypes = [vp, C.POINTER(c_double_p)]
        L.hamr_get_block_prims.argtypes = [vp, C.c_int, C.POINTER(c_double_p)]
        L.hamr_get_block_bface.argtypes = [vp, C.c_int, C.POINTER(c_double_p)]
        L.hamr_debug_emf.argtypes = [vp]
        L.hamr_get_face.argtypes = [vp, C.c_int, C.c_int, c_double_p]
        L.hamr_get_edge.argtypes = [vp, C.c_int, c_double_p]
        L.hamr_get_ctop.argtypes = [vp, c_double_p]
        L.hamr_totals.argtypes = [vp, c_double_p]
        L.hamr_launch_count.argtypes = [vp, C.POINTER(C.c_longlong)]
        L.hamr_profile_begin.argtypes = [vp]
        L.hamr_profile_end.argtypes = [vp, C.c_int, c_double_p, C.POINTER(C.c_longlong)]
        L.hamr_profile_class_name.argtypes = [C.c_int]
        L.hamr_profile_class_name.restype = C.c_char_p
        ip = C.POINTER(C.c_int)
        L.hamr_debug_geometry.argtypes = [vp, C.c_int, C.c_int, c_double_p, ip, ip, ip]
        L.hamr_debug_prim2cons.argtypes = [vp, C.c_int, ip, ip, c_double_p, c_double_p]
        L.hamr_debug_con2prim.argtypes = [vp, C.c_int, ip, ip, c_double_p, c_double_p, c_double_p, c_double_p, ip]
        L.hamr_debug_floors.argtypes = [vp, C.c_int, ip, ip, c_double_p, ip]
        L.hamr_debug_kappa.argtypes = [vp, c_double_p]
        L.hamr_debug_con2prim_entropy.argtypes = [vp, C.c_int, ip, ip, c_double_p, c_double_p, c_double_p, c_double_p,
                                                  c_double_p, ip]
        L.hamr_debug_con2prim_aitken.argtypes = [vp, C.c_int, ip, ip, c_double_p, c_double_p, c_double_p, c_double_p, ip]
        L.hamr_debug_aitken_count.argtypes = [vp, C.POINTER(C.c_longlong)]
        L.hamr_debug_floors_drift.argtypes = [vp, C.c_int, ip, ip, c_double_p, c_double_p, ip]
        L.hamr_bench_fp64.argtypes = [vp, C.c_int, C.c_int, c_double_p, c_double_p]
        L.hamr_refine_radius.argtypes = [vp, C.c_double, c_double_p]
        L.hamr_regrid.argtypes = [vp, C.c_double, C.POINTER(vp)]
        L.hamr_shard_workspace_bytes.argtypes = [C.POINTER(Params), C.c_int, C.c_int, C.POINTER(C.c_size_t)]
        L.hamr_shard_create_in.argtypes = [C.POINTER(Params), C.c_int, C.c_int, vp, C.c_size_t, vp, C.POINTER(vp)]
        L.hamr_shard_attach.argtypes = [vp, C.c_int, vp, C.c_int, C.c_int]
        L.hamr_shard_commit.argtypes = [vp]
        L.hamr_shard_stage.argtypes = [vp, C.c_int]
        L.hamr_shard_ctop_get_dev.argtypes = [vp, vp]
        L.hamr_shard_ctop_set_dev.argtypes = [vp, vp]
        L.hamr_noalloc_setup.argtypes = []
        L.hamr_divb_noalloc.argtypes = [C.POINTER(C.c_int), c_double_p, C.POINTER(vp), vp, vp]
        L.hamr_noalloc_last_error.argtypes = []
        L.hamr_noalloc_last_error.restype = C.c_char_p
        for s in SYMBOLS + DEBUG_SYMBOLS:
            if s not in ("hamr_last_error", "hamr_profile_class_name", "hamr_noalloc_last_error"):
                getattr(L, s).restype = C.c_int
        _LIB = L
    return _LIB


def pack_params(p: dict) -> Params:
    q = Params()
    q.metric, q.recon = int(p["metric"]), int(p["recon"])
    for d in range(3):
        q.n[d] = int(p["n"][d])
        q.bc_lo[d], q.bc_hi[d] = int(p["bc_lo"][d]), int(p["bc_hi"][d])
        q.nb[d] = int(p["nb"][d])
        q.xmin[d], q.xmax[d] = float(p["xmin"][d]), float(p["xmax"][d])
    q.n_deref = len(p["deref_factor"])
    for i, (t, f) in enumerate(zip(p["deref_theta_deg"], p["deref_factor"])):
        q.deref_theta_deg[i], q.deref_factor[i] = float(t), int(f)
    q.lat_max_level = int(p["lat_max_level"])
    q.map = int(p.get("map", 0))
    q.entropy_backup = int(p.get("entropy_backup", 0))
    q.drift_floors = int(p.get("drift_floors", 0))
    q.a = float(p["a"])
    q.gamma_ad, q.cour = float(p["gamma_ad"]), float(p["cour"])
    q.rho_fl_coef, q.rho_fl_pow = float(p["rho_fl_coef"]), float(p["rho_fl_pow"])
    q.u_fl_coef, q.u_fl_pow = float(p["u_fl_coef"]), float(p["u_fl_pow"])
    q.gamma_max = float(p["gamma_max"])
    q.r_refine_max = float(p["r_refine_max"])
    return q


def _dp(a):
    return a.ctypes.data_as(c_double_p)


def _arr(x):
    return np.ascontiguousarray(np.asarray(x, dtype=np.float64))


class Grid:
    """hamr_grid handle.  p: parameter dict as produced by paper_1912_10192_b200.inputs.*_params."""

    def __init__(self, p: dict, torch_arena: bool = False, _handle=None):
        self.L = lib()
        self.p = p
        self.n = tuple(int(v) for v in p["n"])
        self._par = pack_params(p)
        self._arena = None
        h = C.c_void_p(None)
        if _handle is not None:          # a grid the library created itself (hamr_regrid)
            self.h = _handle
            return
        if torch_arena:
            import torch
            nbytes = C.c_size_t(0)
            rc = self.L.hamr_workspace_bytes(C.byref(self._par), C.byref(nbytes))
            if rc != OK:
                raise HamrError(rc, "hamr_workspace_bytes")
            self._arena = torch.empty(nbytes.value + 256, dtype=torch.uint8, device="cuda")
            ptr = (self._arena.data_ptr() + 255) // 256 * 256
            stream = torch.cuda.current_stream().cuda_stream
            rc = self.L.hamr_grid_create_in(C.byref(self._par), C.c_void_p(ptr), C.c_size_t(nbytes.value),
                                            C.c_void_p(stream), C.byref(h))
        else:
            rc = self.L.hamr_grid_create(C.byref(self._par), C.byref(h))
        if rc != OK or not h.value:
            raise HamrError(rc, "hamr_grid_create")
        self.h = h

    # -- life cycle ---------------------------------------------------------------------------------
    def close(self):
        if getattr(self, "h", None):
            self.L.hamr_grid_destroy(self.h)
            self.h = None
            self._arena = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ck(self, rc):
        if rc != OK:
            raise HamrError(rc, (self.L.hamr_last_error(self.h) or b"").decode())

    def _fshape(self, d):
        s = list(self.n)
        s[d] += 1
        return tuple(s)

    # -- state in -----------------------------------------------------------------------------------
    def set_prims(self, hydro, bface=None):
        hy = [_arr(h) for h in hydro]
        assert len(hy) == 5 and all(h.shape == self.n for h in hy)
        hp = (c_double_p * 5)(*[_dp(h) for h in hy])
        if bface is None:
            rc = self.L.hamr_set_prims(self.h, hp, None)
        else:
            bf = [_arr(b) for b in bface]
            assert all(bf[d].shape == self._fshape(d) for d in range(3))
            bp = (c_double_p * 3)(*[_dp(b) for b in bf])
            rc = self.L.hamr_set_prims(self.h, hp, bp)
        return rc

    def set_prims_async(self, hydro, bface=None):
        """hamr_set_prims_async: hydro / bface are C-contiguous float64 numpy arrays in PINNED memory that the caller
        keeps alive and unchanged until wait_input() (or a later sync) has returned"""
        hp = (c_double_p * 5)(*[_dp(h) for h in hydro])
        bp = None if bface is None else (c_double_p * 3)(*[_dp(b) for b in bface])
        return self.L.hamr_set_prims_async(self.h, hp, bp)

    def stage_output(self):
        """hamr_stage_output: the next get_prims() is its eight copies only"""
        self._ck(self.L.hamr_stage_output(self.h))

    def wait_input(self):
        self._ck(self.L.hamr_wait_input(self.h))

    def set_prims_dev(self, hydro, bface=None):
        """hydro / bface: torch CUDA float64 contiguous tensors (device pointers are passed through)."""
        hp = (c_double_p * 5)(*[C.cast(C.c_void_p(t.data_ptr()), c_double_p) for t in hydro])
        bp = None
        if bface is not None:
            bp = (c_double_p * 3)(*[C.cast(C.c_void_p(t.data_ptr()), c_double_p) for t in bface])
        return self.L.hamr_set_prims_dev(self.h, hp, bp)

    # -- the hot path -------------------------------------------------------------------------------
    def step(self, nsteps=1):
        t, dt = C.c_double(0), C.c_double(0)
        self._ck(self.L.hamr_step(self.h, C.c_int(nsteps), C.byref(t), C.byref(dt)))
        return t.value, dt.value

    def step_async(self, nsteps=1):
        self._ck(self.L.hamr_step_async(self.h, C.c_int(nsteps)))

    def sync(self):
        self._ck(self.L.hamr_sync(self.h))

    # -- state out ----------------------------------------------------------------------------------
    def get_prims(self):
        out = [np.empty(self.n) for _ in range(8)]
        self._ck(self.L.hamr_get_prims(self.h, (c_double_p * 8)(*[_dp(o) for o in out])))
        return out

    def get_prims_dev(self, out):
        pp = (c_double_p * 8)(*[C.cast(C.c_void_p(t.data_ptr()), c_double_p) for t in out])
        self._ck(self.L.hamr_get_prims_dev(self.h, pp))

    def get_bface(self):
        out = [np.empty(self._fshape(d)) for d in range(3)]
        self._ck(self.L.hamr_get_bface(self.h, (c_double_p * 3)(*[_dp(o) for o in out])))
        return out

    def divb(self):
        v = C.c_double(0)
        self._ck(self.L.hamr_divb(self.h, C.byref(v)))
        return v.value

    def stats(self):
        c = (C.c_longlong * 4)()
        self._ck(self.L.hamr_get_stats(self.h, c))
        return tuple(c[:])

    def refine_radius(self, rho_cut):
        """hamr_refine_radius: the r_refine_max the density criterion asks for (0: no refined region)"""
        r = C.c_double(0)
        self._ck(self.L.hamr_refine_radius(self.h, float(rho_cut), C.byref(r)))
        return r.value

    def regrid(self, r_refine_max):
        """hamr_regrid: a new Grid with that r_refine_max carrying this grid's state (this grid stays valid)"""
        h = C.c_void_p(None)
        self._ck(self.L.hamr_regrid(self.h, float(r_refine_max), C.byref(h)))
        return Grid(dict(self.p, r_refine_max=float(r_refine_max)), _handle=h)

    def backup_count(self):
        """zones, since the last call, inverted from the entropy row (entropy_backup grids)"""
        n = C.c_longlong(0)
        self._ck(self.L.hamr_get_backup_count(self.h, C.byref(n)))
        return n.value

    @property
    def t(self):
        t = C.c_double(0)
        self._ck(self.L.hamr_get_time(self.h, C.byref(t), None))
        return t.value

    @property
    def dt(self):
        dt = C.c_double(0)
        self._ck(self.L.hamr_get_time(self.h, None, C.byref(dt)))
        return dt.value

    @dt.setter
    def dt(self, v):
        self._ck(self.L.hamr_set_dt(self.h, C.c_double(v)))

    def num_blocks(self):
        return self.L.hamr_num_blocks(self.h)

    def set_block_prims(self, b, hydro, bface=None):
        hy = [_arr(h) for h in hydro]
        hp = (c_double_p * 5)(*[_dp(h) for h in hy])
        bp = None
        if bface is not None:
            bf = [_arr(x) for x in bface]
            bp = (c_double_p * 3)(*[_dp(x) for x in bf])
        return self.L.hamr_set_block_prims(self.h, int(b), hp, bp)

    def set_all_blocks(self, hydro, bface=None):
        """hydro[c] / bface[d]: arrays of shape (nblk, ...) holding every block's dense array"""
        hy = [_arr(h) for h in hydro]
        hp = (c_double_p * 5)(*[_dp(h) for h in hy])
        bp = None
        if bface is not None:
            bf = [_arr(x) for x in bface]
            bp = (c_double_p * 3)(*[_dp(x) for x in bf])
        return self.L.hamr_set_all_blocks(self.h, hp, bp)

    def get_all_blocks(self):
        n = self.block_info(0)[2]
        out = [np.empty((self.num_blocks(),) + tuple(n)) for _ in range(8)]
        self._ck(self.L.hamr_get_all_blocks(self.h, (c_double_p * 8)(*[_dp(o) for o in out])))
        return out

    def commit(self):
        return self.L.hamr_blocks_commit(self.h)

    def get_block_prims(self, b):
        n = self.block_info(b)[2]
        out = [np.empty(n) for _ in range(8)]
        self._ck(self.L.hamr_get_block_prims(self.h, int(b), (c_double_p * 8)(*[_dp(o) for o in out])))
        return out

    def get_block_bface(self, b):
        n = self.block_info(b)[2]
        out = [np.empty(tuple(n[e] + (e == d) for e in range(3))) for d in range(3)]
        self._ck(self.L.hamr_get_block_bface(self.h, int(b), (c_double_p * 3)(*[_dp(o) for o in out])))
        return out

    def set_levels(self, tau):
        if tau is None:
            self._ck(self.L.hamr_set_levels(self.h, None))
        else:
            assert len(tau) == self.num_blocks()
            self._ck(self.L.hamr_set_levels(self.h, (C.c_int * len(tau))(*[int(v) for v in tau])))

    def levels(self):
        return [self.block_info(b)[3] for b in range(self.num_blocks())]

    def block_info(self, b):
        lo, dx = np.zeros(3), np.zeros(3)
        n = (C.c_int * 3)()
        tl = C.c_int(0)
        self._ck(self.L.hamr_block_info(self.h, b, _dp(lo), _dp(dx), n, C.byref(tl)))
        return lo, dx, tuple(n[:]), tl.value

    # -- diagnostics --------------------------------------------------------------------------------
    def debug_emf(self):
        self._ck(self.L.hamr_debug_emf(self.h))

    def get_face(self, d, which):
        out = np.empty(self._fshape(d))
        self._ck(self.L.hamr_get_face(self.h, d, which, _dp(out)))
        return out

    def get_edge(self, f):
        s = [v + 1 for v in self.n]
        s[f] -= 1
        out = np.empty(tuple(s))
        self._ck(self.L.hamr_get_edge(self.h, f, _dp(out)))
        return out

    def ctop(self):
        c = np.zeros(3)
        self._ck(self.L.hamr_get_ctop(self.h, _dp(c)))
        return c

    def totals(self):
        t = np.zeros(5)
        self._ck(self.L.hamr_totals(self.h, _dp(t)))
        return t

    def profile_begin(self):
        self._ck(self.L.hamr_profile_begin(self.h))

    def profile_end(self):
        """{kernel class: (summed device ms, launches)} since profile_begin"""
        ms = (C.c_double * NKCLASS)()
        cnt = (C.c_longlong * NKCLASS)()
        self._ck(self.L.hamr_profile_end(self.h, NKCLASS, ms, cnt))
        return {self.L.hamr_profile_class_name(c).decode(): (ms[c], cnt[c]) for c in range(NKCLASS)}

    def geometry(self, kind, level=0):
        """record table `kind` (0 centres, 1..3 faces) as an array (e1, e2, nrec); entry (ti, tj) = index (ti-3, tj-3)"""
        e1, e2, nr = C.c_int(0), C.c_int(0), C.c_int(0)
        self._ck(self.L.hamr_debug_geometry(self.h, kind, level, None, C.byref(e1), C.byref(e2), C.byref(nr)))
        out = np.empty((e1.value, e2.value, nr.value))
        self._ck(self.L.hamr_debug_geometry(self.h, kind, level, _dp(out), None, None, None))
        return out

    @staticmethod
    def _ij(ti, tj):
        a, b = np.ascontiguousarray(ti, dtype=np.int32), np.ascontiguousarray(tj, dtype=np.int32)
        ip = C.POINTER(C.c_int)
        return a, b, a.ctypes.data_as(ip), b.ctypes.data_as(ip)

    def prim2cons(self, ti, tj, prims):
        """prims (n, 8) at table entries (ti, tj) -> densitised hydro rows U (n, 5)"""
        P = _arr(prims)
        a, b, pa, pb = self._ij(ti, tj)
        U = np.empty((len(a), 5))
        self._ck(self.L.hamr_debug_prim2cons(self.h, len(a), pa, pb, _dp(P), _dp(U)))
        return U

    def con2prim(self, ti, tj, U, Bc, guess):
        """U (n, 5), Bc (n, 3), guess (n, 5) -> hydro primitives (n, 5), rc (n)"""
        U, Bc, gs = _arr(U), _arr(Bc), _arr(guess)
        a, b, pa, pb = self._ij(ti, tj)
        out = np.empty((len(a), 5))
        rc = np.zeros(len(a), dtype=np.int32)
        self._ck(self.L.hamr_debug_con2prim(self.h, len(a), pa, pb, _dp(U), _dp(Bc), _dp(gs), _dp(out),
                                            rc.ctypes.data_as(C.POINTER(C.c_int))))
        return out, rc

    def floors(self, ti, tj, P):
        """floors and ceiling on P (n, 5) -> new P, flags (bit 0 rho floor, 1 u floor, 2 ceiling)"""
        Q = _arr(P).copy()
        a, b, pa, pb = self._ij(ti, tj)
        fl = np.zeros(len(a), dtype=np.int32)
        self._ck(self.L.hamr_debug_floors(self.h, len(a), pa, pb, _dp(Q), fl.ctypes.data_as(C.POINTER(C.c_int))))
        return Q, fl

    def kadv(self):
        """kappa the entropy row gave in the latest update stage, active zones (entropy_backup grids)"""
        out = np.empty(self.n)
        self._ck(self.L.hamr_debug_kappa(self.h, _dp(out)))
        return out

    def con2prim_entropy(self, ti, tj, U, US, Bc, guess):
        """U (n, 5), entropy row US (n), Bc (n, 3), guess (n, 5) -> hydro primitives (n, 5), rc (n)"""
        U, US, Bc, gs = _arr(U), _arr(US), _arr(Bc), _arr(guess)
        a, b, pa, pb = self._ij(ti, tj)
        out = np.empty((len(a), 5))
        rc = np.zeros(len(a), dtype=np.int32)
        self._ck(self.L.hamr_debug_con2prim_entropy(self.h, len(a), pa, pb, _dp(U), _dp(US), _dp(Bc), _dp(gs), _dp(out),
                                                    rc.ctypes.data_as(C.POINTER(C.c_int))))
        return out, rc

    def con2prim_aitken(self, ti, tj, U, Bc, guess):
        """U (n, 5), Bc (n, 3), guess (n, 5) -> hydro primitives (n, 5), rc (n): the Aitken-accelerated inversion"""
        U, Bc, gs = _arr(U), _arr(Bc), _arr(guess)
        a, b, pa, pb = self._ij(ti, tj)
        out = np.empty((len(a), 5))
        rc = np.zeros(len(a), dtype=np.int32)
        self._ck(self.L.hamr_debug_con2prim_aitken(self.h, len(a), pa, pb, _dp(U), _dp(Bc), _dp(gs), _dp(out),
                                                   rc.ctypes.data_as(C.POINTER(C.c_int))))
        return out, rc

    def aitken_count(self):
        n = C.c_longlong(0)
        self._ck(self.L.hamr_debug_aitken_count(self.h, C.byref(n)))
        return n.value

    def floors_drift(self, ti, tj, P, Bc):
        """floors (in the drift frame on a drift_floors grid) and ceiling on P (n, 5) with field Bc (n, 3)"""
        Q, Bc = _arr(P).copy(), _arr(Bc)
        a, b, pa, pb = self._ij(ti, tj)
        fl = np.zeros(len(a), dtype=np.int32)
        self._ck(self.L.hamr_debug_floors_drift(self.h, len(a), pa, pb, _dp(Q), _dp(Bc),
                                                fl.ctypes.data_as(C.POINTER(C.c_int))))
        return Q, fl

    def launch_count(self):
        n = C.c_longlong(0)
        self._ck(self.L.hamr_launch_count(self.h, C.byref(n)))
        return n.value


def divb_noalloc(n, dx, bface_dev_ptrs, out_dev_ptr, stream=None):
    """hamr_divb_noalloc: n (3 ints), dx (3 floats), bface_dev_ptrs (3 device addresses as ints), out_dev_ptr (device
    address of one double), stream (cudaStream_t as int or None).  Enqueues and returns; raises on a non-zero status."""
    L = lib()
    nn = (C.c_int * 3)(*[int(v) for v in n])
    dd = (C.c_double * 3)(*[float(v) for v in dx])
    bp = (C.c_void_p * 3)(*[C.c_void_p(int(a)) for a in bface_dev_ptrs])
    rc = L.hamr_divb_noalloc(nn, dd, bp, C.c_void_p(int(out_dev_ptr)), C.c_void_p(stream))
    if rc != OK:
        raise HamrError(rc, L.hamr_noalloc_last_error().decode())


def bench_fp64(mix=0, iters=20000, stream=None):
    """hamr_bench_fp64: (seconds, thread-level FP64 instructions) of the timed launch on the current device"""
    sec, ins = C.c_double(0), C.c_double(0)
    rc = lib().hamr_bench_fp64(C.c_void_p(stream), int(mix), int(iters), C.byref(sec), C.byref(ins))
    if rc != OK:
        raise HamrError(rc, "hamr_bench_fp64")
    return sec.value, ins.value
