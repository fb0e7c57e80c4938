"""ctypes loader for the CPU oracle (oracle/liborc.so).  Test infrastructure only."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
ORACLE_DIR = os.path.join(os.path.dirname(_HERE), "oracle")
_LIB = None

c_double_p = C.POINTER(C.c_double)


class Params(C.Structure):
    _fields_ = [("metric", C.c_int32), ("recon", C.c_int32), ("n", C.c_int32 * 3),
                ("bc_lo", C.c_int32 * 3), ("bc_hi", C.c_int32 * 3), ("nb", C.c_int32 * 3),
                ("n_deref", C.c_int32), ("deref_factor", C.c_int32 * 4),
                ("lat_max_level", C.c_int32), ("map", C.c_int32),
                ("entropy_backup", C.c_int32), ("drift_floors", C.c_int32),
                ("a", C.c_double), ("xmin", C.c_double * 3), ("xmax", C.c_double * 3),
                ("gamma_ad", C.c_double), ("cour", C.c_double),
                ("rho_fl_coef", C.c_double), ("rho_fl_pow", C.c_double),
                ("u_fl_coef", C.c_double), ("u_fl_pow", C.c_double), ("gamma_max", C.c_double),
                ("deref_theta_deg", C.c_double * 4), ("r_refine_max", C.c_double)]


class Geom(C.Structure):
    _fields_ = [("gcov", C.c_double * 16), ("gcon", C.c_double * 16), ("gdet", C.c_double),
                ("alpha", C.c_double), ("beta", C.c_double * 3)]

    def cov(self):
        return np.array(self.gcov[:]).reshape(4, 4)

    def con(self):
        return np.array(self.gcon[:]).reshape(4, 4)


def build():
    subprocess.check_call(["make", "-s", "-C", ORACLE_DIR], stdout=subprocess.DEVNULL)


def lib():
    global _LIB
    if _LIB is None:
        build()
        L = C.CDLL(os.path.join(ORACLE_DIR, "liborc.so"))
        L.orc_grid_create.restype = C.c_void_p
        L.orc_grid_create.argtypes = [C.POINTER(Params)]
        L.orc_grid_destroy.argtypes = [C.c_void_p]
        L.orc_get_dt.restype = C.c_double
        L.orc_get_dt.argtypes = [C.c_void_p]
        L.orc_set_dt.argtypes = [C.c_void_p, C.c_double]
        for name in ("orc_set_prims", "orc_step", "orc_get_prims", "orc_get_bface", "orc_divb",
                     "orc_get_stats", "orc_get_face", "orc_totals", "orc_debug_emf", "orc_get_edge",
                     "orc_get_centre_emf", "orc_get_ctop", "orc_block_info", "orc_set_block_prims",
                     "orc_get_block_prims", "orc_get_block_bface"):
            getattr(L, name).argtypes = None
        L.orc_bface_mismatch.restype = C.c_double
        L.orc_bface_mismatch.argtypes = [C.c_void_p]
        L.orc_num_blocks.argtypes = [C.c_void_p]
        L.orc_blocks_commit.argtypes = [C.c_void_p]
        L.orc_force_levels.argtypes = [C.c_void_p, C.POINTER(C.c_int)]
        L.orc_geom_at.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, C.POINTER(Geom)]
        L.orc_conn_at.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, c_double_p]
        L.orc_gcov_derivs.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, c_double_p,
                                      c_double_p, c_double_p]
        L.orc_prim_to_UF.argtypes = [c_double_p, C.POINTER(Geom), C.c_double, C.c_int, c_double_p, c_double_p]
        L.orc_state.argtypes = [c_double_p, C.POINTER(Geom)] + [c_double_p] * 5
        L.orc_wavespeeds.argtypes = [c_double_p, C.POINTER(Geom), C.c_double, C.c_int, c_double_p, c_double_p]
        L.orc_source.argtypes = [c_double_p, C.POINTER(Geom), c_double_p, C.c_double, c_double_p]
        L.orc_con2prim.argtypes = [c_double_p, c_double_p, C.POINTER(Geom), C.c_double, c_double_p,
                                   c_double_p, C.POINTER(C.c_int)]
        L.orc_floors.argtypes = [C.POINTER(Params), C.POINTER(Geom), C.c_double, c_double_p, c_double_p,
                                 C.POINTER(C.c_longlong)]
        L.orc_con2prim_aitken.argtypes = [c_double_p, c_double_p, C.POINTER(Geom), C.c_double, c_double_p,
                                          c_double_p, C.POINTER(C.c_int)]
        L.orc_con2prim_entropy.argtypes = [c_double_p, C.c_double, c_double_p, C.POINTER(Geom), C.c_double,
                                           c_double_p, c_double_p, C.POINTER(C.c_int)]
        L.orc_entropy_UF.argtypes = [c_double_p, C.POINTER(Geom), C.c_double, C.c_int, c_double_p, c_double_p]
        L.orc_get_backup_count.argtypes = [C.c_void_p, C.POINTER(C.c_longlong)]
        L.orc_refine_radius.argtypes = [C.c_void_p, C.c_double, c_double_p]
        L.orc_regrid.restype = C.c_void_p
        L.orc_regrid.argtypes = [C.c_void_p, C.c_double]
        L.orc_get_t.restype = C.c_double
        L.orc_get_t.argtypes = [C.c_void_p]
        L.orc_get_kadv.argtypes = [C.c_void_p, c_double_p]
        L.orc_get_block_kadv.argtypes = [C.c_void_p, C.c_int, c_double_p]
        L.orc_get_aitken_count.argtypes = [C.c_void_p, C.POINTER(C.c_longlong)]
        L.orc_ppm_zone.argtypes = [c_double_p] * 3
        L.orc_plm_zone.argtypes = [c_double_p] * 3
        L.orc_hll.argtypes = [c_double_p] * 4 + [C.c_double, C.c_double, c_double_p]
        assert L.orc_sizeof_params() == C.sizeof(Params), (L.orc_sizeof_params(), C.sizeof(Params))
        _LIB = L
    return _LIB


def _dp(a):
    return a.ctypes.data_as(c_double_p)


def _arr(x):
    return np.ascontiguousarray(np.asarray(x, dtype=np.float64))


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
    q.a = float(p["a"])
    q.gamma_ad, q.cour = float(p["gamma_ad"]), float(p["cour"])
    q.rho_fl_coef, q.rho_fl_pow = float(p["rho_fl_coef"]), float(p["rho_fl_pow"])
    q.u_fl_coef, q.u_fl_pow = float(p["u_fl_coef"]), float(p["u_fl_pow"])
    q.gamma_max = float(p["gamma_max"])
    q.r_refine_max = float(p["r_refine_max"])
    q.entropy_backup = int(p.get("entropy_backup", 0))
    q.drift_floors = int(p.get("drift_floors", 0))
    return q


class OrcGrid:
    """Thin wrapper: same call names as the product binding (create/set_prims/step/...)."""

    def __init__(self, p: dict, _handle=None):
        self.L = lib()
        self.p = p
        self.n = tuple(int(v) for v in p["n"])
        self._par = pack_params(p)
        self.h = _handle if _handle is not None else self.L.orc_grid_create(C.byref(self._par))
        if not self.h:
            raise RuntimeError("orc_grid_create failed")
        self.h = C.c_void_p(self.h)

    def refine_radius(self, rho_cut):
        """C-20: the r_refine_max the density criterion asks for (0: no refined region)"""
        r = np.zeros(1)
        assert self.L.orc_refine_radius(self.h, float(rho_cut), _dp(r)) == 0
        return float(r[0])

    def regrid(self, r_refine_max):
        """C-20: a new grid with that r_refine_max carrying this grid's state (this grid stays valid)"""
        h = self.L.orc_regrid(self.h, float(r_refine_max))
        if not h:
            raise RuntimeError("orc_regrid failed")
        return OrcGrid(dict(self.p, r_refine_max=float(r_refine_max)), _handle=h)

    @property
    def t(self):
        return self.L.orc_get_t(self.h)

    def close(self):
        if self.h:
            self.L.orc_grid_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _fshape(self, d):
        s = list(self.n)
        s[d] += 1
        return tuple(s)

    def set_prims(self, hydro, bface=None):
        hy = [_arr(h) for h in hydro]
        assert all(h.shape == self.n for h in hy)
        hp = (c_double_p * 5)(*[_dp(h) for h in hy])
        if bface is None:
            rc = self.L.orc_set_prims(self.h, hp, None)
        else:
            bf = [_arr(b) for b in bface]
            assert all(bf[d].shape == self._fshape(d) for d in range(3))
            bp = (c_double_p * 3)(*[_dp(b) for b in bf])
            rc = self.L.orc_set_prims(self.h, hp, bp)
        return rc

    def step(self, nsteps=1):
        t, dt = C.c_double(0), C.c_double(0)
        rc = self.L.orc_step(self.h, C.c_int(nsteps), C.byref(t), C.byref(dt))
        if rc != 0:
            raise RuntimeError(f"orc_step rc={rc}")
        return t.value, dt.value

    @property
    def dt(self):
        return self.L.orc_get_dt(self.h)

    @dt.setter
    def dt(self, v):
        self.L.orc_set_dt(self.h, C.c_double(v))

    def get_prims(self):
        out = [np.empty(self.n) for _ in range(8)]
        self.L.orc_get_prims(self.h, (c_double_p * 8)(*[_dp(o) for o in out]))
        return out

    def get_bface(self):
        out = [np.empty(self._fshape(d)) for d in range(3)]
        self.L.orc_get_bface(self.h, (c_double_p * 3)(*[_dp(o) for o in out]))
        return out

    def divb(self):
        v = C.c_double(0)
        self.L.orc_divb(self.h, C.byref(v))
        return v.value

    def stats(self):
        c = (C.c_longlong * 4)()
        self.L.orc_get_stats(self.h, c)
        return tuple(c[:])

    def backup_count(self):
        v = C.c_longlong(0)
        self.L.orc_get_backup_count(self.h, C.byref(v))
        return v.value

    def aitken_count(self):
        v = C.c_longlong(0)
        self.L.orc_get_aitken_count(self.h, C.byref(v))
        return v.value

    def kadv(self):
        out = np.empty(self.n)
        rc = self.L.orc_get_kadv(self.h, _dp(out))
        assert rc == 0
        return out

    def totals(self):
        t = np.zeros(5)
        self.L.orc_totals(self.h, _dp(t))
        return t

    def get_face(self, d, which):
        out = np.empty(self._fshape(d))
        self.L.orc_get_face(self.h, C.c_int(d), C.c_int(which), _dp(out))
        return out

    def debug_emf(self):
        self.L.orc_debug_emf(self.h)

    def get_edge(self, f):
        s = [v + 1 for v in self.n]
        s[f] -= 1
        out = np.empty(tuple(s))
        self.L.orc_get_edge(self.h, C.c_int(f), _dp(out))
        return out

    def get_centre_emf(self, f):
        out = np.empty(self.n)
        self.L.orc_get_centre_emf(self.h, C.c_int(f), _dp(out))
        return out

    def ctop(self):
        c = np.zeros(3)
        self.L.orc_get_ctop(self.h, _dp(c))
        return c

    # ---- block-structured grid ----
    def get_padded(self, kind):
        """full padded array (ghosts filled) of a monolithic grid: kind 0..4 hydro, 5..7 Bc, 8..10 Bf"""
        e = tuple(v + 7 for v in self.n)
        out = np.empty(e)
        self.L.orc_get_padded.argtypes = [C.c_void_p, C.c_int, c_double_p]
        assert self.L.orc_get_padded(self.h, int(kind), _dp(out)) == 0
        return out

    def num_blocks(self):
        return self.L.orc_num_blocks(self.h)

    def block_info(self, b):
        xlo, dx = (C.c_double * 3)(), (C.c_double * 3)()
        n = (C.c_int * 3)()
        tau, lev = C.c_int(0), C.c_int(0)
        rc = self.L.orc_block_info(self.h, C.c_int(b), xlo, dx, n, C.byref(tau), C.byref(lev))
        assert rc == 0
        return dict(x_lo=np.array(xlo[:]), dx=np.array(dx[:]), n=tuple(n[:]), tau=tau.value, lev1=lev.value)

    def levels(self):
        return np.array([self.block_info(b)["tau"] for b in range(self.num_blocks())])

    def force_levels(self, tau):
        if tau is None:
            return self.L.orc_force_levels(self.h, None)
        a = (C.c_int * len(tau))(*[int(t) for t in tau])
        return self.L.orc_force_levels(self.h, a)

    def set_block_prims(self, b, hydro, bface=None):
        hy = [_arr(h) for h in hydro]
        hp = (c_double_p * 5)(*[_dp(h) for h in hy])
        if bface is None:
            return self.L.orc_set_block_prims(self.h, C.c_int(b), hp, None)
        bf = [_arr(x) for x in bface]
        bp = (c_double_p * 3)(*[_dp(x) for x in bf])
        return self.L.orc_set_block_prims(self.h, C.c_int(b), hp, bp)

    def commit(self):
        return self.L.orc_blocks_commit(self.h)

    def get_block_kadv(self, b):
        out = np.empty(self.block_info(b)["n"])
        rc = self.L.orc_get_block_kadv(self.h, C.c_int(b), _dp(out))
        assert rc == 0
        return out

    def get_block_prims(self, b):
        n = self.block_info(b)["n"]
        out = [np.empty(n) for _ in range(8)]
        rc = self.L.orc_get_block_prims(self.h, C.c_int(b), (c_double_p * 8)(*[_dp(o) for o in out]))
        assert rc == 0
        return out

    def get_block_bface(self, b):
        n = list(self.block_info(b)["n"])
        out = []
        for d in range(3):
            s = list(n)
            s[d] += 1
            out.append(np.empty(tuple(s)))
        rc = self.L.orc_get_block_bface(self.h, C.c_int(b), (c_double_p * 3)(*[_dp(o) for o in out]))
        assert rc == 0
        return out

    def bface_mismatch(self):
        return self.L.orc_bface_mismatch(self.h)


# ---- per-zone helpers for the pins ---------------------------------------------------------------
def geom_at(metric, a, x1, x2) -> Geom:
    G = Geom()
    lib().orc_geom_at(metric, a, x1, x2, C.byref(G))
    return G


def conn_at(metric, a, x1, x2):
    c = np.zeros(64)
    lib().orc_conn_at(metric, a, x1, x2, _dp(c))
    return c.reshape(4, 4, 4)


def gcov_derivs(metric, a, x1, x2):
    g, d1, d2 = np.zeros(16), np.zeros(16), np.zeros(16)
    lib().orc_gcov_derivs(metric, a, x1, x2, _dp(g), _dp(d1), _dp(d2))
    return g.reshape(4, 4), d1.reshape(4, 4), d2.reshape(4, 4)


def prim_to_UF(P, G, gam, direction=0):
    P = _arr(P)
    U, F = np.zeros(8), np.zeros(8)
    lib().orc_prim_to_UF(_dp(P), C.byref(G), gam, direction, _dp(U), _dp(F))
    return U, F


def state(P, G):
    P = _arr(P)
    o = [np.zeros(4) for _ in range(4)]
    bsq = np.zeros(1)
    lib().orc_state(_dp(P), C.byref(G), _dp(o[0]), _dp(o[1]), _dp(o[2]), _dp(o[3]), _dp(bsq))
    return dict(ucon=o[0], ucov=o[1], bcon=o[2], bcov=o[3], bsq=bsq[0])


def wavespeeds(P, G, gam, direction):
    P = _arr(P)
    a, b = np.zeros(1), np.zeros(1)
    lib().orc_wavespeeds(_dp(P), C.byref(G), gam, direction, _dp(a), _dp(b))
    return a[0], b[0]


def source(P, G, conn, gam):
    P = _arr(P)
    c = _arr(conn).reshape(-1)
    S = np.zeros(5)
    lib().orc_source(_dp(P), C.byref(G), _dp(c), gam, _dp(S))
    return S


def con2prim(U5, Bc, G, gam, Pguess):
    U5, Bc, Pg = _arr(U5), _arr(Bc), _arr(Pguess)
    out = np.zeros(5)
    it = C.c_int(0)
    rc = lib().orc_con2prim(_dp(U5), _dp(Bc), C.byref(G), gam, _dp(Pg), _dp(out), C.byref(it))
    return rc, out, it.value


def floors(p, G, r, P5, Bc=None):
    """floors and Lorentz-factor ceiling (C-13; C-19 with p["drift_floors"] and a field Bc) on one zone: new P5,
    (rho-floor, u-floor, ceiling) hits"""
    par = pack_params(p)
    P = _arr(P5).copy()
    c = (C.c_longlong * 3)()
    B = _arr(Bc) if Bc is not None else None
    lib().orc_floors(C.byref(par), C.byref(G), float(r), _dp(P), _dp(B) if B is not None else None, c)
    return P, tuple(c[:])


def con2prim_aitken(U5, Bc, G, gam, Pguess):
    """C-21: the Aitken-accelerated fixed-point inversion"""
    U5, Bc, Pg = _arr(U5), _arr(Bc), _arr(Pguess)
    out = np.zeros(5)
    it = C.c_int(0)
    rc = lib().orc_con2prim_aitken(_dp(U5), _dp(Bc), C.byref(G), gam, _dp(Pg), _dp(out), C.byref(it))
    return rc, out, it.value


def con2prim_entropy(U5, US, Bc, G, gam, Pguess):
    """C-18: inversion with the entropy row US in place of the energy row"""
    U5, Bc, Pg = _arr(U5), _arr(Bc), _arr(Pguess)
    out = np.zeros(5)
    it = C.c_int(0)
    rc = lib().orc_con2prim_entropy(_dp(U5), float(US), _dp(Bc), C.byref(G), gam, _dp(Pg), _dp(out), C.byref(it))
    return rc, out, it.value


def entropy_UF(P, G, gam, direction):
    P = _arr(P)
    a, b = np.zeros(1), np.zeros(1)
    lib().orc_entropy_UF(_dp(P), C.byref(G), gam, direction, _dp(a), _dp(b))
    return a[0], b[0]


def ppm_zone(a5):
    a5 = _arr(a5)
    l, r = np.zeros(1), np.zeros(1)
    lib().orc_ppm_zone(_dp(a5), _dp(l), _dp(r))
    return l[0], r[0]


def plm_zone(a3):
    a3 = _arr(a3)
    l, r = np.zeros(1), np.zeros(1)
    lib().orc_plm_zone(_dp(a3), _dp(l), _dp(r))
    return l[0], r[0]


def hll(UL, UR, FL, FR, cmin, cmax):
    F = np.zeros(8)
    lib().orc_hll(_dp(_arr(UL)), _dp(_arr(UR)), _dp(_arr(FL)), _dp(_arr(FR)), cmin, cmax, _dp(F))
    return F
