"""GPU checks below the level of a whole step:
 * H0: the device geometry tables against closed forms typed here (not through the oracle): sqrt(-g) = r Sigma sin theta,
   lapse, shift, spatial metric and its inverse, the inverse 4-metric entries of the face records, d ln sqrt(-g) and the
   metric derivatives against Richardson differences of the closed-form metric;
 * the per-zone physics of the kernels (prim -> U, U -> prim, floors / ceiling) on caller-supplied states against the
   oracle's per-zone routines, including the branches a torus run never takes: failed inversion, Lorentz-factor
   ceiling, both floors;
 * whole steps that drive those branches, with all four event counters equal on both sides.
Needs a B200."""
import numpy as np
import pytest

from paper_1912_10192_b200 import inputs as I
from tests._parity import parity_errors

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def H():
    from paper_1912_10192_b200 import build, hamr
    build.build_lib()
    hamr.lib()
    return hamr


# ---- closed forms of DESIGN.md C-1, typed for this test -----------------------------------------------------------
def _gcov4(a, x1, th):
    r = np.exp(x1)
    s2, c2 = np.sin(th) ** 2, np.cos(th) ** 2
    Sig = r * r + a * a * c2
    f = 2.0 * r / Sig
    g = np.zeros((4, 4))
    g[0, 0] = -(1.0 - f)
    g[0, 1] = g[1, 0] = f * r
    g[0, 3] = g[3, 0] = -f * a * s2
    g[1, 1] = (1.0 + f) * r * r
    g[1, 3] = g[3, 1] = -a * s2 * (1.0 + f) * r
    g[2, 2] = Sig
    g[3, 3] = s2 * (Sig + a * a * s2 * (1.0 + f))
    return g


def _richardson(fun, x, h):
    d1 = (fun(x + h) - fun(x - h)) / (2 * h)
    d2 = (fun(x + h / 2) - fun(x - h / 2)) / h
    return (4 * d2 - d1) / 3


def _mirror(th):
    th = abs(th)
    return 2 * np.pi - th if th > np.pi else th


def test_geometry_tables_match_closed_forms(H):
    p = I.torus_params()                                    # cfg 0: a = 0.9375, r in [1.2, 50], 32 x 16
    g = H.Grid(p)
    a = p["a"]
    n = p["n"]
    dx1 = (np.log(p["xmax"][0]) - np.log(p["xmin"][0])) / n[0]
    dx2 = np.pi / n[1]
    x10 = np.log(p["xmin"][0])
    C = g.geometry(0)
    F = [None, g.geometry(1), g.geometry(2), g.geometry(3)]
    assert C.shape == (n[0] + 7, n[1] + 7, 32) and F[1].shape == (n[0] + 7, n[1] + 7, 16)
    hm, hn = [0, 0, 0, 1, 1, 2, 3], [0, 1, 3, 1, 3, 2, 3]
    worst = 0.0
    for ti in range(0, n[0] + 7, 3):
        for tj in range(n[1] + 7):
            i, j = ti - 3, tj - 3
            x1c, x2c = x10 + (i + 0.5) * dx1, (j + 0.5) * dx2
            th = _mirror(x2c)
            sgn = -1.0 if (x2c < 0 or x2c > np.pi) else 1.0
            r = np.exp(x1c)
            Sig = r * r + a * a * np.cos(th) ** 2
            rec = C[ti, tj]
            G4 = _gcov4(a, x1c, th)
            gs = G4[1:, 1:]
            gam = np.array([[rec[0], 0, rec[1]], [0, rec[2], 0], [rec[1], 0, rec[3]]])
            inv = np.array([[rec[4], 0, rec[5]], [0, rec[6], 0], [rec[5], 0, rec[7]]])
            assert np.allclose(gam, gs, rtol=1e-13, atol=1e-13 * np.abs(gs).max())
            assert np.allclose(inv @ gs, np.eye(3), atol=2e-12)
            alpha2 = Sig / (Sig + 2 * r)
            assert abs(rec[8] ** 2 - alpha2) <= 1e-13 * alpha2 and abs(rec[8] * rec[9] - 1) <= 1e-14
            beta1 = 2 * r / (Sig + 2 * r) / r
            assert abs(rec[11] - beta1) <= 1e-12 * beta1 and abs(rec[10] * rec[8] - rec[11]) <= 1e-14 * beta1
            gdet = r * Sig * abs(np.sin(th))
            assert abs(rec[12] - gdet) <= 1e-12 * gdet and abs(rec[12] * rec[13] - 1) <= 1e-14
            # det g = -(r Sigma sin theta)^2 from the closed-form covariant metric, against the table's sqrt(-g)
            assert abs(-np.linalg.det(G4) - rec[12] ** 2) <= 1e-10 * rec[12] ** 2
            # derivatives: Richardson differences of the closed forms (the x2 derivative of a mirrored row flips sign)
            d1 = _richardson(lambda x: _gcov4(a, x, th), x1c, 2e-3)
            d2 = sgn * _richardson(lambda t: _gcov4(a, x1c, t), th, 2e-3)
            for c in range(7):
                wgt = 0.5 if hm[c] == hn[c] else 1.0
                sc = max(abs(G4[hm[c], hn[c]]), 1e-30) + np.abs(d1).max() * 1e-6
                assert abs(rec[16 + c] - wgt * d1[hm[c], hn[c]]) <= 2e-8 * (abs(d1[hm[c], hn[c]]) + sc)
                assert abs(rec[23 + c] - wgt * d2[hm[c], hn[c]]) <= 2e-8 * (abs(d2[hm[c], hn[c]]) + sc)
            lg = lambda x, t: np.log(np.exp(x) * (np.exp(2 * x) + a * a * np.cos(t) ** 2) * abs(np.sin(t)))
            dl1 = _richardson(lambda x: lg(x, th), x1c, 2e-3)
            dl2 = sgn * _richardson(lambda t: lg(x1c, t), th, 2e-3)
            assert abs(rec[14] - dl1) <= 1e-8 * (1 + abs(dl1)) and abs(rec[15] - dl2) <= 1e-8 * (1 + abs(dl2))
            # face records: x1-face at (x1f, x2c), x2-face at (x1c, x2f), x3-face at the centre
            x1f, x2f = x10 + i * dx1, j * dx2
            for kind, (xa, xb) in ((1, (x1f, x2c)), (2, (x1c, x2f)), (3, (x1c, x2c))):
                fr = F[kind][ti, tj]
                thf = _mirror(xb)
                on_axis = kind == 2 and j in (0, n[1])
                if on_axis:
                    assert fr[12] == 0.0 and fr[13] == 0.0   # C-7: pole faces carry sqrt(-g) = 0
                    continue
                Gf = _gcov4(a, xa, thf)
                Ki = np.linalg.inv(Gf)
                assert np.allclose([fr[0], fr[1], fr[2], fr[3]], [Gf[1, 1], Gf[1, 3], Gf[2, 2], Gf[3, 3]], rtol=1e-13,
                                   atol=1e-13 * np.abs(Gf).max())
                rf = np.exp(xa)
                Sf = rf * rf + a * a * np.cos(thf) ** 2
                assert abs(fr[4] ** 2 - Sf / (Sf + 2 * rf)) <= 1e-13 and abs(fr[8] + fr[4] ** 2) <= 1e-15
                assert abs(fr[9] - Ki[0, 0]) <= 1e-10 * abs(Ki[0, 0])
                assert abs(fr[10] - Ki[kind, kind]) <= 1e-9 * abs(Ki[kind, kind])
                assert abs(fr[11] - Ki[0, kind]) <= 1e-10 * (abs(Ki[0, 1]) + 1e-30)
                gd = rf * Sf * abs(np.sin(thf))
                assert abs(fr[12] - gd) <= 1e-12 * gd
            worst = max(worst, abs(rec[12] - gdet) / gdet)
    print("geometry tables: worst relative sqrt(-g) error", worst)
    # Minkowski: identity
    q = I.minkowski_params(n=(4, 4, 4))
    gm = H.Grid(q)
    Cm = gm.geometry(0)
    assert np.all(Cm[..., [0, 2, 3, 4, 6, 7, 8, 9, 12, 13]] == 1.0) and np.all(Cm[..., [1, 5, 10, 11, 14, 15]] == 0.0)
    assert np.all(Cm[..., 16:30] == 0.0)


def _random_states(rng, n, umax=1.0):
    rho = 10.0 ** rng.uniform(-2, 0.5, n)
    u = rho * 10.0 ** rng.uniform(-2, 0, n)
    # the conditioning range of pin P3: u / rho in [1e-2, 1], |B| / sqrt(rho) <~ 1, gamma <~ 2
    ut = rng.normal(size=(n, 3)) * 0.5 * umax
    B = rng.normal(size=(n, 3)) * 0.3 * np.sqrt(rho)[:, None]
    return np.column_stack([rho, u, ut, B])


def test_zone_physics_matches_oracle_and_round_trips(H, orc):
    p = I.torus_params()
    g = H.Grid(p)
    n = p["n"]
    rng = np.random.default_rng(11)
    ns = 400
    ti = rng.integers(3, n[0] + 3, ns)
    tj = rng.integers(3, n[1] + 3, ns)
    dx1 = (np.log(p["xmax"][0]) - np.log(p["xmin"][0])) / n[0]
    x1 = np.log(p["xmin"][0]) + (ti - 3 + 0.5) * dx1
    x2 = (tj - 3 + 0.5) * np.pi / n[1]
    C = g.geometry(0)
    # physical-scale velocities and fields: ut^i and B^i scaled by 1/sqrt(g_ii) so that gamma <~ 2
    P = _random_states(rng, ns)
    sc = np.sqrt(np.stack([C[ti, tj, 0], C[ti, tj, 2], C[ti, tj, 3]], axis=1))
    P[:, 2:5] /= sc
    P[:, 5:8] /= sc
    U = g.prim2cons(ti, tj, P)
    gam = p["gamma_ad"]
    Uo = np.zeros_like(U)
    Po = np.zeros((ns, 5))
    for s in range(ns):
        G = orc.geom_at(p["metric"], p["a"], x1[s], x2[s])
        Uo[s] = orc.prim_to_UF(P[s], G, gam)[0][:5]
    scale = np.abs(Uo).max(axis=1, keepdims=True)
    assert (np.abs(U - Uo) / scale).max() <= 2e-13
    # round trip on the GPU: prim -> U -> prim from a 5 % perturbed guess, <= 1e-12 in the stated conditioning range
    guess = P[:, :5] * (1 + 0.05 * rng.uniform(-1, 1, (ns, 5)))
    out, rc = g.con2prim(ti, tj, U, P[:, 5:8], guess)
    assert np.all(rc == 0)
    assert (np.abs(out[:, :2] - P[:, :2]) / P[:, :2]).max() <= 1e-12
    vn = np.sqrt(((P[:, 2:5] * sc) ** 2).sum(axis=1, keepdims=True))
    assert (np.abs(out[:, 2:5] - P[:, 2:5]) * sc / np.maximum(vn, 1e-3)).max() <= 1e-12
    # and against the oracle's inversion from the same guess
    for s in range(0, ns, 7):
        G = orc.geom_at(p["metric"], p["a"], x1[s], x2[s])
        rco, Po, _ = orc.con2prim(U[s], P[s, 5:8], G, gam, guess[s])
        assert rco == 0
        assert (np.abs(out[s, :2] - Po[:2]) / Po[:2]).max() <= 1e-11
        assert (np.abs(out[s, 2:5] - Po[2:5]) * sc[s]).max() <= 1e-11 * max(vn[s, 0], 1e-3)
    # failed inversion: momentum far beyond what the energy allows; a negative conserved density.  Both sides refuse,
    # and the kernel's result is the guess it was given (C-13: the zone keeps its source state)
    gd = C[ti, tj, 12]
    Ubad = U.copy()
    Ubad[::2, 2] = 50.0 * gd[::2] * (np.abs(Uo[::2, 0]) / gd[::2] + 1.0) * np.sqrt(C[ti[::2], tj[::2], 0])
    Ubad[1::2, 0] = -np.abs(U[1::2, 0])
    outb, rcb = g.con2prim(ti, tj, Ubad, P[:, 5:8], guess)
    nfail_o = 0
    for s in range(ns):
        G = orc.geom_at(p["metric"], p["a"], x1[s], x2[s])
        rco, _, _ = orc.con2prim(Ubad[s], P[s, 5:8], G, gam, guess[s])
        assert (rco != 0) == (rcb[s] != 0), (s, rco, rcb[s])
        nfail_o += rco != 0
    assert nfail_o >= ns // 2 and np.array_equal(outb[rcb != 0], guess[rcb != 0])
    # floors and ceiling: flags and values against the oracle, on states that hit each branch
    Q = P[:, :5].copy()
    r = np.exp(x1)
    Q[0::4, 0] = 1e-7 * r[0::4] ** -1.5                  # below the density floor
    Q[1::4, 1] = -1e-3                                     # below the energy floor
    Q[2::4, 2:5] *= 400.0                                  # far above the Lorentz-factor ceiling
    Qn, fl = g.floors(ti, tj, Q)
    for s in range(ns):
        G = orc.geom_at(p["metric"], p["a"], x1[s], x2[s])
        Pn, c = orc.floors(p, G, r[s], Q[s])
        assert (fl[s] & 1, (fl[s] >> 1) & 1, (fl[s] >> 2) & 1) == c, (s, fl[s], c)
        assert np.allclose(Qn[s], Pn, rtol=1e-13, atol=0)
    assert (fl & 1).sum() >= ns // 4 and ((fl >> 1) & 1).sum() >= ns // 4 and ((fl >> 2) & 1).sum() >= ns // 4 - 1
    # after the ceiling the Lorentz factor is gamma_max
    hit = ((fl >> 2) & 1) == 1
    q = (C[ti, tj, 0] * Qn[:, 2] ** 2 + C[ti, tj, 2] * Qn[:, 3] ** 2 + C[ti, tj, 3] * Qn[:, 4] ** 2
         + 2 * C[ti, tj, 1] * Qn[:, 2] * Qn[:, 4])
    assert np.allclose(np.sqrt(1 + q[hit]), p["gamma_max"], rtol=1e-13)


def _pair(H, orc, p, hyd, bf):
    g, o = H.Grid(p), orc.OrcGrid(p)
    assert g.set_prims(hyd, bf) == 0 and o.set_prims(hyd, bf) == 0
    return g, o


def test_steps_with_lorentz_factor_ceiling_and_with_floors_counts_equal(H, orc):
    # (A) a flow at gamma ~ 60 > gamma_max = 50, smoothly modulated across the flow: every zone hits the ceiling in
    # both stages of every step; (B) a gas at rest below both floors with a smooth pressure modulation: every zone
    # hits both floors.  All four event counters agree exactly with the oracle's, and the primitives to 1e-10.
    n = (16, 8, 32)
    y = (np.arange(n[1]) + 0.5)[None, :, None] / n[1] + np.zeros(n)
    nz = int(np.prod(n))
    p = I.minkowski_params(n=n)
    gam = 60.0 * (1 + 0.05 * np.cos(2 * np.pi * y))
    hyd = [1.0 + 0.1 * np.sin(2 * np.pi * y), np.full(n, 0.5), np.zeros(n), np.zeros(n), np.sqrt(gam ** 2 - 1)]
    g, o = _pair(H, orc, p, hyd, None)
    g.step(1)
    o.step(1)
    sg, so = g.stats(), o.stats()
    assert sg == so == (0, 0, 0, 2 * nz), (sg, so)
    e = parity_errors(p, o.get_prims(), g.get_prims())
    assert max(e.values()) <= 1e-10, e
    P = g.get_prims()
    assert np.allclose(np.sqrt(1 + P[2] ** 2 + P[3] ** 2 + P[4] ** 2), 50.0, rtol=1e-12)
    q = I.minkowski_params(n=n, rho_fl_coef=1e-3, u_fl_coef=1e-4)
    hyd = [2e-4 * (1 + 0.3 * np.sin(2 * np.pi * y)), 3e-5 * (1 + 0.3 * np.cos(2 * np.pi * y)), np.zeros(n), np.zeros(n),
           np.zeros(n)]
    g, o = _pair(H, orc, q, hyd, None)
    g.step(2)
    o.step(2)
    sg, so = g.stats(), o.stats()
    assert sg == so and so[0] == 0 and so[1] >= 2 * nz and so[2] >= 2 * nz, (sg, so)
    e = parity_errors(q, o.get_prims(), g.get_prims())
    assert max(e.values()) <= 2e-10, e


def test_step_with_failed_inversions_keeps_source_state_and_counts_equal(H, orc):
    # the blast of tests/test_oracle_floors_dt_bc.py, 40 x the Courant step: some inversions fail on both sides
    n = (32, 4, 32)
    p = I.minkowski_params(n=n)
    x = (np.arange(n[0]) + 0.5) / n[0]
    rho = np.where(np.abs(x - 0.5) < 0.13, 1.0, 1e-3)[:, None, None] * np.ones(n)
    u = np.where(np.abs(x - 0.5) < 0.13, 1e3, 1e-3)[:, None, None] * np.ones(n)
    hyd = [rho, u, np.zeros(n), np.zeros(n), np.zeros(n)]
    g, o = _pair(H, orc, p, hyd, None)
    g.dt = 40.0 * g.dt
    o.dt = 40.0 * o.dt
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt
    g.step(1)
    o.step(1)
    sg, so = g.stats(), o.stats()
    assert so[0] > 0 and sg == so, (sg, so)
    Pg, Po = g.get_prims(), o.get_prims()
    kept_o = (Po[0] == rho) & (Po[1] == u)
    kept_g = (Pg[0] == rho) & (Pg[1] == u)
    assert np.array_equal(kept_o, kept_g)
    e = parity_errors(p, Po, Pg)
    assert max(e.values()) <= 1e-9, e
