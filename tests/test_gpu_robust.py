"""GPU <-> oracle parity of the robust inversion path (C-18, C-19): the entropy
row and its flux, the entropy inversion, the drift-frame floors, zone by zone and over whole steps, with the event
counters equal on both sides.  Needs a B200."""
import numpy as np
import pytest

from paper_1912_10192_b200 import inputs as I
from tests._parity import parity_errors, rel_max

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def H():
    from paper_1912_10192_b200 import build, hamr
    build.build_lib()
    hamr.lib()
    return hamr


def _pair(H, orc, p, hyd, bf):
    g, o = H.Grid(p), orc.OrcGrid(p)
    assert g.set_prims(hyd, bf) == 0 and o.set_prims(hyd, bf) == 0
    return g, o


def _zone_setup(H, p, ns, seed):
    g = H.Grid(p)
    n = p["n"]
    rng = np.random.default_rng(seed)
    ti = rng.integers(3, n[0] + 3, ns)
    tj = rng.integers(3, n[1] + 3, ns)
    if p["metric"] == I.METRIC_KS:
        dx1 = (np.log(p["xmax"][0]) - np.log(p["xmin"][0])) / n[0]
        x1 = np.log(p["xmin"][0]) + (ti - 3 + 0.5) * dx1
        x2 = (tj - 3 + 0.5) * np.pi / n[1]
    else:
        x1 = (ti - 3 + 0.5) / n[0]
        x2 = (tj - 3 + 0.5) / n[1]
    C = g.geometry(0)
    sc = np.sqrt(np.stack([C[ti, tj, 0], C[ti, tj, 2], C[ti, tj, 3]], axis=1))
    return g, rng, ti, tj, x1, x2, C, sc


def _states(rng, ns, sc, alpha, umax, bmax, cold):
    rho = 10.0 ** rng.uniform(-2, 0.5, ns)
    u = rho * 10.0 ** rng.uniform(-2 - cold, -cold, ns)
    ut = rng.uniform(-umax, umax, (ns, 3)) / sc
    B = rng.uniform(-bmax, bmax, (ns, 3)) * np.sqrt(rho)[:, None] / sc / alpha[:, None]
    return np.column_stack([rho, u, ut, B])


@pytest.mark.parametrize("regime", ["mild", "magnetised", "relativistic", "cold"])
def test_entropy_inversion_matches_oracle(H, orc, regime):
    p = I.torus_params(entropy_backup=1)
    ns = 300
    g, rng, ti, tj, x1, x2, C, sc = _zone_setup(H, p, ns, 21)
    kw = dict(mild=(1.5, 1.0, 0.0), magnetised=(1.0, 30.0, 0.0), relativistic=(12.0, 3.0, 0.0), cold=(1.0, 10.0, 6.0))[regime]
    P = _states(rng, ns, sc, C[ti, tj, 8], *kw)
    gam = p["gamma_ad"]
    U = g.prim2cons(ti, tj, P)
    US = np.zeros(ns)
    Gs = [orc.geom_at(p["metric"], p["a"], x1[s], x2[s]) for s in range(ns)]
    for s in range(ns):
        US[s] = orc.entropy_UF(P[s], Gs[s], gam, 1)[0]
    guess = P[:, :5] * (1 + 0.3 * rng.uniform(-1, 1, (ns, 5)))
    Ue = U.copy()
    Ue[:, 1] = 1e3 * rng.normal(size=ns)        # the energy row is not read
    out, rc = g.con2prim_entropy(ti, tj, Ue, US, P[:, 5:8], guess)
    assert np.all(rc == 0)
    vn = np.sqrt(((P[:, 2:5] * sc) ** 2).sum(axis=1, keepdims=True))
    tol = {"mild": 1e-12, "magnetised": 1e-11, "relativistic": 1e-10, "cold": 1e-11}[regime]   # conditioning
    # round trip on the GPU ...
    assert (np.abs(out[:, :2] - P[:, :2]) / P[:, :2]).max() <= tol
    assert (np.abs(out[:, 2:5] - P[:, 2:5]) * sc / np.maximum(vn, 1e-3)).max() <= tol
    # ... and against the oracle's inversion of the same rows from the same guess
    worst = 0.0
    for s in range(ns):
        rco, Po, _ = orc.con2prim_entropy(U[s], US[s], P[s, 5:8], Gs[s], gam, guess[s])
        assert rco == 0
        worst = max(worst, (np.abs(out[s, :2] - Po[:2]) / Po[:2]).max(),
                    (np.abs(out[s, 2:5] - Po[2:5]) * sc[s]).max() / max(vn[s, 0], 1e-3))
    assert worst <= 10 * tol, worst
    # rows without a state behind them (density, momentum and entropy rescaled independently): the same answer
    V = U.copy()
    V[:, 0] *= rng.uniform(0.3, 3.0, ns)
    V[:, 2:5] *= rng.uniform(0.2, 1.5, (ns, 3))
    VS = US * rng.uniform(0.1, 10.0, ns)
    out2, rc2 = g.con2prim_entropy(ti, tj, V, VS, P[:, 5:8], guess)
    for s in range(ns):
        rco, Po, _ = orc.con2prim_entropy(V[s], VS[s], P[s, 5:8], Gs[s], gam, guess[s])
        assert rco == 0 and rc2[s] == 0
        vs = max(np.sqrt(((Po[2:5] * sc[s]) ** 2).sum()), 1e-3)
        assert (np.abs(out2[s, :2] - Po[:2]) / Po[:2]).max() <= 100 * tol
        assert (np.abs(out2[s, 2:5] - Po[2:5]) * sc[s]).max() <= 100 * tol * vs
    # input without a root: negative density row, negative entropy row, NaN: both sides refuse, the guess is kept
    bad_U, bad_S = U.copy(), US.copy()
    bad_U[0::3, 0] *= -1.0
    bad_S[1::3] *= -1.0
    bad_S[2::3] = np.nan
    out3, rc3 = g.con2prim_entropy(ti, tj, bad_U, bad_S, P[:, 5:8], guess)
    assert np.all(rc3 != 0) and np.array_equal(out3, guess)
    for s in range(0, ns, 11):
        assert orc.con2prim_entropy(bad_U[s], bad_S[s], P[s, 5:8], Gs[s], gam, guess[s])[0] != 0


@pytest.mark.parametrize("metric", [I.METRIC_KS, I.METRIC_MINKOWSKI])
def test_drift_frame_floors_match_oracle(H, orc, metric):
    p = I.torus_params(drift_floors=1) if metric == I.METRIC_KS else \
        I.minkowski_params(n=(8, 8, 8), drift_floors=1, rho_fl_coef=1e-5, u_fl_coef=1e-7)
    ns = 400
    g, rng, ti, tj, x1, x2, C, sc = _zone_setup(H, p, ns, 31 + metric)
    S = _states(rng, ns, sc, C[ti, tj, 8], 3.0, 2.0, 0.0)
    r = np.exp(x1) if metric == I.METRIC_KS else np.ones(ns)
    rfl, ufl = p["rho_fl_coef"] * r ** p["rho_fl_pow"], p["u_fl_coef"] * r ** p["u_fl_pow"]
    Q = S[:, :5].copy()
    Q[0::4, 0] = rfl[0::4] * rng.uniform(1e-3, 0.9, len(Q[0::4]))       # below the density floor
    Q[1::4, 1] = ufl[1::4] * rng.uniform(1e-3, 0.9, len(Q[1::4]))       # below the energy floor
    Q[2::4, 0] = rfl[2::4] * 0.5                                        # below both, and fast: the ceiling follows
    Q[2::4, 1] = -ufl[2::4]
    Q[2::8, 2:5] *= 40.0
    B = S[:, 5:8].copy()
    B[3::8] = 0.0                                                       # no field: the fluid frame
    Q[3::8, 0] = rfl[3::8] * 0.1
    Qn, fl = g.floors_drift(ti, tj, Q, B)
    nhit = np.zeros(3, dtype=int)
    for s in range(ns):
        G = orc.geom_at(p["metric"], p["a"], x1[s], x2[s])
        Pn, c = orc.floors(p, G, r[s], Q[s], B[s])
        assert (fl[s] & 1, (fl[s] >> 1) & 1, (fl[s] >> 2) & 1) == c, (s, fl[s], c)
        nhit += np.array(c)
        assert np.allclose(Qn[s, :2], Pn[:2], rtol=1e-13, atol=0)
        vs = max(np.sqrt(((Pn[2:5] * sc[s]) ** 2).sum()), 1e-6)
        assert (np.abs(Qn[s, 2:5] - Pn[2:5]) * sc[s]).max() <= 1e-12 * vs, (s, Qn[s], Pn)
    assert nhit[0] >= ns // 3 and nhit[1] >= ns // 3 and nhit[2] >= ns // 20, nhit
    # untouched above the floors; a grid without the option applies the fluid-frame floors through the same call
    Q2, fl2 = g.floors_drift(ti, tj, S[:, :5], S[:, 5:8])
    assert np.array_equal(Q2, S[:, :5]) and not fl2.any()
    g0 = H.Grid(dict(p, drift_floors=0))
    Q3, _ = g0.floors_drift(ti, tj, Q, B)
    Q4, _ = g0.floors(ti, tj, Q)
    assert np.array_equal(Q3, Q4)


def _funnel(p):
    """magnetically dominated (b^2 / rho ~ 14), nearly pressureless (u / rho = 1e-9) shear flow: the energy inversion
    returns u < 0 in a third of the zone updates (the recipe of tests/test_oracle_entropy_drift.py)"""
    n = p["n"]
    x, y, z = [(np.arange(m) + 0.5) / m for m in n]
    X, Y, Z = np.meshgrid(x, y, z, indexing="ij")
    rho = 1.0 + 0.3 * np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y)
    u = 1e-9 * (1.0 + 0.2 * np.cos(2 * np.pi * Z))
    u1 = 0.3 * np.sin(2 * np.pi * Y)
    u2 = 0.18 * np.cos(2 * np.pi * (X + Z))
    u3 = 0.12 * np.sin(2 * np.pi * X)
    bface = [np.full((n[0] + 1, n[1], n[2]), 3.0), np.full((n[0], n[1] + 1, n[2]), 1.0),
             np.full((n[0], n[1], n[2] + 1), -2.0)]
    return [rho, u, u1, u2, u3], bface


def _e_scale(P):
    """S-21d: the energy row holds numbers of the size of rho + B^2, and ~12 flux differences of that size, each good
    to one ulp, go into it per stage: where u is far smaller the row fixes it only to ~2e-15 (rho + B^2) in absolute
    terms, and the entropy flux carries that rounding noise from energy-inverted zones into their neighbours.  A
    relative bound of 1e-10 therefore means something down to u ~ 1e-4 (rho + B^2)."""
    return 1e-4 * (P[0] + P[5] ** 2 + P[6] ** 2 + P[7] ** 2)


def _u_error(ref, got):
    return float((np.abs(got[1] - ref[1]) / np.maximum(ref[1], _e_scale(ref))).max())


@pytest.mark.parametrize("drift,n,recon", [(0, (24, 20, 32), I.RECON_PPM), (1, (24, 20, 32), I.RECON_PPM),
                                           (1, (24, 20, 30), I.RECON_PPM), (0, (20, 24, 30), I.RECON_PLM)])
def test_funnel_parity_with_entropy_backup(H, orc, drift, n, recon):
    # n3 = 32: the staged kernels (ring sweeps, warp-per-row x3 sweep, tiled update) with the ninth row; n3 = 30: the
    # generic ones, with PPM and with PLM
    p = I.minkowski_params(n=n, recon=recon, cour=0.5, rho_fl_coef=1e-9, u_fl_coef=1e-13, entropy_backup=1,
                           drift_floors=drift)
    hyd, bf = _funnel(p)
    g, o = _pair(H, orc, p, hyd, bf)
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt
    # the entropy flux of the first flux pass, face by face
    g.debug_emf()
    o.debug_emf()
    gam = p["gamma_ad"]
    ksc = ((gam - 1.0) * hyd[1] / hyd[0] ** gam * hyd[0]).max() * 2.0    # rho kappa u^t, the row's natural size
    for d in range(3):
        a, b = o.get_face(d, 7), g.get_face(d, 7)
        assert np.abs(a - b).max() <= 1e-13 * ksc, (d, np.abs(a - b).max() / ksc)
    nz = int(np.prod(n))
    tot_g = tot_o = 0
    for step, tol in ((1, 1e-10), (2, 1e-8), (3, 1e-7)):
        g.step(1)
        o.step(1)
        Pg, Po = g.get_prims(), o.get_prims()
        # the advected kappa of the last stage, zone by zone (same rounding floor as u, expressed in kappa)
        kg, ko = g.kadv(), o.kadv()
        kfl = (gam - 1.0) * _e_scale(Po) / Po[0] ** gam
        ek = float((np.abs(kg - ko) / np.maximum(np.abs(ko), kfl)).max())
        # zones whose state came from the entropy row in the last stage: u sits on the advected adiabat
        resc_o = np.abs((gam - 1.0) * Po[1] / Po[0] ** gam - ko) <= 1e-9 * np.abs(ko)
        resc_g = np.abs((gam - 1.0) * Pg[1] / Pg[0] ** gam - kg) <= 1e-9 * np.abs(kg)
        assert np.array_equal(resc_o, resc_g) and resc_o.sum() > nz // 20, (step, resc_o.sum(), resc_g.sum())
        e = parity_errors(p, Po, Pg)
        e["u"] = _u_error(Po, Pg)
        print(f"funnel drift={drift} step {step}: {e} kappa {ek:.2e} rescued {resc_o.sum()} of {nz}")
        assert max(e.values()) <= tol and ek <= tol, (step, e, ek)
        sg, so, bg, bo = g.stats(), o.stats(), g.backup_count(), o.backup_count()
        assert sg == so and bg == bo, (step, sg, so, bg, bo)
        assert sg[0] == 0
        tot_g += bg
        tot_o += bo
    assert tot_o > nz // 2                 # PPM: more than one rescue per zone over the three steps, PLM: 0.9
    assert g.divb() <= 1e-12
    for a, b in zip(o.get_bface(), g.get_bface()):
        assert rel_max(a, b) <= 1e-7


def test_torus_with_entropy_backup_and_drift_floors(H, orc):
    """BASELINE cfg 0 with both options: the atmosphere sits at the floors and the energy inversion returns u < 0
    there in hundreds of zone updates, which the entropy row now takes; 1 step <= 1e-10, 10 steps <= 1e-7"""
    p = I.torus_params(entropy_backup=1, drift_floors=1)
    hyd, bf = I.fm_torus(p, seed=0)
    g, o = _pair(H, orc, p, hyd, bf)
    g.step(1)
    o.step(1)
    e1 = parity_errors(p, o.get_prims(), g.get_prims())
    assert max(e1.values()) <= 1e-10, e1
    kg, ko = g.kadv(), o.kadv()
    assert np.abs(kg - ko).max() <= 1e-10 * np.abs(ko).max()
    g.step(9)
    o.step(9)
    e10 = parity_errors(p, o.get_prims(), g.get_prims())
    assert max(e10.values()) <= 1e-7, e10
    sg, so, bg, bo = g.stats(), o.stats(), g.backup_count(), o.backup_count()
    print("torus + NEXT-2: errors", e1, e10, "stats", sg, so, "entropy inversions", bg, bo)
    assert sg[0] == so[0] == 0 and sg[3] == so[3]
    # at the floors a last-bit difference decides whether a zone counts (see test_gpu_parity): counts agree to 2 %
    assert bo > 100 and abs(bg - bo) <= max(3, bo // 50)
    assert g.divb() <= 1e-12


def test_entropy_row_is_passive(H):
    """with no zone in need of the backup the option changes nothing but the kernels that run (their variants that carry
    the ninth row): same primitives as the default grid's to rounding"""
    p = I.minkowski_params(n=(32, 16, 32))
    hyd, bf = I.minkowski_waves(p, seed=2, amp=1e-2)[:2]
    out = []
    for flag in (0, 1):
        g = H.Grid(dict(p, entropy_backup=flag))
        assert g.set_prims(hyd, bf) == 0
        g.step(3)
        out.append(g.get_prims())
        assert g.stats()[0] == 0
        if flag:
            assert g.backup_count() == 0
    e = parity_errors(p, out[0], out[1])
    assert max(e.values()) <= 1e-12, e


def test_cfg2_full_size_with_entropy_backup_and_drift_floors(H, orc):
    """BASELINE cfg 2 (256x128x128 Kerr torus) with both options, in the launch configuration `bench.py --workload cfg2r`
    times: every zone against the oracle after one step and after three, the entropy-inversion count and the ceiling /
    failure counters equal"""
    p = I.torus_params(n=(256, 128, 128), r_out=1000.0, entropy_backup=1, drift_floors=1)
    hyd, bf = I.fm_torus(p, seed=2)
    g, o = _pair(H, orc, p, hyd, bf)
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt
    g.step(1)
    o.step(1)
    e1 = parity_errors(p, o.get_prims(), g.get_prims())
    kg, ko = g.kadv(), o.kadv()
    ek = float(np.abs(kg - ko).max() / np.abs(ko).max())
    print("cfg2 + NEXT-2, 1 step", e1, "advected kappa", ek)
    assert max(e1.values()) <= 1e-10 and ek <= 1e-10, (e1, ek)
    g.step(2)
    o.step(2)
    e3 = parity_errors(p, o.get_prims(), g.get_prims())
    sg, so, bg, bo = g.stats(), o.stats(), g.backup_count(), o.backup_count()
    print("cfg2 + NEXT-2, 3 steps", e3, "stats", sg, so, "entropy inversions", bg, bo)
    assert max(e3.values()) <= 1e-8, e3
    assert sg[0] == so[0] == 0 and sg[3] == so[3]
    # (this torus' atmosphere comes out of the energy inversion below the floors but not below zero: the drift-frame
    # floors act on ~45 % of the zone updates, the entropy inversion on none; it is driven by the other tests)
    assert abs(bg - bo) <= max(3, bo // 50) and abs(sg[2] - so[2]) <= so[2] // 1000 and sg[2] > 10 ** 7
    assert g.divb() <= 1e-12


@pytest.mark.parametrize("regime,tol", [("mild", 1e-12), ("magnetised", 1e-9), ("relativistic", 1e-9)])
def test_aitken_inversion_matches_oracle(H, orc, regime, tol):
    """C-21: the Aitken-accelerated fixed-point inversion zone by zone: round trip, against the oracle's
    from the same guess, from guesses wrong by 1e-6 .. 1e6 (where Newton-Raphson fails for a third), and refusals"""
    p = I.torus_params(entropy_backup=1)
    ns = 300
    g, rng, ti, tj, x1, x2, C, sc = _zone_setup(H, p, ns, 41)
    kw = dict(mild=(1.5, 1.0, 0.0), magnetised=(1.0, 30.0, 0.0), relativistic=(12.0, 3.0, 0.0))[regime]
    P = _states(rng, ns, sc, C[ti, tj, 8], *kw)
    gam = p["gamma_ad"]
    U = g.prim2cons(ti, tj, P)
    Gs = [orc.geom_at(p["metric"], p["a"], x1[s], x2[s]) for s in range(ns)]
    guess = P[:, :5] * (1 + 0.3 * rng.uniform(-1, 1, (ns, 5)))
    out, rc = g.con2prim_aitken(ti, tj, U, P[:, 5:8], guess)
    assert np.all(rc == 0)
    vn = np.sqrt(((P[:, 2:5] * sc) ** 2).sum(axis=1, keepdims=True))
    assert (np.abs(out[:, :2] - P[:, :2]) / P[:, :2]).max() <= tol
    assert (np.abs(out[:, 2:5] - P[:, 2:5]) * sc / np.maximum(vn, 1e-3)).max() <= tol
    worst = 0.0
    for s in range(ns):
        rco, Po, _ = orc.con2prim_aitken(U[s], P[s, 5:8], Gs[s], gam, guess[s])
        assert rco == 0
        worst = max(worst, (np.abs(out[s, :2] - Po[:2]) / Po[:2]).max(),
                    (np.abs(out[s, 2:5] - Po[2:5]) * sc[s]).max() / max(vn[s, 0], 1e-3))
    assert worst <= tol, worst
    # the start is the guess's pressure only
    nfail_newton = 0
    for f in (1e-6, 1e3, 1e6):
        bad = np.zeros((ns, 5))
        bad[:, 0], bad[:, 1] = P[:, 0] * f, P[:, 1] * f
        out2, rc2 = g.con2prim_aitken(ti, tj, U, P[:, 5:8], bad)
        assert np.all(rc2 == 0)
        assert (np.abs(out2[:, :2] - out[:, :2]) / np.abs(out[:, :2])).max() <= 100 * tol
        nfail_newton += int((g.con2prim(ti, tj, U, P[:, 5:8], bad)[1] != 0).sum())
    assert nfail_newton > ns // 10
    # refusals: negative density row, momentum without a real root, NaN: the guess is kept
    Ub = U.copy()
    Ub[0::3, 0] *= -1.0
    Ub[1::3, 2] = 50.0 * C[ti[1::3], tj[1::3], 12] * (np.abs(U[1::3, 0]) + np.abs(U[1::3, 1]) + 1.0) * sc[1::3, 0]
    Ub[2::3, 1] = np.nan
    out3, rc3 = g.con2prim_aitken(ti, tj, Ub, P[:, 5:8], guess)
    assert np.all(rc3 != 0) and np.array_equal(out3, guess)
    for s in range(0, ns, 7):
        assert orc.con2prim_aitken(Ub[s], P[s, 5:8], Gs[s], gam, guess[s])[0] != 0


def test_blast_step_takes_the_whole_inversion_chain(H, orc):
    """a strong blast stepped at 4 x and at 40 x the Courant limit with the robust path on: zones where Newton-Raphson
    does not converge go to the Aitken scheme, what that cannot invert to the entropy row, the rest keeps its source
    state; all three counts and the four event counters equal on both sides, primitives to 1e-10"""
    n = (32, 8, 32)
    p = I.minkowski_params(n=n, entropy_backup=1)
    x = (np.arange(n[0]) + 0.5) / n[0]
    y = (np.arange(n[1]) + 0.5) / n[1]
    core = (np.abs(x - 0.5) < 0.13)[:, None, None] & np.ones(n, dtype=bool)
    rho = np.where(core, 1.0, 1e-3) * (1.0 + 0.05 * np.cos(2 * np.pi * y))[None, :, None]
    u = np.where(core, 1e3, 1e-3) * np.ones(n)
    hyd = [rho, u, np.zeros(n), np.zeros(n), np.zeros(n)]
    seen = np.zeros(3, dtype=int)
    for fac in (4.0, 40.0):
        g, o = _pair(H, orc, p, hyd, None)
        g.dt = fac * g.dt
        o.dt = fac * o.dt
        g.step(1)
        o.step(1)
        cg = (g.stats(), g.aitken_count(), g.backup_count())
        co = (o.stats(), o.aitken_count(), o.backup_count())
        print("blast x", fac, "stats / aitken / entropy:", cg, co)
        assert cg == co
        seen += np.array([co[0][0], co[1], co[2]])
        e = parity_errors(p, o.get_prims(), g.get_prims())
        assert max(e.values()) <= 1e-10, e
    assert seen[0] > 0 and seen[1] > 0 and seen[2] > 0, seen


@pytest.mark.parametrize("case", ["funnel", "torus"])
def test_robust_path_on_a_block_grid(H, orc, case):
    """the entropy row, the backup inversion and the drift-frame floors on a grid cut into blocks that step together (no
    LAT: its registers and correction do not carry the ninth row): the generic block kernels with the ninth row against
    the oracle, whose block-decomposed robust run equals its one-block run bit for bit (tests/test_oracle_entropy_drift.py)"""
    if case == "funnel":
        p = I.minkowski_params(n=(24, 16, 32), nb=(8, 8, 16), cour=0.5, rho_fl_coef=1e-9, u_fl_coef=1e-13, entropy_backup=1,
                               drift_floors=1)
        hyd, bf = _funnel(p)
        steps, tols = 3, (1e-10, 1e-8, 1e-7)
    else:
        p = I.torus_params(n=(32, 16, 16), nb=(8, 8, 8), entropy_backup=1, drift_floors=1)
        hyd, bf = I.fm_torus(p, seed=0)
        steps, tols = 3, (1e-10, 4e-10, 1e-9)
    g, o = _pair(H, orc, p, hyd, bf)
    assert g.num_blocks() == o.num_blocks() > 1
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt
    tot = 0
    for step in range(steps):
        g.step(1)
        o.step(1)
        Pg, Po = g.get_prims(), o.get_prims()
        e = parity_errors(p, Po, Pg)
        if case == "funnel":
            e["u"] = _u_error(Po, Pg)
        sg, so, bg, bo = g.stats(), o.stats(), g.backup_count(), o.backup_count()
        print(f"{case} on blocks, step {step + 1}: {e} stats {sg} {so} entropy inversions {bg} {bo}")
        assert max(e.values()) <= tols[step], (step, e)
        assert sg[0] == so[0] == 0 and sg[3] == so[3]
        if case == "funnel":
            assert sg == so and bg == bo
        else:       # at the floors a last-bit difference decides whether a zone counts (see test_gpu_parity)
            assert abs(bg - bo) <= max(3, bo // 50)
        tot += bo
    assert tot > (np.prod(p["n"]) // 2 if case == "funnel" else 100)
    assert g.divb() <= 1e-12
    for a, b in zip(o.get_bface(), g.get_bface()):
        assert rel_max(a, b) <= 1e-7


@pytest.mark.parametrize("nb", [(0, 0, 0), (8, 4, 16)])
def test_robust_path_with_phi_derefined_rows(H, orc, nb):
    """C-18 / C-19 on a torus whose polar rows are derefined by 4 / 2 / 2 (one block, and blocks stepping together): the
    strided x3 sweep reconstructs kappa of the same groups, the entropy flux goes through the group fix-up"""
    p = I.torus_params(n=(32, 16, 16), nb=nb, deref_theta_deg=(30.0, 12.0), deref_factor=(2, 4), entropy_backup=1, drift_floors=1)
    hyd, bf = I.fm_torus(p, seed=4)
    g, o = _pair(H, orc, p, hyd, bf)
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt
    tot = 0
    for step, tol in ((1, 1e-10), (2, 4e-10), (3, 1e-9)):
        g.step(1)
        o.step(1)
        e = parity_errors(p, o.get_prims(), g.get_prims())
        sg, so, bg, bo = g.stats(), o.stats(), g.backup_count(), o.backup_count()
        print(f"deref + NEXT-2 nb={nb} step {step}: {e} stats {sg} {so} entropy inversions {bg} {bo}")
        assert max(e.values()) <= tol, (step, e)
        assert sg[0] == so[0] == 0 and sg[3] == so[3]
        assert abs(bg - bo) <= max(3, bo // 50)      # at the floors a last-bit difference decides (see test_gpu_parity)
        tot += bo
    assert tot > 100 and g.divb() <= 1e-12
    for a, b in zip(o.get_bface(), g.get_bface()):
        assert rel_max(a, b) <= 1e-7


def test_robust_path_on_a_refined_grid(H, orc):
    """C-18 / C-19 across the x1 refinement interface (blocks stepping together): kappa of the restricted / prolonged ghost
    zones, the fine block's entropy flux taken by the coarse block on the interface face"""
    p = I.torus_params(n=(32, 16, 16), nb=(8, 8, 8), r_refine_max=6.0, entropy_backup=1, drift_floors=1)
    g, o = H.Grid(p), orc.OrcGrid(p)
    infos = []
    for b in range(o.num_blocks()):
        d = o.block_info(b)
        infos.append((d["x_lo"], d["dx"], d["n"]))
    assert len({round(i[1][0], 12) for i in infos}) == 2
    for b, (hyd, bf) in enumerate(I.fm_torus_blocks(p, infos, seed=4)):
        assert g.set_block_prims(b, hyd, bf) == 0 and o.set_block_prims(b, hyd, bf) == 0
    assert g.commit() == 0 and o.commit() == 0
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt
    tot = 0
    for step, tol in ((1, 1e-10), (2, 4e-10), (3, 1e-9)):
        g.step(1)
        o.step(1)
        worst = {}
        for b, (x_lo, dx, n) in enumerate(infos):
            e = parity_errors(I.block_as_grid(p, x_lo, dx, n), o.get_block_prims(b), g.get_block_prims(b))
            for k, v in e.items():
                worst[k] = max(worst.get(k, 0.0), v)
        sg, so, bg, bo = g.stats(), o.stats(), g.backup_count(), o.backup_count()
        print(f"refined + NEXT-2 step {step}: {worst} stats {sg} {so} entropy inversions {bg} {bo}")
        assert max(worst.values()) <= tol, (step, worst)
        assert sg[0] == so[0] == 0 and sg[3] == so[3] and abs(bg - bo) <= max(3, bo // 50)
        tot += bo
    assert tot > 100 and g.divb() <= 1e-12


@pytest.mark.parametrize("case", ["funnel_forced", "torus_courant", "cfg4_features"])
def test_robust_path_under_lat(H, orc, case):
    """C-18 / C-19 / C-21 under local adaptive time-stepping: the registers carry the entropy flux, the correction pass
    corrects the entropy row of the coarse block's boundary zones and inverts them through the same chain (kappa having
    been reset, their entropy row before the correction is density row x kappa of the new primitives).  funnel_forced:
    time levels prescribed in bands (0, 1, 0, 1) on the magnetised funnel, where a third of the zone updates is rescued
    by the entropy row, corrected zones included; torus_courant: Courant-based levels on the torus; cfg4_features:
    blocks + LAT + phi-derefined rows + the x1 refinement level + both options at once"""
    lv = None
    if case == "funnel_forced":
        p = I.minkowski_params(n=(32, 16, 16), nb=(8, 8, 8), lat_max_level=1, cour=0.25, rho_fl_coef=1e-9, u_fl_coef=1e-13,
                               entropy_backup=1, drift_floors=1)
        hyd, bf = _funnel(p)
        tols = (1e-10, 1e-8, 1e-7)
    elif case == "torus_courant":
        p = I.torus_params(n=(32, 16, 16), nb=(8, 8, 8), lat_max_level=1, entropy_backup=1, drift_floors=1)
        hyd, bf = I.fm_torus(p, seed=0)
        tols = (4e-10, 1e-9, 4e-9)
    else:
        p = I.torus_params(n=(32, 16, 16), nb=(8, 4, 16), lat_max_level=1, r_refine_max=4.0, deref_theta_deg=(30.0, 12.0),
                           deref_factor=(2, 4), entropy_backup=1, drift_floors=1)
        tols = (4e-10, 1e-9, 4e-9)
    g, o = H.Grid(p), orc.OrcGrid(p)
    infos = []
    for b in range(o.num_blocks()):
        d = o.block_info(b)
        infos.append((d["x_lo"], d["dx"], d["n"]))
    if case == "funnel_forced":
        lv = [(0, 1, 0, 1)[int(round(x_lo[0] / (dx[0] * n[0]))) % 4] for x_lo, dx, n in infos]
        o.force_levels(lv)
        g.set_levels(lv)
    if case == "cfg4_features":
        for b, (hb, fb) in enumerate(I.fm_torus_blocks(p, infos, seed=4)):
            assert g.set_block_prims(b, hb, fb) == 0 and o.set_block_prims(b, hb, fb) == 0
        assert g.commit() == 0 and o.commit() == 0
    else:
        assert g.set_prims(hyd, bf) == 0 and o.set_prims(hyd, bf) == 0
    assert g.levels() == list(o.levels())
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt
    tot = 0
    for step in range(3):
        g.step(1)
        o.step(1)
        assert g.levels() == list(o.levels())
        worst = {}
        for b, (x_lo, dx, n) in enumerate(infos):
            Po, Pg = o.get_block_prims(b), g.get_block_prims(b)
            e = parity_errors(I.block_as_grid(p, x_lo, dx, n), Po, Pg)
            if case == "funnel_forced":
                e["u"] = _u_error(Po, Pg)
            for k, v in e.items():
                worst[k] = max(worst.get(k, 0.0), v)
        sg, so, bg, bo = g.stats(), o.stats(), g.backup_count(), o.backup_count()
        print(f"{case} step {step + 1}: levels {sorted(set(o.levels()))} {worst} stats {sg} {so} entropy inversions {bg} {bo}")
        assert max(worst.values()) <= tols[step], (step, worst)
        assert sg[0] == so[0] == 0 and sg[3] == so[3]
        if case == "funnel_forced":
            assert sg == so and bg == bo
        else:
            assert abs(bg - bo) <= max(3, bo // 50)
        tot += bo
    assert len(set(o.levels())) > 1 and tot > 100 and g.divb() <= 1e-12


def test_cfg4_full_size_with_entropy_backup_and_drift_floors(H, orc):
    """BASELINE cfg 4 as written (1472 blocks of 16^3: x1 refinement, phi-derefinement 2x / 4x, LAT levels 1 / 2 / 4) with
    both robust options: every zone of every block after one coarse step (4 finest steps), the level assignment equal"""
    import bench
    p, gen, _ = bench.workload("cfg4r")
    g, o = H.Grid(p), orc.OrcGrid(p)
    infos = []
    for b in range(o.num_blocks()):
        d = o.block_info(b)
        infos.append((d["x_lo"], d["dx"], d["n"]))
    assert len(infos) == 1472
    for b, (hb, fb) in enumerate(gen(infos)):
        assert g.set_block_prims(b, hb, fb) == 0 and o.set_block_prims(b, hb, fb) == 0
    assert g.commit() == 0 and o.commit() == 0
    assert g.levels() == list(o.levels()) and sorted(set(o.levels())) == [0, 1, 2]
    g.step(1)
    o.step(1)
    assert g.levels() == list(o.levels())
    worst = {}
    for b, (x_lo, dx, n) in enumerate(infos):
        e = parity_errors(I.block_as_grid(p, x_lo, dx, n), o.get_block_prims(b), g.get_block_prims(b))
        for k, v in e.items():
            worst[k] = max(worst.get(k, 0.0), v)
    sg, so = g.stats(), o.stats()
    print("cfg 4 + NEXT-2, one coarse step:", worst, sg, so, g.backup_count(), o.backup_count())
    assert max(worst.values()) <= 4e-10, worst          # 4 finest steps
    assert sg[0] == so[0] == 0 and sg[3] == so[3] and g.divb() <= 1e-12
