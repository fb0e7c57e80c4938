"""Pins for the robust-inversion path of the oracle (readings C-18, C-19).  CPU only.

C-18: the entropy row, advected beside the eight others, and the inversion that uses it in place of
the energy row.  C-19: floors that add mass and energy in the drift frame.  Every pin fixes the oracle
against something other than the function under test: round trips through the (separately pinned) primitive ->
conserved map, the conserved rows of arbitrary input re-evaluated from the answer, the exact solution of an
advected contact, telescoping sums, and the invariants the drift-frame reading promises, evaluated in numpy.
"""
import numpy as np
import pytest

from paper_1912_10192_b200 import inputs as I

A_SPIN = 0.9375
GAM = 13.0 / 9.0


def pts(rng, n):
    return [(np.log(rng.uniform(1.3, 40.0)), rng.uniform(0.05, np.pi - 0.05)) for _ in range(n)]


def rand_state(rng, G, umax=1.0, bmax=1.0, cold=0.0):
    """random primitives; bmax^2 is the largest magnetisation b^2 / rho, cold lowers u / rho by 10^-cold"""
    g = G.cov()
    rho = 10.0 ** rng.uniform(-2, 1)
    u = rho * 10.0 ** rng.uniform(-2 - cold, 0 - cold)
    ut = rng.uniform(-umax, umax, 3) / np.sqrt(np.diag(g)[1:])
    B = rng.uniform(-bmax, bmax, 3) * np.sqrt(rho) / np.sqrt(np.diag(g)[1:]) / G.alpha
    return np.concatenate(([rho, u], ut, B))


def vel_err(G, P, Pn):
    g = G.cov()
    nrm = np.sqrt(P[2:5] @ g[1:, 1:] @ P[2:5])
    return np.max(np.abs(Pn[2:5] - P[2:5]) * np.sqrt(np.diag(g)[1:])) / max(nrm, 1e-3)


# ---- E1: the entropy row -------------------------------------------------------------------------------------------
def test_e1_entropy_row(orc):
    rng = np.random.default_rng(101)
    for x1, th in pts(rng, 40):
        G = orc.geom_at(1, A_SPIN, x1, th)
        P = rand_state(rng, G)
        for d in (1, 2, 3):
            US, FS = orc.entropy_UF(P, G, GAM, d)
            U, F = orc.prim_to_UF(P, G, GAM, d)
            # the entropy is carried by the mass: U_S / U_rho = F_S / F_rho = kappa, and kappa = p / rho^gamma
            kap = (GAM - 1.0) * P[1] / P[0] ** GAM
            assert np.isclose(US / U[0], kap, rtol=1e-14) and np.isclose(FS / F[0], kap, rtol=1e-13)
            # adiabatic compression by any factor leaves kappa unchanged: rho -> s rho, u -> s^gamma u
            s = rng.uniform(0.1, 10.0)
            Q = P.copy()
            Q[0], Q[1] = s * P[0], s ** GAM * P[1]
            US2, _ = orc.entropy_UF(Q, G, GAM, d)
            U2, _ = orc.prim_to_UF(Q, G, GAM, d)
            assert np.isclose(US2 / U2[0], kap, rtol=1e-13)


# ---- E2: the entropy inversion ---------------------------------------------------------------------------------------
@pytest.mark.parametrize("metric", [0, 1])
@pytest.mark.parametrize("regime", ["mild", "magnetised", "relativistic", "cold"])
def test_e2_roundtrip(orc, metric, regime):
    rng = np.random.default_rng(200 + metric)
    kw = dict(mild=dict(umax=1.5), magnetised=dict(umax=1.0, bmax=30.0), relativistic=dict(umax=12.0, bmax=3.0),
              cold=dict(umax=1.0, bmax=10.0, cold=6.0))[regime]
    worst = 0.0
    for x1, th in pts(rng, 200):
        G = orc.geom_at(metric, A_SPIN, x1, th)
        P = rand_state(rng, G, **kw)
        U, _ = orc.prim_to_UF(P, G, GAM, 0)
        US, _ = orc.entropy_UF(P, G, GAM, 1)
        guess = P[:5] * (1.0 + 0.3 * rng.uniform(-1, 1, 5))
        rc, Pn, it = orc.con2prim_entropy(U[:5], US, P[5:8], G, GAM, guess)
        assert rc == 0 and it <= 60, (rc, it)
        worst = max(worst, abs(Pn[0] - P[0]) / P[0], abs(Pn[1] - P[1]) / P[1], vel_err(G, P, Pn))
    assert worst < (1e-10 if regime == "relativistic" else 1e-12), worst


def test_e2_energy_row_is_not_read_and_guess_does_not_matter(orc):
    rng = np.random.default_rng(210)
    for x1, th in pts(rng, 30):
        G = orc.geom_at(1, A_SPIN, x1, th)
        P = rand_state(rng, G, bmax=5.0)
        U, _ = orc.prim_to_UF(P, G, GAM, 0)
        US, _ = orc.entropy_UF(P, G, GAM, 1)
        r1 = orc.con2prim_entropy(U[:5], US, P[5:8], G, GAM, P[:5])[1]
        V = U[:5].copy()
        V[1] = -7.0 * abs(U[1]) + 3.0     # an energy row no state has
        r2 = orc.con2prim_entropy(V, US, P[5:8], G, GAM, P[:5])[1]
        assert np.array_equal(r1, r2)
        r3 = orc.con2prim_entropy(U[:5], US, P[5:8], G, GAM, P[:5] * np.array([1, 1, -3.0, 5.0, 0.0]))[1]
        assert np.allclose(r1, r3, rtol=1e-12, atol=1e-14)


def test_e2_agrees_with_the_energy_inversion_on_consistent_input(orc):
    rng = np.random.default_rng(220)
    for x1, th in pts(rng, 100):
        G = orc.geom_at(1, A_SPIN, x1, th)
        P = rand_state(rng, G, umax=1.5)
        U, _ = orc.prim_to_UF(P, G, GAM, 0)
        US, _ = orc.entropy_UF(P, G, GAM, 1)
        rc1, Pe, _ = orc.con2prim(U[:5], P[5:8], G, GAM, P[:5] * 1.02)
        rc2, Ps, _ = orc.con2prim_entropy(U[:5], US, P[5:8], G, GAM, P[:5] * 1.02)
        assert rc1 == 0 and rc2 == 0
        assert np.allclose(Pe[:2], Ps[:2], rtol=1e-11) and vel_err(G, Pe, Ps) < 1e-11


def test_e2_answer_reproduces_arbitrary_conserved_rows(orc):
    """not a round trip: density, momentum and entropy rows drawn at random (no state behind them); the state
    returned must give back exactly those rows through the pinned primitive -> conserved map"""
    rng = np.random.default_rng(230)
    done = 0
    for x1, th in pts(rng, 120):
        G = orc.geom_at(1, A_SPIN, x1, th)
        P = rand_state(rng, G, umax=1.0, bmax=3.0)
        U, _ = orc.prim_to_UF(P, G, GAM, 0)
        US, _ = orc.entropy_UF(P, G, GAM, 1)
        V = U[:5].copy()
        V[0] *= rng.uniform(0.3, 3.0)
        V[2:5] *= rng.uniform(-2.0, 2.0, 3)
        VS = US * rng.uniform(0.1, 10.0)
        rc, Pn, _ = orc.con2prim_entropy(V, VS, P[5:8], G, GAM, P[:5])
        assert rc == 0
        Q = np.concatenate((Pn, P[5:8]))
        W, _ = orc.prim_to_UF(Q, G, GAM, 0)
        WS, _ = orc.entropy_UF(Q, G, GAM, 1)
        scale = np.abs(V[2:5]).max() + abs(V[0])
        # conditioning: the momentum along B is the small difference of terms (1 + b^2/rho) gamma^2 times larger
        lor2 = 1.0 + Pn[2:5] @ G.cov()[1:, 1:] @ Pn[2:5]
        sig = orc.state(Q, G)["bsq"] / Pn[0]
        assert np.isclose(W[0], V[0], rtol=1e-12) and np.isclose(WS, VS, rtol=1e-12)
        assert np.allclose(W[2:5], V[2:5], rtol=5e-15 * lor2 * (1.0 + sig) + 1e-12, atol=1e-12 * scale), (lor2, sig)
        assert Pn[0] > 0 and Pn[1] >= 0
        done += 1
    assert done == 120


def test_e2_rejects_what_has_no_root(orc):
    G = orc.geom_at(0, 0.0, 0.0, 1.0)
    P = np.array([1.0, 0.5, 0.1, 0.0, 0.0, 0.2, 0.1, 0.0])
    U, _ = orc.prim_to_UF(P, G, GAM, 0)
    US, _ = orc.entropy_UF(P, G, GAM, 1)
    assert orc.con2prim_entropy(U[:5] * np.array([-1.0, 1, 1, 1, 1]), US, P[5:8], G, GAM, P[:5])[0] == 2   # D < 0
    assert orc.con2prim_entropy(U[:5], -US, P[5:8], G, GAM, P[:5])[0] == 2                                  # kappa < 0
    assert orc.con2prim_entropy(U[:5], np.nan, P[5:8], G, GAM, P[:5])[0] == 2
    assert orc.con2prim_entropy(U[:5], US, P[5:8], G, GAM, P[:5])[0] == 0


# ---- E3: the advected entropy on the grid ----------------------------------------------------------------------------
def _contact_run(orc, N, T=0.2, v=0.4):
    """a density wave carried at uniform pressure and velocity along x1 (an exact solution): rho(x - v t)"""
    p = I.minkowski_params(n=(N, 4, 4), gamma_ad=5.0 / 3.0, cour=0.4, entropy_backup=1)
    gam, pr = p["gamma_ad"], 1.0
    x = (np.arange(N) + 0.5) / N
    lor = 1.0 / np.sqrt(1.0 - v * v)

    def rho_of(xx):
        return 1.0 + 0.3 * np.sin(2 * np.pi * xx)
    shape = (N, 4, 4)
    hyd = [np.broadcast_to(rho_of(x)[:, None, None], shape).copy(), np.full(shape, pr / (gam - 1.0)),
           np.full(shape, lor * v), np.zeros(shape), np.zeros(shape)]
    g = orc.OrcGrid(p)
    g.set_prims(hyd, None)
    t, base = 0.0, None
    while t < T - 1e-14:
        if t + g.dt > T:
            g.dt = T - t
        base = g.get_prims()
        t = g.step(1)[0]
    kadv = g.kadv()
    new = g.get_prims()
    exact = pr / rho_of(x - v * T) ** gam
    err = np.abs(kadv[:, 0, 0] - exact).mean()
    # what a reset from the new primitives would give: differs from the advected value by truncation error only
    kres = (gam - 1.0) * new[1] / new[0] ** gam
    return g, err, base, new, kadv, np.abs(kres - kadv).max(), lor


def test_e3_entropy_is_advected_to_second_order_and_conserved(orc):
    errs = {}
    for N in (32, 64, 128):
        g, err, base, new, kadv, gap, lor = _contact_run(orc, N)
        errs[N] = err
        assert g.stats()[0] == 0 and g.backup_count() == 0
        # telescoping: the sum of the entropy row over a periodic grid does not change in a step.  D = gamma rho on
        # both sides; the last step started from `base` with kappa reset from it
        gam = 5.0 / 3.0

        def dens(P):
            return np.sqrt(1.0 + P[2] ** 2 + P[3] ** 2 + P[4] ** 2) * P[0]
        s0 = (dens(base) * (gam - 1.0) * base[1] / base[0] ** gam).sum()
        s1 = (dens(new) * kadv).sum()
        assert abs(s1 - s0) <= 2e-13 * abs(s0), (s0, s1)
        assert gap < 40 * err + 1e-12
        g.close()
    assert errs[32] / errs[64] > 3.0 and errs[64] / errs[128] > 3.0, errs
    assert errs[128] < 2e-4, errs


def test_e3_entropy_row_is_passive_while_the_energy_inversion_succeeds(orc):
    p0 = I.minkowski_params(n=(16, 12, 8))
    hyd, bface = I.minkowski_waves(p0, seed=5, amp=1e-2)[:2]
    out = []
    for flag in (0, 1):
        g = orc.OrcGrid(dict(p0, entropy_backup=flag))
        g.set_prims(hyd, bface)
        g.step(2)
        out.append(g.get_prims())
        assert g.stats()[0] == 0
        if flag:
            assert g.backup_count() == 0
        g.close()
    for a, b in zip(*out):
        assert np.array_equal(a, b)


def _funnel(p):
    """a magnetically dominated (b^2 / rho ~ 14), nearly pressureless (u / rho = 1e-9) shear flow: the energy row
    holds u as the difference of numbers 1e9 times larger, so the energy inversion returns u < 0 in a third of the
    zone updates"""
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


def test_e3_backup_rescues_the_funnel(orc):
    p0 = I.minkowski_params(n=(16, 16, 8), cour=0.5, rho_fl_coef=1e-9, u_fl_coef=1e-13)
    hyd, bface = _funnel(p0)
    res = {}
    for flag in (0, 1):
        g = orc.OrcGrid(dict(p0, entropy_backup=flag))
        g.set_prims(hyd, bface)
        g.step(3)
        P = g.get_prims()
        res[flag] = (P, g.stats(), g.backup_count() if flag else 0)
        g.close()
    P0, st0, _ = res[0]
    P1, st1, nb = res[1]
    nz = 16 * 16 * 8
    # without the backup the u-floor has to repair the negative energies (more than one hit per zone over the three
    # steps); with it the entropy inversion takes those zones first and the floor is left with the few whose advected
    # entropy went negative (the entropy row is not positivity preserving at second order)
    assert st0[0] == 0 and st0[2] > nz and nb > nz and st1[0] == 0 and st1[2] < st0[2] // 50, (st0, st1, nb)
    gam = p0["gamma_ad"]
    k_init = (gam - 1.0) * hyd[1] / hyd[0] ** gam
    assert np.all(np.isfinite(P1[0])) and P1[1].min() > 0
    # u stays on or above the adiabat it started from; the floored run has zones four decades below it
    k1 = (gam - 1.0) * P1[1] / P1[0] ** gam
    k0 = (gam - 1.0) * P0[1] / P0[0] ** gam
    assert k1.min() > 0.5 * k_init.min() and k0.min() < 1e-3 * k_init.min(), (k1.min(), k0.min(), k_init.min())


# ---- D: drift-frame floors (C-19) ------------------------------------------------------------------------------------
def _split(G, P, B):
    """normal-observer 3-velocity split along / across the field, in numpy"""
    h = G.cov()[1:, 1:]
    gamma = np.sqrt(1.0 + P[2:5] @ h @ P[2:5])
    v = P[2:5] / gamma
    Bs = G.alpha * np.asarray(B)
    Bn = np.sqrt(Bs @ h @ Bs)
    vpar = (v @ h @ Bs) / Bn
    vperp = v - vpar * Bs / Bn
    return gamma, v, vpar, vperp, h


@pytest.mark.parametrize("metric", [0, 1])
def test_d1_drift_frame_invariants(orc, metric):
    rng = np.random.default_rng(300 + metric)
    p = I.torus_params(drift_floors=1, gamma_max=1e6)
    gam = p["gamma_ad"]
    for x1, th in pts(rng, 200):
        G = orc.geom_at(metric, A_SPIN, x1, th)
        r = np.exp(x1) if metric else 1.0
        rfl, ufl = 1e-5 * r ** -1.5, 1e-7 * r ** -2.5
        S = rand_state(rng, G, umax=3.0, bmax=2.0)
        P = S[:5].copy()
        B = S[5:8]
        case = rng.integers(3)
        if case != 1:
            P[0] = rfl * rng.uniform(1e-3, 0.9)
        if case != 0:
            P[1] = ufl * rng.uniform(1e-3, 0.9)
        if case == 0:
            P[1] = P[0] * 0.1 + ufl
        if case == 1:
            P[0] = rfl * 3.0
        Pn, c = orc.floors(dict(p, metric=metric), G, r, P, B)
        assert c == ((case != 1) * 1, (case != 0) * 1, 0)
        assert Pn[0] == max(P[0], rfl) and Pn[1] == max(P[1], ufl)
        g0, v0, vpar0, vperp0, h = _split(G, P, B)
        g1, v1, vpar1, vperp1, _ = _split(G, Pn, B)
        sc = 1.0 / np.sqrt(np.diag(h))
        # the drift velocity is untouched ...
        assert np.allclose(vperp1 / sc, vperp0 / sc, rtol=0, atol=2e-14 * g0 ** 2)
        # ... and so is the momentum along the field, w gamma^2 v_par
        m0 = (P[0] + gam * P[1]) * g0 ** 2 * vpar0
        m1 = (Pn[0] + gam * Pn[1]) * g1 ** 2 * vpar1
        assert np.isclose(m1, m0, rtol=1e-11, atol=1e-300)
        # heavier fluid, same momentum: slower along the field, never faster overall, same direction
        assert abs(vpar1) <= abs(vpar0) * (1 + 1e-14) and vpar1 * vpar0 >= 0 and g1 <= g0 * (1 + 1e-14)
        # the fluid-frame floors (ut kept) would have multiplied that momentum by w'/w
        Pf, _ = orc.floors(dict(p, metric=metric, drift_floors=0), G, r, P, B)
        assert np.array_equal(Pf[2:5], P[2:5])


def test_d1_limits(orc):
    rng = np.random.default_rng(310)
    p = I.torus_params(drift_floors=1)
    for x1, th in pts(rng, 30):
        G = orc.geom_at(1, A_SPIN, x1, th)
        r = np.exp(x1)
        S = rand_state(rng, G, umax=2.0)
        # above both floors: nothing changes, bit for bit
        Pn, c = orc.floors(p, G, r, S[:5], S[5:8])
        assert np.array_equal(Pn, S[:5]) and c == (0, 0, 0)
        low = S[:5].copy()
        low[0] = 1e-12
        # no field: the drift frame is the fluid frame
        a, _ = orc.floors(p, G, r, low, np.zeros(3))
        b, _ = orc.floors(dict(p, drift_floors=0), G, r, low, S[5:8])
        assert np.array_equal(a, b)
        # velocity across the field only: nothing to slow down (v_par = 0), ut unchanged to rounding
        gcv = G.cov()[1:, 1:]
        B = S[5:8]
        ut = low[2:5] - (low[2:5] @ gcv @ B) / (B @ gcv @ B) * B
        q = np.concatenate((low[:2], ut))
        c2, _ = orc.floors(p, G, r, q, B)
        assert np.allclose(c2[2:5], ut, rtol=1e-12, atol=1e-15 * np.abs(ut).max())
        # velocity along the field only, floor far above the state: the fluid is brought almost to rest
        q = np.concatenate(([1e-14, 1e-16], 2.0 * B / np.sqrt(B @ gcv @ B)))
        c3, _ = orc.floors(p, G, r, q, B)
        assert np.sqrt(c3[2:5] @ gcv @ c3[2:5]) < 1e-3


def test_d1_ceiling_follows_the_drift_floors(orc):
    p = I.minkowski_params(drift_floors=1, gamma_max=5.0, rho_fl_coef=1e-6, u_fl_coef=1e-8)
    G = orc.geom_at(0, 0.0, 0.0, 1.0)
    # fast drift across B (gamma 20): the floors leave it alone, the ceiling then rescales ut to gamma_max
    P = np.array([1e-9, 1e-12, 0.0, np.sqrt(20.0 ** 2 - 1.0), 0.0])
    Pn, c = orc.floors(p, G, 1.0, P, [1.0, 0.0, 0.0])
    assert c == (1, 1, 1) and np.isclose(np.sqrt(1 + Pn[2:5] @ Pn[2:5]), 5.0, rtol=1e-14)
    assert Pn[2] == 0.0 and Pn[4] == 0.0


def test_robust_path_block_decomposition_is_the_one_block_run(orc):
    """C-18 / C-19 on a grid cut into blocks that step together: the ninth row lives per block (kappa of the ghost-filled
    source state, entropy flux on the block's own faces), so the decomposition changes nothing: every primitive bit for
    bit, the same event counters and the same number of entropy inversions (the robust analogue of pin P15)"""
    import numpy as np
    from paper_1912_10192_b200 import inputs as I
    for p, gen in ((dict(I.torus_params(n=(32, 16, 16)), entropy_backup=1, drift_floors=1), lambda q: I.fm_torus(q, seed=0)),):
        hyd, bf = gen(p)
        m = orc.OrcGrid(p)
        b = orc.OrcGrid(dict(p, nb=(8, 8, 8)))
        assert m.set_prims(hyd, bf) == 0 and b.set_prims(hyd, bf) == 0
        m.step(3)
        b.step(3)
        assert b.num_blocks() == 16
        assert all(np.array_equal(x, y) for x, y in zip(m.get_prims(), b.get_prims()))
        assert m.stats() == b.stats() and m.backup_count() == b.backup_count() > 100
        assert b.divb() <= 1e-12


@pytest.mark.parametrize("m", [2, 4])
def test_robust_path_on_a_grid_derefined_everywhere_is_the_coarse_phi_grid(orc, m):
    """C-18 / C-19 with C-15 (the robust analogue of pin P14): a grid derefined by m in EVERY row equals, zone for zone, the
    plain grid with N3 / m zones — the strided x3 stencil reconstructs kappa of the same groups, the entropy flux is one
    more flux of the row (group mean / interpolation) — and every event is counted m times (once per member)"""
    import numpy as np
    from paper_1912_10192_b200 import inputs as I
    from tests.test_oracle_deref import _rep_state
    opt = dict(entropy_backup=1, drift_floors=1)
    pc = dict(I.torus_params(n=(16, 8, 8)), **opt)
    pf = dict(I.torus_params(n=(16, 8, 8 * m), deref_theta_deg=(91.0,), deref_factor=(m,)), **opt)
    hyd, bf = I.fm_torus(pc, seed=3)
    c0 = orc.OrcGrid(pc)                       # a phi-dependent field as well: a few steps of evolution first
    assert c0.set_prims(hyd, bf) == 0
    c0.step(3)
    hyd, bf = c0.get_prims()[:5], c0.get_bface()
    c, f = orc.OrcGrid(pc), orc.OrcGrid(pf)
    Hf, Bf = _rep_state(hyd, bf, m)
    assert c.set_prims(hyd, bf) == 0 and f.set_prims(Hf, Bf) == 0
    c.step(4)
    f.step(4)
    for a, b in zip(c.get_prims(), f.get_prims()):
        s = max(np.abs(a).max(), 1e-300)
        for r in range(m):
            assert np.abs(b[:, :, r::m] - a).max() <= 1e-12 * s
    sc, sf = c.stats(), f.stats()
    assert sc[0] == sf[0] == 0 and sf[3] == m * sc[3]
    bc, bf_ = c.backup_count(), f.backup_count()      # (the counter is read and reset)
    assert bc > 100 and bf_ == m * bc
    assert f.divb() <= 1e-12


def test_entropy_row_telescopes_across_the_refinement_interface(orc):
    """C-18 with C-16: the coarse block takes the fine block's entropy flux on the interface face (as it takes the other
    fluxes), so the volume-weighted sum of the entropy row over a periodic box with a refined column is unchanged by a
    step to round-off; with its OWN flux on that face the sum would move at truncation level (checked: the same sum
    with the coarse side's flux differences is off by > 1e-9 on this data).  D = gamma rho in numpy on both sides."""
    import numpy as np
    from paper_1912_10192_b200 import inputs as I
    gam = 4.0 / 3.0
    p = I.minkowski_params(n=(32, 8, 8), nb=(8, 4, 4), r_refine_max=0.3, entropy_backup=1)
    g = orc.OrcGrid(p)
    infos = [g.block_info(b) for b in range(g.num_blocks())]
    assert len({round(d["dx"][0], 12) for d in infos}) == 2          # both levels present
    for b, d in enumerate(infos):
        hyd, bf = I.minkowski_waves(I.block_as_grid(p, d["x_lo"], d["dx"], d["n"]), seed=3, amp=5e-2, noise=1e-3,
                                    box=(1.0, 1.0, 1.0))[:2]
        assert g.set_block_prims(b, hyd, bf) == 0
    assert g.commit() == 0
    g.step(2)

    def dens(P):
        return np.sqrt(1.0 + P[2] ** 2 + P[3] ** 2 + P[4] ** 2) * P[0]
    base = [g.get_block_prims(b) for b in range(g.num_blocks())]
    g.step(1)                                                        # kappa was reset from `base` before this step
    assert g.stats()[0] == 0 and g.backup_count() == 0
    s0 = s1 = 0.0
    for b, d in enumerate(infos):
        vol = d["dx"][0]                                             # x2, x3 widths are the same on both levels
        P0, P1, ka = base[b], g.get_block_prims(b), g.get_block_kadv(b)
        s0 += vol * (dens(P0) * (gam - 1.0) * P0[1] / P0[0] ** gam).sum()
        s1 += vol * (dens(P1) * ka).sum()
    assert abs(s1 - s0) <= 5e-13 * abs(s0), (s0, s1, (s1 - s0) / s0)
