"""Pins for the oracle functions VERDICT round 1 listed as unpinned: floors and Lorentz-factor
ceiling (C-13), the Courant step (C-14; PAPER.md:93 fn. 2: harmonic sum over the three directions), the
outflow branch of the physical boundary fill (C-12) and the failure path of the inversion (C-13: keep the source
state, count).  Each check is against something the mathematics fixes, written here without the oracle.  CPU only."""
import numpy as np

from paper_1912_10192_b200 import inputs as I


def _ks_gcov_spatial(a, r, th):
    """3x3 spatial block of the Kerr-Schild metric in (ln r, theta, phi), typed from DESIGN.md C-1."""
    s2 = np.sin(th) ** 2
    Sig = r * r + a * a * np.cos(th) ** 2
    f = 2.0 * r / Sig
    g = np.zeros((3, 3))
    g[0, 0] = (1.0 + f) * r * r
    g[0, 2] = g[2, 0] = -a * s2 * (1.0 + f) * r
    g[1, 1] = Sig
    g[2, 2] = s2 * (Sig + a * a * s2 * (1.0 + f))
    return g


# ---- floors and ceiling ------------------------------------------------------------------------------------------
def test_floor_values_are_coef_r_pow_and_counted(orc):
    p = I.torus_params()                               # rho floor 1e-5 r^-1.5, u floor 1e-7 r^-2.5 (BASELINE cfg 0)
    for r, th in ((1.3, 0.4), (7.0, 1.5), (41.0, 2.9)):
        G = orc.geom_at(p["metric"], p["a"], np.log(r), th)
        rfl, ufl = 1e-5 * r ** -1.5, 1e-7 * r ** -2.5
        # both below: both floored to exactly the power law, velocities untouched
        P, c = orc.floors(p, G, r, [0.3 * rfl, -2.0 * ufl, 0.01, -0.02, 0.03])
        assert abs(P[0] - rfl) <= 2e-16 * rfl and abs(P[1] - ufl) <= 2e-16 * ufl and c == (1, 1, 0)
        assert np.array_equal(P[2:], [0.01, -0.02, 0.03])
        # only u below; a value exactly AT the floor is not a hit
        P, c = orc.floors(p, G, r, [P[0], 0.5 * ufl, 0.0, 0.0, 0.0])
        assert c == (0, 1, 0) and abs(P[1] - ufl) <= 2e-16 * ufl
        # above both: bitwise unchanged
        Q = [3.0 * rfl, 7.0 * ufl, 0.1, 0.2, -0.1]
        P, c = orc.floors(p, G, r, Q)
        assert np.array_equal(P, Q) and c == (0, 0, 0)
    # a different exponent or coefficient must show: the floor at r = 10 differs from that at r = 1 by 10^pow
    G1 = orc.geom_at(p["metric"], p["a"], 0.0 + np.log(1.5), 1.0)
    G2 = orc.geom_at(p["metric"], p["a"], np.log(15.0), 1.0)
    P1, _ = orc.floors(p, G1, 1.5, [0.0, 0.0, 0, 0, 0])
    P2, _ = orc.floors(p, G2, 15.0, [0.0, 0.0, 0, 0, 0])
    assert abs(P2[0] / P1[0] - 10.0 ** -1.5) <= 1e-15 and abs(P2[1] / P1[1] - 10.0 ** -2.5) <= 1e-15


def test_lorentz_factor_ceiling_rescales_to_gamma_max_along_the_same_direction(orc):
    p = I.torus_params()
    gmax = p["gamma_max"]
    assert gmax == 50.0                                  # DESIGN.md C-13 reading
    rng = np.random.default_rng(3)
    for r, th in ((2.0, 0.7), (9.0, 1.6), (30.0, 2.5)):
        G = orc.geom_at(p["metric"], p["a"], np.log(r), th)
        gs = _ks_gcov_spatial(p["a"], r, th)
        d = rng.normal(size=3)
        d /= np.sqrt(d @ gs @ d)                         # unit vector in the spatial metric
        for gam in (120.0, 50.0 * (1 + 1e-9), 3.0e3):
            ut = np.sqrt(gam * gam - 1.0) * d            # gamma^2 = 1 + g_ij ut^i ut^j
            P, c = orc.floors(p, G, r, [1.0, 1.0, *ut])
            assert c == (0, 0, 1)
            g_after = np.sqrt(1.0 + P[2:] @ gs @ P[2:])
            assert abs(g_after - gmax) <= 1e-13 * gmax
            # direction preserved: the new vector is a positive multiple of the old one
            lam = P[2:] / ut
            assert np.all(lam > 0) and np.ptp(lam) <= 1e-15 * lam.max()
        ut = np.sqrt(49.0 ** 2 - 1.0) * d                # below the ceiling: bitwise unchanged
        P, c = orc.floors(p, G, r, [1.0, 1.0, *ut])
        assert c == (0, 0, 0) and np.array_equal(P[2:], ut)


def test_floors_are_applied_to_the_result_of_the_inversion_in_a_step(orc):
    # a uniform static gas BELOW both floors: the update leaves it unchanged, the inversion returns it, and only
    # then the floors lift it: after one step every zone holds exactly the floor and every zone was counted twice
    # (predictor and corrector)
    p = I.minkowski_params(n=(4, 4, 4), rho_fl_coef=1e-3, u_fl_coef=1e-4)
    n = p["n"]
    g = orc.OrcGrid(p)
    hyd = [np.full(n, v) for v in (2e-4, 3e-5, 0.0, 0.0, 0.0)]
    assert g.set_prims(hyd, None) == 0
    g.step(1)
    P = g.get_prims()
    assert np.all(P[0] == 1e-3) and np.all(P[1] == 1e-4)
    nz = int(np.prod(n))
    assert g.stats() == (0, 2 * nz, 2 * nz, 0)


# ---- Courant step: harmonic sum, not the minimum ---------------------------------------------------------------
def test_dt_is_the_harmonic_sum_over_directions_on_an_anisotropic_box(orc):
    # static uniform magnetised gas in flat space: the speed bounds are +-c_m in every direction, with
    # c_m^2 = c_s^2 + v_A^2 - c_s^2 v_A^2, c_s^2 = gamma p / w, v_A^2 = b^2 / (b^2 + w) (closed form, C-6), so
    # 1/dt = (c_m / C) sum_d 1/dx^d.  With three different spacings min_d dt_d is 1.8 x larger.
    n = (8, 12, 20)
    p = I.minkowski_params(n=n, cour=0.8)
    gam = p["gamma_ad"]
    rho, u, B = 1.3, 0.9, np.array([0.4, -0.7, 0.2])
    g = orc.OrcGrid(p)
    hyd = [np.full(n, v) for v in (rho, u, 0.0, 0.0, 0.0)]
    bf = [np.full(g._fshape(d), B[d]) for d in range(3)]
    assert g.set_prims(hyd, bf) == 0
    w = rho + gam * u
    b2 = B @ B                                           # static fluid: b^mu = (0, B)
    cs2, va2 = gam * (gam - 1.0) * u / w, b2 / (b2 + w)
    cm = np.sqrt(cs2 + va2 - cs2 * va2)
    dx = 1.0 / np.array(n)
    dt_harm = 0.8 / (cm * np.sum(1.0 / dx))
    dt_min = 0.8 * dx.min() / cm
    assert np.allclose(g.ctop(), cm, rtol=1e-13)
    assert abs(g.dt - dt_harm) <= 1e-13 * dt_harm
    assert dt_min / dt_harm > 1.7                        # the two readings are far apart here
    # the same after a step (the corrector's ctop of step n sets dt of step n + 1)
    g.step(1)
    assert abs(g.dt - dt_harm) <= 1e-12 * dt_harm


# ---- outflow boundary ------------------------------------------------------------------------------------------
def test_outflow_ghosts_copy_the_nearest_active_zone_and_the_boundary_face(orc):
    n = (6, 4, 5)
    p = I.minkowski_params(n=n, bc_lo=(I.BC_OUTFLOW, I.BC_PERIODIC, I.BC_PERIODIC),
                           bc_hi=(I.BC_OUTFLOW, I.BC_PERIODIC, I.BC_PERIODIC))
    g = orc.OrcGrid(p)
    i = np.arange(n[0])[:, None, None]
    j = np.arange(n[1])[None, :, None]
    k = np.arange(n[2])[None, None, :]
    # every variable a different linear profile in x1 (so that "zone 1" or "mirror" instead of "zone 0" shows) plus
    # a transverse pattern (so that a transposed copy shows)
    hyd = [1.0 + 0.1 * (c + 1) * i + 0.01 * j + 0.001 * k + 0.0 * i for c in range(5)]
    hyd[2] = 0.02 * i + 0.001 * j + 0 * k; hyd[3] = -0.01 * i + 0 * j + 0.002 * k; hyd[4] = 0.005 * i + 0 * j + 0 * k
    hyd = [np.broadcast_to(h, n).copy() for h in hyd]
    bf = []
    for d in range(3):
        sh = g._fshape(d)
        ii = np.arange(sh[0])[:, None, None]; jj = np.arange(sh[1])[None, :, None]; kk = np.arange(sh[2])[None, None, :]
        bf.append(np.broadcast_to(0.5 + 0.07 * (d + 1) * ii + 0.003 * jj - 0.002 * kk, sh).copy())
    assert g.set_prims(hyd, bf) == 0
    NG = 3
    for c in range(5):
        a = g.get_padded(c)[:, NG:NG + n[1], NG:NG + n[2]]
        for m in range(1, NG + 1):
            assert np.array_equal(a[NG - m], hyd[c][0]), (c, m)              # low ghosts = zone 0
            assert np.array_equal(a[NG + n[0] - 1 + m], hyd[c][n[0] - 1])    # high ghosts = zone n - 1
    # the face field normal to the boundary: ghost faces beyond the boundary face copy the boundary face
    a = g.get_padded(8)[:, NG:NG + n[1], NG:NG + n[2]]
    for m in range(1, NG + 1):
        assert np.array_equal(a[NG - m], bf[0][0]) and np.array_equal(a[NG + n[0] + m], bf[0][n[0]])
    assert np.array_equal(a[NG:NG + n[0] + 1], bf[0])                        # active faces untouched
    # transverse face fields in the ghost zones copy the nearest active zone's faces
    for d in (1, 2):
        a = g.get_padded(8 + d)
        sl = (slice(None), slice(NG, NG + g._fshape(d)[1]), slice(NG, NG + g._fshape(d)[2]))
        a = a[sl]
        for m in range(1, NG + 1):
            assert np.array_equal(a[NG - m], bf[d][0]) and np.array_equal(a[NG + n[0] - 1 + m], bf[d][n[0] - 1])


# ---- failed inversion --------------------------------------------------------------------------------------------
def test_con2prim_failure_returns_a_code_and_the_step_keeps_the_source_state(orc):
    p = I.minkowski_params(n=(16, 4, 4))
    gam = p["gamma_ad"]
    G = orc.geom_at(0, 0.0, 0.5, 0.5)
    # momentum far beyond what the energy allows (|Q| = 10, energy 1e-3, D = 1): no physical (W, v^2) exists
    rc, out, it = orc.con2prim([1.0, 1e-3 + 1.0 - 1.0, 10.0, 0.0, 0.0], [0.0, 0.0, 0.0], G, gam, [1.0, 1.0, 0.1, 0, 0])
    assert rc != 0
    # a negative conserved density cannot be inverted either
    rc2, _, _ = orc.con2prim([-1.0, 1.0, 0.1, 0.0, 0.0], [0.0, 0.0, 0.0], G, gam, [1.0, 1.0, 0.0, 0, 0])
    assert rc2 != 0
    # and a sound state inverts with code 0 from the same kind of guess
    U, _ = orc.prim_to_UF([1.0, 0.5, 0.2, -0.1, 0.3, 0.3, 0.2, -0.1], G, gam)
    rc3, out3, _ = orc.con2prim(U[:5], [0.3, 0.2, -0.1], G, gam, [1.2, 0.4, 0.1, 0, 0.2])
    assert rc3 == 0 and np.allclose(out3, [1.0, 0.5, 0.2, -0.1, 0.3], rtol=1e-12)
    # in a step: a strong blast evolved with a time step 40 x the Courant limit makes U unphysical in some zones.
    # There both stages fail, each keeps its source state (C-13), so the zone ends the step with its initial hydro
    # primitives bit for bit, and each failure is counted
    n = p["n"]
    g = orc.OrcGrid(p)
    x = (np.arange(n[0]) + 0.5) / n[0]
    rho = np.where(np.abs(x - 0.5) < 0.13, 1.0, 1e-3)[:, None, None] * np.ones(n)
    u = np.where(np.abs(x - 0.5) < 0.13, 1e3, 1e-3)[:, None, None] * np.ones(n)
    hyd = [rho, u, np.zeros(n), np.zeros(n), np.zeros(n)]
    assert g.set_prims(hyd, None) == 0
    g.dt = 40.0 * g.dt
    g.step(1)
    st = g.stats()
    P = g.get_prims()
    same = (P[0] == rho) & (P[1] == u) & (P[2] == 0.0)
    # zones next to a jump of the initial data have a non-zero flux divergence: they can only end the step unchanged
    # if both of their inversions failed and kept the source state (zones deep inside a uniform region stay unchanged
    # for the trivial reason)
    jump = np.zeros(n[0], dtype=bool)
    jump[:-1] |= rho[1:, 0, 0] != rho[:-1, 0, 0]
    jump[1:] |= rho[1:, 0, 0] != rho[:-1, 0, 0]
    kept = same & jump[:, None, None]
    assert kept.any(), "no zone at the jump kept its state: the step did not fail where it must"
    assert st[0] >= 2 * int(kept.sum())
    assert not same.all()
