"""Pins P1-P8 for the per-zone pieces of the oracle.  CPU only.

Each pin fixes the oracle against something other than itself: closed forms, invariants, the
independent numpy flat-space system of the input generator, brute-force eigenvalues.
"""
import numpy as np
import pytest

from paper_1912_10192_b200 import inputs as I

A_SPIN = 0.9375


def rand_state(rng, G, orthonormal_scale=True, umax=1.0, bmax=1.0):
    """random primitives in the P3 conditioning range; vector components scaled by 1/sqrt(g_ii)"""
    g = G.cov()
    rho = 10.0 ** rng.uniform(-2, 1)
    u = rho * 10.0 ** rng.uniform(-2, 0)
    ut = rng.uniform(-umax, umax, 3) / np.sqrt(np.diag(g)[1:])
    B = rng.uniform(-bmax, bmax, 3) * np.sqrt(rho) / np.sqrt(np.diag(g)[1:])
    return np.concatenate(([rho, u], ut, B))


def pts(rng, n):
    return [(np.log(rng.uniform(1.3, 40.0)), rng.uniform(0.05, np.pi - 0.05)) for _ in range(n)]


# ---- P1: metric -------------------------------------------------------------------------------------
def test_p1_metric_closed_forms(orc):
    rng = np.random.default_rng(1)
    for x1, th in pts(rng, 50):
        r = np.exp(x1)
        G = orc.geom_at(1, A_SPIN, x1, th)
        g, gi = G.cov(), G.con()
        Sig = r * r + A_SPIN ** 2 * np.cos(th) ** 2
        # determinant: -det g = (r Sigma sin theta)^2 in (t, ln r, theta, phi)
        assert np.isclose(-np.linalg.det(g), (r * Sig * np.sin(th)) ** 2, rtol=1e-12)
        assert np.isclose(G.gdet, r * Sig * abs(np.sin(th)), rtol=1e-14)
        assert np.allclose(g @ gi, np.eye(4), atol=1e-12)
        assert np.allclose(g, g.T) and np.allclose(gi, gi.T)
        # independent numpy restatement used by the input generator
        assert np.allclose(g, I.ks_gcov(A_SPIN, r, th), rtol=1e-14, atol=0)
        # lapse and shift: alpha^2 = Sigma/(Sigma+2r), beta^r = 2r/(Sigma+2r) (divided by r in x1)
        assert np.isclose(G.alpha ** 2, Sig / (Sig + 2 * r), rtol=1e-14)
        assert np.isclose(G.beta[0], 2 * r / (Sig + 2 * r) / r, rtol=1e-14)
        assert G.beta[1] == 0.0 and abs(G.beta[2]) < 1e-16


def test_p1_metric_mirrored_and_minkowski(orc):
    G = orc.geom_at(1, A_SPIN, 1.0, -0.2)
    H = orc.geom_at(1, A_SPIN, 1.0, 0.2)
    assert np.array_equal(G.cov(), H.cov()) and G.gdet == H.gdet
    G = orc.geom_at(1, A_SPIN, 1.0, np.pi + 0.3)
    H = orc.geom_at(1, A_SPIN, 1.0, np.pi - 0.3)
    assert np.allclose(G.cov(), H.cov(), rtol=1e-13)
    M = orc.geom_at(0, 0.0, 0.3, 0.4)
    assert np.array_equal(M.cov(), np.diag([-1.0, 1, 1, 1])) and M.gdet == 1.0 and M.alpha == 1.0
    assert np.all(orc.conn_at(0, 0.0, 0.3, 0.4) == 0.0)


def test_p1_schwarzschild_limit(orc):
    # a = 0: ingoing Eddington-Finkelstein form, g_tt = -(1-2/r), g_tr = 2/r, g_rr = 1+2/r
    r = 7.0
    G = orc.geom_at(1, 0.0, np.log(r), 1.1)
    g = G.cov()
    assert np.isclose(g[0, 0], -(1 - 2 / r)) and np.isclose(g[0, 1], 2 / r * r)
    assert np.isclose(g[1, 1], (1 + 2 / r) * r * r) and np.isclose(g[2, 2], r * r)
    assert np.isclose(g[3, 3], r * r * np.sin(1.1) ** 2) and g[0, 3] == 0.0


# ---- P2: connection ----------------------------------------------------------------------------------
def _fd_dg(orc, x1, x2, k, h):
    e = [0.0, 0.0]
    e[k] = 1.0

    def g(s):
        return orc.geom_at(1, A_SPIN, x1 + s * e[0], x2 + s * e[1]).cov()
    d1 = (g(h) - g(-h)) / (2 * h)
    d2 = (g(h / 2) - g(-h / 2)) / h
    return (4 * d2 - d1) / 3          # Richardson


def test_p2_metric_derivatives_and_connection(orc):
    rng = np.random.default_rng(2)
    for x1, th in pts(rng, 10):
        g, d1, d2 = orc.gcov_derivs(1, A_SPIN, x1, th)
        scale = np.abs(g).max()
        assert np.allclose(d1, _fd_dg(orc, x1, th, 0, 1e-3), atol=2e-9 * scale)
        assert np.allclose(d2, _fd_dg(orc, x1, th, 1, 1e-3), atol=2e-9 * scale)
        # Christoffel symbols rebuilt with numpy from the FD derivatives and numpy's inverse
        dg = np.zeros((4, 4, 4))
        dg[1], dg[2] = _fd_dg(orc, x1, th, 0, 1e-3), _fd_dg(orc, x1, th, 1, 1e-3)
        gi = np.linalg.inv(g)
        ref = 0.5 * (np.einsum("ls,msn->lmn", gi, dg) + np.einsum("ls,nsm->lmn", gi, dg)
                     - np.einsum("ls,smn->lmn", gi, dg))
        conn = orc.conn_at(1, A_SPIN, x1, th)
        assert np.allclose(conn, ref, atol=1e-8 * max(1.0, np.abs(ref).max()))
        assert np.allclose(conn, conn.transpose(0, 2, 1), atol=1e-14 * np.abs(conn).max())
        # metric compatibility contracted: Gamma^m_{m n} = d_n ln sqrt(-g)
        lng = lambda a, b: np.log(orc.geom_at(1, A_SPIN, a, b).gdet)
        h = 1e-5
        assert np.isclose(np.einsum("mmn->n", conn)[1], (lng(x1 + h, th) - lng(x1 - h, th)) / (2 * h), atol=1e-8)
        assert np.isclose(np.einsum("mmn->n", conn)[2], (lng(x1, th + h) - lng(x1, th - h)) / (2 * h), atol=1e-8)


def test_p2_source_vanishes_along_killing_directions(orc):
    # stationary + axisymmetric: T^k_l Gamma^l_{nu k} = 1/2 T^{kl} d_nu g_kl = 0 for nu = t, phi
    rng = np.random.default_rng(3)
    gam = 13.0 / 9.0
    for x1, th in pts(rng, 40):
        G = orc.geom_at(1, A_SPIN, x1, th)
        conn = orc.conn_at(1, A_SPIN, x1, th)
        P = rand_state(rng, G)
        S = orc.source(P, G, conn, gam)
        U, _ = orc.prim_to_UF(P, G, gam, 1)
        scale = np.abs(S).max() + 1e-300
        assert S[0] == 0.0
        assert abs(S[1]) < 1e-12 * scale and abs(S[4]) < 1e-12 * scale
        assert abs(S[2]) > 1e-6 * scale or abs(S[3]) > 1e-6 * scale


def test_p2_source_equals_half_T_dg(orc):
    # S_nu = sqrt(-g) * 1/2 T^{kl} d_nu g_kl with T^{kl} raised by numpy from the oracle's own
    # T^k_l (= F rows / gdet minus the mass flux), FD metric derivative
    rng = np.random.default_rng(4)
    gam = 13.0 / 9.0
    for x1, th in pts(rng, 10):
        G = orc.geom_at(1, A_SPIN, x1, th)
        P = rand_state(rng, G)
        Tmix = np.zeros((4, 4))
        U, _ = orc.prim_to_UF(P, G, gam, 0)
        Tmix[0] = [U[1] - U[0], U[2], U[3], U[4]]
        for d in (1, 2, 3):
            _, F = orc.prim_to_UF(P, G, gam, d)
            Tmix[d] = [F[1] - F[0], F[2], F[3], F[4]]
        Tmix /= G.gdet
        Tup = Tmix @ G.con()
        assert np.allclose(Tup, Tup.T, atol=1e-11 * np.abs(Tup).max())     # T^{kl} symmetric
        S = orc.source(P, G, orc.conn_at(1, A_SPIN, x1, th), gam)
        for nu, k in ((2, 0), (3, 1)):
            ref = G.gdet * 0.5 * np.sum(Tup * _fd_dg(orc, x1, th, k, 1e-3))
            assert np.isclose(S[nu], ref, rtol=1e-7, atol=1e-9 * np.abs(S).max())


# ---- P3/P4: state, conserved variables, inversion -------------------------------------------------------
def test_p3_state_invariants(orc):
    rng = np.random.default_rng(5)
    for x1, th in pts(rng, 40):
        G = orc.geom_at(1, A_SPIN, x1, th)
        P = rand_state(rng, G)
        s = orc.state(P, G)
        assert np.isclose(s["ucon"] @ s["ucov"], -1.0, rtol=1e-12)
        assert abs(s["bcon"] @ s["ucov"]) < 1e-12 * (np.abs(s["bcon"]).max() * np.abs(s["ucov"]).max() + 1e-300)
        assert np.isclose(s["bsq"], s["bcon"] @ G.cov() @ s["bcon"], rtol=1e-12)
        # normal-observer Lorentz factor: gamma = alpha u^t; ut^i is purely spatial-projected
        assert np.isclose(s["ucon"][0] * G.alpha, np.sqrt(1 + P[2:5] @ G.cov()[1:, 1:] @ P[2:5]), rtol=1e-13)


def test_p3_flat_space_U_F_match_independent_system(orc):
    # the generator's numpy flat-space system (complex-step capable) is an independent statement
    rng = np.random.default_rng(6)
    G = orc.geom_at(0, 0.0, 0.0, 0.0)
    gam = 4.0 / 3.0
    for _ in range(40):
        P = rand_state(rng, G, umax=2.0)
        for d in (1, 2, 3):
            nvec = np.zeros(3)
            nvec[d - 1] = 1.0
            Uref, Fref = I._flat_UF(P.astype(np.complex128), gam, nvec)
            U, F = orc.prim_to_UF(P, G, gam, d)
            # oracle rows: (D, T^t_t + D, T^t_i, B^i); T^t_t = -E  -> row 1 = -(E - D)
            assert np.isclose(U[0], Uref[0].real, rtol=1e-13)
            assert np.isclose(U[1], -Uref[1].real, rtol=1e-12, atol=1e-13)
            assert np.allclose(U[2:8], Uref[2:8].real, rtol=1e-12, atol=1e-13)
            assert np.isclose(F[0], Fref[0].real, rtol=1e-12, atol=1e-14)
            assert np.isclose(F[1], -Fref[1].real, rtol=1e-12, atol=1e-13)
            assert np.allclose(F[2:8], Fref[2:8].real, rtol=1e-12, atol=1e-13)
            assert F[4 + d] == 0.0


@pytest.mark.parametrize("metric", [0, 1])
def test_p3_prim_cons_prim_roundtrip(orc, metric):
    rng = np.random.default_rng(7 + metric)
    gam = 13.0 / 9.0
    worst = 0.0
    for x1, th in pts(rng, 300):
        G = orc.geom_at(metric, A_SPIN, x1, th)
        P = rand_state(rng, G, umax=1.5)
        U, _ = orc.prim_to_UF(P, G, gam, 0)
        guess = P[:5] * (1.0 + 0.05 * rng.uniform(-1, 1, 5))
        rc, Pn, it = orc.con2prim(U[:5], P[5:8], G, gam, guess)
        assert rc == 0 and it <= 12
        g = G.cov()
        err = max(abs(Pn[0] - P[0]) / P[0], abs(Pn[1] - P[1]) / P[1])
        nrm = np.sqrt(P[2:5] @ g[1:, 1:] @ P[2:5])
        verr = np.max(np.abs(Pn[2:5] - P[2:5]) * np.sqrt(np.diag(g)[1:])) / max(nrm, 1e-3)
        worst = max(worst, err, verr)
    assert worst < 1e-12, worst


def test_p3_roundtrip_independent_of_guess(orc):
    rng = np.random.default_rng(9)
    gam = 13.0 / 9.0
    for x1, th in pts(rng, 30):
        G = orc.geom_at(1, A_SPIN, x1, th)
        P = rand_state(rng, G)
        U, _ = orc.prim_to_UF(P, G, gam, 0)
        r1 = orc.con2prim(U[:5], P[5:8], G, gam, P[:5] * 1.05)[1]
        r2 = orc.con2prim(U[:5], P[5:8], G, gam, P[:5] * np.array([0.8, 1.2, 0.9, 1.1, 1.0]))[1]
        assert np.allclose(r1, r2, rtol=1e-12, atol=1e-14)


# ---- P5: reconstruction ---------------------------------------------------------------------------------
def test_p5_ppm_plm(orc):
    rng = np.random.default_rng(10)
    for _ in range(50):
        c, s = rng.uniform(-3, 3, 2)
        lin = c + s * np.arange(-2, 3)
        aL, aR = orc.ppm_zone(lin)
        assert np.isclose(aL, c - 0.5 * s, atol=1e-14) and np.isclose(aR, c + 0.5 * s, atol=1e-14)
        aL, aR = orc.plm_zone(lin[1:4])
        assert np.isclose(aL, c - 0.5 * s, atol=1e-14) and np.isclose(aR, c + 0.5 * s, atol=1e-14)
        assert orc.ppm_zone(np.full(5, c)) == (c, c)
        assert orc.plm_zone(np.full(3, c)) == (c, c)
        # monotone data: edge values stay within the neighbouring zone averages
        a = np.sort(rng.uniform(-1, 1, 5))
        aL, aR = orc.ppm_zone(a)
        assert a[1] - 1e-15 <= aL <= a[2] <= aR <= a[3] + 1e-15
        aL, aR = orc.plm_zone(a[1:4])
        assert a[1] <= aL <= a[2] <= aR <= a[3]
        # local extremum -> flat
        b = np.array([0.0, 1.0, 2.0, 1.0, 0.0]) * rng.uniform(0.1, 2)
        assert orc.ppm_zone(b) == (b[2], b[2]) and orc.plm_zone(b[1:4]) == (b[2], b[2])
        # mirror symmetry: reversing the stencil swaps the two edges
        a = rng.uniform(-1, 1, 5)
        l1, r1 = orc.ppm_zone(a)
        l2, r2 = orc.ppm_zone(a[::-1].copy())
        assert np.isclose(l1, r2, atol=1e-15) and np.isclose(r1, l2, atol=1e-15)


def test_p5_ppm_parabola_is_fourth_order_on_smooth_data(orc):
    # zone averages of a cubic: the unlimited interface value is exact (textbook PPM property)
    f_int = lambda x: 0.25 * x ** 4 * 0.3 + x ** 3 / 3 * 0.2 + 0.5 * x * x + 2 * x
    h = 0.1
    edges = (np.arange(6) - 2.5) * h + 5.0
    avg = (f_int(edges[1:]) - f_int(edges[:-1])) / h
    f = lambda x: 0.3 * x ** 3 + 0.2 * x ** 2 + x + 2
    aL, aR = orc.ppm_zone(avg)
    assert np.isclose(aL, f(edges[2]), rtol=1e-12) and np.isclose(aR, f(edges[3]), rtol=1e-12)


# ---- P6: signal speeds ----------------------------------------------------------------------------------
def test_p6_wavespeeds_bracket_flat_eigenvalues(orc):
    rng = np.random.default_rng(11)
    G = orc.geom_at(0, 0.0, 0.0, 0.0)
    gam = 4.0 / 3.0
    for trial in range(60):
        P = rand_state(rng, G, umax=1.5)
        d = 1 + trial % 3
        nvec = np.zeros(3)
        nvec[d - 1] = 1.0
        A0, An = np.zeros((8, 8)), np.zeros((8, 8))
        for c in range(8):
            Pp = P.astype(np.complex128)
            Pp[c] += 1e-30j
            U, F = I._flat_UF(Pp, gam, nvec)
            A0[:, c], An[:, c] = U.imag / 1e-30, F.imag / 1e-30
        keep = [c for c in range(8) if c != 4 + d]           # drop the normal-B row/column
        lam = np.linalg.eigvals(np.linalg.solve(A0[np.ix_(keep, keep)], An[np.ix_(keep, keep)])).real
        vmin, vmax = orc.wavespeeds(P, G, gam, d)
        assert vmin <= lam.min() + 1e-9 and lam.max() <= vmax + 1e-9
        assert -1.0 <= vmin <= vmax <= 1.0


def test_p6_static_and_cold_limits(orc):
    G = orc.geom_at(0, 0.0, 0.0, 0.0)
    gam = 4.0 / 3.0
    P = np.array([1.0, 3.0, 0, 0, 0, 1.0, np.sqrt(2.0), 0.5])
    w = 1.0 + 3.0 + 1.0
    bsq = 1.0 + 2.0 + 0.25
    cs2, va2 = gam * 1.0 / w, bsq / (bsq + w)
    cm = np.sqrt(cs2 + va2 - cs2 * va2)
    for d in (1, 2, 3):
        vmin, vmax = orc.wavespeeds(P, G, gam, d)
        assert np.isclose(vmax, cm, rtol=1e-14) and np.isclose(vmin, -cm, rtol=1e-14)
    # pressureless, unmagnetised: both roots collapse onto the advection speed
    P = np.array([1.0, 1e-30, 0.3, -0.2, 0.5, 0, 0, 0])
    lor = np.sqrt(1 + 0.09 + 0.04 + 0.25)
    for d in (1, 2, 3):
        vmin, vmax = orc.wavespeeds(P, G, gam, d)
        assert np.isclose(vmin, P[1 + d] / lor, atol=1e-12) and np.isclose(vmax, P[1 + d] / lor, atol=1e-12)


def test_p6_kerr_schild_speeds_are_causal_and_ordered(orc):
    # light-cone bound in coordinates: roots of g^{tt} v^2 - 2 g^{td} v + g^{dd} = 0 bracket them
    rng = np.random.default_rng(12)
    gam = 13.0 / 9.0
    for x1, th in pts(rng, 40):
        G = orc.geom_at(1, A_SPIN, x1, th)
        P = rand_state(rng, G)
        gi = G.con()
        for d in (1, 2, 3):
            vmin, vmax = orc.wavespeeds(P, G, gam, d)
            a, b, c = gi[0, 0], -2 * gi[0, d], gi[d, d]
            disc = np.sqrt(b * b - 4 * a * c)
            lo, hi = sorted([(-b + disc) / (2 * a), (-b - disc) / (2 * a)])
            s = orc.state(P, G)
            vadv = s["ucon"][d] / s["ucon"][0]
            assert lo - 1e-12 <= vmin <= vadv <= vmax <= hi + 1e-12


# ---- P7: HLL --------------------------------------------------------------------------------------------
def test_p7_hll(orc):
    rng = np.random.default_rng(13)
    UL, UR, FL, FR = (rng.uniform(-1, 1, 8) for _ in range(4))
    assert np.allclose(orc.hll(UL, UL, FL, FL, 0.3, 0.7), FL, atol=1e-15)       # L = R
    assert np.allclose(orc.hll(UL, UR, FL, FR, 0.0, 0.9), FL, atol=1e-15)       # all waves move right
    assert np.allclose(orc.hll(UL, UR, FL, FR, 0.9, 0.0), FR, atol=1e-15)       # all waves move left
    assert np.allclose(orc.hll(UL, UR, FL, FR, 0.0, 0.0), 0.5 * (FL + FR))      # degenerate fan
    F = orc.hll(UL, UR, FL, FR, 0.4, 0.6)
    assert np.allclose(F, (0.6 * FL + 0.4 * FR - 0.24 * (UR - UL)) / 1.0, atol=1e-15)
    # Rankine-Hugoniot: an isolated jump moving at speed s is captured exactly when cmax = s
    s = 0.35
    FR2 = FL + s * (UR - UL)
    assert np.allclose(orc.hll(UL, UR, FL, FR2, 0.2, s), FL, atol=1e-14)
    # C-7a: a mass flux at rounding level is flushed to exactly zero
    UL2, UR2 = UL.copy(), UL.copy()
    FL2, FR3 = FL.copy(), FL.copy()
    FL2[0], FR3[0] = 1.0, -1.0 + 1e-14
    assert orc.hll(UL2, UR2, FL2, FR3, 0.5, 0.5)[0] == 0.0
