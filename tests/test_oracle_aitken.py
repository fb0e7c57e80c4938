"""Pins for the oracle's Aitken-accelerated inversion (reading C-21; "(multi-)dimensional
Newton-Raphson root-finding method (Noble et al. 2006) or Aitken acceleration scheme (Hamlin & Newman 2013; Newman &
Hamlin 2014)").  CPU only.  The function is fixed against the separately pinned primitive -> conserved map (round
trips), against the Newton-Raphson inversion (two different algorithms, one root), against the cubic it solves
(re-evaluated in numpy from the returned state), and on the property the scheme is used for: it does not need a good
guess."""
import numpy as np
import pytest

A_SPIN = 0.9375
GAM = 13.0 / 9.0


def pts(rng, n):
    return [(np.log(rng.uniform(1.3, 40.0)), rng.uniform(0.05, np.pi - 0.05)) for _ in range(n)]


def rand_state(rng, G, umax=1.0, bmax=1.0):
    """the conditioning range of pin P3 (u / rho in [1e-2, 1]); bmax^2 is the largest b^2 / rho"""
    g = G.cov()
    rho = 10.0 ** rng.uniform(-2, 1)
    u = rho * 10.0 ** rng.uniform(-2, 0)
    ut = rng.uniform(-umax, umax, 3) / np.sqrt(np.diag(g)[1:])
    B = rng.uniform(-bmax, bmax, 3) * np.sqrt(rho) / np.sqrt(np.diag(g)[1:]) / G.alpha
    return np.concatenate(([rho, u], ut, B))


def errs(G, P, Pn):
    g = G.cov()
    nrm = np.sqrt(P[2:5] @ g[1:, 1:] @ P[2:5])
    ve = np.max(np.abs(Pn[2:5] - P[2:5]) * np.sqrt(np.diag(g)[1:])) / max(nrm, 1e-3)
    return max(abs(Pn[0] - P[0]) / P[0], abs(Pn[1] - P[1]) / P[1], ve)


@pytest.mark.parametrize("metric", [0, 1])
@pytest.mark.parametrize("regime,tol", [("mild", 1e-12), ("magnetised", 1e-9), ("relativistic", 1e-9)])
def test_a1_roundtrip_and_agreement_with_newton(orc, metric, regime, tol):
    rng = np.random.default_rng(400 + metric)
    kw = dict(mild=dict(umax=1.5), magnetised=dict(umax=1.0, bmax=30.0), relativistic=dict(umax=12.0, bmax=3.0))[regime]
    worst = both = 0.0
    for x1, th in pts(rng, 200):
        G = orc.geom_at(metric, A_SPIN, x1, th)
        P = rand_state(rng, G, **kw)
        U, _ = orc.prim_to_UF(P, G, GAM, 0)
        guess = P[:5] * (1.0 + 0.3 * rng.uniform(-1, 1, 5))
        rc, Pa, it = orc.con2prim_aitken(U[:5], P[5:8], G, GAM, guess)
        assert rc == 0 and it <= 25, (rc, it)
        worst = max(worst, errs(G, P, Pa))
        rcn, Pn, _ = orc.con2prim(U[:5], P[5:8], G, GAM, guess)
        assert rcn == 0
        both = max(both, errs(G, Pn, Pa))
    assert worst <= tol and both <= tol, (worst, both)


def test_a2_returned_state_solves_the_cubic_and_the_pressure_equation(orc):
    """from the returned state alone: eps = W + Bsq satisfies eps^3 - a eps^2 + d = 0 with a, d rebuilt in numpy from
    the conserved rows, and the pressure is (gamma_ad - 1) u"""
    rng = np.random.default_rng(410)
    for x1, th in pts(rng, 60):
        G = orc.geom_at(1, A_SPIN, x1, th)
        P = rand_state(rng, G, umax=2.0, bmax=3.0)
        U, _ = orc.prim_to_UF(P, G, GAM, 0)
        rc, Pa, _ = orc.con2prim_aitken(U[:5], P[5:8], G, GAM, P[:5] * 1.2)
        assert rc == 0
        g, gi, al = G.cov(), G.con(), G.alpha
        Q = al * np.array([U[1] - U[0], U[2], U[3], U[4]]) / G.gdet
        n_up = -al * gi[:, 0]
        e = -(Q @ n_up)
        M2 = Q @ gi @ Q + (Q @ n_up) ** 2
        Bs = al * P[5:8]
        Bsq = Bs @ g[1:, 1:] @ Bs
        T = Q[1:] @ Bs
        lor2 = 1.0 + Pa[2:5] @ g[1:, 1:] @ Pa[2:5]
        W = (Pa[0] + GAM * Pa[1]) * lor2
        eps = W + Bsq
        a = e + (GAM - 1.0) * Pa[1] + 0.5 * Bsq
        d = 0.5 * (M2 * Bsq - T * T)
        assert abs(eps ** 3 - a * eps ** 2 + d) <= 1e-11 * eps ** 3, (eps, a, d)


def test_a3_a_bad_guess_does_not_matter(orc):
    """the iteration starts from the guess's PRESSURE only: guesses wrong by factors up to 1e6 (and with zero velocity)
    give the same root, where the Newton-Raphson scheme from the same guesses fails for part of them"""
    rng = np.random.default_rng(420)
    nfail_newton = 0
    for x1, th in pts(rng, 150):
        G = orc.geom_at(1, A_SPIN, x1, th)
        P = rand_state(rng, G, umax=3.0, bmax=3.0)
        U, _ = orc.prim_to_UF(P, G, GAM, 0)
        ref = orc.con2prim_aitken(U[:5], P[5:8], G, GAM, P[:5])[1]
        for f in (1e-6, 1e-3, 1e3, 1e6):
            guess = np.array([P[0] * f, P[1] * f, 0.0, 0.0, 0.0])
            rc, Pa, it = orc.con2prim_aitken(U[:5], P[5:8], G, GAM, guess)
            assert rc == 0 and it <= 40, (f, rc, it)
            assert errs(G, ref, Pa) <= 1e-10
            nfail_newton += orc.con2prim(U[:5], P[5:8], G, GAM, guess)[0] != 0
    print("Newton-Raphson failures from the same guesses:", nfail_newton, "of", 600)
    assert nfail_newton > 50


def test_a4_refusals(orc):
    G = orc.geom_at(0, 0.0, 0.0, 1.0)
    P = np.array([1.0, 0.5, 0.1, 0.0, 0.0, 0.2, 0.1, 0.0])
    U, _ = orc.prim_to_UF(P, G, GAM, 0)
    assert orc.con2prim_aitken(U[:5], P[5:8], G, GAM, P[:5])[0] == 0
    V = U[:5].copy()
    V[0] = -V[0]                                             # negative density row
    assert orc.con2prim_aitken(V, P[5:8], G, GAM, P[:5])[0] == 2
    V = U[:5].copy()
    V[2] = 50.0 * (abs(U[0]) + abs(U[1]) + 1.0)              # momentum far beyond what the energy allows: no real root
    assert orc.con2prim_aitken(V, P[5:8], G, GAM, P[:5])[0] != 0
    V = U[:5].copy()
    V[1] = np.nan
    assert orc.con2prim_aitken(V, P[5:8], G, GAM, P[:5])[0] == 2
