"""Pins P8-P13 for the oracle's grid-level algorithm.  CPU only."""
import numpy as np
import pytest

import os

from paper_1912_10192_b200 import inputs as I


def _golden(name):
    """name -> value pairs of a text fixture under tests/golden/ (each file cites its source)"""
    out = {}
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                k, v = line.split()
                out[k] = float(v)
    return out


def run_to(g, T):
    """advance to exactly t = T, clipping the last step"""
    t = 0.0
    steps = 0
    while t < T * (1 - 1e-13):
        if t + g.dt > T:
            g.dt = T - t
        t, _ = g.step(1)
        steps += 1
    return steps


# ---- P8: constrained transport ---------------------------------------------------------------------------
def test_p8_uniform_flow_edge_emf_equals_centre_emf(orc):
    p = I.minkowski_params(n=(6, 5, 4))
    g = orc.OrcGrid(p)
    n = p["n"]
    ut = np.array([0.3, -0.2, 0.45])
    B = np.array([0.7, 1.1, -0.4])
    hyd = [np.full(n, v) for v in (1.0, 2.0, *ut)]
    bf = [np.full(g._fshape(d), B[d]) for d in range(3)]
    g.set_prims(hyd, bf)
    g.debug_emf()
    v = ut / np.sqrt(1 + ut @ ut)
    Eref = -np.cross(v, B)
    for f in range(3):
        assert np.allclose(g.get_centre_emf(f), Eref[f], rtol=1e-14)
        assert np.allclose(g.get_edge(f), Eref[f], rtol=1e-13, atol=1e-15)


@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("sign", [1.0, -1.0])
def test_p8_grid_aligned_flow_corner_emf_equals_face_emf(orc, axis, sign):
    # data vary along `axis` only; flow along it: each edge EMF equals the 1-D face EMF (G&S 2005)
    rng = np.random.default_rng(20 + axis)
    n = [4, 4, 4]
    n[axis] = 12
    p = I.minkowski_params(n=tuple(n))
    g = orc.OrcGrid(p)
    sh = [1, 1, 1]
    sh[axis] = n[axis]
    prof = lambda lo, hi: np.broadcast_to(rng.uniform(lo, hi, n[axis]).reshape(sh), n).copy()
    hyd = [prof(0.5, 2.0), prof(0.5, 2.0), np.zeros(n), np.zeros(n), np.zeros(n)]
    hyd[2 + axis] = sign * prof(0.2, 0.6)
    e, f = (axis + 1) % 3, (axis + 2) % 3
    hyd[2 + e] = prof(-0.3, 0.3)
    bf = [np.zeros(g._fshape(d)) for d in range(3)]
    bf[axis][:] = 0.8                                    # normal field must be uniform (div B = 0)
    for d in (e, f):
        shf = [1, 1, 1]
        shf[axis] = n[axis]
        bf[d][:] = rng.uniform(-1, 1, n[axis]).reshape(shf)
    g.set_prims(hyd, bf)
    assert g.divb() < 1e-14
    g.debug_emf()
    # on `axis`-faces the face EMFs are E_e (which=5) and E_f (which=6)
    for which, comp in ((5, e), (6, f)):
        face = g.get_face(axis, which)
        edge = g.get_edge(comp)
        # edge array: extent n+1 along the two directions != comp; take the rows that coincide
        sl_face = [slice(None)] * 3
        sl_edge = [slice(None)] * 3
        other = 3 - axis - comp
        sl_edge[other] = slice(0, n[other])
        assert np.allclose(edge[tuple(sl_edge)], face[tuple(sl_face)], rtol=1e-13, atol=1e-15)


# ---- P9/P10: div B and conservation on periodic Minkowski --------------------------------------------------
def test_p9_p10_conservation_and_divb_minkowski(orc):
    p = I.minkowski_params(n=(16, 16, 16))
    hyd, bf = I.minkowski_waves(p, seed=1, amp=1e-2, noise=1e-3)   # nonlinear amplitudes on purpose
    g = orc.OrcGrid(p)
    assert g.set_prims(hyd, bf) == 0
    assert g.divb() < 1e-13
    t0 = g.totals()
    g.step(30)
    t1 = g.totals()
    assert g.divb() < 1e-12
    assert g.stats()[0] == 0
    # mass, energy: relative; momenta (~0 net): absolute against the energy scale
    assert abs(t1[0] - t0[0]) < 1e-13 * abs(t0[0])
    assert abs(t1[1] - t0[1]) < 1e-13 * abs(t0[1])
    assert np.all(np.abs(t1[2:] - t0[2:]) < 1e-13 * abs(t0[1]))
    # face-B sums are conserved by CT as well
    b0 = [b.sum() for b in bf]
    b1 = [b.sum() for b in g.get_bface()]
    assert np.allclose(b0, b1, rtol=1e-13)


# ---- P11: second-order convergence of linear fast + Alfven waves -------------------------------------------
def test_p11_phase_speeds_closed_form():
    em = I.flat_eigenmodes()
    gold = _golden("cfg1_wave_speeds.txt")
    for name in ("fast", "alfven", "slow"):
        assert np.isclose(em[name][0], gold[name], rtol=1e-13), name
    # Alfven mode is incompressible and transverse
    r = em["alfven"][1]
    assert abs(r[0]) < 1e-12 and abs(r[1]) < 1e-12 and abs(r[2:5].sum()) < 1e-12 and abs(r[5:8].sum()) < 1e-12


@pytest.mark.parametrize("modes", [("fast",), ("alfven",)])
def test_p11_linear_wave_convergence(orc, modes):
    T = 0.2
    errs = []
    for N in (16, 32, 64):
        p = I.minkowski_params(n=(N, N, N))
        hyd, bf = I.minkowski_waves(p, amp=1e-6, noise=0.0, modes=modes)
        g = orc.OrcGrid(p)
        g.set_prims(hyd, bf)
        run_to(g, T)
        ref_h, ref_b = I.minkowski_waves(p, amp=1e-6, noise=0.0, modes=modes, t=T)
        P = g.get_prims()
        Bf = g.get_bface()
        e = sum(np.abs(P[c] - ref_h[c]).mean() for c in range(5))
        e += sum(np.abs(Bf[d] - ref_b[d]).mean() for d in range(3))
        errs.append(e / 1e-6)
        assert g.divb() < 1e-12
        g.close()
    o1, o2 = np.log2(errs[0] / errs[1]), np.log2(errs[1] / errs[2])
    assert errs[2] < 1e-2, errs            # summed over 8 fields, relative to the wave amplitude
    assert o2 > 1.9 and o1 > 1.5, (errs, o1, o2)   # N=16 has ~9 zones per wavelength along k


# ---- P12: stationary Fishbone-Moncrief torus ------------------------------------------------------------------
def test_p12_fm_initial_data_identities():
    a, gam = 0.9375, 13.0 / 9.0
    rho, u, ut, uphi, inside, info = I.fm_torus_point(a, gam, np.array([12.0, 9.3]), np.array([np.pi / 2, 1.45]))
    gold = _golden("fm_torus_constants.txt")
    assert np.isclose(info["l"], gold["l"], rtol=1e-13)
    assert np.isclose(info["hmax"] - 1, gold["hmax_m1"], rtol=1e-11)
    assert np.isclose(info["rho_max"], gold["rho_max"], rtol=1e-10)
    assert np.isclose(rho[0], 1.0, rtol=1e-12) and inside.all()
    # u^t u_phi = l everywhere in the torus (constant angular momentum), checked in KS
    g = I.ks_gcov(a, np.array([9.3]), np.array([1.45]))[0]
    ucon = np.array([ut[1], 0.0, 0.0, uphi[1]])
    ucov = g @ ucon
    assert np.isclose(ucon @ ucov, -1.0, rtol=1e-12)
    assert np.isclose(ucon[0] * ucov[3], info["l"], rtol=1e-12)


def _torus_drift(orc, n12, T):
    p = I.torus_params(n=(n12[0], n12[1], 1))
    hyd, bf = I.fm_torus(p, pert=0.0, with_B=False)
    g = orc.OrcGrid(p)
    g.set_prims(hyd, None)
    run_to(g, T)
    P = g.get_prims()
    mask = hyd[0] > 0.1
    fails = g.stats()[0]
    g.close()
    return np.abs(P[0] - hyd[0])[mask].mean(), np.abs(P[3])[mask].mean(), fails


def test_p12_stationary_torus_converges(orc):
    T = 10.0
    d = [_torus_drift(orc, n, T) for n in ((32, 16), (64, 32), (128, 64))]
    assert all(x[2] == 0 for x in d)
    e = [x[0] for x in d]
    o1, o2 = np.log2(e[0] / e[1]), np.log2(e[1] / e[2])
    assert e[2] < 2e-3, e
    assert o2 > 1.8 and o1 > 1.5, (e, o1, o2)


# ---- P13: symmetries ---------------------------------------------------------------------------------------------
def test_p13_axisymmetry_and_equatorial_symmetry(orc):
    p = I.torus_params(n=(24, 16, 4))
    hyd, bf = I.fm_torus(p, pert=0.0)
    # axisymmetric, equatorially symmetric perturbation of the pressure
    xc, _, _ = I.grid_coords(p)
    bump = 1.0 + 0.05 * np.cos(3 * xc[0])[:, None, None] * (np.sin(xc[1]) ** 2)[None, :, None]
    hyd[1] = hyd[1] * bump
    g = orc.OrcGrid(p)
    g.set_prims(hyd, bf)
    g.step(5)
    P = g.get_prims()
    assert g.divb() < 1e-12 and g.stats()[0] == 0
    for c in range(8):
        scale = np.abs(P[c]).max() + 1e-300
        assert np.abs(P[c] - P[c][:, :, :1]).max() <= 1e-13 * scale          # axisymmetry
        sgn = -1.0 if c in (3, 5, 7) else 1.0   # ut^theta, B^r, B^phi odd for an A_phi even about the equator
        assert np.abs(P[c] - sgn * P[c][:, ::-1, :]).max() <= 1e-10 * scale, c  # equatorial symmetry
