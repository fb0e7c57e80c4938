"""Pins P14 for the oracle's phi-derefinement (C-15; the polar rows are
derefined in phi, fluxes and conserved quantities averaged over 2^n cells, the reconstruction adapted to
the larger spacing).  CPU only.  What fixes the reading with nothing to compare against:
 * a grid derefined by m in EVERY row is, zone for zone, the plain grid with N3/m zones (strided stencil,
   in-group interpolation, Courant limit with m dx3, group B_c^3);
 * axisymmetric data do not notice the derefinement;
 * with mixed rows and phi-dependent data the group structure is preserved, div B stays at round-off for
   every FINE zone, and mass / energy / momentum are conserved to round-off on a periodic box."""
import numpy as np
import pytest

from paper_1912_10192_b200 import inputs as I


def _rep_state(hyd, bf, m):
    """coarse-phi state -> fine-phi state obeying the C-15 invariant"""
    H = [np.repeat(h, m, axis=2) for h in hyd]
    B = [np.repeat(bf[0], m, axis=2), np.repeat(bf[1], m, axis=2)]
    n3 = hyd[0].shape[2]
    b3 = np.zeros(bf[2].shape[:2] + (n3 * m + 1,))
    for g in range(n3):
        for r in range(m):
            b3[:, :, g * m + r] = bf[2][:, :, g] + (r / m) * (bf[2][:, :, g + 1] - bf[2][:, :, g])
    b3[:, :, n3 * m] = bf[2][:, :, n3]
    B.append(b3)
    return H, B


@pytest.mark.parametrize("m", [2, 4])
def test_p14_deref_everywhere_is_the_coarse_phi_grid(orc, m):
    pc = I.torus_params(n=(16, 8, 8))
    pf = I.torus_params(n=(16, 8, 8 * m), deref_theta_deg=(91.0,), deref_factor=(m,))
    hyd, bf = I.fm_torus(pc, seed=3)
    # a phi-dependent field as well: shear the torus field by a few steps of evolution first
    c0 = orc.OrcGrid(pc)
    assert c0.set_prims(hyd, bf) == 0
    c0.step(3)
    hyd, bf = c0.get_prims()[:5], c0.get_bface()
    assert np.abs(bf[2]).max() > 0
    c, f = orc.OrcGrid(pc), orc.OrcGrid(pf)
    Hf, Bf = _rep_state(hyd, bf, m)
    assert c.set_prims(hyd, bf) == 0 and f.set_prims(Hf, Bf) == 0
    assert abs(c.dt - f.dt) <= 1e-14 * c.dt
    for _ in range(4):
        tc, _ = c.step(1)
        tf, _ = f.step(1)
    assert abs(tc - tf) <= 1e-13 * tc
    Pc, Pf = c.get_prims(), f.get_prims()
    for a, b in zip(Pc, Pf):
        s = max(np.abs(a).max(), 1e-300)
        for r in range(m):
            assert np.abs(b[:, :, r::m] - a).max() <= 1e-12 * s
    Bc, Bff = c.get_bface(), f.get_bface()
    for d in range(2):
        for r in range(m):
            assert np.abs(Bff[d][:, :, r::m] - Bc[d]).max() <= 1e-12 * np.abs(Bc[d]).max()
    assert np.abs(Bff[2][:, :, ::m] - Bc[2]).max() <= 1e-12 * np.abs(Bc[2]).max()
    assert f.divb() <= 1e-12 and f.stats()[0] == 0


def test_p14_axisymmetric_data_do_not_notice(orc):
    p0 = I.torus_params(n=(16, 16, 16))
    p1 = dict(p0, deref_theta_deg=(30.0, 12.0), deref_factor=(2, 4))
    hyd, bf = I.fm_torus(p0, seed=0, pert=0.0)   # no phi-dependent perturbation
    a, b = orc.OrcGrid(dict(p0, nb=(16, 16, 16))), orc.OrcGrid(p1)
    assert a.set_prims(hyd, bf) == 0 and b.set_prims(hyd, bf) == 0
    assert b.dt > a.dt                       # the derefined polar rows no longer set the Courant step
    for _ in range(3):
        dt = a.dt
        b.dt = dt
        a.step(1)
        b.step(1)
    for x, y in zip(a.get_prims() + a.get_bface(), b.get_prims() + b.get_bface()):
        assert np.abs(x - y).max() <= 1e-13 * max(np.abs(x).max(), 1e-300)


def _group_checks(P, Bf, mrow):
    for j, m in enumerate(mrow):
        if m == 1:
            continue
        for c in range(5):                                   # hydro: exactly uniform
            v = P[c][:, j, :].reshape(P[c].shape[0], -1, m)
            assert np.all(v == v[:, :, :1]), (j, c)
        v = Bf[0][:, j, :].reshape(Bf[0].shape[0], -1, m)    # Bf1: uniform to round-off
        assert np.abs(v - v[:, :, :1]).max() <= 1e-13 * max(np.abs(Bf[0]).max(), 1e-300)
        b3 = Bf[2][:, j, :]
        for r in range(1, m):                                # Bf3: linear inside a group
            lin = b3[:, 0:-1:m] + (r / m) * (b3[:, m::m] - b3[:, 0:-1:m])
            assert np.abs(b3[:, r::m] - lin).max() <= 1e-13 * max(np.abs(Bf[2]).max(), 1e-300)
    for j in range(len(mrow) + 1):                           # Bf2 on face j: the coarser grouping
        M = max(mrow[j - 1] if j > 0 else 1, mrow[j] if j < len(mrow) else 1)
        if M > 1:
            v = Bf[1][:, j, :].reshape(Bf[1].shape[0], -1, M)
            assert np.abs(v - v[:, :, :1]).max() <= 1e-13 * max(np.abs(Bf[1]).max(), 1e-300)


def test_p14_mixed_rows_keep_groups_divb_and_conserve(orc):
    # periodic Minkowski box with the x2 extent standing in for (0, 180 deg): rows 0,1,14,15 m=4; 2,3,12,13 m=2
    n = (8, 16, 16)
    p = I.minkowski_params(n=n, deref_theta_deg=(45.0, 22.6), deref_factor=(2, 4))
    mrow = [4, 4, 2, 2] + [1] * 8 + [2, 2, 4, 4]
    hyd, bf = I.minkowski_waves(p, seed=1, amp=2e-2, noise=1e-2)
    # the face field must obey the invariant on entry: use the uniform background field, keep the hydro waves
    bf = [np.full_like(b, v) for b, v in zip(bf, (1.0, np.sqrt(2.0), 0.5))]
    g = orc.OrcGrid(p)
    assert g.set_prims(hyd, bf) == 0
    t0 = g.totals()
    g.step(6)
    P, Bf = g.get_prims(), g.get_bface()
    _group_checks(P, Bf, mrow)
    assert np.abs(Bf[2] - 0.5).max() > 1e-6                  # the field did evolve
    assert g.divb() <= 1e-12 and g.stats()[0] == 0
    t1 = g.totals()
    scale = max(t0[0], abs(t0[1]))
    assert np.abs(t1 - t0).max() / scale < 1e-13, (t1 - t0) / scale


def test_p14_torus_mixed_rows_with_blocks_and_lat(orc):
    # cfg-4-like: polar rows derefined, blocks in (x1, x2) spanning phi, two LAT levels
    p = I.torus_params(n=(32, 16, 16), nb=(8, 4, 16), lat_max_level=1,
                       deref_theta_deg=(30.0, 12.0), deref_factor=(2, 4))
    mrow = [4, 2, 2] + [1] * 10 + [2, 2, 4]
    hyd, bf = I.fm_torus(p, seed=4)
    g = orc.OrcGrid(p)
    assert g.set_prims(hyd, bf) == 0
    g.step(2)
    _group_checks(g.get_prims(), g.get_bface(), mrow)
    assert g.divb() <= 1e-12 and g.stats()[0] == 0


def test_p14_blocks_that_cut_phi_equal_blocks_that_span_it_bitwise(orc):
    """phi-ghost zones of derefined rows are held in GROUP units and the group invariants are exact, so a grid whose
    blocks cut x3 (BASELINE cfg 4's 16^3 blocks) reproduces the phi-spanning decomposition bit for bit, shared
    faces included; mixed rows (m = 4, 2, 1), phi-dependent data"""
    n = (8, 16, 32)
    res = []
    for nb in ((8, 16, 32), (4, 8, 16), (8, 4, 16)):
        p = I.minkowski_params(n=n, nb=nb, deref_theta_deg=(45.0, 22.6), deref_factor=(2, 4))
        hyd, bf = I.minkowski_waves(p, seed=1, amp=2e-2, noise=1e-2)
        bf = [np.full_like(b, v) for b, v in zip(bf, (1.0, np.sqrt(2.0), 0.5))]
        g = orc.OrcGrid(p)
        assert g.set_prims(hyd, bf) == 0
        t0 = g.totals()
        g.step(5)
        assert np.abs(g.totals() - t0).max() / max(t0[0], abs(t0[1])) < 1e-13
        assert g.divb() <= 1e-12 and g.bface_mismatch() == 0.0
        res.append(g.get_prims() + g.get_bface())
    for r in res[1:]:
        for a, b in zip(res[0], r):
            assert np.array_equal(a, b)


def test_p14_phi_cut_blocks_torus_with_lat(orc):
    p = I.torus_params(n=(32, 16, 32), nb=(8, 4, 16), lat_max_level=1, deref_theta_deg=(30.0, 12.0), deref_factor=(2, 4))
    hyd, bf = I.fm_torus(p, seed=4)
    a, b = orc.OrcGrid(p), orc.OrcGrid(dict(p, nb=(8, 4, 32)))
    assert a.set_prims(hyd, bf) == 0 and b.set_prims(hyd, bf) == 0
    a.step(2)
    b.step(2)
    assert len(set(a.levels())) == 2
    for x, y in zip(a.get_prims() + a.get_bface(), b.get_prims() + b.get_bface()):
        assert np.array_equal(x, y)
    assert a.divb() <= 1e-12 and a.bface_mismatch() == 0.0 and a.stats()[0] == 0
