"""Pins for the oracle's transmissive polar boundary.  CPU only.
The ghost zone beyond the pole at (theta_ghost = -theta', phi) IS the zone at (theta', phi + pi).  Checked
against analytic continuation: fields given by formulas that are smooth through the pole (a Cartesian-linear
scalar, the spherical components of a UNIFORM Cartesian vector field) are sampled on the grid; after the
ghost fill every ghost row must hold the formula evaluated at the ghost's own (negative or > pi) theta —
which fixes the half-turn shift and the sign of every component with nothing copied from the implementation."""
import numpy as np
import pytest

from paper_1912_10192_b200 import inputs as I


def _params(n=(8, 8, 16), **kw):
    return I.torus_params(n=n, a=0.0, bc_lo=(I.BC_OUTFLOW, I.BC_POLAR_TRANSMIT, I.BC_PERIODIC),
                          bc_hi=(I.BC_OUTFLOW, I.BC_POLAR_TRANSMIT, I.BC_PERIODIC), **kw)


def _coords(p, stag=-1):
    """padded zone-centre (or face, along stag) coordinates, extended through the poles"""
    xc, xf, dx = I.grid_coords(p)
    n = p["n"]
    ax = []
    for d in range(3):
        lo = (xf[d][0] if d == stag else xc[d][0])
        ax.append(lo + (np.arange(n[d] + 7) - 3) * dx[d])
    return np.meshgrid(np.exp(ax[0]), ax[1], ax[2], indexing="ij")


def test_ghost_rows_are_the_analytic_continuation(orc):
    p = _params()
    n = p["n"]
    o = orc.OrcGrid(p)
    V = np.array([0.3, -0.2, 0.5])                      # a uniform Cartesian vector field

    def sph(r, th, ph):                                 # contravariant (ln r, theta, phi) components, valid for any theta
        st, ct, sp, cp = np.sin(th), np.cos(th), np.sin(ph), np.cos(ph)
        vr = V[0] * st * cp + V[1] * st * sp + V[2] * ct
        vth = (V[0] * ct * cp + V[1] * ct * sp - V[2] * st) / r
        vph = (-V[0] * sp + V[1] * cp) / (r * st)
        return vr / r, vth, vph

    r, th, ph = _coords(p)
    act = (slice(3, 3 + n[0]), slice(3, 3 + n[1]), slice(3, 3 + n[2]))
    rho = 2.0 + 0.01 * r * np.sin(th) * np.cos(ph) + 0.02 * r * np.sin(th) * np.sin(ph)   # linear in x, y
    u1, u2, u3 = sph(r, th, ph)
    full = [rho, 1.0 + 0.0 * rho, u1, u2, u3]
    hyd = [np.ascontiguousarray(f[act]) for f in full]
    assert o.set_prims(hyd, None) == 0
    got = [o.get_padded(c) for c in range(5)]
    gl, gh = slice(0, 3), slice(3 + n[1], 6 + n[1])     # ghost rows below theta = 0 and above theta = pi
    ii, kk = slice(3, 3 + n[0]), slice(0, n[2] + 6)     # all x3 including the periodic ghosts
    for c in (0, 2, 3, 4):
        for rows in (gl, gh):
            a, b = got[c][ii, rows, kk], full[c][ii, rows, kk]
            assert np.abs(a - b).max() <= 1e-13 * np.abs(full[c]).max(), (c, rows)


def test_face_field_ghosts(orc):
    """densitised face fields: Bf1, Bf3 copy (sqrt(-g) uses |sin theta|), Bf2 changes sign, the pole face is 0"""
    p = _params()
    n = p["n"]
    o = orc.OrcGrid(p)
    rng = np.random.default_rng(5)
    bf = [rng.normal(size=tuple(n[e] + (e == d) for e in range(3))) for d in range(3)]
    bf[2][:, :, -1] = bf[2][:, :, 0]
    hyd = [np.ones(n), np.ones(n), np.zeros(n), np.zeros(n), np.zeros(n)]
    assert o.set_prims(hyd, bf) == 0
    h = n[2] // 2
    B1, B2, B3 = (o.get_padded(8 + d) for d in range(3))
    for m in (1, 2, 3):
        for k in range(n[2]):
            ks = (k + h) % n[2]
            assert np.array_equal(B1[3:3 + n[0] + 1, 3 - m, 3 + k], bf[0][:, m - 1, ks])
            assert np.array_equal(B3[3:3 + n[0], 3 - m, 3 + k], bf[2][:, m - 1, ks])
            assert np.array_equal(B2[3:3 + n[0], 3 - m, 3 + k], -bf[1][:, m, ks])
            assert np.array_equal(B2[3:3 + n[0], 3 + n[1] + m, 3 + k], -bf[1][:, n[1] - m, ks])
    assert np.all(B2[3:3 + n[0], 3, 3:3 + n[2]] == 0.0) and np.all(B2[3:3 + n[0], 3 + n[1], 3:3 + n[2]] == 0.0)


def test_axisymmetric_data_reflect_equals_transmit(orc):
    p0 = I.torus_params(n=(16, 16, 8))
    p1 = dict(p0, bc_lo=(I.BC_OUTFLOW, I.BC_POLAR_TRANSMIT, I.BC_PERIODIC), bc_hi=(I.BC_OUTFLOW, I.BC_POLAR_TRANSMIT, I.BC_PERIODIC))
    hyd, bf = I.fm_torus(p0, seed=0, pert=0.0)
    a, b = orc.OrcGrid(p0), orc.OrcGrid(p1)
    assert a.set_prims(hyd, bf) == 0 and b.set_prims(hyd, bf) == 0
    a.step(3)
    b.step(3)
    for x, y in zip(a.get_prims() + a.get_bface(), b.get_prims() + b.get_bface()):
        assert np.array_equal(x, y)


def test_half_turn_equivariance_and_divb(orc):
    """rotating phi-dependent data by half a turn rotates the solution; div B stays at round-off at the poles"""
    p = I.tilted_disk_params(n=(32, 16, 16), bc_lo=(I.BC_OUTFLOW, I.BC_POLAR_TRANSMIT, I.BC_PERIODIC),
                             bc_hi=(I.BC_OUTFLOW, I.BC_POLAR_TRANSMIT, I.BC_PERIODIC))
    hyd, bf = I.tilted_disk(p, seed=3, hr=0.2)
    a, b = orc.OrcGrid(p), orc.OrcGrid(p)
    roll = lambda x, face=False: np.concatenate([np.roll(x[:, :, :-1], 8, axis=2), np.roll(x[:, :, :-1], 8, axis=2)[:, :, :1]], axis=2) if face else np.roll(x, 8, axis=2)
    assert a.set_prims(hyd, bf) == 0
    assert b.set_prims([roll(h) for h in hyd], [roll(bf[0]), roll(bf[1]), roll(bf[2], True)]) == 0
    a.step(4)
    b.step(4)
    for x, y in zip(a.get_prims(), b.get_prims()):
        assert np.abs(roll(x) - y).max() <= 1e-12 * max(np.abs(x).max(), 1e-300)
    assert a.divb() <= 1e-12 and a.stats()[0] == 0


TRANSMIT = dict(bc_lo=(I.BC_OUTFLOW, I.BC_POLAR_TRANSMIT, I.BC_PERIODIC),
                bc_hi=(I.BC_OUTFLOW, I.BC_POLAR_TRANSMIT, I.BC_PERIODIC))


def test_blocks_that_cut_phi_take_the_pole_ghosts_from_the_block_half_a_turn_away(orc):
    """NEXT-1 on blocks that cut x3: the rows beyond the pole lie in ANOTHER block (same x2 row of blocks, half the
    x3 block count further).  Every decomposition must reproduce the single phi-spanning block bit for bit: this
    fixes the partner block, the mirror row, the local x3 index and both signs without reference to the
    implementation of either path.  Tilted disk: the flow and the field cross both poles."""
    n = (16, 16, 32)
    p0 = I.tilted_disk_params(n=n, **TRANSMIT)
    hyd, bf = I.tilted_disk(p0, seed=3, hr=0.2)
    res = []
    for nb in (None, (16, 16, 32), (8, 8, 16), (8, 4, 8), (16, 16, 4)):
        p = p0 if nb is None else dict(p0, nb=nb)
        g = orc.OrcGrid(p)
        assert g.set_prims(hyd, bf) == 0
        g.step(3)
        assert g.divb() <= 1e-12 and g.stats()[0] == 0
        res.append(g.get_prims() + g.get_bface())
    for r in res[1:]:
        for a, b in zip(res[0], r):
            assert np.array_equal(a, b)
    # an odd number of x3 blocks cannot be shifted by half a turn block-wise
    with pytest.raises(RuntimeError):
        orc.OrcGrid(dict(p0, n=(16, 16, 24), nb=(8, 8, 8)))


def _block_data(p, o):
    infos = []
    for b in range(o.num_blocks()):
        d = o.block_info(b)
        infos.append((d["x_lo"], d["dx"], d["n"]))
    return I.fm_torus_blocks(p, infos, seed=4, pert=0.1)


def test_phi_cut_transmit_with_deref_refinement_and_lat(orc):
    """the same identity with everything on: derefined polar rows (group-unit phi ghosts across the pole), one x1
    refinement level (restriction / prolongation in the pole corner) and two time levels"""
    kw = dict(n=(32, 16, 32), lat_max_level=1, deref_theta_deg=(30.0, 12.0), deref_factor=(2, 4),
              r_refine_max=4.0, **TRANSMIT)
    pa, pb = I.torus_params(nb=(8, 4, 16), **kw), I.torus_params(nb=(8, 4, 32), **kw)
    a, b = orc.OrcGrid(pa), orc.OrcGrid(pb)
    assert a.num_blocks() == 2 * b.num_blocks()
    for g, p in ((a, pa), (b, pb)):
        for q, (hyd, bf) in enumerate(_block_data(p, g)):
            assert g.set_block_prims(q, hyd, bf) == 0
        assert g.commit() == 0
    assert any(b.block_info(q)["lev1"] for q in range(b.num_blocks()))
    a.step(2)
    b.step(2)
    assert len(set(a.levels())) == 2
    for q in range(b.num_blocks()):   # b's block q is a's blocks 2q, 2q + 1 side by side in x3
        lo, hi = a.get_block_prims(2 * q), a.get_block_prims(2 * q + 1)
        for x, l, h in zip(b.get_block_prims(q), lo, hi):
            assert np.array_equal(x, np.concatenate([l, h], axis=2))
        lo, hi = a.get_block_bface(2 * q), a.get_block_bface(2 * q + 1)
        for d, (x, l, h) in enumerate(zip(b.get_block_bface(q), lo, hi)):
            assert np.array_equal(x, np.concatenate([l[:, :, :16], h], axis=2))
            if d == 2:
                assert np.array_equal(l[:, :, 16], h[:, :, 0])
    # (faces shared by a coarse and a fine block agree to rounding only: the coarse one is a mean)
    assert a.divb() <= 1e-12 and a.bface_mismatch() <= 1e-12 and a.stats()[0] == 0
