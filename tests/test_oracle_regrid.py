"""Pins for the oracle's regridding of the x1 refinement level (the x1-only part; DESIGN.md
reading C-20; PAPER.md:71-73 refinement criterion and nesting, PAPER.md:117 divergence-free prolongation and
restriction).  CPU only.
 * regridding onto the same lattice is the identity, bit for bit;
 * refine-then-coarsen returns the state (face field bit for bit, hydro to rounding): restriction inverts prolongation;
 * div B stays at round-off through refinement and coarsening of an arbitrary divergence-free field;
 * data linear in x1 are prolonged and restricted exactly (the limited slope of linear data is the slope);
 * the criterion (maximum density per block column) and the contiguity rule, recomputed in numpy;
 * a torus keeps running after the region has been moved: no failed inversion, div B at round-off."""
import numpy as np
import pytest

from paper_1912_10192_b200 import inputs as I


def _infos(g):
    out = []
    for b in range(g.num_blocks()):
        d = g.block_info(b)
        out.append((d["x_lo"], d["dx"], d["n"]))
    return out


def _set_blocks(g, p, fn):
    for b, (x_lo, dx, n) in enumerate(_infos(g)):
        hyd, bf = fn(I.block_as_grid(p, x_lo, dx, n))
        assert g.set_block_prims(b, hyd, bf) == 0
    assert g.commit() == 0


def _state(g):
    return [(g.get_block_prims(b), g.get_block_bface(b)) for b in range(g.num_blocks())]


def _box(r, **kw):
    # unit cube in 4 x 2 x 2 blocks of 8 x 4 x 4, periodic in x2 / x3; columns with x1-centre < r refined
    d = dict(n=(32, 8, 8), nb=(8, 4, 4), r_refine_max=r)
    d.update(kw)
    return I.minkowski_params(**d)


def _waves(p):
    return lambda pg: I.minkowski_waves(pg, seed=3, amp=5e-2, noise=1e-3, box=(1.0, 1.0, 1.0))[:2]


def test_r1_same_lattice_is_identity(orc):
    p = _box(0.3)
    g = orc.OrcGrid(p)
    _set_blocks(g, p, _waves(p))
    g.step(2)
    h = g.regrid(0.3)
    # (the step is set anew from a flux pass on the transferred state, as after hamr_set_prims: C-14)
    assert h.num_blocks() == g.num_blocks() and h.t == g.t and abs(h.dt - g.dt) < 0.01 * g.dt
    for (Pa, Ba), (Pb, Bb) in zip(_state(g), _state(h)):
        assert all(np.array_equal(a, b) for a, b in zip(Pa, Pb)) and all(np.array_equal(a, b) for a, b in zip(Ba, Bb))


def test_r2_refine_then_coarsen_returns_the_state_and_keeps_divb(orc):
    p = _box(0.3)
    g = orc.OrcGrid(p)
    _set_blocks(g, p, _waves(p))
    g.step(1)
    assert g.divb() <= 1e-12
    h = g.regrid(0.6)                                   # columns 0, 1 refined (was: column 0)
    assert h.num_blocks() == (2 * 2 + 2) * 4 and abs(h.t - g.t) == 0.0
    assert h.divb() <= 1e-12
    lev = {tuple(np.round(d[0], 12)): d for d in _infos(h)}
    assert len(lev) == h.num_blocks()
    k = h.regrid(0.3)                                   # and back
    assert k.num_blocks() == g.num_blocks() and k.divb() <= 1e-12
    for (Pa, Ba), (Pb, Bb) in zip(_state(g), _state(k)):
        for c in range(5):
            assert np.allclose(Pa[c], Pb[c], rtol=4e-16, atol=1e-18)
        for d in range(3):
            assert np.array_equal(Ba[d], Bb[d])
    # coarsening everything and refining again loses what only the fine level held, but not the divergence
    z = g.regrid(0.0)
    assert z.num_blocks() == 16 and z.divb() <= 1e-12
    assert z.regrid(0.9).divb() <= 1e-12


def test_r3_linear_data_are_transferred_exactly(orc):
    p = _box(0.3, bc_lo=(I.BC_OUTFLOW, I.BC_PERIODIC, I.BC_PERIODIC), bc_hi=(I.BC_OUTFLOW, I.BC_PERIODIC, I.BC_PERIODIC))
    g = orc.OrcGrid(p)

    def lin(pg):
        n = pg["n"]
        xc, xf, dx = I.grid_coords(pg)
        X = np.broadcast_to(xc[0][:, None, None], n)
        Xf = np.broadcast_to(xf[0][:, None, None], (n[0] + 1, n[1], n[2]))
        hyd = [1.0 + 0.5 * X, 2.0 - 0.3 * X, 0.1 * X, 0.05 + 0.02 * X, -0.03 * X]
        bf = [np.full(Xf.shape, 0.7), 0.2 + 0.1 * np.broadcast_to(xc[0][:, None, None], (n[0], n[1] + 1, n[2])),
              -0.4 * np.broadcast_to(xc[0][:, None, None], (n[0], n[1], n[2] + 1))]
        return hyd, bf
    _set_blocks(g, p, lin)
    h = g.regrid(0.6)
    for b, (x_lo, dx, n) in enumerate(_infos(h)):
        ref, _ = lin(I.block_as_grid(p, x_lo, dx, n))
        got = h.get_block_prims(b)
        touches_edge = x_lo[0] < 1e-12 or x_lo[0] + n[0] * dx[0] > 1 - 1e-12
        for c in range(5):
            a, r_ = got[c], ref[c]
            if touches_edge:      # the outflow ghost flattens the slope of the zone at the domain edge: skip its children
                a, r_ = a[2:-2], r_[2:-2]
            assert np.allclose(a, r_, rtol=1e-14, atol=1e-15), (b, c)
    # restriction of linear data is exact as well (mean of two symmetric samples)
    k = h.regrid(0.0)
    for b, (x_lo, dx, n) in enumerate(_infos(k)):
        ref, _ = lin(I.block_as_grid(p, x_lo, dx, n))
        got = k.get_block_prims(b)
        for c in range(5):
            a, r_ = got[c], ref[c]
            if x_lo[0] < 0.6:     # columns that went through the (edge-flattened) prolongation: interior zones only
                a, r_ = a[1:-1], r_[1:-1]
            assert np.allclose(a, r_, rtol=1e-14, atol=1e-15), (b, c)


def test_r4_criterion_and_contiguity(orc):
    p = I.torus_params(n=(64, 16, 16), nb=(8, 8, 8))
    g = orc.OrcGrid(p)
    infos = _infos(g)
    data = I.fm_torus_blocks(p, infos, seed=4)
    for b, (hyd, bf) in enumerate(data):
        assert g.set_block_prims(b, hyd, bf) == 0
    assert g.commit() == 0
    lo, hi = np.log(p["xmin"][0]), np.log(p["xmax"][0])
    ncol = 8
    colmax = np.zeros(ncol)
    for b, (x_lo, dx, n) in enumerate(infos):
        col = int(round((x_lo[0] - lo) / ((hi - lo) / ncol)))
        colmax[col] = max(colmax[col], g.get_block_prims(b)[0].max())
    for cut in (0.5, 0.05, 1e-3):
        flagged = np.nonzero(colmax >= cut)[0]
        r = g.refine_radius(cut)
        assert len(flagged) > 0
        want = np.exp(lo + (hi - lo) * (flagged.max() + 1) / ncol)   # every column up to the outermost flagged one
        assert abs(r - want) <= 1e-12 * want, (cut, r, want)
        h = g.regrid(r)
        nfine = sum(d["lev1"] for d in (h.block_info(b) for b in range(h.num_blocks())))
        assert nfine == 2 * (flagged.max() + 1) * 4
    assert g.refine_radius(10.0) == 0.0


@pytest.mark.parametrize("lat", [0, 1])
def test_r5_torus_runs_on_after_a_regrid(orc, lat):
    p = I.torus_params(n=(32, 16, 16), nb=(8, 8, 8), lat_max_level=lat)
    g = orc.OrcGrid(p)
    data = I.fm_torus_blocks(p, _infos(g), seed=4)
    for b, (hyd, bf) in enumerate(data):
        assert g.set_block_prims(b, hyd, bf) == 0
    assert g.commit() == 0
    g.step(1)
    r = g.refine_radius(0.3)
    assert r > p["xmin"][0]
    h = g.regrid(r)
    assert h.num_blocks() > g.num_blocks() and h.divb() <= 1e-12 and h.t == g.t
    h.step(2)
    assert h.stats()[0] == 0 and h.divb() <= 1e-12
    for b in range(h.num_blocks()):
        assert all(np.all(np.isfinite(a)) for a in h.get_block_prims(b))
    k = h.regrid(0.0)                                   # and everything coarse again
    assert k.num_blocks() == g.num_blocks()
    k.step(1)
    assert k.stats()[0] == 0 and k.divb() <= 1e-12


def _block_group_checks(g, mrow_global):
    """the C-15 group structure of every block of a phi-derefined grid (blocks spanning x3): hydro exactly uniform in a
    group, Bf1 / Bf2 uniform, Bf3 linear inside a group (to 1e-13 of the field)"""
    from tests.test_oracle_deref import _group_checks
    for b in range(g.num_blocks()):
        d = g.block_info(b)
        J0 = int(round(d["x_lo"][1] / d["dx"][1]))
        n1 = d["n"][1]
        _group_checks(g.get_block_prims(b), g.get_block_bface(b), mrow_global[J0:J0 + n1])


@pytest.mark.parametrize("lat", [0, 1])
def test_r6_regrid_on_a_phi_derefined_grid(orc, lat):
    """C-20 with C-15 (cfg 4 carries both): the group structure of the derefined polar rows goes through copy, prolongation
    and restriction; the same-lattice regrid stays the identity bit for bit; div B stays at round-off; the torus runs on"""
    p = I.torus_params(n=(32, 16, 16), nb=(8, 4, 16), lat_max_level=lat, deref_theta_deg=(30.0, 12.0), deref_factor=(2, 4))
    mrow = [4, 2, 2] + [1] * 10 + [2, 2, 4]
    g = orc.OrcGrid(p)
    data = I.fm_torus_blocks(p, _infos(g), seed=4)
    for b, (hyd, bf) in enumerate(data):
        assert g.set_block_prims(b, hyd, bf) == 0
    assert g.commit() == 0
    g.step(2)
    _block_group_checks(g, mrow)
    same = g.regrid(0.0)                                # same lattice: identity, bit for bit (the projection included)
    for (Pa, Ba), (Pb, Bb) in zip(_state(g), _state(same)):
        assert all(np.array_equal(a, b) for a, b in zip(Pa, Pb)) and all(np.array_equal(a, b) for a, b in zip(Ba, Bb))
    r = g.refine_radius(0.3)
    assert r > p["xmin"][0]
    h = g.regrid(r)                                     # copy + prolongation
    assert h.num_blocks() > g.num_blocks() and h.t == g.t and h.divb() <= 1e-12
    _block_group_checks(h, mrow)
    k = h.regrid(0.0)                                   # restriction: back on the first lattice
    assert k.num_blocks() == g.num_blocks() and k.divb() <= 1e-12
    _block_group_checks(k, mrow)
    for (Pa, Ba), (Pb, Bb) in zip(_state(g), _state(k)):
        for c in range(5):
            assert np.allclose(Pa[c], Pb[c], rtol=4e-16, atol=1e-18)
        for d in range(3):
            assert np.array_equal(Ba[d], Bb[d])          # restriction inverts prolongation on the face field, bit for bit
    h.step(2)
    assert h.stats()[0] == 0 and h.divb() <= 1e-12
    _block_group_checks(h, mrow)
