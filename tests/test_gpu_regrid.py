"""GPU <-> oracle parity of the regridding of the x1 refinement level (the x1-only part;
DESIGN.md C-20): the refinement criterion, the state transfer (copy / prolongation / restriction)
block by block, and the steps that follow on the new lattice, with one global step and with LAT, also on a grid with
phi-derefined polar rows.  Needs a B200."""
import numpy as np
import pytest

from paper_1912_10192_b200 import inputs as I
from tests._parity import parity_errors

pytestmark = pytest.mark.gpu

TOL_1, TOL_10, TOL_DIVB = 1e-10, 1e-7, 1e-12


@pytest.fixture(scope="module")
def H():
    from paper_1912_10192_b200 import build, hamr
    build.build_lib()
    hamr.lib()
    return hamr


def _infos(o):
    out = []
    for b in range(o.num_blocks()):
        d = o.block_info(b)
        out.append((d["x_lo"], d["dx"], d["n"]))
    return out


def _set_both(g, o, data):
    for b, (hyd, bf) in enumerate(data):
        assert g.set_block_prims(b, hyd, bf) == 0 and o.set_block_prims(b, hyd, bf) == 0
    assert g.commit() == 0 and o.commit() == 0


def _check_blocks(p, o, g, tol):
    infos = _infos(o)
    assert g.num_blocks() == len(infos)
    worst = {}
    obf = [o.get_block_bface(b) for b in range(len(infos))]
    scale = max(max(np.abs(a).max() for a in bf) for bf in obf)       # DESIGN.md S-21c
    for b, (x_lo, dx, n) in enumerate(infos):
        lo, dxg, ng, _ = g.block_info(b)
        assert np.allclose(lo, x_lo, rtol=0, atol=1e-13) and np.allclose(dxg, dx, rtol=1e-14) and tuple(ng) == tuple(n)
        pg = I.block_as_grid(p, x_lo, dx, n)
        e = parity_errors(pg, o.get_block_prims(b), g.get_block_prims(b))
        for k, v in e.items():
            worst[k] = max(worst.get(k, 0.0), v)
        for a, c in zip(obf[b], g.get_block_bface(b)):
            assert np.abs(a - c).max() <= tol * max(scale, 1e-300)
    assert max(worst.values()) <= tol, worst
    assert g.divb() <= TOL_DIVB and g.stats()[0] == 0
    return worst


@pytest.mark.parametrize("lat", [0, 1])
def test_torus_regrid_refine_then_coarsen(H, orc, lat):
    """a torus on 4 x 2 x 2 blocks of 8^3, nothing refined: one step, the density criterion picks the columns up to the
    torus, both sides regrid, three steps on the new lattice, then everything coarse again and two more steps"""
    p = I.torus_params(n=(32, 16, 16), nb=(8, 8, 8), lat_max_level=lat)
    g, o = H.Grid(p), orc.OrcGrid(p)
    _set_both(g, o, I.fm_torus_blocks(p, _infos(o), seed=4))
    g.step(1)
    o.step(1)
    rg, ro = g.refine_radius(0.3), o.refine_radius(0.3)
    assert ro > p["xmin"][0] and abs(rg - ro) <= 1e-12 * ro
    assert g.refine_radius(10.0) == 0.0 and o.refine_radius(10.0) == 0.0
    g2, o2 = g.regrid(rg), o.regrid(ro)
    assert g2.num_blocks() == o2.num_blocks() > g.num_blocks()
    assert abs(g2.t - o2.t) <= 1e-13 * o2.t and abs(g2.dt - o2.dt) <= 1e-13 * o2.dt
    if lat:
        assert list(g2.levels()) == list(o2.levels())
    p2 = dict(p, r_refine_max=ro)
    w = _check_blocks(p2, o2, g2, TOL_1)                     # the transferred state itself (one step of history)
    print("after the transfer", w)
    # the old grids are untouched and still usable
    _check_blocks(p, o, g, TOL_1)
    g2.step(3)
    o2.step(3)
    if lat:
        assert list(g2.levels()) == list(o2.levels())
    print("3 steps on the refined lattice", _check_blocks(p2, o2, g2, 4 * TOL_1 if not lat else TOL_10))
    g3, o3 = g2.regrid(0.0), o2.regrid(0.0)
    assert g3.num_blocks() == o3.num_blocks() == g.num_blocks()
    _check_blocks(p, o3, g3, TOL_10)
    g3.step(2)
    o3.step(2)
    print("coarse again + 2 steps", _check_blocks(p, o3, g3, TOL_10))
    for x in (g, g2, g3):
        x.close()


def test_box_regrid_moves_the_region_both_ways(H, orc):
    """periodic-in-x2/x3 unit cube, waves: the refined region grows from one column to two (copy + prolongation in one
    transfer), shrinks back (copy + restriction): the face field returns bit for bit, as in the oracle's own pin"""
    p = I.minkowski_params(n=(32, 8, 8), nb=(8, 4, 4), r_refine_max=0.3)
    g, o = H.Grid(p), orc.OrcGrid(p)
    data = []
    for x_lo, dx, n in _infos(o):
        data.append(I.minkowski_waves(I.block_as_grid(p, x_lo, dx, n), seed=3, amp=5e-2, noise=1e-3, box=(1.0, 1.0, 1.0))[:2])
    _set_both(g, o, data)
    g.step(1)
    o.step(1)
    g2, o2 = g.regrid(0.6), o.regrid(0.6)
    _check_blocks(dict(p, r_refine_max=0.6), o2, g2, TOL_1)
    g3, o3 = g2.regrid(0.3), o2.regrid(0.3)
    _check_blocks(p, o3, g3, TOL_1)
    for b in range(g.num_blocks()):
        for a, c in zip(g.get_block_bface(b), g3.get_block_bface(b)):
            assert np.array_equal(a, c)
    g3.step(2)
    o3.step(2)
    _check_blocks(p, o3, g3, 4 * TOL_1)


def test_regrid_is_refused_where_it_does_not_apply(H):
    mono = H.Grid(I.torus_params())
    hyd, bf = I.fm_torus(I.torus_params(), seed=0)
    assert mono.set_prims(hyd, bf) == 0
    with pytest.raises(H.HamrError):
        mono.regrid(4.0)
    with pytest.raises(H.HamrError):
        mono.refine_radius(0.5)
    p = I.torus_params(n=(32, 16, 16), nb=(8, 8, 8))
    g = H.Grid(p)
    with pytest.raises(H.HamrError):          # no state yet
        g.regrid(4.0)


@pytest.mark.parametrize("lat,n3", [(0, 16), (1, 16), (1, 32)])
def test_regrid_on_a_phi_derefined_grid(H, orc, lat, n3):
    """cfg 4 carries derefined polar rows AND the x1 level: the regrid on such a grid (rows derefined by 4 / 2 / 2; blocks
    that span x3, n3 = 16, or cut it in two, n3 = 32: phi-ghost zones in group units) against the oracle's: transferred
    state, three steps on the refined lattice, back, two more steps"""
    p = I.torus_params(n=(32, 16, n3), nb=(8, 4, 16), lat_max_level=lat, deref_theta_deg=(30.0, 12.0), deref_factor=(2, 4))
    g, o = H.Grid(p), orc.OrcGrid(p)
    _set_both(g, o, I.fm_torus_blocks(p, _infos(o), seed=4))
    g.step(1)
    o.step(1)
    rg, ro = g.refine_radius(0.3), o.refine_radius(0.3)
    assert ro > p["xmin"][0] and abs(rg - ro) <= 1e-12 * ro
    g2, o2 = g.regrid(rg), o.regrid(ro)
    assert g2.num_blocks() == o2.num_blocks() > g.num_blocks()
    assert abs(g2.t - o2.t) <= 1e-13 * o2.t and abs(g2.dt - o2.dt) <= 1e-13 * o2.dt
    if lat:
        assert list(g2.levels()) == list(o2.levels())
    p2 = dict(p, r_refine_max=ro)
    print("after the transfer", _check_blocks(p2, o2, g2, TOL_1))
    g2.step(3)
    o2.step(3)
    if lat:
        assert list(g2.levels()) == list(o2.levels())
    print("3 steps on the refined lattice", _check_blocks(p2, o2, g2, 4 * TOL_1 if not lat else TOL_10))
    g3, o3 = g2.regrid(0.0), o2.regrid(0.0)
    assert g3.num_blocks() == o3.num_blocks() == g.num_blocks()
    _check_blocks(p, o3, g3, TOL_10)
    g3.step(2)
    o3.step(2)
    print("coarse again + 2 steps", _check_blocks(p, o3, g3, TOL_10))
    # the same-lattice regrid of a derefined grid is the identity, bit for bit, on what is evolved: hydro primitives and
    # face field (the cell-centred field is rebuilt from the faces by the commit's division by 2 sqrt(-g), where the update
    # kernel multiplies by the stored reciprocal: one ulp)
    g4 = g3.regrid(0.0)
    for b in range(g3.num_blocks()):
        Pa, Pb = g3.get_block_prims(b), g4.get_block_prims(b)
        assert all(np.array_equal(a, c) for a, c in zip(Pa[:5], Pb[:5]))
        assert all(np.allclose(a, c, rtol=4e-16, atol=0) for a, c in zip(Pa[5:], Pb[5:]))
        assert all(np.array_equal(a, c) for a, c in zip(g3.get_block_bface(b), g4.get_block_bface(b)))
    for x in (g, g2, g3, g4):
        x.close()
