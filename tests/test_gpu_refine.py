"""GPU <-> oracle parity on grids with the x1 refinement level (DESIGN.md §9 C-16;
PAPER.md:71, 137): restricted / prolonged ghosts across the coarse-fine interface, interface flux and EMF
agreement, alone, with LAT, and with phi-derefinement (the full feature set of BASELINE cfg 4).  Needs a B200."""
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


def _check_blocks(p, infos, o, g, tol):
    worst = {}
    # face fields: one scale for the whole grid (a block, or one component in a block, may hold rounding noise only)
    obf = [o.get_block_bface(b) for b in range(len(infos))]
    scale = max(max(np.abs(a).max() for a in bf) for bf in obf)
    for b, (x_lo, dx, n) in enumerate(infos):
        pg = I.block_as_grid(p, x_lo, dx, n)
        e = parity_errors(pg, o.get_block_prims(b), g.get_block_prims(b))
        for k, v in e.items():
            worst[k] = max(worst.get(k, 0.0), v)
        for a, c in zip(obf[b], g.get_block_bface(b)):
            assert np.abs(a - c).max() <= tol * max(scale, 1e-300)
    assert max(worst.values()) <= tol, worst
    assert g.divb() <= TOL_DIVB and g.stats()[0] == 0


def test_refined_lattice_matches_oracle(H, orc):
    p = I.torus_params(n=(32, 16, 16), nb=(8, 8, 8), r_refine_max=4.0)
    g, o = H.Grid(p), orc.OrcGrid(p)
    assert g.num_blocks() == o.num_blocks() and g.num_blocks() > 4 * 2 * 2
    for b in range(g.num_blocks()):
        lo, dx, n, _ = g.block_info(b)
        d = o.block_info(b)
        assert np.allclose(lo, d["x_lo"], rtol=0, atol=1e-13) and np.allclose(dx, d["dx"], rtol=1e-14) and n == d["n"]


@pytest.mark.parametrize("lat", [0, 1])
def test_refined_minkowski_waves(H, orc, lat):
    p = I.minkowski_params(n=(16, 8, 8), nb=(8, 4, 4), r_refine_max=0.5, lat_max_level=lat)   # 2 interfaces
    g, o = H.Grid(p), orc.OrcGrid(p)
    infos = _infos(o)
    if lat:
        lv = [0 if o.block_info(b)["lev1"] else 1 for b in range(o.num_blocks())]
        o.force_levels(lv)
        g.set_levels(lv)
    data = [I.minkowski_waves(I.block_as_grid(p, *inf), amp=1e-2, noise=0.0, box=(1.0, 1.0, 1.0)) for inf in infos]
    _set_both(g, o, data)
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt
    if lat:
        assert g.levels() == list(o.levels()) and len(set(g.levels())) == 2
    t0 = g.totals()
    g.step(1)
    o.step(1)
    _check_blocks(p, infos, o, g, TOL_1 * (2 if lat else 1))
    g.step(5)
    o.step(5)
    _check_blocks(p, infos, o, g, TOL_10)
    t1 = g.totals()
    assert np.abs(t1 - t0).max() / max(t0[0], abs(t0[1])) < 1e-13   # conservative through both interfaces


@pytest.mark.parametrize("extra", [dict(), dict(lat_max_level=2),
                                   dict(nb=(8, 4, 16), lat_max_level=1, deref_theta_deg=(30.0, 12.0), deref_factor=(2, 4))])
def test_refined_torus(H, orc, extra):
    """cfg 0 torus with the block columns inside r < 4 refined (the horizon region), outflow / polar / periodic
    boundaries on the edge blocks; last case: every feature of BASELINE cfg 4 at once"""
    kw = dict(nb=(8, 8, 8), r_refine_max=4.0)
    kw.update(extra)
    p = I.torus_params(n=(32, 16, 16), **kw)
    g, o = H.Grid(p), orc.OrcGrid(p)
    infos = _infos(o)
    assert any(o.block_info(b)["lev1"] for b in range(o.num_blocks()))
    _set_both(g, o, I.fm_torus_blocks(p, infos, seed=4))
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt
    if "lat_max_level" in extra:
        assert g.levels() == list(o.levels())
    g.step(1)
    o.step(1)
    fin = 2 ** extra.get("lat_max_level", 0)
    _check_blocks(p, infos, o, g, TOL_1 * fin)
    assert g.levels() == list(o.levels())   # never skip the continuation: a diverging level assignment is a failure
    g.step(3)
    o.step(3)
    _check_blocks(p, infos, o, g, TOL_10)


@pytest.mark.parametrize("pole", ["reflect", "transmit"])
def test_cfg4_full_size_one_coarse_step(H, orc, pole):
    """BASELINE cfg 4 at full size in the launch configuration bench.py --workload cfg4 times (1472 blocks of 16^3,
    6 029 312 zones, refinement r < 20, derefinement 2x / 4x, LAT levels 1 / 2 / 4): every zone of every block after one
    coarse step (= 4 finest steps) against the oracle.  "transmit": the same grid with the paper's own polar
    boundary (NEXT-1), the pole ghosts of every polar block coming from the block half a turn away."""
    bc = {}
    if pole == "transmit":
        bc = dict(bc_lo=(I.BC_OUTFLOW, I.BC_POLAR_TRANSMIT, I.BC_PERIODIC),
                  bc_hi=(I.BC_OUTFLOW, I.BC_POLAR_TRANSMIT, I.BC_PERIODIC))
    p = I.torus_params(n=(256, 128, 128), r_out=1000.0, nb=(16, 16, 16), lat_max_level=2, r_refine_max=20.0,
                       deref_theta_deg=(15.0, 5.0), deref_factor=(2, 4), **bc)
    g, o = H.Grid(p), orc.OrcGrid(p)
    assert g.num_blocks() == o.num_blocks() == 1472
    infos = _infos(o)
    assert sum(int(np.prod(n)) for _, _, n in infos) == 6029312
    _set_both(g, o, I.fm_torus_blocks(p, infos, seed=4))
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt
    assert g.levels() == list(o.levels()) and set(g.levels()) == {0, 1, 2}
    tg, _ = g.step(1)
    to, _ = o.step(1)
    assert abs(tg - to) <= 1e-13 * to
    _check_blocks(p, infos, o, g, 4 * TOL_1)
    if pole == "reflect":
        # two more coarse steps (12 finest steps in all), the level assignment compared after every coarse step
        for _ in range(2):
            assert g.levels() == list(o.levels())
            tg, _ = g.step(1)
            to, _ = o.step(1)
            assert abs(tg - to) <= 1e-13 * to
        assert g.levels() == list(o.levels())
        _check_blocks(p, infos, o, g, TOL_10)


def test_all_blocks_calls_equal_block_by_block(H):
    """hamr_set_all_blocks / hamr_get_all_blocks (one call, arrays of every block back to back) against the
    block-by-block calls: same state bit for bit"""
    p = I.torus_params(n=(32, 16, 16), nb=(8, 8, 8), r_refine_max=4.0, lat_max_level=1)
    a, b = H.Grid(p), H.Grid(p)
    infos = [a.block_info(q)[:3] for q in range(a.num_blocks())]
    data = I.fm_torus_blocks(p, infos, seed=4)
    for q, (hyd, bf) in enumerate(data):
        assert a.set_block_prims(q, hyd, bf) == 0
    assert a.commit() == 0
    hy = [np.stack([d[0][c] for d in data]) for c in range(5)]
    bf = [np.stack([d[1][c] for d in data]) for c in range(3)]
    assert b.set_all_blocks(hy, bf) == 0
    assert a.dt == b.dt
    a.step(2)
    b.step(2)
    allb = b.get_all_blocks()
    for q in range(a.num_blocks()):
        one = a.get_block_prims(q)
        for c in range(8):
            assert np.array_equal(one[c], allb[c][q])
