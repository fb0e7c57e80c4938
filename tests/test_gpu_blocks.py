"""GPU <-> oracle parity on the block-structured grid (C-16 ghost exchange
between blocks, C-17 local adaptive time-stepping with time-interpolated ghosts, flux / EMF registers,
correction and re-inversion).  Same seeded inputs to both sides through the two
C ABIs; tolerances of BASELINE.json north_star.  Needs a B200."""
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


def _band_levels(g_orc, axis, pattern):
    lv = []
    x00 = g_orc.block_info(0)["x_lo"][axis]
    for b in range(g_orc.num_blocks()):
        info = g_orc.block_info(b)
        pos = int(round((info["x_lo"][axis] - x00) / (info["dx"][axis] * info["n"][axis])))
        lv.append(pattern[pos % len(pattern)])
    return lv


def _check(p, o, g, tol):
    e = parity_errors(p, o.get_prims(), g.get_prims())
    assert max(e.values()) <= tol, e
    ob = o.get_bface()
    s = max(max(np.abs(a).max() for a in ob), 1e-300)   # one scale for the field: a component may hold rounding noise only
    for a, b in zip(ob, g.get_bface()):
        assert np.abs(a - b).max() <= tol * s
    assert g.divb() <= TOL_DIVB
    assert g.stats()[0] == 0
    return e


def test_block_lattice_matches_oracle(H, orc):
    p = I.torus_params(nb=(8, 4, 8))
    g, o = H.Grid(p), orc.OrcGrid(p)
    assert g.num_blocks() == o.num_blocks() == 4 * 4 * 2
    for b in range(g.num_blocks()):
        lo, dx, n, tl = g.block_info(b)
        info = o.block_info(b)
        assert np.allclose(lo, info["x_lo"], rtol=0, atol=1e-14) and np.allclose(dx, info["dx"], rtol=1e-15)
        assert n == info["n"] and tl == 0


@pytest.mark.parametrize("nb", [(8, 8, 8), (16, 4, 8), (32, 16, 16)])
def test_blocks_global_dt_torus(H, orc, nb):
    """C-16: block-decomposed cfg 0 torus (outflow / polar reflect / periodic on the edge blocks) against the
    oracle's block grid, which pin P15 shows is bitwise its monolithic grid."""
    p = I.torus_params(nb=nb)
    hyd, bf = I.fm_torus(p, seed=0)
    g, o = H.Grid(p), orc.OrcGrid(p)
    assert g.set_prims(hyd, bf) == 0 and o.set_prims(hyd, bf) == 0
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt
    g.step(1)
    o.step(1)
    _check(p, o, g, TOL_1)
    assert abs(g.dt - o.dt) <= 1e-12 * o.dt
    tg, _ = g.step(9)
    to, _ = o.step(9)
    _check(p, o, g, TOL_10)
    assert abs(tg - to) <= 1e-12 * to


def test_blocks_equal_monolithic_gpu(H):
    """the product's own block grid against its own monolithic grid (same kernels, different launch shape)"""
    p = I.minkowski_params(n=(24, 16, 16))
    hyd, bf = I.minkowski_waves(p, seed=1, amp=1e-2, noise=1e-3)
    a, b = H.Grid(p), H.Grid(dict(p, nb=(8, 8, 4)))
    assert a.set_prims(hyd, bf) == 0 and b.set_prims(hyd, bf) == 0
    a.step(3)
    b.step(3)
    for x, y in zip(a.get_prims() + a.get_bface(), b.get_prims() + b.get_bface()):
        assert np.abs(x - y).max() <= 1e-13 * max(np.abs(x).max(), 1e-300)


@pytest.mark.parametrize("axis,pattern", [(0, (0, 1, 2, 1)), (1, (1, 0)), (2, (2, 1, 0, 1))])
def test_lat_forced_levels_waves(H, orc, axis, pattern):
    """C-17 with prescribed time levels in bands along each axis: time-interpolated ghosts, registers,
    correction, re-inversion."""
    n = [8, 8, 8]
    n[axis] = 4 * len(pattern)
    p = I.minkowski_params(n=tuple(n), nb=(4, 4, 4), lat_max_level=2)
    hyd, bf = I.minkowski_waves(p, seed=1, amp=1e-2, noise=1e-3)
    g, o = H.Grid(p), orc.OrcGrid(p)
    lv = _band_levels(o, axis, pattern)
    o.force_levels(lv)
    g.set_levels(lv)
    assert g.set_prims(hyd, bf) == 0 and o.set_prims(hyd, bf) == 0
    assert g.levels() == list(o.levels()) and sorted(set(o.levels())) == sorted(set(pattern))
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt
    tg, _ = g.step(1)
    to, _ = o.step(1)
    assert abs(tg - to) <= 1e-13 * to
    _check(p, o, g, TOL_1)
    g.step(2)
    o.step(2)
    _check(p, o, g, TOL_10)


def test_lat_uniform_state_and_conservation(H):
    """properties that hold at any size: a uniform moving state stays uniform through LAT interfaces; mass,
    energy and momentum are conserved to round-off thanks to the flux correction"""
    n = (16, 8, 8)
    p = I.minkowski_params(n=n, nb=(4, 4, 4), lat_max_level=2)
    g = H.Grid(p)
    lv = [(0, 1, 2, 1)[b // 4 % 4] for b in range(g.num_blocks())]
    g.set_levels(lv)
    ref = [1.0, 2.0, 0.3, -0.2, 0.45, 0.7, 1.1, -0.4]
    hyd = [np.full(n, v) for v in ref[:5]]
    bf = [np.full(tuple(n[e] + (e == d) for e in range(3)), ref[5 + d]) for d in range(3)]
    assert g.set_prims(hyd, bf) == 0
    assert set(g.levels()) == {0, 1, 2}
    g.step(3)
    for c, v in enumerate(g.get_prims()):
        assert np.abs(v - ref[c]).max() <= 2e-14, c
    hyd, bf = I.minkowski_waves(p, seed=1, amp=1e-2, noise=0.0)
    assert g.set_prims(hyd, bf) == 0
    t0 = g.totals()
    g.step(4)
    t1 = g.totals()
    scale = max(t0[0], abs(t0[1]))
    assert np.abs(t1 - t0).max() / scale < 1e-13, (t1 - t0) / scale
    assert g.divb() <= TOL_DIVB


def test_lat_courant_levels_torus(H, orc):
    """C-17 with Courant-based levels on the cfg 0 torus cut into 8x4x8 blocks: the levels the product
    chooses equal the oracle's, and the state matches after one coarse step (= 4 finest steps)."""
    p = I.torus_params(nb=(8, 4, 8), lat_max_level=2)
    hyd, bf = I.fm_torus(p, seed=0)
    g, o = H.Grid(p), orc.OrcGrid(p)
    assert g.set_prims(hyd, bf) == 0 and o.set_prims(hyd, bf) == 0
    assert g.levels() == list(o.levels()) and len(set(o.levels())) >= 2
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt
    g.step(1)
    o.step(1)
    _check(p, o, g, TOL_1 * 4)   # 4 finest steps: 4 x the one-step bound
    assert g.levels() == list(o.levels())   # never skip the continuation: a diverging level assignment is a failure
    g.step(2)
    o.step(2)
    _check(p, o, g, TOL_10)


def test_block_grid_parameter_and_call_order_errors(H):
    """error behaviour of the block-structured entry points (include/hamr.h): EINVAL for parameter sets the
    build does not support, ESTATE for calls out of order; nothing throws, nothing aborts"""
    base = I.torus_params(n=(32, 16, 16))
    bad = [dict(nb=(5, 4, 4)),                                                     # does not divide n
           dict(nb=(2, 4, 4)),                                                     # block smaller than the ghost depth
           dict(nb=(8, 4, 8), deref_theta_deg=(30.0,), deref_factor=(4,)),         # 3 groups of ghosts must fit one neighbour
           dict(deref_theta_deg=(30.0,), deref_factor=(3,)),                       # factor must divide N3
           dict(nb=(4, 4, 16), r_refine_max=4.0),                                  # refinement needs nb[0] >= 6
           dict(r_refine_max=4.0),                                                 # refinement needs a block grid
           dict(lat_max_level=5),
           dict(bc_lo=(I.BC_OUTFLOW, I.BC_POLAR_TRANSMIT, I.BC_PERIODIC))]         # transmissive on one pole only
    for kw in bad:
        with pytest.raises(H.HamrError) as ei:
            H.Grid(dict(base, **kw))
        assert ei.value.code == H.EINVAL, kw
    g = H.Grid(dict(base, nb=(8, 8, 8), r_refine_max=4.0))
    hyd, bf = I.fm_torus(base, seed=0)
    assert g.set_prims(hyd, bf) == H.ESTATE          # a refined grid is set block by block
    assert g.commit() == H.ESTATE                    # nothing was set
    with pytest.raises(H.HamrError) as ei:
        g.step(1)
    assert ei.value.code == H.ESTATE
    u = H.Grid(dict(base, nb=(8, 8, 8)))             # unrefined block grid: both ways of setting agree
    assert u.set_prims(hyd, bf) == 0
    ref = u.get_prims()
    v = H.Grid(dict(base, nb=(8, 8, 8)))
    for b in range(v.num_blocks()):
        lo, dx, n, _ = v.block_info(b)
        i0 = [int(round((lo[d] - u.block_info(0)[0][d]) / dx[d])) for d in range(3)]
        sl = tuple(slice(i0[d], i0[d] + n[d]) for d in range(3))
        fsl = [tuple(slice(i0[e], i0[e] + n[e] + (e == d)) for e in range(3)) for d in range(3)]
        assert v.set_block_prims(b, [h[sl] for h in hyd], [bf[d][fsl[d]] for d in range(3)]) == 0
    assert v.commit() == 0
    for a, b_ in zip(ref, v.get_prims()):
        assert np.array_equal(a, b_)
    got = v.get_block_prims(3)
    lo, dx, n, _ = v.block_info(3)
    i0 = [int(round((lo[d] - v.block_info(0)[0][d]) / dx[d])) for d in range(3)]
    assert np.array_equal(got[0], ref[0][tuple(slice(i0[d], i0[d] + n[d]) for d in range(3))])
