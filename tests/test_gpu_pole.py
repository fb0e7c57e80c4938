"""GPU <-> oracle parity with the transmissive polar boundary: the ghost
zone beyond the pole is the mirror row's zone half a turn away in x3.  Monolithic ghost kernel and the block
ghost kernel (with derefined polar rows and LAT on top).  Needs a B200."""
import numpy as np
import pytest

from paper_1912_10192_b200 import inputs as I
from tests._parity import parity_errors

pytestmark = pytest.mark.gpu

TOL_1, TOL_10, TOL_DIVB = 1e-10, 1e-7, 1e-12
TRANSMIT = dict(bc_lo=(I.BC_OUTFLOW, I.BC_POLAR_TRANSMIT, I.BC_PERIODIC),
                bc_hi=(I.BC_OUTFLOW, I.BC_POLAR_TRANSMIT, I.BC_PERIODIC))


@pytest.fixture(scope="module")
def H():
    from paper_1912_10192_b200 import build, hamr
    build.build_lib()
    hamr.lib()
    return hamr


def _run_pair(H, orc, p, hyd, bf, fin=1):
    g, o = H.Grid(p), orc.OrcGrid(p)
    assert g.set_prims(hyd, bf) == 0 and o.set_prims(hyd, bf) == 0
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt
    g.step(1)
    o.step(1)
    e = parity_errors(p, o.get_prims(), g.get_prims())
    assert max(e.values()) <= TOL_1 * fin, e
    if fin == 1 or g.levels() == list(o.levels()):
        g.step(5)
        o.step(5)
        e = parity_errors(p, o.get_prims(), g.get_prims())
        assert max(e.values()) <= TOL_10, e
    ob = o.get_bface()
    scale = max(np.abs(a).max() for a in ob)   # one scale for the field: a component may hold rounding noise only
    for a, b in zip(ob, g.get_bface()):
        assert np.abs(a - b).max() <= TOL_10 * max(scale, 1e-300)
    assert g.divb() <= TOL_DIVB and g.stats()[0] == 0 and o.stats()[0] == 0


@pytest.mark.parametrize("extra", [dict(), dict(nb=(16, 8, 32)), dict(nb=(16, 8, 8)), dict(nb=(32, 32, 16)), dict(nb=(16, 16, 4))])
def test_tilted_disk_through_the_poles(H, orc, extra):
    # a thick (h/r = 0.1) version of the cfg 3 stand-in so that 64x32x32 resolves it: the inclined disk and its
    # field cross both poles.  Monolithic ghost kernel, then the block ghost kernel on blocks that span x3 and
    # on blocks that cut it (the rows beyond the pole come from the block half a turn away).
    p = I.tilted_disk_params(n=(64, 32, 32), **TRANSMIT, **extra)
    hyd, bf = I.tilted_disk(p, seed=3, hr=0.1)
    _run_pair(H, orc, p, hyd, bf)


def test_transmissive_poles_with_blocks_deref_and_lat(H, orc):
    # torus with a 10 % phi-dependent pressure perturbation: the polar rows are derefined (4x, 2x), the blocks sit
    # on two time levels, and the pole ghosts come from half a turn away
    p = I.torus_params(n=(32, 16, 16), nb=(8, 4, 16), lat_max_level=1, deref_theta_deg=(30.0, 12.0),
                       deref_factor=(2, 4), **TRANSMIT)
    hyd, bf = I.fm_torus(p, seed=4, pert=0.1)
    _run_pair(H, orc, p, hyd, bf, fin=2)


def test_transmissive_poles_on_phi_cut_blocks_with_deref_refinement_and_lat(H, orc):
    # everything at once on blocks that cut x3 (BASELINE cfg 4's block shape with the paper's pole): derefined
    # polar rows (group-unit phi ghosts across the pole), one x1 refinement level (restriction / prolongation in
    # the pole corner), two time levels
    p = I.torus_params(n=(32, 16, 32), nb=(8, 4, 16), lat_max_level=1, deref_theta_deg=(30.0, 12.0),
                       deref_factor=(2, 4), r_refine_max=4.0, **TRANSMIT)
    g, o = H.Grid(p), orc.OrcGrid(p)
    infos = []
    for b in range(o.num_blocks()):
        d = o.block_info(b)
        infos.append((d["x_lo"], d["dx"], d["n"]))
    assert any(o.block_info(b)["lev1"] for b in range(o.num_blocks()))
    for b, (hyd, bf) in enumerate(I.fm_torus_blocks(p, infos, seed=4, pert=0.1)):
        assert g.set_block_prims(b, hyd, bf) == 0 and o.set_block_prims(b, hyd, bf) == 0
    assert g.commit() == 0 and o.commit() == 0
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt and g.levels() == list(o.levels())
    assert len(set(g.levels())) == 2

    def check(tol):
        worst = {}
        # face fields: one scale for the whole grid (a block, or one component in a block, may hold rounding noise only)
        obf = [o.get_block_bface(b) for b in range(len(infos))]
        scale = max(max(np.abs(a).max() for a in bf) for bf in obf)
        for b, (x_lo, dx, n) in enumerate(infos):
            e = parity_errors(I.block_as_grid(p, x_lo, dx, n), o.get_block_prims(b), g.get_block_prims(b))
            for k, v in e.items():
                worst[k] = max(worst.get(k, 0.0), v)
            for a, c in zip(obf[b], g.get_block_bface(b)):
                assert np.abs(a - c).max() <= tol * max(scale, 1e-300)
        assert max(worst.values()) <= tol, worst

    g.step(1)
    o.step(1)
    check(2 * TOL_1)
    assert g.levels() == list(o.levels())   # never skip the continuation: a diverging level assignment is a failure
    g.step(3)
    o.step(3)
    check(TOL_10)
    assert g.divb() <= TOL_DIVB and g.stats()[0] == 0 and o.stats()[0] == 0


def test_transmit_differs_from_reflect_and_torus_agrees(H):
    """sanity on the product alone: phi-dependent data see the difference between the two pole treatments;
    axisymmetric data do not"""
    p0 = I.torus_params(n=(32, 16, 16))
    p1 = dict(p0, **TRANSMIT)
    hyd, bf = I.fm_torus(p0, seed=0, pert=0.0)
    a, b = H.Grid(p0), H.Grid(p1)
    assert a.set_prims(hyd, bf) == 0 and b.set_prims(hyd, bf) == 0
    a.step(3)
    b.step(3)
    for x, y in zip(a.get_prims(), b.get_prims()):
        assert np.abs(x - y).max() <= 1e-13 * max(np.abs(x).max(), 1e-300)
    q0 = I.tilted_disk_params(n=(32, 16, 16))
    hyd, bf = I.tilted_disk(q0, seed=3, hr=0.2)
    a, b = H.Grid(q0), H.Grid(dict(q0, **TRANSMIT))
    assert a.set_prims(hyd, bf) == 0 and b.set_prims(hyd, bf) == 0
    a.step(3)
    b.step(3)
    assert np.abs(a.get_prims()[0] - b.get_prims()[0]).max() > 1e-8
