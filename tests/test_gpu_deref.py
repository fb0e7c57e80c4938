"""GPU <-> oracle parity for the phi-derefinement of the polar rows (DESIGN.md §9 C-15;
PAPER.md:101), alone, with blocks in (x1, x2) and with local adaptive time-stepping.  Needs a B200."""
import numpy as np
import pytest

from paper_1912_10192_b200 import inputs as I
from tests._parity import parity_errors
from tests.test_oracle_deref import _group_checks, _rep_state

pytestmark = pytest.mark.gpu

TOL_1, TOL_10, TOL_DIVB = 1e-10, 1e-7, 1e-12
DEREF = dict(deref_theta_deg=(30.0, 12.0), deref_factor=(2, 4))     # 16 rows: m = 4, 2, 2, 1 ... 1, 2, 2, 4
MROW16 = [4, 2, 2] + [1] * 10 + [2, 2, 4]


@pytest.fixture(scope="module")
def H():
    from paper_1912_10192_b200 import build, hamr
    build.build_lib()
    hamr.lib()
    return hamr


def _check(p, o, g, tol):
    e = parity_errors(p, o.get_prims(), g.get_prims())
    assert max(e.values()) <= tol, e
    ob = o.get_bface()
    scale = max(np.abs(a).max() for a in ob)   # one scale for the field: a component may hold rounding noise only
    for a, b in zip(ob, g.get_bface()):
        assert np.abs(a - b).max() <= tol * max(scale, 1e-300)
    assert g.divb() <= TOL_DIVB and g.stats()[0] == 0


@pytest.mark.parametrize("extra", [dict(), dict(nb=(8, 4, 16)), dict(nb=(8, 4, 16), lat_max_level=1),
                                   dict(recon=I.RECON_PLM)])
def test_deref_torus_parity(H, orc, extra):
    p = I.torus_params(n=(32, 16, 16), **DEREF, **extra)
    hyd, bf = I.fm_torus(p, seed=4)
    g, o = H.Grid(p), orc.OrcGrid(p)
    assert g.set_prims(hyd, bf) == 0 and o.set_prims(hyd, bf) == 0
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt
    if "lat_max_level" in extra:
        assert g.levels() == list(o.levels())
    g.step(1)
    o.step(1)
    _check(p, o, g, TOL_1 * (2 if "lat_max_level" in extra else 1))
    g.step(5)
    o.step(5)
    _check(p, o, g, TOL_10)
    _group_checks(g.get_prims(), g.get_bface(), MROW16)


def test_deref_minkowski_mixed_rows(H, orc):
    n = (8, 16, 16)
    p = I.minkowski_params(n=n, deref_theta_deg=(45.0, 22.6), deref_factor=(2, 4))
    mrow = [4, 4, 2, 2] + [1] * 8 + [2, 2, 4, 4]
    hyd, bf = I.minkowski_waves(p, seed=1, amp=2e-2, noise=1e-2)
    bf = [np.full_like(b, v) for b, v in zip(bf, (1.0, np.sqrt(2.0), 0.5))]
    g, o = H.Grid(p), orc.OrcGrid(p)
    assert g.set_prims(hyd, bf) == 0 and o.set_prims(hyd, bf) == 0
    t0 = g.totals()
    g.step(1)
    o.step(1)
    _check(p, o, g, TOL_1)
    g.step(5)
    o.step(5)
    _check(p, o, g, TOL_10)
    _group_checks(g.get_prims(), g.get_bface(), mrow)
    t1 = g.totals()
    assert np.abs(t1 - t0).max() / max(t0[0], abs(t0[1])) < 1e-13


def test_deref_everywhere_is_the_coarse_phi_grid_gpu(H):
    """property that needs no oracle: derefined by m in every row == the plain grid with N3 / m zones"""
    m = 2
    pc = I.torus_params(n=(32, 16, 8))
    pf = I.torus_params(n=(32, 16, 16), deref_theta_deg=(91.0,), deref_factor=(m,))
    hyd, bf = I.fm_torus(pc, seed=3)
    c, f = H.Grid(pc), H.Grid(pf)
    Hf, Bf = _rep_state(hyd, bf, m)
    assert c.set_prims(hyd, bf) == 0 and f.set_prims(Hf, Bf) == 0
    assert abs(c.dt - f.dt) <= 1e-14 * c.dt
    c.step(5)
    f.step(5)
    for a, b in zip(c.get_prims(), f.get_prims()):
        for r in range(m):
            assert np.abs(b[:, :, r::m] - a).max() <= 1e-11 * max(np.abs(a).max(), 1e-300)


def test_deref_on_blocks_that_cut_phi(H, orc):
    """BASELINE cfg 4's block shape: blocks cut x3, so the phi-ghost zones of derefined rows are held in group units
    and the x1 / x2 flux layers are exchanged between phi-neighbours.  Torus with LAT against the oracle, and the
    product's own phi-cut grid against its phi-spanning grid (same answer to round-off, shared faces identical)."""
    p = I.torus_params(n=(32, 16, 32), nb=(8, 4, 16), lat_max_level=1, **DEREF)
    hyd, bf = I.fm_torus(p, seed=4)
    g, o = H.Grid(p), orc.OrcGrid(p)
    assert g.set_prims(hyd, bf) == 0 and o.set_prims(hyd, bf) == 0
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt and g.levels() == list(o.levels())
    g.step(1)
    o.step(1)
    _check(p, o, g, 2 * TOL_1)
    assert g.levels() == list(o.levels())   # never skip the continuation: a diverging level assignment is a failure
    g.step(4)
    o.step(4)
    _check(p, o, g, TOL_10)
    _group_checks(g.get_prims(), g.get_bface(), MROW16)
    q = dict(p, nb=(8, 4, 32), lat_max_level=0)
    a, b = H.Grid(dict(q, nb=(8, 4, 16))), H.Grid(q)
    assert a.set_prims(hyd, bf) == 0 and b.set_prims(hyd, bf) == 0
    a.step(4)
    b.step(4)
    for x, y in zip(a.get_prims() + a.get_bface(), b.get_prims() + b.get_bface()):
        assert np.abs(x - y).max() <= 1e-13 * max(np.abs(x).max(), 1e-300)


def test_deref_minkowski_mixed_rows_phi_cut_blocks(H, orc):
    n = (8, 16, 32)
    p = I.minkowski_params(n=n, nb=(4, 8, 16), deref_theta_deg=(45.0, 22.6), deref_factor=(2, 4))
    mrow = [4, 4, 2, 2] + [1] * 8 + [2, 2, 4, 4]
    hyd, bf = I.minkowski_waves(p, seed=1, amp=2e-2, noise=1e-2)
    bf = [np.full_like(b, v) for b, v in zip(bf, (1.0, np.sqrt(2.0), 0.5))]
    g, o = H.Grid(p), orc.OrcGrid(p)
    assert g.set_prims(hyd, bf) == 0 and o.set_prims(hyd, bf) == 0
    t0 = g.totals()
    g.step(1)
    o.step(1)
    _check(p, o, g, TOL_1)
    g.step(5)
    o.step(5)
    _check(p, o, g, TOL_10)
    _group_checks(g.get_prims(), g.get_bface(), mrow)
    assert np.abs(g.totals() - t0).max() / max(t0[0], abs(t0[1])) < 1e-13
