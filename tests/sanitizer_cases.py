"""Driver for the sanitizer runs of SURVEY section 5 (not a test: run under compute-sanitizer on the B200 box, e.g.
    compute-sanitizer --tool memcheck python tests/sanitizer_cases.py
and for racecheck / initcheck likewise; the summaries are kept under profiles/).  Small grids that reach every kernel
family through the C-ABI: BASELINE cfg 0 (generic marching / x3 / update kernels, polar and outflow ghost fill), a
periodic 32^3 box (TMA ring sweeps, wrapping x3 sweep, tiled update, ghost fill without x3 slots), a derefined torus,
and the refined + derefined + LAT block grid of tests/test_gpu_refine.py::test_refined_torus[extra2]."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_1912_10192_b200 import hamr, inputs as I  # noqa: E402


def main():
    # cfg 0, monolithic
    p = I.torus_params()
    hyd, bf = I.fm_torus(p, seed=0)
    g = hamr.Grid(p)
    assert g.set_prims(hyd, bf) == 0
    g.step(2)
    g.debug_emf()
    assert g.divb() <= 1e-12 and np.all(np.isfinite(g.get_prims()[0]))
    g.close()
    # periodic box: ring, wrap and tile kernels
    q = I.minkowski_params(n=(32, 32, 32))
    hyd, bf = I.minkowski_waves(q, seed=1)
    g = hamr.Grid(q)
    assert g.set_prims(hyd, bf) == 0
    g.step(2)
    assert g.divb() <= 1e-12
    g.close()
    # Kerr torus on the ring path (n3 = 32) and with phi-derefinement (generic kernels + C-15 fix-ups)
    for extra in (dict(), dict(deref_theta_deg=(30.0, 12.0), deref_factor=(2, 4))):
        r = I.torus_params(n=(24, 16, 32), **extra)
        hyd, bf = I.fm_torus(r, seed=3)
        g = hamr.Grid(r)
        assert g.set_prims(hyd, bf) == 0
        g.step(2)
        assert g.divb() <= 1e-12
        g.close()
    # block grid: x1 refinement + derefinement + LAT
    s = I.torus_params(n=(32, 16, 16), nb=(8, 4, 16), r_refine_max=4.0, lat_max_level=1, deref_theta_deg=(30.0, 12.0),
                       deref_factor=(2, 4))
    g = hamr.Grid(s)
    infos = [g.block_info(b)[:3] for b in range(g.num_blocks())]
    for b, (hb, fb) in enumerate(I.fm_torus_blocks(s, infos, seed=4)):
        assert g.set_block_prims(b, hb, fb) == 0
    assert g.commit() == 0
    g.step(2)
    assert g.divb() <= 1e-12
    g.get_block_prims(0)
    g.close()
    print("sanitizer cases ok")


if __name__ == "__main__":
    main()
