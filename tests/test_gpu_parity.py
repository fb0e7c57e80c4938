"""GPU <-> oracle parity through the C-ABI (BASELINE.json north_star: max relative error <= 1e-10 on all
primitives after 1 step, <= 1e-7 after 10 steps, div B <= 1e-12, zero inversion failures).
Same seeded inputs to both sides; element-by-element comparison.  Needs a B200."""
import numpy as np
import pytest

from paper_1912_10192_b200 import inputs as I
from tests._parity import parity_errors, raw_velocity_error, rel_max

pytestmark = pytest.mark.gpu

TOL_1, TOL_10, TOL_DIVB = 1e-10, 1e-7, 1e-12


@pytest.fixture(scope="module")
def H():
    from paper_1912_10192_b200 import build, hamr
    build.build_lib()
    hamr.lib()
    return hamr


def _pair(H, orc, p, hyd, bf):
    g = H.Grid(p)
    o = orc.OrcGrid(p)
    assert g.set_prims(hyd, bf) == 0
    assert o.set_prims(hyd, bf) == 0
    return g, o


def _cases():
    c = {}
    p = I.torus_params()                                        # BASELINE cfg 0
    c["cfg0_torus"] = (p, lambda: I.fm_torus(p, seed=0))
    q = I.minkowski_params(n=(40, 24, 36))                      # ragged sizes: several tiles + tails
    c["minkowski_ragged"] = (q, lambda: I.minkowski_waves(q, seed=1, amp=1e-2, noise=1e-3))
    r = I.torus_params(n=(24, 16, 8), recon=I.RECON_PLM)
    c["torus_plm"] = (r, lambda: I.fm_torus(r, seed=5))
    s = I.minkowski_params(n=(32, 32, 32))                      # BASELINE cfg 1 at oracle-friendly size
    c["cfg1_waves"] = (s, lambda: I.minkowski_waves(s, seed=1))
    return c


CASES = _cases()


def _u_scales(orc, p, o):
    """max |U_c| over the grid for the 5 hydro rows, and max |sqrt(-g) B| (row 5), from the oracle's
    per-zone routines (scales for the flux comparison only)."""
    P = o.get_prims()
    n = p["n"]
    xc, _, _ = I.grid_coords(p)
    out = np.zeros(6)
    for i in range(n[0]):
        for j in range(n[1]):
            G = orc.geom_at(p["metric"], p["a"], xc[0][i], xc[1][j])
            for k in range(0, n[2], max(1, n[2] // 4)):
                U, _ = orc.prim_to_UF([P[c][i, j, k] for c in range(8)], G, p["gamma_ad"])
                out[:5] = np.maximum(out[:5], np.abs(U[:5]))
                out[5] = max(out[5], np.abs(U[5:]).max())
    return out


@pytest.mark.parametrize("name", list(CASES))
def test_face_fluxes_emfs_and_ctop_match(H, orc, name):
    p, gen = CASES[name]
    hyd, bf = gen()
    g, o = _pair(H, orc, p, hyd, bf)
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt          # first dt from the initial flux pass (C-14)
    g.debug_emf()
    o.debug_emf()
    usc = _u_scales(orc, p, o)
    for d in range(3):
        for which in range(7):
            a, b = o.get_face(d, which), g.get_face(d, which)
            # an HLL flux is a difference of terms of size |F| and ctop |U| (ctop <= 1): rounding
            # errors scale with those terms, not with the (possibly cancelling) result
            scale = np.abs(a).max() + usc[min(which, 5)]
            err = np.abs(a - b).max() / scale
            assert err <= 1e-13, (name, d, which, err)
            if which == 0:   # the upwind selector of CT sees the SIGN of the mass flux: must agree exactly
                assert np.array_equal(np.sign(a), np.sign(b)), (name, d)
    for f in range(3):
        a, b = o.get_edge(f), g.get_edge(f)
        assert rel_max(a, b) <= 1e-12, (name, f, rel_max(a, b))
    assert np.allclose(g.ctop(), o.ctop(), rtol=1e-13, atol=0)


@pytest.mark.parametrize("name", list(CASES))
def test_parity_after_1_and_10_steps(H, orc, name):
    p, gen = CASES[name]
    hyd, bf = gen()
    g, o = _pair(H, orc, p, hyd, bf)
    tg, dtg = g.step(1)
    to, dto = o.step(1)
    assert abs(tg - to) <= 1e-13 * to and abs(dtg - dto) <= 1e-13 * dto
    e1 = parity_errors(p, o.get_prims(), g.get_prims())
    assert max(e1.values()) <= TOL_1, (name, e1)
    for a, b in zip(o.get_bface(), g.get_bface()):
        assert rel_max(a, b) <= TOL_1
    g.step(9)
    o.step(9)
    e10 = parity_errors(p, o.get_prims(), g.get_prims())
    assert max(e10.values()) <= TOL_10, (name, e10)
    assert g.divb() <= TOL_DIVB and o.divb() <= TOL_DIVB
    sg, so = g.stats(), o.stats()
    assert sg[0] == 0 and so[0] == 0                 # parity runs must report zero inversion failures
    # failures and ceiling hits agree; the two floor counters are printed only: the atmosphere of the torus sits AT
    # the floors, where a last-bit difference of the inversion decides whether a zone counts as a hit (the counters
    # are compared exactly in tests/test_gpu_zone.py on states well clear of the thresholds)
    assert sg[3] == so[3]
    print(name, "1 step", e1, "10 steps", e10, "velocity error without the S-21a rounding floor (10 steps):",
          raw_velocity_error(p, o.get_prims(), g.get_prims()), "event counters", sg)


def test_divb_and_conservation_minkowski(H):
    p = I.minkowski_params(n=(24, 20, 28))
    hyd, bf = I.minkowski_waves(p, seed=1, amp=1e-2, noise=1e-3)
    g = H.Grid(p)
    assert g.set_prims(hyd, bf) == 0
    assert g.divb() < 1e-13
    t0 = g.totals()
    g.step(30)
    t1 = g.totals()
    assert g.divb() < TOL_DIVB and g.stats()[0] == 0
    assert abs(t1[0] - t0[0]) < 1e-13 * abs(t0[0])
    assert abs(t1[1] - t0[1]) < 1e-13 * abs(t0[1])
    assert np.all(np.abs(t1[2:] - t0[2:]) < 1e-13 * abs(t0[1]))
    b0 = [b.sum() for b in bf]
    b1 = [b.sum() for b in g.get_bface()]
    assert np.allclose(b0, b1, rtol=1e-13)


def test_edge_cases(H, orc):
    # phi slab (N3 = 1), no magnetic field, minimum sizes
    p = I.torus_params(n=(16, 8, 1))
    hyd, _ = I.fm_torus(p, pert=0.0, with_B=False)
    g, o = _pair(H, orc, p, hyd, None)
    g.step(3)
    o.step(3)
    e = parity_errors(p, o.get_prims(), g.get_prims())
    assert max(e.values()) <= 3 * TOL_1, e           # 3 steps
    # smallest non-periodic extents
    q = I.torus_params(n=(3, 3, 3))
    hyd, bf = I.fm_torus(q, seed=7)
    g, o = _pair(H, orc, q, hyd, bf)
    g.step(2)
    o.step(2)
    assert max(parity_errors(q, o.get_prims(), g.get_prims()).values()) <= 2 * TOL_1   # 2 steps
    # call order and bad input
    g2 = H.Grid(q)
    with pytest.raises(H.HamrError) as ei:
        g2.step(1)
    assert ei.value.code == H.ESTATE
    hyd[0] = hyd[0].copy()
    hyd[0][1, 1, 1] = np.nan
    assert g2.set_prims(hyd, bf) == H.ENONFINITE
    # zero steps is a no-op
    g3 = H.Grid(q)
    hyd, bf = I.fm_torus(q, seed=7)
    g3.set_prims(hyd, bf)
    t, _ = g3.step(0)
    assert t == 0.0
    for a, b in zip(g3.get_prims()[:5], hyd):
        assert np.array_equal(a, b)


def test_device_pointer_path_and_torch_arena(H, orc):
    import torch
    p = I.torus_params(n=(24, 12, 16))
    hyd, bf = I.fm_torus(p, seed=3)
    g = H.Grid(p, torch_arena=True)
    hd = [torch.from_numpy(np.ascontiguousarray(h)).cuda() for h in hyd]
    bd = [torch.from_numpy(np.ascontiguousarray(b)).cuda() for b in bf]
    assert g.set_prims_dev(hd, bd) == 0
    g.step(2)
    out = [torch.empty(p["n"], dtype=torch.float64, device="cuda") for _ in range(8)]
    g.get_prims_dev(out)
    torch.cuda.synchronize()
    g2 = H.Grid(p)
    g2.set_prims(hyd, bf)
    g2.step(2)
    ref = g2.get_prims()
    for a, b in zip(ref, out):
        assert np.array_equal(a, b.cpu().numpy())     # same kernels, same inputs: bitwise
    assert g.launch_count() > 0


def test_full_size_headline_config_one_step(H, orc):
    """BASELINE cfg 2 (256x128x128 Kerr torus) in the launch configuration bench.py times: every
    zone compared against the oracle after one step; properties after more steps."""
    p = I.torus_params(n=(256, 128, 128), r_out=1000.0)
    hyd, bf = I.fm_torus(p, seed=2)
    g, o = _pair(H, orc, p, hyd, bf)
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt
    g.step(1)
    o.step(1)
    e1 = parity_errors(p, o.get_prims(), g.get_prims())
    print("cfg2 1 step", e1)
    assert max(e1.values()) <= TOL_1, e1
    g.step(9)
    o.step(9)                                        # ~12 s of oracle: north_star's 1e-7 after 10 steps at full size
    e10 = parity_errors(p, o.get_prims(), g.get_prims())
    print("cfg2 10 steps", e10, "velocity error without the S-21a rounding floor:",
          raw_velocity_error(p, o.get_prims(), g.get_prims()))
    assert max(e10.values()) <= TOL_10, e10
    assert g.divb() <= TOL_DIVB and o.divb() <= TOL_DIVB
    sg, so = g.stats(), o.stats()
    assert sg[0] == so[0] == 0 and sg[3] == so[3]


def _cold_gas_errors(p, ref, got):
    """parity_errors with the internal-energy error measured against max(u, 1e-4 (rho + b^2)) (S-21b): u is
    recovered from W = w gamma^2 ~ rho, itself the result of ~100 fp64 operations (a dozen flux differences, the
    source, the Newton solve); one ulp each moves W, hence u, by ~100 eps (rho + b^2) ~ 1e-14 (rho + b^2) in ABSOLUTE
    terms, so where the gas is cold (cfg 3's disk has u / rho down to 2e-5) a 1e-10 RELATIVE bound on u is below
    the rounding floor of any two fp64 implementations (the oracle's own round trip shows it, pin P3)."""
    e = parity_errors(p, ref, got)
    from tests._parity import centre_gcov_diag_and_norm
    b2 = centre_gcov_diag_and_norm(p, ref[5:8])[1] ** 2
    e["u"] = float(np.max(np.abs(got[1] - ref[1]) / np.maximum(np.abs(ref[1]), 1e-4 * (ref[0] + b2))))
    return e


def test_cfg3_tilted_disk_stand_in(H, orc):
    """BASELINE cfg 3 (synthetic stand-in) at an oracle-friendly 128x64x64: a thin, cold,
    inclined, magnetised sheet crossing the polar rows.  1 and 10 steps, zero inversion failures."""
    p = I.tilted_disk_params(n=(128, 64, 64))
    hyd, bf = I.tilted_disk(p, seed=3)
    g, o = _pair(H, orc, p, hyd, bf)
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt
    g.step(1)
    o.step(1)
    e = _cold_gas_errors(p, o.get_prims(), g.get_prims())
    assert max(e.values()) <= TOL_1, e
    g.step(9)
    o.step(9)
    e = _cold_gas_errors(p, o.get_prims(), g.get_prims())
    assert max(e.values()) <= TOL_10, e
    assert g.divb() <= TOL_DIVB and g.stats()[0] == 0 and o.stats()[0] == 0


def test_cfg3_full_size_one_step(H, orc):
    """BASELINE cfg 3 at the size bench.py --workload cfg3 times (512x256x256, 33.5 M zones): every zone against the
    oracle after one step (norm S-21b for the cold gas, as in the stand-in test above)."""
    p = I.tilted_disk_params()
    assert tuple(p["n"]) == (512, 256, 256)
    hyd, bf = I.tilted_disk(p, seed=3)
    g, o = _pair(H, orc, p, hyd, bf)
    assert abs(g.dt - o.dt) <= 1e-13 * o.dt
    g.step(1)
    o.step(1)
    e = _cold_gas_errors(p, o.get_prims(), g.get_prims())
    print("cfg3 full size, 1 step", e)
    assert max(e.values()) <= TOL_1, e
    sg, so = g.stats(), o.stats()
    assert g.divb() <= TOL_DIVB and sg[0] == so[0] == 0 and sg[3] == so[3]


def test_set_prims_async_equals_set_prims(H):
    """hamr_set_prims_async + hamr_wait_input (host arrays in pinned memory, no wait for the kernels behind the copies)
    leaves the grid in the state hamr_set_prims does: same dt, same primitives after 3 steps, bit for bit; NaN input is
    reported by the next full wait."""
    import torch
    p = I.torus_params()
    hyd, bf = I.fm_torus(p, seed=0)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
    hp, bp = [pin(h) for h in hyd], [pin(b) for b in bf]
    a, b = H.Grid(p), H.Grid(p)
    assert a.set_prims(hyd, bf) == 0
    assert b.set_prims_async(hp, bp) == 0
    b.wait_input()
    for x in hp + bp:
        x[...] = -7.0                      # the input has left the host: the arrays are the caller's again
    assert a.dt == b.dt
    a.step(3)
    b.step(3)
    assert all(np.array_equal(x, y) for x, y in zip(a.get_prims(), b.get_prims()))
    hp2 = [pin(h) for h in hyd]
    hp2[1][3, 4, 5] = np.nan
    assert b.set_prims_async(hp2, None) == 0
    b.wait_input()
    assert H.lib().hamr_sync(b.h) == H.ENONFINITE
    a.close()
    b.close()


def test_stage_output_then_get_prims_equals_get_prims(H):
    """hamr_stage_output gathers the dense output into the staging area ahead of hamr_get_prims: same arrays, bit for bit;
    a step, a new state or another getter in between makes the next hamr_get_prims gather again"""
    p = I.torus_params()
    hyd, bf = I.fm_torus(p, seed=0)
    a, b = H.Grid(p), H.Grid(p)
    assert a.set_prims(hyd, bf) == 0 and b.set_prims(hyd, bf) == 0
    a.step(2)
    b.step_async(2)
    b.stage_output()
    b.sync()
    assert all(np.array_equal(x, y) for x, y in zip(a.get_prims(), b.get_prims()))
    b.stage_output()
    b.get_bface()                        # another getter takes the staging area
    assert all(np.array_equal(x, y) for x, y in zip(a.get_prims(), b.get_prims()))
    b.stage_output()
    a.step(1)
    b.step(1)                            # the staged arrays are stale now
    assert all(np.array_equal(x, y) for x, y in zip(a.get_prims(), b.get_prims()))
    b.stage_output()
    assert b.set_prims(hyd, bf) == 0     # ... and after a new state
    assert all(np.array_equal(x, y) for x, y in zip(hyd, b.get_prims()[:5]))
    r = H.Grid(I.torus_params(n=(32, 16, 16), nb=(8, 8, 8), r_refine_max=4.0))
    assert H.lib().hamr_stage_output(r.h) == H.ESTATE
    for g in (a, b, r):
        g.close()
