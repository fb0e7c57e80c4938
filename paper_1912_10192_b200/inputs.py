"""Seeded synthetic input generators (DESIGN.md §5 "input recipe").

This module serves BOTH the CUDA library and the CPU oracle with identical host arrays.  It holds
none of the method's update arithmetic (no reconstruction, Riemann solver, CT, source, inversion
or time stepping) and imports neither side.  What it does hold is the *initial data*: the analytic
Fishbone-Moncrief torus in Kerr-Schild coordinates (BASELINE.json cfg 0, 2, 4), linear MHD
eigenmodes on a periodic Minkowski box (cfg 1) and a synthetic tilted thin disk (cfg 3; the
paper's own model is unpublished), plus the counter-based random numbers the
recipes draw.  The paper measures on no public dataset; these inputs are the workloads.

Conventions: primitives (rho, u, ut1, ut2, ut3) at zone centres, arrays of shape
(N1, N2, N3) C-ordered (x3 fastest); densitised face field Bf^d = sqrt(-g) B^d on d-faces with
shapes (N1+1,N2,N3), (N1,N2+1,N3), (N1,N2,N3+1).
"""
from __future__ import annotations

import numpy as np

# ------------------------------------------------------------------------------------------------
# counter-based random numbers: u = hash64(seed, global zone index) -> U(-1, 1)
# ------------------------------------------------------------------------------------------------
_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def rand_pm1(seed: int, idx: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser of (seed, idx); independent of traversal order and decomposition."""
    with np.errstate(over="ignore"):
        x = idx.astype(np.uint64) + np.uint64((int(seed) + 1) * 0x9E3779B97F4A7C15 & 0xFFFFFFFFFFFFFFFF)
        x ^= x >> np.uint64(30)
        x *= np.uint64(0xBF58476D1CE4E5B9)
        x ^= x >> np.uint64(27)
        x *= np.uint64(0x94D049BB133111EB)
        x ^= x >> np.uint64(31)
    return (x >> np.uint64(11)).astype(np.float64) * (2.0 ** -52) - 1.0


def zone_index(n) -> np.ndarray:
    return np.arange(int(n[0]) * int(n[1]) * int(n[2]), dtype=np.uint64).reshape(tuple(int(v) for v in n))


# ------------------------------------------------------------------------------------------------
# parameter sets (plain dicts; each binding packs its own struct)
# ------------------------------------------------------------------------------------------------
BC_PERIODIC, BC_OUTFLOW, BC_POLAR, BC_POLAR_TRANSMIT = 0, 1, 2, 3
METRIC_MINKOWSKI, METRIC_KS = 0, 1
RECON_PPM, RECON_PLM = 0, 1


def base_params(**kw) -> dict:
    p = dict(metric=METRIC_KS, recon=RECON_PPM, n=(32, 16, 16), a=0.9375,
             xmin=(1.2, 0.0, 0.0), xmax=(50.0, np.pi, 2.0 * np.pi),
             bc_lo=(BC_OUTFLOW, BC_POLAR, BC_PERIODIC), bc_hi=(BC_OUTFLOW, BC_POLAR, BC_PERIODIC),
             gamma_ad=13.0 / 9.0, cour=0.8,
             rho_fl_coef=1e-5, rho_fl_pow=-1.5, u_fl_coef=1e-7, u_fl_pow=-2.5, gamma_max=50.0,
             nb=(0, 0, 0), deref_theta_deg=(), deref_factor=(), r_refine_max=0.0, lat_max_level=0)
    p.update(kw)
    return p


def torus_params(n=(32, 16, 16), r_out=50.0, **kw) -> dict:
    """BASELINE.json cfg 0 (r_out=50) / cfg 2 (n=(256,128,128), r_out=1000)."""
    return base_params(n=tuple(n), xmax=(r_out, np.pi, 2.0 * np.pi), **kw)


def minkowski_params(n=(128, 128, 128), **kw) -> dict:
    """BASELINE.json cfg 1: periodic unit cube, gamma_ad = 4/3, no floors that bite."""
    d = dict(metric=METRIC_MINKOWSKI, n=tuple(n), a=0.0, xmin=(0.0, 0.0, 0.0), xmax=(1.0, 1.0, 1.0),
             bc_lo=(BC_PERIODIC,) * 3, bc_hi=(BC_PERIODIC,) * 3, gamma_ad=4.0 / 3.0,
             rho_fl_coef=1e-12, rho_fl_pow=0.0, u_fl_coef=1e-14, u_fl_pow=0.0)
    d.update(kw)
    return base_params(**d)


# ------------------------------------------------------------------------------------------------
# Kerr-Schild metric in the internal coordinates (t, x1 = ln r, theta, phi), numpy, for initial data
# ------------------------------------------------------------------------------------------------
def ks_gcov(a: float, r, th):
    """g_{mu nu} in (t, ln r, theta, phi); returns array [..., 4, 4]."""
    r = np.asarray(r, dtype=np.float64)
    th = np.asarray(th, dtype=np.float64)
    s2 = np.sin(th) ** 2
    Sig = r * r + a * a * np.cos(th) ** 2
    f = 2.0 * r / Sig
    g = np.zeros(np.broadcast(r, th).shape + (4, 4))
    g[..., 0, 0] = -(1.0 - f)
    g[..., 0, 1] = g[..., 1, 0] = f * r
    g[..., 0, 3] = g[..., 3, 0] = -f * a * s2
    g[..., 1, 1] = (1.0 + f) * r * r
    g[..., 1, 3] = g[..., 3, 1] = -a * s2 * (1.0 + f) * r
    g[..., 2, 2] = Sig
    g[..., 3, 3] = s2 * (Sig + a * a * s2 * (1.0 + f))
    return g


def ks_lapse_shift(a: float, r, th):
    """alpha, beta^{x1} (others vanish) and sqrt(-g) in (t, ln r, theta, phi)."""
    Sig = r * r + a * a * np.cos(th) ** 2
    alpha = np.sqrt(Sig / (Sig + 2.0 * r))
    beta1 = 2.0 * r / (Sig + 2.0 * r) / r
    gdet = r * Sig * np.abs(np.sin(th))
    return alpha, beta1, gdet


# ------------------------------------------------------------------------------------------------
# Fishbone-Moncrief torus (Fishbone & Moncrief 1976), SURVEY.md App. A-2
# ------------------------------------------------------------------------------------------------
def fm_l(a: float, r_max: float) -> float:
    """l = u^t u_phi of the prograde circular equatorial geodesic at r_max (Boyer-Lindquist)."""
    r = r_max
    Om = 1.0 / (r ** 1.5 + a)
    gtt, gtp, gpp = -(1.0 - 2.0 / r), -2.0 * a / r, r * r + a * a + 2.0 * a * a / r
    ut = 1.0 / np.sqrt(-(gtt + 2.0 * Om * gtp + Om * Om * gpp))
    return float(ut * ut * (gtp + Om * gpp))


def _fm_lnh_raw(a, l, r, th):
    s = np.sin(th)
    Sig = r * r + a * a * np.cos(th) ** 2
    Del = r * r - 2.0 * r + a * a
    A = (r * r + a * a) ** 2 - Del * a * a * s * s
    X = np.sqrt(1.0 + 4.0 * l * l * Sig * Sig * Del / (A * s) ** 2)
    return 0.5 * np.log((1.0 + X) / (Sig * Del / A)) - 0.5 * X - 2.0 * a * r * l / A, X, A, Sig, Del


def fm_torus_point(a, gam, r, th, r_in=6.0, r_max=12.0, kappa=1e-3):
    """rho/rho_max, u/rho_max, u^t, u^phi (KS = BL components since u^r = 0) and an inside mask."""
    l = fm_l(a, r_max)
    r = np.asarray(r, dtype=np.float64)
    th = np.asarray(th, dtype=np.float64)
    r, th = np.broadcast_arrays(r, th)
    s = np.sin(th)
    ok = (np.abs(s) > 1e-12) & (r >= r_in)
    rs = np.where(ok, r, r_max)
    ths = np.where(ok, th, 0.5 * np.pi)
    lnh0 = _fm_lnh_raw(a, l, np.float64(r_in), np.float64(0.5 * np.pi))[0]
    lnh, X, A, Sig, Del = _fm_lnh_raw(a, l, rs, ths)
    lnh = lnh - lnh0
    inside = ok & (lnh > 0.0)
    h = np.exp(np.where(inside, lnh, 0.0))
    hmax = np.exp(_fm_lnh_raw(a, l, np.float64(r_max), np.float64(0.5 * np.pi))[0] - lnh0)
    rho_max = ((hmax - 1.0) * (gam - 1.0) / (kappa * gam)) ** (1.0 / (gam - 1.0))
    rho = ((h - 1.0) * (gam - 1.0) / (kappa * gam)) ** (1.0 / (gam - 1.0))
    u = kappa * rho ** gam / (gam - 1.0)
    uphi_o = np.sqrt(np.maximum(X - 1.0, 0.0) / 2.0)
    sth = np.sin(ths)
    uphi = 2.0 * a * rs * np.sqrt(1.0 + uphi_o ** 2) / np.sqrt(A * Sig * Del) + np.sqrt(Sig / A) * uphi_o / sth
    gtt = -(1.0 - 2.0 * rs / Sig)
    gtp = -2.0 * a * rs * sth ** 2 / Sig
    gpp = A / Sig * sth ** 2
    # g_tt ut^2 + 2 g_tp ut uphi + g_pp uphi^2 = -1, future-directed root
    bq = 2.0 * gtp * uphi
    cq = gpp * uphi ** 2 + 1.0
    ut = (-bq - np.sqrt(bq * bq - 4.0 * gtt * cq)) / (2.0 * gtt)
    return (np.where(inside, rho / rho_max, 0.0), np.where(inside, u / rho_max, 0.0),
            ut, uphi, inside, dict(l=l, hmax=hmax, rho_max=rho_max))


def grid_coords(p: dict):
    """internal-coordinate centres/faces: x1 = ln r for KS."""
    n = p["n"]
    lo = np.array(p["xmin"], dtype=np.float64)
    hi = np.array(p["xmax"], dtype=np.float64)
    if p["metric"] == METRIC_KS:
        lo[0], hi[0] = np.log(lo[0]), np.log(hi[0])
    dx = (hi - lo) / np.array(n, dtype=np.float64)
    xc = [lo[d] + (np.arange(n[d]) + 0.5) * dx[d] for d in range(3)]
    xf = [lo[d] + np.arange(n[d] + 1) * dx[d] for d in range(3)]
    return xc, xf, dx


def fm_torus(p: dict, seed: int = 0, pert: float = 0.02, beta: float = 100.0, with_B: bool = True,
             r_in: float = 6.0, r_max: float = 12.0, bfac=None, zidx=None, ret_bfac: bool = False):
    """BASELINE.json cfg 0 / cfg 2 initial data.  Returns (hydro[5], bface[3]).
    bfac: field normalisation to use instead of the grid's own (blocks of one grid share the base
    grid's); zidx: zone indices keying the pressure perturbation (default: this grid's own);
    ret_bfac: also return the normalisation."""
    a, gam = p["a"], p["gamma_ad"]
    n = p["n"]
    xc, xf, dx = grid_coords(p)
    r2, th2 = np.meshgrid(np.exp(xc[0]), xc[1], indexing="ij")
    rho_t, u_t, ut, uphi, inside, _ = fm_torus_point(a, gam, r2, th2, r_in, r_max)
    rho_fl = p["rho_fl_coef"] * r2 ** p["rho_fl_pow"]
    u_fl = p["u_fl_coef"] * r2 ** p["u_fl_pow"]
    rho = np.maximum(rho_t, rho_fl)
    u = np.maximum(u_t, u_fl)
    alpha, beta1, gdet = ks_lapse_shift(a, r2, th2)
    # ut^i = u^i + gamma beta^i / alpha, gamma = alpha u^t (C-2 inverted); u^1 = u^2 = 0
    ut1 = np.where(inside, ut * beta1, 0.0)
    ut3 = np.where(inside, uphi, 0.0)
    shape = tuple(n)
    hyd = [np.ascontiguousarray(np.broadcast_to(v[:, :, None], shape)) for v in
           (rho, u, ut1, np.zeros_like(rho), ut3)]
    bface = [np.zeros((n[0] + 1, n[1], n[2])), np.zeros((n[0], n[1] + 1, n[2])),
             np.zeros((n[0], n[1], n[2] + 1))]
    if with_B:
        rc, thc = np.meshgrid(np.exp(xf[0]), xf[1], indexing="ij")      # corners (x1-face, x2-face)
        rho_c = fm_torus_point(a, gam, rc, thc, r_in, r_max)[0]
        Aphi = np.maximum(rho_c - 0.2, 0.0)
        B1 = (Aphi[:, 1:] - Aphi[:, :-1]) / dx[1]                        # (N1+1, N2)
        B2 = -(Aphi[1:, :] - Aphi[:-1, :]) / dx[0]                       # (N1, N2+1)
        # b^2 at centres from the face-mean field, for the beta normalisation only
        Bc1 = 0.5 * (B1[1:, :] + B1[:-1, :]) / gdet
        Bc2 = 0.5 * (B2[:, 1:] + B2[:, :-1]) / gdet
        g = ks_gcov(a, r2, th2)
        ucon = np.zeros(r2.shape + (4,))
        ucon[..., 0] = np.where(inside, ut, 1.0 / alpha)
        ucon[..., 1] = np.where(inside, 0.0, -beta1 / alpha)
        ucon[..., 3] = np.where(inside, uphi, 0.0)
        ucov = np.einsum("...mn,...n->...m", g, ucon)
        bt = Bc1 * ucov[..., 1] + Bc2 * ucov[..., 2]
        bcon = np.zeros_like(ucon)
        bcon[..., 0] = bt
        bcon[..., 1] = (Bc1 + bt * ucon[..., 1]) / ucon[..., 0]
        bcon[..., 2] = (Bc2 + bt * ucon[..., 2]) / ucon[..., 0]
        bcon[..., 3] = (bt * ucon[..., 3]) / ucon[..., 0]
        bsq = np.einsum("...m,...mn,...n->...", bcon, g, bcon)
        pmax = ((gam - 1.0) * u).max()
        fac = bfac
        if fac is None and bsq.max() > 0.0:
            fac = np.sqrt(pmax / (0.5 * bsq.max() * beta))
        if fac is not None:
            bface[0][:] = (fac * B1)[:, :, None]
            bface[1][:] = (fac * B2)[:, :, None]
        bfac = fac
    if pert != 0.0:
        hyd[1] = hyd[1] * (1.0 + pert * rand_pm1(seed, zone_index(n) if zidx is None else zidx))
    if ret_bfac:
        return hyd, bface, bfac
    return hyd, bface


def block_as_grid(p: dict, x_lo, dx, n) -> dict:
    """parameter dict describing ONE block (internal-coordinate corner x_lo, spacing dx, n zones) as a
    grid of its own, for sampling analytic initial data on the blocks of a refined grid"""
    lo = np.array(x_lo, dtype=np.float64)
    hi = lo + np.array(dx, dtype=np.float64) * np.array(n, dtype=np.float64)
    if p["metric"] == METRIC_KS:
        lo[0], hi[0] = np.exp(lo[0]), np.exp(hi[0])
    return dict(p, n=tuple(int(v) for v in n), xmin=tuple(lo), xmax=tuple(hi), nb=(0, 0, 0),
                r_refine_max=0.0, lat_max_level=0, deref_theta_deg=(), deref_factor=())


def base_zone_index(p: dict, x_lo, dx, n) -> np.ndarray:
    """index of the BASE-grid zone containing each zone of a block (both children of a refined zone share
    it), for perturbations that must not depend on the decomposition"""
    xc0, _, dx0 = grid_coords(dict(p, nb=(0, 0, 0)))
    lo0 = [xc0[d][0] - 0.5 * dx0[d] for d in range(3)]
    idx = []
    for d in range(3):
        xc = np.array(x_lo[d]) + (np.arange(int(n[d])) + 0.5) * dx[d]
        idx.append(np.floor((xc - lo0[d]) / dx0[d]).astype(np.int64))
    N = p["n"]
    return ((idx[0][:, None, None] * N[1] + idx[1][None, :, None]) * N[2] + idx[2][None, None, :]).astype(np.uint64)


def fm_torus_blocks(p: dict, infos, seed: int = 0, pert: float = 0.02, beta: float = 100.0):
    """cfg 4: the torus sampled on every block of a (possibly x1-refined) block grid.  infos: per block
    (x_lo, dx, n) in internal coordinates.  Field normalisation from the base grid."""
    _, _, bfac = fm_torus(dict(p, nb=(0, 0, 0), r_refine_max=0.0), seed, pert=0.0, beta=beta, ret_bfac=True)
    out = []
    for x_lo, dx, n in infos:
        pg = block_as_grid(p, x_lo, dx, n)
        out.append(fm_torus(pg, seed, pert, beta, bfac=bfac, zidx=base_zone_index(p, x_lo, dx, n)))
    return out


# ------------------------------------------------------------------------------------------------
# linear MHD eigenmodes on a periodic Minkowski box (BASELINE.json cfg 1)
# ------------------------------------------------------------------------------------------------
def _flat_UF(P, gam, nvec):
    """Flat-space conserved vector and flux along the unit vector nvec for primitives
    (rho, u, ut^i, B^i); complex-safe so that the Jacobians come from complex-step differences.
    Used only to build initial eigenmodes."""
    rho, u = P[0], P[1]
    ut = P[2:5]
    B = P[5:8]
    lor = np.sqrt(1.0 + ut @ ut)
    v = ut / lor
    p = (gam - 1.0) * u
    w = rho + u + p
    vB = v @ B
    b0 = lor * vB
    bsq = (B @ B) / (lor * lor) + vB * vB
    bi = B / lor + b0 * v
    eta = w + bsq
    ptot = p + 0.5 * bsq
    D = rho * lor
    S = eta * lor * lor * v - b0 * bi
    E = eta * lor * lor - ptot - b0 * b0
    vn = v @ nvec
    Bn = B @ nvec
    bn = bi @ nvec
    U = np.concatenate(([D, E - D], S, B))
    # momentum flux T^n_i = eta u^n u_i + ptot n_i - b^n b_i ; energy flux T^{n t} = eta lor^2 v^n - b0 b^n
    Fm = eta * lor * lor * vn * v + ptot * nvec - bn * bi
    Fe = eta * lor * lor * vn - b0 * bn
    F = np.concatenate(([D * vn, Fe - D * vn], Fm, B * vn - Bn * v))
    return U, F


def flat_eigenmodes(gam=4.0 / 3.0, rho=1.0, u=3.0, B=(1.0, np.sqrt(2.0), 0.5), kdir=(1.0, 1.0, 1.0)):
    """Right eigenvectors (max-component normalised) and speeds of the +fast, +Alfven and +slow
    modes of the linearised flat-space system about a static background, along kdir."""
    nvec = np.array(kdir, dtype=np.float64)
    nvec /= np.linalg.norm(nvec)
    P0 = np.array([rho, u, 0.0, 0.0, 0.0, *B], dtype=np.complex128)
    A0 = np.zeros((8, 8))
    An = np.zeros((8, 8))
    h = 1e-30
    for c in range(8):
        Pp = P0.copy()
        Pp[c] += 1j * h
        U, F = _flat_UF(Pp, gam, nvec)
        A0[:, c] = U.imag / h
        An[:, c] = F.imag / h
    lam, R = np.linalg.eig(np.linalg.solve(A0, An))
    lam = lam.real
    R = R.real
    order = np.argsort(-lam)
    out = {}
    for name, q in zip(("fast", "alfven", "slow"), order[:3]):
        r = R[:, q] / np.abs(R[:, q]).max()
        if r[np.argmax(np.abs(r))] < 0:
            r = -r
        out[name] = (float(lam[q]), r)
    return out


def minkowski_waves(p: dict, seed: int = 1, amp: float = 1e-6, noise: float = 1e-8,
                    modes=("fast", "alfven"), t: float = 0.0, B0=(1.0, np.sqrt(2.0), 0.5), box=None):
    """cfg 1: background rho=1, p=1, B0, superposed eigenmodes cos(k.x - omega t), k = 2 pi (1,1,1)
    on the unit cube; face B from an edge vector potential (discretely divergence-free); density
    white noise `noise` from `seed`.  `t` translates the modes (the exact linear solution, P11)."""
    gam = p["gamma_ad"]
    n = p["n"]
    xc, xf, dx = grid_coords(p)
    # box: extent of the periodic box when p describes only a block of it (block_as_grid)
    L = np.array(p["xmax"]) - np.array(p["xmin"]) if box is None else np.array(box, dtype=np.float64)
    k = 2.0 * np.pi / L
    kmag = np.linalg.norm(k)
    u0 = 1.0 / (gam - 1.0)
    em = flat_eigenmodes(gam, 1.0, u0, B0, kdir=k)
    Xc = np.meshgrid(*xc, indexing="ij")
    hyd = [np.full(tuple(n), v) for v in (1.0, u0, 0.0, 0.0, 0.0)]
    bface = [np.full((n[0] + 1, n[1], n[2]), B0[0]), np.full((n[0], n[1] + 1, n[2]), B0[1]),
             np.full((n[0], n[1], n[2] + 1), B0[2])]
    cen = [xc[0][:, None, None], xc[1][None, :, None], xc[2][None, None, :]]
    fac = [xf[0][:, None, None], xf[1][None, :, None], xf[2][None, None, :]]
    for m in modes:
        lam, r = em[m]
        om = lam * kmag
        ph = k[0] * Xc[0] + k[1] * Xc[1] + k[2] * Xc[2] - om * t
        for c in range(5):
            hyd[c] = hyd[c] + amp * r[c] * np.cos(ph)
        dB = amp * r[5:8]
        avec = -np.cross(k, dB) / (kmag * kmag)        # A = avec sin(phase): curl A = dB cos(phase)

        def A_edge(d):   # A_d on d-edges: centred along d, on the faces of the other two directions
            xs = [cen[q] if q == d else fac[q] for q in range(3)]
            return avec[d] * np.sin(k[0] * xs[0] + k[1] * xs[1] + k[2] * xs[2] - om * t)
        A1, A2, A3 = A_edge(0), A_edge(1), A_edge(2)   # (N1,N2+1,N3+1), (N1+1,N2,N3+1), (N1+1,N2+1,N3)
        bface[0] = bface[0] + (A3[:, 1:, :] - A3[:, :-1, :]) / dx[1] - (A2[:, :, 1:] - A2[:, :, :-1]) / dx[2]
        bface[1] = bface[1] + (A1[:, :, 1:] - A1[:, :, :-1]) / dx[2] - (A3[1:, :, :] - A3[:-1, :, :]) / dx[0]
        bface[2] = bface[2] + (A2[1:, :, :] - A2[:-1, :, :]) / dx[0] - (A1[:, 1:, :] - A1[:, :-1, :]) / dx[1]
    if box is None:   # periodic images must be bitwise identical
        bface[0][-1] = bface[0][0]
        bface[1][:, -1] = bface[1][:, 0]
        bface[2][:, :, -1] = bface[2][:, :, 0]
    if noise != 0.0:
        hyd[0] = hyd[0] * (1.0 + noise * rand_pm1(seed, zone_index(n)))
    return hyd, bface


# ------------------------------------------------------------------------------------------------
# BASELINE.json cfg 3: tilted thin disk.  The paper's model is unpublished ("in prep."), so
# this is a synthetic stand-in with the same load pattern: a thin (h/r = 0.03), strongly magnetised sheet
# inclined by 65 degrees that crosses the polar rows.  Not an equilibrium.
# ------------------------------------------------------------------------------------------------
def tilted_disk_params(n=(512, 256, 256), **kw) -> dict:
    return base_params(n=tuple(n), xmax=(1000.0, np.pi, 2.0 * np.pi), **kw)


def _disk_frame(r, th, ph, tilt):
    """Cartesian-like position from the KS spatial coordinates, and cylindrical (R', z') about the axis
    z' = (sin tilt, 0, cos tilt)."""
    st, ct = np.sin(th), np.cos(th)
    x, y, z = r * st * np.cos(ph), r * st * np.sin(ph), r * ct
    ax = np.array([np.sin(tilt), 0.0, np.cos(tilt)])
    zp = x * ax[0] + z * ax[2]
    Rp = np.sqrt(np.maximum(r * r - zp * zp, 0.0))
    return (x, y, z), ax, Rp, zp


def _disk_density(Rp, zp, hr, r_in, r_out):
    Rs = np.maximum(Rp, 1e-3 * r_in)
    H = hr * Rs
    taper = np.where(Rp < 0.9 * r_out, 1.0, 0.5 * (1.0 + np.cos(np.pi * np.clip((Rp - 0.9 * r_out) / (0.1 * r_out), 0.0, 1.0))))
    taper = taper * np.clip((Rp - r_in) / (0.1 * r_in), 0.0, 1.0)      # smooth inner edge over 10 % of r_in
    rho = (r_in / Rs) * np.exp(-np.minimum(0.5 * (zp / H) ** 2, 700.0)) * taper
    p = rho * hr * hr / Rs                                             # c_s = (h/r) v_K
    return rho, p


def tilted_disk(p: dict, seed: int = 3, pert: float = 0.01, beta: float = 10.0, hr: float = 0.03,
                tilt_deg: float = 65.0, r_in: float = 10.0, r_out: float = 100.0):
    """cfg 3 stand-in.  Density (R'/r_in)^-1 exp(-z'^2 / 2H^2), H = hr R', between r_in and r_out (tapered);
    p = rho hr^2 / R'; circular motion Omega = R'^-1.5 about the tilted axis; field from the vector
    potential A = R'^2.5 p z'-hat (purely toroidal in the disk frame), discrete curl on the grid edges,
    scaled to p_max / (b^2/2)_max = beta; rho x (1 + pert U) from seed; floors elsewhere.
    Returns (hydro[5], bface[3])."""
    a, gam, n = p["a"], p["gamma_ad"], p["n"]
    tilt = np.deg2rad(tilt_deg)
    xc, xf, dx = grid_coords(p)
    cen = [np.exp(xc[0])[:, None, None], xc[1][None, :, None], xc[2][None, None, :]]
    fac = [np.exp(xf[0])[:, None, None], xf[1][None, :, None], xf[2][None, None, :]]
    r, th, ph = np.broadcast_arrays(*cen)
    (x, y, z), ax, Rp, zp = _disk_frame(r, th, ph, tilt)
    rho_d, p_d = _disk_density(Rp, zp, hr, r_in, r_out)
    rho_fl = p["rho_fl_coef"] * r ** p["rho_fl_pow"]
    u_fl = p["u_fl_coef"] * r ** p["u_fl_pow"]
    inside = rho_d > rho_fl
    rho = np.where(inside, rho_d, rho_fl)
    u = np.where(inside, np.maximum(p_d / (gam - 1.0), u_fl), u_fl)
    # coordinate velocity of the rotation Omega z'-hat x r:  r-dot = 0
    Om = np.maximum(Rp, r_in) ** -1.5
    vx, vy, vz = Om * (ax[1] * z - ax[2] * y), Om * (ax[2] * x - ax[0] * z), Om * (ax[0] * y - ax[1] * x)
    st = np.maximum(np.sin(th), 1e-12)
    v2 = -vz / (r * st)                                   # theta-dot
    v3 = (x * vy - y * vx) / np.maximum(x * x + y * y, 1e-30)   # phi-dot
    g = ks_gcov(a, r, th)
    nrm = g[..., 0, 0] + 2.0 * g[..., 0, 3] * v3 + g[..., 2, 2] * v2 * v2 + g[..., 3, 3] * v3 * v3
    ok = inside & (nrm < -1e-6)
    ut = np.where(ok, 1.0 / np.sqrt(np.maximum(-nrm, 1e-6)), 0.0)
    alpha, beta1, gdet = ks_lapse_shift(a, r, th)
    hyd = [rho, u, np.where(ok, ut * beta1, 0.0), np.where(ok, ut * v2, 0.0), np.where(ok, ut * v3, 0.0)]
    hyd = [np.ascontiguousarray(h) for h in hyd]

    def A_cov(d, rr, tt, pp):      # covariant component d of A = A_z' z'-hat in (ln r, theta, phi)
        rr, tt, pp = np.broadcast_arrays(rr, tt, pp)
        _, _, Rq, zq = _disk_frame(rr, tt, pp, tilt)
        # A_z' = R'^2.5 p: b^2 / p stays bounded in the wings of the Gaussian (a potential ~ sqrt(p) would make
        # the low-density surface layers magnetically dominated, because surfaces of constant z'/R' flare)
        Az = Rq ** 2.5 * _disk_density(Rq, zq, hr, r_in, r_out)[1]
        s, c, sp, cp = np.sin(tt), np.cos(tt), np.sin(pp), np.cos(pp)
        if d == 0:      # A . d r-vec / d ln r = r A . r-hat
            return Az * rr * (ax[0] * s * cp + ax[2] * c)
        if d == 1:      # r A . theta-hat
            return Az * rr * (ax[0] * c * cp - ax[2] * s)
        return Az * rr * s * (-ax[0] * sp)                 # r sin(theta) A . phi-hat
    A1 = A_cov(0, cen[0], fac[1], fac[2])                  # (N1, N2+1, N3+1)
    A2 = A_cov(1, fac[0], cen[1], fac[2])                  # (N1+1, N2, N3+1)
    A3 = A_cov(2, fac[0], fac[1], cen[2])                  # (N1+1, N2+1, N3)
    bface = [(A3[:, 1:, :] - A3[:, :-1, :]) / dx[1] - (A2[:, :, 1:] - A2[:, :, :-1]) / dx[2],
             (A1[:, :, 1:] - A1[:, :, :-1]) / dx[2] - (A3[1:, :, :] - A3[:-1, :, :]) / dx[0],
             (A2[1:, :, :] - A2[:-1, :, :]) / dx[0] - (A1[:, 1:, :] - A1[:, :-1, :]) / dx[1]]
    del A1, A2, A3
    bface[2][:, :, -1] = bface[2][:, :, 0]                 # periodic images bitwise identical
    # normalisation: p_max / (b^2 / 2)_max = beta, b^2 from the face-mean field and the disk velocity
    Bc = [0.5 * (bface[0][1:] + bface[0][:-1]) / gdet, 0.5 * (bface[1][:, 1:] + bface[1][:, :-1]) / gdet,
          0.5 * (bface[2][:, :, 1:] + bface[2][:, :, :-1]) / gdet]
    ucon = np.zeros(r.shape + (4,))
    ucon[..., 0] = np.where(ok, ut, 1.0 / alpha)
    ucon[..., 1] = np.where(ok, 0.0, -beta1 / alpha)
    ucon[..., 2] = hyd[3]
    ucon[..., 3] = hyd[4]
    ucov = np.einsum("...mn,...n->...m", g, ucon)
    bt = Bc[0] * ucov[..., 1] + Bc[1] * ucov[..., 2] + Bc[2] * ucov[..., 3]
    bcon = np.zeros_like(ucon)
    bcon[..., 0] = bt
    for i in range(3):
        bcon[..., 1 + i] = (Bc[i] + bt * ucon[..., 1 + i]) / ucon[..., 0]
    bsq = np.einsum("...m,...mn,...n->...", bcon, g, bcon)
    fac_b = np.sqrt(((gam - 1.0) * u).max() / (0.5 * bsq.max() * beta)) if bsq.max() > 0 else 0.0
    bface = [np.ascontiguousarray(fac_b * b) for b in bface]
    if pert != 0.0:
        hyd[0] = hyd[0] * (1.0 + pert * rand_pm1(seed, zone_index(n)))
    return hyd, bface
