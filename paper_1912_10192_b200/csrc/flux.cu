// flux.cu — fused reconstruct + HLL kernels, one per direction (north_star items 1+2).
// "finite volume shock-capturing Godunov-based HLLE scheme ... third order accurate
// spatial reconstruction (PPM)"; fluxes are evaluated at cell faces.
// Each face: PPM (or PLM-MC) left/right states of the 7 non-normal primitives (C-5), the normal
// field from the staggered face B, U/F of both states (C-4), fast-speed bounds (C-6), HLL flux of
// the 5 hydro rows and the 2 transverse-B rows (= face EMFs, C-7/C-8), and the per-direction
// maximum signal speed for the Courant step (C-14).
//
// The kernels are bound by the FP64 pipe (64 lanes per SM), not by HBM, so the
// design minimises fp64 instructions per face:
//  * every zone's parabola is built ONCE and shared by its two faces: along x1 / x2 a thread
//    marches along the sweep direction carrying the previous zone's right edge in registers (loads
//    stay coalesced along x3); along x3 neighbouring lanes exchange the edge with a warp shuffle;
//  * reconstruction is branch-free (selects, no divergence), divisions by constants are
//    multiplications, each state needs 3 reciprocals and 2 square roots in total.
#include "hamr_host.h"

namespace hamr {

constexpr double SIXTH = 1.0 / 6.0;

// ---- C-5 reconstruction, branch-free ----------------------------------------------------------------
// "dl and dr have the same sign" read off the sign bits (integer pipe; the FP64 pipe is the one these kernels
// saturate).  A zero on either side makes the limited quantity zero by itself, so no product is needed.
__device__ __forceinline__ bool same_sign(double a, double b) { return (__double2hiint(a) ^ __double2hiint(b)) >= 0; }

// van Leer / CW84 limited slope from dl = a_j - a_{j-1}, dr = a_{j+1} - a_j, dc = (a_{j+1} - a_{j-1})/2:
// sign(dc) min(|dc|, 2 |dl|, 2 |dr|) where dl, dr agree in sign, else 0.  The minimum is taken over the SIGNED
// values by magnitude (the compares take |.| as operand modifiers, the selects move the raw words) and the sign
// is imposed once at the end, so no absolute value is ever materialised on the FP64 pipe.
__device__ __forceinline__ double lim_slope(double dl, double dr, double dc) {
  const double m = 2.0 * (fabs(dl) < fabs(dr) ? dl : dr);
  const double lim = fabs(dc) < fabs(m) ? dc : m;
  return same_sign(dl, dr) ? copysign(lim, dl) : 0.0;   // sign(dc) = sign(dl) where the slope survives
}

// TWICE that slope from dl, dr and ds = a_{j+1} - a_{j-1} = 2 dc: sign min(|ds|, 4 |dl|, 4 |dr|).  Scaling by powers of
// two is exact, so 2 lim_slope(dl, dr, ds / 2) == lim_slope2(dl, dr, ds) bit for bit; PPM only ever needs differences of
// slopes times a constant (ppm_iface2), which saves the halving of every centred difference on the FP64 pipe.
__device__ __forceinline__ double lim_slope2(double dl, double dr, double ds) {
  const double m = 4.0 * (fabs(dl) < fabs(dr) ? dl : dr);
  const double lim = fabs(ds) < fabs(m) ? ds : m;
  return same_sign(dl, dr) ? lim : 0.0;   // where dl and dr agree in sign, ds and m carry that sign already
}

// interface value a_{j+1/2} from a_j, d = a_{j+1} - a_j and TWICE the limited slopes of zones j and j+1
constexpr double TWELFTH = 1.0 / 12.0;   // exactly SIXTH / 2
__device__ __forceinline__ double ppm_iface2(double aj, double d, double dm2_j, double dm2_jp) {
  return aj + 0.5 * d - (dm2_jp - dm2_j) * TWELFTH;
}

// monotonised parabola edges of a zone with mean a and interface values l (low side), r (high side)
// CW84 (1.10) in one-sided differences dl = a - l, dr = r - a: where the zone is not an extremum (dl dr > 0) the
// overshoot tests (r - l)(a - (l + r)/2) > (r - l)^2 / 6 and < -(r - l)^2 / 6 divide through by (r - l) to
// |dl| > 2 |dr| and |dr| > 2 |dl|, and the reset edges 3a - 2r, 3a - 2l are a - 2 dr, a + 2 dl; every switch is
// continuous, so the rounding of a test does not matter.  dl = 0 or dr = 0 needs no case of its own: the
// overshoot tests then reset the other edge to a as well.
__device__ __forceinline__ void ppm_mono(double l, double a, double r, double& aL, double& aR) {
  const double dl = a - l, dr = r - a;
  const bool flat = !same_sign(dl, dr);
  // |dl| > 2 |dr| and |dr| > 2 |dl| as the sign of ONE fused multiply-add each (the difference of two doubles is never
  // rounded to zero, so the sign is exact), read off the high word: one FP64 instruction per test instead of two
  const bool over = __double2hiint(fma(-2.0, fabs(dr), fabs(dl))) > 0;
  const bool under = __double2hiint(fma(-2.0, fabs(dl), fabs(dr))) > 0;
  // the resets as PREDICATED writes over l and r (one instruction each instead of the reset value plus two word selects)
  aL = l;
  aR = r;
  asm("{\n\t.reg .pred p;\n\tsetp.ne.s32 p, %1, 0;\n\t@p fma.rn.f64 %0, %2, %3, %4;\n\t}"
      : "+d"(aL) : "r"((int)over), "d"(-2.0), "d"(dr), "d"(a));
  asm("{\n\t.reg .pred p;\n\tsetp.ne.s32 p, %1, 0;\n\t@p fma.rn.f64 %0, %2, %3, %4;\n\t}"
      : "+d"(aR) : "r"((int)(!over && under)), "d"(2.0), "d"(dl), "d"(a));
  asm("{\n\t.reg .pred p;\n\tsetp.ne.s32 p, %2, 0;\n\t@p mov.f64 %0, %3;\n\t@p mov.f64 %1, %3;\n\t}"
      : "+d"(aL), "+d"(aR) : "r"((int)flat), "d"(a));
}

// parabola edges (aL at j-1/2, aR at j+1/2) of zone j from a0..a4 = a[j-2..j+2]
__device__ __forceinline__ void ppm_edges(double a0, double a1, double a2, double a3, double a4, double& aL,
                                          double& aR) {
  const double d10 = a1 - a0, d21 = a2 - a1, d32 = a3 - a2, d43 = a4 - a3;
  const double dm_m = lim_slope2(d10, d21, a2 - a0);
  const double dm_0 = lim_slope2(d21, d32, a3 - a1);
  const double dm_p = lim_slope2(d32, d43, a4 - a2);
  ppm_mono(ppm_iface2(a1, d21, dm_m, dm_0), a2, ppm_iface2(a2, d32, dm_0, dm_p), aL, aR);
}

// PLM with the MC limiter: minmod(2(a1-a0), (a2-a0)/2, 2(a2-a1))
__device__ __forceinline__ void plm_edges(double a0, double a1, double a2, double& aL, double& aR) {
  const double s = lim_slope(a1 - a0, a2 - a1, 0.5 * (a2 - a0));
  aL = a1 - 0.5 * s;
  aR = a1 + 0.5 * s;
}

template <int RECON>
__device__ __forceinline__ void zone_edges(const double* __restrict__ a, int sd, double& aL, double& aR) {
  if (RECON == HAMR_RECON_PPM) ppm_edges(a[-2 * sd], a[-sd], a[0], a[sd], a[2 * sd], aL, aR);
  else plm_edges(a[-sd], a[0], a[sd], aL, aR);
}

// ---- C-2..C-7 on one face ------------------------------------------------------------------------------
// The face record (hamr_dev.cuh FREC_*): the 3+1 split of the face metric.  With u^mu = ut^mu + gamma n^mu and
// n_i = 0 the spatial covariant components need the spatial metric only, u_i = g_ij ut^j, and
// u_t = -alpha gamma + beta^i u_i; likewise b_i = g_ij (b^j + beta^j b^t), b_t = -alpha^2 b^t + beta^i b_i.
// Both metrics have beta^2 = beta^3 = 0 and g_12 = g_23 = 0.
struct FGeo {
  double c11, c13, c22, c33;                 // g_ij
  double alpha, ialpha, boa, beta1, nalpha2; // lapse, 1/lapse, beta^1/lapse, beta^1, -lapse^2
  double k00, kdd, k0d;                      // g^{tt}, g^{dd}, g^{td}
  double gdet, igdet;
};

__device__ __forceinline__ FGeo load_fgeo(const double* __restrict__ rec) {
  double v[NREC_F];
  load_rec(rec, NREC_F - 2, v);
  FGeo G;
  G.c11 = v[FREC_C11]; G.c13 = v[FREC_C13]; G.c22 = v[FREC_C22]; G.c33 = v[FREC_C33];
  G.alpha = v[FREC_ALPHA]; G.ialpha = v[FREC_IALPHA]; G.boa = v[FREC_BOA]; G.beta1 = v[FREC_BETA1];
  G.nalpha2 = v[FREC_NALPHA2]; G.k00 = v[FREC_K00]; G.kdd = v[FREC_KDD]; G.k0d = v[FREC_K0D];
  G.gdet = v[FREC_GDET]; G.igdet = v[FREC_IGDET];
  return G;
}

// the same record from shared memory (every thread of the CTA reads the same words: a broadcast)
__device__ __forceinline__ FGeo load_fgeo_shared(const double* rec) {
  const double2* r2 = reinterpret_cast<const double2*>(rec);
  double v[NREC_F];
#pragma unroll
  for (int q = 0; q < (NREC_F - 2) / 2; q++) { const double2 w = r2[q]; v[2 * q] = w.x; v[2 * q + 1] = w.y; }
  FGeo G;
  G.c11 = v[FREC_C11]; G.c13 = v[FREC_C13]; G.c22 = v[FREC_C22]; G.c33 = v[FREC_C33];
  G.alpha = v[FREC_ALPHA]; G.ialpha = v[FREC_IALPHA]; G.boa = v[FREC_BOA]; G.beta1 = v[FREC_BETA1];
  G.nalpha2 = v[FREC_NALPHA2]; G.k00 = v[FREC_K00]; G.kdd = v[FREC_KDD]; G.k0d = v[FREC_K0D];
  G.gdet = v[FREC_GDET]; G.igdet = v[FREC_IGDET];
  return G;
}

// What the HLL combination needs from one side of the face.  The rows of U and F are never formed: with
// T^mu_nu = eta u^mu u_nu + ptot delta^mu_nu - b^mu b_nu (eta = w + b^2, ptot = p + b^2/2) a weighted sum
// wF F_nu + wU U_nu of the flux and conserved rows is (eta X) u_nu - Y b_nu + wF ptot delta^d_nu with the two scalars
// X = wF u^d + wU u^t, Y = wF b^d + wU b^t: two FMAs per row and side instead of six.
struct Side {
  double rho, ut, ud, eta, ptot, b0, bd;
  double ul[4], bl[4];   // u_mu, b_mu
  double Be, Bf, Fe, Ff; // transverse field components and their flux rows b^e u^d - b^d u^e (C-4)
  double a2, vp, vm;     // C-6: the speed bounds are vp / a2 and -vm / a2, a2 > 0
};

template <int D>
__device__ __forceinline__ void side_state(const double P[8], const FGeo& G, double gam_ad, Side& S) {
  constexpr int dir = D + 1, e = (D + 1) % 3, f = (D + 2) % 3;
  // C-2, C-3
  St T;
  state_3p1(P, G.c11, G.c13, G.c22, G.c33, G.alpha, G.ialpha, G.boa, G.beta1, G.nalpha2, T);
  const double u[4] = {T.ut, T.u1, T.u2, T.u3}, b[4] = {T.b0, T.b1, T.b2, T.b3};
  const double bsq = T.bsq;
  S.ul[0] = T.ul0; S.ul[1] = T.ul1; S.ul[2] = T.ul2; S.ul[3] = T.ul3;
  S.bl[0] = T.bl0; S.bl[1] = T.bl1; S.bl[2] = T.bl2; S.bl[3] = T.bl3;
  // C-4
  const double p = (gam_ad - 1.0) * P[1];
  const double w = P[0] + gam_ad * P[1];
  S.rho = P[0];
  S.ut = u[0];
  S.ud = u[dir];
  S.b0 = b[0];
  S.bd = b[dir];
  S.eta = w + bsq;
  S.ptot = p + 0.5 * bsq;
  S.Be = P[5 + e];
  S.Bf = P[5 + f];
  S.Fe = b[1 + e] * u[dir] - b[dir] * u[1 + e];
  S.Ff = b[1 + f] * u[dir] - b[dir] * u[1 + f];
  // C-6: c_m^2 = c_s^2 + v_A^2 - c_s^2 v_A^2 with c_s^2 = gamma p / w, v_A^2 = b^2 / (b^2 + w)
  // = N / Dq with Dq = w (w + b^2) > 0; the quadratic a2 v^2 - 2 h v + a0 = 0 is multiplied through by Dq (same
  // roots, no division).  With M = Dq - N >= 0: a2 = (u^t)^2 M - g^tt N > 0 (g^tt < 0), so the larger root is
  // (h + sqrt(h^2 - a2 a0)) / a2 and the smaller one (h - sqrt(..)) / a2
  const double gp = gam_ad * p;
  const double Dq = w * S.eta;
  const double N = dmin(dmax(gp * S.eta + bsq * (w - gp), 0.0), Dq);  // clamp c_m^2 to [0, 1]
  const double M = Dq - N;
  S.a2 = (u[0] * u[0]) * M - G.k00 * N;
  const double h = (u[dir] * u[0]) * M - G.k0d * N;
  const double a0 = (u[dir] * u[dir]) * M - G.kdd * N;
  const double disc = sqrt_pos(dmax(h * h - S.a2 * a0, 1e-300));   // the floor is ~1e-130 of the scale of h
  S.vp = h + disc;
  S.vm = disc - h;
}

// HLL (C-7) from the two states: the 7 outputs of the face (5 hydro fluxes, E_f, E_e); returns ctop.
// ENT (C-18): PL[8], PR[8] hold the reconstructed kappa and out[7] receives the flux of the entropy row, which is
// carried by the two parts of the mass flux: kappa_L (rho X)_L + kappa_R (rho X)_R (no flush: C-7a is about CT)
template <int D, bool ENT = false>
__device__ __forceinline__ double face_flux(const double* __restrict__ PL, const double* __restrict__ PR, const FGeo& G,
                                            double gam_ad, double* __restrict__ out) {
  constexpr int dir = D + 1;
  Side L, R;
  side_state<D>(PL, G, gam_ad, L);
  side_state<D>(PR, G, gam_ad, R);
  const double ia = rcp_nr(L.a2 * R.a2);   // one reciprocal for both sides
  const double iL = R.a2 * ia, iR = L.a2 * ia;
  const double cmax = dmax(0.0, dmax(L.vp * iL, R.vp * iR));
  const double cmin = dmax(0.0, dmax(L.vm * iL, R.vm * iR));
  const double sum = cmax + cmin;
  const bool avg = sum < 1e-300;
  const double isg = G.gdet * rcp_nr(sum);
  // F = g [cmax FL + cmin FR - cmax cmin (UR - UL)] / (cmax + cmin);  average if both speeds vanish
  double wl = cmax * isg, wr = cmin * isg;
  if (__builtin_expect(avg, 0)) wl = wr = 0.5 * G.gdet;   // (a branch no lane takes: no select on the common path)
  const double wc = wl * cmin;              // avg: cmin = 0
  const double XL = wl * L.ud + wc * L.ut, XR = wr * R.ud - wc * R.ut;
  double Fh0 = L.rho * XL + R.rho * XR;
  if (ENT) out[7] = PL[8] * (L.rho * XL) + PR[8] * (R.rho * XR);
  // C-7a: a mass flux below 1e-12 of the magnitude of its own HLL terms is rounding noise and is
  // flushed to exactly 0, so that the upwind selector of C-9 sees a tie
  const double mag = L.rho * (wl * fabs(L.ud) + wc * L.ut) + R.rho * (wr * fabs(R.ud) + wc * R.ut);
  if (!avg && fabs(Fh0) <= 1e-12 * mag) Fh0 = 0.0;
  const double AL = L.eta * XL, AR = R.eta * XR;
  const double YL = wl * L.bd + wc * L.b0, YR = wr * R.bd - wc * R.b0;
  double Fh[4];
#pragma unroll
  for (int c = 0; c < 4; c++) Fh[c] = (AL * L.ul[c] - YL * L.bl[c]) + (AR * R.ul[c] - YR * R.bl[c]);
  Fh[dir] += wl * L.ptot + wr * R.ptot;   // delta^d_nu of the flux rows
  Fh[0] += wc * (L.ptot - R.ptot);        // delta^t_nu of the conserved rows
  out[0] = Fh0;
  out[1] = Fh[0] + Fh0;   // the energy row carries T^d_t + rho u^d (C-4)
#pragma unroll
  for (int c = 1; c < 4; c++) out[1 + c] = Fh[c];
  out[5] = -(wl * L.Fe + wr * R.Fe - wc * (R.Be - L.Be));  // C-8: on a d-face, E_f = -F^d(B^e)
  out[6] = wl * L.Ff + wr * R.Ff - wc * (R.Bf - L.Bf);     //                    E_e = +F^d(B^f)
  return dmax(cmax, cmin);
}

__device__ __forceinline__ void store_face(const Dev& Dv, int D, int z, const double out[7]) {
#pragma unroll
  for (int c = 0; c < 5; c++) Dv.F[D][c][z] = out[c];
  Dv.EfB[D][z] = out[5];
  Dv.EfA[D][z] = out[6];
}

// all three kinds of call sites: HLL on one face, results to the face arrays at z
template <int D, bool ENT = false>
__device__ __forceinline__ double face_flux(const double* __restrict__ PL, const double* __restrict__ PR, const FGeo& G,
                                            double gam_ad, const Dev& Dv, int z) {
  double out[8];
  const double ct = face_flux<D, ENT>(PL, PR, G, gam_ad, out);
  store_face(Dv, D, z, out);
  if (ENT) Dv.FK[D][z] = out[7];
  return ct;
}

__device__ __forceinline__ void zero_face(const Dev& Dv, int D, int z) {
  for (int c = 0; c < 5; c++) Dv.F[D][c][z] = 0.0;
  Dv.EfA[D][z] = 0.0;
  Dv.EfB[D][z] = 0.0;
  if (Dv.entropy) Dv.FK[D][z] = 0.0;
}

// C-14 / H5: per-direction maximum signal speed: warp-shuffle max, then one atomic max per warp on the
// bit pattern of the positive double.  BLK: one maximum per block (a warp may straddle two blocks).
template <bool BLK>
__device__ __forceinline__ void ctop_commit(const Dev& Dv, int D, int b, double ctop) {
  if (!BLK) {
    ctop = warp_max(ctop);
    if ((threadIdx.x & 31) == 0 && ctop > 0.0) atomic_max_pos(Dv.scal + S_CTOP0 + D, ctop);
    return;
  }
  const int b0 = __shfl_sync(0xffffffffu, b, 0);
  if (__all_sync(0xffffffffu, b == b0)) {
    ctop = warp_max(ctop);
    if ((threadIdx.x & 31) == 0 && ctop > 0.0) atomic_max_pos(Dv.B.ctopb + b0 * 3 + D, ctop);
  } else if (ctop > 0.0) {
    atomic_max_pos(Dv.B.ctopb + b * 3 + D, ctop);
  }
}

// ---- sweeps along x1 / x2: a thread marches along the sweep direction ---------------------------------
// grid.x covers the flattened transverse index (other, k), k fastest; grid.y the segments of `seg` faces.
// PPM: the thread carries, per variable, a_j, a_{j+1}, the limited slope of zone j and the interface
// value a_{j-1/2}; each step loads ONE new value a_{j+2}, builds ONE new slope and ONE new interface
// value (the expressions are those of ppm_edges, so the result is bitwise the same).
// Tuning constants of the generic kernels, each the best of a measured sweep on cfg 2 (round 1):
// 128 threads per CTA at 128 registers (4 CTAs per SM) for the marching kernels, 96 registers (5 CTAs) for the x3 sweep;
// a_j, a_{j+1} are re-read from L1 each step instead of being carried in registers.
constexpr int MARCH_T = 128, MARCH_MINB = 4, X3_MINB = 5;
// BLK: the launch covers the blocks of Dv.B.list (block-structured grid, H7); s / s2 are the buffer sets
// holding the stage source of blocks with cur == 0 / cur == 2.
// ENT (C-18, monolithic grids): kappa of the zones (Dv.K) is reconstructed as an eighth variable for the entropy flux.
template <int D, int RECON, bool BLK, bool ENT = false>
__global__ void __launch_bounds__(MARCH_T, ENT ? 3 : MARCH_MINB) k_flux_march(Dev Dv, Fields s, Fields s2, int seg,
                                                                                int want_ctop) {
  static_assert(D == 0 || D == 1, "marching kernels sweep x1 or x2");
  const Lay& L = Dv.L;
  constexpr int O = 1 - D;          // the other non-x3 dimension
  constexpr int e = (D + 1) % 3, f = (D + 2) % 3;
  const int ck = L.n[2] + 2;
  const int ntr = (L.n[O] + 2) * ck;
  int tf = blockIdx.x * blockDim.x + threadIdx.x;
  int bslot = 0;
  if (BLK) { bslot = tf / ntr; tf -= bslot * ntr; }
  const bool live = BLK ? bslot < Dv.B.nact : tf < ntr;
  const BCtx C = blk_ctx<BLK>(Dv, BLK ? min(bslot, Dv.B.nact - 1) : 0);
  const int ge2 = BLK ? Dv.B.ge2 : L.e2, n2g = BLK ? Dv.B.n2g : L.n[1];
  double ctop = 0.0;
  if (live) {
    const int k = tf % ck - 1, o = tf / ck - 1;
    const int f0 = blockIdx.y * seg, f1 = min(f0 + seg, L.n[D] + 1);
    const int sd = (D == 0) ? L.S1 : L.S2;
    const bool act = o >= 0 && o < L.n[O] && k >= 0 && k < L.n[2];  // C-14: faces of ACTIVE zones
    const bool ks = Dv.metric == HAMR_METRIC_KERR_SCHILD;
    constexpr int NVR = ENT ? 8 : 7;   // reconstructed variables
    const double* var[8] = {selp<BLK>(s.P[0], s2.P[0], C.cur), selp<BLK>(s.P[1], s2.P[1], C.cur),
                            selp<BLK>(s.P[2], s2.P[2], C.cur), selp<BLK>(s.P[3], s2.P[3], C.cur),
                            selp<BLK>(s.P[4], s2.P[4], C.cur), selp<BLK>(s.Bc[e], s2.Bc[e], C.cur),
                            selp<BLK>(s.Bc[f], s2.Bc[f], C.cur), Dv.K};
    const double* bfn = selp<BLK>(s.Bf[D], s2.Bf[D], C.cur);
    const double* gtab = (D == 0 ? Dv.gf1A : Dv.gf2A) + (BLK ? C.lev * Dv.B.tlevA : 0);
    constexpr int slot[8] = {0, 1, 2, 3, 4, 5 + e, 5 + f, 8};
    int z = C.zoff + (int)L.idx(D == 0 ? f0 - 1 : o, D == 0 ? o : f0 - 1, k);
    double PL[9], PR[9];
    double dm[8], il[8];  // PPM marching state (unused for PLM)
    // the zone below the first face: its right edge, and the marching state of the next zone
#pragma unroll
    for (int v = 0; v < NVR; v++) {
      const double* a = var[v] + z;
      if (RECON == HAMR_RECON_PPM) {
        const double m2 = a[-2 * sd], m1 = a[-sd], c0 = a[0], p1 = a[sd], p2 = a[2 * sd];
        const double d10 = m1 - m2, d21 = c0 - m1, d32 = p1 - c0, d43 = p2 - p1;
        const double dm_m = lim_slope2(d10, d21, c0 - m2);
        const double dm_0 = lim_slope2(d21, d32, p1 - m1);
        const double dm_p = lim_slope2(d32, d43, p2 - c0);
        const double r = ppm_iface2(c0, d32, dm_0, dm_p);
        double aL;
        ppm_mono(ppm_iface2(m1, d21, dm_m, dm_0), c0, r, aL, PL[slot[v]]);
        dm[v] = dm_p; il[v] = r;
      } else {
        double aL;
        plm_edges(a[-sd], a[0], a[sd], aL, PL[slot[v]]);
      }
    }
    for (int fc = f0; fc < f1; fc++) {
      z += sd;
      double carry[8];
#pragma unroll
      for (int v = 0; v < NVR; v++) {
        const double* a = var[v] + z;
        if (RECON == HAMR_RECON_PPM) {
          const double a2 = a[2 * sd];
          const double c0 = a[0], c1 = a[sd];
          const double d21 = c1 - c0, d32 = a2 - c1;
          const double dmp = lim_slope2(d21, d32, a2 - c0);
          const double r = ppm_iface2(c0, d21, dm[v], dmp);
          ppm_mono(il[v], c0, r, PR[slot[v]], carry[v]);
          dm[v] = dmp; il[v] = r;
        } else {
          plm_edges(a[-sd], a[0], a[sd], PR[slot[v]], carry[v]);
        }
      }
      const bool pole = (D == 1) && ks && (C.J0 + fc == 0 || C.J0 + fc == n2g);
      if (pole) {  // C-7: pole faces carry no flux and no state is evaluated there
        zero_face(Dv, D, z);
      } else {
        const int q = C.q0 + ((D == 0) ? fc * ge2 + o : o * ge2 + fc);
        const FGeo G = load_fgeo(gtab + (size_t)q * NREC_F);
        PL[5 + D] = PR[5 + D] = bfn[z] * G.igdet;  // C-5: the normal field is single-valued at the face
        const double ct = face_flux<D, ENT>(PL, PR, G, Dv.gam, Dv, z);
        if (act) ctop = dmax(ctop, ct);
      }
#pragma unroll
      for (int v = 0; v < NVR; v++) PL[slot[v]] = carry[v];
    }
  }
  if (want_ctop) ctop_commit<BLK>(Dv, D, C.b, ctop);
}

// ---- sweeps along x1 / x2 through a shared-memory ring filled by bulk asynchronous copies (TMA) -----------
// north_star: "per-direction fused reconstruct+HLL kernels that stage stencil tiles through shared memory or TMA".
// Monolithic grids with PPM whose x3 extent is a multiple of the CTA width KT and periodic.  A CTA owns KT
// consecutive x3 positions of ONE transverse row o and marches over a segment of faces; every row of the sweep it
// needs (7 variables and the normal face field, KT doubles each, plus the 128-byte geometry record of the row's
// face: all threads of the CTA are on the same (x1, x2)) is brought into a ring of RING slots by 9 bulk copies
// (cp.async.bulk, completion on an mbarrier) issued three rows ahead by one thread.  The marching loop reads shared
// memory only: no load of the loop can miss a cache, no address arithmetic per variable, and the rows in flight
// hold no registers.  The x3-faces of the transverse ghost columns k = -1 and k = n3, which C-9 reads, are the
// periodic images of columns n3 - 1 and 0: their threads store twice.
namespace ring {
constexpr int RING = 6;   // 3 live rows (zones fc, fc + 1, fc + 2) + the rows in flight
static_assert(RING >= 6, "three live rows, one dying, two in flight");
}  // namespace ring

// resident warps per SM the register budget of the staged kernels is set for: 12 (168 registers, no spills) measured
// best of 8 / 10 / 11 / 12 / 13-16 (profiles/r2_experiments.md)
constexpr int RING_WARPS = 12;
// ENT (C-18): kappa of the zones (Dv.K) is a ninth staged array and an eighth reconstructed variable; the flux of the
// entropy row goes to Dv.FK[D] (still 168 registers without spills).
template <int D, int KT, bool ENT = false>
__global__ void __launch_bounds__(KT, RING_WARPS * 32 / KT) k_flux_ring(Dev Dv, Fields s, int seg, int want_ctop) {
  static_assert(D == 0 || D == 1, "marching kernels sweep x1 or x2");
  using namespace ring;
  using namespace tma;
  constexpr int O = 1 - D;
  constexpr int e = (D + 1) % 3, f = (D + 2) % 3;
  constexpr int NW = KT / 32;              // warps of the CTA; warp 0 also is the producer
  constexpr int NVR = ENT ? 8 : 7;         // reconstructed variables
  constexpr int KOFF = 8 * KT + NREC_F;    // where kappa sits in a slot (ENT)
  constexpr int SLOTD = (ENT ? 9 : 8) * KT + NREC_F;   // doubles per ring slot: 7 variables, the face field, the face record (, kappa)
  constexpr int voff[8] = {0, KT, 2 * KT, 3 * KT, 4 * KT, 5 * KT, 6 * KT, KOFF};
  extern __shared__ __align__(128) double ring_mem[];
  unsigned long long* mbar = reinterpret_cast<unsigned long long*>(ring_mem + RING * SLOTD);   // slot filled
  unsigned long long* mbe = mbar + RING;                                                         // slot released
  const Lay& L = Dv.L;
  const int t = threadIdx.x;
  const int k0 = blockIdx.x * KT, k = k0 + t;
  const int o = (int)blockIdx.y - 1;
  const int f0 = blockIdx.z * seg, f1 = min(f0 + seg, L.n[D] + 1);
  const int sd = (D == 0) ? L.S1 : L.S2;
  const int rbase = f0 - 3, rlast = f1 + 1;   // rows (zones along the sweep) this CTA reads
  const double* gtab = (D == 0 ? Dv.gf1A : Dv.gf2A);
  // The producer is one elected lane of warp 0: the next row of every array, and the record of its face, into the
  // next slot.  Its state (row, slot, padded offset of the row, record index) is the same in every thread and
  // advances by constants, so it lives in uniform registers.  A slot is refilled one step after the row in it died:
  // the other warps have announced on the slot's second barrier that they are done with it, and warp 0 waits on that
  // barrier only if one of them lags by more than a step (no CTA-wide barrier inside the loop).
  int prow = rbase, pslot = 0;
  int pz = (int)L.idx(D == 0 ? rbase : o, D == 0 ? o : rbase, k0);
  int pq = (NG * L.e2 + NG) + ((D == 0) ? rbase * L.e2 + o : o * L.e2 + rbase);
  const bool warp0 = t < 32;
  auto issue_next = [&]() {
    if (warp0) {
      if (NW > 1 && prow >= rbase + RING) mbar_wait(mbe + pslot, (unsigned)(((prow - rbase) / RING - 1) & 1));
      if (elect_one()) {
        double* dst = ring_mem + pslot * SLOTD;
        unsigned long long* mb = mbar + pslot;
        const bool face = prow >= f0 && prow < f1;   // rows that are also faces of this segment carry field and record
        mbar_expect(mb, (unsigned)(((face ? 8 * KT + NREC_F : 7 * KT) + (ENT ? KT : 0)) * sizeof(double)));
        if (ENT) bulk_g2s(dst + KOFF, Dv.K + pz, KT * sizeof(double), mb);
        bulk_g2s(dst + 0 * KT, s.P[0] + pz, KT * sizeof(double), mb);
        bulk_g2s(dst + 1 * KT, s.P[1] + pz, KT * sizeof(double), mb);
        bulk_g2s(dst + 2 * KT, s.P[2] + pz, KT * sizeof(double), mb);
        bulk_g2s(dst + 3 * KT, s.P[3] + pz, KT * sizeof(double), mb);
        bulk_g2s(dst + 4 * KT, s.P[4] + pz, KT * sizeof(double), mb);
        bulk_g2s(dst + 5 * KT, s.Bc[e] + pz, KT * sizeof(double), mb);
        bulk_g2s(dst + 6 * KT, s.Bc[f] + pz, KT * sizeof(double), mb);
        if (face) {
          bulk_g2s(dst + 7 * KT, s.Bf[D] + pz, KT * sizeof(double), mb);
          bulk_g2s(dst + 8 * KT, gtab + (size_t)pq * NREC_F, NREC_F * sizeof(double), mb);
        }
      }
    }
    prow++;
    pslot = (pslot + 1 == RING) ? 0 : pslot + 1;
    pz += sd;
    pq += (D == 0) ? L.e2 : 1;
  };
  if (t == 0) {
    for (int c = 0; c < RING; c++) { mbar_init(mbar + c, 1); mbar_init(mbe + c, NW > 1 ? NW - 1 : 1); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
#pragma unroll 1
  for (int c = 0; c < RING; c++)
    if (prow <= rlast) issue_next();
  const bool act = o >= 0 && o < L.n[O];  // C-14: faces of ACTIVE zones (every k of the launch is active)
  const bool ks = Dv.metric == HAMR_METRIC_KERR_SCHILD;
  constexpr int slot[8] = {0, 1, 2, 3, 4, 5 + e, 5 + f, 8};
  int z = (int)L.idx(D == 0 ? f0 - 1 : o, D == 0 ? o : f0 - 1, k);
  // the periodic images: column n3 - 1 also is column -1, column 0 also is column n3
  const int dup = (k == L.n[2] - 1) ? -L.n[2] : (k == 0 ? L.n[2] : 0);
  double PL[9], PR[9], dm[8], il[8];
  double ctop = 0.0;
  // prologue: the parabola of zone f0 - 1 from rows f0 - 3 .. f0 + 1 (slots 0 .. 4 of the first revolution)
#pragma unroll
  for (int c = 0; c < 5; c++) mbar_wait(mbar + c, 0);
  {
    const double* a = ring_mem + t;
#pragma unroll
    for (int v = 0; v < NVR; v++) {
      const double m2 = a[0 * SLOTD + voff[v]], m1 = a[1 * SLOTD + voff[v]], c0 = a[2 * SLOTD + voff[v]],
                   p1 = a[3 * SLOTD + voff[v]], p2 = a[4 * SLOTD + voff[v]];
      const double d10 = m1 - m2, d21 = c0 - m1, d32 = p1 - c0, d43 = p2 - p1;
      const double dm_m = lim_slope2(d10, d21, c0 - m2);
      const double dm_0 = lim_slope2(d21, d32, p1 - m1);
      const double dm_p = lim_slope2(d32, d43, p2 - c0);
      const double r = ppm_iface2(c0, d32, dm_0, dm_p);
      double aL;
      ppm_mono(ppm_iface2(m1, d21, dm_m, dm_0), c0, r, aL, PL[slot[v]]);
      dm[v] = dm_p; il[v] = r;
    }
  }
  // unrolled by two: the marching state alternates between two register sets instead of being moved at the loop end
#pragma unroll 2
  for (int fc = f0; fc < f1; fc++) {
    z += sd;
    __syncwarp();
    const int n0 = fc - rbase;   // ring position of row fc; rows fc + 1, fc + 2 follow
    const int s0 = n0 % RING, s1 = (n0 + 1) % RING, s2 = (n0 + 2) % RING;
    if (NW > 1 && !warp0 && (t & 31) == 0) {   // this warp is done with the rows below fc
      if (fc == f0) { mbar_arrive(mbe + 0); mbar_arrive(mbe + 1); mbar_arrive(mbe + 2); }
      else mbar_arrive(mbe + (n0 + RING - 1) % RING);
    }
    // the rows that died a step ago are replaced (after the prologue: the first two of its three dead rows)
#pragma unroll 1
    while (prow <= rlast && prow <= fc - 2 + RING) issue_next();
    mbar_wait(mbar + s2, (unsigned)(((n0 + 2) / RING) & 1));
    const double* r0 = ring_mem + s0 * SLOTD + t;
    const double* r1 = ring_mem + s1 * SLOTD + t;
    const double* r2 = ring_mem + s2 * SLOTD + t;
    double carry[8];
#pragma unroll
    for (int v = 0; v < NVR; v++) {
      const double c0 = r0[voff[v]], c1 = r1[voff[v]], a2 = r2[voff[v]];
      const double d21 = c1 - c0, d32 = a2 - c1;
      const double dmp = lim_slope2(d21, d32, a2 - c0);
      const double r = ppm_iface2(c0, d21, dm[v], dmp);
      ppm_mono(il[v], c0, r, PR[slot[v]], carry[v]);
      dm[v] = dmp; il[v] = r;
    }
    const bool pole = (D == 1) && ks && (fc == 0 || fc == L.n[1]);
    double out[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};   // C-7: pole faces carry no flux and no state is evaluated there
    if (!pole) {
      const FGeo G = load_fgeo_shared(ring_mem + s0 * SLOTD + 8 * KT);
      PL[5 + D] = PR[5 + D] = r0[7 * KT] * G.igdet;  // C-5: the normal field is single-valued at the face
      const double ct = face_flux<D, ENT>(PL, PR, G, Dv.gam, out);
      if (act) ctop = dmax(ctop, ct);
    }
    store_face(Dv, D, z, out);
    if (ENT) Dv.FK[D][z] = out[7];
    if (dup != 0) {
      store_face(Dv, D, z + dup, out);
      if (ENT) Dv.FK[D][z + dup] = out[7];
    }
#pragma unroll
    for (int v = 0; v < NVR; v++) PL[slot[v]] = carry[v];
  }
  if (want_ctop) ctop_commit<false>(Dv, D, 0, ctop);
}

// ---- sweep along x3: one lane per zone, neighbouring lanes exchange slopes and edges -------------------
// Zones (i, j, k) with i, j in [-1, n], k in [-HLO, n3 + HHI - 1] are flattened with k fastest.  A warp
// owns 32 consecutive zones of which the first HLO and the last HHI only help.
// PPM (HLO = 2, HHI = 1): every lane builds the limited slope of ITS zone once; slopes, interface
// values and right edges travel between lanes by warp shuffle.  PLM (HLO = 1, HHI = 0).
// WRAP (monolithic grids with a periodic x3, the grids the ring kernels serve): the stencil wraps inside the row and
// the face at k = n3 is stored as the periodic image of the face at k = 0, so the x3 ghost zones are never read and the
// per-stage ghost fill skips them (x3_ghosts_unused; bc.cu)
template <int RECON, bool BLK, bool WRAP, bool ENT = false>
__global__ void __launch_bounds__(128, ENT ? 4 : X3_MINB) k_flux_x3(Dev Dv, Fields s, Fields s2, int want_ctop) {
  constexpr int D = 2;
  constexpr int HLO = (RECON == HAMR_RECON_PPM) ? 2 : 1, HHI = (RECON == HAMR_RECON_PPM) ? 1 : 0;
  constexpr int OWN = 32 - HLO - HHI;
  constexpr unsigned FULL = 0xffffffffu;
  const Lay& L = Dv.L;
  const int ck = L.n[2] + (WRAP ? 0 : 1) + HLO + HHI, cj = L.n[1] + 2;
  // 32-bit index arithmetic (the launcher guarantees tot < 2^31): 64-bit division is emulated
  const int per = (L.n[0] + 2) * cj * ck;
  const int tot = BLK ? per * Dv.B.nact : per;
  const int lane = threadIdx.x & 31;
  const int warp = (int)((blockIdx.x * blockDim.x + threadIdx.x) >> 5);
  int ts = warp * OWN + lane - HLO;
  const bool valid = ts >= 0 && ts < tot;
  ts = ts < 0 ? 0 : (ts >= tot ? tot - 1 : ts);  // clamped lanes compute on a real zone and store nothing
  unsigned t = (unsigned)ts;
  int bslot = 0;
  if (BLK) { bslot = (int)(t / (unsigned)per); t -= bslot * per; }
  const BCtx C = blk_ctx<BLK>(Dv, bslot);
  const unsigned tj = t / (unsigned)ck, ti = tj / (unsigned)cj;
  const int k = (int)(t - tj * ck) - HLO;
  const int j = (int)(tj - ti * cj) - 1;
  const int i = (int)ti - 1;
  const int z = C.zoff + (int)L.idx(i, j, k);
  // offsets of zones k - 1, k, k + 1 relative to z (WRAP: their periodic images inside the row)
  int om = -1, o0 = 0, op = 1;
  if (WRAP) {
    const int n3 = L.n[2];
    auto wr = [n3](int q) { return q < 0 ? q + n3 : (q >= n3 ? q - n3 : q); };
    om = wr(k - 1) - k; o0 = wr(k) - k; op = wr(k + 1) - k;
  }
  constexpr int NVR = ENT ? 8 : 7;   // reconstructed variables; C-18: kappa goes to slot 8 of the states
  const double* var[8] = {selp<BLK>(s.P[0], s2.P[0], C.cur), selp<BLK>(s.P[1], s2.P[1], C.cur),
                          selp<BLK>(s.P[2], s2.P[2], C.cur), selp<BLK>(s.P[3], s2.P[3], C.cur),
                          selp<BLK>(s.P[4], s2.P[4], C.cur), selp<BLK>(s.Bc[0], s2.Bc[0], C.cur),
                          selp<BLK>(s.Bc[1], s2.Bc[1], C.cur), Dv.K};
  constexpr int slot[8] = {0, 1, 2, 3, 4, 5, 6, 8};
  // the face's record and normal field are requested together with the stencil: one round trip to memory, not two
  // (helper lanes read the record and field of the real zone they are clamped to)
  const FGeo G = load_fgeo(Dv.gf3A + (BLK ? C.lev * Dv.B.tlevA : 0) + (size_t)(C.q0 + i * (BLK ? Dv.B.ge2 : L.e2) + j) * NREC_F);
  const double bf3 = selp<BLK>(s.Bf[2], s2.Bf[2], C.cur)[z];
  double PL[9], PR[9];
#pragma unroll
  for (int v = 0; v < NVR; v++) {
    const double* a = var[v] + z;
    double aR;
    if (RECON == HAMR_RECON_PPM) {
      const double m1 = a[om], c0 = a[o0], p1 = a[op];
      const double d21 = c0 - m1, d32 = p1 - c0;
      const double dm0 = lim_slope2(d21, d32, p1 - m1);
      const double dmp = __shfl_down_sync(FULL, dm0, 1);         // slope of zone k+1
      const double r = ppm_iface2(c0, d32, dm0, dmp);             // a_{k+1/2}
      const double l = __shfl_up_sync(FULL, r, 1);               // a_{k-1/2}, built by lane-1 from the same expression
      ppm_mono(l, c0, r, PR[slot[v]], aR);
    } else {
      plm_edges(a[om], a[o0], a[op], PR[slot[v]], aR);
    }
    PL[slot[v]] = __shfl_up_sync(FULL, aR, 1);  // right edge of zone k-1 = left state of face k-1/2
  }
  double ctop = 0.0;
  // C-15: the x3-faces of a phi-derefined row are computed by k_deref_x3 with a strided stencil
  const bool fine_row = Dv.mrow == nullptr || __ldg(Dv.mrow + C.J0 + j + NG) == 1;
  if (valid && fine_row && lane >= HLO && lane < 32 - HHI && k >= 0 && k < L.n[2] + (WRAP ? 0 : 1)) {
    PL[7] = PR[7] = bf3 * G.igdet;
    double out[8];
    const double ct = face_flux<D, ENT>(PL, PR, G, Dv.gam, out);
    store_face(Dv, D, z, out);
    if (ENT) Dv.FK[D][z] = out[7];
    if (WRAP && k == 0) {
      store_face(Dv, D, z + L.n[2], out);
      if (ENT) Dv.FK[D][z + L.n[2]] = out[7];
    }
    if (i >= 0 && i < L.n[0] && j >= 0 && j < L.n[1]) ctop = ct;
  }
  if (want_ctop) ctop_commit<BLK>(Dv, D, C.b, ctop);
}

// ---- sweep along x3, one warp per periodic row (monolithic grids the ring kernels serve, n3 = 32 M) ---------------
// A lane owns M CONSECUTIVE zones of the row, so the parabolas of a row are built with the minimum of work: one
// limited slope, one interface value and one monotonisation per zone, three shuffles per lane and variable (the
// neighbours' edge quantities; lane 31 wraps to lane 0: the row is periodic, no lane is spent on halo zones and
// no ghost zone is read).  The left / right states of the row's n3 faces go through shared memory (14 doubles per
// face), because the Riemann problems are then solved with lanes on CONSECUTIVE faces (coalesced stores).
// A warp walks over a contiguous range of rows; each row's stencil lines are prefetched into L2 one row ahead.
// Phase 2 (the row's Riemann problems, M per lane) is a ROLLED loop: unrolled by M = 4 the kernel is 2870 instructions
// (46 KB) per row and waits for its own instructions (no_instruction 0.42 warps per issue); rolled it is 1820 and needs 156
// registers.  Measured on cfg 2 (whole step, the three sweeps side by side): rolled 1.934 ms, by two 1.942, by four 1.963.
constexpr int X3W_U = 1;
template <int M, bool ENT = false>
__global__ void __launch_bounds__(32, RING_WARPS) k_flux_x3_warp(Dev Dv, Fields s, int seg, int want_ctop) {
  constexpr int D = 2;
  constexpr unsigned FULL = 0xffffffffu;
  constexpr int QS = (M == 1) ? 32 : 32 + 16 / M;   // slot stride between a lane's zones: conflict-free both ways
  constexpr int NV = M * QS;                         // doubles per variable and side
  constexpr int NVR = ENT ? 8 : 7;                   // reconstructed variables (C-18: kappa is the eighth)
  __shared__ double lr[2 * NVR * NV];
  __shared__ double sb[32 * M];                      // the normal field of the row's faces (phase 2 is a rolled loop)
  const Lay& L = Dv.L;
  const int lane = threadIdx.x;
  const int n3 = 32 * M, cj = L.n[1] + 2;
  const int nrow = (L.n[0] + 2) * cj;
  const int r0 = blockIdx.x * seg, r1 = min(r0 + seg, nrow);
  const double* var[8] = {s.P[0], s.P[1], s.P[2], s.P[3], s.P[4], s.Bc[0], s.Bc[1], Dv.K};
  const int up = (lane + 31) & 31, dn = (lane + 1) & 31;   // the lanes owning the zones before / after this lane's
  double ctop = 0.0;
  for (int row = r0; row < r1; row++) {
    const int i = row / cj - 1, j = row - (i + 1) * cj - 1;
    const int zr = (int)L.idx(i, j, 0);
    if (row + 1 < r1 && lane < n3 / 16) {   // next row's lines (7 variables + face field) into L2
      const int i2 = (row + 1) / cj - 1, j2 = (row + 1) - (i2 + 1) * cj - 1;
      const int zn = (int)L.idx(i2, j2, 0) + 16 * lane;
#pragma unroll
      for (int v = 0; v < NVR; v++) asm volatile("prefetch.global.L2 [%0];" ::"l"(var[v] + zn));
      asm volatile("prefetch.global.L2 [%0];" ::"l"(s.Bf[2] + zn));
    }
    // the row's face record and the normal field of this lane's faces are requested with the stencil: they are
    // used in phase 2, after the parabolas
    const FGeo G = load_fgeo(Dv.gf3A + (size_t)((NG + i) * L.e2 + NG + j) * NREC_F);
    double bf3[M];
#pragma unroll
    for (int q2 = 0; q2 < M; q2++) bf3[q2] = __ldg(s.Bf[2] + zr + lane + 32 * q2);
#pragma unroll
    for (int q2 = 0; q2 < M; q2++) sb[lane + 32 * q2] = bf3[q2];
    // ---- phase 1: parabolas of the lane's M zones, states of their low faces to shared memory ----
#pragma unroll
    for (int v = 0; v < NVR; v++) {
      double a[M + 2];   // zones M l - 1 .. M l + M
      if (M >= 2) {
        const double2* a2 = reinterpret_cast<const double2*>(var[v] + zr + M * lane);
#pragma unroll
        for (int q = 0; q < M / 2; q++) { const double2 t = __ldg(a2 + q); a[1 + 2 * q] = t.x; a[2 + 2 * q] = t.y; }
      } else {
        a[1] = __ldg(var[v] + zr + lane);
      }
      a[0] = __shfl_sync(FULL, a[M], up);
      a[M + 1] = __shfl_sync(FULL, a[1], dn);
      double dm[M + 1], r[M];
#pragma unroll
      for (int q = 0; q < M; q++) dm[q] = lim_slope2(a[q + 1] - a[q], a[q + 2] - a[q + 1], a[q + 2] - a[q]);
      dm[M] = __shfl_sync(FULL, dm[0], dn);
#pragma unroll
      for (int q = 0; q < M; q++) r[q] = ppm_iface2(a[q + 1], a[q + 2] - a[q + 1], dm[q], dm[q + 1]);
      double l = __shfl_sync(FULL, r[M - 1], up), aRlast = 0.0;
#pragma unroll
      for (int q = 0; q < M; q++) {
        double aL, aR;
        ppm_mono(l, a[q + 1], r[q], aL, aR);
        lr[(NVR + v) * NV + q * QS + lane] = aL;                  // right state of the zone's low face
        if (q + 1 < M) lr[v * NV + (q + 1) * QS + lane] = aR;   // left state of the next zone's low face
        else aRlast = aR;
        l = r[q];
      }
      lr[v * NV + lane] = __shfl_sync(FULL, aRlast, up);        // left state of this lane's first face
    }
    __syncwarp();
    // ---- phase 2: Riemann problems, lanes on consecutive faces ----
    const bool act = i >= 0 && i < L.n[0] && j >= 0 && j < L.n[1];
#pragma unroll X3W_U
    for (int q2 = 0; q2 < M; q2++) {
      const int f = lane + 32 * q2;                  // face = zone index
      const int sl = (f % M) * QS + f / M;
      double PL[9], PR[9];
#pragma unroll
      for (int v = 0; v < 7; v++) { PL[v] = lr[v * NV + sl]; PR[v] = lr[(NVR + v) * NV + sl]; }
      if (ENT) { PL[8] = lr[7 * NV + sl]; PR[8] = lr[(NVR + 7) * NV + sl]; }
      const int z = zr + f;
      PL[7] = PR[7] = sb[f] * G.igdet;
      double out[8];
      const double ct = face_flux<D, ENT>(PL, PR, G, Dv.gam, out);
      if (act) ctop = dmax(ctop, ct);
      store_face(Dv, D, z, out);
      if (ENT) Dv.FK[D][z] = out[7];
      if (f == 0) {   // the face at k = n3 is the periodic image of the face at k = 0
        store_face(Dv, D, z + n3, out);
        if (ENT) Dv.FK[D][z + n3] = out[7];
      }
    }
    __syncwarp();
  }
  if (want_ctop) ctop_commit<false>(Dv, D, 0, ctop);
}

template <int M, bool ENT = false>
static void launch_x3_warp_t(hamr_grid* g, const Dev& Dv, const Fields& src, bool want_ctop) {
  const Lay& L = Dv.L;
  // occupancy cached per host thread and device (a grid is driven by one thread at a time; two grids may be driven concurrently)
  thread_local int per_sm = 0, sms = 148, cached_dev = -1;
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev != cached_dev) {
    int v = 1;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&v, k_flux_x3_warp<M, ENT>, 32, 0);
    per_sm = v < 1 ? 1 : v;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cached_dev = dev;
  }
  const int nrow = (L.n[0] + 2) * (L.n[1] + 2);
  // a whole number of waves of resident warps, at least 8 rows per warp
  const int slots = sms * per_sm;
  int waves = (nrow + 8 * slots - 1) / (8 * slots);
  if (waves < 1) waves = 1;
  int nw = waves * slots;
  if (nw > nrow) nw = nrow;
  const int seg = (nrow + nw - 1) / nw;
  k_flux_x3_warp<M, ENT><<<(nrow + seg - 1) / seg, 32, 0, g->stream>>>(Dv, src, seg, want_ctop ? 1 : 0);
}

static int ring_width(const Dev& Dv);
// M = n3 / 32 of the warp-per-row x3 sweep (0: not served)
static int x3_warp_m(const Dev& Dv) {
  if (ring_width(Dv) == 0) return 0;
  const int n3 = Dv.L.n[2];
  // n3 = 256 (M = 8) needs 32 KB of shared memory per warp (7 resident warps per SM).  With the Riemann problems unrolled it
  // lost to the shuffle kernel on cfg 3 (1.86 vs 1.66 ms); rolled (156 registers) it wins: cfg 3 step 15.37 -> 14.87 ms.
  // With the entropy row (36 KB per warp) the shuffle kernel stays
  return (n3 == 32 || n3 == 64 || n3 == 128 || (n3 == 256 && !Dv.entropy)) ? n3 / 32 : 0;
}

// ---- C-15 (ii): x3-faces of phi-derefined rows -----------------------------------------------------------
// "PPM ... modified for the increased cell spacing".  In a row with factor m the flux exists on
// group-boundary faces only (k a multiple of m); its stencil takes one value per group, zones k + t m,
// t = -3..2 (beyond the block the phi-ghost zones hold groups, C-15); the Courant limit uses m dx3.
// One thread per group-boundary face; rows with m = 1 return at once.
// ENT (C-18): kappa of the same groups is the eighth reconstructed variable, the entropy flux goes to FK
template <int RECON, bool BLK, bool ENT = false>
__global__ void __launch_bounds__(128) k_deref_x3(Dev Dv, Fields s, Fields s2, int want_ctop) {
  constexpr int D = 2;
  const Lay& L = Dv.L;
  const int ck = L.n[2] + 1, cj = L.n[1] + 2;
  const unsigned per = (unsigned)(L.n[0] + 2) * cj * ck;
  unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = t < (BLK ? per * Dv.B.nact : per);
  if (!valid) t = 0;
  int bslot = 0;
  if (BLK) { bslot = (int)(t / per); t -= bslot * per; }
  const BCtx C = blk_ctx<BLK>(Dv, bslot);
  const unsigned tj = t / (unsigned)ck, ti = tj / (unsigned)cj;
  const int k = (int)(t - tj * ck), j = (int)(tj - ti * cj) - 1, i = (int)ti - 1;
  const int m = __ldg(Dv.mrow + C.J0 + j + NG);
  double ctop = 0.0;
  if (valid && m > 1 && k % m == 0) {
    const int n3 = L.n[2];
    const int zrow = C.zoff + (int)L.idx(i, j, 0);
    const double* var[8] = {selp<BLK>(s.P[0], s2.P[0], C.cur), selp<BLK>(s.P[1], s2.P[1], C.cur),
                            selp<BLK>(s.P[2], s2.P[2], C.cur), selp<BLK>(s.P[3], s2.P[3], C.cur),
                            selp<BLK>(s.P[4], s2.P[4], C.cur), selp<BLK>(s.Bc[0], s2.Bc[0], C.cur),
                            selp<BLK>(s.Bc[1], s2.Bc[1], C.cur), Dv.K};
    constexpr int slot[8] = {0, 1, 2, 3, 4, 5, 6, 8};   // kappa goes to slot 8 of the states (slot 7: the normal field)
    int kk[6];   // beyond the block the phi-ghost zones hold whole groups: -1, -2, -3 and n3, n3 + 1, n3 + 2
#pragma unroll
    for (int q = 0; q < 6; q++) {
      const int w = k + (q - 3) * m;
      kk[q] = w < 0 ? w / m : (w >= n3 ? n3 + (w - n3) / m : w);
    }
    double PL[9], PR[9];
#pragma unroll
    for (int v = 0; v < (ENT ? 8 : 7); v++) {
      const double* a = var[v] + zrow;
      const double a0 = a[kk[0]], a1 = a[kk[1]], a2 = a[kk[2]], a3 = a[kk[3]], a4 = a[kk[4]], a5 = a[kk[5]];
      double dum;
      if (RECON == HAMR_RECON_PPM) {
        ppm_edges(a0, a1, a2, a3, a4, dum, PL[slot[v]]);   // left of the face: a_R of group k/m - 1
        ppm_edges(a1, a2, a3, a4, a5, PR[slot[v]], dum);   // right of the face: a_L of group k/m
      } else {
        plm_edges(a1, a2, a3, dum, PL[slot[v]]);
        plm_edges(a2, a3, a4, PR[slot[v]], dum);
      }
    }
    const int ge2 = BLK ? Dv.B.ge2 : L.e2;
    const FGeo G = load_fgeo(Dv.gf3A + (BLK ? C.lev * Dv.B.tlevA : 0) + (size_t)(C.q0 + i * ge2 + j) * NREC_F);
    const int z = zrow + k;
    PL[7] = PR[7] = selp<BLK>(s.Bf[2], s2.Bf[2], C.cur)[z] * G.igdet;
    const double ct = face_flux<D, ENT>(PL, PR, G, Dv.gam, Dv, z);
    if (i >= 0 && i < L.n[0] && j >= 0 && j < L.n[1]) ctop = ct / (double)m;
  }
  if (want_ctop) ctop_commit<BLK>(Dv, D, C.b, ctop);
}

void launch_deref_x3(hamr_grid* g, const Dev& Dv0, const Fields& src, const Fields& src2, bool want_ctop) {
  if (!Dv0.mrow) return;
  Dev Dv = Dv0;   // on a block grid only the listed blocks that hold derefined rows
  if (Dv0.B.nblk > 0 && Dv0.B.dlist) { Dv.B.list = Dv0.B.dlist; Dv.B.nact = Dv0.B.ndact; }
  const Lay& L = Dv.L;
  const bool ppm = Dv.recon == HAMR_RECON_PPM, blk = Dv.B.nblk > 0;
  if (blk && Dv.B.nact == 0) return;
  const long long tot = (long long)(L.n[0] + 2) * (L.n[1] + 2) * (L.n[2] + 1) * (blk ? Dv.B.nact : 1);
  const unsigned nb = (unsigned)((tot + 127) / 128);
  const int wc = want_ctop ? 1 : 0;
  Launch l_(g, K_FLUX3);
  if (Dv.entropy) {   // C-18
    if (ppm && !blk) k_deref_x3<HAMR_RECON_PPM, false, true><<<nb, 128, 0, g->stream>>>(Dv, src, src2, wc);
    else if (ppm) k_deref_x3<HAMR_RECON_PPM, true, true><<<nb, 128, 0, g->stream>>>(Dv, src, src2, wc);
    else if (!blk) k_deref_x3<HAMR_RECON_PLM_MC, false, true><<<nb, 128, 0, g->stream>>>(Dv, src, src2, wc);
    else k_deref_x3<HAMR_RECON_PLM_MC, true, true><<<nb, 128, 0, g->stream>>>(Dv, src, src2, wc);
    return;
  }
  if (ppm && !blk) k_deref_x3<HAMR_RECON_PPM, false><<<nb, 128, 0, g->stream>>>(Dv, src, src2, wc);
  else if (ppm) k_deref_x3<HAMR_RECON_PPM, true><<<nb, 128, 0, g->stream>>>(Dv, src, src2, wc);
  else if (!blk) k_deref_x3<HAMR_RECON_PLM_MC, false><<<nb, 128, 0, g->stream>>>(Dv, src, src2, wc);
  else k_deref_x3<HAMR_RECON_PLM_MC, true><<<nb, 128, 0, g->stream>>>(Dv, src, src2, wc);
}

// picks the number of faces per marching segment so that the grid fills whole waves of resident
// blocks (148 SMs x blocks per SM) with little prologue overhead
template <int D, int RECON, bool BLK, bool ENT>
static int pick_segment(const Lay& L, int nbx) {
  thread_local int cached_seg = 0, cached_dev = -1;   // per host thread: no shared mutable state between grids
  thread_local long long cached_key = -1;
  const int nf = L.n[D] + 1;
  const long long key = (long long)nf * (1LL << 32) + nbx;
  int dev = 0, sms = 148, per_sm = 2;
  cudaGetDevice(&dev);
  if (key == cached_key && dev == cached_dev) return cached_seg;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_flux_march<D, RECON, BLK, ENT>, MARCH_T, 0);
  if (per_sm < 1) per_sm = 1;
  const double slots = (double)sms * per_sm;
  double best = -1.0;
  int best_seg = nf < 16 ? nf : 16;
  for (int nseg = 1; nseg <= nf && nseg <= 64; nseg++) {
    const int seg = (nf + nseg - 1) / nseg;
    if (seg < 8 && nseg > 1) break;
    const int ns = (nf + seg - 1) / seg;
    const double blocks = (double)nbx * ns;
    const double waves = ceil(blocks / slots);
    // useful work / occupied slots-time: wave fill x (faces / (faces + one prologue zone per segment))
    const double eff = blocks / (waves * slots) * ((double)nf / ((double)ns * (seg + 1)));
    if (eff > best) { best = eff; best_seg = seg; }
  }
  cached_key = key;
  cached_dev = dev;
  cached_seg = best_seg;
  return best_seg;
}

template <int D, int RECON, bool BLK, bool ENT = false>
static void launch_march_t(hamr_grid* g, const Dev& Dv, const Fields& src, const Fields& src2, bool want_ctop) {
  const Lay& L = Dv.L;
  const int O = 1 - D;
  const long long ntr = (long long)(L.n[O] + 2) * (L.n[2] + 2) * (BLK ? Dv.B.nact : 1);
  const int nbx = (int)((ntr + MARCH_T - 1) / MARCH_T);
  const int seg = pick_segment<D, RECON, BLK, ENT>(L, nbx);
  dim3 grid(nbx, (L.n[D] + 1 + seg - 1) / seg);
  k_flux_march<D, RECON, BLK, ENT><<<grid, MARCH_T, 0, g->stream>>>(Dv, src, src2, seg, want_ctop ? 1 : 0);
}

// the ring kernel: segment length such that the grid fills whole waves of resident CTAs
template <int D, int KT, bool ENT = false>
static void launch_ring_t(hamr_grid* g, const Dev& Dv, const Fields& src, bool want_ctop) {
  const Lay& L = Dv.L;
  const int O = 1 - D;
  const size_t smem = (size_t)ring::RING * (((ENT ? 9 : 8) * KT + NREC_F) * sizeof(double)) + 2 * ring::RING * sizeof(unsigned long long);
  // the attribute and the occupancy are per function and device; cached per host thread
  thread_local int per_sm = 0, sms = 148, cached_dev = -1;
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev != cached_dev) {
    cudaFuncSetAttribute(k_flux_ring<D, KT, ENT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    int v = 1;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&v, k_flux_ring<D, KT, ENT>, KT, smem);
    per_sm = v < 1 ? 1 : v;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cached_dev = dev;
  }
  const int nf = L.n[D] + 1, nrow = (L.n[2] / KT) * (L.n[O] + 2);
  const double slots = (double)sms * per_sm;
  double best = -1.0;
  int best_seg = nf;
  for (int nseg = 1; nseg <= nf && nseg <= 64; nseg++) {
    const int seg = (nf + nseg - 1) / nseg;
    if (seg < 8 && nseg > 1) break;
    const int ns = (nf + seg - 1) / seg;
    const double blocks = (double)nrow * ns, waves = ceil(blocks / slots);
    // useful work / occupied slot-time: wave fill x (faces / (faces + one prologue zone per segment))
    const double eff = blocks / (waves * slots) * ((double)nf / ((double)ns * (seg + 1)));
    if (eff > best) { best = eff; best_seg = seg; }
  }
  dim3 grid(L.n[2] / KT, L.n[O] + 2, (nf + best_seg - 1) / best_seg);
  k_flux_ring<D, KT, ENT><<<grid, KT, smem, g->stream>>>(Dv, src, best_seg, want_ctop ? 1 : 0);
}

// the shared-memory ring serves monolithic PPM grids whose x3 extent is periodic, not derefined, and a multiple of 32
static int ring_width(const Dev& Dv) {
  const int n3 = Dv.L.n[2];
  if (Dv.B.nblk > 0 || Dv.recon != HAMR_RECON_PPM || Dv.mrow || Dv.bc_lo[2] != HAMR_BC_PERIODIC) return 0;
  if (Dv.L.n[0] + 2 > 65535 || Dv.L.n[1] + 2 > 65535) return 0;
  // one warp per CTA: 64 / 128 threads (slots released through the second mbarrier) measured 3-7 % slower
  return n3 % 32 == 0 ? 32 : 0;
}

// On those grids no kernel of a stage reads a zone beyond the x3 range: the ring kernels and the wrapping x3 sweep
// work on k in [0, n3) and store the periodic images, the centre-EMF kernel does the same (ct.cu), and the ghost
// fill leaves the x3 ghost slots alone (bc.cu).
bool x3_ghosts_unused(const Dev& Dv) { return ring_width(Dv) != 0; }

template <int D>
static void launch_march(hamr_grid* g, const Dev& Dv, const Fields& src, const Fields& src2, bool want_ctop) {
  Launch l_(g, K_FLUX1 + D);
  const bool ppm = Dv.recon == HAMR_RECON_PPM, blk = Dv.B.nblk > 0;
  if (ring_width(Dv) == 32)
    return Dv.entropy ? launch_ring_t<D, 32, true>(g, Dv, src, want_ctop) : launch_ring_t<D, 32, false>(g, Dv, src, want_ctop);
  if (Dv.entropy) {   // C-18
    if (ppm && !blk) launch_march_t<D, HAMR_RECON_PPM, false, true>(g, Dv, src, src2, want_ctop);
    else if (ppm) launch_march_t<D, HAMR_RECON_PPM, true, true>(g, Dv, src, src2, want_ctop);
    else if (!blk) launch_march_t<D, HAMR_RECON_PLM_MC, false, true>(g, Dv, src, src2, want_ctop);
    else launch_march_t<D, HAMR_RECON_PLM_MC, true, true>(g, Dv, src, src2, want_ctop);
    return;
  }
  if (ppm && !blk) launch_march_t<D, HAMR_RECON_PPM, false>(g, Dv, src, src2, want_ctop);
  else if (ppm) launch_march_t<D, HAMR_RECON_PPM, true>(g, Dv, src, src2, want_ctop);
  else if (!blk) launch_march_t<D, HAMR_RECON_PLM_MC, false>(g, Dv, src, src2, want_ctop);
  else launch_march_t<D, HAMR_RECON_PLM_MC, true>(g, Dv, src, src2, want_ctop);
}

static void launch_x3(hamr_grid* g, const Dev& Dv, const Fields& src, const Fields& src2, bool want_ctop) {
  const Lay& L = Dv.L;
  const bool ppm = Dv.recon == HAMR_RECON_PPM, blk = Dv.B.nblk > 0;
  const int own = ppm ? 29 : 31, halo = ppm ? 3 : 1;
  const bool x3wrap = x3_ghosts_unused(Dv);
  const long long tot = (long long)(L.n[0] + 2) * (L.n[1] + 2) * (L.n[2] + (x3wrap ? 0 : 1) + halo) * (blk ? Dv.B.nact : 1);
  const long long warps = (tot + own - 1) / own + 1;
  const unsigned nb = (unsigned)((warps + 3) / 4);
  const int wc = want_ctop ? 1 : 0;
  {
    Launch l_(g, K_FLUX3);
    switch (x3_warp_m(Dv) * (Dv.entropy ? -1 : 1)) {
      case 1: launch_x3_warp_t<1>(g, Dv, src, want_ctop); return;
      case 2: launch_x3_warp_t<2>(g, Dv, src, want_ctop); return;
      case 4: launch_x3_warp_t<4>(g, Dv, src, want_ctop); return;
      case 8: launch_x3_warp_t<8>(g, Dv, src, want_ctop); return;
      case -1: launch_x3_warp_t<1, true>(g, Dv, src, want_ctop); return;
      case -2: launch_x3_warp_t<2, true>(g, Dv, src, want_ctop); return;
      case -4: launch_x3_warp_t<4, true>(g, Dv, src, want_ctop); return;
      default: break;
    }
    if (Dv.entropy && blk && ppm) k_flux_x3<HAMR_RECON_PPM, true, false, true><<<nb, 128, 0, g->stream>>>(Dv, src, src2, wc);
    else if (Dv.entropy && blk) k_flux_x3<HAMR_RECON_PLM_MC, true, false, true><<<nb, 128, 0, g->stream>>>(Dv, src, src2, wc);
    else if (Dv.entropy && x3wrap) k_flux_x3<HAMR_RECON_PPM, false, true, true><<<nb, 128, 0, g->stream>>>(Dv, src, src2, wc);
    else if (Dv.entropy && ppm) k_flux_x3<HAMR_RECON_PPM, false, false, true><<<nb, 128, 0, g->stream>>>(Dv, src, src2, wc);
    else if (Dv.entropy) k_flux_x3<HAMR_RECON_PLM_MC, false, false, true><<<nb, 128, 0, g->stream>>>(Dv, src, src2, wc);
    else if (x3wrap) k_flux_x3<HAMR_RECON_PPM, false, true><<<nb, 128, 0, g->stream>>>(Dv, src, src2, wc);
    else if (ppm && !blk) k_flux_x3<HAMR_RECON_PPM, false, false><<<nb, 128, 0, g->stream>>>(Dv, src, src2, wc);
    else if (ppm) k_flux_x3<HAMR_RECON_PPM, true, false><<<nb, 128, 0, g->stream>>>(Dv, src, src2, wc);
    else if (!blk) k_flux_x3<HAMR_RECON_PLM_MC, false, false><<<nb, 128, 0, g->stream>>>(Dv, src, src2, wc);
    else k_flux_x3<HAMR_RECON_PLM_MC, true, false><<<nb, 128, 0, g->stream>>>(Dv, src, src2, wc);
  }
  if (Dv.mrow) launch_deref_x3(g, Dv, src, src2, want_ctop);   // C-15: strided x3 fluxes of the derefined rows
}

// launches issued while this object lives go to `st` instead of the grid's stream
struct OnStream {
  hamr_grid* g;
  cudaStream_t keep;
  OnStream(hamr_grid* g_, cudaStream_t st) : g(g_), keep(g_->stream) { g->stream = st; }
  ~OnStream() { g->stream = keep; }
};

// src / src2: the stage source in the buffer sets of blocks with cur == 0 / 2 (monolithic: src2 unused).
// The three sweeps read the same source and write disjoint arrays (and disjoint Courant slots), so they are issued on
// three streams between a fork and a join (inside a captured step: three parallel branches of the graph): the tail of
// one sweep's last wave is filled by the next sweep's first, and the small launches of the upper LAT levels, which
// leave most SMs idle, run side by side.  with_cemf: the caller's next call is launch_ct_on with the same source; its
// centre-EMF kernel is then issued here, beside the sweeps.  Not while the per-kernel timers are on (they bracket launches on one stream).
void launch_flux_on(hamr_grid* g, const Dev& Dv, const Fields& src, const Fields& src2, bool want_ctop, bool with_cemf) {
  if (Dv.B.nblk > 0 && Dv.B.nact == 0) return;
  const bool fork = g->aux[0] && g->aux[1] && !g->prof;
  if (fork) {
    cudaEventRecord(g->ev_fork, g->stream);
    cudaStreamWaitEvent(g->aux[0], g->ev_fork, 0);
    cudaStreamWaitEvent(g->aux[1], g->ev_fork, 0);
    { OnStream os(g, g->aux[0]); launch_march<1>(g, Dv, src, src2, want_ctop); }
    { OnStream os(g, g->aux[1]); launch_x3(g, Dv, src, src2, want_ctop); }
    launch_march<0>(g, Dv, src, src2, want_ctop);
    if (with_cemf) {
      // the centre EMFs (C-8) need the source only: a memory-bound kernel beside the issue-bound sweeps
      launch_centre_emf_on(g, Dv, src, src2);
      g->cemf_done = true;
    }
    cudaEventRecord(g->ev_join[0], g->aux[0]);
    cudaEventRecord(g->ev_join[1], g->aux[1]);
    cudaStreamWaitEvent(g->stream, g->ev_join[0], 0);
    cudaStreamWaitEvent(g->stream, g->ev_join[1], 0);
  } else {
    launch_march<0>(g, Dv, src, src2, want_ctop);
    launch_march<1>(g, Dv, src, src2, want_ctop);
    launch_x3(g, Dv, src, src2, want_ctop);
  }
  if (Dv.mrow) {  // C-15: the group structure on all face values
    launch_deref_fix_flux(g, Dv);
    launch_deref_flux_layers(g, Dv);
  }
}

void launch_flux(hamr_grid* g, const Fields& src, bool want_ctop, bool with_cemf) {
  if (g->D.entropy) launch_kappa(g, g->D, src, src);   // C-18: kappa of the (ghost-filled) source state for the entropy flux
  launch_flux_on(g, g->D, src, src, want_ctop, with_cemf);
}

}  // namespace hamr
