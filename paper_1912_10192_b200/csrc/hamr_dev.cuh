// hamr_dev.cuh — data layout and per-zone device physics shared by the CUDA kernels of libhamr.
// Product code (sm_100a, fp64).  Shares nothing with oracle/.
//
// Formulas: the standard forms behind the paper's citations as read in DESIGN.md §3 (C-n):
//   C-2 four-velocity, C-3 magnetic four-vector, C-4 stress-energy / conserved vector / fluxes
//   (Eq. 1), C-5 PPM / PLM-MC, C-6 signal speeds, C-7 HLLE
//   (PAPER.md:41), C-13 2-D Newton-Raphson inversion and floors.
//
// Both supported metrics (Minkowski; Kerr-Schild in x1 = ln r, x2 = theta, x3 = phi)
// share one sparsity pattern: g_{02} = g_{12} = g_{23} = 0 and g^{02} = g^{03} = g^{12} = g^{23} = 0.
// Only the 7 + 6 non-zero components are stored and multiplied.
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

namespace hamr {

constexpr int NG = 3;     // ghost layers: a PPM face needs zones j-3 .. j+2 (C-5)
constexpr int NNBR = 36;  // entries per block of the neighbour table (27 by offset + 9 across a transmissive pole)
constexpr int LEAD = 13;  // leading pad so that active zone k = 0 sits on a 128-byte boundary

// ---- array layout ------------------------------------------------------------------------------
// One padded fp64 array per variable, x3 fastest.  Zone (i,j,k), -NG <= idx <= n+NG, lives at
// off0 + i*S1 + j*S2 + k.  Face/edge arrays use the same index for the face on the LOW side.
struct Lay {
  int n[3];       // active zones
  int e1, e2;     // padded extents n + 2NG + 1 along x1, x2
  int p3;         // pitch along x3: n3 + 2NG + 1 rounded up to a multiple of 16 doubles
  int S1, S2;     // strides (S3 = 1)
  long long off0; // index of zone (0,0,0)
  long long len;  // doubles per array
  int n2d;        // e1*e2 entries per 2-D geometry component
  __host__ __device__ __forceinline__ long long idx(int i, int j, int k) const {
    return off0 + (long long)i * S1 + (long long)j * S2 + k;
  }
  __host__ __device__ __forceinline__ int idx2(int i, int j) const { return (i + NG) * e2 + (j + NG); }
  __host__ __device__ __forceinline__ int str(int d) const { return d == 0 ? S1 : (d == 1 ? S2 : 1); }
};

// ---- geometry tables: one record per (i, j) of a 2-D table incl. ghosts ------------------------------
// The kernels read a geometry RECORD with all lanes of a warp on the same (i, j): a record is one (faces) or two
// (centres) 128-byte lines, so a warp's geometry costs one or two L1 / L2 round trips.  Records hold the 3+1 split
// of the metric, which is what the per-zone physics below works with: spatial metric g_ij (the only non-zero
// off-diagonal spatial component of either metric is g_13), lapse alpha, shift beta^1 (beta^2 = beta^3 = 0),
// sqrt(-g).  Face records exist for x1-faces, x2-faces and x3-faces (the latter at the centre's (x1, x2)).
constexpr int NREC_C = 32, NREC_F = 16;
enum FaceRec {
  FREC_C11 = 0, FREC_C13, FREC_C22, FREC_C33,              // spatial metric g_ij
  FREC_ALPHA, FREC_IALPHA, FREC_BOA, FREC_BETA1,           // lapse, 1/lapse, beta^1/lapse, beta^1
  FREC_NALPHA2, FREC_K00, FREC_KDD, FREC_K0D,              // -lapse^2, g^{tt}, g^{dd}, g^{td} of the face's direction d
  FREC_GDET, FREC_IGDET                                    // sqrt(-g), 1/sqrt(-g) (0 on the polar axis); 2 pad
};
// centre record: the first 16 doubles are CGeo below; then the metric derivatives the source term contracts
// (C-12): H1[7], H2[7] = the x1- and x2-derivatives of (g_00, g_01, g_03, g_11, g_13, g_22, g_33) with the
// diagonal ones halved, so that (1/2) v^k v^l d_nu g_kl = sum_c H[c] (v v)_c over the 7 distinct products
enum CentreRec {
  CREC_C11 = 0, CREC_C13, CREC_C22, CREC_C33,              // spatial metric g_ij
  CREC_I11, CREC_I13, CREC_I22, CREC_I33,                  // its inverse gamma^ij
  CREC_ALPHA, CREC_IALPHA, CREC_BOA, CREC_BETA1,           // lapse, 1/lapse, beta^1/lapse, beta^1
  CREC_GDET, CREC_IGDET, CREC_DLG1, CREC_DLG2,             // sqrt(-g), its reciprocal, d_1 and d_2 of ln sqrt(-g)
  CREC_H1 = 16, CREC_H2 = 23, CREC_END = 30
};
enum HComp { H00 = 0, H01, H03, H11, H13, H22, H33, NH };

struct CGeo {
  double c11, c13, c22, c33;
  double i11, i13, i22, i33;
  double alpha, ialpha, boa, beta1;
  double gdet, igdet, dlg1, dlg2;
};

__device__ __forceinline__ void load_rec(const double* __restrict__ rec, int n, double* v) {
  const double2* r2 = reinterpret_cast<const double2*>(rec);
#pragma unroll
  for (int q = 0; q < n / 2; q++) {
    const double2 t = __ldg(r2 + q);
    v[2 * q] = t.x;
    v[2 * q + 1] = t.y;
  }
}
__device__ __forceinline__ CGeo load_cgeo(const double* __restrict__ rec) {
  double v[16];
  load_rec(rec, 16, v);
  CGeo G;
  G.c11 = v[CREC_C11]; G.c13 = v[CREC_C13]; G.c22 = v[CREC_C22]; G.c33 = v[CREC_C33];
  G.i11 = v[CREC_I11]; G.i13 = v[CREC_I13]; G.i22 = v[CREC_I22]; G.i33 = v[CREC_I33];
  G.alpha = v[CREC_ALPHA]; G.ialpha = v[CREC_IALPHA]; G.boa = v[CREC_BOA]; G.beta1 = v[CREC_BETA1];
  G.gdet = v[CREC_GDET]; G.igdet = v[CREC_IGDET]; G.dlg1 = v[CREC_DLG1]; G.dlg2 = v[CREC_DLG2];
  return G;
}

// ---- reciprocal, reciprocal square root, square root for finite, normal, non-zero arguments ----------------
// The hardware seed (MUFU.RCP64H / MUFU.RSQ64H, ~20 bits) refined by fused multiply-adds, without the range
// checks and slow-path calls of the library routines.  Results are within 2 ulp; nothing here decides a branch.
__device__ __forceinline__ double rcp_nr(double a) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
  double e = fma(-a, y, 1.0);
  y = fma(y, e, y);          // relative error e^2 ~ 2^-40
  e = fma(-a, y, 1.0);
  return fma(y, e, y);
}
__device__ __forceinline__ double rsqrt_pos(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-x, y * y, 1.0);
  return fma(fma(e, 0.375, 0.5), y * e, y);   // y (1 + e/2 + 3 e^2/8): relative error ~ e^3 ~ 2^-60
}
__device__ __forceinline__ double sqrt_pos(double x) {
  const double y = rsqrt_pos(x), s = x * y;
  return fma(fma(-s, s, x), 0.5 * y, s);      // one Heron correction of s = x y
}

// plain compare-select min / max (no NaN special-casing, unlike fmin / fmax)
__device__ __forceinline__ double dmin(double a, double b) { return a < b ? a : b; }
__device__ __forceinline__ double dmax(double a, double b) { return a > b ? a : b; }

// ---- C-2, C-3: four-velocity and magnetic four-vector in the 3+1 split --------------------------------
// With u^mu = ut^mu + gamma n^mu and n_i = 0: u_i = g_ij ut^j, gamma^2 = 1 + ut^i u_i, u^t = gamma / alpha,
// u^i = ut^i - gamma beta^i / alpha, u_t = -alpha gamma + beta^i u_i.  With b^t = B^i u_i,
// b^i = (B^i + b^t u^i) / u^t: b_i = g_ij (b^j + beta^j b^t), b_t = -alpha^2 b^t + beta^i b_i.
struct St {
  double ut, u1, u2, u3;        // u^mu
  double ul0, ul1, ul2, ul3;    // u_mu
  double b0, b1, b2, b3;        // b^mu
  double bl0, bl1, bl2, bl3;    // b_mu
  double bsq, gam, iut;         // b^2, Lorentz factor, 1/u^t
};

// P = (rho, u, ut1, ut2, ut3, B1, B2, B3); nalpha2 = -alpha^2
__device__ __forceinline__ void state_3p1(const double P[8], double c11, double c13, double c22, double c33,
                                          double alpha, double ialpha, double boa, double beta1, double nalpha2,
                                          St& S) {
  S.ul1 = c11 * P[2] + c13 * P[4];
  S.ul2 = c22 * P[3];
  S.ul3 = c13 * P[2] + c33 * P[4];
  const double q1 = 1.0 + (P[2] * S.ul1 + P[3] * S.ul2 + P[4] * S.ul3);
  const double rg = rsqrt_pos(q1);   // q1 >= 1; gamma = q1 rg and 1/u^t = alpha rg share one special-function call
  S.gam = q1 * rg;
  S.iut = alpha * rg;
  S.ut = S.gam * ialpha;
  S.u1 = P[2] - S.gam * boa;
  S.u2 = P[3];
  S.u3 = P[4];
  S.ul0 = beta1 * S.ul1 - alpha * S.gam;
  S.b0 = P[5] * S.ul1 + P[6] * S.ul2 + P[7] * S.ul3;
  S.b1 = (P[5] + S.b0 * S.u1) * S.iut;
  S.b2 = (P[6] + S.b0 * S.u2) * S.iut;
  S.b3 = (P[7] + S.b0 * S.u3) * S.iut;
  const double bt1 = S.b1 + S.b0 * beta1;
  S.bl1 = c11 * bt1 + c13 * S.b3;
  S.bl2 = c22 * S.b2;
  S.bl3 = c13 * bt1 + c33 * S.b3;
  S.bl0 = nalpha2 * S.b0 + beta1 * S.bl1;
  S.bsq = S.b0 * S.bl0 + S.b1 * S.bl1 + S.b2 * S.bl2 + S.b3 * S.bl3;
}
__device__ __forceinline__ void get_state(const double P[8], const CGeo& G, St& S) {
  state_3p1(P, G.c11, G.c13, G.c22, G.c33, G.alpha, G.ialpha, G.boa, G.beta1, -(G.alpha * G.alpha), S);
}

// ---- C-4: the hydro rows of the conserved vector -----------------------------------------------------------
// U = g (rho u^t, T^t_t + rho u^t, T^t_1, T^t_2, T^t_3), T^t_nu = eta u^t u_nu + ptot delta^t_nu - b^t b_nu
__device__ __forceinline__ void prim_to_U5(const double P[8], const St& S, double gdet, double gam_ad,
                                           double U[5]) {
  const double p = (gam_ad - 1.0) * P[1];
  const double eta = P[0] + gam_ad * P[1] + S.bsq;
  const double ptot = p + 0.5 * S.bsq;
  const double eu = eta * S.ut;
  const double D = P[0] * S.ut;
  U[0] = gdet * D;
  U[1] = gdet * (eu * S.ul0 + ptot - S.b0 * S.bl0 + D);
  U[2] = gdet * (eu * S.ul1 - S.b0 * S.bl1);
  U[3] = gdet * (eu * S.ul2 - S.b0 * S.bl2);
  U[4] = gdet * (eu * S.ul3 - S.b0 * S.bl3);
}

// ---- C-12: geometric source ----------------------------------------------------------------------------
// S_nu = g T^kappa_lambda Gamma^lambda_{nu kappa} = (g/2) T^{kappa lambda} d_nu g_{kappa lambda}; both metrics are
// stationary and independent of x3, so S_t = S_3 = 0 identically.  With T^{kl} = eta u^k u^l + ptot g^{kl} - b^k b^l
// and g^{kl} d_nu g_kl = 2 d_nu ln sqrt(-g):  S_nu = g [ sum_c H_nu[c] (eta (u u)_c - (b b)_c) + ptot d_nu ln sqrt(-g) ]
// over the 7 distinct products (00, 01, 03, 11, 13, 22, 33); rec: the zone's centre record
__device__ __forceinline__ void source_12(const double P[8], const St& S, const CGeo& G, double gam_ad,
                                          const double* __restrict__ rec, double& S1, double& S2) {
  const double eta = P[0] + gam_ad * P[1] + S.bsq;
  const double ptot = (gam_ad - 1.0) * P[1] + 0.5 * S.bsq;
  double w[NH];
  w[H00] = eta * S.ut * S.ut - S.b0 * S.b0;
  w[H01] = eta * S.ut * S.u1 - S.b0 * S.b1;
  w[H03] = eta * S.ut * S.u3 - S.b0 * S.b3;
  w[H11] = eta * S.u1 * S.u1 - S.b1 * S.b1;
  w[H13] = eta * S.u1 * S.u3 - S.b1 * S.b3;
  w[H22] = eta * S.u2 * S.u2 - S.b2 * S.b2;
  w[H33] = eta * S.u3 * S.u3 - S.b3 * S.b3;
  double h[2 * NH];
  load_rec(rec + CREC_H1, 2 * NH, h);
  double a1 = ptot * G.dlg1, a2 = ptot * G.dlg2;
#pragma unroll
  for (int c = 0; c < NH; c++) { a1 += h[c] * w[c]; a2 += h[NH + c] * w[c]; }
  S1 = G.gdet * a1;
  S2 = G.gdet * a2;
}

// ---- C-13: conserved -> primitive, 2-unknown (W = w gamma^2, v^2) Newton-Raphson (Noble et al. 2006) -------
// In the 3+1 split the scheme's inputs are what the normal observer measures: D = alpha rho u^t = rho gamma,
// Q_i = alpha T^t_i, the energy -Q.n = -(T^t_t - beta^i T^t_i) (rest mass removed from the energy row, C-4),
// curlyB^i = alpha B^i, and all contractions use the spatial metric and its inverse.
// U: densitised hydro rows; Bc: NEW cell-centred field; Pg: guess.  Returns 0 ok, 1 no convergence / non-finite.
__device__ __forceinline__ int con2prim(const double U[5], const double Bc[3], const CGeo& G, double gam_ad,
                                        const double Pg[5], double Pout[5]) {
  const double D = G.alpha * (U[0] * G.igdet);
  const double m1 = U[2] * G.igdet, m2 = U[3] * G.igdet, m3 = U[4] * G.igdet;   // T^t_i
  const double Qdotn = (U[1] - U[0]) * G.igdet - G.beta1 * m1;                  // Q.n = T^t_t - beta^1 T^t_1
  const double Q1 = G.alpha * m1, Q2 = G.alpha * m2, Q3 = G.alpha * m3;
  const double Qu1 = G.i11 * Q1 + G.i13 * Q3, Qu2 = G.i22 * Q2, Qu3 = G.i13 * Q1 + G.i33 * Q3;   // Q~^i
  const double Qtsq = Q1 * Qu1 + Q2 * Qu2 + Q3 * Qu3;
  const double B1 = G.alpha * Bc[0], B2 = G.alpha * Bc[1], B3 = G.alpha * Bc[2];
  const double Bsq = B1 * (G.c11 * B1 + G.c13 * B3) + B2 * (G.c22 * B2) + B3 * (G.c13 * B1 + G.c33 * B3);
  const double QdB = Q1 * B1 + Q2 * B2 + Q3 * B3;
  const double QdB2 = QdB * QdB;
  const double cg = (gam_ad - 1.0) / gam_ad;
  // guess from Pg: W = (rho + gamma_ad u) gamma^2, v^2 = 1 - 1/gamma^2
  const double g2 = 1.0 + (Pg[2] * (G.c11 * Pg[2] + G.c13 * Pg[4]) + Pg[3] * (G.c22 * Pg[3]) +
                           Pg[4] * (G.c13 * Pg[2] + G.c33 * Pg[4]));
  double W = (Pg[0] + gam_ad * Pg[1]) * g2;
  double v2 = dmin(dmax(1.0 - rcp_nr(g2), 0.0), 1.0 - 1e-15);
  int extra = -1;
  bool conv = false;
  for (int it = 0; it < 30; it++) {
    const double omv = 1.0 - v2;                   // in [1e-15, 1]
    const double rs = rsqrt_pos(omv), sq = omv * rs;
    const double iW = rcp_nr(W);
    const double t = QdB2 * iW * iW;               // (Q.B)^2 / W^2
    const double BW = Bsq + W;
    const double f1 = Qtsq - v2 * BW * BW + t * (BW + W);
    const double f2 = (cg * (W * omv - D * sq) - W) - Qdotn - 0.5 * (Bsq * (1.0 + v2) - t);
    const double j11 = -2.0 * BW * (v2 + t * iW);
    const double j12 = -BW * BW;
    const double j21 = cg * omv - 1.0 - t * iW;
    const double j22 = cg * (0.5 * D * rs - W) - 0.5 * Bsq;
    const double idet = rcp_nr(j11 * j22 - j12 * j21);
    const double dW = (j12 * f2 - j22 * f1) * idet;
    const double dv = (j21 * f1 - j11 * f2) * idet;
    W = fabs(W + dW);
    v2 = dmin(dmax(v2 + dv, 0.0), 1.0 - 1e-15);
    if (extra >= 0) {
      if (++extra >= 2) { conv = true; break; }
    } else if (fabs(dW) <= 1e-12 * W && fabs(dv) <= 1e-12) {
      extra = 0;  // converged: take 2 more iterations so the result does not depend on the guess
    }
  }
  // a non-finite iterate never passes the convergence test (comparisons with NaN are false)
  if (!conv) return 1;
  const double rs = rsqrt_pos(1.0 - v2);           // gamma
  const double rho = D * rcp_nr(rs);
  const double iW = rcp_nr(W);
  const double u = (W * (1.0 - v2) - rho) * rcp_nr(gam_ad);
  if (!(fabs(rho) <= 1.79e308) || !(fabs(u) <= 1.79e308) || !(W <= 1.79e308)) return 1;
  Pout[0] = rho;
  Pout[1] = u;
  const double fac = rs * rcp_nr(W + Bsq), qw = QdB * iW;
  Pout[2] = fac * (Qu1 + qw * B1);
  Pout[3] = fac * (Qu2 + qw * B2);
  Pout[4] = fac * (Qu3 + qw * B3);
  return 0;
}

// floors and Lorentz-factor ceiling on primitives (C-13)
__device__ __forceinline__ void ceiling_only(const CGeo& G, double gamma_max, double Pn[5], int& ngc) {
  const double q = Pn[2] * (G.c11 * Pn[2] + G.c13 * Pn[4]) + Pn[3] * (G.c22 * Pn[3]) + Pn[4] * (G.c13 * Pn[2] + G.c33 * Pn[4]);
  if (q > gamma_max * gamma_max - 1.0) {   // gamma^2 = 1 + q > gamma_max^2
    const double fac = sqrt((gamma_max * gamma_max - 1.0) / q);
    Pn[2] *= fac; Pn[3] *= fac; Pn[4] *= fac;
    ngc = 1;
  }
}
__device__ __forceinline__ void floors_ceiling(const CGeo& G, double rfl, double ufl, double gamma_max, double Pn[5],
                                               int& nrf, int& nuf, int& ngc) {
  if (Pn[0] < rfl) { Pn[0] = rfl; nrf = 1; }
  if (Pn[1] < ufl) { Pn[1] = ufl; nuf = 1; }
  ceiling_only(G, gamma_max, Pn, ngc);
}

// kappa = (gamma_ad - 1) u rho^-gamma_ad through exp / log (each good to an ulp; |gamma_ad ln rho| < 100 keeps the
// result within 1e-14 of the correctly rounded power at a third of the cost of the library's pow)
__device__ __forceinline__ double kappa_of(double rho, double u, double gam_ad) {
  return (gam_ad - 1.0) * u * exp(-gam_ad * log(rho));
}

// ---- C-18: the entropy row and the inversion that uses it ------------------------
// kappa = p / rho^gamma_ad is carried by the mass: the row is gdet rho u^t kappa with flux gdet rho u^d kappa and no
// source.  Where the energy inversion fails (or returns rho <= 0 or u < 0) the zone is inverted from the density,
// momentum and ENTROPY rows instead.  The normal observer sees D = gamma rho and D kappa, so kappa = US / U[0] is
// known and one unknown is left, q = gamma^2 - 1:
//   W(q) = w gamma^2 = D gamma + A gamma^(2 - gamma_ad),   A = gamma_ad / (gamma_ad - 1) kappa D^gamma_ad,
//   f(q) = q / (1 + q) (Bsq + W)^2 - (Q.B)^2 (Bsq + 2 W) / W^2 - Qt^2 = 0        (momentum equation of Noble et al. 2006)
// f grows monotonically from f(0) <= 0 (gamma_ad < 2): Newton steps kept inside a bracket that is first grown by
// factors of 4.  The energy row U[1] is not read.  Returns 0 ok, 1 no root found / input without one.
static __device__ __noinline__ int con2prim_entropy(const double* __restrict__ U, double US, const double* __restrict__ Bc,
                                             const CGeo* __restrict__ Gp, double gam_ad,
                                             const double* __restrict__ Pg, double* __restrict__ Pout) {
  const CGeo& G = *Gp;
  const double D = G.alpha * (U[0] * G.igdet);
  const double kap = US / U[0];
  if (!(D > 0.0) || !(kap >= 0.0) || !(D <= 1.79e308) || !(kap <= 1.79e308)) return 1;
  const double Q1 = G.alpha * (U[2] * G.igdet), Q2 = G.alpha * (U[3] * G.igdet), Q3 = G.alpha * (U[4] * G.igdet);
  const double Qu1 = G.i11 * Q1 + G.i13 * Q3, Qu2 = G.i22 * Q2, Qu3 = G.i13 * Q1 + G.i33 * Q3;
  const double Qtsq = Q1 * Qu1 + Q2 * Qu2 + Q3 * Qu3;
  const double B1 = G.alpha * Bc[0], B2 = G.alpha * Bc[1], B3 = G.alpha * Bc[2];
  const double Bsq = B1 * (G.c11 * B1 + G.c13 * B3) + B2 * (G.c22 * B2) + B3 * (G.c13 * B1 + G.c33 * B3);
  const double QdB = Q1 * B1 + Q2 * B2 + Q3 * B3, QdB2 = QdB * QdB;
  const double A = gam_ad / (gam_ad - 1.0) * kap * pow(D, gam_ad);
  if (!(Qtsq <= 1.79e308) || !(Bsq <= 1.79e308) || !(A <= 1.79e308)) return 1;
  double W = 0.0, df = 0.0;
  auto feval = [&](double q) {
    const double q1 = 1.0 + q, g = sqrt(q1);
    const double gp = pow(q1, -0.5 * gam_ad);              // gamma^(-gamma_ad)
    W = D * g + A * gp * q1;
    const double dW = 0.5 * (D / g + A * (2.0 - gam_ad) * gp);
    const double v2 = q / q1, BW = Bsq + W, iW = 1.0 / W, t = QdB2 * iW * iW;
    df = BW * BW / (q1 * q1) + 2.0 * BW * dW * (v2 + t * iW);
    return v2 * BW * BW - t * (BW + W) - Qtsq;
  };
  double lo = 0.0, hi = 1.0;
  for (int nb = 0; feval(hi) < 0.0; nb++) {
    if (nb >= 60) return 1;
    lo = hi;
    hi *= 4.0;
  }
  double q = Pg[2] * (G.c11 * Pg[2] + G.c13 * Pg[4]) + Pg[3] * (G.c22 * Pg[3]) + Pg[4] * (G.c13 * Pg[2] + G.c33 * Pg[4]);
  if (!(q > lo && q < hi)) q = 0.5 * (lo + hi);
  bool conv = false;
  for (int it = 0; it < 100 && !conv; it++) {
    const double f = feval(q);
    if (!(fabs(f) <= 1.79e308) || !(fabs(df) <= 1.79e308)) return 1;
    if (f < 0.0) lo = q; else hi = q;
    double qn = q - f / df;
    if (!(qn > lo && qn < hi)) qn = 0.5 * (lo + hi);
    conv = fabs(qn - q) <= 1e-14 * (1.0 + qn);
    q = qn;
  }
  if (!conv) return 1;
  feval(q);
  const double gamma = sqrt(1.0 + q);
  const double rho = D / gamma;
  const double u = kap * pow(rho, gam_ad) / (gam_ad - 1.0);
  if (!(rho <= 1.79e308) || !(u <= 1.79e308) || !(W <= 1.79e308)) return 1;
  Pout[0] = rho;
  Pout[1] = u;
  const double fac = gamma / (W + Bsq), qw = QdB / W;
  Pout[2] = fac * (Qu1 + qw * B1);
  Pout[3] = fac * (Qu2 + qw * B2);
  Pout[4] = fac * (Qu3 + qw * B3);
  return 0;
}

// ---- C-21 ("... or Aitken acceleration scheme (Hamlin & Newman 2013; Newman & Hamlin
// 2014)"): the second primary inversion, tried where the Newton-Raphson one does not converge ----------------------------
// Fixed-point iteration on the gas pressure p.  With the normal observer's e = -Q.n, M^2 = Qt^2, T = Q.B and
// eps = W + Bsq, energy and momentum equations combine into a cubic for eps at given p,
//   eps^3 - a eps^2 + d = 0,  a = e + p + Bsq/2,  d = (M^2 Bsq - T^2)/2 >= 0,
// with largest root eps = (a/3)(1 + 2 cos((2/3) asin sqrt(27 d/(4 a^3)))); then W = eps - Bsq,
// v^2 = (M^2 W^2 + T^2 (Bsq + 2W))/(W eps)^2, rho = D sqrt(1 - v^2), p' = (gamma_ad - 1)/gamma_ad (W (1 - v^2) - rho).
// Every third value is Aitken's extrapolation p2 - (p2 - p1)^2 / ((p2 - p1) - (p1 - p0)).  The start is the guess's
// pressure only.  Returns 0 ok, 1 no convergence / no real root / non-finite.
static __device__ __noinline__ int con2prim_aitken(const double* __restrict__ U, const double* __restrict__ Bc,
                                                   const CGeo* __restrict__ Gp, double gam_ad,
                                                   const double* __restrict__ Pg, double* __restrict__ Pout) {
  const CGeo& G = *Gp;
  const double D = G.alpha * (U[0] * G.igdet);
  const double m1 = U[2] * G.igdet, m2 = U[3] * G.igdet, m3 = U[4] * G.igdet;
  const double e = -((U[1] - U[0]) * G.igdet - G.beta1 * m1);
  const double Q1 = G.alpha * m1, Q2 = G.alpha * m2, Q3 = G.alpha * m3;
  const double Qu1 = G.i11 * Q1 + G.i13 * Q3, Qu2 = G.i22 * Q2, Qu3 = G.i13 * Q1 + G.i33 * Q3;
  const double M2 = Q1 * Qu1 + Q2 * Qu2 + Q3 * Qu3;
  const double B1 = G.alpha * Bc[0], B2 = G.alpha * Bc[1], B3 = G.alpha * Bc[2];
  const double Bsq = B1 * (G.c11 * B1 + G.c13 * B3) + B2 * (G.c22 * B2) + B3 * (G.c13 * B1 + G.c33 * B3);
  const double T = Q1 * B1 + Q2 * B2 + Q3 * B3;
  const double d = fmax(0.0, 0.5 * (M2 * Bsq - T * T));
  const double cg = (gam_ad - 1.0) / gam_ad;
  if (!(fabs(e) <= 1.79e308) || !(M2 <= 1.79e308) || !(Bsq <= 1.79e308) || !(D > 0.0)) return 1;
  double W = 0.0, v2 = 0.0, a = 0.0;
  bool bad = false, clamped = false;
  auto step = [&](double p) {
    a = e + p + 0.5 * Bsq;
    if (!(a > 0.0)) { bad = true; return p; }
    const double s2 = 27.0 * d / (4.0 * a * a * a);
    if (!(s2 <= 1.0)) { bad = true; return p; }
    const double eps = (a / 3.0) * (1.0 + 2.0 * cos((2.0 / 3.0) * asin(sqrt(s2))));
    W = eps - Bsq;
    if (!(W > 0.0)) { bad = true; return p; }
    v2 = (M2 * W * W + T * T * (Bsq + 2.0 * W)) / ((W * eps) * (W * eps));
    clamped = !(v2 <= 1.0 - 1e-15);   // more momentum than this energy can carry: refused at the end
    v2 = dmin(dmax(v2, 0.0), 1.0 - 1e-15);
    return cg * (W * (1.0 - v2) - D * sqrt(1.0 - v2));
  };
  double p0 = (gam_ad - 1.0) * Pg[1];
  bool conv = false;
  for (int it = 0; it < 60 && !conv; it++) {
    const double p1 = step(p0);
    const double p2 = step(p1);
    if (bad || !(fabs(p2) <= 1.79e308)) return 1;
    conv = fabs(p2 - p1) <= 1e-13 * fabs(p2) + 1e-16 * a;
    const double den = (p2 - p1) - (p1 - p0);
    const double pa = p2 - (p2 - p1) * (p2 - p1) / den;
    p0 = (conv || den == 0.0 || !(fabs(pa) <= 1.79e308)) ? p2 : pa;
  }
  if (!conv) return 1;
  step(p0);
  if (bad || clamped) return 1;
  const double gamma = 1.0 / sqrt(1.0 - v2);
  const double rho = D / gamma;
  const double u = (W / (gamma * gamma) - rho) / gam_ad;
  if (!(fabs(rho) <= 1.79e308) || !(fabs(u) <= 1.79e308) || !(W <= 1.79e308)) return 1;
  Pout[0] = rho;
  Pout[1] = u;
  const double fac = gamma / (W + Bsq), qw = T / W;
  Pout[2] = fac * (Qu1 + qw * B1);
  Pout[3] = fac * (Qu2 + qw * B2);
  Pout[4] = fac * (Qu3 + qw * B3);
  return 0;
}

// ---- C-19 (Ressler et al. 2017): floors applied in the drift frame ---------------
// The matter added to reach the floors carries no momentum along the field and does not change the velocity across
// it: with v = ut / gamma = v_perp + v_par Bhat in the normal observer's frame, v_perp is kept and v_par follows
// from the conserved field-aligned momentum  m = w gamma^2 v_par  (w = rho + gamma_ad u):
//   v_par' = 2 m s / (w' + sqrt(w'^2 + 4 m^2 s)),  s = 1 - v_perp^2.     Called only for a zone below a floor.
// (inline: on a torus whose atmosphere sits at the floors this runs for almost half of the zone updates; reciprocals
// and roots from the hardware seed as in the rest of the per-zone physics)
__device__ __forceinline__ void floors_drift(const CGeo& G, const double Bc[3], double gam_ad, double rho_new, double u_new,
                                             double Pn[5]) {
  const double B1 = G.alpha * Bc[0], B2 = G.alpha * Bc[1], B3 = G.alpha * Bc[2];
  const double Bl1 = G.c11 * B1 + G.c13 * B3, Bl2 = G.c22 * B2, Bl3 = G.c13 * B1 + G.c33 * B3;
  const double Bsq = B1 * Bl1 + B2 * Bl2 + B3 * Bl3;
  if (!(Bsq > 1e-300)) { Pn[0] = rho_new; Pn[1] = u_new; return; }   // no field: the fluid frame
  const double q1 = 1.0 + (Pn[2] * (G.c11 * Pn[2] + G.c13 * Pn[4]) + Pn[3] * (G.c22 * Pn[3]) + Pn[4] * (G.c13 * Pn[2] + G.c33 * Pn[4]));
  const double ig = rsqrt_pos(q1);                                   // 1 / gamma
  const double v1 = Pn[2] * ig, v2 = Pn[3] * ig, v3 = Pn[4] * ig;
  const double iB = rsqrt_pos(Bsq);
  const double vpar = (v1 * Bl1 + v2 * Bl2 + v3 * Bl3) * iB;
  const double h1 = B1 * iB, h2 = B2 * iB, h3 = B3 * iB;             // unit vector along the field
  const double p1 = v1 - vpar * h1, p2 = v2 - vpar * h2, p3 = v3 - vpar * h3;
  const double vperp2 = p1 * (G.c11 * p1 + G.c13 * p3) + p2 * (G.c22 * p2) + p3 * (G.c13 * p1 + G.c33 * p3);
  const double m = (Pn[0] + gam_ad * Pn[1]) * q1 * vpar;
  const double wn = rho_new + gam_ad * u_new, s = 1.0 - vperp2;
  const double vpn = 2.0 * m * s * rcp_nr(wn + sqrt_pos(wn * wn + 4.0 * m * m * s));
  const double gn = rsqrt_pos(s - vpn * vpn);
  Pn[0] = rho_new;
  Pn[1] = u_new;
  Pn[2] = gn * (p1 + vpn * h1);
  Pn[3] = gn * (p2 + vpn * h2);
  Pn[4] = gn * (p3 + vpn * h3);
}

// positive doubles order like their bit patterns: max-reduce through an unsigned 64-bit atomic
__device__ __forceinline__ void atomic_max_pos(double* addr, double v) {
  atomicMax(reinterpret_cast<unsigned long long*>(addr), (unsigned long long)__double_as_longlong(v));
}

__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// ---- bulk asynchronous copies global -> shared (TMA) with mbarrier completion --------------------------------
namespace tma {
__device__ __forceinline__ unsigned su32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* b, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(su32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* b) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(su32(b)) : "memory");
}
__device__ __forceinline__ void mbar_expect(unsigned long long* b, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(su32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* b) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(su32(dst)),
               "l"(src), "r"(bytes), "r"(su32(b))
               : "memory");
}
// asks for [src, src + bytes) to be brought into L2 (no destination, no completion: a hint)
__device__ __forceinline__ void bulk_prefetch_l2(const void* src, unsigned bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}
// one lane of a converged warp
__device__ __forceinline__ bool elect_one() {
  unsigned p;
  asm volatile("{\n.reg .pred P;\nelect.sync _|P, 0xffffffff;\nselp.u32 %0, 1, 0, P;\n}" : "=r"(p));
  return p != 0;
}
__device__ __forceinline__ void mbar_wait(unsigned long long* b, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "HAMR_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra HAMR_DONE;\n"
      "bra HAMR_WAIT;\n"
      "HAMR_DONE:\n"
      "}" ::"r"(su32(b)),
      "r"(parity)
      : "memory");
}
}  // namespace tma

// ---- C-15: phi-ghost slots of derefined rows are in GROUP units -------------------------------------------
// x3 index inside the periodic neighbour that ghost slot k of an array whose row (or x2-face) has grouping mg
// holds: ghost zone -g is group -g (the neighbour's zone n3 - g mg), ghost zone n3 - 1 + g is group g - 1 beyond the
// edge (its zone (g - 1) mg); x3-faces likewise hold group-boundary faces.  k must lie outside the block.
__device__ __forceinline__ int deref_ghost_k(int k, int n3, int mg) { return k < 0 ? n3 + k * mg : (k - n3) * mg; }
// An x2-face array follows the grouping M of its FACE (the coarser of its two rows).  A zone row with factor m whose
// ghost slot k holds one of ITS groups finds the covering face value in this slot of the face array.
__device__ __forceinline__ int deref_face2_slot(int k, int n3, int m, int M) {
  if (M == m) return k;
  if (k < 0) return -((-k * m + M - 1) / M);
  if (k >= n3) return n3 + ((k - n3) * m) / M;
  return k;
}

}  // namespace hamr
