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

// ---- geometry tables (2-D over (i,j) incl. ghosts, SoA by component) ------------------------------
enum GeoComp {
  C00 = 0, C01, C03, C11, C13, C22, C33,  // covariant metric
  K00, K01, K11, K13, K22, K33,           // contravariant metric
  GDET, ALPHA, IALPHA, BOA,               // sqrt(-g), lapse, 1/lapse, beta^1/lapse
  IGDET,                                  // 1/sqrt(-g) (0 on the polar axis)
  NGEO
};
// centre-only extras: x1- and x2-derivatives of the 7 covariant components (for the source, C-12)
enum DgComp { D00 = 0, D01, D03, D11, D13, D22, D33, NDG };

struct Geo {
  double c00, c01, c03, c11, c13, c22, c33;
  double k00, k01, k11, k13, k22, k33;
  double gdet, alpha, ialpha, boa, igdet;
};

__device__ __forceinline__ Geo load_geo(const double* __restrict__ tab, int n2d, int q) {
  Geo G;
  G.c00 = __ldg(tab + C00 * n2d + q); G.c01 = __ldg(tab + C01 * n2d + q);
  G.c03 = __ldg(tab + C03 * n2d + q); G.c11 = __ldg(tab + C11 * n2d + q);
  G.c13 = __ldg(tab + C13 * n2d + q); G.c22 = __ldg(tab + C22 * n2d + q);
  G.c33 = __ldg(tab + C33 * n2d + q);
  G.k00 = __ldg(tab + K00 * n2d + q); G.k01 = __ldg(tab + K01 * n2d + q);
  G.k11 = __ldg(tab + K11 * n2d + q); G.k13 = __ldg(tab + K13 * n2d + q);
  G.k22 = __ldg(tab + K22 * n2d + q); G.k33 = __ldg(tab + K33 * n2d + q);
  G.gdet = __ldg(tab + GDET * n2d + q); G.alpha = __ldg(tab + ALPHA * n2d + q);
  G.ialpha = __ldg(tab + IALPHA * n2d + q); G.boa = __ldg(tab + BOA * n2d + q);
  G.igdet = __ldg(tab + IGDET * n2d + q);
  return G;
}

// The hot kernels read a geometry RECORD with all lanes of a warp on the same (i, j): with the SoA tables that is one
// cache line (one L2 round trip when it misses L1) per COMPONENT, 15-50 per face or zone.  They therefore read
// array-of-records copies: a centre record is 32 doubles (the 18 components of Geo in GeoComp order, then the 7 x1-
// and the 7 x2-derivatives of the covariant metric) = two 128-byte lines; a face record is 16 doubles = one line.
// Face records exist for the x1-faces, the x2-faces and the x3-faces (the latter at the zone centre's (x1, x2)) and
// hold the 3+1 split of the face metric that the flux kernels work with (flux.cu):
constexpr int NREC_C = 32, NREC_F = 16;
enum FaceRec {
  FREC_C11 = 0, FREC_C13, FREC_C22, FREC_C33,              // spatial metric g_ij
  FREC_ALPHA, FREC_IALPHA, FREC_BOA, FREC_BETA1,           // lapse, 1/lapse, beta^1/lapse, beta^1
  FREC_NALPHA2, FREC_K00, FREC_KDD, FREC_K0D,              // -lapse^2, g^{tt}, g^{dd}, g^{td} of the face's direction d
  FREC_GDET, FREC_IGDET                                    // sqrt(-g), 1/sqrt(-g) (0 on the polar axis); 2 pad
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
__device__ __forceinline__ Geo load_geo_rec(const double* __restrict__ rec) {
  double v[18];
  load_rec(rec, 18, v);
  Geo G;
  G.c00 = v[0]; G.c01 = v[1]; G.c03 = v[2]; G.c11 = v[3]; G.c13 = v[4]; G.c22 = v[5]; G.c33 = v[6];
  G.k00 = v[7]; G.k01 = v[8]; G.k11 = v[9]; G.k13 = v[10]; G.k22 = v[11]; G.k33 = v[12];
  G.gdet = v[13]; G.alpha = v[14]; G.ialpha = v[15]; G.boa = v[16]; G.igdet = v[17];
  return G;
}

// ---- C-2, C-3: four-velocity and magnetic four-vector -----------------------------------------------
struct St {
  double ucon[4], ucov[4], bcon[4], bcov[4], bsq;
};

// q = g_ij ut^i ut^j
__device__ __forceinline__ double vsq_tilde(const Geo& G, double v1, double v2, double v3) {
  return G.c11 * v1 * v1 + G.c22 * v2 * v2 + G.c33 * v3 * v3 + 2.0 * (G.c13 * v1 * v3);
}

__device__ __forceinline__ void lower(const Geo& G, const double v[4], double w[4]) {
  w[0] = G.c00 * v[0] + G.c01 * v[1] + G.c03 * v[3];
  w[1] = G.c01 * v[0] + G.c11 * v[1] + G.c13 * v[3];
  w[2] = G.c22 * v[2];
  w[3] = G.c03 * v[0] + G.c13 * v[1] + G.c33 * v[3];
}

// P = (rho, u, ut1, ut2, ut3, B1, B2, B3)
__device__ __forceinline__ void get_state(const double P[8], const Geo& G, St& S) {
  const double gam = sqrt(1.0 + vsq_tilde(G, P[2], P[3], P[4]));
  S.ucon[0] = gam * G.ialpha;
  S.ucon[1] = P[2] - gam * G.boa;   // beta^2 = beta^3 = 0 for both metrics
  S.ucon[2] = P[3];
  S.ucon[3] = P[4];
  lower(G, S.ucon, S.ucov);
  S.bcon[0] = P[5] * S.ucov[1] + P[6] * S.ucov[2] + P[7] * S.ucov[3];
  const double iut = 1.0 / S.ucon[0];
  S.bcon[1] = (P[5] + S.bcon[0] * S.ucon[1]) * iut;
  S.bcon[2] = (P[6] + S.bcon[0] * S.ucon[2]) * iut;
  S.bcon[3] = (P[7] + S.bcon[0] * S.ucon[3]) * iut;
  lower(G, S.bcon, S.bcov);
  S.bsq = S.bcon[0] * S.bcov[0] + S.bcon[1] * S.bcov[1] + S.bcon[2] * S.bcov[2] + S.bcon[3] * S.bcov[3];
}

// ---- C-4: conserved vector and flux -----------------------------------------------------------------
// T^mu_nu = (w + b^2) u^mu u_nu + (p + b^2/2) delta^mu_nu - b^mu b_nu for fixed mu
// hydro rows only: U = g (rho u^t, T^t_t + rho u^t, T^t_1, T^t_2, T^t_3)
__device__ __forceinline__ void prim_to_U5(const double P[8], const St& S, double gdet, double gam_ad,
                                           double U[5]) {
  const double p = (gam_ad - 1.0) * P[1];
  const double eta = P[0] + P[1] + p + S.bsq;
  const double ptot = p + 0.5 * S.bsq;
  const double eu = eta * S.ucon[0], b0 = S.bcon[0];
  const double D = P[0] * S.ucon[0];
  U[0] = gdet * D;
  U[1] = gdet * (eu * S.ucov[0] + ptot - b0 * S.bcov[0] + D);
  U[2] = gdet * (eu * S.ucov[1] - b0 * S.bcov[1]);
  U[3] = gdet * (eu * S.ucov[2] - b0 * S.bcov[2]);
  U[4] = gdet * (eu * S.ucov[3] - b0 * S.bcov[3]);
}

// ---- C-6: bounds on the fast-wave coordinate speeds along direction index dir = 1..3 ----------------
// A = g^{dd}, Bq = g^{tt}, Cq = g^{td}
__device__ __forceinline__ void wavespeeds(const double P[8], const St& S, double gam_ad, double A,
                                           double Bq, double Cq, int dir, double& vmin, double& vmax) {
  const double p = (gam_ad - 1.0) * P[1];
  const double w = P[0] + P[1] + p;
  const double cs2 = gam_ad * p / w;
  const double va2 = S.bsq / (S.bsq + w);
  double cm2 = cs2 + va2 - cs2 * va2;
  cm2 = fmin(fmax(cm2, 0.0), 1.0);
  const double ut = S.ucon[0], ud = S.ucon[dir];
  const double a2 = ut * ut - (Bq + ut * ut) * cm2;
  const double a1 = 2.0 * (ud * ut - (Cq + ud * ut) * cm2);
  const double a0 = ud * ud - (A + ud * ud) * cm2;
  const double disc = sqrt(fmax(a1 * a1 - 4.0 * a2 * a0, 0.0));
  const double i2 = 1.0 / (2.0 * a2);
  const double v1 = (a1 + disc) * i2;
  const double v2 = (a1 - disc) * i2;
  vmax = fmax(v1, v2);
  vmin = fmin(v1, v2);
}

// ---- C-5: reconstruction -----------------------------------------------------------------------------
__device__ __forceinline__ double ppm_slope(double am, double a0, double ap) {
  const double dl = a0 - am, dr = ap - a0;
  if (dl * dr <= 0.0) return 0.0;
  const double dc = 0.5 * (ap - am);
  const double lim = fmin(fabs(dc), fmin(2.0 * fabs(dl), 2.0 * fabs(dr)));
  return dc > 0.0 ? lim : -lim;
}

// parabola edges of the zone with value a2 from a0..a4 = a[j-2..j+2] (Colella & Woodward 1984)
__device__ __forceinline__ void ppm_zone(double a0, double a1, double a2, double a3, double a4,
                                         double& aL, double& aR) {
  const double dm_m = ppm_slope(a0, a1, a2);
  const double dm_0 = ppm_slope(a1, a2, a3);
  const double dm_p = ppm_slope(a2, a3, a4);
  aL = a1 + 0.5 * (a2 - a1) - (dm_0 - dm_m) / 6.0;
  aR = a2 + 0.5 * (a3 - a2) - (dm_p - dm_0) / 6.0;
  if ((aR - a2) * (a2 - aL) <= 0.0) {
    aL = aR = a2;
  } else {
    const double d = aR - aL;
    const double c = a2 - 0.5 * (aL + aR);
    if (d * c > d * d / 6.0) aL = 3.0 * a2 - 2.0 * aR;
    else if (d * c < -d * d / 6.0) aR = 3.0 * a2 - 2.0 * aL;
  }
}

// PLM with the MC limiter: minmod(2(a1-a0), (a2-a0)/2, 2(a2-a1))
__device__ __forceinline__ void plm_zone(double a0, double a1, double a2, double& aL, double& aR) {
  const double dl = 2.0 * (a1 - a0), dr = 2.0 * (a2 - a1), dc = 0.5 * (a2 - a0);
  double s = 0.0;
  if (dl * dr > 0.0) {
    s = fmin(fabs(dc), fmin(fabs(dl), fabs(dr)));
    if (dc < 0.0) s = -s;
  }
  aL = a1 - 0.5 * s;
  aR = a1 + 0.5 * s;
}

// positive doubles order like their bit patterns: max-reduce through an unsigned 64-bit atomic
__device__ __forceinline__ void atomic_max_pos(double* addr, double v) {
  atomicMax(reinterpret_cast<unsigned long long*>(addr), (unsigned long long)__double_as_longlong(v));
}

// plain compare-select min / max (no NaN special-casing, unlike fmin / fmax)
__device__ __forceinline__ double dmin(double a, double b) { return a < b ? a : b; }
__device__ __forceinline__ double dmax(double a, double b) { return a > b ? a : b; }

__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// C-13: 2-unknown (W = w gamma^2, v^2) Newton-Raphson.  U: densitised hydro rows; Bc: NEW cell-centred
// field; Pg: guess (the stage's source state).  Returns 0 ok, 1 no convergence, 2 non-finite.
__device__ __forceinline__ int con2prim(const double U[5], const double Bc[3], const Geo& G, double gam_ad,
                                        const double Pg[5], double Pout[5]) {
  const double ig = 1.0 / G.gdet;
  const double alpha = G.alpha;
  const double rhout = U[0] * ig;
  const double D = alpha * rhout;
  // Q_mu = alpha T^t_mu with rho u^t removed from the energy row (C-4)
  const double Q0 = alpha * (U[1] * ig - rhout), Q1 = alpha * (U[2] * ig), Q2 = alpha * (U[3] * ig),
               Q3 = alpha * (U[4] * ig);
  const double B1 = alpha * Bc[0], B2 = alpha * Bc[1], B3 = alpha * Bc[2];
  const double Qc0 = G.k00 * Q0 + G.k01 * Q1;
  const double Qc1 = G.k01 * Q0 + G.k11 * Q1 + G.k13 * Q3;
  const double Qc2 = G.k22 * Q2;
  const double Qc3 = G.k13 * Q1 + G.k33 * Q3;
  const double n0 = -alpha * G.k00, n1 = -alpha * G.k01;  // n^mu = -alpha g^{mu t}; n^2 = n^3 = 0
  const double Qdotn = Q0 * n0 + Q1 * n1;
  const double QQ = Q0 * Qc0 + Q1 * Qc1 + Q2 * Qc2 + Q3 * Qc3;
  const double Qtsq = QQ + Qdotn * Qdotn;
  const double QdB = Q1 * B1 + Q2 * B2 + Q3 * B3;
  const double Bsq = vsq_tilde(G, B1, B2, B3);
  const double QdB2 = QdB * QdB;
  const double cg = (gam_ad - 1.0) / gam_ad;

  const double g2 = 1.0 + vsq_tilde(G, Pg[2], Pg[3], Pg[4]);
  double W = (Pg[0] + gam_ad * Pg[1]) * g2;
  double v2 = 1.0 - 1.0 / g2;
  v2 = fmin(fmax(v2, 0.0), 1.0 - 1e-15);

  int extra = -1;
  bool conv = false;
  for (int it = 0; it < 30; it++) {
    const double omv = 1.0 - v2;
    const double sq = sqrt(omv);
    const double p = cg * (W * omv - D * sq);
    const double dpdW = cg * omv;
    const double dpdv = cg * (-W + D / (2.0 * sq));
    const double BW = Bsq + W;
    const double iW = 1.0 / W;
    const double iW2 = iW * iW, iW3 = iW2 * iW;
    const double f1 = Qtsq - v2 * BW * BW + QdB2 * (Bsq + 2.0 * W) * iW2;
    const double f2 = -Qdotn - 0.5 * Bsq * (1.0 + v2) + 0.5 * QdB2 * iW2 - W + p;
    const double j11 = -2.0 * v2 * BW - 2.0 * QdB2 * BW * iW3;
    const double j12 = -BW * BW;
    const double j21 = -QdB2 * iW3 - 1.0 + dpdW;
    const double j22 = -0.5 * Bsq + dpdv;
    const double idet = 1.0 / (j11 * j22 - j12 * j21);
    const double dW = -(j22 * f1 - j12 * f2) * idet;
    const double dv = -(-j21 * f1 + j11 * f2) * idet;
    if (!isfinite(dW) || !isfinite(dv)) return 2;
    W = fabs(W + dW);
    v2 = fmin(fmax(v2 + dv, 0.0), 1.0 - 1e-15);
    if (extra >= 0) {
      if (++extra >= 2) { conv = true; break; }
    } else if (fabs(dW) <= 1e-12 * fabs(W) && fabs(dv) <= 1e-12) {
      extra = 0;  // converged: take 2 more iterations so the result does not depend on the guess
    }
  }
  if (!conv) return 1;
  const double gamma = 1.0 / sqrt(1.0 - v2);
  const double rho = D / gamma;
  const double u = (W / (gamma * gamma) - rho) / gam_ad;
  if (!isfinite(rho) || !isfinite(u) || !isfinite(W)) return 2;
  Pout[0] = rho;
  Pout[1] = u;
  const double fac = gamma / (W + Bsq), qw = QdB / W;
  Pout[2] = fac * (Qc1 + Qdotn * n1 + qw * B1);
  Pout[3] = fac * (Qc2 + qw * B2);
  Pout[4] = fac * (Qc3 + qw * B3);
  return 0;
}

// floors and Lorentz-factor ceiling on primitives (C-13)
__device__ __forceinline__ void floors_ceiling(const Geo& G, double rfl, double ufl, double gamma_max, double Pn[5],
                                               int& nrf, int& nuf, int& ngc) {
  if (Pn[0] < rfl) { Pn[0] = rfl; nrf = 1; }
  if (Pn[1] < ufl) { Pn[1] = ufl; nuf = 1; }
  const double gamma = sqrt(1.0 + vsq_tilde(G, Pn[2], Pn[3], Pn[4]));
  if (gamma > gamma_max) {
    const double fac = sqrt((gamma_max * gamma_max - 1.0) / (gamma * gamma - 1.0));
    Pn[2] *= fac; Pn[3] *= fac; Pn[4] *= fac;
    ngc = 1;
  }
}

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
