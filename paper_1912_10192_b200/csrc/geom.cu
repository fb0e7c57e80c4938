// geom.cu — one-time metric precompute ("Kerr-Schild foliation ...
// x1 = log r, x2 = theta, x3 = phi"; "need to store metric components").
// Tables are 2-D over (x1, x2) including ghosts, because both metrics are independent of x3; one record per
// (i, j) for zone centres and for each kind of face (hamr_dev.cuh CentreRec / FaceRec).
//
// How the numbers are made (C-1).  The Kerr metric in Kerr-Schild coordinates (t, r, theta, phi) is
// built in its Kerr-Schild FORM, flat space in spheroidal coordinates plus a null dyad,
//     g_mn = g0_mn + f l_m l_n,   f = 2 r / Sigma,   l = (1, 1, 0, -a sin^2 theta),
//     g0 = diag(-1, 1, Sigma, (r^2 + a^2) sin^2 theta) with g0_{r phi} = -a sin^2 theta,
// and differentiated by the product rule; the change to x1 = ln r multiplies every r index by r.  Everything else in
// a record is DERIVED from these covariant components by the 3+1 split, numerically, on the table itself:
// shift beta^i = gamma^ij g_0j (gamma^ij the inverse of the spatial block), lapse alpha^2 = beta^i g_0i - g_00,
// sqrt(-g) = alpha sqrt(det gamma), g^tt = -1/alpha^2, g^ti = beta^i/alpha^2, g^ij = gamma^ij - beta^i beta^j/alpha^2,
// d ln sqrt(-g) = (1/2) g^kl d g_kl.  No closed form of the inverse metric or of the determinant is typed in; the
// closed forms (alpha^2 = Sigma / (Sigma + 2 r), sqrt(-g) = r Sigma sin theta, ...) are what tests/ check the tables against.
#include "hamr_host.h"

namespace hamr {

struct Metric4 {
  double g[4][4];    // covariant components in the internal coordinates
  double d1[4][4];   // their x1-derivatives
  double d2[4][4];   // their x2-derivatives
  bool axis;         // the point lies on the polar axis (the spatial metric is singular there)
};

__device__ static void metric_at(int metric, double a, double x1, double x2, Metric4& M) {
  for (int m = 0; m < 4; m++)
    for (int n = 0; n < 4; n++) M.g[m][n] = M.d1[m][n] = M.d2[m][n] = 0.0;
  M.axis = false;
  if (metric == HAMR_METRIC_MINKOWSKI) {
    M.g[0][0] = -1.0;
    M.g[1][1] = M.g[2][2] = M.g[3][3] = 1.0;
    return;
  }
  const double pi = 3.14159265358979323846;
  const double r = exp(x1);
  // rows beyond a pole carry the metric of their mirror image: theta -> -theta or 2 pi - theta.  The metric is even
  // about both poles, so the x2-derivative of the mirrored function is minus the derivative at the image point
  double th = x2, sgn2 = 1.0;
  if (th < 0.0) { th = -th; sgn2 = -1.0; }
  if (th > pi) { th = 2.0 * pi - th; sgn2 = -1.0; }
  const double sn = sin(th), cs = cos(th);
  const double sn2 = sn * sn, d_sn2 = 2.0 * sn * cs;           // sin^2 theta and its theta-derivative
  const double Sig = r * r + a * a * cs * cs;
  const double dSig[2] = {2.0 * r, -a * a * d_sn2};            // d/dr, d/dtheta
  const double f = 2.0 * r / Sig;
  const double df[2] = {(2.0 - f * dSig[0]) / Sig, -f * dSig[1] / Sig};
  const double l[4] = {1.0, 1.0, 0.0, -a * sn2};
  const double dl3[2] = {0.0, -a * d_sn2};                     // only l_phi varies
  double g0[4][4] = {}, dg0[2][4][4] = {};
  g0[0][0] = -1.0;
  g0[1][1] = 1.0;
  g0[2][2] = Sig;                    dg0[0][2][2] = dSig[0];                 dg0[1][2][2] = dSig[1];
  g0[3][3] = (r * r + a * a) * sn2;  dg0[0][3][3] = 2.0 * r * sn2;           dg0[1][3][3] = (r * r + a * a) * d_sn2;
  g0[1][3] = g0[3][1] = -a * sn2;    dg0[1][1][3] = dg0[1][3][1] = -a * d_sn2;
  const double jac[4] = {1.0, r, 1.0, 1.0};                    // d(t, r, theta, phi) / d(t, x1, x2, x3), diagonal
  for (int m = 0; m < 4; m++) {
    for (int n = 0; n < 4; n++) {
      const double sc = jac[m] * jac[n];
      const double gmn = g0[m][n] + f * l[m] * l[n];
      double dg[2];
      for (int c = 0; c < 2; c++) {
        const double dlm = (m == 3) ? dl3[c] : 0.0, dln = (n == 3) ? dl3[c] : 0.0;
        dg[c] = dg0[c][m][n] + df[c] * l[m] * l[n] + f * (dlm * l[n] + l[m] * dln);
      }
      const int nr = (m == 1) + (n == 1);                      // r indices: d(r^nr)/dx1 = nr r^nr
      M.g[m][n] = sc * gmn;
      M.d1[m][n] = nr * sc * gmn + sc * r * dg[0];
      M.d2[m][n] = sgn2 * sc * dg[1];
    }
  }
  M.axis = sn2 < 1e-28;
}

// the 3+1 split of a covariant metric with g_02 = g_12 = g_23 = 0 (both supported metrics)
struct Split {
  double c11, c13, c22, c33, i11, i13, i22, i33, alpha, beta1, gdet;
  double k[4][4];   // contravariant components
};

__device__ static Split split_3p1(const Metric4& M) {
  Split S;
  S.c11 = M.g[1][1]; S.c13 = M.g[1][3]; S.c22 = M.g[2][2]; S.c33 = M.g[3][3];
  for (int m = 0; m < 4; m++)
    for (int n = 0; n < 4; n++) S.k[m][n] = 0.0;
  if (M.axis) {   // never used: faces on the axis carry no flux (C-7) and no zone centre lies on it
    S.i11 = S.i13 = S.i22 = S.i33 = 0.0;
    S.alpha = 1.0; S.beta1 = 0.0; S.gdet = 0.0;
    return S;
  }
  const double det2 = S.c11 * S.c33 - S.c13 * S.c13;
  S.i11 = S.c33 / det2; S.i13 = -S.c13 / det2; S.i33 = S.c11 / det2; S.i22 = 1.0 / S.c22;
  const double b1 = M.g[0][1], b3 = M.g[0][3];                 // beta_i = g_0i
  S.beta1 = S.i11 * b1 + S.i13 * b3;                           // beta^3 = i13 b1 + i33 b3 vanishes for both metrics
  const double alpha2 = S.beta1 * b1 - M.g[0][0];
  S.alpha = sqrt(alpha2);
  S.gdet = S.alpha * sqrt(S.c22 * det2);
  S.k[0][0] = -1.0 / alpha2;
  S.k[0][1] = S.k[1][0] = S.beta1 / alpha2;
  S.k[1][1] = S.i11 - S.beta1 * S.beta1 / alpha2;
  S.k[1][3] = S.k[3][1] = S.i13;
  S.k[2][2] = S.i22;
  S.k[3][3] = S.i33;
  return S;
}

// d: the face's direction index 1..3 (g^{dd}, g^{td} go into the record)
__device__ static void store_face_rec(double* rec, const Split& S, int d, bool zero_gdet) {
  double v[NREC_F] = {};
  v[FREC_C11] = S.c11; v[FREC_C13] = S.c13; v[FREC_C22] = S.c22; v[FREC_C33] = S.c33;
  v[FREC_ALPHA] = S.alpha; v[FREC_IALPHA] = 1.0 / S.alpha; v[FREC_BOA] = S.beta1 / S.alpha; v[FREC_BETA1] = S.beta1;
  v[FREC_NALPHA2] = -(S.alpha * S.alpha);
  v[FREC_K00] = S.k[0][0]; v[FREC_KDD] = S.k[d][d]; v[FREC_K0D] = S.k[0][d];
  const double gd = zero_gdet ? 0.0 : S.gdet;
  v[FREC_GDET] = gd; v[FREC_IGDET] = gd > 0.0 ? 1.0 / gd : 0.0;
  for (int c = 0; c < NREC_F; c++) rec[c] = v[c];
}

// e1 x e2 table entries; entry (ti, tj) is the zone with index (ti - NG, tj - NG) counted from the
// domain's low corner in zones of spacing dx1 (the table of one x1 refinement level), n2glob zones in x2
__global__ void k_geometry(Dev D, int e1, int e2, double dx1, int n2glob, double* rho_fl, double* u_fl, double* gcA,
                           double* gf1A, double* gf2A, double* gf3A) {
  const int q = blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= e1 * e2) return;
  const int i = q / e2 - NG, j = q % e2 - NG;
  // an x1 slab (NEXT-4) counts from the GLOBAL low corner, so that its tables equal the global grid's bit for bit
  const int ig = i + D.ioff;
  const double xc1 = D.x0[0] + ((double)ig + 0.5) * dx1, xf1 = D.x0[0] + (double)ig * dx1;
  const double xc2 = D.x0[1] + ((double)j + 0.5) * D.dx[1], xf2 = D.x0[1] + (double)j * D.dx[1];
  Metric4 M;
  metric_at(D.metric, D.a, xc1, xc2, M);
  Split S = split_3p1(M);
  {
    double v[NREC_C] = {};
    v[CREC_C11] = S.c11; v[CREC_C13] = S.c13; v[CREC_C22] = S.c22; v[CREC_C33] = S.c33;
    v[CREC_I11] = S.i11; v[CREC_I13] = S.i13; v[CREC_I22] = S.i22; v[CREC_I33] = S.i33;
    v[CREC_ALPHA] = S.alpha; v[CREC_IALPHA] = 1.0 / S.alpha; v[CREC_BOA] = S.beta1 / S.alpha; v[CREC_BETA1] = S.beta1;
    v[CREC_GDET] = S.gdet; v[CREC_IGDET] = S.gdet > 0.0 ? 1.0 / S.gdet : 0.0;
    double dl1 = 0.0, dl2 = 0.0;   // d ln sqrt(-g) = (1/2) g^kl d g_kl
    for (int m = 0; m < 4; m++)
      for (int n = 0; n < 4; n++) { dl1 += S.k[m][n] * M.d1[m][n]; dl2 += S.k[m][n] * M.d2[m][n]; }
    v[CREC_DLG1] = 0.5 * dl1; v[CREC_DLG2] = 0.5 * dl2;
    const int hm[NH] = {0, 0, 0, 1, 1, 2, 3}, hn[NH] = {0, 1, 3, 1, 3, 2, 3};   // HComp order
    for (int c = 0; c < NH; c++) {
      const double w = hm[c] == hn[c] ? 0.5 : 1.0;   // (1/2) d g_kl, both orders of an off-diagonal pair
      v[CREC_H1 + c] = w * M.d1[hm[c]][hn[c]];
      v[CREC_H2 + c] = w * M.d2[hm[c]][hn[c]];
    }
    double* rec = gcA + (size_t)q * NREC_C;
    for (int c = 0; c < NREC_C; c++) rec[c] = v[c];
  }
  store_face_rec(gf3A + (size_t)q * NREC_F, S, 3, false);
  metric_at(D.metric, D.a, xf1, xc2, M);
  S = split_3p1(M);
  store_face_rec(gf1A + (size_t)q * NREC_F, S, 1, false);
  metric_at(D.metric, D.a, xc1, xf2, M);
  S = split_3p1(M);
  // pole faces (C-7): sqrt(-g) = 0
  store_face_rec(gf2A + (size_t)q * NREC_F, S, 2, D.metric == HAMR_METRIC_KERR_SCHILD && (j == 0 || j == n2glob));
  if (j == -NG) {  // floors depend on x1 only (C-13): coef * r^pow, r = 1 on the Cartesian map
    const double r = (D.metric == HAMR_METRIC_KERR_SCHILD) ? exp(xc1) : 1.0;
    rho_fl[i + NG] = D.rho_fl_coef * pow(r, D.rho_fl_pow);
    u_fl[i + NG] = D.u_fl_coef * pow(r, D.u_fl_pow);
  }
}

void launch_geometry_tab(hamr_grid* g, int e1, int e2, double dx1, int n2glob, double* rho_fl, double* u_fl,
                         double* gcA, double* gf1A, double* gf2A, double* gf3A) {
  Launch l_(g, K_OTHER);
  k_geometry<<<(e1 * e2 + 127) / 128, 128, 0, g->stream>>>(g->D, e1, e2, dx1, n2glob, rho_fl, u_fl, gcA, gf1A, gf2A,
                                                          gf3A);
}

}  // namespace hamr
