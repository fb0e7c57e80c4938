// geom.cu — one-time metric precompute ("Kerr-Schild foliation ...
// x1 = log r, x2 = theta, x3 = phi"; "need to store metric components").
// Tables are 2-D over (x1, x2) including ghosts, because both metrics are independent of x3.
#include "hamr_host.h"

namespace hamr {

// Kerr-Schild in internal coordinates (t, ln r, theta, phi), C-1.
// dg1/dg2: x1- and x2-derivatives of the 7 non-zero covariant components (analytic).
__device__ static void metric_at(int metric, double a, double x1, double x2, Geo& G, double dg1[NDG],
                                 double dg2[NDG]) {
  for (int c = 0; c < NDG; c++) dg1[c] = dg2[c] = 0.0;
  if (metric == HAMR_METRIC_MINKOWSKI) {
    G.c00 = -1.0; G.c01 = 0.0; G.c03 = 0.0; G.c11 = 1.0; G.c13 = 0.0; G.c22 = 1.0; G.c33 = 1.0;
    G.k00 = -1.0; G.k01 = 0.0; G.k11 = 1.0; G.k13 = 0.0; G.k22 = 1.0; G.k33 = 1.0;
    G.gdet = 1.0; G.alpha = 1.0; G.ialpha = 1.0; G.boa = 0.0;
    return;
  }
  const double pi = 3.14159265358979323846;
  const double r = exp(x1);
  // polar ghosts use the mirrored theta; the metric is even about both poles, so d/dtheta of the
  // mirrored function is minus the derivative at the image point
  double th = x2;
  const bool mirrored = (x2 < 0.0) || (x2 > pi);
  if (th < 0.0) th = -th;
  if (th > pi) th = 2.0 * pi - th;
  const double s = sin(th), c = cos(th);
  const double s2 = s * s, sc2 = 2.0 * s * c;
  const double a2 = a * a;
  const double Sig = r * r + a2 * c * c;
  const double Sig_r = 2.0 * r, Sig_th = -2.0 * a2 * s * c;
  const double f = 2.0 * r / Sig;
  const double f_r = 2.0 * (a2 * c * c - r * r) / (Sig * Sig);
  const double f_th = 4.0 * r * a2 * s * c / (Sig * Sig);
  const double q = Sig + a2 * s2 * (1.0 + f);
  // covariant components in (t, r, theta, phi) and their r-, theta-derivatives
  const double g[NDG] = {-(1.0 - f), f, -f * a * s2, 1.0 + f, -a * s2 * (1.0 + f), Sig, s2 * q};
  const double gr[NDG] = {f_r, f_r, -a * s2 * f_r, f_r, -a * s2 * f_r, Sig_r, s2 * (Sig_r + a2 * s2 * f_r)};
  const double gt[NDG] = {f_th, f_th, -a * (f_th * s2 + f * sc2), f_th, -a * (sc2 * (1.0 + f) + s2 * f_th),
                          Sig_th, sc2 * q + s2 * (Sig_th + a2 * (sc2 * (1.0 + f) + s2 * f_th))};
  // x1 = ln r: each index equal to 1 carries a factor r; d/dx1 = r d/dr
  const int cnt[NDG] = {0, 1, 0, 2, 1, 0, 0};
  double gi[NDG];
  for (int m = 0; m < NDG; m++) {
    const double sf = cnt[m] == 0 ? 1.0 : (cnt[m] == 1 ? r : r * r);
    gi[m] = sf * g[m];
    dg1[m] = cnt[m] * gi[m] + sf * r * gr[m];
    dg2[m] = (mirrored ? -1.0 : 1.0) * sf * gt[m];
  }
  G.c00 = gi[0]; G.c01 = gi[1]; G.c03 = gi[2]; G.c11 = gi[3]; G.c13 = gi[4]; G.c22 = gi[5]; G.c33 = gi[6];
  G.gdet = r * Sig * fabs(s);
  if (s2 < 1e-28) {  // on the polar axis the inverse metric is singular; the record is never used
    G.k00 = G.k01 = G.k11 = G.k13 = G.k22 = G.k33 = 0.0;
    G.gdet = 0.0; G.alpha = 1.0; G.ialpha = 1.0; G.boa = 0.0;
    return;
  }
  const double Delta = r * r - 2.0 * r + a2;
  G.k00 = -(1.0 + f);
  G.k01 = f / r;
  G.k11 = (Delta / Sig) / (r * r);
  G.k13 = (a / Sig) / r;
  G.k22 = 1.0 / Sig;
  G.k33 = 1.0 / (Sig * s2);
  G.alpha = 1.0 / sqrt(-G.k00);
  G.ialpha = 1.0 / G.alpha;
  const double beta1 = -G.k01 / G.k00;
  G.boa = beta1 / G.alpha;
}

__device__ static void store_geo(double* tab, int n2d, int q, const Geo& G) {
  tab[C00 * n2d + q] = G.c00; tab[C01 * n2d + q] = G.c01; tab[C03 * n2d + q] = G.c03;
  tab[C11 * n2d + q] = G.c11; tab[C13 * n2d + q] = G.c13; tab[C22 * n2d + q] = G.c22;
  tab[C33 * n2d + q] = G.c33;
  tab[K00 * n2d + q] = G.k00; tab[K01 * n2d + q] = G.k01; tab[K11 * n2d + q] = G.k11;
  tab[K13 * n2d + q] = G.k13; tab[K22 * n2d + q] = G.k22; tab[K33 * n2d + q] = G.k33;
  tab[GDET * n2d + q] = G.gdet; tab[ALPHA * n2d + q] = G.alpha; tab[IALPHA * n2d + q] = G.ialpha;
  tab[BOA * n2d + q] = G.boa;
  tab[IGDET * n2d + q] = G.gdet > 0.0 ? 1.0 / G.gdet : 0.0;
}

// e1 x e2 table entries; entry (ti, tj) is the zone with index (ti - NG, tj - NG) counted from the
// domain's low corner in zones of spacing dx1 (the table of one x1 refinement level), n2glob zones in x2
// face record of the array-of-records tables (hamr_dev.cuh); kdd / k0d: g^{dd}, g^{td} of the face's direction
__device__ static void store_face_rec(double* rec, const Geo& G, double kdd, double k0d) {
  double v[NREC_F] = {};
  v[FREC_C11] = G.c11; v[FREC_C13] = G.c13; v[FREC_C22] = G.c22; v[FREC_C33] = G.c33;
  v[FREC_ALPHA] = G.alpha; v[FREC_IALPHA] = G.ialpha; v[FREC_BOA] = G.boa; v[FREC_BETA1] = G.boa * G.alpha;
  v[FREC_NALPHA2] = -(G.alpha * G.alpha); v[FREC_K00] = G.k00; v[FREC_KDD] = kdd; v[FREC_K0D] = k0d;
  v[FREC_GDET] = G.gdet; v[FREC_IGDET] = G.gdet > 0.0 ? 1.0 / G.gdet : 0.0;
  for (int c = 0; c < NREC_F; c++) rec[c] = v[c];
}

__global__ void k_geometry(Dev D, int e1, int e2, int n2d, double dx1, int n2glob, double* gc, double* gf1,
                           double* gf2, double* dgc, double* rho_fl, double* u_fl, double* gcA, double* gf1A,
                           double* gf2A, double* gf3A) {
  const int q = blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= e1 * e2) return;
  const int i = q / e2 - NG, j = q % e2 - NG;
  const double xc1 = D.x0[0] + ((double)i + 0.5) * dx1, xf1 = D.x0[0] + (double)i * dx1;
  const double xc2 = D.x0[1] + ((double)j + 0.5) * D.dx[1], xf2 = D.x0[1] + (double)j * D.dx[1];
  Geo G;
  double d1[NDG], d2[NDG];
  metric_at(D.metric, D.a, xc1, xc2, G, d1, d2);
  store_geo(gc, n2d, q, G);
  for (int c = 0; c < NDG; c++) {
    dgc[c * n2d + q] = d1[c];
    dgc[(NDG + c) * n2d + q] = d2[c];
  }
  {
    double* rec = gcA + (size_t)q * NREC_C;   // the same numbers, one record per (i, j)
    for (int c = 0; c < NGEO; c++) rec[c] = gc[c * n2d + q];
    for (int c = 0; c < NDG; c++) { rec[NGEO + c] = d1[c]; rec[NGEO + NDG + c] = d2[c]; }
  }
  store_face_rec(gf3A + (size_t)q * NREC_F, G, G.k33, 0.0);   // g^{t3} = 0 for both metrics
  metric_at(D.metric, D.a, xf1, xc2, G, d1, d2);
  store_geo(gf1, n2d, q, G);
  store_face_rec(gf1A + (size_t)q * NREC_F, G, G.k11, G.k01);
  metric_at(D.metric, D.a, xc1, xf2, G, d1, d2);
  if (D.metric == HAMR_METRIC_KERR_SCHILD && (j == 0 || j == n2glob)) G.gdet = 0.0;  // pole faces (C-7)
  store_geo(gf2, n2d, q, G);
  store_face_rec(gf2A + (size_t)q * NREC_F, G, G.k22, 0.0);
  if (j == -NG) {  // floors depend on x1 only (C-13): coef * r^pow, r = 1 on the Cartesian map
    const double r = (D.metric == HAMR_METRIC_KERR_SCHILD) ? exp(xc1) : 1.0;
    rho_fl[i + NG] = D.rho_fl_coef * pow(r, D.rho_fl_pow);
    u_fl[i + NG] = D.u_fl_coef * pow(r, D.u_fl_pow);
  }
}

void launch_geometry_tab(hamr_grid* g, int e1, int e2, int n2d, double dx1, int n2glob, double* gc, double* gf1,
                         double* gf2, double* dgc, double* rho_fl, double* u_fl, double* gcA, double* gf1A,
                         double* gf2A, double* gf3A) {
  Launch l_(g, K_OTHER);
  k_geometry<<<(e1 * e2 + 127) / 128, 128, 0, g->stream>>>(g->D, e1, e2, n2d, dx1, n2glob, gc, gf1, gf2, dgc,
                                                         rho_fl, u_fl, gcA, gf1A, gf2A, gf3A);
}

}  // namespace hamr
