// ORACLE (test infrastructure) — geometry, C-1 of DESIGN.md §3.
// PAPER.md:41 (§2): "spherical polar coordinates r, theta, phi in a Kerr-Schild foliation. The grid
// is uniform in internal coordinates x0=t, x1=log r, x2=theta, x3=phi".
#include "orc.hpp"
#include <cstring>

namespace orc {

static double mirror_theta(double th) {
  // C-1: polar ghosts use the mirrored theta (|theta| or 2pi - theta); KS depends on sin^2, cos^2
  const double pi = 3.14159265358979323846;
  if (th < 0.0) th = -th;
  if (th > pi) th = 2.0 * pi - th;
  return th;
}

// Kerr-Schild covariant metric in (t, r, theta, phi) and its r- and theta-derivatives.
static void ks_cov(double a, double r, double th, double g[4][4], double dgr[4][4],
                   double dgth[4][4]) {
  std::memset(g, 0, 16 * sizeof(double));
  std::memset(dgr, 0, 16 * sizeof(double));
  std::memset(dgth, 0, 16 * sizeof(double));
  const double s = std::sin(th), c = std::cos(th);
  const double s2 = s * s, sc2 = 2.0 * s * c;  // d(s2)/dth = 2 s c
  const double Sig = r * r + a * a * c * c;
  const double Sig_r = 2.0 * r, Sig_th = -2.0 * a * a * s * c;
  const double f = 2.0 * r / Sig;
  const double f_r = 2.0 * (a * a * c * c - r * r) / (Sig * Sig);
  const double f_th = 4.0 * r * a * a * s * c / (Sig * Sig);

  g[0][0] = -(1.0 - f);            dgr[0][0] = f_r;                 dgth[0][0] = f_th;
  g[0][1] = f;                     dgr[0][1] = f_r;                 dgth[0][1] = f_th;
  g[0][3] = -f * a * s2;           dgr[0][3] = -a * s2 * f_r;       dgth[0][3] = -a * (f_th * s2 + f * sc2);
  g[1][1] = 1.0 + f;               dgr[1][1] = f_r;                 dgth[1][1] = f_th;
  g[1][3] = -a * s2 * (1.0 + f);   dgr[1][3] = -a * s2 * f_r;       dgth[1][3] = -a * (sc2 * (1.0 + f) + s2 * f_th);
  g[2][2] = Sig;                   dgr[2][2] = Sig_r;               dgth[2][2] = Sig_th;
  const double q = Sig + a * a * s2 * (1.0 + f);
  g[3][3] = s2 * q;
  dgr[3][3] = s2 * (Sig_r + a * a * s2 * f_r);
  dgth[3][3] = sc2 * q + s2 * (Sig_th + a * a * (sc2 * (1.0 + f) + s2 * f_th));
  for (int m = 0; m < 4; m++)
    for (int n = 0; n < m; n++) {
      g[m][n] = g[n][m];
      dgr[m][n] = dgr[n][m];
      dgth[m][n] = dgth[n][m];
    }
}

void gcov_and_derivs(int metric, double a, double x1, double x2, double g[4][4], double dg1[4][4],
                     double dg2[4][4]) {
  if (metric == 0) {
    std::memset(g, 0, 16 * sizeof(double));
    std::memset(dg1, 0, 16 * sizeof(double));
    std::memset(dg2, 0, 16 * sizeof(double));
    g[0][0] = -1.0;
    g[1][1] = g[2][2] = g[3][3] = 1.0;
    return;
  }
  const double r = std::exp(x1);
  // d/dtheta at a mirrored point: the metric is even in theta about both poles, so the derivative
  // of the mirrored function is -(derivative at the mirror image).  Ghost-row connections are
  // never used (sources are evaluated at active zones only); the sign is kept right anyway.
  const double pi = 3.14159265358979323846;
  const bool mirrored = (x2 < 0.0) || (x2 > pi);
  const double th = mirror_theta(x2);
  double gk[4][4], dr[4][4], dth[4][4];
  ks_cov(a, r, th, gk, dr, dth);
  // x1 = ln r:  g'_{mu nu} = s_mu s_nu g_{mu nu},  s = (1, r, 1, 1)
  // d/dx1 = r d/dr;  r d/dr (r^n g) = n r^n g + r^n r dg/dr with n = #indices equal to 1
  for (int m = 0; m < 4; m++)
    for (int n = 0; n < 4; n++) {
      const int cnt = (m == 1) + (n == 1);
      const double sf = (cnt == 0) ? 1.0 : (cnt == 1 ? r : r * r);
      g[m][n] = sf * gk[m][n];
      dg1[m][n] = cnt * g[m][n] + sf * r * dr[m][n];
      dg2[m][n] = (mirrored ? -1.0 : 1.0) * sf * dth[m][n];
    }
}

void geom_at(int metric, double a, double x1, double x2, Geom& G) {
  std::memset(&G, 0, sizeof(G));
  if (metric == 0) {
    G.gcov[0][0] = G.gcon[0][0] = -1.0;
    for (int i = 1; i < 4; i++) G.gcov[i][i] = G.gcon[i][i] = 1.0;
    G.gdet = 1.0;
    G.alpha = 1.0;
    return;
  }
  const double r = std::exp(x1);
  const double th = mirror_theta(x2);
  const double s = std::sin(th), c = std::cos(th);
  const double s2 = s * s;
  const double Sig = r * r + a * a * c * c;
  G.gdet = r * Sig * std::fabs(s);  // C-1: sqrt(-g) = r Sigma |sin theta|
  double d1[4][4], d2[4][4];
  gcov_and_derivs(metric, a, x1, x2, G.gcov, d1, d2);
  if (s2 < 1e-28) {  // on the polar axis: inverse metric singular; record never used (C-7)
    G.gdet = 0.0;
    G.alpha = 1.0;
    return;
  }
  // inverse KS metric (C-1), Delta = r^2 - 2r + a^2, then g'^{mu nu} = g^{mu nu}/(s_mu s_nu)
  const double f = 2.0 * r / Sig;
  const double Delta = r * r - 2.0 * r + a * a;
  double gi[4][4];
  std::memset(gi, 0, sizeof(gi));
  gi[0][0] = -(1.0 + f);
  gi[0][1] = gi[1][0] = f;
  gi[1][1] = Delta / Sig;
  gi[1][3] = gi[3][1] = a / Sig;
  gi[2][2] = 1.0 / Sig;
  gi[3][3] = 1.0 / (Sig * s2);
  for (int m = 0; m < 4; m++)
    for (int n = 0; n < 4; n++) {
      const int cnt = (m == 1) + (n == 1);
      const double sf = (cnt == 0) ? 1.0 : (cnt == 1 ? r : r * r);
      G.gcon[m][n] = gi[m][n] / sf;
    }
  G.alpha = 1.0 / std::sqrt(-G.gcon[0][0]);
  for (int i = 0; i < 3; i++) G.beta[i] = -G.gcon[0][i + 1] / G.gcon[0][0];
}

void conn_at(int metric, double a, double x1, double x2, double conn[4][4][4]) {
  std::memset(conn, 0, 64 * sizeof(double));
  if (metric == 0) return;
  Geom G;
  geom_at(metric, a, x1, x2, G);
  if (G.gdet == 0.0) return;
  double g[4][4], dg[4][4][4];  // dg[k][m][n] = d_k g_{mn}
  std::memset(dg, 0, sizeof(dg));
  gcov_and_derivs(metric, a, x1, x2, g, dg[1], dg[2]);
  // Gamma^l_{mn} = 1/2 g^{ls} (d_m g_{sn} + d_n g_{sm} - d_s g_{mn})
  for (int l = 0; l < 4; l++)
    for (int m = 0; m < 4; m++)
      for (int n = 0; n < 4; n++) {
        double acc = 0.0;
        for (int s = 0; s < 4; s++)
          acc += G.gcon[l][s] * (dg[m][s][n] + dg[n][s][m] - dg[s][m][n]);
        conn[l][m][n] = 0.5 * acc;
      }
}

}  // namespace orc
