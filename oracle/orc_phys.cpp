// ORACLE (test infrastructure) — per-zone physics: C-2..C-7, C-12 (source), C-13 of DESIGN.md §3.
// PAPER.md:45-47 (Eq. 1: dU/dt = -dF^i/dx^i + S; U conserved, F fluxes, S the warping source);
// PAPER.md:41 (HLLE, PPM); PAPER.md:49 (Newton-Raphson inversion, Noble et al. 2006).
#include "orc.hpp"
#include <algorithm>

namespace orc {

// C-2 four-velocity from primitives, C-3 magnetic four-vector
void get_state(const double P[8], const Geom& G, State& S) {
  double q = 0.0;
  for (int i = 1; i < 4; i++)
    for (int j = 1; j < 4; j++) q += G.gcov[i][j] * P[1 + i] * P[1 + j];
  S.gamma = std::sqrt(1.0 + q);
  S.ucon[0] = S.gamma / G.alpha;
  for (int i = 1; i < 4; i++) S.ucon[i] = P[1 + i] - S.gamma * G.beta[i - 1] / G.alpha;
  for (int m = 0; m < 4; m++) {
    double acc = 0.0;
    for (int n = 0; n < 4; n++) acc += G.gcov[m][n] * S.ucon[n];
    S.ucov[m] = acc;
  }
  S.bcon[0] = P[5] * S.ucov[1] + P[6] * S.ucov[2] + P[7] * S.ucov[3];
  for (int i = 1; i < 4; i++) S.bcon[i] = (P[4 + i] + S.bcon[0] * S.ucon[i]) / S.ucon[0];
  for (int m = 0; m < 4; m++) {
    double acc = 0.0;
    for (int n = 0; n < 4; n++) acc += G.gcov[m][n] * S.bcon[n];
    S.bcov[m] = acc;
  }
  S.bsq = 0.0;
  for (int m = 0; m < 4; m++) S.bsq += S.bcon[m] * S.bcov[m];
}

// C-4: T^mu_nu = (w + b^2) u^mu u_nu + (p + b^2/2) delta^mu_nu - b^mu b_nu for fixed mu
static void mhd_row(const double P[8], const State& S, double gam, int mu, double T[4]) {
  const double p = (gam - 1.0) * P[1];
  const double w = P[0] + P[1] + p;
  const double eta = w + S.bsq;
  const double ptot = p + 0.5 * S.bsq;
  for (int nu = 0; nu < 4; nu++)
    T[nu] = eta * S.ucon[mu] * S.ucov[nu] + (mu == nu ? ptot : 0.0) - S.bcon[mu] * S.bcov[nu];
}

// C-4: U = g (rho u^t, T^t_t + rho u^t, T^t_1, T^t_2, T^t_3, B^1, B^2, B^3)
void prim_to_U(const double P[8], const State& S, const Geom& G, double gam, double U[8]) {
  double T[4];
  mhd_row(P, S, gam, 0, T);
  const double D = P[0] * S.ucon[0];
  U[0] = G.gdet * D;
  U[1] = G.gdet * (T[0] + D);
  U[2] = G.gdet * T[1];
  U[3] = G.gdet * T[2];
  U[4] = G.gdet * T[3];
  for (int i = 0; i < 3; i++) U[5 + i] = G.gdet * P[5 + i];
}

// C-4: F^d = g (rho u^d, T^d_t + rho u^d, T^d_i, b^i u^d - b^d u^i)
void prim_to_F(const double P[8], const State& S, const Geom& G, double gam, int dir, double F[8]) {
  double T[4];
  mhd_row(P, S, gam, dir, T);
  const double m = P[0] * S.ucon[dir];
  F[0] = G.gdet * m;
  F[1] = G.gdet * (T[0] + m);
  F[2] = G.gdet * T[1];
  F[3] = G.gdet * T[2];
  F[4] = G.gdet * T[3];
  for (int i = 1; i < 4; i++)
    F[4 + i] = G.gdet * (S.bcon[i] * S.ucon[dir] - S.bcon[dir] * S.ucon[i]);
}

// C-6: bounds on the fast-wave coordinate speeds along `dir`
void wavespeeds(const double P[8], const State& S, const Geom& G, double gam, int dir,
                double& vmin, double& vmax) {
  const double p = (gam - 1.0) * P[1];
  const double w = P[0] + P[1] + p;
  const double cs2 = gam * p / w;
  const double va2 = S.bsq / (S.bsq + w);
  double cm2 = cs2 + va2 - cs2 * va2;
  cm2 = std::min(std::max(cm2, 0.0), 1.0);
  const double A = G.gcon[dir][dir], Bq = G.gcon[0][0], C = G.gcon[0][dir];
  const double ut = S.ucon[0], ud = S.ucon[dir];
  const double a2 = ut * ut - (Bq + ut * ut) * cm2;
  const double a1 = 2.0 * (ud * ut - (C + ud * ut) * cm2);
  const double a0 = ud * ud - (A + ud * ud) * cm2;
  const double disc = std::sqrt(std::max(a1 * a1 - 4.0 * a2 * a0, 0.0));
  const double v1 = (a1 + disc) / (2.0 * a2);
  const double v2 = (a1 - disc) / (2.0 * a2);
  vmax = std::max(v1, v2);
  vmin = std::min(v1, v2);
}

// C-7 HLL(E) flux for all 8 rows (the row of the face-normal field is identically 0).
// DESIGN.md §3 C-7a: a mass flux smaller than 1e-12 of the magnitude of its own HLL terms is
// rounding noise and is flushed to exactly 0, so that the upwind selector of C-9 sees a tie.
void hll(const double UL[8], const double UR[8], const double FL[8], const double FR[8],
         double cmin, double cmax, double F[8]) {
  const double sum = cmax + cmin;
  if (sum < 1e-300) {
    for (int c = 0; c < 8; c++) F[c] = 0.5 * (FL[c] + FR[c]);
  } else {
    for (int c = 0; c < 8; c++)
      F[c] = (cmax * FL[c] + cmin * FR[c] - cmax * cmin * (UR[c] - UL[c])) / sum;
    const double mag = (cmax * std::fabs(FL[0]) + cmin * std::fabs(FR[0]) +
                        cmax * cmin * (std::fabs(UR[0]) + std::fabs(UL[0]))) / sum;
    if (std::fabs(F[0]) <= 1e-12 * mag) F[0] = 0.0;
  }
}

// C-12: S_nu = g T^kappa_lambda Gamma^lambda_{nu kappa}, nu = 0..3 ; S(rho) = 0.
// Rows follow U: (0, S_t, S_1, S_2, S_3).
void source(const double P[8], const State& S, const Geom& G, const double conn[4][4][4],
            double gam, double Ssrc[5]) {
  double T[4][4];
  for (int k = 0; k < 4; k++) mhd_row(P, S, gam, k, T[k]);
  Ssrc[0] = 0.0;
  for (int nu = 0; nu < 4; nu++) {
    double acc = 0.0;
    for (int k = 0; k < 4; k++)
      for (int l = 0; l < 4; l++) acc += T[k][l] * conn[l][nu][k];
    Ssrc[1 + nu] = G.gdet * acc;
  }
}

// C-13 conserved -> primitive: 2-unknown (W, v^2) Newton-Raphson of Noble et al. 2006
// (PAPER.md:49).  U: densitised hydro rows; Bc: cell-centred B^i of the NEW field.
// Failure codes: 1 no convergence, 2 non-finite.  A converged root with rho <= 0 or u < 0 is NOT a
// failure: the floors that follow repair it (DESIGN.md §3 S-8).
int con2prim(const double U[5], const double Bc[3], const Geom& G, double gam,
             const double Pguess[5], double Pout[5], int* iters) {
  const double ig = 1.0 / G.gdet;
  const double alpha = G.alpha;
  // undensitise; remove rho u^t from the energy row (C-4)
  const double rhout = U[0] * ig;
  double Tt[4] = {U[1] * ig - rhout, U[2] * ig, U[3] * ig, U[4] * ig};
  const double D = alpha * rhout;
  double Qcov[4], Qcon[4], Bs[4] = {0.0, alpha * Bc[0], alpha * Bc[1], alpha * Bc[2]};
  for (int m = 0; m < 4; m++) Qcov[m] = alpha * Tt[m];
  for (int m = 0; m < 4; m++) {
    double acc = 0.0;
    for (int n = 0; n < 4; n++) acc += G.gcon[m][n] * Qcov[n];
    Qcon[m] = acc;
  }
  double ncon[4];
  for (int m = 0; m < 4; m++) ncon[m] = -alpha * G.gcon[m][0];
  double Qdotn = 0.0, QQ = 0.0;
  for (int m = 0; m < 4; m++) {
    Qdotn += Qcov[m] * ncon[m];
    QQ += Qcov[m] * Qcon[m];
  }
  const double Qtsq = QQ + Qdotn * Qdotn;
  double QdB = 0.0, Bsq = 0.0;
  for (int i = 1; i < 4; i++) {
    QdB += Qcov[i] * Bs[i];
    for (int j = 1; j < 4; j++) Bsq += G.gcov[i][j] * Bs[i] * Bs[j];
  }
  const double QdB2 = QdB * QdB;
  const double cg = (gam - 1.0) / gam;

  // guess from P_src: W0 = (rho + gamma_ad u) gamma^2, v2_0 = 1 - 1/gamma^2
  double q = 0.0;
  for (int i = 1; i < 4; i++)
    for (int j = 1; j < 4; j++) q += G.gcov[i][j] * Pguess[1 + i] * Pguess[1 + j];
  const double g2 = 1.0 + q;
  double W = (Pguess[0] + gam * Pguess[1]) * g2;
  double v2 = 1.0 - 1.0 / g2;
  v2 = std::min(std::max(v2, 0.0), 1.0 - 1e-15);

  int extra = -1, it = 0;
  bool conv = false;
  for (it = 0; it < 30; it++) {
    const double omv = 1.0 - v2;
    const double sq = std::sqrt(omv);
    const double p = cg * (W * omv - D * sq);
    const double dpdW = cg * omv;
    const double dpdv = cg * (-W + D / (2.0 * sq));
    const double BW = Bsq + W;
    const double W2 = W * W, W3 = W2 * W;
    const double f1 = Qtsq - v2 * BW * BW + QdB2 * (Bsq + 2.0 * W) / W2;
    const double f2 = -Qdotn - 0.5 * Bsq * (1.0 + v2) + QdB2 / (2.0 * W2) - W + p;
    const double j11 = -2.0 * v2 * BW - 2.0 * QdB2 * BW / W3;
    const double j12 = -BW * BW;
    const double j21 = -QdB2 / W3 - 1.0 + dpdW;
    const double j22 = -0.5 * Bsq + dpdv;
    const double det = j11 * j22 - j12 * j21;
    const double dW = -(j22 * f1 - j12 * f2) / det;
    const double dv = -(-j21 * f1 + j11 * f2) / det;
    if (!std::isfinite(dW) || !std::isfinite(dv)) {
      if (iters) *iters = it;
      return 2;
    }
    W = std::fabs(W + dW);
    v2 = std::min(std::max(v2 + dv, 0.0), 1.0 - 1e-15);
    if (extra >= 0) {
      if (++extra >= 2) { conv = true; it++; break; }
    } else if (std::fabs(dW) <= 1e-12 * std::fabs(W) && std::fabs(dv) <= 1e-12) {
      extra = 0;  // converged: take 2 more iterations (C-13)
    }
  }
  if (iters) *iters = it;
  if (!conv) return 1;
  const double gamma = 1.0 / std::sqrt(1.0 - v2);
  const double rho = D / gamma;
  const double u = (W / (gamma * gamma) - rho) / gam;
  if (!std::isfinite(rho) || !std::isfinite(u) || !std::isfinite(W)) return 2;
  Pout[0] = rho;
  Pout[1] = u;
  for (int i = 1; i < 4; i++) {
    const double Qt = Qcon[i] + Qdotn * ncon[i];
    Pout[1 + i] = gamma / (W + Bsq) * (Qt + QdB * Bs[i] / W);
  }
  return 0;
}

// ---- C-18: entropy advection and the backup inversion ("H-AMR also advects the entropy (Noble et al.
// 2009), which is then used in place of the energy equation to recover the primitive variables") -----------------
// For an ideal gas p = (gamma_ad - 1) u the quantity kappa = p / rho^gamma_ad is a function of the specific entropy
// only, so along smooth adiabatic flow  d(kappa)/d(tau) = 0, which with mass conservation is the conservation law
//   d_t (gdet rho kappa u^t) + d_i (gdet rho kappa u^i) = 0            (no source term).
double entropy_kappa(double rho, double u, double gam) { return (gam - 1.0) * u / std::pow(rho, gam); }

void entropy_UF(const double P[8], const State& S, const Geom& G, double gam, int dir, double& US, double& FS) {
  const double k = entropy_kappa(P[0], P[1], gam);
  US = G.gdet * P[0] * k * S.ucon[0];
  FS = G.gdet * P[0] * k * S.ucon[dir];
}

// The inversion.  In the normal observer's frame (n_mu = (-alpha, 0, 0, 0)) the conserved rows give
//   D = gamma rho,  Q_mu = alpha T^t_mu,  curly-B^i = alpha B^i,  and  alpha (rho kappa u^t) = D kappa,
// so kappa = US / U[0] is known at once.  With  q = ut^2 = gamma^2 - 1  as the one unknown:
//   rho = D / gamma,  p = kappa rho^gamma_ad,  w = rho + gamma_ad/(gamma_ad - 1) p,
//   W(q) = w gamma^2 = D gamma + c kappa D^gamma_ad gamma^(2 - gamma_ad),   c = gamma_ad / (gamma_ad - 1),
// and the squared momentum equation of Noble et al. 2006 (their Eq. 27, the f1 of con2prim above) closes it:
//   f(q) = v^2 (Bsq + W)^2 - (Q.B)^2 (Bsq + 2 W) / W^2 - Qt^2 = 0,   v^2 = q / (1 + q).
// W grows with q for gamma_ad < 2, each term of f grows with W and with v^2, f(0) <= 0 and f -> infinity: the
// root exists and is unique.  It is found by Newton's method kept inside a bracket [lo, hi] (a step that leaves the
// bracket is replaced by its midpoint), from the guess q of P_guess, until |dq| <= 1e-14 (1 + q); cap 100.
int con2prim_entropy(const double U[5], double US, const double Bc[3], const Geom& G, double gam,
                     const double Pguess[5], double Pout[5], int* iters) {
  if (iters) *iters = 0;
  const double ig = 1.0 / G.gdet;
  const double alpha = G.alpha;
  const double rhout = U[0] * ig;
  const double D = alpha * rhout;
  const double kappa = US / U[0];
  if (!(D > 0.0) || !(kappa >= 0.0) || !std::isfinite(D) || !std::isfinite(kappa)) return 2;
  // momentum rows exactly as in con2prim (the energy row U[1] is NOT read: Q_t follows from Q.n below only through
  // the spatial rows, see Qtsq)
  double Qcov[4] = {0.0, alpha * U[2] * ig, alpha * U[3] * ig, alpha * U[4] * ig};
  double Bs[4] = {0.0, alpha * Bc[0], alpha * Bc[1], alpha * Bc[2]};
  // Qt^2 = Qt_i Qt^i with Qt_mu = Q_mu + (Q.n) n_mu: its spatial covariant part is Q_i itself (n_i = 0), and for a
  // vector orthogonal to n the square is the 3-metric's inverse applied to the spatial part:
  //   Qt^2 = gamma^ij Q_i Q_j,  gamma^ij = g^ij + beta^i beta^j / alpha^2   (so Q_t is never needed)
  double Qtsq = 0.0, Qtcon[4] = {0.0, 0.0, 0.0, 0.0};
  for (int i = 1; i < 4; i++) {
    double acc = 0.0;
    for (int j = 1; j < 4; j++)
      acc += (G.gcon[i][j] + G.beta[i - 1] * G.beta[j - 1] / (alpha * alpha)) * Qcov[j];
    Qtcon[i] = acc;
    Qtsq += Qcov[i] * acc;
  }
  double QdB = 0.0, Bsq = 0.0;
  for (int i = 1; i < 4; i++) {
    QdB += Qcov[i] * Bs[i];
    for (int j = 1; j < 4; j++) Bsq += G.gcov[i][j] * Bs[i] * Bs[j];
  }
  const double QdB2 = QdB * QdB;
  const double c = gam / (gam - 1.0);
  const double A = c * kappa * std::pow(D, gam);  // W = D g + A g^(2 - gamma_ad)
  if (!std::isfinite(Qtsq) || !std::isfinite(Bsq) || !std::isfinite(A)) return 2;

  auto feval = [&](double q, double& W, double& df) {
    const double g = std::sqrt(1.0 + q);
    const double gp = std::pow(g, -gam);            // g^(-gamma_ad)
    W = D * g + A * gp * (1.0 + q);                 // g^(2 - gamma_ad) = g^(-gamma_ad) (1 + q)
    const double dW = D / (2.0 * g) + A * 0.5 * (2.0 - gam) * gp;
    const double v2 = q / (1.0 + q), BW = Bsq + W;
    const double W2 = W * W, W3 = W2 * W;
    df = BW * BW / ((1.0 + q) * (1.0 + q)) + 2.0 * BW * dW * (v2 + QdB2 / W3);
    return v2 * BW * BW - QdB2 * (Bsq + 2.0 * W) / W2 - Qtsq;
  };
  double W, df;
  // bracket: f(0) <= 0; hi grows by factors of 4 from 1 until f(hi) >= 0
  double lo = 0.0, hi = 1.0;
  int nb = 0;
  while (feval(hi, W, df) < 0.0) {
    lo = hi;
    hi *= 4.0;
    if (++nb > 60) return 1;
  }
  double q = 0.0;
  for (int i = 1; i < 4; i++)
    for (int j = 1; j < 4; j++) q += G.gcov[i][j] * Pguess[1 + i] * Pguess[1 + j];
  if (!(q > lo && q < hi)) q = 0.5 * (lo + hi);
  bool conv = false;
  int it;
  for (it = 0; it < 100; it++) {
    const double f = feval(q, W, df);
    if (!std::isfinite(f) || !std::isfinite(df)) { if (iters) *iters = it; return 2; }
    if (f < 0.0) lo = q; else hi = q;
    double qn = q - f / df;
    if (!(qn > lo && qn < hi)) qn = 0.5 * (lo + hi);
    const double dq = qn - q;
    q = qn;
    if (std::fabs(dq) <= 1e-14 * (1.0 + q)) { conv = true; it++; break; }
  }
  if (iters) *iters = it;
  if (!conv) return 1;
  feval(q, W, df);
  const double gamma = std::sqrt(1.0 + q);
  const double rho = D / gamma;
  const double u = kappa * std::pow(rho, gam) / (gam - 1.0);
  if (!std::isfinite(rho) || !std::isfinite(u) || !std::isfinite(W)) return 2;
  Pout[0] = rho;
  Pout[1] = u;
  for (int i = 1; i < 4; i++) Pout[1 + i] = gamma / (W + Bsq) * (Qtcon[i] + QdB * Bs[i] / W);
  return 0;
}

// ---- C-21: the Aitken-accelerated inversion ("... or Aitken acceleration scheme (Hamlin & Newman 2013;
// Newman & Hamlin 2014)"): the second primary inversion, tried where the Newton-Raphson one does not converge -------
// A fixed-point iteration on the gas pressure.  With the normal observer's e = -Q.n (total energy density, rest mass
// included), M^2 = Qt^2, T = Q.B, and  eps = W + Bsq  (W = w gamma^2), the energy equation
//   e = W - p + Bsq/2 + (Bsq v^2 - T^2/W^2)/2   and the momentum equation   M^2 = eps^2 v^2 - T^2 (2W + Bsq)/W^2
// combine (Bsq (2W + Bsq) - eps^2 = -W^2) into a cubic for eps at GIVEN pressure:
//   eps^3 - a eps^2 + d = 0,   a = e + p + Bsq/2,   d = (M^2 Bsq - T^2)/2 >= 0,
// whose largest root, for 0 <= d <= 4 a^3/27, is  eps = (a/3)(1 + 2 cos((2/3) asin sqrt(27 d/(4 a^3)))).
// Then W = eps - Bsq, v^2 = (M^2 W^2 + T^2 (Bsq + 2W))/(W eps)^2, rho = D sqrt(1 - v^2), and the new pressure
// p' = (gamma_ad - 1)/gamma_ad (W (1 - v^2) - rho).  Every third value of the sequence is replaced by Aitken's
// extrapolation  p2 - (p2 - p1)^2/((p2 - p1) - (p1 - p0)).  Start: p of P_guess.  Stop when two successive plain
// iterates differ by <= 1e-13 |p| + 1e-16 a; cap 60 double steps.  Returns 0 ok, 1 no convergence or a converged
// pressure whose v^2 had to be clamped below 1 (no state carries that momentum), 2 no real root / non-finite.  A converged root with u < 0 is returned as such (as in con2prim).
int con2prim_aitken(const double U[5], const double Bc[3], const Geom& G, double gam,
                    const double Pguess[5], double Pout[5], int* iters) {
  if (iters) *iters = 0;
  const double ig = 1.0 / G.gdet, alpha = G.alpha;
  const double rhout = U[0] * ig;
  const double D = alpha * rhout;
  double Qcov[4] = {alpha * (U[1] * ig - rhout), alpha * U[2] * ig, alpha * U[3] * ig, alpha * U[4] * ig};
  double Qcon[4], ncon[4], Bs[4] = {0.0, alpha * Bc[0], alpha * Bc[1], alpha * Bc[2]};
  for (int m = 0; m < 4; m++) {
    double acc = 0.0;
    for (int n = 0; n < 4; n++) acc += G.gcon[m][n] * Qcov[n];
    Qcon[m] = acc;
    ncon[m] = -alpha * G.gcon[m][0];
  }
  double Qdotn = 0.0, QQ = 0.0, T = 0.0, Bsq = 0.0;
  for (int m = 0; m < 4; m++) { Qdotn += Qcov[m] * ncon[m]; QQ += Qcov[m] * Qcon[m]; }
  for (int i = 1; i < 4; i++) {
    T += Qcov[i] * Bs[i];
    for (int j = 1; j < 4; j++) Bsq += G.gcov[i][j] * Bs[i] * Bs[j];
  }
  const double M2 = QQ + Qdotn * Qdotn, e = -Qdotn;
  const double d = std::max(0.0, 0.5 * (M2 * Bsq - T * T));
  const double cg = (gam - 1.0) / gam;
  if (!std::isfinite(e) || !std::isfinite(M2) || !std::isfinite(Bsq) || !(D > 0.0)) return 2;
  double W = 0.0, v2 = 0.0, a = 0.0;
  int bad = 0;
  bool clamped = false;
  auto step = [&](double p) {
    a = e + p + 0.5 * Bsq;
    if (!(a > 0.0)) { bad = 2; return p; }
    const double s2 = 27.0 * d / (4.0 * a * a * a);
    if (!(s2 <= 1.0)) { bad = 2; return p; }
    const double eps = (a / 3.0) * (1.0 + 2.0 * std::cos((2.0 / 3.0) * std::asin(std::sqrt(s2))));
    W = eps - Bsq;
    if (!(W > 0.0)) { bad = 2; return p; }
    v2 = (M2 * W * W + T * T * (Bsq + 2.0 * W)) / ((W * eps) * (W * eps));
    clamped = !(v2 <= 1.0 - 1e-15);   // more momentum than this energy can carry: iterated on, refused at the end
    v2 = std::min(std::max(v2, 0.0), 1.0 - 1e-15);
    return cg * (W * (1.0 - v2) - D * std::sqrt(1.0 - v2));
  };
  double p0 = (gam - 1.0) * Pguess[1];
  bool conv = false;
  int it;
  for (it = 0; it < 60 && !conv; it++) {
    const double p1 = step(p0);
    const double p2 = step(p1);
    if (bad || !std::isfinite(p2)) { if (iters) *iters = it; return 2; }
    conv = std::fabs(p2 - p1) <= 1e-13 * std::fabs(p2) + 1e-16 * a;
    const double den = (p2 - p1) - (p1 - p0);
    const double pa = p2 - (p2 - p1) * (p2 - p1) / den;
    p0 = (conv || den == 0.0 || !std::isfinite(pa)) ? p2 : pa;
  }
  if (iters) *iters = it;
  if (!conv) return 1;
  step(p0);   // W, v^2 of the converged pressure
  if (bad) return 2;
  if (clamped) return 1;
  const double gamma = 1.0 / std::sqrt(1.0 - v2);
  const double rho = D / gamma;
  const double u = (W / (gamma * gamma) - rho) / gam;
  if (!std::isfinite(rho) || !std::isfinite(u) || !std::isfinite(W)) return 2;
  Pout[0] = rho;
  Pout[1] = u;
  for (int i = 1; i < 4; i++) Pout[1 + i] = gamma / (W + Bsq) * (Qcon[i] + Qdotn * ncon[i] + T * Bs[i] / W);
  return 0;
}

// C-5 PPM (Colella & Woodward 1984) on a uniform grid, zone j = a[2]
static double ppm_slope(double am, double a0, double ap) {
  const double dl = a0 - am, dr = ap - a0;
  if (dl * dr <= 0.0) return 0.0;
  const double dc = 0.5 * (ap - am);
  const double lim = std::min(std::fabs(dc), std::min(2.0 * std::fabs(dl), 2.0 * std::fabs(dr)));
  return dc > 0.0 ? lim : -lim;
}

void ppm_zone(const double a[5], double& aL, double& aR) {
  const double dm_m = ppm_slope(a[0], a[1], a[2]);
  const double dm_0 = ppm_slope(a[1], a[2], a[3]);
  const double dm_p = ppm_slope(a[2], a[3], a[4]);
  aL = a[1] + 0.5 * (a[2] - a[1]) - (dm_0 - dm_m) / 6.0;  // a_{j-1/2}
  aR = a[2] + 0.5 * (a[3] - a[2]) - (dm_p - dm_0) / 6.0;  // a_{j+1/2}
  const double aj = a[2];
  if ((aR - aj) * (aj - aL) <= 0.0) {
    aL = aR = aj;
  } else {
    const double d = aR - aL;
    const double c = aj - 0.5 * (aL + aR);
    if (d * c > d * d / 6.0) aL = 3.0 * aj - 2.0 * aR;
    else if (d * c < -d * d / 6.0) aR = 3.0 * aj - 2.0 * aL;
  }
}

void plm_zone(const double a[3], double& aL, double& aR) {
  // MC limiter: minmod(2(a_j - a_{j-1}), (a_{j+1} - a_{j-1})/2, 2(a_{j+1} - a_j))
  const double dl = 2.0 * (a[1] - a[0]), dr = 2.0 * (a[2] - a[1]), dc = 0.5 * (a[2] - a[0]);
  double s = 0.0;
  if (dl * dr > 0.0) {
    s = std::min(std::fabs(dc), std::min(std::fabs(dl), std::fabs(dr)));
    if (dc < 0.0) s = -s;
  }
  aL = a[1] - 0.5 * s;
  aR = a[1] + 0.5 * s;
}

}  // namespace orc
