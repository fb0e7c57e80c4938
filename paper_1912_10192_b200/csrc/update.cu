// update.cu — face-B update, geometric source, conservative update, conserved-to-primitive inversion,
// floors and ceiling in ONE kernel (SURVEY §8(a) H2 second half, H3, H4; north_star items 3-5).
// "the source terms are added at cell centers to compute the cell-centered values of the
// conserved quantities U at the new time"; "(multi-)dimensional Newton-Raphson ...
// Noble et al. 2006"; floors.  DESIGN.md C-10, C-12, C-13.
// The conserved vector never touches HBM: U_base, div F, S and the inversion stay in registers.
#include "hamr_host.h"

namespace hamr {

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

// face-B update of the d-face on the low side of z (C-10):
// Bf^d -= dt [ (E_f(e+) - E_f(e-))/dx^e - (E_e(f+) - E_e(f-))/dx^f ], (d,e,f) cyclic
template <int d>
__device__ __forceinline__ double bf_new(const Dev& Dv, const double* __restrict__ base, long long z, double dt,
                                         const long long S[3], const double idx[3]) {
  constexpr int e = (d + 1) % 3, f = (d + 2) % 3;
  const double curl = (Dv.Ee[f][z + S[e]] - Dv.Ee[f][z]) * idx[e] - (Dv.Ee[e][z + S[f]] - Dv.Ee[e][z]) * idx[f];
  return base[z] - dt * curl;
}

template <bool SAME>  // SAME: predictor, source state == base state
__global__ void __launch_bounds__(128) k_update(Dev Dv, Fields src, Fields base, Fields out, double dtfac) {
  const Lay& L = Dv.L;
  const int c2 = L.n[2] + 1, c1 = L.n[1] + 1;
  const long long tot = (long long)(L.n[0] + 1) * c1 * c2;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = t < tot;
  int nfail = 0, nrf = 0, nuf = 0, ngc = 0, bad = 0;
  if (valid) {
    const int k = (int)(t % c2);
    const int j = (int)((t / c2) % c1);
    const int i = (int)(t / ((long long)c2 * c1));
    const long long z = L.idx(i, j, k);
    const double dt = dtfac * Dv.scal[S_DT];
    const long long S[3] = {L.S1, L.S2, 1};
    const double idx[3] = {1.0 / Dv.dx[0], 1.0 / Dv.dx[1], 1.0 / Dv.dx[2]};
    const bool in0 = i < L.n[0], in1 = j < L.n[1], in2 = k < L.n[2];
    const bool ks = Dv.metric == HAMR_METRIC_KERR_SCHILD;
    double lo[3] = {0.0, 0.0, 0.0};
    if (in1 && in2) { lo[0] = bf_new<0>(Dv, base.Bf[0], z, dt, S, idx); out.Bf[0][z] = lo[0]; }
    if (in0 && in2) {
      lo[1] = (ks && (j == 0 || j == L.n[1])) ? 0.0 : bf_new<1>(Dv, base.Bf[1], z, dt, S, idx);
      out.Bf[1][z] = lo[1];
    }
    if (in0 && in1) { lo[2] = bf_new<2>(Dv, base.Bf[2], z, dt, S, idx); out.Bf[2][z] = lo[2]; }
    if (in0 && in1 && in2) {
      const int q = L.idx2(i, j);
      const Geo G = load_geo(Dv.gc, L.n2d, q);
      // new cell-centred field from the new faces (the high faces are recomputed, bit-identically)
      double Bn[3];
      {
        const double h0 = bf_new<0>(Dv, base.Bf[0], z + S[0], dt, S, idx);
        const double h1 = (ks && j + 1 == L.n[1]) ? 0.0 : bf_new<1>(Dv, base.Bf[1], z + S[1], dt, S, idx);
        const double h2 = bf_new<2>(Dv, base.Bf[2], z + S[2], dt, S, idx);
        const double i2g = 1.0 / (2.0 * G.gdet);
        Bn[0] = (lo[0] + h0) * i2g;
        Bn[1] = (lo[1] + h1) * i2g;
        Bn[2] = (lo[2] + h2) * i2g;
      }
      double Ps[8], U[5], Ssrc1, Ssrc2;
#pragma unroll
      for (int c = 0; c < 5; c++) Ps[c] = src.P[c][z];
#pragma unroll
      for (int c = 0; c < 3; c++) Ps[5 + c] = src.Bc[c][z];
      {
        St Ss;
        get_state(Ps, G, Ss);
        if (SAME) prim_to_U5(Ps, Ss, G.gdet, Dv.gam, U);
        // C-12 source: S_nu = g T^kappa_lambda Gamma^lambda_{nu kappa} = (g/2) T^{kappa lambda} d_nu g_{kappa lambda};
        // both metrics are stationary and independent of x3, so S_t = S_3 = 0 identically
        const double p = (Dv.gam - 1.0) * Ps[1];
        const double eta = Ps[0] + Ps[1] + p + Ss.bsq;
        const double ptot = p + 0.5 * Ss.bsq;
        const double* u = Ss.ucon;
        const double* b = Ss.bcon;
        const double T00 = eta * u[0] * u[0] + ptot * G.k00 - b[0] * b[0];
        const double T01 = eta * u[0] * u[1] + ptot * G.k01 - b[0] * b[1];
        const double T03 = eta * u[0] * u[3] - b[0] * b[3];
        const double T11 = eta * u[1] * u[1] + ptot * G.k11 - b[1] * b[1];
        const double T13 = eta * u[1] * u[3] + ptot * G.k13 - b[1] * b[3];
        const double T22 = eta * u[2] * u[2] + ptot * G.k22 - b[2] * b[2];
        const double T33 = eta * u[3] * u[3] + ptot * G.k33 - b[3] * b[3];
        const double* d1 = Dv.dgc + q;
        const int n2d = L.n2d;
        double a1 = 0.5 * (T00 * __ldg(d1 + D00 * n2d) + T11 * __ldg(d1 + D11 * n2d) + T22 * __ldg(d1 + D22 * n2d) +
                           T33 * __ldg(d1 + D33 * n2d)) +
                    T01 * __ldg(d1 + D01 * n2d) + T03 * __ldg(d1 + D03 * n2d) + T13 * __ldg(d1 + D13 * n2d);
        const double* d2 = d1 + NDG * n2d;
        double a2 = 0.5 * (T00 * __ldg(d2 + D00 * n2d) + T11 * __ldg(d2 + D11 * n2d) + T22 * __ldg(d2 + D22 * n2d) +
                           T33 * __ldg(d2 + D33 * n2d)) +
                    T01 * __ldg(d2 + D01 * n2d) + T03 * __ldg(d2 + D03 * n2d) + T13 * __ldg(d2 + D13 * n2d);
        Ssrc1 = G.gdet * a1;
        Ssrc2 = G.gdet * a2;
      }
      if (!SAME) {
        double Pb[8];
#pragma unroll
        for (int c = 0; c < 5; c++) Pb[c] = base.P[c][z];
#pragma unroll
        for (int c = 0; c < 3; c++) Pb[5 + c] = base.Bc[c][z];
        St Sb;
        get_state(Pb, G, Sb);
        prim_to_U5(Pb, Sb, G.gdet, Dv.gam, U);
      }
      // U_new = U_base - dt sum_d (F^d_+ - F^d_-)/dx^d + dt S
#pragma unroll
      for (int c = 0; c < 5; c++) {
        double div = 0.0;
#pragma unroll
        for (int d = 0; d < 3; d++) div += (Dv.F[d][c][z + S[d]] - Dv.F[d][c][z]) * idx[d];
        const double sc = (c == 2) ? Ssrc1 : (c == 3 ? Ssrc2 : 0.0);
        U[c] = U[c] - dt * div + dt * sc;
      }
      double Pn[5];
      const int rc = con2prim(U, Bn, G, Dv.gam, Ps, Pn);
      if (rc != 0) {  // C-13: keep the source state's hydro primitives, count the failure
        nfail = 1;
#pragma unroll
        for (int c = 0; c < 5; c++) Pn[c] = Ps[c];
      }
      // floors and Lorentz-factor ceiling (C-13)
      const double rfl = __ldg(Dv.rho_fl + i + NG), ufl = __ldg(Dv.u_fl + i + NG);
      if (Pn[0] < rfl) { Pn[0] = rfl; nrf = 1; }
      if (Pn[1] < ufl) { Pn[1] = ufl; nuf = 1; }
      const double gamma = sqrt(1.0 + vsq_tilde(G, Pn[2], Pn[3], Pn[4]));
      if (gamma > Dv.gamma_max) {
        const double fac = sqrt((Dv.gamma_max * Dv.gamma_max - 1.0) / (gamma * gamma - 1.0));
        Pn[2] *= fac; Pn[3] *= fac; Pn[4] *= fac;
        ngc = 1;
      }
#pragma unroll
      for (int c = 0; c < 5; c++) {
        out.P[c][z] = Pn[c];
        if (!isfinite(Pn[c])) bad = 1;
      }
#pragma unroll
      for (int c = 0; c < 3; c++) out.Bc[c][z] = Bn[c];
    }
  }
  // warp-aggregated event counters
  const unsigned m_f = __ballot_sync(0xffffffffu, nfail), m_r = __ballot_sync(0xffffffffu, nrf),
                 m_u = __ballot_sync(0xffffffffu, nuf), m_g = __ballot_sync(0xffffffffu, ngc),
                 m_b = __ballot_sync(0xffffffffu, bad);
  if ((threadIdx.x & 31) == 0) {
    if (m_f) atomicAdd(Dv.cnt + N_C2PFAIL, (unsigned long long)__popc(m_f));
    if (m_r) atomicAdd(Dv.cnt + N_RHOFL, (unsigned long long)__popc(m_r));
    if (m_u) atomicAdd(Dv.cnt + N_UFL, (unsigned long long)__popc(m_u));
    if (m_g) atomicAdd(Dv.cnt + N_GCEIL, (unsigned long long)__popc(m_g));
    if (m_b) atomicAdd(Dv.cnt + N_NONFINITE, (unsigned long long)__popc(m_b));
  }
}

void launch_update(hamr_grid* g, const Fields& src, const Fields& base, const Fields& out, double dtfac,
                   bool src_is_base) {
  const Lay& L = g->D.L;
  const long long tot = (long long)(L.n[0] + 1) * (L.n[1] + 1) * (L.n[2] + 1);
  const unsigned nb = (unsigned)((tot + 127) / 128);
  Launch l_(g, src_is_base ? K_UPDATE_P : K_UPDATE_C);
  if (src_is_base) k_update<true><<<nb, 128, 0, g->stream>>>(g->D, src, base, out, dtfac);
  else k_update<false><<<nb, 128, 0, g->stream>>>(g->D, src, base, out, dtfac);
}

}  // namespace hamr
