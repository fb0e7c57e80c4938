// flux.cu — fused reconstruct + HLL kernels, one per direction (north_star items 1+2).
// "finite volume shock-capturing Godunov-based HLLE scheme ... third order accurate
// spatial reconstruction (PPM)"; fluxes are evaluated at cell faces.
// Each face: PPM (or PLM-MC) left/right states of the 7 non-normal primitives (C-5), the normal
// field from the staggered face B, U/F of both states (C-4), fast-speed bounds (C-6), HLL flux of
// the 5 hydro rows and the 2 transverse-B rows (= face EMFs, C-7/C-8), and the per-direction
// maximum signal speed for the Courant step (C-14).
#include "hamr_host.h"

namespace hamr {

// HLL for one row
__device__ __forceinline__ double hll1(double UL, double UR, double FL, double FR, double cmin, double cmax,
                                       double cc, double isum, bool avg) {
  return avg ? 0.5 * (FL + FR) : (cmax * FL + cmin * FR - cc * (UR - UL)) * isum;
}

// Physics of one face along direction D (0..2) from the two reconstructed states.
// Fh[0..4]: hydro flux; EA = E_e, EB = E_f on the face with (D, e, f) cyclic; returns ctop.
template <int D>
__device__ __forceinline__ double face_physics(const double PL[8], const double PR[8], const Geo& G,
                                               double gam_ad, double Fh[5], double& EA, double& EB) {
  constexpr int dir = D + 1, e = (D + 1) % 3, f = (D + 2) % 3;
  const double A = (D == 0) ? G.k11 : (D == 1 ? G.k22 : G.k33);
  const double Cq = (D == 0) ? G.k01 : 0.0;
  double UL[7], UR[7], FL[7], FR[7];
  double vminL, vmaxL, vminR, vmaxR;
#pragma unroll
  for (int side = 0; side < 2; side++) {
    const double* P = side ? PR : PL;
    double* U = side ? UR : UL;
    double* F = side ? FR : FL;
    St S;
    get_state(P, G, S);
    const double p = (gam_ad - 1.0) * P[1];
    const double eta = P[0] + P[1] + p + S.bsq;
    const double ptot = p + 0.5 * S.bsq;
    const double eu0 = eta * S.ucon[0], eud = eta * S.ucon[dir];
    const double b0 = S.bcon[0], bd = S.bcon[dir];
    const double Dn = P[0] * S.ucon[0], m = P[0] * S.ucon[dir];
    U[0] = G.gdet * Dn;
    U[1] = G.gdet * (eu0 * S.ucov[0] + ptot - b0 * S.bcov[0] + Dn);
    F[0] = G.gdet * m;
    F[1] = G.gdet * (eud * S.ucov[0] - bd * S.bcov[0] + m);
#pragma unroll
    for (int c = 1; c < 4; c++) {
      U[1 + c] = G.gdet * (eu0 * S.ucov[c] - b0 * S.bcov[c]);
      F[1 + c] = G.gdet * (eud * S.ucov[c] + (c == dir ? ptot : 0.0) - bd * S.bcov[c]);
    }
    // transverse field rows: U = g B^i, F = g (b^i u^d - b^d u^i)
    U[5] = G.gdet * P[5 + e];
    U[6] = G.gdet * P[5 + f];
    F[5] = G.gdet * (S.bcon[1 + e] * S.ucon[dir] - bd * S.ucon[1 + e]);
    F[6] = G.gdet * (S.bcon[1 + f] * S.ucon[dir] - bd * S.ucon[1 + f]);
    wavespeeds(P, S, gam_ad, A, G.k00, Cq, dir, side ? vminR : vminL, side ? vmaxR : vmaxL);
  }
  const double cmax = fmax(0.0, fmax(vmaxL, vmaxR));
  const double cmin = fmax(0.0, fmax(-vminL, -vminR));
  const double sum = cmax + cmin;
  const bool avg = sum < 1e-300;
  const double isum = avg ? 0.0 : 1.0 / sum;
  const double cc = cmax * cmin;
#pragma unroll
  for (int c = 0; c < 5; c++) Fh[c] = hll1(UL[c], UR[c], FL[c], FR[c], cmin, cmax, cc, isum, avg);
  const double Fe = hll1(UL[5], UR[5], FL[5], FR[5], cmin, cmax, cc, isum, avg);
  const double Ff = hll1(UL[6], UR[6], FL[6], FR[6], cmin, cmax, cc, isum, avg);
  if (!avg) {
    // C-7a: a mass flux below 1e-12 of the magnitude of its own HLL terms is rounding noise and is
    // flushed to exactly 0, so that the upwind selector of C-9 sees a tie
    const double mag = (cmax * fabs(FL[0]) + cmin * fabs(FR[0]) + cc * (fabs(UR[0]) + fabs(UL[0]))) * isum;
    if (fabs(Fh[0]) <= 1e-12 * mag) Fh[0] = 0.0;
  }
  EB = -Fe;  // C-8: on a d-face, E_f = -F^d(B^e)
  EA = Ff;   //                    E_e = +F^d(B^f)
  return fmax(cmax, cmin);
}

// v1: one thread per face, stencil read straight from global memory (L1/L2 catch the reuse).
template <int D, int RECON>
__global__ void __launch_bounds__(128) k_flux(Dev Dv, Fields s, int want_ctop) {
  const Lay& L = Dv.L;
  constexpr int e = (D + 1) % 3, f = (D + 2) % 3;
  // box of faces: 0..n along D, one transverse ghost layer on each side (needed by CT)
  int lo[3] = {-1, -1, -1}, cntd[3];
  lo[D] = 0;
  for (int d = 0; d < 3; d++) cntd[d] = (d == D) ? L.n[d] + 1 : L.n[d] + 2;
  const long long tot = (long long)cntd[0] * cntd[1] * cntd[2];
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  double ctop = 0.0;
  if (t < tot) {
    const int k = (int)(t % cntd[2]) + lo[2];
    const int j = (int)((t / cntd[2]) % cntd[1]) + lo[1];
    const int i = (int)(t / ((long long)cntd[2] * cntd[1])) + lo[0];
    const long long z = L.idx(i, j, k);
    const int q = L.idx2(i, j);
    const bool pole = (D == 1) && Dv.metric == HAMR_METRIC_KERR_SCHILD && (j == 0 || j == L.n[1]);
    double Fh[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, EA = 0.0, EB = 0.0;
    if (!pole) {  // C-7: pole faces carry no flux and no state is evaluated there
      const Geo G = load_geo(D == 0 ? Dv.gf1 : (D == 1 ? Dv.gf2 : Dv.gc), L.n2d, q);
      const long long sd = (D == 0) ? L.S1 : (D == 1 ? L.S2 : 1);
      double PL[8], PR[8];
      const double* var[7] = {s.P[0], s.P[1], s.P[2], s.P[3], s.P[4], s.Bc[e], s.Bc[f]};
      const int slot[7] = {0, 1, 2, 3, 4, 5 + e, 5 + f};
#pragma unroll
      for (int v = 0; v < 7; v++) {
        const double* a = var[v] + z;
        double aL, aR, dummy;
        if (RECON == HAMR_RECON_PPM) {
          const double m3 = a[-3 * sd], m2 = a[-2 * sd], m1 = a[-sd], c0 = a[0], p1 = a[sd], p2 = a[2 * sd];
          ppm_zone(m3, m2, m1, c0, p1, dummy, aR);  // left of the face: a_R of zone j-1
          ppm_zone(m2, m1, c0, p1, p2, aL, dummy);  // right of the face: a_L of zone j
        } else {
          const double m2 = a[-2 * sd], m1 = a[-sd], c0 = a[0], p1 = a[sd];
          plm_zone(m2, m1, c0, dummy, aR);
          plm_zone(m1, c0, p1, aL, dummy);
        }
        PL[slot[v]] = aR;
        PR[slot[v]] = aL;
      }
      PL[5 + D] = PR[5 + D] = s.Bf[D][z] / G.gdet;  // C-5: the normal field is single-valued at the face
      const double ct = face_physics<D>(PL, PR, G, Dv.gam, Fh, EA, EB);
      // C-14: the Courant maximum runs over the faces of ACTIVE zones
      const int id[3] = {i, j, k};
      bool act = true;
      for (int d = 0; d < 3; d++)
        if (d != D && (id[d] < 0 || id[d] >= L.n[d])) act = false;
      if (act) ctop = ct;
    }
#pragma unroll
    for (int c = 0; c < 5; c++) Dv.F[D][c][z] = Fh[c];
    Dv.EfA[D][z] = EA;
    Dv.EfB[D][z] = EB;
  }
  if (want_ctop) {
    ctop = warp_max(ctop);
    if ((threadIdx.x & 31) == 0 && ctop > 0.0) atomic_max_pos(Dv.scal + S_CTOP0 + D, ctop);
  }
}

template <int D>
static void launch_flux_d(hamr_grid* g, const Fields& src, bool want_ctop) {
  const Lay& L = g->D.L;
  long long tot = 1;
  for (int d = 0; d < 3; d++) tot *= (d == D) ? L.n[d] + 1 : L.n[d] + 2;
  const unsigned nb = (unsigned)((tot + 127) / 128);
  Launch l_(g, K_FLUX1 + D);
  if (g->D.recon == HAMR_RECON_PPM)
    k_flux<D, HAMR_RECON_PPM><<<nb, 128, 0, g->stream>>>(g->D, src, want_ctop ? 1 : 0);
  else
    k_flux<D, HAMR_RECON_PLM_MC><<<nb, 128, 0, g->stream>>>(g->D, src, want_ctop ? 1 : 0);
}

void launch_flux(hamr_grid* g, const Fields& src, bool want_ctop) {
  launch_flux_d<0>(g, src, want_ctop);
  launch_flux_d<1>(g, src, want_ctop);
  launch_flux_d<2>(g, src, want_ctop);
}

}  // namespace hamr
