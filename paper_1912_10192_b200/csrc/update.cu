// update.cu — face-B update, geometric source, conservative update, conserved-to-primitive inversion,
// floors and ceiling in ONE kernel (SURVEY §8(a) H2 second half, H3, H4; north_star items 3-5).
// "the source terms are added at cell centers to compute the cell-centered values of the
// conserved quantities U at the new time"; "(multi-)dimensional Newton-Raphson ...
// Noble et al. 2006"; floors.  DESIGN.md C-10, C-12, C-13.
// The conserved vector never touches HBM: U_base, div F, S and the inversion stay in registers.
#include "hamr_host.h"

namespace hamr {

// face-B update of the d-face on the low side of z (C-10):
// Bf^d -= dt [ (E_f(e+) - E_f(e-))/dx^e - (E_e(f+) - E_e(f-))/dx^f ], (d,e,f) cyclic
// All index arithmetic is 32-bit (an array holds fewer than 2^31 doubles, checked at creation).
template <int d>
__device__ __forceinline__ double bf_new(const Dev& Dv, const double* __restrict__ base, int z, double dt,
                                         const int S[3], const double idx[3]) {
  constexpr int e = (d + 1) % 3, f = (d + 2) % 3;
  const double curl = (__ldg(Dv.Ee[f] + z + S[e]) - __ldg(Dv.Ee[f] + z)) * idx[e] -
                      (__ldg(Dv.Ee[e] + z + S[f]) - __ldg(Dv.Ee[e] + z)) * idx[f];
  return __ldg(base + z) - dt * curl;
}

template <bool BLK>
__device__ __forceinline__ Fields pick_fields(const Fields& a, const Fields& b, int cur) {
  Fields f;
#pragma unroll
  for (int c = 0; c < 5; c++) f.P[c] = selp<BLK>(a.P[c], b.P[c], cur);
#pragma unroll
  for (int c = 0; c < 3; c++) { f.Bc[c] = selp<BLK>(a.Bc[c], b.Bc[c], cur); f.Bf[c] = selp<BLK>(a.Bf[c], b.Bf[c], cur); }
  return f;
}

#ifndef HAMR_UPD_MINB
#define HAMR_UPD_MINB 6
#endif
#ifndef HAMR_UPD_MINB_PRED
#define HAMR_UPD_MINB_PRED 7
#endif
#ifndef HAMR_UPD_RELOAD
#define HAMR_UPD_RELOAD 1
#endif
template <bool SAME, bool BLK>  // SAME: predictor, source state == base state
__global__ void __launch_bounds__(128, SAME ? HAMR_UPD_MINB_PRED : HAMR_UPD_MINB) k_update(Dev Dv, Roles ra, Roles rb, double dtfac) {
  const Lay& L = Dv.L;
  // k runs over [0, n3): warps start on 128-byte lines when n3 is a multiple of 32; the thread at k = 0 also
  // builds the x3-face at k = n3
  const int c2 = L.n[2], c1 = L.n[1] + 1;
  const unsigned per = (unsigned)(L.n[0] + 1) * c1 * c2;
  unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = t < (BLK ? per * Dv.B.nact : per);
  int nfail = 0, nrf = 0, nuf = 0, ngc = 0, bad = 0;
  if (valid) {
    int bslot = 0;
    if (BLK) { bslot = (int)(t / per); t -= bslot * per; }
    const BCtx C = blk_ctx<BLK>(Dv, bslot);
    const Fields src = pick_fields<BLK>(ra.src, rb.src, C.cur), base = pick_fields<BLK>(ra.base, rb.base, C.cur),
                 out = pick_fields<BLK>(ra.out, rb.out, C.cur);
    const unsigned tj = t / (unsigned)c2;
    const int k = (int)(t - tj * c2);
    const int i = (int)(tj / (unsigned)c1);
    const int j = (int)(tj - i * c1);
    const int z = C.zoff + (int)L.idx(i, j, k);
    const double dt = dtfac * Dv.scal[S_DT];
    const int S[3] = {L.S1, L.S2, 1};
    const double idx[3] = {1.0 / ((BLK && C.lev) ? 0.5 * Dv.dx[0] : Dv.dx[0]), 1.0 / Dv.dx[1], 1.0 / Dv.dx[2]};
    const bool in0 = i < L.n[0], in1 = j < L.n[1];
    const bool ks = Dv.metric == HAMR_METRIC_KERR_SCHILD;
    const int Jg = C.J0 + j, n2g = BLK ? Dv.B.n2g : L.n[1];
    double lo[3] = {0.0, 0.0, 0.0};
    if (in1) { lo[0] = bf_new<0>(Dv, base.Bf[0], z, dt, S, idx); out.Bf[0][z] = lo[0]; }
    if (in0) {
      lo[1] = (ks && (Jg == 0 || Jg == n2g)) ? 0.0 : bf_new<1>(Dv, base.Bf[1], z, dt, S, idx);
      out.Bf[1][z] = lo[1];
    }
    if (in0 && in1) {
      lo[2] = bf_new<2>(Dv, base.Bf[2], z, dt, S, idx);
      out.Bf[2][z] = lo[2];
      if (k == 0) out.Bf[2][z + L.n[2]] = bf_new<2>(Dv, base.Bf[2], z + L.n[2], dt, S, idx);
      const double* grec = Dv.gcA + (BLK ? C.lev * Dv.B.tlevA : 0) + (size_t)(C.q0 + i * (BLK ? Dv.B.ge2 : L.e2) + j) * NREC_C;
      const CGeo G = load_cgeo(grec);
      // new cell-centred field from the new faces (the high faces are recomputed, bit-identically)
      double Bn[3];
      {
        const double h0 = bf_new<0>(Dv, base.Bf[0], z + S[0], dt, S, idx);
        const double h1 = (ks && Jg + 1 == n2g) ? 0.0 : bf_new<1>(Dv, base.Bf[1], z + S[1], dt, S, idx);
        double h2 = bf_new<2>(Dv, base.Bf[2], z + S[2], dt, S, idx), l2 = lo[2];
        if (Dv.mrow) {
          // C-15: in a phi-derefined row B_c^3 is the GROUP's value, from the group's two outer x3-faces
          const int m = __ldg(Dv.mrow + Jg + NG);
          if (m > 1) {
            const int zg = z - (k % m);
            l2 = bf_new<2>(Dv, base.Bf[2], zg, dt, S, idx);
            h2 = bf_new<2>(Dv, base.Bf[2], zg + m, dt, S, idx);
          }
        }
        const double i2g = 0.5 * G.igdet;
        Bn[0] = (lo[0] + h0) * i2g;
        Bn[1] = (lo[1] + h1) * i2g;
        Bn[2] = (l2 + h2) * i2g;
      }
      double Ps[8], U[5], Ssrc1, Ssrc2;
#pragma unroll
      for (int c = 0; c < 5; c++) Ps[c] = __ldg(src.P[c] + z);
#pragma unroll
      for (int c = 0; c < 3; c++) Ps[5 + c] = __ldg(src.Bc[c] + z);
      {
        St Ss;
        get_state(Ps, G, Ss);
        if (SAME) prim_to_U5(Ps, Ss, G.gdet, Dv.gam, U);
        source_12(Ps, Ss, G, Dv.gam, grec, Ssrc1, Ssrc2);   // C-12: on the stage's source state
      }
      if (!SAME) {
        double Pb[8];
#pragma unroll
        for (int c = 0; c < 5; c++) Pb[c] = __ldg(base.P[c] + z);
#pragma unroll
        for (int c = 0; c < 3; c++) Pb[5 + c] = __ldg(base.Bc[c] + z);
        St Sb;
        get_state(Pb, G, Sb);
        prim_to_U5(Pb, Sb, G.gdet, Dv.gam, U);
      }
      // U_new = U_base - dt sum_d (F^d_+ - F^d_-)/dx^d + dt S
#pragma unroll
      for (int c = 0; c < 5; c++) {
        double div = 0.0;
#pragma unroll
        for (int d = 0; d < 3; d++) div += (__ldg(Dv.F[d][c] + z + S[d]) - __ldg(Dv.F[d][c] + z)) * idx[d];
        const double sc = (c == 2) ? Ssrc1 : (c == 3 ? Ssrc2 : 0.0);
        U[c] = U[c] - dt * div + dt * sc;
      }
      double Pn[5], Pg[5];
#if HAMR_UPD_RELOAD
      // the geometry record and the guess are re-read (L1 / L2 hits) instead of being kept in registers
      // across the flux divergence: lower register pressure, more resident warps
      const double* gtab = grec;
      asm volatile("" : "+l"(gtab));
      const CGeo G2 = load_cgeo(gtab);
      const double* sp[5] = {src.P[0], src.P[1], src.P[2], src.P[3], src.P[4]};
#pragma unroll
      for (int c = 0; c < 5; c++) { const double* a = sp[c]; asm volatile("" : "+l"(a)); Pg[c] = a[z]; }
#else
      const CGeo& G2 = G;
#pragma unroll
      for (int c = 0; c < 5; c++) Pg[c] = Ps[c];
#endif
      if (con2prim(U, Bn, G2, Dv.gam, Pg, Pn) != 0) {  // C-13: keep the source state's hydro primitives, count the failure
        nfail = 1;
#pragma unroll
        for (int c = 0; c < 5; c++) Pn[c] = Pg[c];
      }
      // floors and Lorentz-factor ceiling (C-13)
      const int fi = C.I0 + i + NG + (BLK ? C.lev * Dv.B.flev : 0);
      floors_ceiling(G2, __ldg(Dv.rho_fl + fi), __ldg(Dv.u_fl + fi), Dv.gamma_max, Pn, nrf, nuf, ngc);
#pragma unroll
      for (int c = 0; c < 5; c++) {
        out.P[c][z] = Pn[c];
        if (!(fabs(Pn[c]) <= 1.79e308)) bad = 1;
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

// ra / rb: the stage's roles in the buffer sets of blocks with cur == 0 / 2 (monolithic: rb unused)
void launch_update_on(hamr_grid* g, const Dev& Dv, const Roles& ra, const Roles& rb, double dtfac, bool same) {
  const Lay& L = Dv.L;
  const bool blk = Dv.B.nblk > 0;
  if (blk && Dv.B.nact == 0) return;
  const long long tot = (long long)(L.n[0] + 1) * (L.n[1] + 1) * L.n[2] * (blk ? Dv.B.nact : 1);
  const unsigned nb = (unsigned)((tot + 127) / 128);
  Launch l_(g, same ? K_UPDATE_P : K_UPDATE_C);
  if (same && !blk) k_update<true, false><<<nb, 128, 0, g->stream>>>(Dv, ra, rb, dtfac);
  else if (same) k_update<true, true><<<nb, 128, 0, g->stream>>>(Dv, ra, rb, dtfac);
  else if (!blk) k_update<false, false><<<nb, 128, 0, g->stream>>>(Dv, ra, rb, dtfac);
  else k_update<false, true><<<nb, 128, 0, g->stream>>>(Dv, ra, rb, dtfac);
}

void launch_update(hamr_grid* g, const Fields& src, const Fields& base, const Fields& out, double dtfac,
                   bool src_is_base) {
  const Roles r = {src, base, out};
  launch_update_on(g, g->D, r, r, dtfac, src_is_base);
}

}  // namespace hamr
