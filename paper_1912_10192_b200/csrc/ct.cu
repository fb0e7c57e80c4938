// ct.cu — constrained transport: centre EMFs and velocity-upwinded edge EMFs.
// "magnetic fields are evolved on a staggered grid, where the electric fields have been
// velocity upwinded to add dissipation (Gardiner & Stone 2005)".  DESIGN.md C-8 (centre EMF
// E^c_k = -eps_kmn v^m (g B^n)), C-9 (edge EMF from 4 face EMFs, 4 centre EMFs and the sign of the
// HLL mass fluxes; edges on the polar axis carry E1 = E3 = 0).
#include "hamr_host.h"

namespace hamr {

// centre EMFs on active zones plus one ghost layer.  WRAP (x3_ghosts_unused): k runs over [0, n3) and the two x3
// ghost columns are stored as the periodic images of columns n3 - 1 and 0 (their zones are not read)
// 16 CTAs of 128 threads per SM (32 registers): 0.063 -> 0.058 ms on cfg 2 (it is bound by memory latency); the edge
// kernel below gains nothing from the same cap (0.105 ms at 40 or 32 registers)
template <bool BLK, bool WRAP>
__global__ void __launch_bounds__(128, 16) k_centre_emf(Dev Dv, Fields s0, Fields s2) {
  const Lay& L = Dv.L;
  const int c2 = L.n[2] + (WRAP ? 0 : 2), c1 = L.n[1] + 2;
  const unsigned per = (unsigned)(L.n[0] + 2) * c1 * c2;
  unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (BLK ? per * Dv.B.nact : per)) return;
  int bslot = 0;
  if (BLK) { bslot = (int)(t / per); t -= bslot * per; }
  const BCtx C = blk_ctx<BLK>(Dv, bslot);
  const unsigned tj = t / (unsigned)c2, ti = tj / (unsigned)c1;
  const int k = (int)(t - tj * c2) - (WRAP ? 0 : 1);
  const int j = (int)(tj - ti * c1) - 1;
  const int i = (int)ti - 1;
  const long long z = C.zoff + L.idx(i, j, k);
  const int q = C.q0 + i * (BLK ? Dv.B.ge2 : L.e2) + j;
  Fields s;
  for (int c = 2; c < 5; c++) s.P[c] = selp<BLK>(s0.P[c], s2.P[c], C.cur);
  for (int c = 0; c < 3; c++) s.Bc[c] = selp<BLK>(s0.Bc[c], s2.Bc[c], C.cur);
  // the zone's geometry record (array-of-records table: two cache lines instead of seven, hamr_dev.cuh)
  const double* rec = Dv.gcA + (BLK ? C.lev * Dv.B.tlevA : 0) + (size_t)q * NREC_C;
  const double c11 = __ldg(rec + CREC_C11), c13 = __ldg(rec + CREC_C13), c22 = __ldg(rec + CREC_C22),
               c33 = __ldg(rec + CREC_C33), gdet = __ldg(rec + CREC_GDET), ialpha = __ldg(rec + CREC_IALPHA),
               boa = __ldg(rec + CREC_BOA);
  const double v1 = s.P[2][z], v2 = s.P[3][z], v3 = s.P[4][z];
  const double gam = sqrt(1.0 + (c11 * v1 * v1 + c22 * v2 * v2 + c33 * v3 * v3 + 2.0 * (c13 * v1 * v3)));
  const double iut = 1.0 / (gam * ialpha);
  const double w1 = (v1 - gam * boa) * iut, w2 = v2 * iut, w3 = v3 * iut;  // v^i = u^i / u^t
  const double B1 = gdet * s.Bc[0][z], B2 = gdet * s.Bc[1][z], B3 = gdet * s.Bc[2][z];
  const double e0 = -(w2 * B3 - w3 * B2), e1 = -(w3 * B1 - w1 * B3), e2 = -(w1 * B2 - w2 * B1);
  Dv.Cc[0][z] = e0;
  Dv.Cc[1][z] = e1;
  Dv.Cc[2][z] = e2;
  if (WRAP) {
    const int n3 = L.n[2];
    const long long zd = (k == n3 - 1) ? z - n3 : (k == 0 ? z + n3 : -1);
    if (zd >= 0) { Dv.Cc[0][zd] = e0; Dv.Cc[1][zd] = e1; Dv.Cc[2][zd] = e2; }
  }
}

__device__ __forceinline__ double up(double m, double lo, double hi) {
  return m > 0.0 ? lo : (m < 0.0 ? hi : 0.5 * (lo + hi));
}

// E_f at edge (d-1/2, e-1/2) of zone z, (f, d, e) cyclic.  X = E_f on d-faces, Y = E_f on e-faces,
// C = centre E_f, md / me = HLL mass fluxes through d- / e-faces.
__device__ __forceinline__ double edge_emf(const double* __restrict__ X, const double* __restrict__ Y,
                                           const double* __restrict__ C, const double* __restrict__ md,
                                           const double* __restrict__ me, long long z, long long sD,
                                           long long sE) {
  const double Xz = X[z], Xe = X[z - sE], Yz = Y[z], Yd = Y[z - sD];
  const double Cz = C[z], Cd = C[z - sD], Ce = C[z - sE], Cde = C[z - sD - sE];
  return 0.25 * (Xz + Xe + Yz + Yd) +
         0.25 * (up(md[z - sE], Yd - Cde, Yz - Ce) - up(md[z], Cd - Yd, Cz - Yz)) +
         0.25 * (up(me[z - sD], Xe - Cde, Xz - Cd) - up(me[z], Ce - Xe, Cz - Xz));
}

// one thread per zone corner: the three edge EMFs on the low edges of zone (i,j,k), 0 <= idx <= n
template <bool BLK>
__global__ void __launch_bounds__(128) k_edge_emf(Dev Dv) {
  const Lay& L = Dv.L;
  const int c2 = L.n[2] + 1, c1 = L.n[1] + 1;
  const unsigned per = (unsigned)(L.n[0] + 1) * c1 * c2;
  unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (BLK ? per * Dv.B.nact : per)) return;
  int bslot = 0;
  if (BLK) { bslot = (int)(t / per); t -= bslot * per; }
  const BCtx C = blk_ctx<BLK>(Dv, bslot);
  const unsigned tj = t / (unsigned)c2, ti = tj / (unsigned)c1;
  const int k = (int)(t - tj * c2);
  const int j = (int)(tj - ti * c1);
  const int i = (int)ti;
  const long long z = C.zoff + L.idx(i, j, k);
  const bool pole = Dv.metric == HAMR_METRIC_KERR_SCHILD && (C.J0 + j == 0 || C.J0 + j == (BLK ? Dv.B.n2g : L.n[1]));
  const long long S[3] = {L.S1, L.S2, 1};
  const int id[3] = {i, j, k};
#pragma unroll
  for (int f = 0; f < 3; f++) {
    const int d = (f + 1) % 3, e = (f + 2) % 3;
    if (id[f] >= L.n[f]) continue;
    double E = 0.0;
    if (!(f != 1 && pole))
      // X = E_f on d-faces: f = d + 2 -> EfB[d];  Y = E_f on e-faces: f = e + 1 -> EfA[e]
      E = edge_emf(Dv.EfB[d], Dv.EfA[e], Dv.Cc[f], Dv.F[d][0], Dv.F[e][0], z, S[d], S[e]);
    Dv.Ee[f][z] = E;
  }
}

// centre EMFs of the stage source (C-8); launch_flux_on may have issued this beside the flux sweeps (g->cemf_done)
void launch_centre_emf_on(hamr_grid* g, const Dev& Dv, const Fields& src, const Fields& src2) {
  const Lay& L = Dv.L;
  const bool blk = Dv.B.nblk > 0;
  if (blk && Dv.B.nact == 0) return;
  const long long mult = blk ? Dv.B.nact : 1;
  const bool wrap = x3_ghosts_unused(Dv);
  const long long tot = (long long)(L.n[0] + 2) * (L.n[1] + 2) * (L.n[2] + (wrap ? 0 : 2)) * mult;
  Launch l_(g, K_CEMF);
  if (blk) k_centre_emf<true, false><<<(unsigned)((tot + 127) / 128), 128, 0, g->stream>>>(Dv, src, src2);
  else if (wrap) k_centre_emf<false, true><<<(unsigned)((tot + 127) / 128), 128, 0, g->stream>>>(Dv, src, src2);
  else k_centre_emf<false, false><<<(unsigned)((tot + 127) / 128), 128, 0, g->stream>>>(Dv, src, src2);
}

void launch_ct_on(hamr_grid* g, const Dev& Dv, const Fields& src, const Fields& src2) {
  const Lay& L = Dv.L;
  const bool blk = Dv.B.nblk > 0;
  if (blk && Dv.B.nact == 0) return;
  const long long mult = blk ? Dv.B.nact : 1;
  if (g->cemf_done) g->cemf_done = false;   // issued with the flux sweeps of the same source
  else launch_centre_emf_on(g, Dv, src, src2);
  const long long tot = (long long)(L.n[0] + 1) * (L.n[1] + 1) * (L.n[2] + 1) * mult;
  Launch l_(g, K_EDGE);
  if (blk) k_edge_emf<true><<<(unsigned)((tot + 127) / 128), 128, 0, g->stream>>>(Dv);
  else k_edge_emf<false><<<(unsigned)((tot + 127) / 128), 128, 0, g->stream>>>(Dv);
}

void launch_ct(hamr_grid* g, const Fields& src) { launch_ct_on(g, g->D, src, src); }

}  // namespace hamr
