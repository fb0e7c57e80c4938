// deref.cu — phi-derefinement of the polar rows ("internal SMR"; DESIGN.md §9 C-15).
// near the poles the grid is derefined in phi; the code "averages the fluxes and conserved
// quantities ... over 2^n cells" and adapts the reconstruction to the larger cell spacing.
//
// Reading (C-15): a row with factor m treats every aligned group of m phi-zones as one zone, but all
// arrays stay on the FINE grid.  After the flux kernels the face values of derefined rows are given the
// group structure (x1-/x2-face values -> group mean; x3-face values between group boundaries -> linear
// interpolation of the boundary faces, which flux.cu: k_deref_x3 computes with a strided stencil), after
// the edge-EMF kernel likewise (E3 -> group mean, E1 / E2 between group-boundary edges -> interpolation).
// Every fine face and fine edge then carries ONE value, so the unchanged update conserves and the
// unchanged CT keeps div B per fine zone; the hydro state of a group is that of its first member.
// An x2-face (and its edges) between two rows uses the coarser of the two rows' groupings.
//
// All of this touches ~17 % of the rows of BASELINE cfg 4 and is HBM-bound streaming work; one thread
// owns one group of one (i, j) column, so no two threads touch the same value.
#include "hamr_host.h"

namespace hamr {

// C-15: factor of global x2 row J by the polar angle of its zone centre (degrees; on the Cartesian map the
// x2 extent stands for (0, 180)): the largest factor whose threshold the row lies inside.  Rows beyond a
// pole take their mirror row's factor, rows beyond a periodic x2 boundary their image's.
int deref_row_factor(const hamr_params& p, long long J) {
  if (p.n_deref <= 0) return 1;
  const long long N2 = p.n[1];
  if (p.bc_lo[1] == HAMR_BC_PERIODIC) J = ((J % N2) + N2) % N2;
  if (J < 0) J = -J - 1;
  if (J >= N2) J = 2 * N2 - 1 - J;
  if (J < 0 || J >= N2) return 1;
  const double th = ((double)J + 0.5) / (double)N2 * 180.0;
  int m = 1;
  for (int t = 0; t < p.n_deref && t < 4; t++)
    if ((th < p.deref_theta_deg[t] || th > 180.0 - p.deref_theta_deg[t]) && p.deref_factor[t] > m) m = p.deref_factor[t];
  return m;
}

// thread -> (block, i, j, k) over i in [ilo, n1 + ihi), j in [jlo, n2 + jhi), k in [0, n3)
struct DIdx { int i, j, k; bool valid; BCtx C; };
template <bool BLK>
__device__ __forceinline__ DIdx deref_idx(const Dev& Dv, int ilo, int ihi, int jlo, int jhi) {
  const Lay& L = Dv.L;
  const int ci = L.n[0] + ihi - ilo, cj = L.n[1] + jhi - jlo, ck = L.n[2];
  const unsigned per = (unsigned)ci * cj * ck;
  unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  DIdx r;
  r.valid = t < (BLK ? per * Dv.B.nact : per);
  if (!r.valid) t = 0;
  int bslot = 0;
  if (BLK) { bslot = (int)(t / per); t -= bslot * per; }
  r.C = blk_ctx<BLK>(Dv, bslot);
  const unsigned tj = t / (unsigned)ck, ti = tj / (unsigned)cj;
  r.k = (int)(t - tj * ck);
  r.j = (int)(tj - ti * cj) + jlo;
  r.i = (int)ti + ilo;
  return r;
}

// group mean in place (members z0 .. z0 + m - 1, m a power of two <= 16) by a pairwise (tree) sum: the mean of
// m IDENTICAL values is then that value exactly, so quantities that are already uniform in the group are left
// bit-for-bit alone and blocks that recompute a shared value from copies of each other's groups agree
template <int M>
__device__ __forceinline__ void group_mean_t(double* __restrict__ a) {
  double v[M];   // registers: M is a compile-time constant
#pragma unroll
  for (int r = 0; r < M; r++) v[r] = a[r];
#pragma unroll
  for (int w = 1; w < M; w *= 2)
#pragma unroll
    for (int r = 0; r + w < M; r += 2 * w) v[r] = v[r] + v[r + w];
  const double mean = v[0] / (double)M;
#pragma unroll
  for (int r = 0; r < M; r++) a[r] = mean;
}
__device__ __forceinline__ void group_mean(double* __restrict__ a, long long zrow, int k0, int m) {
  double* g = a + zrow + k0;
  if (m == 2) group_mean_t<2>(g);
  else if (m == 4) group_mean_t<4>(g);
  else if (m == 8) group_mean_t<8>(g);
  else group_mean_t<16>(g);
}

// members 1 .. m-1 become the linear interpolation of the values at k0 and k0 + m
__device__ __forceinline__ void group_interp(double* __restrict__ a, long long zrow, int k0, int m) {
  const double lo = a[zrow + k0], hi = a[zrow + k0 + m];
  for (int r = 1; r < m; r++) a[zrow + k0 + r] = lo + ((double)r / (double)m) * (hi - lo);
}

// C-15 (iii): after the three flux kernels
template <bool BLK>
__global__ void __launch_bounds__(128) k_deref_fix_flux(Dev Dv) {
  const Lay& L = Dv.L;
  const DIdx T = deref_idx<BLK>(Dv, -1, 1, -1, 1);   // i, j in [-1, n]: the transverse ghost layer included
  if (!T.valid) return;
  const int i = T.i, j = T.j, k = T.k, n3 = L.n[2];
  const int m = __ldg(Dv.mrow + T.C.J0 + j + NG);
  const int M = max(m, __ldg(Dv.mrow + T.C.J0 + j - 1 + NG));   // x2-face j lies between rows j-1 and j
  const long long zrow = T.C.zoff + L.idx(i, j, 0);
  // blockIdx.y: the quantity (five hydro fluxes, the two transverse face EMFs): seven independent threads per
  // group instead of one thread walking 21 read-modify-write chains one after the other
  const int c = blockIdx.y;   // 7 (C-18): the entropy flux, one more flux of the row
  double* const a0 = c < 5 ? Dv.F[0][c] : (c == 5 ? Dv.EfA[0] : (c == 6 ? Dv.EfB[0] : Dv.FK[0]));
  double* const a1 = c < 5 ? Dv.F[1][c] : (c == 5 ? Dv.EfA[1] : (c == 6 ? Dv.EfB[1] : Dv.FK[1]));
  double* const a2 = c < 5 ? Dv.F[2][c] : (c == 5 ? Dv.EfA[2] : (c == 6 ? Dv.EfB[2] : Dv.FK[2]));
  if (m > 1 && k % m == 0) {
    if (i >= 0) group_mean(a0, zrow, k, m);                 // x1-faces of the row
    group_interp(a2, zrow, k, m);                           // x3-faces inside the group
  }
  if (j >= 0 && M > 1 && k % M == 0) group_mean(a1, zrow, k, M);   // x2-face on the low side of row j
}

// C-15 (iv): after the edge-EMF kernel
template <bool BLK>
__global__ void __launch_bounds__(128) k_deref_fix_edges(Dev Dv) {
  const Lay& L = Dv.L;
  const DIdx T = deref_idx<BLK>(Dv, 0, 1, 0, 1);     // i in [0, n1], j in [0, n2]
  if (!T.valid) return;
  const int i = T.i, j = T.j, k = T.k, n3 = L.n[2];
  const int m = __ldg(Dv.mrow + T.C.J0 + j + NG);
  const int M = max(m, __ldg(Dv.mrow + T.C.J0 + j - 1 + NG));
  const long long zrow = T.C.zoff + L.idx(i, j, 0);
  if (M > 1 && k % M == 0) {
    group_mean(Dv.Ee[2], zrow, k, M);                            // E3 at (i-1/2, j-1/2, k)
    if (i < L.n[0]) group_interp(Dv.Ee[0], zrow, k, M);          // E1 at (i, j-1/2, k-1/2)
  }
  if (m > 1 && k % m == 0 && j < L.n[1]) group_interp(Dv.Ee[1], zrow, k, m);   // E2 at (i-1/2, j, k-1/2)
}

// C-15 (v) and (i): one inversion per group, and the whole invariant re-imposed EXACTLY after every update: the
// first member's primitives and B_c are the group's; Bf1 (row grouping) and Bf2 (the grouping of its face)
// likewise; Bf3 on in-group faces is re-interpolated from the group's outer faces.  The update leaves these true
// to round-off only; exactness keeps blocks that cut x3 bit-for-bit consistent on the faces they share and
// costs div B nothing beyond round-off that does not accumulate.
template <bool BLK>
__global__ void __launch_bounds__(128) k_deref_sync(Dev Dv, Fields o0, Fields o2) {
  const Lay& L = Dv.L;
  const DIdx T = deref_idx<BLK>(Dv, 0, 1, 0, 1);     // i in [0, n1], j in [0, n2]: the high faces included
  if (!T.valid) return;
  const int i = T.i, j = T.j, k = T.k;
  const int m = __ldg(Dv.mrow + T.C.J0 + j + NG);
  const int M = max(m, __ldg(Dv.mrow + T.C.J0 + j - 1 + NG));
  const long long z = T.C.zoff + L.idx(i, j, k);
  const int r = k % m, R = k % M;
  if (m > 1 && r != 0 && j < L.n[1]) {
    { double* a = selp<BLK>(o0.Bf[0], o2.Bf[0], T.C.cur); a[z] = a[z - r]; }
    if (i < L.n[0]) {
#pragma unroll
      for (int c = 0; c < 5; c++) { double* a = selp<BLK>(o0.P[c], o2.P[c], T.C.cur); a[z] = a[z - r]; }
#pragma unroll
      for (int c = 0; c < 3; c++) { double* a = selp<BLK>(o0.Bc[c], o2.Bc[c], T.C.cur); a[z] = a[z - r]; }
      double* a = selp<BLK>(o0.Bf[2], o2.Bf[2], T.C.cur);
      const double lo = a[z - r], hi = a[z - r + m];
      a[z] = lo + ((double)r / (double)m) * (hi - lo);
    }
  }
  if (M > 1 && R != 0 && i < L.n[0]) { double* a = selp<BLK>(o0.Bf[1], o2.Bf[1], T.C.cur); a[z] = a[z - R]; }
}

// C-15 (iii): the x1- and x2-face values of derefined rows in the transverse phi-ghost layer (k = -1, k = n3; they
// feed the edge EMFs of C-9 on the phi-boundary) are the phi-NEIGHBOUR's group means, not this block's own
// per-zone values: where rows with different factors meet, the mean changes the value.  Same-level neighbours
// only (across time levels the LAT correction makes shared edges agree); a monolithic grid wraps onto itself.
template <bool BLK>
__global__ void __launch_bounds__(128) k_deref_flux_layers(Dev Dv) {
  const Lay& L = Dv.L;
  const int c1 = L.n[1] + 1;
  const unsigned per = 2u * (L.n[0] + 1) * c1;
  unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (BLK ? per * Dv.B.nact : per)) return;
  int bslot = 0;
  if (BLK) { bslot = (int)(t / per); t -= bslot * per; }
  const BCtx C = blk_ctx<BLK>(Dv, bslot);
  const int side = (int)(t & 1);
  t >>= 1;
  const int j = (int)(t % (unsigned)c1), i = (int)(t / (unsigned)c1), n3 = L.n[2];
  const int m = __ldg(Dv.mrow + C.J0 + j + NG);
  const int M = max(m, __ldg(Dv.mrow + C.J0 + j - 1 + NG));
  if (M == 1) return;
  int q = C.b;
  if (BLK) {
    q = __ldg(Dv.B.nbr + C.b * NNBR + 12 + (side ? 2 : 0));       // offset (0, 0, -1) / (0, 0, +1)
    if (q < 0 || Dv.B.tau[q] != Dv.B.tau[C.b] || Dv.B.info[q].y != C.lev) return;
  }
  const long long zd = C.zoff + L.idx(i, j, side ? n3 : -1);
  const long long zs = (BLK ? (long long)q * Dv.B.blen : 0) + L.idx(i, j, side ? 0 : n3 - 1);
  if (m > 1 && j < L.n[1]) {
#pragma unroll
    for (int c = 0; c < 5; c++) Dv.F[0][c][zd] = Dv.F[0][c][zs];
    Dv.EfA[0][zd] = Dv.EfA[0][zs];
    Dv.EfB[0][zd] = Dv.EfB[0][zs];
  }
  if (i < L.n[0]) {
#pragma unroll
    for (int c = 0; c < 5; c++) Dv.F[1][c][zd] = Dv.F[1][c][zs];
    Dv.EfA[1][zd] = Dv.EfA[1][zs];
    Dv.EfB[1][zd] = Dv.EfB[1][zs];
  }
}

// C-15 (i): puts an initial state onto the invariant: hydro primitives -> group mean, x3-face field between
// group boundaries -> interpolation.  Bf1, Bf2 are expected to be group-uniform (any axisymmetric field is).
template <bool BLK>
__global__ void __launch_bounds__(128) k_deref_project(Dev Dv, Fields s0, Fields s2) {
  const Lay& L = Dv.L;
  const DIdx T = deref_idx<BLK>(Dv, 0, 0, 0, 0);
  if (!T.valid) return;
  const int m = __ldg(Dv.mrow + T.C.J0 + T.j + NG);
  if (m == 1 || T.k % m != 0) return;
  const long long zrow = T.C.zoff + L.idx(T.i, T.j, 0);
#pragma unroll
  for (int c = 0; c < 5; c++) group_mean(selp<BLK>(s0.P[c], s2.P[c], T.C.cur), zrow, T.k, m);
  group_interp(selp<BLK>(s0.Bf[2], s2.Bf[2], T.C.cur), zrow, T.k, m);
}

// the launch of a C-15 kernel: on a block grid only the listed blocks that hold derefined rows
static Dev deref_dev(const Dev& Dv) {
  Dev D = Dv;
  if (Dv.B.nblk > 0 && Dv.B.dlist) { D.B.list = Dv.B.dlist; D.B.nact = Dv.B.ndact; }
  return D;
}

static unsigned nblocks_for(const Dev& Dv, int ci, int cj) {
  const long long tot = (long long)ci * cj * Dv.L.n[2] * (Dv.B.nblk > 0 ? Dv.B.nact : 1);
  return (unsigned)((tot + 127) / 128);
}

void launch_deref_fix_flux(hamr_grid* g, const Dev& Dv0) {
  const Dev Dv = deref_dev(Dv0);
  if (!Dv.mrow || (Dv.B.nblk > 0 && Dv.B.nact == 0)) return;
  Launch l_(g, K_OTHER);
  const unsigned nb = nblocks_for(Dv, Dv.L.n[0] + 2, Dv.L.n[1] + 2);
  const unsigned nq = Dv.entropy ? 8 : 7;
  if (Dv.B.nblk > 0) k_deref_fix_flux<true><<<dim3(nb, nq), 128, 0, g->stream>>>(Dv);
  else k_deref_fix_flux<false><<<dim3(nb, nq), 128, 0, g->stream>>>(Dv);
}

void launch_deref_flux_layers(hamr_grid* g, const Dev& Dv0) {
  const Dev Dv = deref_dev(Dv0);
  if (!Dv.mrow || (Dv.B.nblk > 0 && Dv.B.nact == 0)) return;
  Launch l_(g, K_OTHER);
  const long long tot = 2LL * (Dv.L.n[0] + 1) * (Dv.L.n[1] + 1) * (Dv.B.nblk > 0 ? Dv.B.nact : 1);
  const unsigned nb = (unsigned)((tot + 127) / 128);
  if (Dv.B.nblk > 0) k_deref_flux_layers<true><<<nb, 128, 0, g->stream>>>(Dv);
  else k_deref_flux_layers<false><<<nb, 128, 0, g->stream>>>(Dv);
}

void launch_deref_fix_edges(hamr_grid* g, const Dev& Dv0) {
  const Dev Dv = deref_dev(Dv0);
  if (!Dv.mrow || (Dv.B.nblk > 0 && Dv.B.nact == 0)) return;
  Launch l_(g, K_OTHER);
  const unsigned nb = nblocks_for(Dv, Dv.L.n[0] + 1, Dv.L.n[1] + 1);
  if (Dv.B.nblk > 0) k_deref_fix_edges<true><<<nb, 128, 0, g->stream>>>(Dv);
  else k_deref_fix_edges<false><<<nb, 128, 0, g->stream>>>(Dv);
}

void launch_deref_sync(hamr_grid* g, const Dev& Dv0, const Fields& out, const Fields& out2) {
  const Dev Dv = deref_dev(Dv0);
  if (!Dv.mrow || (Dv.B.nblk > 0 && Dv.B.nact == 0)) return;
  Launch l_(g, K_OTHER);
  const unsigned nb = nblocks_for(Dv, Dv.L.n[0] + 1, Dv.L.n[1] + 1);
  if (Dv.B.nblk > 0) k_deref_sync<true><<<nb, 128, 0, g->stream>>>(Dv, out, out2);
  else k_deref_sync<false><<<nb, 128, 0, g->stream>>>(Dv, out, out2);
}

void launch_deref_project(hamr_grid* g, const Dev& Dv0, const Fields& s, const Fields& s2) {
  const Dev Dv = deref_dev(Dv0);
  if (!Dv.mrow || (Dv.B.nblk > 0 && Dv.B.nact == 0)) return;
  Launch l_(g, K_OTHER);
  const unsigned nb = nblocks_for(Dv, Dv.L.n[0], Dv.L.n[1]);
  if (Dv.B.nblk > 0) k_deref_project<true><<<nb, 128, 0, g->stream>>>(Dv, s, s2);
  else k_deref_project<false><<<nb, 128, 0, g->stream>>>(Dv, s, s2);
}

}  // namespace hamr
