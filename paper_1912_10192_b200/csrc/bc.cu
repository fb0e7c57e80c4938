// bc.cu — physical boundary fill (C-12) and cell-centred B in ghosts (C-10).
// Boundaries (BASELINE.json cfg 0; PAPER.md:79 discusses the polar boundary): outflow copies the
// nearest active zone / boundary face, polar reflect mirrors about the axis with ut^2, Bf^2
// changing sign, periodic wraps.  The fill order x1, x2, x3 of the definition (edge and corner
// ghosts take values already filled along earlier dimensions) is reproduced in ONE launch by
// composing the three index maps: every ghost value is a signed copy of one active value.
#include "hamr_host.h"

namespace hamr {

__device__ __forceinline__ int pmod(int g, int n) {
  int r = g % n;
  return r < 0 ? r + n : r;
}

// source index along one dimension for padded index g; `stag`: the array is a face array along
// this dimension (active faces 0..n) else zone-centred (active 0..n-1).  flip is set when the
// value comes from a reflection.
__device__ __forceinline__ int map_idx(int g, int n, int bc_lo, int bc_hi, bool stag, bool& flip) {
  const int hi = stag ? n : n - 1;
  if (g >= 0 && g <= hi) return g;
  if (g < 0) {
    const int m = -g;
    if (bc_lo == HAMR_BC_PERIODIC) return pmod(g, n);
    if (bc_lo == HAMR_BC_OUTFLOW) return 0;
    flip = true;
    return stag ? m : m - 1;
  }
  const int m = g - hi;
  if (bc_hi == HAMR_BC_PERIODIC) return stag ? ((m % n == 0) ? n : m % n) : g % n;
  if (bc_hi == HAMR_BC_OUTFLOW) return hi;
  flip = true;
  return n - m;
}

// value of array `a` (vector component vc = -1 scalar / 0..2; face array along sd = -1 / 0..2) at
// any padded location, as the fill would leave it.  pa: on an x1 slab (NEXT-4) the array's slot in the neighbour
// tables (buffer set * 11 + array), -1 otherwise: beyond a side that has a neighbour slab the value is the neighbour's
// active value (ghost zones of a block on another GPU are fetched over NVLink), the x2 / x3 maps
// composed with it as with any other x1 rule.
__device__ __forceinline__ double ghost_value(const Dev& D, const double* __restrict__ a, int vc, int sd,
                                              int i, int j, int k, int pa = -1) {
  const Lay& L = D.L;
  bool f0 = false, f1 = false, f2 = false;
  int si;
  const bool own = !(D.peer && pa >= 0 && ((i < 0 && D.peer->on[0]) || (i > (sd == 0 ? L.n[0] : L.n[0] - 1) && D.peer->on[1])));
  if (own) {
    si = map_idx(i, L.n[0], D.bc_lo[0], D.bc_hi[0], sd == 0, f0);
  } else if (i < 0) {       // the neighbour's face n1' is this slab's face 0: faces and zones shift alike
    si = i + D.peer->n1[0];
    a = D.peer->a[0][pa];
  } else {
    si = i - L.n[0];
    a = D.peer->a[1][pa];
  }
  const int sj = map_idx(j, L.n[1], D.bc_lo[1], D.bc_hi[1], sd == 1, f1);
  int sk = map_idx(k, L.n[2], D.bc_lo[2], D.bc_hi[2], sd == 2, f2);
  if (D.mrow && D.bc_lo[2] == HAMR_BC_PERIODIC && (k < 0 || k > (sd == 2 ? L.n[2] : L.n[2] - 1))) {
    // C-15: the phi-ghost slots of a derefined row hold whole groups; an x2-face array follows its face's grouping
    const int mj = __ldg(D.mrow + j + NG);
    const int mg = sd == 1 ? max(mj, __ldg(D.mrow + max(j - 1, -NG) + NG)) : mj;
    if (mg > 1) sk = deref_ghost_k(k, L.n[2], mg);
  }
  // NEXT-1 transmissive pole: the zone beyond the pole is the mirror row's zone half a turn away
  if (f1 && D.bc_lo[1] == HAMR_BC_POLAR_TRANSMIT) sk = (sk % L.n[2] + L.n[2] / 2) % L.n[2];
  double v = a[L.idx(si, sj, sk)];
  // a reflecting wall carries no normal flux: the wall face itself is 0
  if (own && sd == 0 && ((si == 0 && D.bc_lo[0] >= HAMR_BC_POLAR_REFLECT) || (si == L.n[0] && D.bc_hi[0] >= HAMR_BC_POLAR_REFLECT))) v = 0.0;
  if (sd == 1 && ((sj == 0 && D.bc_lo[1] >= HAMR_BC_POLAR_REFLECT) || (sj == L.n[1] && D.bc_hi[1] >= HAMR_BC_POLAR_REFLECT))) v = 0.0;
  if (sd == 2 && ((sk == 0 && D.bc_lo[2] >= HAMR_BC_POLAR_REFLECT) || (sk == L.n[2] && D.bc_hi[2] >= HAMR_BC_POLAR_REFLECT))) v = 0.0;
  const bool neg = (vc == 0 && f0) || (vc == 1 && f1) || (vc == 2 && f2);
  return neg ? -v : v;
}

// One padded location (i,j,k).  Writes ghost P, ghost Bf and Bc of ghost zones (of all zones if `all`
// is set: used once for the initial state).
// pq: 11 * (the buffer set s is) on an x1 slab, negative otherwise
__device__ __forceinline__ void ghost_cell(const Dev& D, const Fields& s, int all, int i, int j, int k, int pq) {
  const Lay& L = D.L;
  const int id[3] = {i, j, k};
  bool in_c[3], extra[3];
  for (int d = 0; d < 3; d++) {
    in_c[d] = id[d] >= 0 && id[d] < L.n[d];
    extra[d] = id[d] == L.n[d] + NG;
  }
  const bool zone_active = in_c[0] && in_c[1] && in_c[2];
  const bool zone_slot = !(extra[0] || extra[1] || extra[2]);
  if (zone_active && !all) {
    // interior: only wall faces of reflecting boundaries need attention
    for (int d = 0; d < 3; d++)
      if (id[d] == 0 && D.bc_lo[d] >= HAMR_BC_POLAR_REFLECT) s.Bf[d][L.idx(i, j, k)] = 0.0;
    return;
  }
  const long long z = L.idx(i, j, k);
  if (zone_slot && !zone_active) {
    for (int c = 0; c < 5; c++) s.P[c][z] = ghost_value(D, s.P[c], c - 2, -1, i, j, k, pq + c);
  }
  double lo[3], hi[3];
  for (int d = 0; d < 3; d++) {
    // face array along d: valid slot if the transverse indices are zone slots
    const int o1 = (d + 1) % 3, o2 = (d + 2) % 3;
    if (extra[o1] || extra[o2]) { lo[d] = hi[d] = 0.0; continue; }
    lo[d] = ghost_value(D, s.Bf[d], d, d, i, j, k, pq + 8 + d);
    const bool face_active = in_c[o1] && in_c[o2] && id[d] >= 0 && id[d] <= L.n[d];
    const bool wall = face_active && ((id[d] == 0 && D.bc_lo[d] >= HAMR_BC_POLAR_REFLECT) ||
                                      (id[d] == L.n[d] && D.bc_hi[d] >= HAMR_BC_POLAR_REFLECT));
    if (!face_active || wall) s.Bf[d][z] = lo[d];  // ghost_value returns 0 on a reflecting wall
    if (!extra[d]) hi[d] = ghost_value(D, s.Bf[d], d, d, i + (d == 0), j + (d == 1), k + (d == 2), pq + 8 + d);
  }
  if (zone_slot && pq >= 0 && in_c[1] && in_c[2] && ((i < 0 && D.peer->on[0]) || (i >= L.n[0] && D.peer->on[1]))) {
    // NEXT-4: this ghost zone IS an active zone of the neighbour slab, whose B_c came out of its update kernel (a
    // product with the stored 1 / sqrt(-g), not the division below): take that value, as the one-grid run would
    for (int d = 0; d < 3; d++) s.Bc[d][z] = ghost_value(D, s.Bc[d], -1, -1, i, j, k, pq + 5 + d);
    return;
  }
  if (zone_slot) {
    const double g = __ldg(D.gcA + (size_t)L.idx2(i, j) * NREC_C + CREC_GDET);
    if (D.mrow) {
      const int m = __ldg(D.mrow + j + NG), n3 = L.n[2];
      if (k >= 0 && k < n3) {
        if (m > 1) {   // C-15: B_c^3 of a phi-derefined row is the group's value, from the group's two outer x3-faces
          const int k0 = k - k % m;
          lo[2] = ghost_value(D, s.Bf[2], 2, 2, i, j, k0, pq + 10);
          hi[2] = ghost_value(D, s.Bf[2], 2, 2, i, j, k0 + m, pq + 10);
        }
      } else {
        // a phi-ghost slot holds a whole group of THIS row; its two x2-faces are stored in their faces' groupings
        const int Mlo = max(m, __ldg(D.mrow + max(j - 1, -NG) + NG)), Mhi = max(m, __ldg(D.mrow + min(j + 1, L.n[1] + NG) + NG));
        if (Mlo != m) lo[1] = ghost_value(D, s.Bf[1], 1, 1, i, j, deref_face2_slot(k, n3, m, Mlo), pq + 9);
        if (Mhi != m) hi[1] = ghost_value(D, s.Bf[1], 1, 1, i, j + 1, deref_face2_slot(k, n3, m, Mhi), pq + 9);
      }
    }
    for (int d = 0; d < 3; d++) s.Bc[d][z] = (lo[d] + hi[d]) / (2.0 * g);
  }
}

// every padded location (initial state; grids with a reflecting x1 or x3 wall)
__global__ void __launch_bounds__(256) k_ghosts(Dev D, Fields s, int all, int pq) {
  const Lay& L = D.L;
  const int e3 = L.n[2] + 2 * NG + 1;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long tot = (long long)L.e1 * L.e2 * e3;
  if (t >= tot) return;
  ghost_cell(D, s, all, (int)(t / ((long long)e3 * L.e2)) - NG, (int)((t / e3) % L.e2) - NG, (int)(t % e3) - NG, pq);
}

// The ghost shell only (the per-stage fill; ~12 % of the padded grid for cfg 2):
//  part A: (i,j) columns with i or j outside the active range (plus the j = 0 wall row of a reflecting
//          axis): every k;   part B: active (i,j) columns: the 2 NG + 1 ghost slots in k.
// nox3: the stage kernels of this grid never read x3 ghost zones (x3_ghosts_unused, flux.cu): part A covers
// k in [0, n3) only and there is no part B.
__global__ void __launch_bounds__(256) k_ghosts_shell(Dev D, Fields s, int nj, long long nA_, int nox3, int pq) {
  const Lay& L = D.L;
  // 32-bit index arithmetic (an array holds < 2^31 doubles, checked at creation): 64-bit division is emulated
  const unsigned e3 = nox3 ? L.n[2] : L.n[2] + 2 * NG + 1;
  const unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned nA = (unsigned)nA_;
  if (t < nA) {
    unsigned row = t / e3;
    const int k = (int)(t - row * e3) - (nox3 ? 0 : NG);
    int i, j;
    const unsigned e2 = L.e2, lo_rows = NG * e2, mid_rows = (unsigned)L.n[0] * nj;
    if (row < lo_rows) {
      const unsigned a = row / e2;
      i = (int)a - NG; j = (int)(row - a * e2) - NG;
    } else if (row < lo_rows + mid_rows) {
      row -= lo_rows;
      const unsigned a = row / (unsigned)nj;
      i = (int)a;
      const int q = (int)(row - a * nj);  // -3, -2, -1, [0,] n2 .. n2 + 3
      j = q < NG ? q - NG : (nj == 2 * NG + 2 ? (q == NG ? 0 : L.n[1] + q - NG - 1) : L.n[1] + q - NG);
    } else {
      row -= lo_rows + mid_rows;
      const unsigned a = row / e2;
      i = L.n[0] + (int)a; j = (int)(row - a * e2) - NG;
    }
    ghost_cell(D, s, 0, i, j, k, pq);
    return;
  }
  if (nox3) return;
  const unsigned u = t - nA;
  const unsigned nB = (unsigned)L.n[0] * L.n[1] * 8;
  if (u >= nB) return;
  const int q = (int)(u & 7);
  if (q == 7) return;
  const unsigned col = u >> 3;
  const int i = (int)(col / (unsigned)L.n[1]), j = (int)(col - (unsigned)i * L.n[1]);
  if (nj == 2 * NG + 2 && j == 0) return;  // the wall row was done in part A
  const int n3 = L.n[2];
  const int k = q < NG ? q - NG : n3 + q - NG;
  // periodic x3 on a row that is not derefined and touches no reflecting wall face: the slots are plain
  // copies of the image zone; same values and the same B_c arithmetic as ghost_cell
  const bool fast = D.bc_lo[2] == HAMR_BC_PERIODIC && !D.mrow && n3 > NG &&
                    !(j + 1 == L.n[1] && D.bc_hi[1] >= HAMR_BC_POLAR_REFLECT) &&
                    !(i + 1 == L.n[0] && D.bc_hi[0] >= HAMR_BC_POLAR_REFLECT);
  if (!fast) { ghost_cell(D, s, 0, i, j, k, pq); return; }
  if (q == 6) { s.Bf[2][L.idx(i, j, k)] = s.Bf[2][L.idx(i, j, NG)]; return; }
  const int ks = k < 0 ? k + n3 : k - n3;
  const long long z = L.idx(i, j, k), zs = L.idx(i, j, ks);
#pragma unroll
  for (int c = 0; c < 5; c++) s.P[c][z] = s.P[c][zs];
  const double lo0 = s.Bf[0][zs], hi0 = s.Bf[0][L.idx(i + 1, j, ks)];
  const double lo1 = s.Bf[1][zs], hi1 = s.Bf[1][L.idx(i, j + 1, ks)];
  const int klo = k < 0 ? n3 + k : (k == n3 ? n3 : k - n3);
  const int khi = k == -1 ? 0 : (k < 0 ? n3 + k + 1 : k + 1 - n3);
  const double lo2 = s.Bf[2][L.idx(i, j, klo)], hi2 = s.Bf[2][L.idx(i, j, khi)];
  s.Bf[0][z] = lo0;
  s.Bf[1][z] = lo1;
  if (k != n3) s.Bf[2][z] = lo2;
  const double g2 = 2.0 * __ldg(D.gcA + (size_t)L.idx2(i, j) * NREC_C + CREC_GDET);
  s.Bc[0][z] = (lo0 + hi0) / g2;
  s.Bc[1][z] = (lo1 + hi1) / g2;
  s.Bc[2][z] = (lo2 + hi2) / g2;
}

void launch_ghosts(hamr_grid* g, const Fields& s, bool all) {
  const Lay& L = g->D.L;
  const int e3 = L.n[2] + 2 * NG + 1;
  int pq = -64;   // x1 slab: which of the three buffer sets s is (the neighbours' sets rotate in step with ours)
  if (g->D.peer)
    for (int q = 0; q < 3; q++) if (g->s[q].P[0] == s.P[0]) pq = 11 * q;
  Launch l_(g, K_GHOSTS);
  if (all || g->D.bc_lo[0] >= HAMR_BC_POLAR_REFLECT || g->D.bc_lo[2] >= HAMR_BC_POLAR_REFLECT) {
    const long long tot = (long long)L.e1 * L.e2 * e3;
    k_ghosts<<<(unsigned)((tot + 255) / 256), 256, 0, g->stream>>>(g->D, s, all ? 1 : 0, pq);
    return;
  }
  const int nj = 2 * NG + 1 + (g->D.bc_lo[1] >= HAMR_BC_POLAR_REFLECT ? 1 : 0);
  const long long rows = (long long)(2 * NG + 1) * L.e2 + (long long)L.n[0] * nj;
    const bool nox3 = x3_ghosts_unused(g->D);
  const long long nA = rows * (nox3 ? L.n[2] : e3);
  const long long tot = nA + (nox3 ? 0 : (long long)L.n[0] * L.n[1] * 8);
  k_ghosts_shell<<<(unsigned)((tot + 255) / 256), 256, 0, g->stream>>>(g->D, s, nj, nA, nox3 ? 1 : 0, pq);
}

}  // namespace hamr
