// ORACLE (test infrastructure) — the per-block stage: boundary fill, reconstruct + HLL, CT,
// source + update + inversion, Courant dt.  DESIGN.md §3 C-5..C-14.
#include "orc_grid.hpp"
#include <algorithm>
#include <cstring>

namespace orc {


static const int CYC[3][3] = {{0, 1, 2}, {1, 2, 0}, {2, 0, 1}};  // (d, e, f) cyclic

// C-15: phi-derefinement factor of global x2 row J by its zone-centre polar angle: the largest factor
// whose threshold (degrees from either pole) the row lies inside.  Rows beyond a pole (ghosts) take
// the factor of their mirror image (of their periodic image if x2 is periodic).
int deref_factor_of_row(const Params& par, long long J) {
  if (par.n_deref <= 0) return 1;
  const long long N2 = par.n[1];
  if (par.bc_lo[1] == 0) J = ((J % N2) + N2) % N2;   // periodic x2: the image row
  if (J < 0) J = -J - 1;                              // beyond a pole: the mirror row
  if (J >= N2) J = 2 * N2 - 1 - J;
  if (J < 0 || J >= N2) return 1;
  // polar angle of the zone centre in degrees; on the Cartesian map the x2 extent plays (0, 180)
  const double th = ((double)J + 0.5) / (double)N2 * 180.0;
  int m = 1;
  for (int t = 0; t < par.n_deref && t < 4; t++)
    if (th < par.deref_theta_deg[t] || th > 180.0 - par.deref_theta_deg[t]) m = std::max(m, (int)par.deref_factor[t]);
  return m;
}

void block_init(const Params& par, Block& b) {
  for (int d = 0; d < 3; d++) b.e[d] = b.n[d] + 2 * NG + 1;
  const size_t n2d = (size_t)b.e[0] * b.e[1];
  b.gc.resize(n2d);
  b.gf1.resize(n2d);
  b.gf2.resize(n2d);
  b.conn.assign(n2d * 64, 0.0);
  b.pole2.assign(b.e[1], 0);
  b.mrow.assign(b.e[1], 1);
  for (int j = -NG; j <= b.n[1] + NG; j++) {
    const long long J = b.I0[1] + j;
    if (par.metric == 1 && (J == 0 || J == par.n[1])) b.pole2[j + NG] = 1;
    b.mrow[j + NG] = deref_factor_of_row(par, J);
  }
  for (int i = -NG; i <= b.n[0] + NG; i++)
    for (int j = -NG; j <= b.n[1] + NG; j++) {
      const size_t q = b.idx2(i, j);
      geom_at(par.metric, par.a, b.xc(0, i), b.xc(1, j), b.gc[q]);
      geom_at(par.metric, par.a, b.xf(0, i), b.xc(1, j), b.gf1[q]);
      geom_at(par.metric, par.a, b.xc(0, i), b.xf(1, j), b.gf2[q]);
      if (b.pole2[j + NG]) b.gf2[q].gdet = 0.0;
      double c[4][4][4];
      conn_at(par.metric, par.a, b.xc(0, i), b.xc(1, j), c);
      std::memcpy(&b.conn[q * 64], c, sizeof(c));
    }
  const size_t n = b.size();
  b.sn.alloc(n);
  b.sh.alloc(n);
  b.snew.alloc(n);
  for (int d = 0; d < 3; d++) {
    for (int c = 0; c < 5; c++) b.F[d][c].assign(n, 0.0);
    if (par.entropy_backup) b.FK[d].assign(n, 0.0);
    for (int c = 0; c < 3; c++) b.Ef[d][c].assign(n, 0.0);
    b.Ee[d].assign(n, 0.0);
    b.Cc[d].assign(n, 0.0);
    b.ctop[d] = 0.0;
  }
}

// ---- physical boundaries (C-12) -------------------------------------------------------------------
// kind: 0 centred along d, 1 staggered along d (a d-face array); sgn: reflection sign
static void fill_dim(const Block& b, std::vector<double>& a, int d, int bc_lo, int bc_hi,
                     bool do_lo, bool do_hi, bool stag, double sgn) {
  const int n = b.n[d];
  const int str[3] = {b.e[1] * b.e[2], b.e[2], 1};
  const int o1 = (d + 1) % 3, o2 = (d + 2) % 3;
  for (int p = 0; p < b.e[o1]; p++)
    for (int q = 0; q < b.e[o2]; q++) {
      double* base = a.data() + (size_t)p * str[o1] + (size_t)q * str[o2] + (size_t)NG * str[d];
      auto at = [&](int i) -> double& { return base[(ptrdiff_t)i * str[d]]; };
      for (int m = 1; m <= NG; m++) {
        if (do_lo) {
          const int g = -m;
          if (bc_lo == 0) at(g) = at(((g % n) + n) % n);
          else if (bc_lo == 1) at(g) = at(0);
          else at(g) = sgn * (stag ? at(m) : at(m - 1));
        }
        if (do_hi) {
          const int g = stag ? n + m : n - 1 + m;
          if (bc_hi == 0) at(g) = stag ? at(m % n == 0 ? n : m % n) : at((g % n + n) % n);
          else if (bc_hi == 1) at(g) = stag ? at(n) : at(n - 1);
          else at(g) = sgn * (stag ? at(n - m) : at(n - m));
        }
      }
      if (stag) {  // a reflecting wall carries no normal flux: the wall face itself is 0
        if (do_lo && bc_lo == 2) at(0) = 0.0;
        if (do_hi && bc_hi == 2) at(n) = 0.0;
      }
    }
}

// NEXT-1 transmissive pole: the zone beyond the pole at (theta_ghost = -theta', phi) IS the zone
// at (theta', phi + pi).  Along the extended meridian the theta basis vector reverses, the r and phi ones do
// not, so the ghost takes the mirror row's value half a turn away, with the x2 components (ut^2, Bf^2)
// changing sign; Bf^2 on the pole face is 0 (zero area).  Needs an even N3, a periodic x3 of extent 2 pi and
// a block that spans x3.  stag2 / stag3: the array is staggered along x2 / x3.
static void fill_polar_transmit(const Block& b, std::vector<double>& a, bool do_lo, bool do_hi, bool stag2,
                                bool stag3, double sgn) {
  const int n2 = b.n[1], n3 = b.n[2], half = n3 / 2;
  for (int i = -NG; i < b.n[0] + NG + 1; i++)
    for (int g = 1; g <= NG; g++)
      for (int side = 0; side < 2; side++) {
        if (!(side ? do_hi : do_lo)) continue;
        const int jg = side ? (stag2 ? n2 + g : n2 - 1 + g) : -g;      // the ghost row (or x2-face)
        const int js = side ? n2 - g : (stag2 ? g : g - 1);            // its mirror image
        // factor of the SOURCE row's x3 grouping: a phi-ghost slot holds a whole group (C-15); an x2-face
        // array follows the grouping of its face (the coarser of its two rows)
        const int m = stag2 ? std::max(b.mrow[js - 1 + NG], b.mrow[js + NG]) : b.mrow[js + NG];
        for (int k = -NG; k < n3 + NG + 1; k++) {
          int o2;
          int kz = deref_ghost_k(k, n3, m, stag3, o2);                // fine x3 index, possibly beyond the block
          kz = ((kz + o2 * n3) % n3 + n3) % n3;                        // periodic: back into the block
          const int ks = (kz + half) % n3;                             // half a turn away; face n3 is face 0
          a[b.idx(i, jg, k)] = sgn * a[b.idx(i, js, ks)];
        }
      }
  if (stag2)
    for (int i = -NG; i < b.n[0] + NG + 1; i++)
      for (int k = -NG; k < n3 + NG + 1; k++) {
        if (do_lo) a[b.idx(i, 0, k)] = 0.0;
        if (do_hi) a[b.idx(i, n2, k)] = 0.0;
      }
}

void fill_physical_bc(const Params& par, Block& b, Fields& s) {
  for (int d = 0; d < 3; d++) {  // order x1, x2, x3 so that edge and corner ghosts are defined
    bool lo = b.phys_lo[d], hi = b.phys_hi[d];
    // a transmissive pole on blocks that cut x3 is closed by the block exchange (orc_blocks.cpp)
    if (d == 1 && (b.xpole_lo || b.xpole_hi)) {
      for (int i = -NG; i < b.n[0] + NG + 1; i++)
        for (int k = -NG; k < b.n[2] + NG + 1; k++) {   // Bf^2 on the pole face is 0 (zero area)
          if (lo && b.xpole_lo) s.Bf[1][b.idx(i, 0, k)] = 0.0;
          if (hi && b.xpole_hi) s.Bf[1][b.idx(i, b.n[1], k)] = 0.0;
        }
      lo = lo && !b.xpole_lo;
      hi = hi && !b.xpole_hi;
    }
    if (!lo && !hi) continue;
    const int bl = par.bc_lo[d], bh = par.bc_hi[d];
    if (d == 1 && (bl == 3 || bh == 3)) {
      // both poles transmissive (a mix with another kind on the other pole is not supported)
      for (int c = 0; c < 5; c++) fill_polar_transmit(b, s.P[c], lo, hi, false, false, c == 3 ? -1.0 : 1.0);
      for (int c = 0; c < 3; c++) fill_polar_transmit(b, s.Bf[c], lo, hi, c == 1, c == 2, c == 1 ? -1.0 : 1.0);
      continue;
    }
    for (int c = 0; c < 5; c++)
      fill_dim(b, s.P[c], d, bl, bh, lo, hi, false, (c == 2 + d) ? -1.0 : 1.0);
    for (int c = 0; c < 3; c++)
      fill_dim(b, s.Bf[c], d, bl, bh, lo, hi, c == d, (c == d) ? -1.0 : 1.0);
  }
}

// C-10: B^d_c = (Bf^d_- + Bf^d_+) / (2 g_c)
void compute_Bc(const Block& b, Fields& s, bool active_only) {
  const int lo = active_only ? 0 : -NG;
  const int str[3] = {b.e[1] * b.e[2], b.e[2], 1};
#pragma omp parallel for collapse(2)
  for (int i = lo; i < b.n[0] - lo; i++)
    for (int j = lo; j < b.n[1] - lo; j++) {
      const double g = b.gc[b.idx2(i, j)].gdet;
      const int m = b.mrow[j + NG], n3 = b.n[2];
      for (int k = lo; k < b.n[2] - lo; k++) {
        const size_t z = b.idx(i, j, k);
        for (int d = 0; d < 3; d++)
          s.Bc[d][z] = (s.Bf[d][z] + s.Bf[d][z + str[d]]) / (2.0 * g);
        if (k < 0 || k >= n3) {
          // a phi-ghost slot holds a whole group of THIS row; the two x2-faces of the zone are stored in the
          // grouping of their own faces
          const int Mlo = std::max(b.mrow[std::max(j - 1, -NG) + NG], m);
          const int Mhi = std::max(m, b.mrow[std::min(j + 1, b.n[1] + NG) + NG]);
          if (Mlo != m || Mhi != m) {
            const double flo = s.Bf[1][b.idx(i, j, deref_face2_slot(k, n3, m, Mlo))];
            const double fhi = s.Bf[1][b.idx(i, j + 1, deref_face2_slot(k, n3, m, Mhi))];
            s.Bc[1][z] = (flo + fhi) / (2.0 * g);
          }
        } else if (m > 1) {
          // C-15 (iii): in a derefined row B_c^3 is the GROUP's value, from the group's two outer x3-faces
          // (a phi-ghost zone holds a whole group and its two ghost faces are that group's outer faces)
          const int k0 = k - k % m;
          s.Bc[2][z] = (s.Bf[2][b.idx(i, j, k0)] + s.Bf[2][b.idx(i, j, k0 + m)]) / (2.0 * g);
        }
      }
    }
}

// ---- reconstruct + HLL on one face (C-5, C-6, C-7) -------------------------------------------------
// face on the low side of zone z along d.  st6[v][0..5]: the six zone values a[j-3 .. j+2] of the
// seven reconstructed variables around the face (j = the zone on the high side).
// C-18: with par.entropy_backup an eighth variable, kappa = (gamma_ad - 1) u / rho^gamma_ad of the zones (b.K, filled
// by flux_pass), is reconstructed like the others and the HLL flux of the entropy row goes to b.FK.
static void face_flux_core(const Params& par, Block& b, const Fields& s, int d, int i, int j, size_t z,
                           const double st6[8][6], double* ctop) {
  const int e = CYC[d][1], f = CYC[d][2];
  const Geom& G = (d == 0) ? b.gf1[b.idx2(i, j)] : (d == 1) ? b.gf2[b.idx2(i, j)] : b.gc[b.idx2(i, j)];
  if (d == 1 && b.pole2[j + NG]) {  // C-7: pole faces carry no flux; no state is evaluated
    for (int c = 0; c < 5; c++) b.F[d][c][z] = 0.0;
    b.Ef[d][e][z] = b.Ef[d][f][z] = 0.0;
    if (par.entropy_backup) b.FK[d][z] = 0.0;
    return;
  }
  double PL[8], PR[8], kL = 0.0, kR = 0.0;
  const int slot[7] = {0, 1, 2, 3, 4, 5 + e, 5 + f};
  for (int v = 0; v < (par.entropy_backup ? 8 : 7); v++) {
    const double* a = st6[v];
    double aL, aR, dummy;
    if (par.recon == 0) {
      ppm_zone(a, dummy, aR);      // left of the face: a_R of zone j-1 from a[j-3 .. j+1]
      ppm_zone(a + 1, aL, dummy);  // right of the face: a_L of zone j from a[j-2 .. j+2]
    } else {
      plm_zone(a + 1, dummy, aR);  // a[j-2 .. j]
      plm_zone(a + 2, aL, dummy);  // a[j-1 .. j+1]
    }
    if (v == 7) { kL = aR; kR = aL; continue; }
    PL[slot[v]] = aR;
    PR[slot[v]] = aL;
  }
  PL[5 + d] = PR[5 + d] = s.Bf[d][z] / G.gdet;  // C-5: normal field is single-valued at the face
  State SL, SR;
  get_state(PL, G, SL);
  get_state(PR, G, SR);
  double UL[8], UR[8], FL[8], FR[8], Fh[8];
  prim_to_U(PL, SL, G, par.gamma_ad, UL);
  prim_to_U(PR, SR, G, par.gamma_ad, UR);
  prim_to_F(PL, SL, G, par.gamma_ad, d + 1, FL);
  prim_to_F(PR, SR, G, par.gamma_ad, d + 1, FR);
  double vminL, vmaxL, vminR, vmaxR;
  wavespeeds(PL, SL, G, par.gamma_ad, d + 1, vminL, vmaxL);
  wavespeeds(PR, SR, G, par.gamma_ad, d + 1, vminR, vmaxR);
  const double cmax = std::max(0.0, std::max(vmaxL, vmaxR));
  const double cmin = std::max(0.0, std::max(-vminL, -vminR));
  hll(UL, UR, FL, FR, cmin, cmax, Fh);
  for (int c = 0; c < 5; c++) b.F[d][c][z] = Fh[c];
  // C-8: on a d-face, E_f = -F^d(B^e), E_e = +F^d(B^f)
  b.Ef[d][f][z] = -Fh[5 + e];
  b.Ef[d][e][z] = Fh[5 + f];
  if (par.entropy_backup) {
    // the entropy row (C-18) through the same HLL formula: U_S = gdet rho kappa u^t, F_S = gdet rho kappa u^d with the
    // reconstructed kappa; gdet rho u^t and gdet rho u^d are row 0 of U and F
    const double USL = UL[0] * kL, USR = UR[0] * kR, FSL = FL[0] * kL, FSR = FR[0] * kR;
    // (slot 1: slot 0 of hll is the mass row with its C-7a flush, which does not apply here)
    double U2L[8] = {0.0, USL}, U2R[8] = {0.0, USR}, F2L[8] = {0.0, FSL}, F2R[8] = {0.0, FSR}, F2[8];
    hll(U2L, U2R, F2L, F2R, cmin, cmax, F2);
    b.FK[d][z] = F2[1];
  }
  if (ctop) *ctop = std::max(cmax, cmin);
}

static void face_flux(const Params& par, Block& b, const Fields& s, int d, int i, int j, int k,
                      double* ctop) {
  const int str[3] = {b.e[1] * b.e[2], b.e[2], 1};
  const size_t z = b.idx(i, j, k);
  const ptrdiff_t sd = str[d];
  const int e = CYC[d][1], f = CYC[d][2];
  const double* var[7] = {s.P[0].data(), s.P[1].data(), s.P[2].data(), s.P[3].data(),
                          s.P[4].data(), s.Bc[e].data(), s.Bc[f].data()};
  double st6[8][6];
  for (int v = 0; v < 7; v++)
    for (int t = 0; t < 6; t++) st6[v][t] = var[v][(ptrdiff_t)z + (t - 3) * sd];
  if (par.entropy_backup)
    for (int t = 0; t < 6; t++) st6[7][t] = b.K[(ptrdiff_t)z + (t - 3) * sd];
  face_flux_core(par, b, s, d, i, j, z, st6, ctop);
}

// C-15 (ii): x3-face on a group boundary of a phi-derefined row (k a multiple of m): the stencil takes
// one value per GROUP, i.e. zones k + t m, t = -3..2; beyond the block the phi-ghost zones hold groups.
static void face_flux_x3_deref(const Params& par, Block& b, const Fields& s, int i, int j, int k, int m,
                               double* ctop) {
  const size_t z = b.idx(i, j, k);
  const int n3 = b.n[2];
  const double* var[7] = {s.P[0].data(), s.P[1].data(), s.P[2].data(), s.P[3].data(),
                          s.P[4].data(), s.Bc[0].data(), s.Bc[1].data()};
  double st6[8][6];
  for (int v = 0; v < 7; v++)
    for (int t = 0; t < 6; t++) {
      int kk = k + (t - 3) * m;                      // first zone of the group, in fine zones
      if (kk < 0) kk = kk / m;                       // groups beyond the low edge: ghost zones -1, -2, -3
      else if (kk >= n3) kk = n3 + (kk - n3) / m;    // beyond the high edge: ghost zones n3, n3 + 1, n3 + 2
      st6[v][t] = var[v][b.idx(i, j, kk)];
      if (v == 0 && par.entropy_backup) st6[7][t] = b.K[b.idx(i, j, kk)];   // C-18: kappa of the same groups
    }
  face_flux_core(par, b, s, 2, i, j, z, st6, ctop);
}

void flux_pass(const Params& par, Block& b, const Fields& src) {
  if (par.entropy_backup) {  // C-18: kappa of every zone of the source state, ghosts included
    b.K.resize(b.size());
    for (size_t z = 0; z < b.size(); z++) b.K[z] = entropy_kappa(src.P[0][z], src.P[1][z], par.gamma_ad);
  }
  for (int d = 0; d < 3; d++) {
    int lo[3] = {-1, -1, -1}, hi[3] = {b.n[0], b.n[1], b.n[2]};  // one transverse ghost layer (CT)
    lo[d] = 0;
    hi[d] = b.n[d];
    double cmaxd = 0.0;
#pragma omp parallel for collapse(2) reduction(max : cmaxd)
    for (int i = lo[0]; i <= hi[0]; i++)
      for (int j = lo[1]; j <= hi[1]; j++)
        for (int k = lo[2]; k <= hi[2]; k++) {
          double ct = 0.0;
          const int m = b.mrow[j + NG];
          if (d == 2 && m > 1) {
            // C-15 (ii): fluxes only on group-boundary faces (the others are interpolated by
            // deref_fix_fluxes); the Courant limit of the row uses the group width m dx3
            if (k < 0 || k > b.n[2] || k % m != 0) continue;
            face_flux_x3_deref(par, b, src, i, j, k, m, &ct);
            ct /= (double)m;
          } else {
            face_flux(par, b, src, d, i, j, k, &ct);
          }
          const int id[3] = {i, j, k};
          bool act = true;  // C-14: the Courant maximum runs over the faces of ACTIVE zones
          for (int t = 0; t < 3; t++)
            if (t != d && (id[t] < 0 || id[t] >= b.n[t])) act = false;
          if (act) cmaxd = std::max(cmaxd, ct);
        }
    b.ctop[d] = cmaxd;
  }
}

// ---- phi-derefinement fix-ups (C-15; "averages the fluxes ... over 2^n cells") --------------
// Everything is stored on the fine grid.  After the flux pass the face quantities of derefined rows are
// given the group structure: x1- and x2-face values become their group mean, x3-face values between
// group boundaries the linear interpolation of the two boundary faces.  With one value per fine face
// and per fine edge, the unchanged update conserves and the unchanged CT keeps div B per FINE zone.
static inline int face2_factor(const Block& b, int j) {  // x2-face j lies between rows j-1 and j
  return std::max(b.mrow[j - 1 + NG], b.mrow[j + NG]);
}

// pairwise (tree) sum of m = 2^p values: the mean of m IDENTICAL values is then that value exactly, so group
// quantities that are already uniform are left bit-for-bit alone (blocks that share a group boundary stay
// consistent)
static double tree_sum(const double* v, int m) {
  if (m == 1) return v[0];
  return tree_sum(v, m / 2) + tree_sum(v + m / 2, m / 2);
}

static void group_mean(std::vector<double>& a, const Block& b, int i, int j, int m) {
  const int n3 = b.n[2];
  for (int k0 = 0; k0 < n3; k0 += m) {
    const double mean = tree_sum(&a[b.idx(i, j, k0)], m) / (double)m;
    for (int r = 0; r < m; r++) a[b.idx(i, j, k0 + r)] = mean;
  }
}

static void group_interp(std::vector<double>& a, const Block& b, int i, int j, int m) {
  const int n3 = b.n[2];
  for (int k0 = 0; k0 < n3; k0 += m) {
    const double lo = a[b.idx(i, j, k0)], hi = a[b.idx(i, j, k0 + m)];
    for (int r = 1; r < m; r++) a[b.idx(i, j, k0 + r)] = lo + ((double)r / (double)m) * (hi - lo);
  }
}

void deref_fix_fluxes(const Params& par, Block& b) {
  if (par.n_deref <= 0) return;
  for (int i = -1; i <= b.n[0]; i++)
    for (int j = -1; j <= b.n[1]; j++) {
      const int m = b.mrow[j + NG];
      const bool ent = par.entropy_backup != 0;   // C-18: the entropy flux is one more flux of the row
      if (m > 1 && i >= 0) {          // x1-faces of the row
        if (ent) group_mean(b.FK[0], b, i, j, m);
        for (int c = 0; c < 5; c++) group_mean(b.F[0][c], b, i, j, m);
        group_mean(b.Ef[0][1], b, i, j, m);
        group_mean(b.Ef[0][2], b, i, j, m);
      }
      if (m > 1) {                    // x3-faces of the row: in-group faces
        if (ent) group_interp(b.FK[2], b, i, j, m);
        for (int c = 0; c < 5; c++) group_interp(b.F[2][c], b, i, j, m);
        group_interp(b.Ef[2][0], b, i, j, m);
        group_interp(b.Ef[2][1], b, i, j, m);
      }
      if (j >= 0) {                   // x2-face between rows j-1 and j: the coarser of the two groupings
        const int M = face2_factor(b, j);
        if (M > 1) {
          if (ent) group_mean(b.FK[1], b, i, j, M);
          for (int c = 0; c < 5; c++) group_mean(b.F[1][c], b, i, j, M);
          group_mean(b.Ef[1][2], b, i, j, M);
          group_mean(b.Ef[1][0], b, i, j, M);
        }
      }
    }
}

// C-15 (iv): E3 is a group mean; E1 and E2 exist on group-boundary phi-edges, the ones in between are
// their linear interpolation.  Edges on an x2-face row use the coarser grouping of the two rows.
void deref_fix_edges(const Params& par, Block& b) {
  if (par.n_deref <= 0) return;
  const int n3 = b.n[2];
  for (int i = 0; i <= b.n[0]; i++)
    for (int j = 0; j <= b.n[1]; j++) {
      const int m = b.mrow[j + NG], M = face2_factor(b, j);
      if (M > 1) {                                         // E3 at (i-1/2, j-1/2, k)
        for (int k0 = 0; k0 < n3; k0 += M) {
          double sum = 0.0;
          sum = tree_sum(&b.Ee[2][b.idx(i, j, k0)], M);
          for (int r = 0; r < M; r++) b.Ee[2][b.idx(i, j, k0 + r)] = sum / (double)M;
        }
      }
      if (M > 1 && i < b.n[0]) group_interp(b.Ee[0], b, i, j, M);   // E1 at (i, j-1/2, k-1/2)
      if (m > 1 && j < b.n[1]) group_interp(b.Ee[1], b, i, j, m);   // E2 at (i-1/2, j, k-1/2)
    }
}

// C-15 (v): one inversion per group: the group's first member's result is the group's
// The whole invariant (i) is re-imposed EXACTLY after every update: hydro and B_c of a group are its first
// member's; Bf1 (row grouping) and Bf2 (the coarser grouping of the two rows of its face) likewise; Bf3 on
// in-group faces is re-interpolated from the group's outer faces.  The update leaves all of these true to
// round-off only (the interpolated EMFs differ in the last bit between members); making them exact keeps
// neighbouring blocks, which recompute shared faces from copies of each other's groups, bit-for-bit
// consistent, and costs div B nothing beyond round-off that does not accumulate.
void deref_sync_groups(const Params& par, Block& b, Fields& s) {
  if (par.n_deref <= 0) return;
  for (int i = 0; i <= b.n[0]; i++)
    for (int j = 0; j <= b.n[1]; j++) {
      const int m = b.mrow[j + NG], M = face2_factor(b, j);
      for (int k = 0; k < b.n[2]; k++) {
        const size_t z = b.idx(i, j, k);
        if (m > 1 && k % m != 0 && j < b.n[1]) {
          const size_t z0 = b.idx(i, j, k - k % m);
          s.Bf[0][z] = s.Bf[0][z0];
          if (i < b.n[0]) {
            for (int c = 0; c < 5; c++) s.P[c][z] = s.P[c][z0];
            for (int c = 0; c < 3; c++) s.Bc[c][z] = s.Bc[c][z0];
          }
        }
        if (M > 1 && k % M != 0 && i < b.n[0]) s.Bf[1][z] = s.Bf[1][b.idx(i, j, k - k % M)];
      }
      if (m > 1 && i < b.n[0] && j < b.n[1]) group_interp(s.Bf[2], b, i, j, m);
    }
}

// C-15 (i): puts an initial state onto the invariant: hydro primitives become their group mean; the
// x3-face field between group boundaries the linear interpolation of the boundary faces.  The face
// fields Bf1, Bf2 are expected to be group-uniform already (true for any axisymmetric field).
void deref_project(const Params& par, Block& b, Fields& s) {
  if (par.n_deref <= 0) return;
  for (int i = 0; i <= b.n[0]; i++)
    for (int j = 0; j < b.n[1]; j++) {
      const int m = b.mrow[j + NG];
      if (m <= 1) continue;
      if (i < b.n[0]) {
        for (int c = 0; c < 5; c++)
          for (int k0 = 0; k0 < b.n[2]; k0 += m) {
            const double sum = tree_sum(&s.P[c][b.idx(i, j, k0)], m);
            for (int r = 0; r < m; r++) s.P[c][b.idx(i, j, k0 + r)] = sum / (double)m;
          }
        group_interp(s.Bf[2], b, i, j, m);
      }
    }
  deref_sync_groups(par, b, s);   // Bf1, Bf2 onto their first member as well
}

// ---- constrained transport (C-8, C-9) -------------------------------------------------------------
static inline double up(double m, double lo, double hi) {
  return m > 0.0 ? lo : (m < 0.0 ? hi : 0.5 * (lo + hi));
}

void ct_edges(const Params& par, Block& b, const Fields& s) {
  const int str[3] = {b.e[1] * b.e[2], b.e[2], 1};
  // centre EMFs E^c_k = -eps_{kmn} v^m Bdens^n on active zones plus one ghost layer
#pragma omp parallel for collapse(2)
  for (int i = -1; i <= b.n[0]; i++)
    for (int j = -1; j <= b.n[1]; j++)
      for (int k = -1; k <= b.n[2]; k++) {
        const size_t z = b.idx(i, j, k);
        const Geom& G = b.gc[b.idx2(i, j)];
        double P[8];
        for (int c = 0; c < 5; c++) P[c] = s.P[c][z];
        for (int c = 0; c < 3; c++) P[5 + c] = s.Bc[c][z];
        State S;
        get_state(P, G, S);
        const double v[3] = {S.ucon[1] / S.ucon[0], S.ucon[2] / S.ucon[0], S.ucon[3] / S.ucon[0]};
        const double B[3] = {G.gdet * P[5], G.gdet * P[6], G.gdet * P[7]};
        b.Cc[0][z] = -(v[1] * B[2] - v[2] * B[1]);
        b.Cc[1][z] = -(v[2] * B[0] - v[0] * B[2]);
        b.Cc[2][z] = -(v[0] * B[1] - v[1] * B[0]);
      }
  // edge EMF E_f at (d-1/2, e-1/2), (d,e,f) cyclic
  for (int f = 0; f < 3; f++) {
    const int d = CYC[f][1], e = CYC[f][2];
    const ptrdiff_t sD = str[d], sE = str[e];
    const std::vector<double>&X = b.Ef[d][f], &Y = b.Ef[e][f], &C = b.Cc[f];
    const std::vector<double>&md = b.F[d][0], &me = b.F[e][0];
    int hi[3] = {b.n[0], b.n[1], b.n[2]};
    hi[f] = b.n[f] - 1;
#pragma omp parallel for collapse(2)
    for (int i = 0; i <= hi[0]; i++)
      for (int j = 0; j <= hi[1]; j++)
        for (int k = 0; k <= hi[2]; k++) {
          const size_t z = b.idx(i, j, k);
          // C-9: edges on the polar axis carry E1 = E3 = 0 exactly
          if (f != 1 && b.pole2[j + NG]) { b.Ee[f][z] = 0.0; continue; }
          const double E =
              0.25 * (X[z] + X[z - sE] + Y[z] + Y[z - sD]) +
              0.25 * (up(md[z - sE], Y[z - sD] - C[z - sD - sE], Y[z] - C[z - sE]) -
                      up(md[z], C[z - sD] - Y[z - sD], C[z] - Y[z])) +
              0.25 * (up(me[z - sD], X[z - sE] - C[z - sD - sE], X[z] - C[z - sD]) -
                      up(me[z], C[z - sE] - X[z - sE], C[z] - X[z]));
          b.Ee[f][z] = E;
        }
  }
  (void)par;
}

// ---- floors and ceiling (C-13; PAPER.md:59 says only "below a certain threshold") -----------------
// C-19 (par.drift_floors; "injects mass and internal energy in the drift frame of the jet ... (Ressler et
// al. 2017)"): the mass and energy added to reach the floors are added in the frame that moves with the part of the
// velocity perpendicular to the magnetic field.  In the normal observer's frame, with v^i = ut^i / gamma and
// curly-B^i = alpha B^i:   v^i = v_perp^i + v_par Bhat^i,   v_par = (v . B) / |B|.
//   * v_perp (the E x B drift: E = -v x B does not see v_par) is left unchanged: no drag on the field lines;
//   * the momentum along the field, m_par = w gamma^2 v_par (w = rho + gamma_ad u; the electromagnetic momentum
//     is perpendicular to B), is conserved: the added matter carries none, so v_par drops and cannot run away.
// With w' the enthalpy after the floors:  w' v_par' / (1 - v_perp^2 - v_par'^2) = m_par, whose root of the sign of
// m_par is  v_par' = 2 m_par s / (w' + sqrt(w'^2 + 4 m_par^2 s)),  s = 1 - v_perp^2.   B = 0: the fluid frame.
void floors_and_ceiling(const Params& par, const Geom& G, double r, double P[5], const double* Bc, Stats& st) {
  const double rfl = par.rho_fl_coef * std::pow(r, par.rho_fl_pow);
  const double ufl = par.u_fl_coef * std::pow(r, par.u_fl_pow);
  const bool lowr = P[0] < rfl, lowu = P[1] < ufl;
  double Bsq = 0.0;
  if (par.drift_floors && Bc && (lowr || lowu))
    for (int i = 1; i < 4; i++)
      for (int j = 1; j < 4; j++) Bsq += G.gcov[i][j] * (G.alpha * Bc[i - 1]) * (G.alpha * Bc[j - 1]);
  if (Bsq > 0.0) {
    double q = 0.0;
    for (int i = 1; i < 4; i++)
      for (int j = 1; j < 4; j++) q += G.gcov[i][j] * P[1 + i] * P[1 + j];
    const double gamma = std::sqrt(1.0 + q);
    double v[3], vB = 0.0;
    for (int i = 0; i < 3; i++) v[i] = P[2 + i] / gamma;
    for (int i = 1; i < 4; i++)
      for (int j = 1; j < 4; j++) vB += G.gcov[i][j] * v[i - 1] * (G.alpha * Bc[j - 1]);
    const double Bn = std::sqrt(Bsq);
    const double vpar = vB / Bn;
    double vperp[3], vperp2 = 0.0;
    for (int i = 0; i < 3; i++) vperp[i] = v[i] - vpar * (G.alpha * Bc[i]) / Bn;
    for (int i = 1; i < 4; i++)
      for (int j = 1; j < 4; j++) vperp2 += G.gcov[i][j] * vperp[i - 1] * vperp[j - 1];
    const double mpar = (P[0] + par.gamma_ad * P[1]) * gamma * gamma * vpar;
    if (lowr) { P[0] = rfl; st.rho_floor++; }
    if (lowu) { P[1] = ufl; st.u_floor++; }
    const double wn = P[0] + par.gamma_ad * P[1];
    const double s = 1.0 - vperp2;
    const double vparn = 2.0 * mpar * s / (wn + std::sqrt(wn * wn + 4.0 * mpar * mpar * s));
    const double gn = 1.0 / std::sqrt(s - vparn * vparn);
    for (int i = 0; i < 3; i++) P[2 + i] = gn * (vperp[i] + vparn * (G.alpha * Bc[i]) / Bn);
  } else {
    if (lowr) { P[0] = rfl; st.rho_floor++; }
    if (lowu) { P[1] = ufl; st.u_floor++; }
  }
  double q = 0.0;
  for (int i = 1; i < 4; i++)
    for (int j = 1; j < 4; j++) q += G.gcov[i][j] * P[1 + i] * P[1 + j];
  const double gamma = std::sqrt(1.0 + q);
  if (gamma > par.gamma_max) {
    const double fac = std::sqrt((par.gamma_max * par.gamma_max - 1.0) / (gamma * gamma - 1.0));
    for (int i = 2; i < 5; i++) P[i] *= fac;
    st.gam_ceil++;
  }
}

// ---- B update, source, conservative update, inversion (C-10, C-12, C-13) ---------------------------
void update(const Params& par, Block& b, const Fields& src, const Fields& base, Fields& out,
            double dt, Stats& st) {
  const int str[3] = {b.e[1] * b.e[2], b.e[2], 1};
  // C-10: Bf^d -= dt [ (E_f(e+) - E_f(e-))/dx^e - (E_e(f+) - E_e(f-))/dx^f ]
  for (int d = 0; d < 3; d++) {
    const int e = CYC[d][1], f = CYC[d][2];
    int hi[3] = {b.n[0] - 1, b.n[1] - 1, b.n[2] - 1};
    hi[d] = b.n[d];
#pragma omp parallel for collapse(2)
    for (int i = 0; i <= hi[0]; i++)
      for (int j = 0; j <= hi[1]; j++)
        for (int k = 0; k <= hi[2]; k++) {
          const size_t z = b.idx(i, j, k);
          if (d == 1 && b.pole2[j + NG]) { out.Bf[d][z] = 0.0; continue; }
          const double curl = (b.Ee[f][z + str[e]] - b.Ee[f][z]) / b.dx[e] -
                              (b.Ee[e][z + str[f]] - b.Ee[e][z]) / b.dx[f];
          out.Bf[d][z] = base.Bf[d][z] - dt * curl;
        }
  }
  compute_Bc(b, out, true);
  long long nfail = 0, nrf = 0, nuf = 0, ngc = 0, nent = 0, nait = 0;
  if (par.entropy_backup) b.Kadv.assign(b.size(), 0.0);
#pragma omp parallel for collapse(2) reduction(+ : nfail, nrf, nuf, ngc, nent, nait)
  for (int i = 0; i < b.n[0]; i++)
    for (int j = 0; j < b.n[1]; j++) {
      const Geom& G = b.gc[b.idx2(i, j)];
      const double(*conn)[4][4] = (const double(*)[4][4]) & b.conn[b.idx2(i, j) * 64];
      const double r = (par.metric == 1) ? std::exp(b.xc(0, i)) : 1.0;
      for (int k = 0; k < b.n[2]; k++) {
        const size_t z = b.idx(i, j, k);
        double Pb[8], Ps[8], Ub[8], Ssrc[5], U[5];
        for (int c = 0; c < 5; c++) { Pb[c] = base.P[c][z]; Ps[c] = src.P[c][z]; }
        for (int c = 0; c < 3; c++) { Pb[5 + c] = base.Bc[c][z]; Ps[5 + c] = src.Bc[c][z]; }
        State Sb, Ss;
        get_state(Pb, G, Sb);
        prim_to_U(Pb, Sb, G, par.gamma_ad, Ub);
        get_state(Ps, G, Ss);
        source(Ps, Ss, G, conn, par.gamma_ad, Ssrc);
        for (int c = 0; c < 5; c++) {
          double div = 0.0;
          for (int d = 0; d < 3; d++) div += (b.F[d][c][z + str[d]] - b.F[d][c][z]) / b.dx[d];
          U[c] = Ub[c] - dt * div + dt * Ssrc[c];
        }
        const double Bn[3] = {out.Bc[0][z], out.Bc[1][z], out.Bc[2][z]};
        double Pn[5];
        int rc = con2prim(U, Bn, G, par.gamma_ad, Ps, Pn, nullptr);
        if (par.entropy_backup && rc != 0) {
          // C-21: the second primary inversion, where the Newton-Raphson one did not converge
          double Pa[5];
          if (con2prim_aitken(U, Bn, G, par.gamma_ad, Ps, Pa, nullptr) == 0) {
            for (int c = 0; c < 5; c++) Pn[c] = Pa[c];
            rc = 0;
            nait++;
          }
        }
        if (par.entropy_backup) {
          // C-18: the entropy row, advanced like the others (no source term), and the backup inversion wherever
          // the energy inversion failed or returned a state without positive density and non-negative energy
          double USb, Fdummy;
          entropy_UF(Pb, Sb, G, par.gamma_ad, 1, USb, Fdummy);
          double div = 0.0;
          for (int d = 0; d < 3; d++) div += (b.FK[d][z + str[d]] - b.FK[d][z]) / b.dx[d];
          const double US = USb - dt * div;
          b.Kadv[z] = US / U[0];
          if (rc != 0 || !(Pn[0] > 0.0) || !(Pn[1] >= 0.0)) {
            double Pe[5];
            // an entropy row that went negative (kappa < 0) or has no root leaves what the energy inversion gave:
            // its converged state for the floors to repair, or its failure
            if (con2prim_entropy(U, US, Bn, G, par.gamma_ad, Ps, Pe, nullptr) == 0) {
              for (int c = 0; c < 5; c++) Pn[c] = Pe[c];
              rc = 0;
              nent++;
            }
          }
        }
        if (rc != 0) {  // C-13: keep the source state's hydro primitives, count the failure
          nfail++;
          for (int c = 0; c < 5; c++) Pn[c] = Ps[c];
        }
        Stats loc = {0, 0, 0, 0, 0, 0};
        floors_and_ceiling(par, G, r, Pn, Bn, loc);
        nrf += loc.rho_floor; nuf += loc.u_floor; ngc += loc.gam_ceil;
        for (int c = 0; c < 5; c++) out.P[c][z] = Pn[c];
      }
    }
  st.c2p_entropy += nent; st.c2p_aitken += nait; st.c2p_fail += nfail; st.rho_floor += nrf; st.u_floor += nuf; st.gam_ceil += ngc;
  deref_sync_groups(par, b, out);
}

// C-14 (PAPER.md:93 fn. 2): 1/dt = sum_d 1/dt_d, dt_d = C dx^d / max ctop_d
double dt_from_ctop(const Params& par, const Block& b) {
  double s = 0.0;
  for (int d = 0; d < 3; d++) s += b.ctop[d] / b.dx[d];
  return par.cour / s;
}

}  // namespace orc
