// ORACLE (test infrastructure) — block-structured grid: block lattice, ghost exchange between
// blocks, local adaptive time-stepping with flux / EMF correction.  DESIGN.md §9 (C-16, C-17);
// PAPER.md:71 (blocks, boundary-cell transfer), PAPER.md:105 (LAT: per-block dt in factors of 2),
// PAPER.md:137 (flux / EMF synchronisation between time levels, correction added to the coarse
// block's boundary cells, extra inversion there).
#include "orc_grid.hpp"
#include <algorithm>
#include <cstring>
#include <stdexcept>

namespace orc {

static const int CYC[3][3] = {{0, 1, 2}, {1, 2, 0}, {2, 0, 1}};  // (d, e, f) cyclic

// ---- block lattice (C-16) -----------------------------------------------------------------------
void blocks_build(Grid& g) {
  const Params& par = g.par;
  double lo[3], hi[3], dx0[3];
  int nb[3], NB[3];
  for (int d = 0; d < 3; d++) { lo[d] = par.xmin[d]; hi[d] = par.xmax[d]; }
  if (par.metric == 1) { lo[0] = std::log(par.xmin[0]); hi[0] = std::log(par.xmax[0]); }
  for (int d = 0; d < 3; d++) {
    nb[d] = par.nb[d] > 0 ? par.nb[d] : par.n[d];
    if (par.n[d] % nb[d] != 0) throw std::runtime_error("n[d] is not a multiple of nb[d]");
    NB[d] = par.n[d] / nb[d];
    dx0[d] = (hi[d] - lo[d]) / par.n[d];
  }
  // x1 slots: a base block column whose x1-centre has r < r_refine_max is replaced by two children
  // with dx1/2 (C-16; PAPER.md:71 per-dimension splitting)
  struct Slot { int col, lev, child; };
  std::vector<Slot> slots;
  bool seen_coarse = false;
  for (int col = 0; col < NB[0]; col++) {
    bool refined = false;
    if (par.r_refine_max > 0.0) {
      // centre of the column: r on the Kerr-Schild map, x1 itself on the Cartesian map
      const double xc = lo[0] + ((double)col + 0.5) * nb[0] * dx0[0];
      refined = (par.metric == 1 ? std::exp(xc) : xc) < par.r_refine_max;
    }
    if (refined && seen_coarse) throw std::runtime_error("refined columns must be contiguous from r_in");
    // a coarse ghost layer of NG zones is the restriction of 2 NG fine zones of ONE neighbour
    if (refined && nb[0] < 2 * NG) throw std::runtime_error("x1 refinement needs nb[0] >= 6");
    if (refined) { slots.push_back({col, 1, 0}); slots.push_back({col, 1, 1}); }
    else { slots.push_back({col, 0, 0}); seen_coarse = true; }
  }
  if (par.n_deref > 0) {
    // C-15: the strided x3 stencil of a derefined row wraps inside the block
    // C-15: groups never straddle blocks and a ghost depth of 3 groups fits one neighbour; factors are powers of 2
    if (par.bc_lo[2] != 0) throw std::runtime_error("phi-derefinement needs a periodic x3");
    for (int t = 0; t < par.n_deref && t < 4; t++) {
      const int f = par.deref_factor[t];
      if (f < 1 || (f & (f - 1)) != 0 || nb[2] % f != 0 || nb[2] < 3 * f)
        throw std::runtime_error("deref factor must be a power of two with 3 factor <= nb[2], dividing it");
    }
  }
  g.nslot[0] = (int)slots.size(); g.nslot[1] = NB[1]; g.nslot[2] = NB[2];
  g.lattice.assign((size_t)g.nslot[0] * NB[1] * NB[2], -1);
  g.blocks.clear();
  g.blocks.resize(g.lattice.size());
  int id = 0;
  for (int s = 0; s < g.nslot[0]; s++)
    for (int bj = 0; bj < NB[1]; bj++)
      for (int bk = 0; bk < NB[2]; bk++, id++) {
        Block& b = g.blocks[id];
        g.lattice[((size_t)s * NB[1] + bj) * NB[2] + bk] = id;
        b.slot[0] = s; b.slot[1] = bj; b.slot[2] = bk;
        b.lev1 = slots[s].lev;
        for (int d = 0; d < 3; d++) { b.n[d] = nb[d]; b.dx[d] = dx0[d]; b.x0[d] = lo[d]; }
        b.I0[0] = slots[s].lev ? (long long)(2 * slots[s].col + slots[s].child) * nb[0]
                               : (long long)slots[s].col * nb[0];
        if (b.lev1) b.dx[0] = dx0[0] / 2.0;
        b.I0[1] = (long long)bj * nb[1];
        b.I0[2] = (long long)bk * nb[2];
        for (int d = 0; d < 3; d++) {
          // periodic dimensions are closed through the neighbour table, not through fill_physical_bc
          b.phys_lo[d] = b.slot[d] == 0 && par.bc_lo[d] != 0;
          b.phys_hi[d] = b.slot[d] == g.nslot[d] - 1 && par.bc_hi[d] != 0;
        }
        b.tau = 0; b.tb_u = 0; b.dt_u = 2; b.has_new = false;
        // NEXT-1: with x3 cut into blocks the rows beyond a transmissive pole belong to another block
        b.xpole_lo = b.phys_lo[1] && par.bc_lo[1] == 3 && NB[2] > 1;
        b.xpole_hi = b.phys_hi[1] && par.bc_hi[1] == 3 && NB[2] > 1;
      }
  for (Block& b : g.blocks) {
    for (int o0 = -1; o0 <= 1; o0++)
      for (int o1 = -1; o1 <= 1; o1++)
        for (int o2 = -1; o2 <= 1; o2++) {
          const int o[3] = {o0, o1, o2};
          int s[3];
          bool inside = true;
          for (int d = 0; d < 3; d++) {
            s[d] = b.slot[d] + o[d];
            if (s[d] < 0 || s[d] >= g.nslot[d]) {
              if (par.bc_lo[d] == 0) s[d] = (s[d] + g.nslot[d]) % g.nslot[d];
              else inside = false;
            }
          }
          b.nbr[o0 + 1][o1 + 1][o2 + 1] =
              inside ? g.lattice[((size_t)s[0] * g.nslot[1] + s[1]) * g.nslot[2] + s[2]] : -1;
        }
  }
  for (Block& b : g.blocks)
    for (int o0 = -1; o0 <= 1; o0++)
      for (int o2 = -1; o2 <= 1; o2++) {
        const int s0 = b.slot[0] + o0;                   // x1 is never periodic together with a pole
        const int s2 = ((b.slot[2] + g.nslot[2] / 2 + o2) % g.nslot[2] + g.nslot[2]) % g.nslot[2];
        const bool inside = s0 >= 0 && s0 < g.nslot[0] && (b.xpole_lo || b.xpole_hi);
        b.pnbr[o0 + 1][o2 + 1] = inside ? g.lattice[((size_t)s0 * g.nslot[1] + b.slot[1]) * g.nslot[2] + s2] : -1;
      }
  for (Block& b : g.blocks) {
    // C-16 ghost geometry on a refined x1 level uses the block's own (fine or coarse) spacing
    if (b.lev1) {
      // pole2 / geometry use global x2 index and the block's own x1 spacing: block_init reads
      // I0 and dx, which are already those of the block's level
    }
    block_init(par, b);
    const size_t n = b.size();
    for (int d = 0; d < 3; d++) {
      for (int c = 0; c < 5; c++) { b.FA[d][c].assign(n, 0.0); b.FA2[d][c].assign(n, 0.0); }
      b.EA[d].assign(n, 0.0);
      b.EA2[d].assign(n, 0.0);
      if (par.entropy_backup) { b.FKA[d].assign(n, 0.0); b.FKA2[d].assign(n, 0.0); }
      b.ctop_last[d] = 0.0;
    }
  }
}

// ---- ghost exchange (C-16 same-level copy; C-17 time interpolation) ----------------------------------
// value at integer time s_u (units of dt_0/2) of an array of block q given its three time levels
static inline double sample(const Block& q, const std::vector<double>& an, const std::vector<double>& ah,
                            const std::vector<double>& aw, size_t z, long long s_u) {
  if (s_u == q.tb_u) return an[z];                       // a completed state: copy
  if (q.has_new) {                                       // completed states bracket s: linear in time
    const double w = (double)(s_u - q.tb_u) / (double)q.dt_u;
    return (1.0 - w) * an[z] + w * aw[z];
  }
  const double w = (double)(s_u - q.tb_u) / (double)(q.dt_u / 2);  // state n and its predictor state
  return (1.0 - w) * an[z] + w * ah[z];
}

// NEXT-1 on blocks that cut x3 (fill_polar_transmit in orc_grid.cpp is the same rule inside one
// block): ghost row j beyond a transmissive pole is the mirror row of the block half a turn away, at the same
// local x3 index; ut^2 and Bf^2 change sign.
static inline bool across_pole(const Block& b, int o1) { return (o1 < 0 && b.xpole_lo) || (o1 > 0 && b.xpole_hi); }
static inline int pole_mirror(const Block& b, int j, bool face2) {
  if (j < 0) return face2 ? -j : -j - 1;
  return b.n[1] - (j - (face2 ? b.n[1] : b.n[1] - 1));
}
// x3 grouping of the SOURCE row js (of x2-face js: the coarser of the two rows it separates)
static inline int pole_group(const Block& b, int js, bool face2) {
  return face2 ? std::max(b.mrow[js - 1 + NG], b.mrow[js + NG]) : b.mrow[js + NG];
}

static void exchange_block(Grid& g, Block& b, Fields& dst, long long s_u) {
  auto off = [](int idx, int n, bool face) { return idx < 0 ? -1 : (idx > (face ? n : n - 1) ? 1 : 0); };
  for (int i = -NG; i < b.n[0] + NG + 1; i++)
    for (int j = -NG; j < b.n[1] + NG + 1; j++)
      for (int k = -NG; k < b.n[2] + NG + 1; k++) {
        const int id[3] = {i, j, k};
        const size_t z = b.idx(i, j, k);
        // a = 0: zone-centred hydro primitives; a = 1 + d: the d-face field
        for (int a = 0; a < 4; a++) {
          int o[3], lq[3];
          bool ghost = false, valid = true;
          for (int d = 0; d < 3; d++) {
            const bool face = (a == 1 + d);
            if (!face && id[d] > b.n[d] + NG - 1) valid = false;  // index n+3 exists for faces only
            o[d] = off(id[d], b.n[d], face);
            if (o[d] != 0) ghost = true;
          }
          if (!valid) continue;
          const bool xp = across_pole(b, o[1]);
          // the block itself if no offset
          int qi = xp ? b.pnbr[o[0] + 1][o[2] + 1] : b.nbr[o[0] + 1][o[1] + 1][o[2] + 1];
          if (qi < 0) continue;                          // outside the domain: physical boundary
          for (int d = 0; d < 3; d++) lq[d] = id[d] - o[d] * b.n[d];
          if (xp) lq[1] = pole_mirror(b, j, a == 2);
          // C-15: the phi-ghost slots of a derefined row are in group units
          if (o[2] != 0) {
            // an x2-face array follows the grouping of its face, the coarser of the two rows it separates
            const int mg = xp ? pole_group(b, lq[1], a == 2)
                              : (a == 2 ? std::max(b.mrow[std::max(j - 1, -NG) + NG], b.mrow[j + NG]) : b.mrow[j + NG]);
            int o2;
            if (mg > 1) lq[2] = deref_ghost_k(k, b.n[2], mg, a == 3, o2);
          }
          // C-17: a face on the plane between two blocks on different time levels has ONE value in
          // every stage source, that of the finer block (own boundary faces included)
          if (a > 0 && (id[a - 1] == 0 || id[a - 1] == b.n[a - 1])) {
            const int d = a - 1;
            int o2[3] = {o[0], o[1], o[2]};
            o2[d] = id[d] == 0 ? -1 : 1;
            const int q2 = xp ? b.pnbr[o2[0] + 1][o2[2] + 1] : b.nbr[o2[0] + 1][o2[1] + 1][o2[2] + 1];
            if (q2 >= 0 && g.blocks[q2].tau < g.blocks[qi].tau && g.blocks[q2].lev1 == g.blocks[qi].lev1) {
              qi = q2;
              lq[d] = id[d] == 0 ? b.n[d] : 0;
              ghost = true;
            }
          }
          if (!ghost) continue;
          const Block& q = g.blocks[qi];
          if (q.lev1 != b.lev1) continue;                // coarse <-> fine: exchange_refined()
          const size_t zq = q.idx(lq[0], lq[1], lq[2]);
          if (a == 0) {
            for (int c = 0; c < 5; c++) {
              const double v = sample(q, q.sn.P[c], q.sh.P[c], q.snew.P[c], zq, s_u);
              dst.P[c][z] = (xp && c == 3) ? -v : v;
            }
          } else {
            const int d = a - 1;
            const double v = sample(q, q.sn.Bf[d], q.sh.Bf[d], q.snew.Bf[d], zq, s_u);
            dst.Bf[d][z] = (xp && d == 1) ? -v : v;
          }
        }
      }
}

// ---- ghost exchange across the x1 refinement interface (C-16) ------------------------------------------------
// A refined block has dx1/2 and unchanged dx2, dx3, so only the x1 index changes meaning across the
// interface.  kind: 0..4 hydro primitive, 5 + d the d-face field.  All reads go through sample().
static double sample_kind(const Block& q, int kind, int i, int j, int k, long long s_u) {
  const size_t z = q.idx(i, j, k);
  if (kind < 5) return sample(q, q.sn.P[kind], q.sh.P[kind], q.snew.P[kind], z, s_u);
  const int d = kind - 5;
  return sample(q, q.sn.Bf[d], q.sh.Bf[d], q.snew.Bf[d], z, s_u);
}

// C-16 restriction: coarse value = arithmetic mean of the two fine values it covers (primitives and
// densitised transverse faces alike)
static double restrict2(const Block& qf, int kind, int i0, int j, int k, long long s_u) {
  return 0.5 * (sample_kind(qf, kind, i0, j, k, s_u) + sample_kind(qf, kind, i0 + 1, j, k, s_u));
}

static void exchange_refined(Grid& g, Block& b, Fields& dst, long long s_u) {
  for (int side = 0; side < 2; side++) {
    const int o0 = side ? 1 : -1;
    for (int o1 = -1; o1 <= 1; o1++)
      for (int o2 = -1; o2 <= 1; o2++) {
        const bool xp = across_pole(b, o1);
        const int qi = xp ? b.pnbr[o0 + 1][o2 + 1] : b.nbr[o0 + 1][o1 + 1][o2 + 1];
        if (qi < 0 || g.blocks[qi].lev1 == b.lev1) continue;
        const Block& q = g.blocks[qi];
        // the block on b's own side of the interface in the same transverse position (b itself for
        // o1 = o2 = 0): it covers the zones just outside q
        const int ri = xp ? b.pnbr[1][o2 + 1] : b.nbr[1][o1 + 1][o2 + 1];
        const Block& r = g.blocks[ri];
        const int n0 = b.n[0];
        // ranges of the padded indices that fall into q
        auto range = [&](int o, int n, int& lo, int& hi, bool face) {
          if (o < 0) { lo = -NG; hi = -1; }
          else if (o > 0) { lo = face ? n + 1 : n; hi = face ? n + NG : n + NG - 1; }
          else { lo = 0; hi = face ? n : n - 1; }
        };
        for (int kind = 0; kind < 8; kind++) {
          if (kind > 0 && kind < 5) continue;          // the five hydro variables share kind 0's geometry
          const int fd = kind >= 5 ? kind - 5 : -1;    // face direction
          int lo[3], hi[3];
          range(o0, b.n[0], lo[0], hi[0], fd == 0);
          range(o1, b.n[1], lo[1], hi[1], fd == 1);
          range(o2, b.n[2], lo[2], hi[2], fd == 2);
          for (int i = lo[0]; i <= hi[0]; i++)
            for (int j = lo[1]; j <= hi[1]; j++)
              for (int k = lo[2]; k <= hi[2]; k++) {
                int o2u;
                const int lj = xp ? pole_mirror(b, j, fd == 1) : j - o1 * b.n[1];
                const int mg = xp ? pole_group(b, lj, fd == 1)
                                  : (fd == 1 ? std::max(b.mrow[std::max(j - 1, -NG) + NG], b.mrow[j + NG]) : b.mrow[j + NG]);
                const int lk = o2 != 0 ? deref_ghost_k(k, b.n[2], mg, fd == 2, o2u) : k;
                const int nk = kind == 0 ? 5 : 1;
                for (int c = 0; c < nk; c++) {
                  const int kd = kind == 0 ? c : kind;
                  double v;
                  if (b.lev1 == 0) {
                    // ---- coarse ghost from fine data
                    if (fd == 0) {               // normal face: coincident fine face, copied
                      const int t = side ? i - n0 : -i;            // 1..3 coarse faces from the interface
                      v = sample_kind(q, kd, side ? 2 * t : n0 - 2 * t, lj, lk, s_u);
                    } else {                     // zones and transverse faces: mean of the two fine ones
                      const int t = side ? i - n0 : -1 - i;        // 0..2 coarse zones from the interface
                      v = restrict2(q, kd, side ? 2 * t : n0 - 2 * t - 2, lj, lk, s_u);
                    }
                  } else {
                    // ---- fine ghost from coarse data
                    if (fd == 0) {
                      // normal faces: coincident ones copied, in-between ones the mean of their neighbours
                      const int t = side ? i - n0 : -i;            // 1..3 fine faces from the interface
                      const int c0 = side ? t / 2 : n0 - t / 2;    // coarse face at or just inside
                      if (t % 2 == 0) v = sample_kind(q, kd, c0, lj, lk, s_u);
                      else v = 0.5 * (sample_kind(q, kd, c0, lj, lk, s_u) +
                                      sample_kind(q, kd, side ? c0 + 1 : c0 - 1, lj, lk, s_u));
                    } else {
                      // zones and transverse faces: piecewise linear in x1 with the MC-limited slope,
                      // evaluated a quarter of a coarse zone off the coarse centre
                      const int t = side ? i - n0 : -1 - i;        // 0..2 fine zones from the interface
                      const int ic = side ? t / 2 : n0 - 1 - t / 2;
                      const bool high_half = side ? (t % 2 == 1) : (t % 2 == 0);
                      double a3[3];
                      for (int w = -1; w <= 1; w++) {
                        const int iw = ic + w;
                        if (iw >= 0 && iw < n0) a3[w + 1] = sample_kind(q, kd, iw, lj, lk, s_u);
                        else a3[w + 1] = restrict2(r, kd, side ? n0 - 2 : 0, lj, lk, s_u);  // covered by fine zones
                      }
                      double aL, aR;
                      plm_zone(a3, aL, aR);
                      v = 0.5 * (a3[1] + (high_half ? aR : aL));
                    }
                  }
                  if (xp && (kd == 3 || fd == 1)) v = -v;   // ut^2, Bf^2 reverse across the pole
                  if (kind == 0) dst.P[c][b.idx(i, j, k)] = v;
                  else dst.Bf[fd][b.idx(i, j, k)] = v;
                }
              }
        }
      }
  }
}

// C-16: where a coarse and a fine block on the same time level share the x1 interface, the fine block's
// F^1 and the edge EMFs E_2, E_3 lying in the interface plane are authoritative: the coarse block
// overwrites its own with them before its update (equal face areas and edge lengths: plain copies).
static void interface_agreement(Grid& g, int tau) {
  for (Block& c : g.blocks) {
    if (c.tau != tau || c.lev1 != 0) continue;
    for (int side = 0; side < 2; side++) {
      const int qi = c.nbr[side ? 2 : 0][1][1];
      if (qi < 0) continue;
      const Block& q = g.blocks[qi];
      if (q.lev1 == c.lev1 || q.tau != c.tau) continue;
      const int ic = side ? c.n[0] : 0, iq = side ? 0 : q.n[0];
      for (int j = 0; j <= c.n[1]; j++)
        for (int k = 0; k <= c.n[2]; k++) {
          const size_t zc = c.idx(ic, j, k), zq = q.idx(iq, j, k);
          if (j < c.n[1] && k < c.n[2]) {
            for (int cc = 0; cc < 5; cc++) c.F[0][cc][zc] = q.F[0][cc][zq];
            if (g.par.entropy_backup) c.FK[0][zc] = q.FK[0][zq];   // C-18: the entropy flux is one more flux of the face
          }
          if (j < c.n[1]) c.Ee[1][zc] = q.Ee[1][zq];   // E2 on edges along x2 at (i-1/2, k-1/2)
          if (k < c.n[2]) c.Ee[2][zc] = q.Ee[2][zq];   // E3 on edges along x3 at (i-1/2, j-1/2)
        }
    }
  }
}

// C-15: the x1- and x2-face fluxes of a derefined row in the transverse phi-ghost layer (k = -1 and k = n3;
// they feed the edge EMFs of C-9 on the block's phi-boundary) must be the phi-neighbour's group means, not
// this block's own per-zone values: where rows with different factors meet, the mean changes the value.
// Same-level neighbours only (across time levels the LAT correction makes the shared edges agree).
static void deref_exchange_flux_layers(Grid& g, int tau) {
  if (g.par.n_deref <= 0) return;
  for (Block& b : g.blocks) {
    if (b.tau != tau) continue;
    const int n3 = b.n[2];
    for (int side = 0; side < 2; side++) {
      const int qi = b.nbr[1][1][side ? 2 : 0];
      if (qi < 0) continue;
      const Block& q = g.blocks[qi];
      if (q.tau != b.tau || q.lev1 != b.lev1) continue;
      const int kd = side ? n3 : -1, ks = side ? 0 : n3 - 1;
      for (int i = 0; i <= b.n[0]; i++)
        for (int j = 0; j <= b.n[1]; j++) {
          const int m = b.mrow[j + NG], M = std::max(m, b.mrow[j - 1 + NG]);
          const size_t zd = b.idx(i, j, kd), zs = q.idx(i, j, ks);
          if (m > 1 && j < b.n[1]) {
            for (int c = 0; c < 5; c++) b.F[0][c][zd] = q.F[0][c][zs];
            b.Ef[0][1][zd] = q.Ef[0][1][zs];
            b.Ef[0][2][zd] = q.Ef[0][2][zs];
          }
          if (M > 1 && i < b.n[0]) {
            for (int c = 0; c < 5; c++) b.F[1][c][zd] = q.F[1][c][zs];
            b.Ef[1][2][zd] = q.Ef[1][2][zs];
            b.Ef[1][0][zd] = q.Ef[1][0][zs];
          }
        }
    }
  }
}

// ---- one stage of C-12 on every block of one time level ------------------------------------------------
static void stage_level(Grid& g, int tau, bool corrector) {
  for (Block& b : g.blocks) {
    if (b.tau != tau) continue;
    Fields& src = corrector ? b.sh : b.sn;
    exchange_block(g, b, src, b.tb_u + (corrector ? b.dt_u / 2 : 0));
    exchange_refined(g, b, src, b.tb_u + (corrector ? b.dt_u / 2 : 0));
    fill_physical_bc(g.par, b, src);
    compute_Bc(b, src, false);
  }
  for (Block& b : g.blocks) {
    if (b.tau != tau) continue;
    Fields& src = corrector ? b.sh : b.sn;
    flux_pass(g.par, b, src);
    deref_fix_fluxes(g.par, b);
  }
  deref_exchange_flux_layers(g, tau);
  for (Block& b : g.blocks) {
    if (b.tau != tau) continue;
    Fields& src = corrector ? b.sh : b.sn;
    ct_edges(g.par, b, src);
    deref_fix_edges(g.par, b);
  }
  interface_agreement(g, tau);
  for (Block& b : g.blocks) {
    if (b.tau != tau) continue;
    Fields& src = corrector ? b.sh : b.sn;
    const double dtb = g.dt * (double)(b.dt_u / 2);      // dt_b = 2^tau dt_0
    if (corrector) {
      // C-17 registers: R1 = dt_b * (F, E) of this corrector; R2 accumulates the two steps that
      // make up one step of a neighbour on the next coarser level
      const bool first = (b.tb_u % (2 * b.dt_u)) == 0;
      const size_t n = b.size();
      for (int d = 0; d < 3; d++) {
        for (int c = 0; c < 5; c++)
          for (size_t z = 0; z < n; z++) {
            const double v = dtb * b.F[d][c][z];
            b.FA[d][c][z] = v;
            b.FA2[d][c][z] = first ? v : b.FA2[d][c][z] + v;
          }
        for (size_t z = 0; z < n; z++) {
          const double v = dtb * b.Ee[d][z];
          b.EA[d][z] = v;
          b.EA2[d][z] = first ? v : b.EA2[d][z] + v;
        }
        if (g.par.entropy_backup)   // C-18: the entropy flux is one more flux of the face
          for (size_t z = 0; z < n; z++) {
            const double v = dtb * b.FK[d][z];
            b.FKA[d][z] = v;
            b.FKA2[d][z] = first ? v : b.FKA2[d][z] + v;
          }
        b.ctop_last[d] = b.ctop[d];
      }
    }
    update(g.par, b, src, b.sn, corrector ? b.snew : b.sh, corrector ? dtb : 0.5 * dtb, g.stats);
  }
  if (corrector)
    for (Block& b : g.blocks)
      if (b.tau == tau) b.has_new = true;
}

// ---- C-17 correct(tau-1 -> tau) ---------------------------------------------------------------------
// For every block c on level tau with a neighbour on level tau-1 (across a face, edge or corner):
//  * edge EMFs on c's boundary that a finer block shares are replaced by the finer block's
//    time-integrated EMF; every active face of c touching a replaced edge is rebuilt from the base
//    field with the corrected EMFs; the normal field on a face shared with a finer block is copied;
//  * the flux difference on faces shared with a finer block is added to c's boundary zones;
//  * the touched zones are re-inverted.
static void correct_level(Grid& g, int tau) {
  const Params& par = g.par;
  for (Block& c : g.blocks) {
    if (c.tau != tau) continue;
    bool any = false;
    for (int a = 0; a < 27; a++) {
      const int q = (&c.nbr[0][0][0])[a];
      if (q >= 0 && g.blocks[q].tau == tau - 1) any = true;
    }
    if (!any) continue;
    const int str[3] = {c.e[1] * c.e[2], c.e[2], 1};
    const size_t n = c.size();
    std::vector<double> EC[3];
    std::vector<char> erep[3], ftouch[3], zmask(n, 0);
    std::vector<double> dU[5], dUS(n, 0.0);
    for (int d = 0; d < 3; d++) { EC[d] = c.EA[d]; erep[d].assign(n, 0); ftouch[d].assign(n, 0); }
    for (int cc = 0; cc < 5; cc++) dU[cc].assign(n, 0.0);
    // (1) replace boundary edge EMFs by the finer sharer's accumulated value
    for (int f = 0; f < 3; f++) {
      const int d = CYC[f][1], e = CYC[f][2];
      int hi[3] = {c.n[0], c.n[1], c.n[2]};
      hi[f] = c.n[f] - 1;
      for (int i = 0; i <= hi[0]; i++)
        for (int j = 0; j <= hi[1]; j++)
          for (int k = 0; k <= hi[2]; k++) {
            const int id[3] = {i, j, k};
            const int od = id[d] == 0 ? -1 : (id[d] == c.n[d] ? 1 : 0);
            const int oe = id[e] == 0 ? -1 : (id[e] == c.n[e] ? 1 : 0);
            if (od == 0 && oe == 0) continue;
            const int cand[3][2] = {{od, 0}, {0, oe}, {od, oe}};
            for (int t = 0; t < 3; t++) {
              if (cand[t][0] == 0 && cand[t][1] == 0) continue;
              int o[3] = {0, 0, 0};
              o[d] = cand[t][0]; o[e] = cand[t][1];
              const int qi = c.nbr[o[0] + 1][o[1] + 1][o[2] + 1];
              if (qi < 0) continue;
              const Block& q = g.blocks[qi];
              if (q.tau != tau - 1) continue;
              int lq[3] = {i, j, k};
              lq[d] -= o[d] * c.n[d];
              lq[e] -= o[e] * c.n[e];
              const size_t z = c.idx(i, j, k);
              EC[f][z] = q.EA2[f][q.idx(lq[0], lq[1], lq[2])];
              erep[f][z] = 1;
              break;
            }
          }
    }
    // (2) rebuild every active face touching a replaced edge: Bf = base - curl(EC)   (C-10 with dt E -> EC)
    for (int d = 0; d < 3; d++) {
      const int e = CYC[d][1], f = CYC[d][2];
      int hi[3] = {c.n[0] - 1, c.n[1] - 1, c.n[2] - 1};
      hi[d] = c.n[d];
      for (int i = 0; i <= hi[0]; i++)
        for (int j = 0; j <= hi[1]; j++)
          for (int k = 0; k <= hi[2]; k++) {
            const size_t z = c.idx(i, j, k);
            if (!(erep[f][z] || erep[f][z + str[e]] || erep[e][z] || erep[e][z + str[f]])) continue;
            if (d == 1 && c.pole2[j + NG]) continue;
            const double curl = (EC[f][z + str[e]] - EC[f][z]) / c.dx[e] - (EC[e][z + str[f]] - EC[e][z]) / c.dx[f];
            c.snew.Bf[d][z] = c.sn.Bf[d][z] - curl;
            ftouch[d][z] = 1;
          }
    }
    // (3) faces shared with a finer face-neighbour: copy its normal field, add the flux difference
    for (int d = 0; d < 3; d++)
      for (int side = 0; side < 2; side++) {
        int o[3] = {0, 0, 0};
        o[d] = side ? 1 : -1;
        const int qi = c.nbr[o[0] + 1][o[1] + 1][o[2] + 1];
        if (qi < 0) continue;
        const Block& q = g.blocks[qi];
        if (q.tau != tau - 1) continue;
        const int e = CYC[d][1], f = CYC[d][2];
        for (int p = 0; p < c.n[e]; p++)
          for (int r = 0; r < c.n[f]; r++) {
            int lc[3], lq[3], lz[3];
            lc[d] = side ? c.n[d] : 0; lc[e] = p; lc[f] = r;        // c's boundary face
            lq[d] = side ? 0 : q.n[d]; lq[e] = p; lq[f] = r;        // the same face in q
            lz[d] = side ? c.n[d] - 1 : 0; lz[e] = p; lz[f] = r;    // c's boundary zone
            const size_t zf = c.idx(lc[0], lc[1], lc[2]), zq = q.idx(lq[0], lq[1], lq[2]);
            const size_t zz = c.idx(lz[0], lz[1], lz[2]);
            c.snew.Bf[d][zf] = q.sn.Bf[d][zq];   // q has completed both steps: its sn is at c's new time
            ftouch[d][zf] = 1;
            for (int cc = 0; cc < 5; cc++) {
              const double dF = q.FA2[d][cc][zq] - c.FA[d][cc][zf];
              // U_new = U - (dt F_hi - dt F_lo)/dx: the high face enters with -, the low face with +
              dU[cc][zz] += (side ? -dF : dF) / c.dx[d];
            }
            if (par.entropy_backup) {
              const double dF = q.FKA2[d][zq] - c.FKA[d][zf];
              dUS[zz] += (side ? -dF : dF) / c.dx[d];
            }
            zmask[zz] = 1;
          }
      }
    // zones with a touched face
    for (int d = 0; d < 3; d++)
      for (int i = 0; i < c.n[0]; i++)
        for (int j = 0; j < c.n[1]; j++)
          for (int k = 0; k < c.n[2]; k++) {
            const size_t z = c.idx(i, j, k);
            if (ftouch[d][z] || ftouch[d][z + str[d]]) zmask[z] = 1;
          }
    // (4) re-invert: U = U(P^{n+1}, old B_c) + dU with the rebuilt B_c
    for (int i = 0; i < c.n[0]; i++)
      for (int j = 0; j < c.n[1]; j++) {
        const Geom& G = c.gc[c.idx2(i, j)];
        const double r = (par.metric == 1) ? std::exp(c.xc(0, i)) : 1.0;
        for (int k = 0; k < c.n[2]; k++) {
          const size_t z = c.idx(i, j, k);
          if (!zmask[z]) continue;
          double P[8], U[8], Bn[3], Pn[5];
          for (int cc = 0; cc < 5; cc++) P[cc] = c.snew.P[cc][z];
          for (int cc = 0; cc < 3; cc++) P[5 + cc] = c.snew.Bc[cc][z];
          State S;
          get_state(P, G, S);
          prim_to_U(P, S, G, par.gamma_ad, U);
          for (int cc = 0; cc < 5; cc++) U[cc] += dU[cc][z];
          for (int d = 0; d < 3; d++) {
            Bn[d] = (c.snew.Bf[d][z] + c.snew.Bf[d][z + str[d]]) / (2.0 * G.gdet);
            c.snew.Bc[d][z] = Bn[d];
          }
          int rc = con2prim(U, Bn, G, par.gamma_ad, P, Pn, nullptr);
          if (par.entropy_backup) {
            // C-18 / C-21 under LAT: the corrected rows go through the same chain as in the update.  kappa was reset from
            // the zone's new primitives, so its entropy row before the correction is its density row times kappa(P)
            if (rc != 0) {
              double Pa[5];
              if (con2prim_aitken(U, Bn, G, par.gamma_ad, P, Pa, nullptr) == 0) {
                for (int cc = 0; cc < 5; cc++) Pn[cc] = Pa[cc];
                rc = 0;
                g.stats.c2p_aitken++;
              }
            }
            if (rc != 0 || !(Pn[0] > 0.0) || !(Pn[1] >= 0.0)) {
              const double US = (U[0] - dU[0][z]) * entropy_kappa(P[0], P[1], par.gamma_ad) + dUS[z];
              double Pe[5];
              if (con2prim_entropy(U, US, Bn, G, par.gamma_ad, P, Pe, nullptr) == 0) {
                for (int cc = 0; cc < 5; cc++) Pn[cc] = Pe[cc];
                rc = 0;
                g.stats.c2p_entropy++;
              }
            }
          }
          if (rc != 0) {
            g.stats.c2p_fail++;
            for (int cc = 0; cc < 5; cc++) Pn[cc] = P[cc];
          }
          floors_and_ceiling(par, G, r, Pn, par.drift_floors ? Bn : nullptr, g.stats);
          for (int cc = 0; cc < 5; cc++) c.snew.P[cc][z] = Pn[cc];
        }
      }
    deref_sync_groups(par, c, c.snew);
  }
}

static void rotate_level(Grid& g, int tau) {
  for (Block& b : g.blocks) {
    if (b.tau != tau) continue;
    for (int c = 0; c < 5; c++) b.sn.P[c].swap(b.snew.P[c]);
    for (int c = 0; c < 3; c++) { b.sn.Bc[c].swap(b.snew.Bc[c]); b.sn.Bf[c].swap(b.snew.Bf[c]); }
    b.tb_u += b.dt_u;
    b.has_new = false;
  }
}

// C-17: advance(tau) = predictor, first half of the finer levels, corrector, second half, correction
static void advance(Grid& g, int tau) {
  stage_level(g, tau, false);
  if (tau > 0) advance(g, tau - 1);
  stage_level(g, tau, true);
  if (tau > 0) {
    advance(g, tau - 1);
    correct_level(g, tau);
  }
  rotate_level(g, tau);
}

// ---- time step and time levels (C-14, C-17) ---------------------------------------------------------------
static void assign_levels(Grid& g) {
  const Params& par = g.par;
  const int tmax = par.lat_max_level;
  if (tmax <= 0) {
    // global step: per-direction maximum over the whole grid, then the harmonic sum (C-14)
    double s = 0.0;
    for (int d = 0; d < 3; d++) {
      double m = 0.0;
      for (const Block& b : g.blocks) m = std::max(m, b.ctop_last[d] / b.dx[d]);
      s += m;
    }
    g.dt = par.cour / s;
    for (Block& b : g.blocks) { b.tau = 0; }
  } else {
    // per-block Courant step, levels in factors of 2 relative to the smallest
    std::vector<double> dtb(g.blocks.size());
    double dt0 = 1e300;
    for (size_t i = 0; i < g.blocks.size(); i++) {
      dtb[i] = dt_from_ctop(par, g.blocks[i]);
      dt0 = std::min(dt0, dtb[i]);
    }
    if (!g.forced_tau.empty()) {
      // test hook: prescribed levels; dt_0 is the largest step every block can take on its level
      dt0 = 1e300;
      for (size_t i = 0; i < g.blocks.size(); i++) {
        g.blocks[i].tau = std::min(tmax, std::max(0, g.forced_tau[i]));
        dt0 = std::min(dt0, dtb[i] / (double)(1 << g.blocks[i].tau));
      }
    } else {
      for (size_t i = 0; i < g.blocks.size(); i++) {
        int tau = 0;
        double lim = 2.0 * dt0;
        while (tau < tmax && dtb[i] >= lim) { tau++; lim *= 2.0; }
        g.blocks[i].tau = tau;
      }
    }
    // neighbours across faces, edges and corners differ by at most one level: lower until they do
    for (bool changed = true; changed;) {
      changed = false;
      std::vector<int> nt(g.blocks.size());
      for (size_t i = 0; i < g.blocks.size(); i++) {
        const Block& b = g.blocks[i];
        int t = b.tau;
        for (int a = 0; a < 27; a++) {
          const int q = (&b.nbr[0][0][0])[a];
          if (q >= 0) t = std::min(t, g.blocks[q].tau + 1);
        }
        for (int a = 0; a < 9; a++) {   // the blocks across a transmissive pole are neighbours too
          const int q = (&b.pnbr[0][0])[a];
          if (q >= 0) t = std::min(t, g.blocks[q].tau + 1);
        }
        nt[i] = t;
        if (t != b.tau) changed = true;
      }
      for (size_t i = 0; i < g.blocks.size(); i++) g.blocks[i].tau = nt[i];
    }
    g.dt = dt0;
  }
  for (Block& b : g.blocks) {
    b.tb_u = 0;
    b.dt_u = 2LL << b.tau;
    b.has_new = false;
  }
}

void blocks_initial_dt(Grid& g) {
  for (Block& b : g.blocks) { b.tau = 0; b.tb_u = 0; b.dt_u = 2; b.has_new = false; }
  for (Block& b : g.blocks) {
    exchange_block(g, b, b.sn, 0);
    exchange_refined(g, b, b.sn, 0);
    fill_physical_bc(g.par, b, b.sn);
    compute_Bc(b, b.sn, false);
  }
  for (Block& b : g.blocks) {
    flux_pass(g.par, b, b.sn);                 // C-14: one flux pass sets the first dt
    for (int d = 0; d < 3; d++) b.ctop_last[d] = b.ctop[d];
  }
  assign_levels(g);
}

void blocks_coarse_step(Grid& g) {
  const int tmax = std::max(0, g.par.lat_max_level);
  advance(g, tmax);
  g.t += g.dt * (double)(1 << tmax);
  assign_levels(g);
}

// ---- C-20 (the x1-only part): regridding ---------------------------------------------------------
// PAPER.md:73 "H-AMR allows the user to implement an arbitrary refinement criterion ... a cutoff on the maximum density in
// each block"; PAPER.md:71 blocks are split per dimension; "(de-)refinement ... including the divergence-free
// prolongation and restriction of magnetic fields (Balsara 2001)".  This grid has ONE refinement level along x1 whose
// block columns must be contiguous from the inner edge (C-16), so a regrid moves the outer edge of the refined region.
//
// Criterion: a block column wants refinement if any of its blocks holds a zone with rho >= rho_cut; the refined region
// is every column up to the outermost such column (the nesting rule of PAPER.md:73 with one level: no resolution jump
// greater than two exists).  Returned as the r_refine_max that selects exactly those columns; 0: none.
double blocks_refine_radius(const Grid& g, double rho_cut) {
  const Params& par = g.par;
  const int nb0 = par.nb[0] > 0 ? par.nb[0] : par.n[0];
  const int ncol = par.n[0] / nb0;
  int cmax = -1;
  for (const Block& b : g.blocks) {
    const int col = b.lev1 ? (int)(b.I0[0] / nb0) / 2 : (int)(b.I0[0] / nb0);
    double m = 0.0;
    for (int i = 0; i < b.n[0]; i++)
      for (int j = 0; j < b.n[1]; j++)
        for (int k = 0; k < b.n[2]; k++) m = std::max(m, b.sn.P[0][b.idx(i, j, k)]);
    if (m >= rho_cut) cmax = std::max(cmax, col);
  }
  if (cmax < 0) return 0.0;
  double lo = par.xmin[0], hi = par.xmax[0];
  if (par.metric == 1) { lo = std::log(lo); hi = std::log(hi); }
  const double edge = lo + (hi - lo) * (double)(cmax + 1) / (double)ncol;   // high edge of column cmax
  return par.metric == 1 ? std::exp(edge) : edge;
}

// Transfer of the state of `go` (all blocks at the same time: between coarse steps) onto the lattice of `gn`, which
// differs in r_refine_max only.  Per new block: same level as before -> copy; newly refined -> prolongation of the old
// coarse block; newly coarsened -> restriction of the two old fine blocks.
//   prolongation: hydro primitives piecewise linear in x1 with the MC-limited slope of the coarse values, evaluated a
//     quarter of a coarse zone off the coarse centre (the operator of the ghost fill, C-16); x1-faces: coincident ones
//     copied, the new one in the middle of a coarse zone is the MEAN of that zone's two x1-faces; x2- and x3-faces: both
//     children take the coarse zone's face value.  Each child then has the coarse zone's transverse divergence and, over
//     half the width, half of its x1 difference: the coarse zone's divergence, i.e. zero if that was (the lowest-order
//     member of Balsara 2001's divergence-free prolongation).
//   restriction: hydro primitives and transverse faces are the mean of the two fine values, x1-faces the coincident
//     fine faces: the coarse divergence is the mean of the two children's.
void blocks_regrid(Grid& go, Grid& gn) {
  const Params& par = go.par;
  const int nb0 = par.nb[0] > 0 ? par.nb[0] : par.n[0];
  const int ncol = par.n[0] / nb0;
  const int nref_o = go.nslot[0] - ncol, nref_n = gn.nslot[0] - ncol;
  if (nb0 % 2 != 0 && nref_o != nref_n) throw std::runtime_error("regrid needs an even nb[0]");
  // ghosts of the old state (the slopes of the prolongation read one zone beyond the block)
  for (Block& b : go.blocks) {
    exchange_block(go, b, b.sn, b.tb_u);
    exchange_refined(go, b, b.sn, b.tb_u);
    fill_physical_bc(go.par, b, b.sn);
  }
  auto old_block = [&](int slot0, int bj, int bk) -> const Block& {
    return go.blocks[go.lattice[((size_t)slot0 * go.nslot[1] + bj) * go.nslot[2] + bk]];
  };
  for (Block& b : gn.blocks) {
    const int n0 = b.n[0], n1 = b.n[1], n2 = b.n[2];
    const int col = b.lev1 ? (int)(b.I0[0] / nb0) / 2 : (int)(b.I0[0] / nb0);
    const int child = b.lev1 ? (int)(b.I0[0] / nb0) % 2 : 0;
    const bool old_fine = col < nref_o;
    Fields& d = b.sn;
    if ((b.lev1 != 0) == old_fine) {
      // ---- same level: copy
      const Block& q = old_block(old_fine ? 2 * col + child : col + nref_o, b.slot[1], b.slot[2]);
      for (int i = 0; i <= n0; i++)
        for (int j = 0; j <= n1; j++)
          for (int k = 0; k <= n2; k++) {
            const size_t z = b.idx(i, j, k);
            if (i < n0 && j < n1 && k < n2)
              for (int c = 0; c < 5; c++) d.P[c][z] = q.sn.P[c][z];
            if (j < n1 && k < n2) d.Bf[0][z] = q.sn.Bf[0][z];
            if (i < n0 && k < n2) d.Bf[1][z] = q.sn.Bf[1][z];
            if (i < n0 && j < n1) d.Bf[2][z] = q.sn.Bf[2][z];
          }
    } else if (b.lev1) {
      // ---- newly refined: prolongation of the old coarse block; this child covers its zones [h n0/2, (h+1) n0/2)
      const Block& q = old_block(col + nref_o, b.slot[1], b.slot[2]);
      const int c0 = child * (n0 / 2);
      for (int i = 0; i <= n0; i++)
        for (int j = 0; j <= n1; j++)
          for (int k = 0; k <= n2; k++) {
            const size_t z = b.idx(i, j, k);
            const int ic = c0 + i / 2;
            if (i < n0 && j < n1 && k < n2)
              for (int c = 0; c < 5; c++) {
                const double a3[3] = {q.sn.P[c][q.idx(ic - 1, j, k)], q.sn.P[c][q.idx(ic, j, k)], q.sn.P[c][q.idx(ic + 1, j, k)]};
                double aL, aR;
                plm_zone(a3, aL, aR);
                d.P[c][z] = 0.5 * (a3[1] + ((i & 1) ? aR : aL));
              }
            if (j < n1 && k < n2) {
              const int f2 = 2 * c0 + i;                 // the face's position in half coarse zones
              d.Bf[0][z] = (f2 % 2 == 0) ? q.sn.Bf[0][q.idx(f2 / 2, j, k)]
                                         : 0.5 * (q.sn.Bf[0][q.idx(f2 / 2, j, k)] + q.sn.Bf[0][q.idx(f2 / 2 + 1, j, k)]);
            }
            if (i < n0 && k < n2) d.Bf[1][z] = q.sn.Bf[1][q.idx(ic, j, k)];
            if (i < n0 && j < n1) d.Bf[2][z] = q.sn.Bf[2][q.idx(ic, j, k)];
          }
    } else {
      // ---- newly coarsened: restriction of the two old fine blocks
      for (int i = 0; i <= n0; i++) {
        const int hh = (i == n0) ? 1 : ((i < n0 / 2) ? 0 : 1);   // the child holding coarse zone i (coarse face n0: the second)
        const Block& q = old_block(2 * col + hh, b.slot[1], b.slot[2]);
        const int i0 = 2 * i - hh * n0;                   // first of the two fine zones / the coincident fine face
        for (int j = 0; j <= n1; j++)
          for (int k = 0; k <= n2; k++) {
            const size_t z = b.idx(i, j, k);
            if (i < n0 && j < n1 && k < n2)
              for (int c = 0; c < 5; c++) d.P[c][z] = 0.5 * (q.sn.P[c][q.idx(i0, j, k)] + q.sn.P[c][q.idx(i0 + 1, j, k)]);
            if (j < n1 && k < n2) d.Bf[0][z] = q.sn.Bf[0][q.idx(i0, j, k)];
            if (i < n0 && k < n2) d.Bf[1][z] = 0.5 * (q.sn.Bf[1][q.idx(i0, j, k)] + q.sn.Bf[1][q.idx(i0 + 1, j, k)]);
            if (i < n0 && j < n1) d.Bf[2][z] = 0.5 * (q.sn.Bf[2][q.idx(i0, j, k)] + q.sn.Bf[2][q.idx(i0 + 1, j, k)]);
          }
      }
    }
  }
  // C-15: on a phi-derefined grid the transfer keeps the group structure (every member of a group goes through the same
  // arithmetic on the same values) except for the last bit of the in-group x3-faces after a restriction (the mean of two
  // interpolated values is not bitwise the interpolation of the means): the invariant is imposed as after set_prims
  for (Block& b : gn.blocks) deref_project(gn.par, b, b.sn);
  gn.t = go.t;
  gn.have_state = true;
  blocks_initial_dt(gn);
}

}  // namespace orc
