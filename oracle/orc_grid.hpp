// ORACLE (test infrastructure) — block data structure and the per-block stage (C-5..C-14).
#pragma once
#include "orc.hpp"

namespace orc {

struct Fields {                    // one time level of one block ("flat arrays")
  std::vector<double> P[5];        // rho, u, ut1, ut2, ut3 at zone centres
  std::vector<double> Bc[3];       // cell-centred B^i (C-10)
  std::vector<double> Bf[3];       // densitised face field g*B^d on d-faces
  void alloc(size_t n) {
    for (auto& v : P) v.assign(n, 0.0);
    for (auto& v : Bc) v.assign(n, 0.0);
    for (auto& v : Bf) v.assign(n, 0.0);
  }
};

struct Block {
  int n[3];                        // active zones
  int e[3];                        // padded extents n + 2NG + 1 (the +1 holds the last face/edge)
  long long I0[3];                 // global index of local zone 0, in zones of this block's level
  int lev1;                        // x1 refinement level (0 or 1), C-16
  double dx[3];
  double x0[3];                    // internal-coordinate origin of the GLOBAL grid
  bool phys_lo[3], phys_hi[3];     // side lies on the domain boundary
  int tau;                         // LAT time level (C-17)
  std::vector<int> mrow;           // phi-derefinement factor per local x2 row incl. ghosts (C-15)

  std::vector<Geom> gc, gf1, gf2;  // 2-D tables over (i,j) incl. ghosts: centres, x1-, x2-faces
  std::vector<double> conn;        // Gamma at centres, 64 per (i,j)
  std::vector<char> pole2;         // x2-face row j lies on the polar axis

  Fields sn, sh, snew;             // time n, n+1/2 and the state being written
  // ---- block-structured grid (C-16, C-17; orc_blocks.cpp) ----
  int slot[3];                     // position in the block lattice (x1 slot, x2 block, x3 block)
  int nbr[3][3][3];                // neighbour block ids by offset (-1: outside the domain)
  // NEXT-1 on blocks that cut x3: the ghost rows beyond a transmissive pole lie in the block row half a turn
  // away; pnbr[o0 + 1][o2 + 1] is the block at (slot0 + o0, same slot1, slot2 + nslot2 / 2 + o2)
  bool xpole_lo, xpole_hi;
  int pnbr[3][3];
  long long tb_u, dt_u;            // LAT: time of sn and own step, in units of (finest dt)/2
  bool has_new;                    // snew holds the completed state at tb_u + dt_u
  std::vector<double> FA[3][5];    // flux register R1: dt_b * F of the latest corrector (C-17)
  std::vector<double> EA[3];       // EMF register R1: dt_b * E_edge of the latest corrector
  std::vector<double> FA2[3][5];   // R2: R1 summed over the two steps inside one step of the next
  std::vector<double> EA2[3];      //     coarser time level
  std::vector<double> FKA[3], FKA2[3];   // C-18 under LAT: the same two registers for the entropy flux
  double ctop_last[3];             // ctop of this block's most recent corrector (or initial) pass
  std::vector<double> K;           // C-18: kappa of the flux pass's source state, every zone incl. ghosts
  std::vector<double> FK[3];       // C-18: entropy fluxes on d-faces
  std::vector<double> Kadv;        // C-18: kappa the entropy row gives after the latest update (before it is reset)
  std::vector<double> F[3][5];     // hydro fluxes on d-faces
  std::vector<double> Ef[3][3];    // Ef[d][c]: E_c on d-faces, c != d (C-8)
  std::vector<double> Ee[3];       // edge EMFs (C-9)
  std::vector<double> Cc[3];       // centre EMFs (C-8)
  double ctop[3];

  size_t size() const { return (size_t)e[0] * e[1] * e[2]; }
  size_t idx(int i, int j, int k) const {
    return ((size_t)(i + NG) * e[1] + (j + NG)) * e[2] + (k + NG);
  }
  size_t idx2(int i, int j) const { return (size_t)(i + NG) * e[1] + (j + NG); }
  double xc(int d, int i) const { return x0[d] + ((double)(I0[d] + i) + 0.5) * dx[d]; }
  double xf(int d, int i) const { return x0[d] + (double)(I0[d] + i) * dx[d]; }
};

struct Stats { long long c2p_fail, rho_floor, u_floor, gam_ceil, c2p_entropy, c2p_aitken; };

struct Grid {
  Params par;
  std::vector<Block> blocks;
  double t, dt;                    // dt: the global step, or the finest-level step dt_0 under LAT
  bool have_state;
  Stats stats;
  std::string err;
  int nslot[3];                    // block lattice extents
  std::vector<int> lattice;        // block id by (slot1, slot2, slot3)
  bool multi;                      // more than one block, or any of deref / refine / LAT
  std::vector<int> forced_tau;     // test hook: fixed time levels instead of the Courant-based ones
};

// orc_blocks.cpp (C-15..C-17)
void blocks_build(Grid& g);                       // block lattice, neighbours, geometry
void blocks_exchange(Grid& g, int level, int stage_half);  // ghost fill of the level's stage source
void blocks_initial_dt(Grid& g);                  // flux pass on every block, first dt / levels
void blocks_coarse_step(Grid& g);                 // one (coarse) step: advance(tau_max)
double blocks_refine_radius(const Grid& g, double rho_cut);   // C-20: the refinement criterion as an r_refine_max
void blocks_regrid(Grid& go, Grid& gn);           // C-20: state of go onto the lattice of gn (built, differing in r_refine_max)

void block_init(const Params& par, Block& b);           // geometry tables, allocation
void fill_physical_bc(const Params& par, Block& b, Fields& s);
void compute_Bc(const Block& b, Fields& s, bool active_only);
void flux_pass(const Params& par, Block& b, const Fields& src);
void ct_edges(const Params& par, Block& b, const Fields& src);
// out may alias base (every zone/face reads only its own base value)
void update(const Params& par, Block& b, const Fields& src, const Fields& base, Fields& out,
            double dt, Stats& st);
double dt_from_ctop(const Params& par, const Block& b);
// C-15: the phi-ghost slots of a row with factor m are in GROUP units: ghost zone -g holds group -g (the
// neighbour's zones n3 - g m ...), ghost zone n3 - 1 + g holds group g - 1 beyond the edge (the neighbour's zone
// (g - 1) m); ghost x3-faces likewise hold group-boundary faces.  Returns the neighbour offset o2 and the x3
// index inside the neighbour.  m = 1: the ordinary ghost zones.  Needs n3 >= 3 m.
inline int deref_ghost_k(int k, int n3, int m, bool face3, int& o2) {
  const int hi = face3 ? n3 : n3 - 1;
  if (k < 0) { o2 = -1; return n3 + k * m; }
  if (k > hi) { o2 = 1; return face3 ? (k - n3) * m : (k - n3) * m; }
  o2 = 0;
  return k;
}
// C-15: an x2-face array (Bf2) follows the grouping of its FACE (the coarser of the two rows it separates), so
// its phi-ghost slots are in units of that grouping.  A zone row with factor m whose ghost slot k holds one of
// ITS groups finds the face value that covers that group in this slot of the face array with grouping M >= m.
inline int deref_face2_slot(int k, int n3, int m, int M) {
  if (M == m) return k;
  if (k < 0) { const int g = -k; return -((g * m + M - 1) / M); }     // group -g of the row lies in face group -ceil(g m / M)
  if (k >= n3) { const int g = k - n3; return n3 + (g * m) / M; }     // group g beyond the edge: face group floor(g m / M)
  return k;
}
// C-15 phi-derefinement (orc_grid.cpp)
int deref_factor_of_row(const Params& par, long long J);
void deref_fix_fluxes(const Params& par, Block& b);
void deref_fix_edges(const Params& par, Block& b);
void deref_sync_groups(const Params& par, Block& b, Fields& s);
void deref_project(const Params& par, Block& b, Fields& s);
// Bc: the zone's cell-centred field (read only with par.drift_floors; may be NULL)
void floors_and_ceiling(const Params& par, const Geom& G, double r, double P[5], const double* Bc, Stats& st);

}  // namespace orc
