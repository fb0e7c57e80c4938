// ORACLE (test infrastructure) — grid driver and the C entry points that tests/_orc.py loads with
// ctypes.  Time stepping follows DESIGN.md §3 C-12 (predictor/corrector = one zone-cycle,
// PAPER.md:41, 141) and C-14 (harmonic Courant dt, PAPER.md:93 fn. 2).
#include "orc_grid.hpp"
#include <algorithm>
#include <cstring>
#include <new>
#include <stdexcept>

namespace orc {

static const double PI = 3.14159265358979323846;

static bool params_ok(const Params& p, std::string& why) {
  for (int d = 0; d < 3; d++) {
    if (p.n[d] < 1) { why = "n[d] < 1"; return false; }
    if (!(p.xmax[d] > p.xmin[d])) { why = "xmax <= xmin"; return false; }
    if ((p.bc_lo[d] == 0) != (p.bc_hi[d] == 0)) { why = "periodic must be set on both sides"; return false; }
  }
  if (p.metric == 1 && !(p.xmin[0] > 0.0)) { why = "r_in <= 0"; return false; }
  if (p.bc_lo[1] == 3 || p.bc_hi[1] == 3) {   // NEXT-1 transmissive pole
    // blocks that cut x3 come in an even number, so that half a turn is a whole number of blocks
    const bool cut_ok = p.nb[2] <= 0 || p.nb[2] == p.n[2] || (p.n[2] % p.nb[2] == 0 && (p.n[2] / p.nb[2]) % 2 == 0);
    if (p.bc_lo[1] != p.bc_hi[1] || p.bc_lo[2] != 0 || p.n[2] % 2 != 0 || !cut_ok) {
      why = "transmissive poles need both poles, a periodic even x3 and blocks that span x3 or cut it into an even number";
      return false;
    }
  }
  if (!(p.gamma_ad > 1.0) || !(p.cour > 0.0)) { why = "gamma_ad/cour"; return false; }
  if (p.entropy_backup || p.drift_floors) {  // C-18, C-19: one block, or blocks that step together on one lattice level
    if ((p.entropy_backup & ~1) || (p.drift_floors & ~1)) { why = "entropy_backup / drift_floors are 0 or 1"; return false; }
    if (p.entropy_backup && !(p.gamma_ad < 2.0)) { why = "the entropy inversion needs gamma_ad < 2"; return false; }
  }
  return true;
}

// internal-coordinate extents: x1 = ln r for the Kerr-Schild map
static void internal_extent(const Params& p, double lo[3], double hi[3]) {
  for (int d = 0; d < 3; d++) { lo[d] = p.xmin[d]; hi[d] = p.xmax[d]; }
  if (p.metric == 1) { lo[0] = std::log(p.xmin[0]); hi[0] = std::log(p.xmax[0]); }
}

static Grid* grid_new(const Params& par) {
  Grid* g = new Grid();
  g->par = par;
  g->t = 0.0;
  g->dt = 0.0;
  g->have_state = false;
  g->stats = Stats{0, 0, 0, 0, 0, 0};
  if (!params_ok(par, g->err)) { delete g; return nullptr; }
  g->multi = par.nb[0] > 0 || par.nb[1] > 0 || par.nb[2] > 0 || par.n_deref > 0 ||
             par.lat_max_level > 0 || par.r_refine_max > 0.0;
  if (g->multi) {
    try { blocks_build(*g); } catch (const std::exception& e) { delete g; return nullptr; }
    return g;
  }
  g->nslot[0] = g->nslot[1] = g->nslot[2] = 1;
  double lo[3], hi[3];
  internal_extent(par, lo, hi);
  g->blocks.resize(1);
  Block& b = g->blocks[0];
  for (int d = 0; d < 3; d++) {
    b.n[d] = par.n[d];
    b.I0[d] = 0;
    b.dx[d] = (hi[d] - lo[d]) / par.n[d];
    b.x0[d] = lo[d];
    b.phys_lo[d] = b.phys_hi[d] = true;
  }
  b.lev1 = 0;
  b.tau = 0;
  b.xpole_lo = b.xpole_hi = false;
  block_init(par, b);
  return g;
}

// one stage of C-12 on the single block
static void stage(Grid& g, Fields& src, const Fields& base, Fields& out, double dts) {
  Block& b = g.blocks[0];
  fill_physical_bc(g.par, b, src);
  compute_Bc(b, src, false);
  flux_pass(g.par, b, src);
  ct_edges(g.par, b, src);
  update(g.par, b, src, base, out, dts, g.stats);
}

static void full_step(Grid& g) {
  Block& b = g.blocks[0];
  const double dt = g.dt;
  stage(g, b.sn, b.sn, b.sh, 0.5 * dt);     // predictor: src = base = n, dt/2 -> n+1/2
  stage(g, b.sh, b.sn, b.snew, dt);         // corrector: src = n+1/2, base = n, dt -> n+1
  for (int c = 0; c < 5; c++) b.sn.P[c].swap(b.snew.P[c]);
  for (int c = 0; c < 3; c++) { b.sn.Bc[c].swap(b.snew.Bc[c]); b.sn.Bf[c].swap(b.snew.Bf[c]); }
  g.t += dt;
  g.dt = dt_from_ctop(g.par, b);            // C-14: corrector ctop of step n sets dt of step n+1
}

static bool state_finite(const Grid& g) {
  for (const Block& b : g.blocks)
    for (int i = 0; i < b.n[0]; i++)
      for (int j = 0; j < b.n[1]; j++)
        for (int k = 0; k < b.n[2]; k++) {
          const size_t z = b.idx(i, j, k);
          for (int c = 0; c < 5; c++)
            if (!std::isfinite(b.sn.P[c][z])) return false;
        }
  return true;
}

// dense <-> block transfers.  Global arrays (orc_set_prims etc.) exist for grids without x1
// refinement: block b holds the sub-box starting at I0.  stag = -1 zone-centred, else the face dim.
static void scatter(const Grid& g, Block& b, std::vector<double>& dst, const double* src, int stag,
                    bool global) {
  int m[3] = {b.n[0], b.n[1], b.n[2]}, M[3] = {g.par.n[0], g.par.n[1], g.par.n[2]};
  if (stag >= 0) { m[stag] += 1; M[stag] += 1; }
  for (int i = 0; i < m[0]; i++)
    for (int j = 0; j < m[1]; j++)
      for (int k = 0; k < m[2]; k++) {
        double v = global ? src[((size_t)(b.I0[0] + i) * M[1] + (b.I0[1] + j)) * M[2] + (b.I0[2] + k)]
                          : src[((size_t)i * m[1] + j) * m[2] + k];
        if (stag == 1 && b.pole2[j + NG]) v = 0.0;      // C-12: Bf2 on the pole face is 0
        dst[b.idx(i, j, k)] = v;
      }
}
static void gather(const Grid& g, const Block& b, const std::vector<double>& src, double* dst, int stag,
                   bool global) {
  int m[3] = {b.n[0], b.n[1], b.n[2]}, M[3] = {g.par.n[0], g.par.n[1], g.par.n[2]};
  if (stag >= 0) { m[stag] += 1; M[stag] += 1; }
  for (int i = 0; i < m[0]; i++)
    for (int j = 0; j < m[1]; j++)
      for (int k = 0; k < m[2]; k++) {
        const double v = src[b.idx(i, j, k)];
        if (global) dst[((size_t)(b.I0[0] + i) * M[1] + (b.I0[1] + j)) * M[2] + (b.I0[2] + k)] = v;
        else dst[((size_t)i * m[1] + j) * m[2] + k] = v;
      }
}
static bool has_refinement(const Grid& g) {
  for (const Block& b : g.blocks) if (b.lev1) return true;
  return false;
}

}  // namespace orc

using namespace orc;

extern "C" {

int orc_sizeof_params() { return (int)sizeof(Params); }

void* orc_grid_create(const Params* p) {
  if (!p) return nullptr;
  try { return grid_new(*p); } catch (const std::bad_alloc&) { return nullptr; }
}

void orc_grid_destroy(void* h) { delete (Grid*)h; }

// C-20: the refinement criterion (max density per block column >= rho_cut) as the r_refine_max it asks for
int orc_refine_radius(void* h, double rho_cut, double* r_new) {
  Grid& g = *(Grid*)h;
  if (!g.multi || !g.have_state || !r_new) return 1;
  *r_new = blocks_refine_radius(g, rho_cut);
  return 0;
}
// C-20: a new grid with r_refine_max = r_new holding the state of h (which stays valid); NULL if the grid is not a
// block grid between coarse steps or the new lattice is not admissible
void* orc_regrid(void* h, double r_new) {
  Grid& go = *(Grid*)h;
  if (!go.multi || !go.have_state) return nullptr;
  Params p = go.par;
  p.r_refine_max = r_new;
  Grid* gn = nullptr;
  try {
    gn = grid_new(p);
    if (!gn) return nullptr;
    if (!gn->multi) { delete gn; return nullptr; }
    blocks_regrid(go, *gn);
  } catch (const std::exception&) {
    delete gn;
    return nullptr;
  }
  return gn;
}

// hydro[c]: N1*N2*N3 active zones, x3 fastest.  bface[d]: d-faces, extent n[d]+1 along d; NULL -> 0.
int orc_set_prims(void* h, const double* const hydro[5], const double* const bface[3]) {
  Grid& g = *(Grid*)h;
  if (g.multi) {
    if (has_refinement(g)) return 1;   // refined grids are set block by block
    for (Block& b : g.blocks) {
      for (int c = 0; c < 5; c++) scatter(g, b, b.sn.P[c], hydro[c], -1, true);
      for (int d = 0; d < 3; d++) {
        std::fill(b.sn.Bf[d].begin(), b.sn.Bf[d].end(), 0.0);
        if (bface && bface[d]) scatter(g, b, b.sn.Bf[d], bface[d], d, true);
      }
      deref_project(g.par, b, b.sn);
    }
    blocks_initial_dt(g);
    g.t = 0.0;
    g.have_state = true;
    g.stats = Stats{0, 0, 0, 0, 0, 0};
    return state_finite(g) ? 0 : 5;
  }
  Block& b = g.blocks[0];
  for (int c = 0; c < 5; c++)
    for (int i = 0; i < b.n[0]; i++)
      for (int j = 0; j < b.n[1]; j++)
        for (int k = 0; k < b.n[2]; k++)
          b.sn.P[c][b.idx(i, j, k)] = hydro[c][((size_t)i * b.n[1] + j) * b.n[2] + k];
  for (int d = 0; d < 3; d++) {
    int m[3] = {b.n[0], b.n[1], b.n[2]};
    m[d] += 1;
    std::fill(b.sn.Bf[d].begin(), b.sn.Bf[d].end(), 0.0);
    if (!bface || !bface[d]) continue;
    for (int i = 0; i < m[0]; i++)
      for (int j = 0; j < m[1]; j++)
        for (int k = 0; k < m[2]; k++) {
          double v = bface[d][((size_t)i * m[1] + j) * m[2] + k];
          if (d == 1 && b.pole2[j + NG]) v = 0.0;   // C-12: Bf2 on the pole face is 0
          b.sn.Bf[d][b.idx(i, j, k)] = v;
        }
  }
  fill_physical_bc(g.par, b, b.sn);
  compute_Bc(b, b.sn, false);
  flux_pass(g.par, b, b.sn);               // C-14: one flux pass sets dt of step 0
  g.dt = dt_from_ctop(g.par, b);
  g.t = 0.0;
  g.have_state = true;
  g.stats = Stats{0, 0, 0, 0, 0, 0};
  return state_finite(g) ? 0 : 5;
}

int orc_step(void* h, int nsteps, double* t_out, double* dt_last) {
  Grid& g = *(Grid*)h;
  if (!g.have_state) return 4;
  double dtl = 0.0;
  for (int s = 0; s < nsteps; s++) {
    dtl = g.dt;
    if (g.multi) blocks_coarse_step(g);
    else full_step(g);
  }
  if (t_out) *t_out = g.t;
  if (dt_last) *dt_last = dtl;
  return state_finite(g) ? 0 : 5;
}

double orc_get_dt(void* h) { return ((Grid*)h)->dt; }
double orc_get_t(void* h) { return ((Grid*)h)->t; }
void orc_set_dt(void* h, double dt) { ((Grid*)h)->dt = dt; }

int orc_get_prims(void* h, double* const prims[8]) {
  Grid& g = *(Grid*)h;
  if (g.multi) {
    if (has_refinement(g)) return 1;
    for (const Block& b : g.blocks)
      for (int c = 0; c < 8; c++) gather(g, b, (c < 5) ? b.sn.P[c] : b.sn.Bc[c - 5], prims[c], -1, true);
    return 0;
  }
  Block& b = g.blocks[0];
  for (int c = 0; c < 8; c++) {
    const std::vector<double>& a = (c < 5) ? b.sn.P[c] : b.sn.Bc[c - 5];
    for (int i = 0; i < b.n[0]; i++)
      for (int j = 0; j < b.n[1]; j++)
        for (int k = 0; k < b.n[2]; k++)
          prims[c][((size_t)i * b.n[1] + j) * b.n[2] + k] = a[b.idx(i, j, k)];
  }
  return 0;
}

int orc_get_bface(void* h, double* const bface[3]) {
  Grid& g = *(Grid*)h;
  if (g.multi) {
    if (has_refinement(g)) return 1;
    // a face shared by two blocks is written twice; orc_bface_mismatch() reports whether the copies agree
    for (const Block& b : g.blocks)
      for (int d = 0; d < 3; d++) gather(g, b, b.sn.Bf[d], bface[d], d, true);
    return 0;
  }
  Block& b = g.blocks[0];
  for (int d = 0; d < 3; d++) {
    int m[3] = {b.n[0], b.n[1], b.n[2]};
    m[d] += 1;
    for (int i = 0; i < m[0]; i++)
      for (int j = 0; j < m[1]; j++)
        for (int k = 0; k < m[2]; k++)
          bface[d][((size_t)i * m[1] + j) * m[2] + k] = b.sn.Bf[d][b.idx(i, j, k)];
  }
  return 0;
}

// C-11: max over zones of |div| / sum_d (|Bf+| + |Bf-|)/(2 dx^d), zones with a denominator below
// 1e-12 of its global maximum count 0.
int orc_divb(void* h, double* out) {
  Grid& g = *(Grid*)h;
  double denmax = 0.0;
  for (int pass = 0; pass < 2; pass++) {
    double worst = 0.0;
    for (const Block& b : g.blocks) {
    const int str[3] = {b.e[1] * b.e[2], b.e[2], 1};
    for (int i = 0; i < b.n[0]; i++)
      for (int j = 0; j < b.n[1]; j++)
        for (int k = 0; k < b.n[2]; k++) {
          const size_t z = b.idx(i, j, k);
          double div = 0.0, den = 0.0;
          for (int d = 0; d < 3; d++) {
            const double lo = b.sn.Bf[d][z], hi = b.sn.Bf[d][z + str[d]];
            div += (hi - lo) / b.dx[d];
            den += (std::fabs(hi) + std::fabs(lo)) / (2.0 * b.dx[d]);
          }
          if (pass == 0) denmax = std::max(denmax, den);
          else if (den > 1e-12 * denmax) worst = std::max(worst, std::fabs(div) / den);
        }
    }
    if (pass == 1) *out = worst;
  }
  return 0;
}

int orc_get_stats(void* h, long long counts[4]) {
  Grid& g = *(Grid*)h;
  counts[0] = g.stats.c2p_fail; counts[1] = g.stats.rho_floor;
  counts[2] = g.stats.u_floor;  counts[3] = g.stats.gam_ceil;
  g.stats.c2p_fail = g.stats.rho_floor = g.stats.u_floor = g.stats.gam_ceil = 0;
  return 0;
}
// zones, since the last call, whose primitives came from the entropy inversion (C-18)
int orc_get_backup_count(void* h, long long* n) {
  Grid& g = *(Grid*)h;
  *n = g.stats.c2p_entropy;
  g.stats.c2p_entropy = 0;
  return 0;
}
// zones, since the last call, whose primitives came from the Aitken-accelerated inversion (C-21)
int orc_get_aitken_count(void* h, long long* n) {
  Grid& g = *(Grid*)h;
  *n = g.stats.c2p_aitken;
  g.stats.c2p_aitken = 0;
  return 0;
}
// kappa = (entropy row) / (density row) of the latest update, before it is reset from the primitives; active zones
int orc_get_kadv(void* h, double* out) {
  Grid& g = *(Grid*)h;
  Block& b = g.blocks[0];
  if (!g.par.entropy_backup || b.Kadv.empty()) return 1;
  for (int i = 0; i < b.n[0]; i++)
    for (int j = 0; j < b.n[1]; j++)
      for (int k = 0; k < b.n[2]; k++) out[((size_t)i * b.n[1] + j) * b.n[2] + k] = b.Kadv[b.idx(i, j, k)];
  return 0;
}

// the same for block bi of a block grid (block-local dense array)
int orc_get_block_kadv(void* h, int bi, double* out) {
  Grid& g = *(Grid*)h;
  if (bi < 0 || bi >= (int)g.blocks.size()) return 1;
  Block& b = g.blocks[bi];
  if (!g.par.entropy_backup || b.Kadv.empty()) return 1;
  for (int i = 0; i < b.n[0]; i++)
    for (int j = 0; j < b.n[1]; j++)
      for (int k = 0; k < b.n[2]; k++) out[((size_t)i * b.n[1] + j) * b.n[2] + k] = b.Kadv[b.idx(i, j, k)];
  return 0;
}

// Face fluxes / EMFs of the most recent flux pass, for face-by-face parity (debug access).
// which: 0..4 hydro flux F^d[c]; 5,6 the two face EMFs E_e, E_f with (d,e,f) cyclic; 7 the entropy flux (C-18).
int orc_get_face(void* h, int d, int which, double* out) {
  Grid& g = *(Grid*)h;
  Block& b = g.blocks[0];
  static const int CY[3][3] = {{0, 1, 2}, {1, 2, 0}, {2, 0, 1}};
  if (which == 7 && !g.par.entropy_backup) return 1;
  const std::vector<double>& a = (which == 7) ? b.FK[d] : (which < 5) ? b.F[d][which] : b.Ef[d][CY[d][which - 4]];
  int m[3] = {b.n[0], b.n[1], b.n[2]};
  m[d] += 1;
  for (int i = 0; i < m[0]; i++)
    for (int j = 0; j < m[1]; j++)
      for (int k = 0; k < m[2]; k++) out[((size_t)i * m[1] + j) * m[2] + k] = a[b.idx(i, j, k)];
  return 0;
}

// Conserved totals over active zones: sum of U[c] dV for c = 0..4 (P10), U from sn.
int orc_totals(void* h, double tot[5]) {
  Grid& g = *(Grid*)h;
  for (int c = 0; c < 5; c++) tot[c] = 0.0;
  for (const Block& b : g.blocks) {
  const double dV = b.dx[0] * b.dx[1] * b.dx[2];
  for (int i = 0; i < b.n[0]; i++)
    for (int j = 0; j < b.n[1]; j++) {
      const Geom& G = b.gc[b.idx2(i, j)];
      for (int k = 0; k < b.n[2]; k++) {
        const size_t z = b.idx(i, j, k);
        double P[8], U[8];
        for (int c = 0; c < 5; c++) P[c] = b.sn.P[c][z];
        for (int c = 0; c < 3; c++) P[5 + c] = b.sn.Bc[c][z];
        State S;
        get_state(P, G, S);
        prim_to_U(P, S, G, g.par.gamma_ad, U);
        for (int c = 0; c < 5; c++) tot[c] += U[c] * dV;
      }
    }
  }
  return 0;
}

// ---- block enumeration (C-16, C-17) -------------------------------------------------------------
int orc_num_blocks(void* h) { return (int)((Grid*)h)->blocks.size(); }
// x_lo: internal coordinates of the block's low corner
int orc_block_info(void* h, int bi, double x_lo[3], double dx[3], int n[3], int* tau, int* lev1) {
  Grid& g = *(Grid*)h;
  if (bi < 0 || bi >= (int)g.blocks.size()) return 1;
  const Block& b = g.blocks[bi];
  for (int d = 0; d < 3; d++) { x_lo[d] = b.xf(d, 0); dx[d] = b.dx[d]; n[d] = b.n[d]; }
  *tau = b.tau;
  *lev1 = b.lev1;
  return 0;
}
int orc_set_block_prims(void* h, int bi, const double* const hydro[5], const double* const bface[3]) {
  Grid& g = *(Grid*)h;
  if (!g.multi || bi < 0 || bi >= (int)g.blocks.size()) return 1;
  Block& b = g.blocks[bi];
  for (int c = 0; c < 5; c++) scatter(g, b, b.sn.P[c], hydro[c], -1, false);
  for (int d = 0; d < 3; d++) {
    std::fill(b.sn.Bf[d].begin(), b.sn.Bf[d].end(), 0.0);
    if (bface && bface[d]) scatter(g, b, b.sn.Bf[d], bface[d], d, false);
  }
  return 0;
}
// test hook: prescribe the LAT level of every block (NULL: back to Courant-based levels)
int orc_force_levels(void* h, const int* tau) {
  Grid& g = *(Grid*)h;
  g.forced_tau.clear();
  if (tau) g.forced_tau.assign(tau, tau + g.blocks.size());
  return 0;
}
// after every block has been set: ghost fill, first dt and time levels
int orc_blocks_commit(void* h) {
  Grid& g = *(Grid*)h;
  if (!g.multi) return 1;
  for (Block& b : g.blocks) deref_project(g.par, b, b.sn);
  blocks_initial_dt(g);
  g.t = 0.0;
  g.have_state = true;
  g.stats = Stats{0, 0, 0, 0, 0, 0};
  return state_finite(g) ? 0 : 5;
}
int orc_get_block_prims(void* h, int bi, double* const prims[8]) {
  Grid& g = *(Grid*)h;
  if (bi < 0 || bi >= (int)g.blocks.size()) return 1;
  const Block& b = g.blocks[bi];
  for (int c = 0; c < 8; c++) gather(g, b, (c < 5) ? b.sn.P[c] : b.sn.Bc[c - 5], prims[c], -1, false);
  return 0;
}
int orc_get_block_bface(void* h, int bi, double* const bface[3]) {
  Grid& g = *(Grid*)h;
  if (bi < 0 || bi >= (int)g.blocks.size()) return 1;
  const Block& b = g.blocks[bi];
  for (int d = 0; d < 3; d++) gather(g, b, b.sn.Bf[d], bface[d], d, false);
  return 0;
}
// largest difference between the two copies of a face field value on faces shared by two blocks
double orc_bface_mismatch(void* h) {
  Grid& g = *(Grid*)h;
  double worst = 0.0;
  for (const Block& b : g.blocks)
    for (int d = 0; d < 3; d++) {
      int o[3] = {0, 0, 0};
      o[d] = 1;
      const int qi = b.nbr[o[0] + 1][o[1] + 1][o[2] + 1];
      if (qi < 0 || g.blocks[qi].lev1 != b.lev1) continue;
      const Block& q = g.blocks[qi];
      const int e = (d + 1) % 3, f = (d + 2) % 3;
      for (int p = 0; p < b.n[e]; p++)
        for (int r = 0; r < b.n[f]; r++) {
          int lb[3], lq[3];
          lb[d] = b.n[d]; lb[e] = p; lb[f] = r;
          lq[d] = 0; lq[e] = p; lq[f] = r;
          worst = std::max(worst, std::fabs(b.sn.Bf[d][b.idx(lb[0], lb[1], lb[2])] -
                                            q.sn.Bf[d][q.idx(lq[0], lq[1], lq[2])]));
        }
    }
  return worst;
}

// ---- per-zone entry points for the pins -------------------------------------------------------
void orc_geom_at(int metric, double a, double x1, double x2, Geom* G) { geom_at(metric, a, x1, x2, *G); }
void orc_conn_at(int metric, double a, double x1, double x2, double* conn64) {
  conn_at(metric, a, x1, x2, *(double(*)[4][4][4])conn64);
}
void orc_gcov_derivs(int metric, double a, double x1, double x2, double* g, double* d1, double* d2) {
  gcov_and_derivs(metric, a, x1, x2, *(double(*)[4][4])g, *(double(*)[4][4])d1, *(double(*)[4][4])d2);
}
void orc_prim_to_UF(const double* P, const Geom* G, double gam, int dir, double* U, double* F) {
  State S;
  get_state(P, *G, S);
  prim_to_U(P, S, *G, gam, U);
  if (dir >= 1) prim_to_F(P, S, *G, gam, dir, F);
}
void orc_state(const double* P, const Geom* G, double* ucon, double* ucov, double* bcon, double* bcov,
               double* bsq) {
  State S;
  get_state(P, *G, S);
  for (int m = 0; m < 4; m++) { ucon[m] = S.ucon[m]; ucov[m] = S.ucov[m]; bcon[m] = S.bcon[m]; bcov[m] = S.bcov[m]; }
  *bsq = S.bsq;
}
void orc_wavespeeds(const double* P, const Geom* G, double gam, int dir, double* vmin, double* vmax) {
  State S;
  get_state(P, *G, S);
  wavespeeds(P, S, *G, gam, dir, *vmin, *vmax);
}
void orc_source(const double* P, const Geom* G, const double* conn64, double gam, double* S5) {
  State S;
  get_state(P, *G, S);
  source(P, S, *G, *(const double(*)[4][4][4])conn64, gam, S5);
}
int orc_con2prim(const double* U5, const double* Bc, const Geom* G, double gam, const double* Pguess,
                 double* Pout, int* iters) {
  return con2prim(U5, Bc, *G, gam, Pguess, Pout, iters);
}
// floors and Lorentz-factor ceiling of C-13 on one zone at radius r; counts3: rho-floor, u-floor, ceiling hits
// Bc3: the zone's field (read with par->drift_floors; may be NULL)
void orc_floors(const Params* par, const Geom* G, double r, double* P5, const double* Bc3, long long* counts3) {
  Stats st = {0, 0, 0, 0, 0, 0};
  floors_and_ceiling(*par, *G, r, P5, Bc3, st);
  counts3[0] = st.rho_floor; counts3[1] = st.u_floor; counts3[2] = st.gam_ceil;
}
int orc_con2prim_aitken(const double* U5, const double* Bc, const Geom* G, double gam, const double* Pguess,
                        double* Pout, int* iters) {
  return con2prim_aitken(U5, Bc, *G, gam, Pguess, Pout, iters);
}
int orc_con2prim_entropy(const double* U5, double US, const double* Bc, const Geom* G, double gam,
                         const double* Pguess, double* Pout, int* iters) {
  return con2prim_entropy(U5, US, Bc, *G, gam, Pguess, Pout, iters);
}
void orc_entropy_UF(const double* P, const Geom* G, double gam, int dir, double* US, double* FS) {
  State S;
  get_state(P, *G, S);
  entropy_UF(P, S, *G, gam, dir, *US, *FS);
}
void orc_ppm_zone(const double* a5, double* aL, double* aR) { ppm_zone(a5, *aL, *aR); }
void orc_plm_zone(const double* a3, double* aL, double* aR) { plm_zone(a3, *aL, *aR); }
void orc_hll(const double* UL, const double* UR, const double* FL, const double* FR, double cmin,
             double cmax, double* F) { hll(UL, UR, FL, FR, cmin, cmax, F); }

}  // extern "C"

// ---- debug access for the CT pins (P8): run fill + flux + CT on the current state --------------
extern "C" {
int orc_debug_emf(void* h) {
  Grid& g = *(Grid*)h;
  Block& b = g.blocks[0];
  fill_physical_bc(g.par, b, b.sn);
  compute_Bc(b, b.sn, false);
  flux_pass(g.par, b, b.sn);
  ct_edges(g.par, b, b.sn);
  return 0;
}
// edge EMF E_f on edges (extent n+1 along the two directions != f), x3 fastest
int orc_get_edge(void* h, int f, double* out) {
  Grid& g = *(Grid*)h;
  Block& b = g.blocks[0];
  int m[3] = {b.n[0] + 1, b.n[1] + 1, b.n[2] + 1};
  m[f] -= 1;
  for (int i = 0; i < m[0]; i++)
    for (int j = 0; j < m[1]; j++)
      for (int k = 0; k < m[2]; k++)
        out[((size_t)i * m[1] + j) * m[2] + k] = b.Ee[f][b.idx(i, j, k)];
  return 0;
}
// centre EMF E^c_f on active zones
int orc_get_centre_emf(void* h, int f, double* out) {
  Grid& g = *(Grid*)h;
  Block& b = g.blocks[0];
  for (int i = 0; i < b.n[0]; i++)
    for (int j = 0; j < b.n[1]; j++)
      for (int k = 0; k < b.n[2]; k++)
        out[((size_t)i * b.n[1] + j) * b.n[2] + k] = b.Cc[f][b.idx(i, j, k)];
  return 0;
}
void orc_get_ctop(void* h, double* c3) {
  Grid& g = *(Grid*)h;
  for (int d = 0; d < 3; d++) c3[d] = g.blocks[0].ctop[d];
}
}

// failure-code histogram of con2prim since creation (debug): codes 1..4

// number of OpenMP threads the oracle's loops use (reported by bench.py's cpu_baseline leg)
#include <omp.h>
extern "C" int orc_omp_threads() { return omp_get_max_threads(); }
// the timing harness runs the oracle on one core and on all of them
extern "C" void orc_set_threads(int n) { omp_set_num_threads(n > 0 ? n : omp_get_num_procs()); }

// debug access for the boundary pins: fills the ghosts of the single block's current state and returns one
// full padded array (kind 0..4 hydro, 5..7 Bc, 8..10 Bf), extents n + 2 NG + 1 per dimension, x3 fastest
extern "C" int orc_get_padded(void* h, int kind, double* out) {
  Grid& g = *(Grid*)h;
  if (g.multi || kind < 0 || kind > 10) return 1;
  Block& b = g.blocks[0];
  fill_physical_bc(g.par, b, b.sn);
  compute_Bc(b, b.sn, false);
  const std::vector<double>& a = kind < 5 ? b.sn.P[kind] : (kind < 8 ? b.sn.Bc[kind - 5] : b.sn.Bf[kind - 8]);
  std::memcpy(out, a.data(), a.size() * sizeof(double));
  return 0;
}
