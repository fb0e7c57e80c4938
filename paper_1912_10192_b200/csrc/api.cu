// api.cu — the C-ABI of libhamr (include/hamr.h): grid life cycle, state in/out, the step driver.
// The time integrator is the 2nd-order predictor/corrector of PAPER.md:41, 141 (C-12):
//   predictor: src = base = state n,  dt/2 -> n+1/2 ;  corrector: src = n+1/2, base = n, dt -> n+1,
// each stage = ghost fill -> reconstruct+HLL x3 -> CT EMFs -> B update + source + update + inversion.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>
#include "../../include/hamr_debug.h"
#include "hamr_host.h"

using namespace hamr;

namespace {

constexpr int N_STATE_ARR = 11, N_ARR = 3 * N_STATE_ARR + 15 + 3 + 3 + 3 + 3;
constexpr int N_REG_ARR = 15 + 3;  // LAT flux / EMF registers (C-17)

bool is_block_grid(const hamr_params& p) { return p.nb[0] > 0 || p.nb[1] > 0 || p.nb[2] > 0 || p.lat_max_level > 0; }
bool params_ok(const hamr_params& p, std::string& why);

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

bool params_ok(const hamr_params& p, std::string& why) {
  for (int d = 0; d < 3; d++) {
    if (p.n[d] < 1) { why = "n[d] < 1"; return false; }
    if (!(p.xmax[d] > p.xmin[d])) { why = "xmax <= xmin"; return false; }
    if (p.bc_lo[d] < 0 || p.bc_lo[d] > 3 || p.bc_hi[d] < 0 || p.bc_hi[d] > 3) { why = "bad boundary kind"; return false; }
    if (d != 1 && (p.bc_lo[d] == HAMR_BC_POLAR_TRANSMIT || p.bc_hi[d] == HAMR_BC_POLAR_TRANSMIT)) {
      why = "the transmissive polar boundary applies to x2 only";
      return false;
    }
    if ((p.bc_lo[d] == HAMR_BC_PERIODIC) != (p.bc_hi[d] == HAMR_BC_PERIODIC)) {
      why = "periodic must be set on both sides";
      return false;
    }
    if (p.bc_lo[d] != HAMR_BC_PERIODIC && p.n[d] < NG) { why = "non-periodic dimension needs n >= 3"; return false; }
  }
  if (p.bc_lo[1] == HAMR_BC_POLAR_TRANSMIT || p.bc_hi[1] == HAMR_BC_POLAR_TRANSMIT) {
    // blocks that cut x3 come in an even number: half a turn is then a whole number of blocks
    const bool cut_ok = p.nb[2] <= 0 || p.nb[2] == p.n[2] || (p.n[2] % p.nb[2] == 0 && (p.n[2] / p.nb[2]) % 2 == 0);
    if (p.bc_lo[1] != p.bc_hi[1] || p.bc_lo[2] != HAMR_BC_PERIODIC || p.n[2] % 2 != 0 || !cut_ok) {
      why = "transmissive poles need both poles, a periodic even x3 and blocks that span x3 or cut it into an even number";
      return false;
    }
  }
  if (p.metric != HAMR_METRIC_MINKOWSKI && p.metric != HAMR_METRIC_KERR_SCHILD) { why = "bad metric"; return false; }
  if (p.map != HAMR_MAP_DEFAULT &&
      p.map != (p.metric == HAMR_METRIC_KERR_SCHILD ? HAMR_MAP_LOGR_SPHERICAL : HAMR_MAP_CARTESIAN)) {
    why = "coordinate map and metric do not go together (Minkowski: Cartesian, Kerr-Schild: log-r spherical)";
    return false;
  }
  if (p.metric == HAMR_METRIC_KERR_SCHILD) {
    // the x2-faces J = 0 and J = N2 are treated as the polar axis (no flux, no normal field, pole-edge EMFs 0):
    // x2 must span exactly (0, pi) with a polar boundary on both sides
    const double pi = 3.14159265358979323846;
    const bool polar_lo = p.bc_lo[1] == HAMR_BC_POLAR_REFLECT || p.bc_lo[1] == HAMR_BC_POLAR_TRANSMIT;
    const bool polar_hi = p.bc_hi[1] == HAMR_BC_POLAR_REFLECT || p.bc_hi[1] == HAMR_BC_POLAR_TRANSMIT;
    if (std::fabs(p.xmin[1]) > 1e-12 || std::fabs(p.xmax[1] - pi) > 1e-12 * pi || !polar_lo || !polar_hi) {
      why = "the spherical map needs x2 = (0, pi) with a polar boundary kind on both sides";
      return false;
    }
  }
  if (p.recon != HAMR_RECON_PPM && p.recon != HAMR_RECON_PLM_MC) { why = "bad recon"; return false; }
  if (p.metric == HAMR_METRIC_KERR_SCHILD && !(p.xmin[0] > 0.0)) { why = "r_in <= 0"; return false; }
  if (!(p.gamma_ad > 1.0) || !(p.cour > 0.0) || !(p.gamma_max > 1.0)) { why = "gamma_ad / cour / gamma_max"; return false; }
  if (p.r_refine_max > 0.0 && !is_block_grid(p)) { why = "x1 refinement needs a block grid (nb)"; return false; }
  if (p.n_deref < 0 || p.n_deref > 4) { why = "n_deref must be 0..4"; return false; }
  if (p.n_deref > 0) {
    // C-15: the strided x3 stencil of a derefined row wraps inside the grid / block
    if (p.bc_lo[2] != HAMR_BC_PERIODIC) { why = "phi-derefinement needs a periodic x3"; return false; }
    // groups never straddle blocks and a ghost depth of 3 groups fits one neighbour; factors are powers of two
    const int nb3 = p.nb[2] > 0 ? p.nb[2] : p.n[2];
    for (int t = 0; t < p.n_deref; t++) {
      const int f = p.deref_factor[t];
      if (f < 1 || f > 16 || (f & (f - 1)) != 0 || nb3 % f != 0 || nb3 < 3 * f) {
        why = "deref factor must be a power of two <= 16 that divides nb[2], with 3 factor <= nb[2]";
        return false;
      }
    }
  }
  if (p.lat_max_level < 0 || p.lat_max_level > 3) { why = "lat_max_level must be 0..3"; return false; }
  if ((p.entropy_backup & ~1) || (p.drift_floors & ~1)) { why = "entropy_backup / drift_floors are 0 or 1"; return false; }
  if (p.entropy_backup || p.drift_floors) {   // NEXT-2 (C-18, C-19): one block, or blocks that step together on one lattice level
    if (p.entropy_backup && !(p.gamma_ad < 2.0)) { why = "the entropy inversion needs gamma_ad < 2"; return false; }
  }
  if (is_block_grid(p)) {
    int ns[3], bn[3];
    if (p.nb[0] < 0 || p.nb[1] < 0 || p.nb[2] < 0 || blk_count(p, ns, bn) <= 0) {
      why = "block size must divide n and be >= 3";
      return false;
    }
  }
  return true;
}

// Layout of one padded block (monolithic grid: the one block).  On a block grid every array holds nblk
// blocks of blen doubles back to back and the geometry tables are global.
struct GridShape {
  int nblk;        // 0: monolithic
  int blen;        // doubles per block per array
  int te1, te2;    // extents of the geometry tables
  int nlev;        // x1 refinement levels carrying a table set (1 or 2, C-16)
  int narr;        // fp64 arrays of Lay::len doubles
};

bool make_layout(const hamr_params& p, Lay& L, GridShape& G) {
  int ns[3], bn[3] = {p.n[0], p.n[1], p.n[2]};
  G.nblk = is_block_grid(p) ? blk_count(p, ns, bn) : 0;
  for (int d = 0; d < 3; d++) L.n[d] = bn[d];
  L.e1 = bn[0] + 2 * NG + 1;
  L.e2 = bn[1] + 2 * NG + 1;
  L.p3 = (int)align_up((size_t)bn[2] + 2 * NG + 1, 16);
  L.S2 = L.p3;
  L.S1 = L.e2 * L.p3;
  L.off0 = ((long long)NG * L.e2 + NG) * L.p3 + NG + LEAD;
  const long long blen = (long long)align_up((size_t)L.e1 * L.e2 * L.p3 + 32, 32);
  L.len = blen * (G.nblk > 0 ? G.nblk : 1);
  if (L.len >= (1LL << 31)) return false;   // kernels index one array with 32-bit offsets
  G.blen = (int)blen;
  G.nlev = (G.nblk > 0 && blk_has_refinement(p)) ? 2 : 1;
  G.te1 = G.nlev * p.n[0] + 2 * NG + 1;   // the level-1 table is indexed in fine zones
  G.te2 = p.n[1] + 2 * NG + 1;
  L.n2d = G.te1 * G.te2;
  G.narr = N_ARR + ((G.nblk > 0 && p.lat_max_level > 0) ? N_REG_ARR + (p.entropy_backup ? 3 : 0) : 0) + (p.entropy_backup ? 4 : 0);
  return true;
}

struct ArenaPlan {
  size_t arr, tabs, recs, scal, cnt, peer, stage, blk, mrow, total;
  size_t stage_doubles;
};

ArenaPlan plan_arena(const hamr_params& p, const Lay& L, const GridShape& G) {
  ArenaPlan a;
  size_t off = 0;
  a.arr = off; off += (size_t)G.narr * L.len * 8;
  a.tabs = off; off += align_up((size_t)G.nlev * ((size_t)2 * G.te1 * 8), 256);   // floor tables
  a.recs = off; off += align_up((size_t)G.nlev * (NREC_C + 3 * NREC_F) * L.n2d * 8, 256);   // geometry records
  a.scal = off; off += 256;
  a.cnt = off; off += 256;
  a.peer = off; off += align_up(sizeof(PeerTab), 256);   // NEXT-4: neighbour-slab table (unused on other grids)
  a.stage_doubles = (size_t)8 * (p.n[0] + 1) * (p.n[1] + 1) * (p.n[2] + 1);
  // block-by-block state: every block has its own staging slot, so hamr_set_block_prims need not wait for the
  // previous block's copies (the stream is synchronised once, in hamr_blocks_commit)
  if (G.nblk > 0)
    a.stage_doubles = std::max(a.stage_doubles, (size_t)G.nblk * 8 * (L.n[0] + 1) * (L.n[1] + 1) * (L.n[2] + 1));
  a.stage = off; off += align_up(a.stage_doubles * 8, 256);
  a.blk = off; off += G.nblk > 0 ? blk_table_bytes(G.nblk, (long long)L.e1 * L.e2 * (L.n[2] + 2 * NG + 1)) : 0;
  a.mrow = off; off += p.n_deref > 0 ? align_up((size_t)G.te2 * sizeof(int), 256) : 0;
  a.total = off;
  return a;
}

void destroy_aux(hamr_grid* g) {
  if (!g->aux[0]) return;
  cudaStreamSynchronize(g->aux[0]);
  cudaStreamSynchronize(g->aux[1]);
  cudaStreamDestroy(g->aux[0]);
  cudaStreamDestroy(g->aux[1]);
  cudaEventDestroy(g->ev_fork);
  cudaEventDestroy(g->ev_join[0]);
  cudaEventDestroy(g->ev_join[1]);
  g->aux[0] = g->aux[1] = nullptr;
}

int fail(hamr_grid* g, int code, const char* what, cudaError_t e = cudaSuccess) {
  if (g) {
    g->err = what;
    if (e != cudaSuccess) { g->err += ": "; g->err += cudaGetErrorString(e); }
  }
  return code;
}

#define CK(call)                                                    \
  do {                                                              \
    cudaError_t e_ = (call);                                        \
    if (e_ != cudaSuccess) return fail(g, HAMR_ECUDA, #call, e_);   \
  } while (0)

// An x1 slab of a global grid (NEXT-4): zones [i_lo, i_lo + n1) of n1_global; p carries the slab's n[0] and the
// GLOBAL extents and boundary kinds.
struct SlabSpec { int i_lo, n1_global; };

bool slab_ok(const hamr_params& gp, int i_lo, int n1, std::string& why) {
  if (!params_ok(gp, why)) return false;
  if (is_block_grid(gp) || gp.r_refine_max > 0.0) { why = "a slab is cut from a grid of one block"; return false; }
  if (i_lo < 0 || n1 < NG || i_lo + n1 > gp.n[0]) { why = "a slab needs 0 <= i_lo, n1 >= 3, i_lo + n1 <= n[0]"; return false; }
  return true;
}

int create_common(const hamr_params* p, void* arena, size_t arena_bytes, void* stream, bool own,
                  hamr_grid** out, const SlabSpec* slab = nullptr) {
  if (out) *out = nullptr;
  if (!p || !out) return HAMR_EINVAL;
  std::string why;
  if (!params_ok(*p, why)) return HAMR_EINVAL;
  hamr_grid* g = new (std::nothrow) hamr_grid();
  if (!g) return HAMR_ENOMEM;
  g->par = *p;
  Dev& D = g->D;
  std::memset(&D, 0, sizeof(D));
  GridShape gs;
  if (!make_layout(*p, D.L, gs)) { delete g; return HAMR_EINVAL; }
  const ArenaPlan ap = plan_arena(*p, D.L, gs);
  g->bh.on = false;
  g->bh.nblk = 0;
  g->bh.h_ctop = nullptr;
  g->bh.h_ints = nullptr;
  g->own_arena = own;
  g->own_stream = own;
  g->arena = nullptr;
  g->stream = nullptr;
  g->aux[0] = g->aux[1] = nullptr;
  g->cemf_done = false;
  g->h_pinned = nullptr;
  g->have_state = false;
  g->out_staged = false;
  g->blocks_open = false;
  g->dead = false;
  g->launches = 0;
  g->prof = false;
  g->ev_used = 0;
  g->step_graph[0] = g->step_graph[1] = nullptr;
  g->graph_launches = 0;
  g->plain_steps = 0;
  g->sharded = slab != nullptr;
  g->n1_global = slab ? slab->n1_global : p->n[0];
  std::memset(&g->peers, 0, sizeof(g->peers));
  g->shard_committed = false;
  g->shard_stage = 0;
  for (int a = 0; a < 2; a++) for (int b = 0; b < 2; b++) g->stage_graph[a][b] = nullptr;
  g->isn = 0; g->ish = 1; g->inew = 2;
  cudaError_t e;
  if (own) {
    if ((e = cudaStreamCreateWithFlags(&g->stream, cudaStreamNonBlocking)) != cudaSuccess) { delete g; return HAMR_ECUDA; }
    if ((e = cudaMalloc(&g->arena, ap.total)) != cudaSuccess) {
      cudaStreamDestroy(g->stream);
      delete g;
      return e == cudaErrorMemoryAllocation ? HAMR_ENOMEM : HAMR_ECUDA;
    }
    g->arena_bytes = ap.total;
  } else {
    if (!arena || ((uintptr_t)arena & 255) != 0) { delete g; return HAMR_EINVAL; }
    if (arena_bytes < ap.total) { delete g; return HAMR_ENOMEM; }
    g->arena = arena;
    g->arena_bytes = arena_bytes;
    g->stream = (cudaStream_t)stream;
  }
  // side streams and events of the fork / join in launch_flux_on; without them the sweeps run one after the other
  if (cudaStreamCreateWithFlags(&g->aux[0], cudaStreamNonBlocking) != cudaSuccess ||
      cudaStreamCreateWithFlags(&g->aux[1], cudaStreamNonBlocking) != cudaSuccess ||
      cudaEventCreateWithFlags(&g->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&g->ev_join[0], cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&g->ev_join[1], cudaEventDisableTiming) != cudaSuccess) {
    g->aux[0] = g->aux[1] = nullptr;
    cudaGetLastError();
  }
  g->ev_input = nullptr;
  if (cudaEventCreateWithFlags(&g->ev_input, cudaEventDisableTiming) != cudaSuccess) {
    g->ev_input = nullptr;
    cudaGetLastError();
  }
  if ((e = cudaMallocHost((void**)&g->h_pinned, 64 * sizeof(double))) != cudaSuccess) {
    if (g->ev_input) cudaEventDestroy(g->ev_input);
    destroy_aux(g);
    if (own) { cudaFree(g->arena); cudaStreamDestroy(g->stream); }
    delete g;
    return HAMR_ECUDA;
  }
  // internal coordinates: x1 = ln r on the Kerr-Schild map
  double lo[3], hi[3];
  for (int d = 0; d < 3; d++) { lo[d] = p->xmin[d]; hi[d] = p->xmax[d]; }
  if (p->metric == HAMR_METRIC_KERR_SCHILD) { lo[0] = std::log(p->xmin[0]); hi[0] = std::log(p->xmax[0]); }
  D.metric = p->metric;
  D.recon = p->recon;
  for (int d = 0; d < 3; d++) {
    D.bc_lo[d] = p->bc_lo[d];
    D.bc_hi[d] = p->bc_hi[d];
    D.dx[d] = (hi[d] - lo[d]) / (d == 0 ? g->n1_global : p->n[d]);
    D.x0[d] = lo[d];
  }
  D.ioff = slab ? slab->i_lo : 0;
  D.a = p->a; D.gam = p->gamma_ad; D.cour = p->cour; D.gamma_max = p->gamma_max;
  D.rho_fl_coef = p->rho_fl_coef; D.rho_fl_pow = p->rho_fl_pow;
  D.u_fl_coef = p->u_fl_coef; D.u_fl_pow = p->u_fl_pow;

  char* base = (char*)g->arena;
  double* arr = (double*)(base + ap.arr);
  int ia = 0;
  auto next = [&]() { return arr + (size_t)(ia++) * D.L.len; };
  for (int s = 0; s < 3; s++) {
    for (int c = 0; c < 5; c++) g->s[s].P[c] = next();
    for (int c = 0; c < 3; c++) g->s[s].Bc[c] = next();
    for (int c = 0; c < 3; c++) g->s[s].Bf[c] = next();
  }
  for (int d = 0; d < 3; d++) for (int c = 0; c < 5; c++) D.F[d][c] = next();
  for (int d = 0; d < 3; d++) D.EfA[d] = next();
  for (int d = 0; d < 3; d++) D.EfB[d] = next();
  for (int d = 0; d < 3; d++) D.Ee[d] = next();
  for (int d = 0; d < 3; d++) D.Cc[d] = next();
  if (gs.nblk > 0 && p->lat_max_level > 0) {
    for (int d = 0; d < 3; d++) for (int c = 0; c < 5; c++) D.B.FA2[d][c] = next();
    for (int d = 0; d < 3; d++) D.B.EA2[d] = next();
    if (p->entropy_backup) for (int d = 0; d < 3; d++) D.B.FKA2[d] = next();   // C-18 under LAT
  }
  D.entropy = p->entropy_backup;
  D.drift = p->drift_floors;
  if (D.entropy) {   // C-18: kappa of the stage source and the entropy flux per direction
    D.K = next();
    for (int d = 0; d < 3; d++) D.FK[d] = next();
  }
  D.B.nblk = gs.nblk;
  D.B.blen = gs.blen;
  D.B.ge2 = gs.te2;
  D.B.n2g = p->n[1];
  // floor tables [level][rho | u], geometry records [level][centres | x1-faces | x2-faces | x3-faces]
  D.B.flev = 2 * gs.te1;
  double* rfl = (double*)(base + ap.tabs);
  double* ufl = rfl + gs.te1;
  D.rho_fl = rfl; D.u_fl = ufl;
  double* gcA = (double*)(base + ap.recs);
  double* gf1A = gcA + (size_t)NREC_C * D.L.n2d;
  double* gf2A = gf1A + (size_t)NREC_F * D.L.n2d;
  double* gf3A = gf2A + (size_t)NREC_F * D.L.n2d;
  D.gcA = gcA; D.gf1A = gf1A; D.gf2A = gf2A; D.gf3A = gf3A;
  D.B.tlevA = (NREC_C + 3 * NREC_F) * D.L.n2d;
  D.scal = (double*)(base + ap.scal);
  D.cnt = (unsigned long long*)(base + ap.cnt);
  D.peer = slab ? (const PeerTab*)(base + ap.peer) : nullptr;
  g->stage = (double*)(base + ap.stage);
  g->stage_doubles = ap.stage_doubles;

  e = cudaMemsetAsync(g->arena, 0, ap.total, g->stream);
  if (e == cudaSuccess) {
    launch_geometry_tab(g, gs.te1, gs.te2, D.dx[0], p->n[1], rfl, ufl, gcA, gf1A, gf2A, gf3A);
    if (gs.nlev > 1)   // C-16: the refined level's tables, dx1 / 2
      launch_geometry_tab(g, gs.te1, gs.te2, 0.5 * D.dx[0], p->n[1], rfl + D.B.flev, ufl + D.B.flev, gcA + D.B.tlevA,
                          gf1A + D.B.tlevA, gf2A + D.B.tlevA, gf3A + D.B.tlevA);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess && gs.nblk > 0 && blk_setup(g, base + ap.blk) != HAMR_OK) e = cudaErrorUnknown;
  if (e == cudaSuccess && p->n_deref > 0) {   // C-15: derefinement factor per global x2 row incl. ghosts
    std::vector<int> mrow(gs.te2);
    bool any = false;
    for (int t = 0; t < gs.te2; t++) { mrow[t] = deref_row_factor(*p, (long long)t - NG); any = any || mrow[t] > 1; }
    if (any) {
      e = cudaMemcpyAsync(base + ap.mrow, mrow.data(), (size_t)gs.te2 * sizeof(int), cudaMemcpyHostToDevice, g->stream);
      if (e == cudaSuccess) e = cudaStreamSynchronize(g->stream);
      D.mrow = (const int*)(base + ap.mrow);
    }
  }
  if (e == cudaSuccess) e = cudaStreamSynchronize(g->stream);
  if (e != cudaSuccess) {
    destroy_aux(g);
    cudaFreeHost(g->h_pinned);
    if (g->bh.h_ctop) cudaFreeHost(g->bh.h_ctop);
    if (g->bh.h_ints) cudaFreeHost(g->bh.h_ints);
    if (own) { cudaFree(g->arena); cudaStreamDestroy(g->stream); }
    delete g;
    return HAMR_ECUDA;
  }
  *out = g;
  return HAMR_OK;
}

// reads n device scalars into host memory (synchronises)
int read_scal(hamr_grid* g, int first, int n, double* out) {
  CK(cudaMemcpyAsync(g->h_pinned, g->D.scal + first, n * sizeof(double), cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  for (int c = 0; c < n; c++) out[c] = g->h_pinned[c];
  return HAMR_OK;
}

int check_state(hamr_grid* g) {  // after a sync point: non-finite flag, sticky CUDA errors
  unsigned long long* h = (unsigned long long*)(g->h_pinned + 32);
  CK(cudaMemcpyAsync(h, g->D.cnt + N_NONFINITE, sizeof(unsigned long long), cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  CK(cudaGetLastError());
  if (*h != 0) {
    g->dead = true;
    return fail(g, HAMR_ENONFINITE, "non-finite primitives detected");
  }
  return HAMR_OK;
}

void enqueue_stage(hamr_grid* g, const Fields& src, const Fields& base, const Fields& out, double dtfac,
                   bool same, bool want_ctop) {
  launch_ghosts(g, src, false);
  launch_flux(g, src, want_ctop, true);
  launch_ct(g, src);
  launch_deref_fix_edges(g, g->D);
  launch_update(g, src, base, out, dtfac, same);
  launch_deref_sync(g, g->D, out, out);
}

void enqueue_step(hamr_grid* g) {
  const Fields& sn = g->s[g->isn];
  const Fields& sh = g->s[g->ish];
  const Fields& sw = g->s[g->inew];
  enqueue_stage(g, sn, sn, sh, 0.5, true, false);
  enqueue_stage(g, sh, sn, sw, 1.0, false, true);
  const int tmp = g->isn; g->isn = g->inew; g->inew = tmp;
  launch_dt(g, 1);  // C-14: the corrector's ctop of step n sets dt of step n+1
}

// One step of a monolithic grid.  The 15 launches of a step are captured once per buffer parity into a CUDA graph and
// replayed (every kernel argument is fixed for a grid: dt and the Courant maxima live on the device); the first step
// runs launch by launch (it also sets the per-kernel attributes and occupancy caches, which must not happen under
// capture), and so does every step while the per-kernel timers are on.
int step_once(hamr_grid* g) {
  // (the legacy default stream cannot be captured: a grid created on it keeps launching kernel by kernel)
  if (g->prof || g->plain_steps < 1 || g->stream == nullptr || g->stream == cudaStreamLegacy) {
    enqueue_step(g);
    g->plain_steps++;
    return HAMR_OK;
  }
  const int par = g->isn == 0 ? 0 : 1;
  if (!g->step_graph[par]) {
    const int isn = g->isn, ish = g->ish, inew = g->inew;
    const long long l0 = g->launches;
    cudaGraph_t graph = nullptr;
    CK(cudaStreamBeginCapture(g->stream, cudaStreamCaptureModeThreadLocal));
    enqueue_step(g);
    cudaError_t e = cudaStreamEndCapture(g->stream, &graph);
    g->isn = isn; g->ish = ish; g->inew = inew;      // the capture enqueued nothing: the state has not moved
    g->graph_launches = g->launches - l0;
    g->launches = l0;
    if (e == cudaSuccess) e = cudaGraphInstantiate(&g->step_graph[par], graph, 0);
    if (graph) cudaGraphDestroy(graph);
    if (e != cudaSuccess) return fail(g, HAMR_ECUDA, "capturing the step as a CUDA graph", e);
  }
  CK(cudaGraphLaunch(g->step_graph[par], g->stream));
  g->launches += g->graph_launches;
  const int tmp = g->isn; g->isn = g->inew; g->inew = tmp;
  return HAMR_OK;
}

// dev: device pointers (no staging, no wait).  nowait (host pointers): the copies and kernels are enqueued and the call
// returns; the caller's arrays must stay unchanged until hamr_wait_input (or any later wait on the stream) has returned
int set_prims_common(hamr_grid* g, const double* const hydro[5], const double* const bface[3], bool dev, bool nowait = false) {
  if (!g) return HAMR_EINVAL;
  if (g->dead) return fail(g, HAMR_ESTATE, "grid unusable after a non-finite state");
  if (!hydro) return fail(g, HAMR_EINVAL, "hydro is NULL");
  for (int c = 0; c < 5; c++) if (!hydro[c]) return fail(g, HAMR_EINVAL, "hydro[c] is NULL");
  const bool blk = g->bh.on;
  const int* N = g->par.n;
  g->out_staged = false;
  if (blk && g->bh.refined) return fail(g, HAMR_ESTATE, "a grid with x1 refinement is set block by block (hamr_set_block_prims)");
  if (blk) {
    g->isn = 0; g->ish = 1; g->inew = 2;
    CK(cudaMemsetAsync(g->D.B.cur, 0, (size_t)g->bh.nblk * sizeof(int), g->stream));
  }
  const Fields& sn = g->s[g->isn];
  const size_t nz = (size_t)N[0] * N[1] * N[2];
  // host arrays: ALL copies first, then the pack kernels (a copy behind a kernel on the same stream would leave the
  // host link idle while that kernel waits for SMs another grid is using)
  const double* srcs[8];
  size_t off = 5 * nz;
  for (int c = 0; c < 5; c++) {
    srcs[c] = hydro[c];
    if (!dev) {
      double* st = stage_take(g) + (size_t)c * nz;
      CK(cudaMemcpyAsync(st, hydro[c], nz * 8, cudaMemcpyHostToDevice, g->stream));
      srcs[c] = st;
    }
  }
  for (int d = 0; d < 3; d++) {
    int m[3] = {N[0], N[1], N[2]};
    m[d] += 1;
    const size_t nf = (size_t)m[0] * m[1] * m[2];
    srcs[5 + d] = (bface && bface[d]) ? bface[d] : nullptr;
    if (srcs[5 + d] && !dev) {
      if (off + nf > g->stage_doubles) return fail(g, HAMR_ENOMEM, "staging buffer too small");
      double* st = stage_take(g) + off;
      CK(cudaMemcpyAsync(st, srcs[5 + d], nf * 8, cudaMemcpyHostToDevice, g->stream));
      srcs[5 + d] = st;
      off += nf;
    }
  }
  if (nowait && g->ev_input) CK(cudaEventRecord(g->ev_input, g->stream));   // every input array has left the host
  for (int c = 0; c < 5; c++) {
    if (blk) blk_pack(g, srcs[c], c, -1, false);
    else launch_pack(g, srcs[c], sn.P[c], -1, false);
  }
  for (int d = 0; d < 3; d++) {
    if (blk) blk_pack(g, srcs[5 + d], 5 + d, d, d == 1);
    else launch_pack(g, srcs[5 + d], sn.Bf[d], d, d == 1);
  }
  CK(cudaMemsetAsync(g->D.scal, 0, NSCAL * sizeof(double), g->stream));
  CK(cudaMemsetAsync(g->D.cnt, 0, NCNT * sizeof(unsigned long long), g->stream));
  if (g->sharded) {
    // NEXT-4: the ghost fill reads the neighbour slabs, which may not hold their state yet: hamr_shard_commit does the
    // rest once every slab has been set
    launch_deref_project(g, g->D, sn, sn);
    launch_deref_sync(g, g->D, sn, sn);
    g->have_state = false;
    g->shard_committed = false;
    launch_check_finite(g, sn);
    CK(cudaGetLastError());
    if (dev || nowait) return HAMR_OK;
    return check_state(g);
  }
  if (blk) {
    const int rc = blk_initial(g);
    if (rc != HAMR_OK) return fail(g, rc, "block grid initialisation failed");
    blk_check_finite(g);
  } else {
    launch_deref_project(g, g->D, sn, sn);
    launch_deref_sync(g, g->D, sn, sn);
    launch_ghosts(g, sn, true);
    launch_flux(g, sn, true);   // C-14: one flux pass sets dt of step 0
    launch_dt(g, 0);
    launch_check_finite(g, sn);
  }
  g->have_state = true;
  CK(cudaGetLastError());
  if (dev || nowait) return HAMR_OK;
  return check_state(g);
}

// kind (block grids): 0..4 P, 5..7 Bc, 8..10 Bf of the current state
int get_dense(hamr_grid* g, const double* padded, double* out, int stag, bool dev, size_t stage_off, int kind = -1) {
  const int* N = g->par.n;
  int m[3] = {N[0], N[1], N[2]};
  if (stag >= 0) m[stag] += 1;
  const size_t nf = (size_t)m[0] * m[1] * m[2];
  if (g->bh.on && kind < 0) return fail(g, HAMR_ESTATE, "not available on a block-structured grid");
  if (g->bh.on && g->bh.refined) return fail(g, HAMR_ESTATE, "a grid with x1 refinement is read block by block (hamr_get_block_prims)");
  if (dev) {
    if (g->bh.on) blk_unpack(g, kind, out);
    else launch_unpack(g, padded, out, m);
  } else {
    double* st = stage_take(g) + stage_off;
    if (g->bh.on) blk_unpack(g, kind, st);
    else launch_unpack(g, padded, st, m);
    CK(cudaMemcpyAsync(out, st, nf * 8, cudaMemcpyDeviceToHost, g->stream));
  }
  return HAMR_OK;
}

}  // namespace

extern "C" {

int hamr_workspace_bytes(const hamr_params* p, size_t* bytes) {
  std::string why;
  if (!p || !bytes || !params_ok(*p, why)) return HAMR_EINVAL;
  Lay L;
  GridShape gs;
  if (!make_layout(*p, L, gs)) return HAMR_EINVAL;
  *bytes = plan_arena(*p, L, gs).total;
  return HAMR_OK;
}

int hamr_grid_create(const hamr_params* p, hamr_grid** out) {
  return create_common(p, nullptr, 0, nullptr, true, out);
}

int hamr_grid_create_in(const hamr_params* p, void* arena, size_t arena_bytes, void* cuda_stream,
                        hamr_grid** out) {
  return create_common(p, arena, arena_bytes, cuda_stream, false, out);
}

int hamr_grid_destroy(hamr_grid* g) {
  if (!g) return HAMR_EINVAL;
  cudaStreamSynchronize(g->stream);
  cudaFreeHost(g->h_pinned);
  if (g->bh.h_ctop) cudaFreeHost(g->bh.h_ctop);
  if (g->bh.h_ints) cudaFreeHost(g->bh.h_ints);
  for (cudaEvent_t e : g->ev) cudaEventDestroy(e);
  if (g->ev_input) cudaEventDestroy(g->ev_input);
  for (int c = 0; c < 2; c++)
    if (g->step_graph[c]) cudaGraphExecDestroy(g->step_graph[c]);
  for (int a = 0; a < 2; a++)
    for (int b = 0; b < 2; b++)
      if (g->stage_graph[a][b]) cudaGraphExecDestroy(g->stage_graph[a][b]);
  destroy_aux(g);
  if (g->own_arena) cudaFree(g->arena);
  if (g->own_stream) cudaStreamDestroy(g->stream);
  delete g;
  return HAMR_OK;
}

int hamr_set_prims(hamr_grid* g, const double* const hydro[5], const double* const bface[3]) {
  return set_prims_common(g, hydro, bface, false);
}
int hamr_set_prims_dev(hamr_grid* g, const double* const hydro[5], const double* const bface[3]) {
  return set_prims_common(g, hydro, bface, true);
}

int hamr_set_prims_async(hamr_grid* g, const double* const hydro[5], const double* const bface[3]) {
  return set_prims_common(g, hydro, bface, false, true);
}

int hamr_wait_input(hamr_grid* g) {
  if (!g) return HAMR_EINVAL;
  if (!g->ev_input) { CK(cudaStreamSynchronize(g->stream)); return HAMR_OK; }
  CK(cudaEventSynchronize(g->ev_input));
  return HAMR_OK;
}

int hamr_step_async(hamr_grid* g, int nsteps) {
  if (!g || nsteps < 0) return HAMR_EINVAL;
  g->out_staged = false;
  if (g->dead) return fail(g, HAMR_ESTATE, "grid unusable after a non-finite state");
  if (g->sharded) return fail(g, HAMR_ESTATE, "an x1 slab steps through hamr_shard_stage (its neighbours must keep pace)");
  if (!g->have_state) return fail(g, HAMR_ESTATE, "hamr_step before hamr_set_prims");
  if (g->bh.on) {
    const int rc = blk_step(g, nsteps);
    if (rc != HAMR_OK) return fail(g, rc, "block grid step failed");
  } else {
    for (int s = 0; s < nsteps; s++) {
      const int rc = step_once(g);
      if (rc != HAMR_OK) return rc;
    }
  }
  CK(cudaGetLastError());
  return HAMR_OK;
}

int hamr_sync(hamr_grid* g) {
  if (!g) return HAMR_EINVAL;
  return check_state(g);
}

int hamr_step(hamr_grid* g, int nsteps, double* t_out, double* dt_last_out) {
  int rc = hamr_step_async(g, nsteps);
  if (rc != HAMR_OK) return rc;
  double v[6];
  rc = read_scal(g, 0, 6, v);
  if (rc != HAMR_OK) return rc;
  if (t_out) *t_out = v[S_T];
  if (dt_last_out) *dt_last_out = v[S_DTLAST];
  return check_state(g);
}

int hamr_get_prims(hamr_grid* g, double* const prims[8]) {
  if (!g || !prims) return HAMR_EINVAL;
  if (!g->have_state) return fail(g, HAMR_ESTATE, "no state");
  const Fields& sn = g->s[g->isn];
  const size_t nz = (size_t)g->par.n[0] * g->par.n[1] * g->par.n[2];
  // all unpack kernels first (into the staging area), then the eight copies back to back: the host link does not wait
  // for a kernel between two copies.  After hamr_stage_output the unpacked arrays are there already
  if (!g->out_staged) {
    double* st = stage_take(g);
    for (int c = 0; c < 8; c++) {
      if (!prims[c]) continue;
      int rc = get_dense(g, c < 5 ? sn.P[c] : sn.Bc[c - 5], st + (size_t)c * nz, -1, true, 0, c);
      if (rc != HAMR_OK) return rc;
    }
  }
  for (int c = 0; c < 8; c++)
    if (prims[c]) CK(cudaMemcpyAsync(prims[c], g->stage + (size_t)c * nz, nz * 8, cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  return HAMR_OK;
}

int hamr_stage_output(hamr_grid* g) {
  if (!g) return HAMR_EINVAL;
  if (!g->have_state) return fail(g, HAMR_ESTATE, "no state");
  const Fields& sn = g->s[g->isn];
  const size_t nz = (size_t)g->par.n[0] * g->par.n[1] * g->par.n[2];
  double* st = stage_take(g);
  for (int c = 0; c < 8; c++) {
    int rc = get_dense(g, c < 5 ? sn.P[c] : sn.Bc[c - 5], st + (size_t)c * nz, -1, true, 0, c);
    if (rc != HAMR_OK) return rc;
  }
  CK(cudaGetLastError());
  g->out_staged = true;
  return HAMR_OK;
}

int hamr_get_prims_dev(hamr_grid* g, double* const prims[8]) {
  if (!g || !prims) return HAMR_EINVAL;
  if (!g->have_state) return fail(g, HAMR_ESTATE, "no state");
  const Fields& sn = g->s[g->isn];
  for (int c = 0; c < 8; c++) {
    if (!prims[c]) continue;
    const int rc = get_dense(g, c < 5 ? sn.P[c] : sn.Bc[c - 5], prims[c], -1, true, 0, c);
    if (rc != HAMR_OK) return rc;
  }
  CK(cudaGetLastError());
  return HAMR_OK;
}

int hamr_get_bface(hamr_grid* g, double* const bface[3]) {
  if (!g || !bface) return HAMR_EINVAL;
  if (!g->have_state) return fail(g, HAMR_ESTATE, "no state");
  const Fields& sn = g->s[g->isn];
  const int* N = g->par.n;
  size_t off = 0;
  for (int d = 0; d < 3; d++) {
    if (!bface[d]) continue;
    int rc = get_dense(g, sn.Bf[d], bface[d], d, false, off, 8 + d);
    if (rc != HAMR_OK) return rc;
    off += (size_t)(N[0] + 1) * (N[1] + 1) * (N[2] + 1);
  }
  CK(cudaStreamSynchronize(g->stream));
  return HAMR_OK;
}

int hamr_divb(hamr_grid* g, double* out) {
  if (!g || !out) return HAMR_EINVAL;
  if (!g->have_state) return fail(g, HAMR_ESTATE, "no state");
  if (g->bh.on) blk_divb(g);
  else launch_divb(g, g->s[g->isn]);
  return read_scal(g, S_DIVB, 1, out);
}

int hamr_get_stats(hamr_grid* g, long long counts[4]) {
  if (!g || !counts) return HAMR_EINVAL;
  unsigned long long* h = (unsigned long long*)(g->h_pinned + 32);
  CK(cudaMemcpyAsync(h, g->D.cnt, 4 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, g->stream));
  CK(cudaMemsetAsync(g->D.cnt, 0, 4 * sizeof(unsigned long long), g->stream));
  CK(cudaStreamSynchronize(g->stream));
  for (int c = 0; c < 4; c++) counts[c] = (long long)h[c];
  return HAMR_OK;
}

int hamr_get_backup_count(hamr_grid* g, long long* n) {
  if (!g || !n) return HAMR_EINVAL;
  unsigned long long* h = (unsigned long long*)(g->h_pinned + 32);
  CK(cudaMemcpyAsync(h, g->D.cnt + N_ENTROPY, sizeof(unsigned long long), cudaMemcpyDeviceToHost, g->stream));
  CK(cudaMemsetAsync(g->D.cnt + N_ENTROPY, 0, sizeof(unsigned long long), g->stream));
  CK(cudaStreamSynchronize(g->stream));
  *n = (long long)h[0];
  return HAMR_OK;
}

int hamr_get_time(hamr_grid* g, double* t, double* dt_next) {
  if (!g) return HAMR_EINVAL;
  double v[2];
  int rc = read_scal(g, S_T, 2, v);
  if (rc != HAMR_OK) return rc;
  if (t) *t = v[0];
  if (dt_next) *dt_next = v[1];
  return HAMR_OK;
}

int hamr_set_dt(hamr_grid* g, double dt) {
  if (!g || !(dt > 0.0)) return HAMR_EINVAL;
  g->h_pinned[48] = dt;
  CK(cudaMemcpyAsync(g->D.scal + S_DT, g->h_pinned + 48, sizeof(double), cudaMemcpyHostToDevice, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  return HAMR_OK;
}

const char* hamr_last_error(const hamr_grid* g) { return g ? g->err.c_str() : "null grid"; }

int hamr_num_blocks(const hamr_grid* g) { return g ? (g->bh.on ? g->bh.nblk : 1) : 0; }

int hamr_block_info(const hamr_grid* g, int b, double x_lo[3], double dx[3], int n[3], int* time_level) {
  if (!g || b < 0 || b >= hamr_num_blocks(g)) return HAMR_EINVAL;
  for (int d = 0; d < 3; d++) {
    const double dxd = (d == 0 && g->bh.on && g->bh.lev1[b]) ? 0.5 * g->D.dx[0] : g->D.dx[d];
    if (x_lo) x_lo[d] = g->D.x0[d] + (g->bh.on ? g->bh.I0[(size_t)b * 3 + d] * dxd : (d == 0 ? g->D.ioff * dxd : 0.0));
    if (dx) dx[d] = dxd;
    if (n) n[d] = g->D.L.n[d];
  }
  if (time_level) *time_level = g->bh.on ? g->bh.tau[b] : 0;
  return HAMR_OK;
}

// ---- block-by-block state access (required on grids with x1 refinement) ---------------------------------
int hamr_set_block_prims(hamr_grid* g, int b, const double* const hydro[5], const double* const bface[3]) {
  if (!g || !g->bh.on || b < 0 || b >= g->bh.nblk || !hydro) return HAMR_EINVAL;
  if (g->dead) return fail(g, HAMR_ESTATE, "grid unusable after a non-finite state");
  for (int c = 0; c < 5; c++) if (!hydro[c]) return fail(g, HAMR_EINVAL, "hydro[c] is NULL");
  const Lay& L = g->D.L;
  if (!g->blocks_open) {   // first block of a new state: every block back to buffer set 0
    CK(cudaMemsetAsync(g->D.B.cur, 0, (size_t)g->bh.nblk * sizeof(int), g->stream));
    g->blocks_open = true;
    g->have_state = false;
  }
  const size_t nz = (size_t)L.n[0] * L.n[1] * L.n[2];
  size_t off = (size_t)b * 8 * (L.n[0] + 1) * (L.n[1] + 1) * (L.n[2] + 1);   // the block's own staging slot
  for (int c = 0; c < 5; c++) {
    double* st = stage_take(g) + off;
    CK(cudaMemcpyAsync(st, hydro[c], nz * 8, cudaMemcpyHostToDevice, g->stream));
    blk_pack_one(g, b, st, c, -1, false);
    off += nz;
  }
  for (int d = 0; d < 3; d++) {
    int m[3] = {L.n[0], L.n[1], L.n[2]};
    m[d] += 1;
    const size_t nf = (size_t)m[0] * m[1] * m[2];
    const double* src = (bface && bface[d]) ? bface[d] : nullptr;
    if (src) {
      double* st = stage_take(g) + off;
      CK(cudaMemcpyAsync(st, src, nf * 8, cudaMemcpyHostToDevice, g->stream));
      src = st;
      off += nf;
    }
    blk_pack_one(g, b, src, 5 + d, d, d == 1);
  }
  // the caller's arrays may be pageable: cudaMemcpyAsync from pageable memory returns only after the data
  // have been staged, so they may be reused on return; the device side completes before hamr_blocks_commit returns
  return HAMR_OK;
}

// every block in one call: the per-block arrays of hamr_set_block_prims back to back in block order
int hamr_set_all_blocks(hamr_grid* g, const double* const hydro[5], const double* const bface[3]) {
  if (!g || !g->bh.on || !hydro) return HAMR_EINVAL;
  if (g->dead) return fail(g, HAMR_ESTATE, "grid unusable after a non-finite state");
  for (int c = 0; c < 5; c++) if (!hydro[c]) return fail(g, HAMR_EINVAL, "hydro[c] is NULL");
  const Lay& L = g->D.L;
  const size_t nb = (size_t)g->bh.nblk;
  CK(cudaMemsetAsync(g->D.B.cur, 0, nb * sizeof(int), g->stream));
  g->have_state = false;
  const size_t nz = (size_t)L.n[0] * L.n[1] * L.n[2] * nb;
  size_t off = 0;
  for (int c = 0; c < 5; c++) {
    double* st = stage_take(g) + off;
    CK(cudaMemcpyAsync(st, hydro[c], nz * 8, cudaMemcpyHostToDevice, g->stream));
    blk_pack_one(g, -1, st, c, -1, false);
    off += nz;
  }
  for (int d = 0; d < 3; d++) {
    int m[3] = {L.n[0], L.n[1], L.n[2]};
    m[d] += 1;
    const size_t nf = (size_t)m[0] * m[1] * m[2] * nb;
    const double* src = (bface && bface[d]) ? bface[d] : nullptr;
    if (src) {
      double* st = stage_take(g) + off;
      CK(cudaMemcpyAsync(st, src, nf * 8, cudaMemcpyHostToDevice, g->stream));
      src = st;
      off += nf;
    }
    blk_pack_one(g, -1, src, 5 + d, d, d == 1);
  }
  g->blocks_open = true;
  return hamr_blocks_commit(g);
}

int hamr_get_all_blocks(hamr_grid* g, double* const prims[8]) {
  if (!g || !g->bh.on || !prims) return HAMR_EINVAL;
  if (!g->have_state) return fail(g, HAMR_ESTATE, "no state");
  const Lay& L = g->D.L;
  const size_t nz = (size_t)L.n[0] * L.n[1] * L.n[2] * g->bh.nblk;
  for (int c = 0; c < 8; c++) {
    if (!prims[c]) continue;
    double* st = stage_take(g) + (size_t)c * nz;
    blk_unpack_one(g, -1, c, st);
    CK(cudaMemcpyAsync(prims[c], st, nz * 8, cudaMemcpyDeviceToHost, g->stream));
  }
  CK(cudaStreamSynchronize(g->stream));
  return HAMR_OK;
}

int hamr_blocks_commit(hamr_grid* g) {
  if (!g || !g->bh.on) return HAMR_EINVAL;
  g->out_staged = false;
  if (!g->blocks_open) return fail(g, HAMR_ESTATE, "hamr_blocks_commit without hamr_set_block_prims");
  g->blocks_open = false;
  g->isn = 0; g->ish = 1; g->inew = 2;
  CK(cudaMemsetAsync(g->D.scal, 0, NSCAL * sizeof(double), g->stream));
  CK(cudaMemsetAsync(g->D.cnt, 0, NCNT * sizeof(unsigned long long), g->stream));
  const int rc = blk_initial(g);
  if (rc != HAMR_OK) return fail(g, rc, "block grid initialisation failed");
  blk_check_finite(g);
  g->have_state = true;
  CK(cudaGetLastError());
  return check_state(g);
}

// ---- C-20: regridding of the x1 refinement level (the x1-only part) ----------------------------------
int hamr_refine_radius(hamr_grid* g, double rho_cut, double* r_refine_max) {
  if (!g || !r_refine_max) return HAMR_EINVAL;
  if (!g->bh.on) return fail(g, HAMR_EINVAL, "the refinement criterion needs a block grid (nb)");
  if (!g->have_state) return fail(g, HAMR_ESTATE, "no state");
  const int rc = blk_refine_radius(g, rho_cut, r_refine_max);
  return rc == HAMR_OK ? rc : fail(g, rc, "hamr_refine_radius");
}

int hamr_regrid(hamr_grid* g, double r_refine_max, hamr_grid** out) {
  if (out) *out = nullptr;
  if (!g || !out) return HAMR_EINVAL;
  if (!g->bh.on) return fail(g, HAMR_EINVAL, "regridding needs a block grid (nb)");
  if (!g->have_state || g->blocks_open) return fail(g, HAMR_ESTATE, "no committed state");
  if (g->dead) return fail(g, HAMR_ESTATE, "grid unusable after a non-finite state");
  hamr_params p = g->par;
  p.r_refine_max = r_refine_max > 0.0 ? r_refine_max : 0.0;
  hamr_grid* gn = nullptr;
  int rc = hamr_grid_create(&p, &gn);
  if (rc != HAMR_OK) return fail(g, rc, "regrid: the new lattice was refused (refined columns must leave a block grid)");
  if (!gn->bh.on) { hamr_grid_destroy(gn); return fail(g, HAMR_EINVAL, "regrid: the new grid is not a block grid"); }
  double tt[2];
  rc = read_scal(g, S_T, 2, tt);
  if (rc == HAMR_OK) rc = blk_regrid(g, gn);
  if (rc != HAMR_OK) { hamr_grid_destroy(gn); return fail(g, rc, "regrid: state transfer failed"); }
  // as hamr_blocks_commit: ghosts, B_c, one flux pass for the step and the time levels (C-14), then the clock
  gn->isn = 0; gn->ish = 1; gn->inew = 2;
  cudaError_t e = cudaMemsetAsync(gn->D.scal, 0, NSCAL * sizeof(double), gn->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(gn->D.cnt, 0, NCNT * sizeof(unsigned long long), gn->stream);
  if (e == cudaSuccess) rc = blk_initial(gn);
  gn->h_pinned[57] = tt[0];
  if (e == cudaSuccess && rc == HAMR_OK)
    e = cudaMemcpyAsync(gn->D.scal + S_T, gn->h_pinned + 57, sizeof(double), cudaMemcpyHostToDevice, gn->stream);
  if (e != cudaSuccess || rc != HAMR_OK) { hamr_grid_destroy(gn); return fail(g, e != cudaSuccess ? HAMR_ECUDA : rc, "regrid: initialisation of the new grid failed"); }
  blk_check_finite(gn);
  gn->have_state = true;
  rc = check_state(gn);
  if (rc != HAMR_OK) { hamr_grid_destroy(gn); return fail(g, rc, "regrid: non-finite state after the transfer"); }
  *out = gn;
  return HAMR_OK;
}

static int get_block(hamr_grid* g, int b, int kind0, int nkind, double* const out[]) {
  if (!g || !g->bh.on || b < 0 || b >= g->bh.nblk || !out) return HAMR_EINVAL;
  if (!g->have_state) return fail(g, HAMR_ESTATE, "no state");
  const Lay& L = g->D.L;
  size_t off = 0;
  for (int c = 0; c < nkind; c++) {
    if (!out[c]) continue;
    const int kind = kind0 + c, stag = kind >= 8 ? kind - 8 : -1;
    int m[3] = {L.n[0], L.n[1], L.n[2]};
    if (stag >= 0) m[stag] += 1;
    const size_t nf = (size_t)m[0] * m[1] * m[2];
    double* st = stage_take(g) + off;
    blk_unpack_one(g, b, kind, st);
    CK(cudaMemcpyAsync(out[c], st, nf * 8, cudaMemcpyDeviceToHost, g->stream));
    off += nf;
  }
  CK(cudaStreamSynchronize(g->stream));
  return HAMR_OK;
}

int hamr_get_block_prims(hamr_grid* g, int b, double* const prims[8]) { return get_block(g, b, 0, 8, prims); }
int hamr_get_block_bface(hamr_grid* g, int b, double* const bface[3]) { return get_block(g, b, 8, 3, bface); }

// ---- NEXT-4: x1 slabs with ghost layers read from peer memory ------------------
static hamr_params slab_params(const hamr_params& gp, int n1) {
  hamr_params p = gp;
  p.n[0] = n1;
  return p;
}

int hamr_shard_workspace_bytes(const hamr_params* gp, int i_lo, int n1, size_t* bytes) {
  std::string why;
  if (!gp || !bytes || !slab_ok(*gp, i_lo, n1, why)) return HAMR_EINVAL;
  const hamr_params p = slab_params(*gp, n1);
  return hamr_workspace_bytes(&p, bytes);
}

int hamr_shard_create_in(const hamr_params* gp, int i_lo, int n1, void* arena, size_t arena_bytes, void* cuda_stream,
                         hamr_grid** out) {
  if (out) *out = nullptr;
  std::string why;
  if (!gp || !out || !slab_ok(*gp, i_lo, n1, why)) return HAMR_EINVAL;
  const hamr_params p = slab_params(*gp, n1);
  const SlabSpec sp = {i_lo, gp->n[0]};
  return create_common(&p, arena, arena_bytes, cuda_stream, false, out, &sp);
}

int hamr_shard_attach(hamr_grid* g, int side, const void* peer_arena, int peer_i_lo, int peer_n1) {
  if (!g || !g->sharded || side < 0 || side > 1) return HAMR_EINVAL;
  if (!peer_arena || ((uintptr_t)peer_arena & 255) != 0) return fail(g, HAMR_EINVAL, "peer arena is NULL or not 256-byte aligned");
  const int i_lo = g->D.ioff, n1 = g->par.n[0], n1g = g->n1_global;
  const bool periodic = g->par.bc_lo[0] == HAMR_BC_PERIODIC && n1 < n1g;
  bool fits;
  if (side == 0) fits = i_lo > 0 ? peer_i_lo + peer_n1 == i_lo : (periodic && peer_i_lo + peer_n1 == n1g);
  else fits = i_lo + n1 < n1g ? peer_i_lo == i_lo + n1 : (periodic && peer_i_lo == 0);
  if (peer_n1 < NG || peer_i_lo < 0 || !fits) return fail(g, HAMR_EINVAL, "the neighbour slab does not adjoin this side (or is thinner than 3 zones)");
  // the neighbour's arena is laid out by the same plan: its 33 state arrays come first
  const hamr_params pp = slab_params(g->par, peer_n1);
  Lay PL;
  GridShape pgs;
  if (!make_layout(pp, PL, pgs)) return fail(g, HAMR_EINVAL, "neighbour layout");
  if (PL.S1 != g->D.L.S1 || PL.S2 != g->D.L.S2) return fail(g, HAMR_EINVAL, "neighbour layout differs in x2 / x3");
  const ArenaPlan pap = plan_arena(pp, PL, pgs);
  const double* arr = (const double*)((const char*)peer_arena + pap.arr);
  for (int q = 0; q < 3 * N_STATE_ARR; q++) g->peers.a[side][q] = arr + (size_t)q * PL.len;
  g->peers.n1[side] = peer_n1;
  g->peers.on[side] = 1;
  CK(cudaMemcpyAsync((void*)g->D.peer, &g->peers, sizeof(PeerTab), cudaMemcpyHostToDevice, g->stream));
  CK(cudaStreamSynchronize(g->stream));   // g->peers may change before an asynchronous copy from pageable memory has read it
  g->shard_committed = false;
  return HAMR_OK;
}

static bool slab_sides_attached(const hamr_grid* g) {
  const int i_lo = g->D.ioff, n1 = g->par.n[0], n1g = g->n1_global;
  const bool periodic = g->par.bc_lo[0] == HAMR_BC_PERIODIC && n1 < n1g;
  const bool need_lo = i_lo > 0 || periodic, need_hi = i_lo + n1 < n1g || periodic;
  return (!need_lo || g->peers.on[0]) && (!need_hi || g->peers.on[1]);
}

int hamr_shard_commit(hamr_grid* g) {
  if (!g || !g->sharded) return HAMR_EINVAL;
  if (g->dead) return fail(g, HAMR_ESTATE, "grid unusable after a non-finite state");
  if (!slab_sides_attached(g)) return fail(g, HAMR_ESTATE, "a side without a physical boundary has no neighbour slab (hamr_shard_attach)");
  const Fields& sn = g->s[g->isn];
  launch_ghosts(g, sn, true);
  launch_flux(g, sn, true);   // C-14: one flux pass gives this slab's Courant maxima for the first step
  g->have_state = true;
  g->shard_committed = true;
  g->shard_stage = 3;
  CK(cudaGetLastError());
  return HAMR_OK;
}

int hamr_shard_stage(hamr_grid* g, int stage) {
  if (!g || !g->sharded || stage < 0 || stage > 1) return HAMR_EINVAL;
  if (g->dead) return fail(g, HAMR_ESTATE, "grid unusable after a non-finite state");
  if (!g->shard_committed) return fail(g, HAMR_ESTATE, "hamr_shard_stage before hamr_shard_commit");
  if (g->shard_stage != stage) return fail(g, HAMR_ESTATE, "stages out of order: commit, ctop get / set, stage 0, stage 1, ctop get / set, ...");
  g->out_staged = false;
  const Fields& sn = g->s[g->isn];
  const Fields& sh = g->s[g->ish];
  const Fields& sw = g->s[g->inew];
  auto enqueue = [&]() {
    if (stage == 0) enqueue_stage(g, sn, sn, sh, 0.5, true, false);
    else enqueue_stage(g, sh, sn, sw, 1.0, false, true);
  };
  // as step_once: the stage's launches are captured once per buffer parity and replayed (every argument, the
  // neighbour table included, is fixed for the grid); the first step, the legacy stream and the timers launch plainly
  const int par = g->isn == 0 ? 0 : 1;
  if (g->prof || g->plain_steps < 2 || g->stream == nullptr || g->stream == cudaStreamLegacy) {
    enqueue();
    g->plain_steps++;
  } else {
    if (!g->stage_graph[stage][par]) {
      const long long l0 = g->launches;
      cudaGraph_t graph = nullptr;
      CK(cudaStreamBeginCapture(g->stream, cudaStreamCaptureModeThreadLocal));
      enqueue();
      cudaError_t e = cudaStreamEndCapture(g->stream, &graph);
      g->stage_launches[stage][par] = g->launches - l0;
      g->launches = l0;
      if (e == cudaSuccess) e = cudaGraphInstantiate(&g->stage_graph[stage][par], graph, 0);
      if (graph) cudaGraphDestroy(graph);
      if (e != cudaSuccess) return fail(g, HAMR_ECUDA, "capturing the stage as a CUDA graph", e);
    }
    CK(cudaGraphLaunch(g->stage_graph[stage][par], g->stream));
    g->launches += g->stage_launches[stage][par];
  }
  if (stage == 0) {
    g->shard_stage = 1;
  } else {
    const int tmp = g->isn; g->isn = g->inew; g->inew = tmp;
    g->shard_stage = 2;
  }
  CK(cudaGetLastError());
  return HAMR_OK;
}

int hamr_shard_ctop_get_dev(hamr_grid* g, double* ctop3_dev) {
  if (!g || !g->sharded || !ctop3_dev) return HAMR_EINVAL;
  if (!g->shard_committed || g->shard_stage < 2) return fail(g, HAMR_ESTATE, "the Courant maxima are complete after hamr_shard_commit or stage 1");
  launch_ctop_out(g, ctop3_dev);
  CK(cudaGetLastError());
  return HAMR_OK;
}

int hamr_shard_ctop_set_dev(hamr_grid* g, const double* ctop3_dev) {
  if (!g || !g->sharded || !ctop3_dev) return HAMR_EINVAL;
  if (!g->shard_committed || g->shard_stage < 2) return fail(g, HAMR_ESTATE, "hamr_shard_ctop_set_dev follows hamr_shard_commit or stage 1");
  launch_dt_slab(g, ctop3_dev, g->shard_stage == 2);   // after a step: advance the clock; after a commit: first dt only
  g->shard_stage = 0;
  CK(cudaGetLastError());
  return HAMR_OK;
}

int hamr_set_levels(hamr_grid* g, const int* tau) {
  if (!g || !g->bh.on) return HAMR_EINVAL;
  return blk_set_levels(g, tau);
}

int hamr_debug_emf(hamr_grid* g) {
  if (!g) return HAMR_EINVAL;
  if (!g->have_state) return fail(g, HAMR_ESTATE, "no state");
  if (g->bh.on) return fail(g, HAMR_ESTATE, "not available on a block-structured grid");
  const Fields& sn = g->s[g->isn];
  launch_ghosts(g, sn, false);
  launch_zero_ctop(g);
  launch_flux(g, sn, true, true);
  launch_ct(g, sn);
  launch_deref_fix_edges(g, g->D);
  launch_dt(g, 2);
  CK(cudaStreamSynchronize(g->stream));
  CK(cudaGetLastError());
  return HAMR_OK;
}

int hamr_get_face(hamr_grid* g, int d, int which, double* out) {
  if (!g || !out || d < 0 || d > 2 || which < 0 || which > 7 || (which == 7 && !g->D.entropy)) return HAMR_EINVAL;
  const double* a = which == 7 ? g->D.FK[d] : (which < 5 ? g->D.F[d][which] : (which == 5 ? g->D.EfA[d] : g->D.EfB[d]));
  int rc = get_dense(g, a, out, d, false, 0);
  if (rc != HAMR_OK) return rc;
  CK(cudaStreamSynchronize(g->stream));
  return HAMR_OK;
}

int hamr_debug_kappa(hamr_grid* g, double* out) {
  if (!g || !out || !g->D.entropy) return HAMR_EINVAL;
  if (!g->have_state) return fail(g, HAMR_ESTATE, "no state");
  int rc = get_dense(g, g->D.K, out, -1, false, 0);
  if (rc != HAMR_OK) return rc;
  CK(cudaStreamSynchronize(g->stream));
  return HAMR_OK;
}

int hamr_get_edge(hamr_grid* g, int f, double* out) {
  if (!g || !out || f < 0 || f > 2) return HAMR_EINVAL;
  if (g->bh.on) return fail(g, HAMR_ESTATE, "not available on a block-structured grid");
  const Lay& L = g->D.L;
  int m[3] = {L.n[0] + 1, L.n[1] + 1, L.n[2] + 1};
  m[f] -= 1;
  double* st = stage_take(g);
  launch_unpack(g, g->D.Ee[f], st, m);
  CK(cudaMemcpyAsync(out, st, (size_t)m[0] * m[1] * m[2] * 8, cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  return HAMR_OK;
}

int hamr_get_ctop(hamr_grid* g, double ctop[3]) {
  if (!g || !ctop) return HAMR_EINVAL;
  return read_scal(g, S_CTOPL0, 3, ctop);
}

int hamr_totals(hamr_grid* g, double tot[5]) {
  if (!g || !tot) return HAMR_EINVAL;
  if (!g->have_state) return fail(g, HAMR_ESTATE, "no state");
  if (g->bh.on) blk_totals(g);
  else launch_totals(g, g->s[g->isn]);
  return read_scal(g, S_TOT0, 5, tot);
}

int hamr_profile_begin(hamr_grid* g) {
  if (!g) return HAMR_EINVAL;
  CK(cudaStreamSynchronize(g->stream));
  g->ev_used = 0;
  g->prof = true;
  return HAMR_OK;
}

int hamr_profile_end(hamr_grid* g, int nclass, double ms[], long long count[]) {
  if (!g || !ms || !count || nclass < NKCLASS) return HAMR_EINVAL;
  g->prof = false;
  CK(cudaStreamSynchronize(g->stream));
  for (int c = 0; c < nclass; c++) { ms[c] = 0.0; count[c] = 0; }
  for (size_t i = 0; i < g->ev_used; i++) {
    float t = 0.f;
    CK(cudaEventElapsedTime(&t, g->ev[2 * i], g->ev[2 * i + 1]));
    ms[g->ev_cls[i]] += (double)t;
    count[g->ev_cls[i]]++;
  }
  g->ev_used = 0;
  return HAMR_OK;
}

const char* hamr_profile_class_name(int c) {
  static const char* names[NKCLASS] = {"ghosts", "flux_x1", "flux_x2", "flux_x3", "centre_emf", "edge_emf",
                                       "update_predictor", "update_corrector", "dt", "other"};
  return (c >= 0 && c < NKCLASS) ? names[c] : "";
}

int hamr_launch_count(const hamr_grid* g, long long* n) {
  if (!g || !n) return HAMR_EINVAL;
  *n = g->launches;
  return HAMR_OK;
}

}  // extern "C"
