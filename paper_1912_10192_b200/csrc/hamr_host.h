// hamr_host.h — host-side grid object and kernel launchers of libhamr (internal; product code).
#pragma once
#include <string>
#include <vector>
#include "../../include/hamr.h"
#include "hamr_dev.cuh"

namespace hamr {

// one time level: hydro primitives, cell-centred B, densitised face B (all padded, on the device)
struct Fields {
  double* P[5];
  double* Bc[3];
  double* Bf[3];
};

// device scalars (one small array)
enum Scal { S_T = 0, S_DT, S_CTOP0, S_CTOP1, S_CTOP2, S_DTLAST, S_DENMAX, S_DIVB, S_TOT0 /* ..+4 */,
            S_CTOPL0 = 13 /* ..+2: ctop of the last finished pass */, NSCAL = 16 };
// device counters
enum Cnt { N_C2PFAIL = 0, N_RHOFL, N_UFL, N_GCEIL, N_NONFINITE, N_ENTROPY /* zones inverted from the entropy row (C-18) */, N_AITKEN /* ... by the Aitken scheme (C-21) */, NCNT = 8 };

// Block-structured grid: every per-variable array holds nblk
// padded blocks back to back (block b at doubles [b*blen, (b+1)*blen)); a launch works on the blocks
// listed in `list` (all blocks of one time level).  nblk == 0: monolithic grid.
struct BlkDev {
  int nblk;                  // blocks on the grid
  int nact;                  // blocks in this launch
  int blen;                  // doubles per block per array
  int ge2;                   // row pitch of the (global, per x1-level) geometry tables
  int n2g;                   // global N2 (pole faces: J == 0 or J == n2g)
  int flev;                  // offset in doubles of the level-1 floor tables
  int tlevA;                 // offset in doubles of the level-1 geometry records
  const int* list;           // [nact] block ids of this launch
  const int* dlist;          // [ndact] those of them that hold phi-derefined rows (C-15 kernels); NULL: use list
  int ndact;
  const int4* info;          // [nblk] {table index of local zone (0,0), x1 level, I0, J0}
  const int* nbr;            // [nblk][NNBR]: 27 neighbour blocks by offset (-1 outside the domain), then the 9 blocks
                             // half a turn away across a transmissive pole, by (o0 + 1) * 3 + (o2 + 1) (NEXT-1; -1 if none)
  const int* phys;           // [nblk] bit d: low side of dim d is a physical boundary, bit 3+d: high side
  const int* K0;             // [nblk] global x3 index of local zone 0
  int* tau;                  // [nblk] LAT time level (C-17)
  int* cur;                  // [nblk] which of the 3 buffers holds the block's time-n state (0 or 2)
  // ghost-source table (blocks.cu): for every padded location of every block and each of the four array kinds
  // (zone-centred, x1-, x2-, x3-faces) WHERE the ghost fill takes the value from, packed in 64 bits; a pure function of
  // the block tables and the time levels, rebuilt when the levels change.  [nblk][4][gloc]; NULL: computed on the fly
  const unsigned long long* gsrc;
  int gloc;                  // padded locations per block: e1 * e2 * (n3 + 2 NG + 1)
  int* flags;                // [nblk] bit 0: ghost fill is a plain copy; bit 1: has a finer-level neighbour
  double* ctopb;             // [nblk][3] max signal speed of the block's last corrector pass (C-14)
  double* FA2[3][5];         // flux registers: dt_b F summed over the steps inside one coarser step (C-17)
  double* EA2[3];            // EMF registers
  double* FKA2[3];           // C-18 under LAT: the register of the entropy flux (NULL without the entropy row)
};

// x1-slab sharding: the state arrays of the neighbour slabs, as device pointers
// valid on THIS device (peer memory over NVLink, or the same device).  Lives in device memory; the ghost fill reads the
// x1 ghost layers of a side that has a neighbour straight from the neighbour's active zones.
struct PeerTab {
  const double* a[2][33];    // [side: 0 low x1, 1 high x1][buffer set * 11 + array: P 0..4, Bc 5..7, Bf 8..10]
  int n1[2];                 // the neighbour's zone count along x1
  int on[2];                 // side has a neighbour
};

struct Dev {                 // everything a kernel may need, passed by value
  Lay L;
  BlkDev B;
  const PeerTab* peer;       // NEXT-4: neighbour slabs (NULL: the grid is not a slab)
  int ioff;                  // NEXT-4: global x1 index of local zone 0 (geometry tables, floors)
  int metric, recon;
  int bc_lo[3], bc_hi[3];
  double dx[3], x0[3];       // internal-coordinate spacing and origin
  double a, gam, cour, gamma_max;
  double rho_fl_coef, rho_fl_pow, u_fl_coef, u_fl_pow;
  const double* gcA;         // geometry records (hamr_dev.cuh): centres [n2d][32],
  const double* gf1A;        // x1-faces [n2d][16],
  const double* gf2A;        // x2-faces [n2d][16] (pole rows: gdet = 0),
  const double* gf3A;        // x3-faces [n2d][16] (centre (x1, x2))
  const double* rho_fl;      // [e1] floor per x1 index
  const double* u_fl;
  int entropy, drift;        // C-18 entropy row + backup inversion, C-19 drift-frame floors (hamr_params; monolithic grids)
  double* K;                 // C-18: kappa = (gamma_ad - 1) u / rho^gamma_ad of the stage's source state, every zone
                             // incl. ghosts (k_kappa); the update kernel leaves the advected kappa of the active zones in it
  double* FK[3];             // C-18: flux of the entropy row on d-faces
  double* F[3][5];           // hydro fluxes on d-faces
  double* EfA[3];            // on d-faces: E_e, (d,e,f) cyclic  (C-8)
  double* EfB[3];            // on d-faces: E_f
  double* Ee[3];             // edge EMFs (C-9)
  double* Cc[3];             // centre EMFs (C-8)
  const int* mrow;           // phi-derefinement factor per global x2 row incl. ghosts (C-15); NULL: none
  double* scal;              // [NSCAL]
  unsigned long long* cnt;   // [NCNT]
};

// the three roles of a stage (C-12) in the buffer sets of blocks with cur == 0 (a) / cur == 2 (b)
struct Roles { Fields src, base, out; };

// per-thread view of the block a BLK kernel thread works on (monolithic: constants)
struct BCtx { int b, zoff, q0, lev, cur, I0, J0; };
template <bool BLK>
__device__ __forceinline__ BCtx blk_ctx(const Dev& Dv, int slot) {
  BCtx c;
  if (BLK) {
    c.b = __ldg(Dv.B.list + slot);
    const int4 inf = __ldg(Dv.B.info + c.b);
    c.zoff = c.b * Dv.B.blen; c.q0 = inf.x; c.lev = inf.y; c.I0 = inf.z; c.J0 = inf.w;
    c.cur = Dv.B.cur[c.b];
  } else {
    c.b = 0; c.zoff = 0; c.q0 = NG * Dv.L.e2 + NG; c.lev = 0; c.cur = 0; c.I0 = 0; c.J0 = 0;
  }
  return c;
}
// buffer selection: a block's time-n state lives in buffer set a (cur == 0) or b (cur == 2)
template <bool BLK>
__device__ __forceinline__ const double* selp(const double* a, const double* b, int cur) { return (BLK && cur) ? b : a; }
template <bool BLK>
__device__ __forceinline__ double* selp(double* a, double* b, int cur) { return (BLK && cur) ? b : a; }

}  // namespace hamr

namespace hamr {
// kernel classes for the per-kernel timers (hamr_profile_*)
enum KClass { K_GHOSTS = 0, K_FLUX1, K_FLUX2, K_FLUX3, K_CEMF, K_EDGE, K_UPDATE_P, K_UPDATE_C, K_DT, K_OTHER, NKCLASS };
}

namespace hamr {
// host side of the block-structured grid (blocks.cu)
struct BlkHost {
  bool on;                   // block-structured grid (more than one block, or LAT)
  bool refined;              // some block columns carry the x1 refinement level (C-16)
  int nblk, tmax;            // blocks; highest LAT level (0: one global dt)
  int nslot[3];              // block lattice extents
  std::vector<int> nbr;      // [nblk][NNBR] host mirror of the neighbour table
  std::vector<int> lev1;     // [nblk] x1 refinement level
  std::vector<int> tau;      // [nblk] current time level
  std::vector<int> I0;       // [nblk][3]
  std::vector<int> phys;     // [nblk] physical-boundary sides
  std::vector<int> forced;   // test hook: prescribed time levels (empty: Courant-based)
  int* d_lists;              // device [5][nblk]: blocks of level 0..3, then every block
  int* d_clists;             // device [4][nblk]: blocks of level tau with a neighbour on tau - 1
  int* d_dlists;             // device [5][nblk]: per list, the blocks that hold phi-derefined rows
  int nlist[4], nclist[4], ndlist[5];
  std::vector<char> hasderef;  // [nblk] some row of the block (or of its transverse ghost layer) is derefined
  long long tb_u[4];         // LAT clocks per level, units of (finest dt)/2 (C-17)
  int dt_u[4];
  int has_new[4];
  double* h_ctop;            // pinned [nblk][3]
  int* h_ints;               // pinned [16][nblk]
  double dt0;                // host copy of the finest step (LAT)
  unsigned long long* d_gsrc;  // device ghost-source table (NULL: none)
  std::vector<int> gsrc_tau;   // the time levels the table was built for (empty: not built)
};
}

struct hamr_grid {
  hamr_params par;
  hamr::BlkHost bh;
  hamr::Dev D;
  hamr::Fields s[3];         // rotating: sn (time n), sh (n+1/2), snew
  int isn, ish, inew;
  void* arena;               // device memory base
  size_t arena_bytes;
  bool own_arena, own_stream;
  cudaStream_t stream;
  cudaStream_t aux[2];       // side streams of the fork / join around independent launches of a stage (flux.cu); NULL: none
  cudaEvent_t ev_fork, ev_join[2];
  cudaEvent_t ev_input;      // recorded behind the last host-to-device copy of hamr_set_prims_async (hamr_wait_input); NULL: none
  bool cemf_done;            // launch_flux_on has issued the centre-EMF kernel of the coming launch_ct_on
  double* stage;             // device staging buffer for dense <-> padded transfers
  size_t stage_doubles;
  double* h_pinned;          // small pinned host buffer for scalar read-back
  bool have_state, dead;
  bool out_staged;           // the staging area holds the dense primitives of the current state (hamr_stage_output)
  bool blocks_open;          // hamr_set_block_prims calls are being collected; hamr_blocks_commit closes
  long long launches;
  std::string err;
  // per-kernel timers: CUDA event pairs on the grid's stream around every launch while enabled
  bool prof;
  std::vector<cudaEvent_t> ev;   // pairs: start, stop
  std::vector<int> ev_cls;
  size_t ev_used;
  // the step sequence of a monolithic grid as a CUDA graph: one executable graph per parity of
  // the rotating state buffers, captured on first use after one plain step has run
  cudaGraphExec_t step_graph[2];
  long long graph_launches;      // kernel launches one replay stands for
  int plain_steps;               // steps enqueued launch by launch so far
  // NEXT-4: the grid is an x1 slab [i_lo, i_lo + n[0]) of a global grid of n1_global zones
  bool sharded;
  int n1_global;
  hamr::PeerTab peers;           // host copy of D.peer
  bool shard_committed;          // hamr_shard_commit has run on the current state
  int shard_stage;               // next stage hamr_shard_stage expects (0 / 1), 2: the step's hamr_shard_ctop_set_dev
  cudaGraphExec_t stage_graph[2][2];   // [stage][parity of the rotating buffers]: a slab's stage as a CUDA graph
  long long stage_launches[2][2];      // kernel launches one replay stands for
};

namespace hamr {
// the staging area for a new use: whatever hamr_stage_output left there is gone
inline double* stage_take(hamr_grid* g) { g->out_staged = false; return g->stage; }
// brackets one kernel launch with an event pair when profiling is on; always counts the launch
struct Launch {
  hamr_grid* g;
  bool on;
  Launch(hamr_grid* g_, int cls) : g(g_), on(g_->prof) {
    g->launches++;
    if (!on) return;
    if (g->ev_used * 2 + 2 > g->ev.size()) {
      cudaEvent_t a, b;
      cudaEventCreate(&a);
      cudaEventCreate(&b);
      g->ev.push_back(a);
      g->ev.push_back(b);
      g->ev_cls.push_back(cls);
    }
    g->ev_cls[g->ev_used] = cls;
    cudaEventRecord(g->ev[g->ev_used * 2], g->stream);
  }
  ~Launch() {
    if (!on) return;
    cudaEventRecord(g->ev[g->ev_used * 2 + 1], g->stream);
    g->ev_used++;
  }
};
}

namespace hamr {

// kernel launchers (each returns after enqueueing on g->stream)
void launch_ghosts(hamr_grid* g, const Fields& s, bool bc_active_too);
void launch_flux(hamr_grid* g, const Fields& src, bool want_ctop, bool with_cemf = false);
void launch_ct(hamr_grid* g, const Fields& src);
void launch_kappa(hamr_grid* g, const Dev& Dv, const Fields& src, const Fields& src2);   // misc.cu: C-18, fills Dv.K from the source state (after its ghost fill)
bool x3_ghosts_unused(const Dev& Dv);   // flux.cu: the stage kernels of this grid never read x3 ghost zones
void launch_update(hamr_grid* g, const Fields& src, const Fields& base, const Fields& out, double dtfac,
                   bool src_is_base);
void launch_dt(hamr_grid* g, int mode);  // 0 set dt, 1 advance t + set dt, 2 latch ctop only
void launch_ctop_out(hamr_grid* g, double* out3);                    // NEXT-4: this slab's Courant maxima -> out3 (device)
void launch_dt_slab(hamr_grid* g, const double* in3, bool advance);  // NEXT-4: dt from the maxima over all slabs (device)
void launch_pack(hamr_grid* g, const double* dense, double* padded, int stag, bool zero_pole);
void launch_unpack(hamr_grid* g, const double* padded, double* dense, const int m[3]);
void launch_divb(hamr_grid* g, const Fields& s);
void launch_totals(hamr_grid* g, const Fields& s);
void launch_check_finite(hamr_grid* g, const Fields& s);
void launch_zero_ctop(hamr_grid* g);
void launch_flux_on(hamr_grid* g, const Dev& Dv, const Fields& src, const Fields& src2, bool want_ctop, bool with_cemf = false);
void launch_centre_emf_on(hamr_grid* g, const Dev& Dv, const Fields& src, const Fields& src2);
void launch_ct_on(hamr_grid* g, const Dev& Dv, const Fields& src, const Fields& src2);
void launch_update_on(hamr_grid* g, const Dev& Dv, const Roles& ra, const Roles& rb, double dtfac, bool same);
// deref.cu / flux.cu: phi-derefinement (C-15)
void launch_deref_x3(hamr_grid* g, const Dev& Dv, const Fields& src, const Fields& src2, bool want_ctop);
void launch_deref_fix_flux(hamr_grid* g, const Dev& Dv);
void launch_deref_flux_layers(hamr_grid* g, const Dev& Dv);
void launch_deref_fix_edges(hamr_grid* g, const Dev& Dv);
void launch_deref_sync(hamr_grid* g, const Dev& Dv, const Fields& out, const Fields& out2);
void launch_deref_project(hamr_grid* g, const Dev& Dv, const Fields& s, const Fields& s2);
int deref_row_factor(const hamr_params& p, long long J);
void launch_geometry_tab(hamr_grid* g, int e1, int e2, double dx1, int n2glob, double* rho_fl, double* u_fl,
                         double* gcA, double* gf1A, double* gf2A, double* gf3A);

// blocks.cu: block-structured grid (H7)
int blk_count(const hamr_params& p, int nslot[3], int bn[3]);       // number of blocks (0 if invalid)
int blk_has_refinement(const hamr_params& p);
void blk_pack_one(hamr_grid* g, int b, const double* dense, int kind, int stag, bool zero_pole);
void blk_unpack_one(hamr_grid* g, int b, int kind, double* dense);
size_t blk_table_bytes(int nblk, long long nloc);                   // device bytes of the block tables; nloc: padded locations per block
int blk_setup(hamr_grid* g, void* tables);                          // lattice, neighbour tables, lists
void blk_pack(hamr_grid* g, const double* dense, int kind, int stag, bool zero_pole);  // kind: 0..4 P, 5..7 Bf
void blk_unpack(hamr_grid* g, int kind, double* dense);             // kind: 0..4 P, 5..7 Bc, 8..10 Bf
int blk_initial(hamr_grid* g);                                      // ghosts, first flux pass, dt / levels
int blk_step(hamr_grid* g, int nsteps);                             // nsteps coarse steps
int blk_set_levels(hamr_grid* g, const int* tau);
int blk_refine_radius(hamr_grid* g, double rho_cut, double* r_new);   // C-20: refinement criterion -> r_refine_max
int blk_regrid(hamr_grid* go, hamr_grid* gn);                         // C-20: state of go onto the lattice of gn
void blk_divb(hamr_grid* g);
void blk_totals(hamr_grid* g);
void blk_check_finite(hamr_grid* g);

}  // namespace hamr
