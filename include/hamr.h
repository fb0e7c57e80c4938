/* hamr.h — C ABI of the B200-native H-AMR hot path (Liska et al., arXiv:1912.10192).
 *
 * What the library computes: the per-zone GRMHD conservative update
 *     d_t(sqrt(-g) U) + d_i(sqrt(-g) F^i) = sqrt(-g) S ,  div B = 0          (Eq. 1)
 * on a grid uniform in the internal coordinates x1 = ln r, x2 = theta, x3 = phi of a Kerr-Schild
 * foliation, with HLLE fluxes and PPM reconstruction, a staggered
 * constrained-transport magnetic field with velocity-upwinded EMFs, source terms at
 * zone centres, a Newton-Raphson conserved-to-primitive inversion,
 * floors, a 2nd-order predictor/corrector and the harmonic
 * Courant time step (PAPER.md:93 fn. 2).  The readings of every point the paper leaves open are
 * in DESIGN.md §3.  Every step runs in hand-written CUDA kernels for sm_100a; there is no CPU path.
 *
 * Conventions
 *  - all floating point is IEEE fp64; units G = c = M = 1;
 *  - all arrays are SoA, dense, index order [i1][i2][i3] with i3 fastest, ACTIVE zones only (the
 *    library owns the ghost zones);
 *  - primitives: rho, u, ut1, ut2, ut3 (ut^i = spatial 4-velocity projected normal to the lapse
 *    observer, C-2), cell-centred B^i;  face field Bf^d = sqrt(-g) B^d on d-faces, with
 *    shapes (N1+1,N2,N3), (N1,N2+1,N3), (N1,N2,N3+1);
 *  - pointers are HOST pointers unless the function name ends in _dev, in which case they are
 *    DEVICE pointers read or written on the grid's stream;
 *  - the caller owns every array it passes; the library copies in or out before returning
 *    (host variants synchronise the grid's stream; _dev variants and hamr_step_async do not);
 *  - every call returns a hamr_status, never throws, never aborts; no global state;
 *  - one CUDA stream per grid; a grid must not be used from two host threads at once.
 */
#ifndef HAMR_H
#define HAMR_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct hamr_grid hamr_grid; /* opaque; owns (or borrows, see hamr_grid_create_in) device memory */

typedef enum {
  HAMR_OK = 0,
  HAMR_EINVAL = 1,     /* bad argument or parameter set                                         */
  HAMR_ENOMEM = 2,     /* device or host allocation failed / arena too small                    */
  HAMR_ECUDA = 3,      /* a CUDA call failed; hamr_last_error() has the text                    */
  HAMR_ESTATE = 4,     /* call out of order, e.g. hamr_step before hamr_set_prims               */
  HAMR_ENONFINITE = 5  /* NaN/Inf detected in the evolved primitives; the grid is unusable      */
} hamr_status;

typedef enum { HAMR_METRIC_MINKOWSKI = 0, HAMR_METRIC_KERR_SCHILD = 1 } hamr_metric_t;
/* HAMR_BC_POLAR_TRANSMIT (x2 only, both sides, "transmissive polar boundary"): the ghost zone beyond
 * the pole is the zone on the mirror row half a turn away in x3, with the x2 components (ut2, Bf2) changing sign;
 * needs an even N3, a periodic x3 of extent 2 pi, and blocks that span x3 or cut it into an EVEN number (the
 * rows beyond the pole then come from the block half a turn away). */
typedef enum { HAMR_BC_PERIODIC = 0, HAMR_BC_OUTFLOW = 1, HAMR_BC_POLAR_REFLECT = 2, HAMR_BC_POLAR_TRANSMIT = 3 } hamr_bc_t;
typedef enum { HAMR_RECON_PPM = 0, HAMR_RECON_PLM_MC = 1 } hamr_recon_t;
/* Coordinate map of the internal coordinates ("any self-consistent coordinate system (and metric) can be
 * chosen"): the Cartesian box (x^i linear) or x1 = ln r, x2 = theta, x3 = phi.  Two pairs are built: Minkowski on the
 * Cartesian box and Kerr-Schild on the logarithmic spherical-polar map; HAMR_MAP_DEFAULT picks the metric's own map,
 * any other pair is rejected with HAMR_EINVAL. */
typedef enum { HAMR_MAP_DEFAULT = 0, HAMR_MAP_CARTESIAN = 1, HAMR_MAP_LOGR_SPHERICAL = 2 } hamr_map_t;

/* Parameter block (plain data). */
typedef struct {
  int metric;            /* hamr_metric_t                                                        */
  int recon;             /* hamr_recon_t (PPM; PLM+MC is the allowed alternative)   */
  int n[3];              /* base zones N1, N2, N3                                                */
  int bc_lo[3], bc_hi[3];/* hamr_bc_t per side; periodic must be set on both sides of a dim     */
  int nb[3];             /* block size; {0,0,0} = one block (block-structured grid: DESIGN.md §9)*/
  int n_deref;           /* number of phi-derefinement thresholds, 0 = none       */
  int deref_factor[4];   /* derefinement factor per threshold (see "phi-derefinement" below)            */
  int lat_max_level;     /* local adaptive time-stepping levels; 0 = global dt    */
  int map;               /* hamr_map_t                                                           */
  int entropy_backup;    /* 1: advect the entropy and invert with it where the energy inversion fails */
  int drift_floors;      /* 1: floors inject mass / energy in the drift frame; 0: fluid frame        */
  double a;              /* black-hole spin (ignored for Minkowski)                              */
  double xmin[3], xmax[3]; /* PHYSICAL extents: (r_in, r_out), (0, pi), (0, 2pi), or the box.  On the spherical
                            map x2 must span exactly (0, pi) with a polar boundary kind on both sides: the faces
                            at theta = 0, pi are treated as the polar axis (no flux, no normal field, C-7 / C-9) */
  double gamma_ad;       /* adiabatic index, p = (gamma_ad - 1) u                                */
  double cour;           /* Courant factor C of dt_d = C dx^d / max ctop_d (PAPER.md:93 fn. 2)   */
  double rho_fl_coef, rho_fl_pow, u_fl_coef, u_fl_pow; /* floor = coef * r^pow (r = 1 Cartesian) */
  double gamma_max;      /* Lorentz-factor ceiling                                               */
  double deref_theta_deg[4]; /* thresholds in degrees from either pole                                   */
  double r_refine_max;   /* x1-refinement radius (see below); <= 0 = none           */
} hamr_params;

/* ---- life cycle ------------------------------------------------------------------------------ */
/* Builds the grid: allocates all device arrays (cudaMalloc, own stream) and runs the metric
 * precompute kernel (g_{mu nu}, g^{mu nu}, sqrt(-g), lapse, shift at centres and faces, metric
 * derivatives for the source).  *out is NULL on failure. */
int hamr_grid_create(const hamr_params* p, hamr_grid** out);
/* Bytes of device memory a grid with these parameters needs. */
int hamr_workspace_bytes(const hamr_params* p, size_t* bytes);
/* Same as hamr_grid_create, but the device arrays live in caller-owned device memory `arena`
 * (>= hamr_workspace_bytes, 256-byte aligned; e.g. a torch CUDA tensor) and all work is issued on
 * the caller's `cuda_stream` (a cudaStream_t cast to void*; NULL = the legacy default stream).
 * The arena must outlive the grid; hamr_grid_destroy does not free it. */
int hamr_grid_create_in(const hamr_params* p, void* arena, size_t arena_bytes, void* cuda_stream,
                        hamr_grid** out);
int hamr_grid_destroy(hamr_grid* g);

/* ---- state in -------------------------------------------------------------------------------- */
/* Sets the state at t = 0: hydro[c] = rho, u, ut1, ut2, ut3 at zone centres (N1*N2*N3 each);
 * bface[d] = sqrt(-g) B^d on d-faces (NULL, or NULL entries, = 0).  Fills ghosts, derives the
 * cell-centred field (C-10) and runs one flux pass to set the first dt (C-14).
 * Returns HAMR_ENONFINITE if the input contains NaN/Inf. */
int hamr_set_prims(hamr_grid* g, const double* const hydro[5], const double* const bface[3]);
int hamr_set_prims_dev(hamr_grid* g, const double* const hydro[5], const double* const bface[3]);
/* hamr_set_prims with HOST arrays that does not wait: the eight host-to-device copies and the kernels behind them are
 * enqueued on the grid's stream and the call returns.  The arrays should be page-locked (pinned; pageable memory makes
 * every copy synchronous) and must stay UNCHANGED until hamr_wait_input has returned, which waits for the copies only
 * (not for the kernels behind them): the host link is then free for another grid's input while this grid's first flux
 * pass and step run.  NaN / Inf input is reported by the next full wait (hamr_sync, hamr_step: HAMR_ENONFINITE).  On a
 * block-structured grid the call waits as hamr_set_prims does (the first time levels are assigned on the host). */
int hamr_set_prims_async(hamr_grid* g, const double* const hydro[5], const double* const bface[3]);
int hamr_wait_input(hamr_grid* g);   /* spins on the event behind the last copy (no sleep: the wake-up would idle the link) */

/* ---- the hot path ---------------------------------------------------------------------------- */
/* Advances nsteps full steps (predictor + corrector = one zone-cycle each): ghost
 * fill, reconstruct + HLL per direction, CT EMFs + face-B update, source + update, con2prim +
 * floors, Courant dt reduction — all on the device.  t_out / dt_last_out (host, may be NULL)
 * receive the time reached and the dt of the last step; the call synchronises the stream. */
int hamr_step(hamr_grid* g, int nsteps, double* t_out, double* dt_last_out);
/* Enqueues nsteps steps and returns without synchronising (errors surface at the next sync).  Exception: on a
 * grid with lat_max_level > 0 the host reads the per-block Courant limits back once per coarse step to assign
 * the time levels and build the per-level block lists (one 24 B x blocks copy), so the call waits for all but
 * the last coarse step. */
int hamr_step_async(hamr_grid* g, int nsteps);
int hamr_sync(hamr_grid* g); /* waits for the stream; reports HAMR_ENONFINITE / HAMR_ECUDA */

/* ---- state out ------------------------------------------------------------------------------- */
int hamr_get_prims(hamr_grid* g, double* const prims[8]); /* 5 hydro + cell-centred B^i */
/* Enqueues, without waiting, the kernels that gather the eight dense arrays hamr_get_prims returns into the grid's staging
 * area; a hamr_get_prims that follows (with no step, state change or other getter on the grid in between) then consists
 * of its eight device-to-host copies only.  Lets a caller that shares the host link among several grids take the link
 * when the data are ready to leave, not before (hamr_step_async, hamr_stage_output, hamr_sync, then hamr_get_prims).
 * Not on grids with x1 refinement (HAMR_ESTATE: their state is read block by block). */
int hamr_stage_output(hamr_grid* g);
int hamr_get_prims_dev(hamr_grid* g, double* const prims[8]);
int hamr_get_bface(hamr_grid* g, double* const bface[3]);
/* max over zones of |div| / sum_d (|Bf+| + |Bf-|)/(2 dx^d), div = sum_d (Bf^d_+ - Bf^d_-)/dx^d;
 * zones whose denominator is below 1e-12 of its global maximum count 0 (C-11). */
int hamr_divb(hamr_grid* g, double* max_norm_divb);
/* counts since the last call: con2prim failures, rho-floor, u-floor, gamma-ceiling hits */
int hamr_get_stats(hamr_grid* g, long long counts[4]);
/* zones, since the last call, whose primitives came from the entropy inversion (entropy_backup; see below) */
int hamr_get_backup_count(hamr_grid* g, long long* n);
int hamr_get_time(hamr_grid* g, double* t, double* dt_next);
int hamr_set_dt(hamr_grid* g, double dt_next); /* overrides the next step's dt (run-to-time) */
const char* hamr_last_error(const hamr_grid* g); /* never NULL; valid until the next call on g */

/* ---- robust inversion path (C-18, C-19) ------------------------ */
/* entropy_backup = 1 ("H-AMR also advects the entropy (Noble et al. 2009), which is then used in place of
 * the energy equation to recover the primitive variables"): a ninth conserved row, sqrt(-g) rho u^t kappa with
 * kappa = p / rho^gamma_ad, is advanced in every stage beside the others (HLL flux of the reconstructed kappa, no
 * source term) and, wherever the 2-unknown energy inversion does not converge or returns rho <= 0 or u < 0, the zone
 * is inverted from the density, momentum and entropy rows instead (one unknown, bracketed Newton).  Before that, where
 * the Newton-Raphson inversion did not converge, the Aitken-accelerated fixed-point inversion the paper names beside it
 * is tried: the chain is Newton-Raphson, Aitken, entropy, failure path (C-21).  kappa is reset
 * from the new primitives after every update, so the state handed in and out stays the eight primitives.  A zone
 * whose entropy row has no admissible root (kappa < 0) keeps what the energy inversion gave it: its converged state,
 * for the floors to repair, or the failure path of hamr_get_stats counts[0].  Needs gamma_ad < 2.
 * drift_floors = 1 ("injects mass and internal energy in the drift frame of the jet ... (Ressler et al.
 * 2017)"): a zone below a floor is raised to it with the velocity perpendicular to the magnetic field unchanged and
 * the momentum along the field, (rho + gamma_ad u) gamma^2 v_par, conserved; zones without field get the fluid-frame
 * floors.  The Lorentz-factor ceiling follows as before.
 * Both options work on every grid the library builds: one block, blocks, phi-derefined polar rows (the strided x3 sweep
 * reconstructs kappa of the same groups, the entropy flux goes through the group fix-up like the other fluxes), the x1
 * refinement level (the coarse block takes the fine block's entropy flux on the interface face) and LAT (the flux
 * registers carry the entropy flux; the correction pass corrects the entropy row of the coarse block's boundary zones —
 * kappa having been reset, their row before the correction is density row x kappa of the new primitives — and inverts
 * them through the same chain, with the drift-frame floors if they are on).  The staged kernels
 * carry the ninth row where they serve the grid (cfg 2 with both options: 80 % of its plain rate). */

/* ---- regridding of the x1 refinement level (the x1-only part; C-20) ------------------ */
/* "H-AMR allows the user to implement an arbitrary refinement criterion.  For example ... a cutoff on the
 * maximum density in each block"; "(de-)refinement ... including the divergence-free prolongation and
 * restriction of magnetic fields (Balsara 2001)".  The grid carries ONE refinement level along x1 whose block columns are
 * contiguous from the inner x1 edge (r < r_refine_max), so a regrid moves the outer edge of the refined region.
 * hamr_refine_radius evaluates the density criterion on the current state: a block column wants refinement if one of its
 * blocks holds a zone with rho >= rho_cut; *r_refine_max receives the radius (x1 on the Cartesian map) that refines every
 * column up to the outermost such column, 0 if there is none.  Synchronises the stream.
 * hamr_regrid creates a NEW grid (own device memory and stream, as hamr_grid_create) with g's parameters but for
 * r_refine_max, transfers g's state onto it on the device and initialises it as hamr_blocks_commit does (ghosts, first
 * step and time levels from a flux pass, C-14); the time is carried over.  g stays valid and unchanged; the caller
 * destroys both.  Blocks that keep their level are copied bit for bit; newly refined blocks are the prolongation of their
 * parent (hydro: piecewise linear in x1 with the MC-limited slope; x1-faces: coincident ones copied, the new one the mean
 * of the parent zone's two; transverse faces: the parent's value), newly coarsened ones the restriction of their two
 * children (means; coincident x1-faces copied): every new zone has the divergence of the zone(s) it came from, so
 * div B stays at round-off.  On a phi-derefined grid the group structure of the polar rows (C-15) goes through the transfer
 * (every member of a group sees the same arithmetic) and is imposed again on the new grid as after hamr_blocks_commit.
 * Needs a block grid (nb) with an even nb[0], between steps; HAMR_EINVAL otherwise (also if r_refine_max does not give an
 * admissible lattice). */
int hamr_refine_radius(hamr_grid* g, double rho_cut, double* r_refine_max);
int hamr_regrid(hamr_grid* g, double r_refine_max, hamr_grid** out);

/* ---- one entry point that allocates nothing -------------------------------------------------------------------- */
/* For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it): the div B diagnostic of hamr_divb ("divergence-free evolution of the magnetic field"; C-11)
 * on caller-owned DENSE device arrays, without a grid object.  The scratch memory of its two-pass reduction is a
 * file-scope device array of fixed size inside the library (1 MB, held by every GPU that loads the library until the
 * process exits); the call itself makes no cudaMalloc / cudaFree and calls no allocating library routine.
 *   n[3]: zones; dx[3]: zone widths (both host); bface_dev[d]: DEVICE pointer to sqrt(-g) B^d on d-faces, extent
 *   n[d] + 1 along d, x3 fastest (the layout hamr_set_prims takes); out_dev: DEVICE pointer to one double that
 *   receives max over zones of |div| / sum_d (|Bf+| + |Bf-|) / (2 dx^d), zones whose denominator is below 1e-12 of its
 *   maximum counting 0 (hamr_divb's definition); cuda_stream: a cudaStream_t cast to void* (NULL: the default stream).
 * Four kernels are enqueued on the stream and the call returns without synchronising; the caller owns every array.
 * Limit: n[0] n[1] n[2] <= HAMR_NOALLOC_MAX_ZONES, else HAMR_EINVAL and nothing is launched (hamr_noalloc_last_error
 * says so); larger fields go through hamr_divb on a grid.  Every call on a device shares the one scratch array, which
 * keeps the last call's contents (each call writes every slot before it reads it, so nothing needs clearing): calls
 * that overlap on the GPU (streams without ordering between them, several host threads) race: serialise them.
 * hamr_noalloc_setup resolves the scratch array's device address for the CURRENT device (once per device; no
 * allocation); hamr_divb_noalloc does the same on first use, so calling it beforehand matters only where even that
 * first look-up must happen outside a captured or timed region. */
#define HAMR_NOALLOC_MAX_ZONES 16777216
int hamr_noalloc_setup(void);
int hamr_divb_noalloc(const int n[3], const double dx[3], const double* const bface_dev[3], double* out_dev,
                      void* cuda_stream);
const char* hamr_noalloc_last_error(void); /* never NULL; per host thread; "" after a successful call */

/* ---- x1 slabs over peer memory: one grid on several GPUs ----------------------- */
/* "H-AMR uses ... NVLINK for intra-node GPU-GPU ... communication" — blocks on different GPUs exchange
 * their boundary zones every stage; PAPER.md:93 fn. 2: one Courant step for the whole grid.  Here the unit that is
 * distributed is an x1 SLAB of a one-block grid: zones [i_lo, i_lo + n1) of the n[0] zones of `global` (global extents and
 * boundary kinds; n1 >= 3).  One process per GPU holds one slab; a slab's geometry tables, floors and zone widths are those
 * of the global grid bit for bit, and so is every zone it computes: slabs stepped in lockstep reproduce the one-grid
 * result exactly.  There is NO exchange buffer and no pack / unpack step: the per-stage ghost fill of a slab reads the
 * three x1 ghost layers of a side that has a neighbour straight from the neighbour's active zones through a device
 * pointer to the neighbour's arena (the x2 / x3 boundary maps composed with it as with the physical x1 rules), i.e. over
 * NVLink when that arena lives on a peer GPU (CUDA IPC / symmetric memory; the caller maps it) and through L2 / HBM when
 * both slabs live on one GPU.  The interface face i_lo is held by both slabs, which advance it with bitwise equal EMFs.
 * What the caller provides between the calls is ordering and one reduction (the Python binding's shard.py does it with
 * torch.distributed: an all-reduce on the grid's stream is both):
 *     every slab: hamr_set_prims(_dev)              | its part of the state (zones and faces i_lo .. i_lo + n1)
 *     -- all slabs have been set --                 | barrier
 *     every slab: hamr_shard_commit                 | ghosts from the neighbours, first flux pass
 *     hamr_shard_ctop_get_dev -> MAX over slabs -> hamr_shard_ctop_set_dev      | first dt (C-14)
 *     per step:   hamr_shard_stage(0)               | predictor: reads the neighbours' time-n state
 *                 -- all slabs have finished stage 0 --
 *                 hamr_shard_stage(1)               | corrector: reads the neighbours' predictor state
 *                 hamr_shard_ctop_get_dev -> MAX over slabs -> hamr_shard_ctop_set_dev   | clock + next dt; also the barrier
 * A slab never writes to a neighbour's memory; the buffer set a stage writes is never the one a neighbour reads in that
 * stage, so the two ordering points per step are all the synchronisation there is.  hamr_step on a slab returns
 * HAMR_ESTATE.  State out: the usual getters, per slab.  Needs a grid of one block (nb = 0, no LAT, no x1 refinement);
 * phi-derefinement and the robust inversion options (entropy_backup, drift_floors) are allowed.  A periodic x1 closes the ring (the last slab is the
 * first one's low neighbour); with one slab covering the whole grid no neighbour is needed.
 * hamr_shard_attach: `peer_arena` is the neighbour slab's arena (the pointer ITS hamr_shard_create_in was given, as
 * seen from this process and device), (peer_i_lo, peer_n1) its extent; side 0 = low x1, 1 = high x1.  The library reads
 * the neighbour's state arrays at the offsets its own arena plan gives for that extent; nothing is copied or owned.
 * hamr_shard_ctop_get_dev / _set_dev take DEVICE pointers to three doubles (max signal speed per dimension, C-14) and
 * enqueue on the grid's stream without synchronising. */
int hamr_shard_workspace_bytes(const hamr_params* global, int i_lo, int n1, size_t* bytes);
int hamr_shard_create_in(const hamr_params* global, int i_lo, int n1, void* arena, size_t arena_bytes,
                         void* cuda_stream, hamr_grid** out);
int hamr_shard_attach(hamr_grid* g, int side, const void* peer_arena, int peer_i_lo, int peer_n1);
int hamr_shard_commit(hamr_grid* g);
int hamr_shard_stage(hamr_grid* g, int stage);
int hamr_shard_ctop_get_dev(hamr_grid* g, double* ctop3_dev);
int hamr_shard_ctop_set_dev(hamr_grid* g, const double* ctop3_dev);

/* ---- block-structured grid (BASELINE.json cfg 4) ------------------ */
/* A grid with nb != {0,0,0} or lat_max_level > 0 is cut into blocks of nb zones (nb[d] = 0: the whole
 * extent; nb[d] must divide n[d] and be >= 3).  Blocks exchange ghost zones directly;
 * with lat_max_level = L > 0 every block steps with dt_0 * 2^tau, tau <= L chosen from its own Courant
 * limit at every coarse step, neighbours differing by at most one level; ghosts of a
 * block on another time level are interpolated in time, and at the end of each coarse block's step
 * its boundary zones are corrected with the finer neighbour's accumulated fluxes and EMFs and
 * inverted again (C-16, C-17).  On such a grid hamr_step(nsteps) takes
 * nsteps COARSE steps of 2^L finest steps each; set / get calls take the same global arrays.
 * All kernels of a stage run once over all blocks of a time level (no per-block launches). */
int hamr_num_blocks(const hamr_grid* g);
/* x_lo: internal coordinates of the block's low corner; time_level: its current LAT level tau */
int hamr_block_info(const hamr_grid* g, int b, double x_lo[3], double dx[3], int n[3],
                    int* time_level);
/* phi-derefinement of the polar rows (C-15): with n_deref > 0 an x2 row whose zone-centre
 * polar angle lies within deref_theta_deg[t] degrees of either pole is derefined in x3 by deref_factor[t] (the
 * largest factor that applies; BASELINE cfg 4: {15, 5} degrees -> {2, 4}).  A row with factor m treats every
 * aligned group of m phi-zones as one zone: fluxes and EMFs are group means (or interpolated between group
 * boundaries), the x3 reconstruction takes one value per group, the Courant limit uses m dx3; all arrays keep
 * the fine shapes.  hamr_set_prims projects the hydro input onto group means; the face field given must be
 * uniform within groups (any axisymmetric field is).  Needs a periodic x3; factors are powers of two <= 16
 * that divide the x3 block size nb3 with 3 * factor <= nb3.  Works on monolithic and block grids and under LAT. */
/* One x1 refinement level (PAPER.md:71 per-dimension refinement; C-16): with r_refine_max > 0 every
 * block column whose x1-centre has r < r_refine_max (x1 < r_refine_max on the Cartesian map) is replaced by
 * two blocks of nb zones with dx1 / 2; such columns must be contiguous from the low x1 side and nb[0] >= 6.
 * Ghost zones across the coarse/fine interface are restricted (mean of the two fine values) or prolonged
 * (piecewise linear in x1, MC-limited); the coarse block takes the fine block's interface fluxes and EMFs.
 * A refined grid has no global zone array: its state is set and read block by block.  Arrays are dense,
 * block-local, x3 fastest: hydro[c] nb0*nb1*nb2, bface[d] with nb[d]+1 along d (NULL = 0); the caller keeps
 * them and, unlike with the other host calls, must leave them UNCHANGED until hamr_blocks_commit has returned
 * (the copies of all blocks are queued on the stream and waited for once, in commit; with 1472 blocks a wait
 * per block would dominate).  After the last hamr_set_block_prims, hamr_blocks_commit fills ghosts, projects onto the
 * derefinement invariant, and finds the first dt and time levels (HAMR_ENONFINITE on NaN/Inf input).
 * Also valid on unrefined block grids. */
int hamr_set_block_prims(hamr_grid* g, int b, const double* const hydro[5], const double* const bface[3]);
int hamr_blocks_commit(hamr_grid* g);
int hamr_get_block_prims(hamr_grid* g, int b, double* const prims[8]);   /* 5 hydro + cell-centred B^i */
/* Every block in one call (8 large copies instead of 8 per block): each array holds the per-block dense arrays of
 * the calls above back to back in block order.  hamr_set_all_blocks includes the commit and copies before it
 * returns; hamr_get_all_blocks fills prims (NULL entries skipped) and synchronises. */
int hamr_set_all_blocks(hamr_grid* g, const double* const hydro[5], const double* const bface[3]);
int hamr_get_all_blocks(hamr_grid* g, double* const prims[8]);
int hamr_get_block_bface(hamr_grid* g, int b, double* const bface[3]);
/* Test hooks and diagnostics (flux / EMF getters, per-kernel timers, geometry tables, zone-level physics
 * entry points, the FP64 peak measurement) are declared in hamr_debug.h. */

#ifdef __cplusplus
}
#endif
#endif /* HAMR_H */
