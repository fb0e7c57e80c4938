/* hamr_debug.h — test hooks and diagnostics of libhamr (not part of the hot path's public surface).
 *
 * Used by the parity tests (tests/) and by bench.py: getters for intermediate results of a stage, per-kernel device
 * timers, the geometry tables, zone-level entry points to the per-zone physics (so that the branches a whole-grid
 * run rarely takes — failed inversion, Lorentz-factor ceiling, floors — can be driven directly and compared with the
 * oracle), the LAT level override, and a measurement of the FP64 pipe's peak.  Same conventions as hamr.h:
 * host pointers, the caller owns every array, every call returns a hamr_status.
 */
#ifndef HAMR_DEBUG_H
#define HAMR_DEBUG_H
#include "hamr.h"
#ifdef __cplusplus
extern "C" {
#endif

/* Test hook: prescribes the LAT level of every block (tau[hamr_num_blocks], clamped to
 * 0..lat_max_level, then lowered until neighbours differ by at most one); NULL restores the
 * Courant-based choice.  Takes effect at the next hamr_set_prims / coarse step.  The caller keeps tau. */
int hamr_set_levels(hamr_grid* g, const int* tau);

/* ---- diagnostics used by the parity tests (not part of the hot path) -------------------------- */
/* Runs ghost fill + flux pass + CT EMFs on the current state (no update). */
int hamr_debug_emf(hamr_grid* g);
/* which 0..4: hydro flux F^d[c] of the last flux pass; 5, 6: the two face EMFs E_e, E_f with
 * (d, e, f) cyclic (C-8); 7: the flux of the entropy row (entropy_backup grids, C-18).
 * out: d-face array, extent n[d]+1 along d. */
int hamr_get_face(hamr_grid* g, int d, int which, double* out);
/* edge EMF E_f (extent n+1 along the two directions != f). */
int hamr_get_edge(hamr_grid* g, int f, double* out);
int hamr_get_ctop(hamr_grid* g, double ctop[3]); /* per-direction max signal speed of the last corrector pass */
/* conserved totals sum_zones U[c] dV, c = 0..4, of the current state */
int hamr_totals(hamr_grid* g, double tot[5]);
/* Per-kernel device timers.  Between hamr_profile_begin and hamr_profile_end every kernel launch on
 * the grid's stream is bracketed by a CUDA event pair; _end synchronises and returns, per kernel
 * class c < HAMR_NKCLASS, the summed device time ms[c] and the number of launches count[c].
 * nclass must be >= HAMR_NKCLASS. */
#define HAMR_NKCLASS 10
int hamr_profile_begin(hamr_grid* g);
int hamr_profile_end(hamr_grid* g, int nclass, double ms[], long long count[]);
const char* hamr_profile_class_name(int c); /* "" if out of range */
/* kernel launches issued on this grid's stream since creation */
int hamr_launch_count(const hamr_grid* g, long long* n);


/* ---- geometry tables (C-1) -------------------------------------------------------- */
/* Copies one record table of refinement level `level` (0, or 1 on a grid with x1 refinement) to the host.
 * kind 0: zone centres, 32 doubles per entry: g_11 g_13 g_22 g_33 | gamma^11 gamma^13 gamma^22 gamma^33 | alpha
 * 1/alpha beta^1/alpha beta^1 | sqrt(-g) 1/sqrt(-g) d_1 ln sqrt(-g) d_2 ln sqrt(-g) | H1[7] H2[7] | 2 pad, where
 * H_nu = x^nu-derivatives of (g_00 g_01 g_03 g_11 g_13 g_22 g_33), the diagonal ones halved;
 * kind 1, 2, 3: x1-, x2-, x3-faces, 16 doubles per entry: g_11 g_13 g_22 g_33 | alpha 1/alpha beta^1/alpha beta^1 |
 * -alpha^2 g^tt g^dd g^td | sqrt(-g) 1/sqrt(-g) | 2 pad.
 * Entry (ti, tj), ti < *e1, tj < *e2, is zone / face index (ti - 3, tj - 3) of the table's level (ghosts included).
 * out may be NULL to query the extents; otherwise it holds e1 * e2 * nrec doubles. */
int hamr_debug_geometry(hamr_grid* g, int kind, int level, double* out, int* e1, int* e2, int* nrec);

/* ---- per-zone physics on caller-supplied states (C-2 .. C-4, C-13) ------------------------------------ */
/* n states; state s uses the centre geometry of table entry (ti[s], tj[s]) of level 0.  All arrays are host arrays,
 * state-major: prims n x 8 (rho, u, ut1..3, B1..3), U n x 5 (densitised hydro rows). */
int hamr_debug_prim2cons(hamr_grid* g, int n, const int* ti, const int* tj, const double* prims, double* U);
/* The inversion as the update kernel runs it: U (n x 5), new cell-centred field Bc (n x 3), guess (n x 5) ->
 * out (n x 5) and rc (n): 0 ok, 1 failed (out then holds the guess, as the kernels keep it). */
int hamr_debug_con2prim(hamr_grid* g, int n, const int* ti, const int* tj, const double* U, const double* Bc,
                        const double* guess, double* out, int* rc);
/* Floors and Lorentz-factor ceiling applied to P (n x 5, in place); flags[s] bit 0: rho floor, 1: u floor,
 * 2: ceiling.  The floor of state s is that of x1 table index ti[s]. */
int hamr_debug_floors(hamr_grid* g, int n, const int* ti, const int* tj, double* P, int* flags);

/* ---- robust inversion path (C-18, C-19) ------------------------------------------------------------------ */
/* kappa = (entropy row) / (density row) that the latest update stage advected, on the active zones (N1*N2*N3), before
 * it was reset from the new primitives.  entropy_backup grids only. */
int hamr_debug_kappa(hamr_grid* g, double* out);
/* The entropy inversion as the update kernel runs it: U (n x 5; the energy row U[.][1] is not read), entropy row US (n),
 * new field Bc (n x 3), guess (n x 5) -> out (n x 5), rc (n): 0 ok, 1 no admissible root (out then holds the guess). */
int hamr_debug_con2prim_entropy(hamr_grid* g, int n, const int* ti, const int* tj, const double* U, const double* US,
                                const double* Bc, const double* guess, double* out, int* rc);
/* The Aitken-accelerated inversion (C-21) as the update kernels run it where the Newton-Raphson one did not
 * converge: arguments and codes as hamr_debug_con2prim.  hamr_debug_aitken_count: zones, since the last call, whose
 * primitives came from it (entropy_backup grids). */
int hamr_debug_con2prim_aitken(hamr_grid* g, int n, const int* ti, const int* tj, const double* U, const double* Bc,
                               const double* guess, double* out, int* rc);
int hamr_debug_aitken_count(hamr_grid* g, long long* n);
/* hamr_debug_floors with the zone's field Bc (n x 3): drift-frame floors (C-19) when the grid has drift_floors = 1 */
int hamr_debug_floors_drift(hamr_grid* g, int n, const int* ti, const int* tj, double* P, const double* Bc, int* flags);

/* ---- FP64 pipe peak ("measure it with an FMA-chain microbenchmark") ---------------------------------- */
/* Runs `iters` rounds of 8 independent dependent-chains of FP64 instructions per thread on every SM of the current
 * device (stream = cudaStream_t cast to void*, NULL = default) and returns the device time of the timed launch and
 * the thread-level FP64 instructions it executed.  mix 0: all DFMA (peak FLOP rate = 2 x instructions / time);
 * mix 1: the flux kernels' blend, one third DFMA and two thirds DADD / DMUL (the pipe issues all three at the same
 * rate, so the instruction rate is the same and the FLOP rate is 4/3 x instructions / time);
 * mix 2: the flux kernels' whole instruction blend: per three FP64 arithmetic instructions one double compare-and-select
 * (DSETP + 2 FSEL) and two integer instructions (three in SASS), i.e. 4 FP64-pipe instructions to 5 others
 * (k_flux_ring: about 380 to 430 per face); thread_instructions then counts the FP64-pipe instructions (arithmetic + compares).  What this rate
 * falls short of mix 1's is what the other instructions cost the FP64 pipe in issue slots. */
int hamr_bench_fp64(void* cuda_stream, int mix, int iters, double* seconds, double* thread_instructions);

#ifdef __cplusplus
}
#endif
#endif /* HAMR_DEBUG_H */
