// ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT.
//
// Plain, slow, fp64 CPU restatement of the H-AMR per-zone GRMHD update (Liska et al.,
// arXiv:1912.10192; /root/reference/PAPER.md).  It exists to check the CUDA library against and
// to be timed as the CPU baseline.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may load it.  It shares no code with
// paper_1912_10192_b200/ (no headers, helpers, tables or constants) and never calls it.
//
// The paper prints one equation (Eq. 1) and names every ingredient by citation
// (PAPER.md:41 HLLE + PPM + 2nd-order time stepping + log-r Kerr-Schild grid; PAPER.md:47
// staggered CT with velocity-upwinded EMFs, sources at centres; PAPER.md:49 Newton-Raphson
// inversion; PAPER.md:59 floors; PAPER.md:93 fn.2 harmonic dt).  The formulas are the standard
// ones of those citations as read in DESIGN.md §3 ("C-n" below = that reading).
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): see DESIGN.md §4.  Readings that no pin can
// distinguish from a reasonable alternative are listed there as "parity unpinned".
#pragma once
#include <cmath>
#include <cstdint>
#include <vector>
#include <string>

namespace orc {

constexpr int NG = 3;  // ghost layers: PPM face stencil j-3..j+2 (C-5)

// ---- parameters (C layout; mirrored by tests/_orc.py with ctypes) -----------------------------
struct Params {
  int32_t metric;        // 0 Minkowski (Cartesian), 1 Kerr-Schild in x1=ln r, x2=theta, x3=phi
  int32_t recon;         // 0 PPM, 1 PLM with MC limiter
  int32_t n[3];          // base zones
  int32_t bc_lo[3], bc_hi[3];  // 0 periodic, 1 outflow, 2 polar reflect
  int32_t nb[3];         // block size; 0,0,0 -> one block
  int32_t n_deref;       // number of phi-derefinement thresholds (C-15)
  int32_t deref_factor[4];
  int32_t lat_max_level; // C-17; 0 -> global dt
  int32_t map;
  int32_t entropy_backup;  // C-18 (NEXT-2): advect the entropy, invert with it where the energy inversion fails
  int32_t drift_floors;    // C-19 (NEXT-2): floors inject mass / energy in the drift frame instead of the fluid frame
  double a;              // spin
  double xmin[3], xmax[3];   // PHYSICAL extents ((r_in,r_out),(0,pi),(0,2pi)) or box
  double gamma_ad, cour;
  double rho_fl_coef, rho_fl_pow, u_fl_coef, u_fl_pow;  // floor = coef * r^pow (r=1 Cartesian)
  double gamma_max;
  double deref_theta_deg[4];
  double r_refine_max;   // C-16; <=0 none
};

// ---- geometry (C-1) -----------------------------------------------------------------------------
struct Geom {
  double gcov[4][4], gcon[4][4];
  double gdet;           // sqrt(-g) of the internal coordinates
  double alpha;          // lapse
  double beta[3];        // shift beta^i, i=1..3
};

// Metric of the internal coordinates at (x1, x2); x2 outside (0,pi) is mirrored (C-1).
// `singular` (pole) fills zeros and gdet=0: such records are never used (C-7, C-9).
void geom_at(int metric, double a, double x1, double x2, Geom& G);
// Christoffel symbols conn[lam][mu][nu] = Gamma^lam_{mu nu} from ANALYTIC metric derivatives.
void conn_at(int metric, double a, double x1, double x2, double conn[4][4][4]);
// covariant metric and its x1-, x2-derivatives in internal coordinates (used by conn_at; exported
// for the pins)
void gcov_and_derivs(int metric, double a, double x1, double x2, double g[4][4], double dg1[4][4],
                     double dg2[4][4]);

// ---- per-zone physics (C-2..C-7, C-12, C-13) -----------------------------------------------------
// primitives P = (rho, u, ut1, ut2, ut3, B1, B2, B3)
struct State {
  double ucon[4], ucov[4], bcon[4], bcov[4], bsq, gamma;
};
void get_state(const double P[8], const Geom& G, State& S);
void prim_to_U(const double P[8], const State& S, const Geom& G, double gam, double U[8]);
void prim_to_F(const double P[8], const State& S, const Geom& G, double gam, int dir, double F[8]);
void wavespeeds(const double P[8], const State& S, const Geom& G, double gam, int dir,
                double& vmin, double& vmax);
void source(const double P[8], const State& S, const Geom& G, const double conn[4][4][4],
            double gam, double Ssrc[5]);
// returns 0 ok, >0 failure code; P_out[0..4] hydro primitives (B untouched = input Bc)
int con2prim(const double U[5], const double Bc[3], const Geom& G, double gam,
             const double Pguess[5], double Pout[5], int* iters);

// C-21: the Aitken-accelerated fixed-point inversion, same arguments and codes as con2prim
int con2prim_aitken(const double U[5], const double Bc[3], const Geom& G, double gam,
                    const double Pguess[5], double Pout[5], int* iters);

// ---- C-18 entropy as a backup for the energy equation (Noble et al. 2009) ------------------------
// kappa = p / rho^gamma_ad = (gamma_ad - 1) u / rho^gamma_ad: constant along smooth flow lines
double entropy_kappa(double rho, double u, double gam);
// conserved entropy and its flux along dir (1..3): gdet rho kappa u^t, gdet rho kappa u^dir
void entropy_UF(const double P[8], const State& S, const Geom& G, double gam, int dir, double& US, double& FS);
// inversion with the entropy row US in place of the energy row U[1] (which is not read): a 1-unknown root find.
// returns 0 ok, 1 no convergence / no bracket, 2 non-finite or non-positive D or US
int con2prim_entropy(const double U[5], double US, const double Bc[3], const Geom& G, double gam,
                     const double Pguess[5], double Pout[5], int* iters);

// ---- reconstruction (C-5) ------------------------------------------------------------------------
// zone j's parabola edges from a[j-2..j+2] given as a[0..4]
void ppm_zone(const double a[5], double& aL, double& aR);
void plm_zone(const double a[3], double& aL, double& aR);

// ---- HLL (C-7) -----------------------------------------------------------------------------------
void hll(const double UL[8], const double UR[8], const double FL[8], const double FR[8],
         double cmin, double cmax, double F[8]);

}  // namespace orc
