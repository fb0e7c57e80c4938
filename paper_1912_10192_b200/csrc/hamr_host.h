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
enum Cnt { N_C2PFAIL = 0, N_RHOFL, N_UFL, N_GCEIL, N_NONFINITE, NCNT = 8 };

struct Dev {                 // everything a kernel may need, passed by value
  Lay L;
  int metric, recon;
  int bc_lo[3], bc_hi[3];
  double dx[3], x0[3];       // internal-coordinate spacing and origin
  double a, gam, cour, gamma_max;
  double rho_fl_coef, rho_fl_pow, u_fl_coef, u_fl_pow;
  const double* gc;          // geometry at centres  [NGEO][n2d]
  const double* gf1;         // at x1-faces
  const double* gf2;         // at x2-faces (pole rows: gdet = 0)
  const double* dgc;         // [2][NDG][n2d]: d_1 g, d_2 g at centres
  const double* rho_fl;      // [e1] floor per x1 index
  const double* u_fl;
  double* F[3][5];           // hydro fluxes on d-faces
  double* EfA[3];            // on d-faces: E_e, (d,e,f) cyclic  (C-8)
  double* EfB[3];            // on d-faces: E_f
  double* Ee[3];             // edge EMFs (C-9)
  double* Cc[3];             // centre EMFs (C-8)
  double* scal;              // [NSCAL]
  unsigned long long* cnt;   // [NCNT]
};

}  // namespace hamr

namespace hamr {
// kernel classes for the per-kernel timers (hamr_profile_*)
enum KClass { K_GHOSTS = 0, K_FLUX1, K_FLUX2, K_FLUX3, K_CEMF, K_EDGE, K_UPDATE_P, K_UPDATE_C, K_DT, K_OTHER, NKCLASS };
}

struct hamr_grid {
  hamr_params par;
  hamr::Dev D;
  hamr::Fields s[3];         // rotating: sn (time n), sh (n+1/2), snew
  int isn, ish, inew;
  void* arena;               // device memory base
  size_t arena_bytes;
  bool own_arena, own_stream;
  cudaStream_t stream;
  double* stage;             // device staging buffer for dense <-> padded transfers
  size_t stage_doubles;
  double* h_pinned;          // small pinned host buffer for scalar read-back
  bool have_state, dead;
  long long launches;
  std::string err;
  // per-kernel timers: CUDA event pairs on the grid's stream around every launch while enabled
  bool prof;
  std::vector<cudaEvent_t> ev;   // pairs: start, stop
  std::vector<int> ev_cls;
  size_t ev_used;
};

namespace hamr {
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
void launch_geometry(hamr_grid* g, double* gc, double* gf1, double* gf2, double* dgc, double* rho_fl,
                     double* u_fl);
void launch_ghosts(hamr_grid* g, const Fields& s, bool bc_active_too);
void launch_flux(hamr_grid* g, const Fields& src, bool want_ctop);
void launch_ct(hamr_grid* g, const Fields& src);
void launch_update(hamr_grid* g, const Fields& src, const Fields& base, const Fields& out, double dtfac,
                   bool src_is_base);
void launch_dt(hamr_grid* g, int mode);  // 0 set dt, 1 advance t + set dt, 2 latch ctop only
void launch_pack(hamr_grid* g, const double* dense, double* padded, int stag, bool zero_pole);
void launch_unpack(hamr_grid* g, const double* padded, double* dense, const int m[3]);
void launch_divb(hamr_grid* g, const Fields& s);
void launch_totals(hamr_grid* g, const Fields& s);
void launch_check_finite(hamr_grid* g, const Fields& s);
void launch_zero_ctop(hamr_grid* g);

}  // namespace hamr
