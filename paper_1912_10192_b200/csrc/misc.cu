// misc.cu — small kernels around the hot path: Courant dt finisher, dense <-> padded
// transfers for the C-ABI, div B diagnostic (C-11), conserved totals, finite check.
#include "hamr_host.h"

namespace hamr {

// C-14 (PAPER.md:93 fn. 2): 1/dt = sum_d 1/dt_d, dt_d = C dx^d / max ctop_d.  One thread; dt never
// leaves the device between steps.
// mode 0: set dt from ctop; 1: advance t by the dt just used, then set dt; 2: only latch ctop
__global__ void k_dt(Dev Dv, int mode) {
  double* s = Dv.scal;
  if (mode == 1) {
    s[S_T] += s[S_DT];
    s[S_DTLAST] = s[S_DT];
  }
  double sum = 0.0;
  for (int d = 0; d < 3; d++) {
    sum += s[S_CTOP0 + d] / Dv.dx[d];
    s[S_CTOPL0 + d] = s[S_CTOP0 + d];
    s[S_CTOP0 + d] = 0.0;  // ready for the next corrector pass
  }
  if (mode != 2) s[S_DT] = Dv.cour / sum;
}

// NEXT-4 (x1 slabs): the Courant maxima leave the grid for the max over all slabs (one global step) ...
__global__ void k_ctop_out(Dev Dv, double* __restrict__ out3) {
  for (int d = 0; d < 3; d++) out3[d] = Dv.scal[S_CTOP0 + d];
}
// ... and come back reduced: the arithmetic of k_dt on them
__global__ void k_dt_slab(Dev Dv, const double* __restrict__ in3, int advance) {
  double* s = Dv.scal;
  if (advance) {
    s[S_T] += s[S_DT];
    s[S_DTLAST] = s[S_DT];
  }
  double sum = 0.0;
  for (int d = 0; d < 3; d++) {
    sum += in3[d] / Dv.dx[d];
    s[S_CTOPL0 + d] = in3[d];
    s[S_CTOP0 + d] = 0.0;
  }
  s[S_DT] = Dv.cour / sum;
}

void launch_ctop_out(hamr_grid* g, double* out3) {
  Launch l_(g, K_DT);
  k_ctop_out<<<1, 1, 0, g->stream>>>(g->D, out3);
}
void launch_dt_slab(hamr_grid* g, const double* in3, bool advance) {
  Launch l_(g, K_DT);
  k_dt_slab<<<1, 1, 0, g->stream>>>(g->D, in3, advance ? 1 : 0);
}

__global__ void k_zero_ctop(Dev Dv) {
  Dv.scal[S_CTOP0] = Dv.scal[S_CTOP1] = Dv.scal[S_CTOP2] = 0.0;
}

void launch_dt(hamr_grid* g, int mode) {
  Launch l_(g, K_DT);
  k_dt<<<1, 1, 0, g->stream>>>(g->D, mode);
}

// dense (m0, m1, m2), x3 fastest  ->  padded array; zero_pole: Bf^2 on the polar axis is 0 (C-12)
__global__ void k_pack(Dev Dv, const double* __restrict__ dense, double* __restrict__ padded, int m0, int m1,
                       int m2, int zero_pole) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (long long)m0 * m1 * m2) return;
  const int k = (int)(t % m2), j = (int)((t / m2) % m1), i = (int)(t / ((long long)m2 * m1));
  double v = dense ? dense[t] : 0.0;
  if (zero_pole && Dv.metric == HAMR_METRIC_KERR_SCHILD && (j == 0 || j == Dv.L.n[1])) v = 0.0;
  padded[Dv.L.idx(i, j, k)] = v;
}

__global__ void k_unpack(Dev Dv, const double* __restrict__ padded, double* __restrict__ dense, int m0, int m1,
                         int m2) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (long long)m0 * m1 * m2) return;
  const int k = (int)(t % m2), j = (int)((t / m2) % m1), i = (int)(t / ((long long)m2 * m1));
  dense[t] = padded[Dv.L.idx(i, j, k)];
}

void launch_pack(hamr_grid* g, const double* dense, double* padded, int stag, bool zero_pole) {
  int m[3] = {g->D.L.n[0], g->D.L.n[1], g->D.L.n[2]};
  if (stag >= 0) m[stag] += 1;
  const long long tot = (long long)m[0] * m[1] * m[2];
  Launch l_(g, K_OTHER);
  k_pack<<<(unsigned)((tot + 255) / 256), 256, 0, g->stream>>>(g->D, dense, padded, m[0], m[1], m[2],
                                                                 zero_pole ? 1 : 0);
}

void launch_unpack(hamr_grid* g, const double* padded, double* dense, const int m[3]) {
  const long long tot = (long long)m[0] * m[1] * m[2];
  Launch l_(g, K_OTHER);
  k_unpack<<<(unsigned)((tot + 255) / 256), 256, 0, g->stream>>>(g->D, padded, dense, m[0], m[1], m[2]);
}

// C-11, two passes: max denominator, then max |div| / den over zones with den > 1e-12 denmax
__global__ void k_divb(Dev Dv, Fields s, int pass) {
  const Lay& L = Dv.L;
  const long long tot = (long long)L.n[0] * L.n[1] * L.n[2];
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  double val = 0.0;
  if (t < tot) {
    const int k = (int)(t % L.n[2]), j = (int)((t / L.n[2]) % L.n[1]), i = (int)(t / ((long long)L.n[2] * L.n[1]));
    const long long z = L.idx(i, j, k);
    const long long S[3] = {L.S1, L.S2, 1};
    double div = 0.0, den = 0.0;
    for (int d = 0; d < 3; d++) {
      const double lo = s.Bf[d][z], hi = s.Bf[d][z + S[d]];
      div += (hi - lo) / Dv.dx[d];
      den += (fabs(hi) + fabs(lo)) / (2.0 * Dv.dx[d]);
    }
    if (pass == 0) val = den;
    else if (den > 1e-12 * Dv.scal[S_DENMAX]) val = fabs(div) / den;
  }
  val = warp_max(val);
  if ((threadIdx.x & 31) == 0 && val > 0.0) atomic_max_pos(Dv.scal + (pass == 0 ? S_DENMAX : S_DIVB), val);
}

__global__ void k_zero_scal(Dev Dv, int first, int count) {
  for (int c = 0; c < count; c++) Dv.scal[first + c] = 0.0;
}

void launch_divb(hamr_grid* g, const Fields& s) {
  const Lay& L = g->D.L;
  const long long tot = (long long)L.n[0] * L.n[1] * L.n[2];
  const unsigned nb = (unsigned)((tot + 255) / 256);
  Launch l_(g, K_OTHER);
  g->launches += 2;
  k_zero_scal<<<1, 1, 0, g->stream>>>(g->D, S_DENMAX, 2);
  k_divb<<<nb, 256, 0, g->stream>>>(g->D, s, 0);
  k_divb<<<nb, 256, 0, g->stream>>>(g->D, s, 1);
}

// sum over active zones of U[c] dV (conservation diagnostic, P10)
__global__ void k_totals(Dev Dv, Fields s) {
  const Lay& L = Dv.L;
  const long long tot = (long long)L.n[0] * L.n[1] * L.n[2];
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  double U[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
  if (t < tot) {
    const int k = (int)(t % L.n[2]), j = (int)((t / L.n[2]) % L.n[1]), i = (int)(t / ((long long)L.n[2] * L.n[1]));
    const long long z = L.idx(i, j, k);
    const CGeo G = load_cgeo(Dv.gcA + (size_t)L.idx2(i, j) * NREC_C);
    double P[8];
    for (int c = 0; c < 5; c++) P[c] = s.P[c][z];
    for (int c = 0; c < 3; c++) P[5 + c] = s.Bc[c][z];
    St S;
    get_state(P, G, S);
    prim_to_U5(P, S, G.gdet, Dv.gam, U);
    const double dV = Dv.dx[0] * Dv.dx[1] * Dv.dx[2];
    for (int c = 0; c < 5; c++) U[c] *= dV;
  }
  for (int c = 0; c < 5; c++) {
    double v = U[c];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) atomicAdd(Dv.scal + S_TOT0 + c, v);
  }
}

void launch_totals(hamr_grid* g, const Fields& s) {
  const Lay& L = g->D.L;
  const long long tot = (long long)L.n[0] * L.n[1] * L.n[2];
  Launch l_(g, K_OTHER);
  g->launches += 1;
  k_zero_scal<<<1, 1, 0, g->stream>>>(g->D, S_TOT0, 5);
  k_totals<<<(unsigned)((tot + 255) / 256), 256, 0, g->stream>>>(g->D, s);
}

__global__ void k_check_finite(Dev Dv, Fields s) {
  const Lay& L = Dv.L;
  const long long tot = (long long)L.n[0] * L.n[1] * L.n[2];
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  int bad = 0;
  if (t < tot) {
    const int k = (int)(t % L.n[2]), j = (int)((t / L.n[2]) % L.n[1]), i = (int)(t / ((long long)L.n[2] * L.n[1]));
    const long long z = L.idx(i, j, k);
    for (int c = 0; c < 5; c++) bad |= !isfinite(s.P[c][z]);
    for (int c = 0; c < 3; c++) bad |= !isfinite(s.Bc[c][z]);
  }
  const unsigned m = __ballot_sync(0xffffffffu, bad);
  if ((threadIdx.x & 31) == 0 && m) atomicAdd(Dv.cnt + N_NONFINITE, (unsigned long long)__popc(m));
}

void launch_check_finite(hamr_grid* g, const Fields& s) {
  const Lay& L = g->D.L;
  const long long tot = (long long)L.n[0] * L.n[1] * L.n[2];
  Launch l_(g, K_OTHER);
  k_check_finite<<<(unsigned)((tot + 255) / 256), 256, 0, g->stream>>>(g->D, s);
}

// C-18: kappa = p / rho^gamma_ad of every zone of the stage's source state, ghosts included (run after
// the ghost fill), for the entropy flux of the generic flux kernels.  Slots no kernel reads (rho = 0) get 0.
// On a block grid the stage source of a block is in buffer set s (cur == 0) or s2 (cur == 2)
__global__ void k_kappa(Dev Dv, Fields s, Fields s2) {
  long long z = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  bool second = false;
  if (Dv.B.nblk > 0) {          // the blocks of the launch's list (under LAT: one time level)
    const long long slot = z / Dv.B.blen;
    if (slot >= Dv.B.nact) return;
    const int b = __ldg(Dv.B.list + slot);
    z = (long long)b * Dv.B.blen + (z - slot * Dv.B.blen);
    second = Dv.B.cur[b] != 0;
  } else if (z >= Dv.L.len) return;
  const double rho = (second ? s2.P[0] : s.P[0])[z], u = (second ? s2.P[1] : s.P[1])[z];
  Dv.K[z] = rho > 0.0 ? kappa_of(rho, u, Dv.gam) : 0.0;
}

void launch_kappa(hamr_grid* g, const Dev& Dv, const Fields& s, const Fields& s2) {
  const long long tot = Dv.B.nblk > 0 ? (long long)Dv.B.nact * Dv.B.blen : Dv.L.len;
  if (tot == 0) return;
  Launch l_(g, K_OTHER);
  k_kappa<<<(unsigned)((tot + 255) / 256), 256, 0, g->stream>>>(Dv, s, s2);
}

void launch_zero_ctop(hamr_grid* g) {
  Launch l_(g, K_OTHER);
  k_zero_ctop<<<1, 1, 0, g->stream>>>(g->D);
}

}  // namespace hamr
