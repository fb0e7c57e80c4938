// update.cu — face-B update, geometric source, conservative update, conserved-to-primitive inversion,
// floors and ceiling in ONE kernel (SURVEY §8(a) H2 second half, H3, H4; north_star items 3-5).
// "the source terms are added at cell centers to compute the cell-centered values of the
// conserved quantities U at the new time"; "(multi-)dimensional Newton-Raphson ...
// Noble et al. 2006"; floors.  DESIGN.md C-10, C-12, C-13.
// The conserved vector never touches HBM: U_base, div F, S and the inversion stay in registers.
#include "hamr_host.h"

namespace hamr {

// face-B update of the d-face on the low side of z (C-10):
// Bf^d -= dt [ (E_f(e+) - E_f(e-))/dx^e - (E_e(f+) - E_e(f-))/dx^f ], (d,e,f) cyclic
// All index arithmetic is 32-bit (an array holds fewer than 2^31 doubles, checked at creation).
template <int d>
__device__ __forceinline__ double bf_new(const Dev& Dv, const double* __restrict__ base, int z, double dt,
                                         const int S[3], const double idx[3]) {
  constexpr int e = (d + 1) % 3, f = (d + 2) % 3;
  const double curl = (__ldg(Dv.Ee[f] + z + S[e]) - __ldg(Dv.Ee[f] + z)) * idx[e] -
                      (__ldg(Dv.Ee[e] + z + S[f]) - __ldg(Dv.Ee[e] + z)) * idx[f];
  return __ldg(base + z) - dt * curl;
}

template <bool BLK>
__device__ __forceinline__ Fields pick_fields(const Fields& a, const Fields& b, int cur) {
  Fields f;
#pragma unroll
  for (int c = 0; c < 5; c++) f.P[c] = selp<BLK>(a.P[c], b.P[c], cur);
#pragma unroll
  for (int c = 0; c < 3; c++) { f.Bc[c] = selp<BLK>(a.Bc[c], b.Bc[c], cur); f.Bf[c] = selp<BLK>(a.Bf[c], b.Bf[c], cur); }
  return f;
}

// generic kernel: 6 CTAs of 128 threads per SM for the corrector (80 registers), 5 for the predictor (96, no spills):
// measured best of 3-7 on cfg 2 (profiles/r2_experiments.md)
constexpr int UPD_MINB = 6, UPD_MINB_PRED = 5;
// ROB (monolithic grids): the robust path.  With Dv.entropy the entropy row is advanced beside the
// others and inverts the zones whose energy inversion failed or came back with rho <= 0 or u < 0 (C-18); with Dv.drift
// the floors add mass and energy in the drift frame (C-19).
template <bool SAME, bool BLK, bool ROB = false>  // SAME: predictor, source state == base state
__global__ void __launch_bounds__(128, ROB ? 4 : (SAME ? UPD_MINB_PRED : UPD_MINB)) k_update(Dev Dv, Roles ra, Roles rb, double dtfac) {
  const Lay& L = Dv.L;
  // k runs over [0, n3): warps start on 128-byte lines when n3 is a multiple of 32; the thread at k = 0 also
  // builds the x3-face at k = n3
  const int c2 = L.n[2], c1 = L.n[1] + 1;
  const unsigned per = (unsigned)(L.n[0] + 1) * c1 * c2;
  unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = t < (BLK ? per * Dv.B.nact : per);
  int nfail = 0, nrf = 0, nuf = 0, ngc = 0, bad = 0, nent = 0, nait = 0;
  if (valid) {
    int bslot = 0;
    if (BLK) { bslot = (int)(t / per); t -= bslot * per; }
    const BCtx C = blk_ctx<BLK>(Dv, bslot);
    const Fields src = pick_fields<BLK>(ra.src, rb.src, C.cur), base = pick_fields<BLK>(ra.base, rb.base, C.cur),
                 out = pick_fields<BLK>(ra.out, rb.out, C.cur);
    const unsigned tj = t / (unsigned)c2;
    const int k = (int)(t - tj * c2);
    const int i = (int)(tj / (unsigned)c1);
    const int j = (int)(tj - i * c1);
    const int z = C.zoff + (int)L.idx(i, j, k);
    const double dt = dtfac * Dv.scal[S_DT];
    const int S[3] = {L.S1, L.S2, 1};
    const double idx[3] = {1.0 / ((BLK && C.lev) ? 0.5 * Dv.dx[0] : Dv.dx[0]), 1.0 / Dv.dx[1], 1.0 / Dv.dx[2]};
    const bool in0 = i < L.n[0], in1 = j < L.n[1];
    const bool ks = Dv.metric == HAMR_METRIC_KERR_SCHILD;
    const int Jg = C.J0 + j, n2g = BLK ? Dv.B.n2g : L.n[1];
    double lo[3] = {0.0, 0.0, 0.0};
    if (in1) { lo[0] = bf_new<0>(Dv, base.Bf[0], z, dt, S, idx); out.Bf[0][z] = lo[0]; }
    if (in0) {
      lo[1] = (ks && (Jg == 0 || Jg == n2g)) ? 0.0 : bf_new<1>(Dv, base.Bf[1], z, dt, S, idx);
      out.Bf[1][z] = lo[1];
    }
    if (in0 && in1) {
      lo[2] = bf_new<2>(Dv, base.Bf[2], z, dt, S, idx);
      out.Bf[2][z] = lo[2];
      if (k == 0) out.Bf[2][z + L.n[2]] = bf_new<2>(Dv, base.Bf[2], z + L.n[2], dt, S, idx);
      const double* grec = Dv.gcA + (BLK ? C.lev * Dv.B.tlevA : 0) + (size_t)(C.q0 + i * (BLK ? Dv.B.ge2 : L.e2) + j) * NREC_C;
      const CGeo G = load_cgeo(grec);
      // new cell-centred field from the new faces (the high faces are recomputed, bit-identically)
      double Bn[3];
      {
        const double h0 = bf_new<0>(Dv, base.Bf[0], z + S[0], dt, S, idx);
        const double h1 = (ks && Jg + 1 == n2g) ? 0.0 : bf_new<1>(Dv, base.Bf[1], z + S[1], dt, S, idx);
        double h2 = bf_new<2>(Dv, base.Bf[2], z + S[2], dt, S, idx), l2 = lo[2];
        if (Dv.mrow) {
          // C-15: in a phi-derefined row B_c^3 is the GROUP's value, from the group's two outer x3-faces
          const int m = __ldg(Dv.mrow + Jg + NG);
          if (m > 1) {
            const int zg = z - (k % m);
            l2 = bf_new<2>(Dv, base.Bf[2], zg, dt, S, idx);
            h2 = bf_new<2>(Dv, base.Bf[2], zg + m, dt, S, idx);
          }
        }
        const double i2g = 0.5 * G.igdet;
        Bn[0] = (lo[0] + h0) * i2g;
        Bn[1] = (lo[1] + h1) * i2g;
        Bn[2] = (l2 + h2) * i2g;
      }
      double Ps[8], U[5], Ssrc1, Ssrc2;
#pragma unroll
      for (int c = 0; c < 5; c++) Ps[c] = __ldg(src.P[c] + z);
#pragma unroll
      for (int c = 0; c < 3; c++) Ps[5 + c] = __ldg(src.Bc[c] + z);
      {
        St Ss;
        get_state(Ps, G, Ss);
        if (SAME) prim_to_U5(Ps, Ss, G.gdet, Dv.gam, U);
        source_12(Ps, Ss, G, Dv.gam, grec, Ssrc1, Ssrc2);   // C-12: on the stage's source state
      }
      double rho_b = Ps[0], u_b = Ps[1];   // ROB: the base state's density and energy (C-18)
      if (!SAME) {
        double Pb[8];
#pragma unroll
        for (int c = 0; c < 5; c++) Pb[c] = __ldg(base.P[c] + z);
#pragma unroll
        for (int c = 0; c < 3; c++) Pb[5 + c] = __ldg(base.Bc[c] + z);
        St Sb;
        get_state(Pb, G, Sb);
        prim_to_U5(Pb, Sb, G.gdet, Dv.gam, U);
        rho_b = Pb[0]; u_b = Pb[1];
      }
      double US = 0.0;
      if (ROB && Dv.entropy) {
        // C-18: the entropy row of the base state is its density row times kappa; no source term
        double div = 0.0;
#pragma unroll
        for (int d = 0; d < 3; d++) div += (__ldg(Dv.FK[d] + z + S[d]) - __ldg(Dv.FK[d] + z)) * idx[d];
        US = U[0] * kappa_of(rho_b, u_b, Dv.gam) - dt * div;
      }
      // U_new = U_base - dt sum_d (F^d_+ - F^d_-)/dx^d + dt S
#pragma unroll
      for (int c = 0; c < 5; c++) {
        double div = 0.0;
#pragma unroll
        for (int d = 0; d < 3; d++) div += (__ldg(Dv.F[d][c] + z + S[d]) - __ldg(Dv.F[d][c] + z)) * idx[d];
        const double sc = (c == 2) ? Ssrc1 : (c == 3 ? Ssrc2 : 0.0);
        U[c] = U[c] - dt * div + dt * sc;
      }
      double Pn[5], Pg[5];
      // the geometry record and the guess are re-read (L1 / L2 hits) instead of being kept in registers
      // across the flux divergence: lower register pressure, more resident warps
      const double* gtab = grec;
      asm volatile("" : "+l"(gtab));
      const CGeo G2 = load_cgeo(gtab);
      const double* sp[5] = {src.P[0], src.P[1], src.P[2], src.P[3], src.P[4]};
#pragma unroll
      for (int c = 0; c < 5; c++) { const double* a = sp[c]; asm volatile("" : "+l"(a)); Pg[c] = a[z]; }
      int rc = con2prim(U, Bn, G2, Dv.gam, Pg, Pn);
      if (ROB && Dv.entropy) {
        Dv.K[z] = US / U[0];   // the advected kappa (diagnostic: k_kappa overwrites it before the next flux pass)
        if (rc != 0 || !(Pn[0] > 0.0) || !(Pn[1] >= 0.0)) {
          // the rare calls work on copies, so that the common path's U, Bn, Pg and record stay in registers
          double Pe[5], Uc[5], Bc[3], Pc[5];
          CGeo Gc = G2;
#pragma unroll
          for (int c = 0; c < 5; c++) { Uc[c] = U[c]; Pc[c] = Pg[c]; }
#pragma unroll
          for (int c = 0; c < 3; c++) Bc[c] = Bn[c];
          // C-21: the second primary inversion where Newton-Raphson did not converge
          if (rc != 0 && con2prim_aitken(Uc, Bc, &Gc, Dv.gam, Pc, Pe) == 0) {
#pragma unroll
            for (int c = 0; c < 5; c++) Pn[c] = Pe[c];
            rc = 0;
            nait = 1;
          }
          // C-18: the entropy row where no energy inversion gave an admissible state.  An entropy row that went
          // negative or has no root leaves what the energy inversion gave: its state for the floors, or its failure
          if ((rc != 0 || !(Pn[0] > 0.0) || !(Pn[1] >= 0.0)) && con2prim_entropy(Uc, US, Bc, &Gc, Dv.gam, Pc, Pe) == 0) {
#pragma unroll
            for (int c = 0; c < 5; c++) Pn[c] = Pe[c];
            rc = 0;
            nent = 1;
          }
        }
      }
      if (rc != 0) {  // C-13: keep the source state's hydro primitives, count the failure
        nfail = 1;
#pragma unroll
        for (int c = 0; c < 5; c++) Pn[c] = Pg[c];
      }
      // floors and Lorentz-factor ceiling (C-13)
      const int fi = C.I0 + i + NG + (BLK ? C.lev * Dv.B.flev : 0);
      const double rfl = __ldg(Dv.rho_fl + fi), ufl = __ldg(Dv.u_fl + fi);
      if (ROB && Dv.drift) {
        nrf = Pn[0] < rfl;
        nuf = Pn[1] < ufl;
        if (nrf | nuf) floors_drift(G2, Bn, Dv.gam, nrf ? rfl : Pn[0], nuf ? ufl : Pn[1], Pn);
        ceiling_only(G2, Dv.gamma_max, Pn, ngc);
      } else {
        floors_ceiling(G2, rfl, ufl, Dv.gamma_max, Pn, nrf, nuf, ngc);
      }
#pragma unroll
      for (int c = 0; c < 5; c++) {
        out.P[c][z] = Pn[c];
        if (!(fabs(Pn[c]) <= 1.79e308)) bad = 1;
      }
#pragma unroll
      for (int c = 0; c < 3; c++) out.Bc[c][z] = Bn[c];
    }
  }
  // warp-aggregated event counters
  const unsigned m_f = __ballot_sync(0xffffffffu, nfail), m_r = __ballot_sync(0xffffffffu, nrf),
                 m_u = __ballot_sync(0xffffffffu, nuf), m_g = __ballot_sync(0xffffffffu, ngc),
                 m_b = __ballot_sync(0xffffffffu, bad);
  if (ROB) {
    const unsigned m_e = __ballot_sync(0xffffffffu, nent), m_a = __ballot_sync(0xffffffffu, nait);
    if ((threadIdx.x & 31) == 0 && m_e) atomicAdd(Dv.cnt + N_ENTROPY, (unsigned long long)__popc(m_e));
    if ((threadIdx.x & 31) == 0 && m_a) atomicAdd(Dv.cnt + N_AITKEN, (unsigned long long)__popc(m_a));
  }
  if ((threadIdx.x & 31) == 0) {
    if (m_f) atomicAdd(Dv.cnt + N_C2PFAIL, (unsigned long long)__popc(m_f));
    if (m_r) atomicAdd(Dv.cnt + N_RHOFL, (unsigned long long)__popc(m_r));
    if (m_u) atomicAdd(Dv.cnt + N_UFL, (unsigned long long)__popc(m_u));
    if (m_g) atomicAdd(Dv.cnt + N_GCEIL, (unsigned long long)__popc(m_g));
    if (m_b) atomicAdd(Dv.cnt + N_NONFINITE, (unsigned long long)__popc(m_b));
  }
}

// ---- the same update on monolithic grids, staged through shared memory by bulk asynchronous copies (TMA) --------
// A CTA owns TJ consecutive x2 rows over the whole x3 extent and marches along x1.  Every array with reuse between
// zones (15 flux arrays: each value feeds two zones; 3 edge EMFs: eight uses; 3 base face fields: two uses) is brought
// in as ONE contiguous chunk per plane (rows j0 .. j0 + TJ, whole x3 pitch: the k + 1 and j + 1 neighbours come with
// it).  Arrays read at planes i and i + 1 (F^1, E_2, E_3, Bf^1) keep two planes (the march reuses plane i + 1 as the
// next step's plane i), the others one.  A step first consumes everything staged (new faces, new B_c, flux
// divergence), the CTA synchronises, one thread requests the next plane into the SAME buffers, and the long
// dependent part (states, source, Newton inversion, floors) runs while those copies land.  Zone-centred arrays
// without reuse (source / base state in, new state out) are read and written directly, requested at the top of the step.
namespace tile {
constexpr int TJ = 2;            // rows per CTA: 1 / 3 / 4 measured 5-19 % slower (profiles/r2_experiments.md)
constexpr int NA = 8, NB = 13;   // arrays keeping two planes / one plane
}

// ROB: the robust path of k_update above (C-18 entropy row and backup inversion, C-19 drift-frame floors).  The three
// entropy fluxes are not staged (a third CTA-plane set would halve the CTAs per SM): each zone reads its six values
// directly, requested with the zone-centred inputs at the top of the step.
constexpr bool PREFETCH_STATE = true;
template <bool SAME, int NT, bool ROB = false>
__global__ void __launch_bounds__(NT, 512 / NT) k_update_tile(Dev Dv, Roles r, double dtfac, int seg) {
  using namespace tile;
  using namespace tma;
  extern __shared__ __align__(128) double tile_mem[];
  const Lay& L = Dv.L;
  const int AS = (TJ + 1) * L.p3;                  // doubles per staged array and plane
  unsigned long long* full = reinterpret_cast<unsigned long long*>(tile_mem + (2 * NA + NB) * AS);
  const int t = threadIdx.x, lane = t & 31, w = t >> 5;
  const int wpr = (L.n[2] + 31) >> 5;              // warps per x3 row
  const int jj = w / wpr, k = (w - jj * wpr) * 32 + lane;
  const int j0 = blockIdx.x * TJ, j = j0 + jj;
  const int i0 = blockIdx.y * seg, i1 = min(i0 + seg, L.n[0] + 1);
  const bool live = jj < TJ && j <= L.n[1] && k < L.n[2];
  const bool in1 = j < L.n[1];
  const bool ks = Dv.metric == HAMR_METRIC_KERR_SCHILD;
  const double dt = dtfac * Dv.scal[S_DT];
  const double ix0 = 1.0 / Dv.dx[0], ix1 = 1.0 / Dv.dx[1], ix2 = 1.0 / Dv.dx[2];
  // class A: F^1[0..4], Ee[1], Ee[2], Bf^1 ; class B: F^2[0..4], F^3[0..4], Ee[0], Bf^2, Bf^3
  const double* srcA[NA] = {Dv.F[0][0], Dv.F[0][1], Dv.F[0][2], Dv.F[0][3], Dv.F[0][4], Dv.Ee[1], Dv.Ee[2], r.base.Bf[0]};
  const double* srcB[NB] = {Dv.F[1][0], Dv.F[1][1], Dv.F[1][2], Dv.F[1][3], Dv.F[1][4], Dv.F[2][0], Dv.F[2][1],
                            Dv.F[2][2], Dv.F[2][3], Dv.F[2][4], Dv.Ee[0], r.base.Bf[1], r.base.Bf[2]};
  const unsigned bytes = (unsigned)(AS * sizeof(double));
  const bool warp0 = t < 32;
  // request plane pa of the class A arrays (into the buffer of its parity) and / or plane pb of the class B arrays
  auto request = [&](int pa0, int pa1, int pb) {
    if (warp0 && elect_one()) {
      const int na = pa1 - pa0 + 1;
      mbar_expect(full, (unsigned)((na * NA + (pb >= 0 ? NB : 0)) * bytes));
      for (int pa = pa0; pa <= pa1; pa++) {
        const int zc = (int)L.idx(pa, j0, 0);
#pragma unroll
        for (int a = 0; a < NA; a++) bulk_g2s(tile_mem + (2 * a + (pa & 1)) * AS, srcA[a] + zc, bytes, full);
      }
      if (pb >= 0) {
        const int zc = (int)L.idx(pb, j0, 0);
#pragma unroll
        for (int b = 0; b < NB; b++) bulk_g2s(tile_mem + (2 * NA + b) * AS, srcB[b] + zc, bytes, full);
      }
    }
  };
  if (t == 0) {
    mbar_init(full, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  request(i0, i0 + 1, i0);
  int nfail = 0, nrf = 0, nuf = 0, ngc = 0, bad = 0, nent = 0, nait = 0;
  const int sk = jj * L.p3 + k;                    // this thread's element inside a staged chunk
  for (int i = i0; i < i1; i++) {
    const bool in0 = i < L.n[0];
    const bool zone = live && in0 && in1;
    const int z = (int)L.idx(i, j, k);
    // corrector: the zone-centred inputs of the NEXT plane (two whole rows per array: one contiguous chunk) are asked into
    // L2 now, so that the direct loads at the top of the next step, which its early state evaluation waits for, find them
    // there: 0.374 -> 0.335 ms on cfg 2.  The predictor, which uses its inputs after the staged part, loses by it
    // (0.276 -> 0.291 ms) and does without
    if (PREFETCH_STATE && !SAME && warp0 && i + 1 < L.n[0] && i + 1 < i1 && elect_one()) {
      const int zn = (int)L.idx(i + 1, j0, 0);
      const unsigned pb = (unsigned)(2 * L.p3 * sizeof(double));
#pragma unroll
      for (int c = 0; c < 5; c++) bulk_prefetch_l2(r.src.P[c] + zn, pb);
#pragma unroll
      for (int c = 0; c < 3; c++) bulk_prefetch_l2(r.src.Bc[c] + zn, pb);
      if (!SAME) {
#pragma unroll
        for (int c = 0; c < 5; c++) bulk_prefetch_l2(r.base.P[c] + zn, pb);
#pragma unroll
        for (int c = 0; c < 3; c++) bulk_prefetch_l2(r.base.Bc[c] + zn, pb);
      }
    }
    // zone-centred inputs without reuse: requested now, used after the staged part
    double Ps[8], Pb[8];
    if (zone) {
#pragma unroll
      for (int c = 0; c < 5; c++) Ps[c] = __ldg(r.src.P[c] + z);
#pragma unroll
      for (int c = 0; c < 3; c++) Ps[5 + c] = __ldg(r.src.Bc[c] + z);
      if (!SAME) {
#pragma unroll
        for (int c = 0; c < 5; c++) Pb[c] = __ldg(r.base.P[c] + z);
#pragma unroll
        for (int c = 0; c < 3; c++) Pb[5 + c] = __ldg(r.base.Bc[c] + z);
      }
    }
    double divK = 0.0;   // C-18: divergence of the entropy flux
    if (ROB && zone && Dv.entropy)
      divK = (__ldg(Dv.FK[0] + z + L.S1) - __ldg(Dv.FK[0] + z)) * ix0 + (__ldg(Dv.FK[1] + z + L.S2) - __ldg(Dv.FK[1] + z)) * ix1 +
             (__ldg(Dv.FK[2] + z + 1) - __ldg(Dv.FK[2] + z)) * ix2;
    // The corrector evaluates its two input states BEFORE the staged part (16 doubles of input become 7 of result
    // while the copies land: measured 0.393 -> 0.369 ms); the predictor, with one input state, is faster the other
    // way round (0.274 vs 0.293 ms)
    constexpr bool EARLY = !SAME;
    const double* grec = Dv.gcA + (size_t)((NG + i) * L.e2 + NG + j) * NREC_C;
    double U[5], S1 = 0.0, S2 = 0.0;
    if (EARLY && zone) {
      const CGeo G = load_cgeo(grec);
      St Ss, Sb;
      get_state(Ps, G, Ss);
      source_12(Ps, Ss, G, Dv.gam, grec, S1, S2);   // C-12: on the stage's source state
      get_state(Pb, G, Sb);
      prim_to_U5(Pb, Sb, G.gdet, Dv.gam, U);
    }
    mbar_wait(full, (unsigned)((i - i0) & 1));
    const double* A0 = tile_mem + (i & 1) * AS + sk;          // class A, plane i     (array a at + 2 a AS)
    const double* A1 = tile_mem + ((i + 1) & 1) * AS + sk;    // class A, plane i + 1
    const double* B0 = tile_mem + 2 * NA * AS + sk;           // class B, plane i     (array b at + b AS)
    const int p3 = L.p3;
    double Bn[3] = {0.0, 0.0, 0.0}, div[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    if (live) {
      // C-10: Bf^d -= dt [ (E_f(e+) - E_f(e-))/dx^e - (E_e(f+) - E_e(f-))/dx^f ], (d,e,f) cyclic; the low faces of the
      // zone are stored, the high faces are the neighbours' low faces recomputed from the same expression
      const double* E1a = A0 + 10 * AS;  const double* E1b = A1 + 10 * AS;   // Ee[1] at planes i, i + 1
      const double* E2a = A0 + 12 * AS;  const double* E2b = A1 + 12 * AS;   // Ee[2]
      const double* E0 = B0 + 10 * AS;                                        // Ee[0]
      const double* F0a = A0 + 14 * AS;  const double* F0b = A1 + 14 * AS;   // base Bf^1
      const double* Bf1 = B0 + 11 * AS;  const double* Bf2 = B0 + 12 * AS;
      const int Jg = j, n2g = L.n[1];
      const double lo0 = F0a[0] - dt * ((E2a[p3] - E2a[0]) * ix1 - (E1a[1] - E1a[0]) * ix2);
      const double hi0 = F0b[0] - dt * ((E2b[p3] - E2b[0]) * ix1 - (E1b[1] - E1b[0]) * ix2);
      double lo1 = Bf1[0] - dt * ((E0[1] - E0[0]) * ix2 - (E2b[0] - E2a[0]) * ix0);
      double hi1 = Bf1[p3] - dt * ((E0[p3 + 1] - E0[p3]) * ix2 - (E2b[p3] - E2a[p3]) * ix0);
      const double lo2 = Bf2[0] - dt * ((E1b[0] - E1a[0]) * ix0 - (E0[p3] - E0[0]) * ix1);
      const double hi2 = Bf2[1] - dt * ((E1b[1] - E1a[1]) * ix0 - (E0[p3 + 1] - E0[1]) * ix1);
      if (ks && (Jg == 0 || Jg == n2g)) lo1 = 0.0;     // C-12: no field through the polar axis
      if (ks && Jg + 1 == n2g) hi1 = 0.0;
      if (in1) r.out.Bf[0][z] = lo0;
      if (in0) r.out.Bf[1][z] = lo1;
      if (in0 && in1) {
        r.out.Bf[2][z] = lo2;
        if (k == 0) {   // the x3-face at k = n3 of this row
          const int q = L.n[2];
          r.out.Bf[2][z + q] = Bf2[q] - dt * ((E1b[q] - E1a[q]) * ix0 - (E0[p3 + q] - E0[q]) * ix1);
        }
        Bn[0] = lo0 + hi0; Bn[1] = lo1 + hi1; Bn[2] = lo2 + hi2;   // times 1 / (2 sqrt(-g)) below
#pragma unroll
        for (int c = 0; c < 5; c++)
          div[c] = (A1[2 * c * AS] - A0[2 * c * AS]) * ix0 + (B0[c * AS + p3] - B0[c * AS]) * ix1 +
                   (B0[(5 + c) * AS + 1] - B0[(5 + c) * AS]) * ix2;
      }
    }
    __syncthreads();   // everything staged for this plane has been read
    if (i + 1 < i1) request(i + 2, i + 2, i + 1);
    if (zone) {
      const CGeo G = load_cgeo(grec);
      const double i2g = 0.5 * G.igdet;
      Bn[0] *= i2g; Bn[1] *= i2g; Bn[2] *= i2g;
      if (!EARLY) {
        St Ss;
        get_state(Ps, G, Ss);
        prim_to_U5(Ps, Ss, G.gdet, Dv.gam, U);
        source_12(Ps, Ss, G, Dv.gam, grec, S1, S2);   // C-12: on the stage's source state
      }
      double US = 0.0;
      if (ROB && Dv.entropy) {   // C-18: the base state's entropy row is its density row times kappa; no source term
        const double rho_b = SAME ? Ps[0] : Pb[0], u_b = SAME ? Ps[1] : Pb[1];
        US = U[0] * kappa_of(rho_b, u_b, Dv.gam) - dt * divK;
      }
      // U_new = U_base - dt sum_d (F^d_+ - F^d_-)/dx^d + dt S
#pragma unroll
      for (int c = 0; c < 5; c++) {
        const double sc = (c == 2) ? S1 : (c == 3 ? S2 : 0.0);
        U[c] = U[c] - dt * div[c] + dt * sc;
      }
      double Pn[5];
      int rc = con2prim(U, Bn, G, Dv.gam, Ps, Pn);
      if (ROB && Dv.entropy) {
        Dv.K[z] = US / U[0];   // the advected kappa (diagnostic: k_kappa overwrites it before the next flux pass)
        if (rc != 0 || !(Pn[0] > 0.0) || !(Pn[1] >= 0.0)) {
          // the rare calls work on copies, so that the common path's U, Bn, Ps and record stay in registers
          double Pe[5], Uc[5], Bc[3], Pc[5];
          CGeo Gc = G;
#pragma unroll
          for (int c = 0; c < 5; c++) { Uc[c] = U[c]; Pc[c] = Ps[c]; }
#pragma unroll
          for (int c = 0; c < 3; c++) Bc[c] = Bn[c];
          // C-21: the second primary inversion where Newton-Raphson did not converge
          if (rc != 0 && con2prim_aitken(Uc, Bc, &Gc, Dv.gam, Pc, Pe) == 0) {
#pragma unroll
            for (int c = 0; c < 5; c++) Pn[c] = Pe[c];
            rc = 0;
            nait++;
          }
          // C-18: the entropy row where no energy inversion gave an admissible state.  An entropy row that went
          // negative or has no root leaves what the energy inversion gave: its state for the floors, or its failure
          if ((rc != 0 || !(Pn[0] > 0.0) || !(Pn[1] >= 0.0)) && con2prim_entropy(Uc, US, Bc, &Gc, Dv.gam, Pc, Pe) == 0) {
#pragma unroll
            for (int c = 0; c < 5; c++) Pn[c] = Pe[c];
            rc = 0;
            nent++;
          }
        }
      }
      if (rc != 0) {  // C-13: keep the source state's hydro primitives, count the failure
        nfail++;
#pragma unroll
        for (int c = 0; c < 5; c++) Pn[c] = Ps[c];
      }
      int frf = 0, fuf = 0, fgc = 0;
      const double rfl = __ldg(Dv.rho_fl + i + NG), ufl = __ldg(Dv.u_fl + i + NG);
      if (ROB && Dv.drift) {   // C-19
        frf = Pn[0] < rfl;
        fuf = Pn[1] < ufl;
        if (frf | fuf) floors_drift(G, Bn, Dv.gam, frf ? rfl : Pn[0], fuf ? ufl : Pn[1], Pn);
        ceiling_only(G, Dv.gamma_max, Pn, fgc);
      } else {
        floors_ceiling(G, rfl, ufl, Dv.gamma_max, Pn, frf, fuf, fgc);
      }
      nrf += frf; nuf += fuf; ngc += fgc;
#pragma unroll
      for (int c = 0; c < 5; c++) {
        r.out.P[c][z] = Pn[c];
        if (!(fabs(Pn[c]) <= 1.79e308)) bad = 1;
      }
#pragma unroll
      for (int c = 0; c < 3; c++) r.out.Bc[c][z] = Bn[c];
    }
  }
  // warp-aggregated event counters (a thread has seen many zones: sums, not flags)
  const int s_f = __reduce_add_sync(0xffffffffu, nfail), s_r = __reduce_add_sync(0xffffffffu, nrf),
            s_u = __reduce_add_sync(0xffffffffu, nuf), s_g = __reduce_add_sync(0xffffffffu, ngc),
            s_b = __reduce_add_sync(0xffffffffu, bad);
  if (ROB) {
    const int s_e = __reduce_add_sync(0xffffffffu, nent), s_a = __reduce_add_sync(0xffffffffu, nait);
    if (lane == 0 && s_e) atomicAdd(Dv.cnt + N_ENTROPY, (unsigned long long)s_e);
    if (lane == 0 && s_a) atomicAdd(Dv.cnt + N_AITKEN, (unsigned long long)s_a);
  }
  if (lane == 0) {
    if (s_f) atomicAdd(Dv.cnt + N_C2PFAIL, (unsigned long long)s_f);
    if (s_r) atomicAdd(Dv.cnt + N_RHOFL, (unsigned long long)s_r);
    if (s_u) atomicAdd(Dv.cnt + N_UFL, (unsigned long long)s_u);
    if (s_g) atomicAdd(Dv.cnt + N_GCEIL, (unsigned long long)s_g);
    if (s_b) atomicAdd(Dv.cnt + N_NONFINITE, (unsigned long long)s_b);
  }
}

template <bool SAME, int NT, bool ROB = false>
static void launch_tile_t(hamr_grid* g, const Dev& Dv, const Roles& r, double dtfac) {
  using namespace tile;
  const Lay& L = Dv.L;
  const size_t smem = (size_t)(2 * NA + NB) * (TJ + 1) * L.p3 * sizeof(double) + 16;
  // cached per host thread, device and shared-memory size (which depends on the x3 pitch only).  The function's limit
  // is raised to the device's opt-in maximum, never to this grid's size: another thread's grid may need more.
  thread_local size_t cached_smem = 0;
  thread_local int per_sm = 1, sms = 148, cached_dev = -1;
  int dev = 0;
  cudaGetDevice(&dev);
  if (cached_smem != smem || cached_dev != dev) {
    int optin = 0;
    cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    cudaFuncSetAttribute(k_update_tile<SAME, NT, ROB>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    int v = 1;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&v, k_update_tile<SAME, NT, ROB>, NT, smem);
    per_sm = v < 1 ? 1 : v;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cached_smem = smem;
    cached_dev = dev;
  }
  const int np = L.n[0] + 1, ntile = (L.n[1] + 1 + TJ - 1) / TJ;
  const double slots = (double)sms * per_sm;
  double best = -1.0;
  int best_seg = np;
  for (int nseg = 1; nseg <= np && nseg <= 64; nseg++) {
    const int sg = (np + nseg - 1) / nseg;
    if (sg < 8 && nseg > 1) break;
    const int ns = (np + sg - 1) / sg;
    const double blocks = (double)ntile * ns, waves = ceil(blocks / slots);
    // wave fill x (planes / (planes + one exposed load latency per segment, about half a plane of work))
    const double eff = blocks / (waves * slots) * ((double)np / ((double)ns * (sg + 0.5)));
    if (eff > best) { best = eff; best_seg = sg; }
  }
  dim3 grid(ntile, (np + best_seg - 1) / best_seg);
  k_update_tile<SAME, NT, ROB><<<grid, NT, smem, g->stream>>>(Dv, r, dtfac, best_seg);
}

// the tiled kernel serves monolithic grids without derefinement whose staged planes fit shared memory
static int tile_threads(const Dev& Dv) {
  using namespace tile;
  if (Dv.B.nblk > 0 || Dv.mrow) return 0;
  const int nt = 32 * ((Dv.L.n[2] + 31) / 32) * TJ;
  const size_t smem = (size_t)(2 * NA + NB) * (TJ + 1) * Dv.L.p3 * sizeof(double) + 16;
  if (nt > 512 || smem > 227 * 1024) return 0;
  return nt <= 64 ? 64 : (nt <= 128 ? 128 : (nt <= 256 ? 256 : 512));
}

// ra / rb: the stage's roles in the buffer sets of blocks with cur == 0 / 2 (monolithic: rb unused)
void launch_update_on(hamr_grid* g, const Dev& Dv, const Roles& ra, const Roles& rb, double dtfac, bool same) {
  const Lay& L = Dv.L;
  const bool blk = Dv.B.nblk > 0;
  if (blk && Dv.B.nact == 0) return;
  const long long tot = (long long)(L.n[0] + 1) * (L.n[1] + 1) * L.n[2] * (blk ? Dv.B.nact : 1);
  const unsigned nb = (unsigned)((tot + 127) / 128);
  Launch l_(g, same ? K_UPDATE_P : K_UPDATE_C);
  const bool rob = Dv.entropy || Dv.drift;   // NEXT-2
  if (rob) {
    switch (tile_threads(Dv)) {
      case 64: return same ? launch_tile_t<true, 64, true>(g, Dv, ra, dtfac) : launch_tile_t<false, 64, true>(g, Dv, ra, dtfac);
      case 128: return same ? launch_tile_t<true, 128, true>(g, Dv, ra, dtfac) : launch_tile_t<false, 128, true>(g, Dv, ra, dtfac);
      case 256: return same ? launch_tile_t<true, 256, true>(g, Dv, ra, dtfac) : launch_tile_t<false, 256, true>(g, Dv, ra, dtfac);
      case 512: return same ? launch_tile_t<true, 512, true>(g, Dv, ra, dtfac) : launch_tile_t<false, 512, true>(g, Dv, ra, dtfac);
      default: break;
    }
    if (same && !blk) k_update<true, false, true><<<nb, 128, 0, g->stream>>>(Dv, ra, rb, dtfac);
    else if (same) k_update<true, true, true><<<nb, 128, 0, g->stream>>>(Dv, ra, rb, dtfac);
    else if (!blk) k_update<false, false, true><<<nb, 128, 0, g->stream>>>(Dv, ra, rb, dtfac);
    else k_update<false, true, true><<<nb, 128, 0, g->stream>>>(Dv, ra, rb, dtfac);
    return;
  }
  switch (tile_threads(Dv)) {
    case 64: return same ? launch_tile_t<true, 64>(g, Dv, ra, dtfac) : launch_tile_t<false, 64>(g, Dv, ra, dtfac);
    case 128: return same ? launch_tile_t<true, 128>(g, Dv, ra, dtfac) : launch_tile_t<false, 128>(g, Dv, ra, dtfac);
    case 256: return same ? launch_tile_t<true, 256>(g, Dv, ra, dtfac) : launch_tile_t<false, 256>(g, Dv, ra, dtfac);
    case 512: return same ? launch_tile_t<true, 512>(g, Dv, ra, dtfac) : launch_tile_t<false, 512>(g, Dv, ra, dtfac);
    default: break;
  }
  if (same && !blk) k_update<true, false><<<nb, 128, 0, g->stream>>>(Dv, ra, rb, dtfac);
  else if (same) k_update<true, true><<<nb, 128, 0, g->stream>>>(Dv, ra, rb, dtfac);
  else if (!blk) k_update<false, false><<<nb, 128, 0, g->stream>>>(Dv, ra, rb, dtfac);
  else k_update<false, true><<<nb, 128, 0, g->stream>>>(Dv, ra, rb, dtfac);
}

void launch_update(hamr_grid* g, const Fields& src, const Fields& base, const Fields& out, double dtfac,
                   bool src_is_base) {
  const Roles r = {src, base, out};
  launch_update_on(g, g->D, r, r, dtfac, src_is_base);
}

}  // namespace hamr
