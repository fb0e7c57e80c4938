// blocks.cu — block-structured grid on one GPU.
// the grid is a set of blocks that "directly transfer boundary cells" to one another;
// local adaptive time-stepping — every block steps with its own dt, a power of two
// times the smallest; at the interface between time levels the fluxes and EMFs of the
// finer block are accumulated and the coarse block's boundary zones are corrected with the
// difference, "an additional conserved to primitive variable inversion needs to be performed for
// these boundary cells".  Readings C-16 (same-level ghost copy, physical boundaries on the blocks
// that touch the domain edge) and C-17 (schedule, time-interpolated ghosts, registers, correction).
//
// B200 design: blocks are far too small to fill the GPU one at a time (16^3 zones; PAPER.md:185
// wants >~50^3 per launch), so every kernel of a stage is launched ONCE for all blocks of a time
// level: arrays hold the padded blocks back to back, a launch carries the list of its blocks, and
// a thread finds its block from its flat index.  No stream-per-block, no host loop over blocks.
#include <algorithm>
#include <cmath>
#include <cstring>
#include "hamr_host.h"

namespace hamr {

// the three buffer sets of the state arrays; a block's time-n state is s[cur], its predictor state
// s[1], the state being written by its corrector s[2 - cur]
struct Bufs { Fields s[3]; };

// LAT clock of every time level (C-17), in units of (finest dt)/2: time of the level's time-n state,
// its step, and whether its corrector has completed (so that s[2 - cur] holds the state at tb + dt)
struct LevT { long long tb[4]; int dtu[4]; int hasnew[4]; };

__device__ __forceinline__ const double* buf_arr(const Bufs& B, int buf, int kind) {
  // kind 0..4: hydro primitive; 5..7: face field along kind - 5
  const Fields& f0 = B.s[0];
  const Fields& f1 = B.s[1];
  const Fields& f2 = B.s[2];
  const double* a0 = kind < 5 ? f0.P[kind] : f0.Bf[kind - 5];
  const double* a1 = kind < 5 ? f1.P[kind] : f1.Bf[kind - 5];
  const double* a2 = kind < 5 ? f2.P[kind] : f2.Bf[kind - 5];
  return buf == 0 ? a0 : (buf == 1 ? a1 : a2);
}

// k_blk_ghosts calls blk_fetch_ref from eleven places.  Out of line the kernel is slower (measured on cfg 4: 0.260 ->
// 0.286 ms): the calls spill their arguments.  A single looped call site was no faster either: each iteration consumes
// its load at once, which serialises the DRAM round trips the unrolled form overlaps.
template <typename T>
__device__ __forceinline__ T pick4(const T v[4], int i) {
  return i == 0 ? v[0] : (i == 1 ? v[1] : (i == 2 ? v[2] : v[3]));
}

// Where the ghost fill of C-16 / C-12 takes the value at padded index id[] of an array of block b from:
// the per-dimension physical-boundary maps (outflow copy, polar mirror; fill order x1, x2, x3) are
// composed with the neighbour lookup, so that every ghost value is ONE signed sample of an active value.
struct GSrc {
  int q;        // block holding the value
  int zl;       // offset of the value inside that block
  int negmask;  // bit d: a mirror along d was applied (the component along d changes sign)
  bool ghost;   // sampled from a neighbour (else read from b's own active storage)
  bool zero;    // a reflecting wall face: the value is 0
  bool mod;     // differs from what b's own storage holds at id[]
  bool moved;   // a physical-boundary map changed the index (outflow copy, mirror, half turn)
  // C-16: the neighbour is on the other x1 refinement level: the value is a restriction / prolongation
  bool ref;
  int rq;       // the block on b's own side of the interface in the same transverse position
  int side;     // the neighbour lies on the high (1) or low (0) x1 side
  int mi, lj, lk;  // b's padded x1 index of the value; the neighbour's transverse indices
};

// sd: the array is staggered along sd (-1: zone-centred)
// norule: every neighbour is on b's own time level, so no face is owned by a finer block
__device__ __forceinline__ GSrc blk_src(const Dev& Dv, int b, int phys, int sd, const int id[3], bool norule) {
  const Lay& L = Dv.L;
  int m[3], o[3];
  GSrc s;
  s.negmask = 0;
  s.zero = false;
#pragma unroll
  for (int d = 0; d < 3; d++) {
    const int n = L.n[d], hi = (sd == d) ? n : n - 1, g = id[d];
    m[d] = g; o[d] = 0;
    if (g < 0) {
      if (phys & (1 << d)) {
        if (Dv.bc_lo[d] == HAMR_BC_OUTFLOW) m[d] = 0;
        else { m[d] = (sd == d) ? -g : -g - 1; s.negmask |= 1 << d; }
      } else o[d] = -1;
    } else if (g > hi) {
      if (phys & (8 << d)) {
        if (Dv.bc_hi[d] == HAMR_BC_OUTFLOW) m[d] = hi;
        else { m[d] = n - (g - hi); s.negmask |= 1 << d; }
      } else o[d] = 1;
    }
    // a reflecting wall carries no normal flux: the wall face itself is 0
    if (sd == d && ((m[d] == 0 && (phys & (1 << d)) && Dv.bc_lo[d] >= HAMR_BC_POLAR_REFLECT) ||
                    (m[d] == n && (phys & (8 << d)) && Dv.bc_hi[d] >= HAMR_BC_POLAR_REFLECT)))
      s.zero = true;
  }
  // C-15: the phi-ghost slots of a derefined row hold whole groups; an x2-face array follows its face's grouping
  int kz = m[2] - o[2] * L.n[2];            // x3 index inside the block that holds the value
  if (Dv.mrow && o[2] != 0) {
    const int J = Dv.B.info[b].w + id[1];
    const int mj = __ldg(Dv.mrow + J + NG);
    const int mg = sd == 1 ? max(mj, __ldg(Dv.mrow + max(J - 1, -NG) + NG)) : mj;
    if (mg > 1) kz = deref_ghost_k(id[2], L.n[2], mg);
  }
  const int* nb = Dv.B.nbr + b * NNBR;
  // NEXT-1 transmissive pole: the mirror row's zone half a turn away in x3: inside the block if
  // it spans x3, else at the same local index of the block half the x3 block count further (xp: the nine
  // such blocks replace the neighbour table)
  bool xp = false;
  if (((s.negmask >> 1) & 1) && Dv.bc_lo[1] == HAMR_BC_POLAR_TRANSMIT) {
    xp = __ldg(nb + 27 + 4) >= 0;
    if (xp) {
      if (Dv.mrow && o[2] != 0) {   // C-15 group units follow the SOURCE row (face) m[1]
        const int J = Dv.B.info[b].w + m[1];
        const int mj = __ldg(Dv.mrow + J + NG);
        const int mg = sd == 1 ? max(mj, __ldg(Dv.mrow + J - 1 + NG)) : mj;
        kz = mg > 1 ? deref_ghost_k(id[2], L.n[2], mg) : m[2] - o[2] * L.n[2];
      }
    } else {
      const int n3 = L.n[2];
      kz = (kz % n3 + n3 / 2) % n3;
      o[2] = 0;
    }
  }
  // neighbour by offset; across the pole the x2 offset is spent on the mirror
  auto nbq = [&](int a0, int a1, int a2) {
    return __ldg(xp ? nb + 27 + (a0 + 1) * 3 + (a2 + 1) : nb + (a0 + 1) * 9 + (a1 + 1) * 3 + (a2 + 1));
  };
  s.ghost = xp || (o[0] | o[1] | o[2]) != 0;
  s.q = s.ghost ? nbq(o[0], o[1], o[2]) : b;
  int lq[3] = {m[0] - o[0] * L.n[0], m[1] - o[1] * L.n[1], kz};
  // C-17: a face on the plane between two blocks on different time levels has ONE value in every stage
  // source, that of the finer block
  if (!norule && sd >= 0 && (m[sd] == 0 || m[sd] == L.n[sd])) {
    int o2[3] = {o[0], o[1], o[2]};
    o2[sd] = m[sd] == 0 ? -1 : 1;
    const int q2 = (xp && sd == 1) ? -1 : nbq(o2[0], o2[1], o2[2]);
    if (q2 >= 0 && s.q >= 0 && Dv.B.tau[q2] < Dv.B.tau[s.q] && Dv.B.info[q2].y == Dv.B.info[s.q].y) {
      s.q = q2;
      lq[sd] = m[sd] == 0 ? L.n[sd] : 0;
      s.ghost = true;
    }
  }
  s.moved = m[0] != id[0] || m[1] != id[1] || m[2] != id[2] || s.negmask != 0;
  s.mod = s.ghost || s.zero || (sd >= 0 && ((s.negmask >> sd) & 1)) || m[0] != id[0] || m[1] != id[1] || kz != id[2];
  s.zl = (int)L.idx(lq[0], lq[1], lq[2]);
  s.ref = false;
  if (!norule && o[0] != 0 && s.q >= 0 && Dv.B.info[s.q].y != Dv.B.info[b].y) {
    s.ref = true;
    s.rq = nbq(0, o[1], o[2]);
    s.side = o[0] > 0 ? 1 : 0;
    s.mi = m[0]; s.lj = lq[1]; s.lk = lq[2];
  }
  return s;
}

// ---- the ghost-source table -------------------------------------------------------------------------------------------
// blk_src is a pure function of (block, array kind, padded location) once the time levels are fixed, and it is most of
// the ghost kernel's instructions (neighbour look-ups, boundary maps, the finer-face rule).  k_blk_src_table evaluates
// it once per level assignment for every location; the ghost kernel then reads 8 bytes instead.  Packed: bits 0..31 the
// offset zl, 32..53 q + 1, 54..56 negmask, 57 ghost, 58 zero, 59 mod, 60 moved, 63 "not in the table" (the value is a
// restriction / prolongation across the x1 refinement interface, whose five extra fields are computed on the fly).
__device__ __forceinline__ unsigned long long gsrc_pack(const GSrc& s) {
  if (s.ref) return 1ull << 63;
  return (unsigned long long)(unsigned)s.zl | ((unsigned long long)(unsigned)(s.q + 1) << 32) |
         ((unsigned long long)(s.negmask & 7) << 54) | ((unsigned long long)s.ghost << 57) |
         ((unsigned long long)s.zero << 58) | ((unsigned long long)s.mod << 59) | ((unsigned long long)s.moved << 60);
}

__device__ __noinline__ void blk_src_slow(const Dev* Dv, int b, int phys, int sd, int i0, int i1, int i2, int norule, GSrc* out) {
  const int id[3] = {i0, i1, i2};
  *out = blk_src(*Dv, b, phys, sd, id, norule != 0);
}

// tb: the block's part of the table (NULL: no table); loc: the padded location of id[] (every caller's id[] lies inside
// the padded block: the thread's own location, its + 1 neighbour along a dimension that is not the extra slot, or a
// derefinement group slot of the same row)
__device__ __forceinline__ GSrc blk_src_tab(const Dev& Dv, const unsigned long long* __restrict__ tb, int loc, int b,
                                            int phys, int sd, const int id[3], bool norule) {
  if (tb) {
    const unsigned long long w = __ldg(tb + (size_t)(sd + 1) * Dv.B.gloc + loc);
    if (!(w >> 63)) {
      GSrc s;
      s.zl = (int)(unsigned)(w & 0xffffffffull);
      s.q = (int)((w >> 32) & 0x3fffffull) - 1;
      s.negmask = (int)((w >> 54) & 7);
      s.ghost = (w >> 57) & 1;
      s.zero = (w >> 58) & 1;
      s.mod = (w >> 59) & 1;
      s.moved = (w >> 60) & 1;
      s.ref = false;
      s.rq = -1; s.side = 0; s.mi = 0; s.lj = 0; s.lk = 0;
      return s;
    }
  }
  GSrc s;
  blk_src_slow(&Dv, b, phys, sd, id[0], id[1], id[2], norule ? 1 : 0, &s);
  return s;
}

// one thread per padded location of every block: the four sources of the location
__global__ void __launch_bounds__(256) k_blk_src_table(const __grid_constant__ Dev Dv, unsigned long long* __restrict__ tab) {
  const Lay& L = Dv.L;
  const int e3 = L.n[2] + 2 * NG + 1;
  const unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (unsigned)Dv.B.gloc) return;
  const int b = blockIdx.y;
  const unsigned tj = t / (unsigned)e3, ti = tj / (unsigned)L.e2;
  const int id[3] = {(int)ti - NG, (int)(tj - ti * L.e2) - NG, (int)(t - tj * e3) - NG};
  const int phys = __ldg(Dv.B.phys + b);
  const bool same = (Dv.B.flags[b] & 4) != 0;
#pragma unroll 1
  for (int sd = -1; sd < 3; sd++)
    tab[((size_t)b * 4 + (sd + 1)) * Dv.B.gloc + t] = gsrc_pack(blk_src(Dv, b, phys, sd, id, same));
}

// C-17 time sampling of block q at time s_u: which buffers and with what weight
struct QTime { int b0, b1; double w; };  // value = (1 - w) a[b0] + w a[b1]; b1 < 0: a plain copy of a[b0]
__device__ __forceinline__ QTime blk_qtime(const Dev& Dv, const LevT& lt, int q, long long s_u) {
  const int tq = Dv.B.tau[q], cq = Dv.B.cur[q];
  const long long tb = pick4(lt.tb, tq);
  const int dtu = pick4(lt.dtu, tq);
  QTime t;
  t.b0 = cq; t.b1 = -1; t.w = 0.0;
  if (s_u == tb) return t;                                  // a completed state: copy
  if (pick4(lt.hasnew, tq)) {                               // completed states bracket s_u
    t.b1 = 2 - cq;
    t.w = (double)(s_u - tb) / (double)dtu;
  } else {                                                  // the time-n state and the predictor state
    t.b1 = 1;
    t.w = (double)(s_u - tb) / (double)(dtu / 2);
  }
  return t;
}

__device__ __forceinline__ double blk_at(const Dev& Dv, const Bufs& B, int kind, int q, const QTime& t, int i, int j,
                                        int k) {
  const long long z = (long long)q * Dv.B.blen + Dv.L.idx(i, j, k);
  double v = buf_arr(B, t.b0, kind)[z];
  if (t.b1 >= 0) v = (1.0 - t.w) * v + t.w * buf_arr(B, t.b1, kind)[z];
  return v;
}

// C-16 ghost value across the x1 refinement interface.  levb: b's level.  Coarse ghosts: zones and
// transverse faces are the mean of the two fine values they cover, normal faces the coincident fine face.
// Fine ghosts: zones and transverse faces are piecewise linear in x1 with the MC-limited slope of the
// coarse values (the coarse value beyond the interface is the restriction of the fine block rq), a quarter
// of a coarse zone off the coarse centre; normal faces copy coincident coarse faces, in-between ones are
// the mean of their two coarse neighbours.
__device__ __forceinline__ double blk_fetch_ref(const Dev& Dv, const Bufs& B, const LevT& lt, int levb, int kind,
                                                const GSrc& s, long long s_u) {
  if (s.zero) return 0.0;
  const int n0 = Dv.L.n[0];
  const bool hi = s.side != 0, normal = kind == 5;
  const int i = s.mi, j = s.lj, k = s.lk, q = s.q;
  const QTime tq = blk_qtime(Dv, lt, q, s_u);
  double v;
  if (levb == 0) {
    if (normal) {
      const int t = hi ? i - n0 : -i;                       // 1..3 coarse faces from the interface
      v = blk_at(Dv, B, kind, q, tq, hi ? 2 * t : n0 - 2 * t, j, k);
    } else {
      const int t = hi ? i - n0 : -1 - i;                   // 0..2 coarse zones from the interface
      const int i0 = hi ? 2 * t : n0 - 2 * t - 2;
      v = 0.5 * (blk_at(Dv, B, kind, q, tq, i0, j, k) + blk_at(Dv, B, kind, q, tq, i0 + 1, j, k));
    }
  } else {
    if (normal) {
      const int t = hi ? i - n0 : -i;                       // 1..3 fine faces from the interface
      const int c0 = hi ? t / 2 : n0 - t / 2;
      v = blk_at(Dv, B, kind, q, tq, c0, j, k);
      if (t & 1) v = 0.5 * (v + blk_at(Dv, B, kind, q, tq, hi ? c0 + 1 : c0 - 1, j, k));
    } else {
      const int t = hi ? i - n0 : -1 - i;                   // 0..2 fine zones from the interface
      const int ic = hi ? t / 2 : n0 - 1 - t / 2;
      const bool high_half = hi ? (t & 1) != 0 : (t & 1) == 0;
      double a3[3];
#pragma unroll
      for (int w = -1; w <= 1; w++) {
        const int iw = ic + w;
        if (iw >= 0 && iw < n0) {
          a3[w + 1] = blk_at(Dv, B, kind, q, tq, iw, j, k);
        } else {                                            // covered by two fine zones of rq
          const QTime tr = blk_qtime(Dv, lt, s.rq, s_u);
          const int i0 = hi ? n0 - 2 : 0;
          a3[w + 1] = 0.5 * (blk_at(Dv, B, kind, s.rq, tr, i0, j, k) + blk_at(Dv, B, kind, s.rq, tr, i0 + 1, j, k));
        }
      }
      // C-16: piecewise linear in x1 with the MC-limited slope of the three coarse values, a quarter of a coarse
      // zone off the coarse centre
      const double dl = a3[1] - a3[0], dr = a3[2] - a3[1];
      double sl = 0.0;
      if (dl * dr > 0.0) {
        sl = fmin(0.5 * fabs(a3[2] - a3[0]), 2.0 * fmin(fabs(dl), fabs(dr)));
        if (dl < 0.0) sl = -sl;
      }
      v = 0.5 * (a3[1] + (high_half ? a3[1] + 0.5 * sl : a3[1] - 0.5 * sl));
    }
  }
  const int vc = kind >= 5 ? kind - 5 : (kind >= 2 ? kind - 2 : -1);
  return (vc >= 0 && ((s.negmask >> vc) & 1)) ? -v : v;
}

__device__ __forceinline__ double blk_fetch(const Dev& Dv, const Bufs& B, int b, int own_buf, int kind,
                                            const GSrc& s, const QTime& qt) {
  if (s.zero) return 0.0;
  const int vc = kind >= 5 ? kind - 5 : (kind >= 2 ? kind - 2 : -1);
  double v;
  if (!s.ghost) {
    v = buf_arr(B, own_buf, kind)[(long long)b * Dv.B.blen + s.zl];
  } else {
    const long long z = (long long)s.q * Dv.B.blen + s.zl;
    v = buf_arr(B, qt.b0, kind)[z];
    if (qt.b1 >= 0) v = (1.0 - qt.w) * v + qt.w * buf_arr(B, qt.b1, kind)[z];
  }
  return (vc >= 0 && ((s.negmask >> vc) & 1)) ? -v : v;
}

// 4 CTAs of 256 threads per SM (64 registers): with the sources read from the table 3 / 4 / 5 / 6 / 8 CTAs measured
// 0.299 / 0.260 / 0.285 / 0.306 / 0.303 ms per launch on cfg 4 (0.317 before the table, at 5)
constexpr int GHOST_MINB = 4;
// Ghost fill of the stage source of every listed block: neighbour exchange with time interpolation
// (C-16, C-17), physical boundaries (C-12), cell-centred B wherever a face changed (C-10).
// role: 0 the source is the block's time-n state, 1 its predictor state.  all: also derive B_c on the
// active zones (initial state).  zero_ctop: reset the block's Courant maxima (before a corrector pass).
// Block flags (host, per level assignment): bit 0 "simple": no physical side and all 26 neighbours on
// the block's own time level -> every ghost value (B_c included) is a plain copy of the neighbour's
// stage source; bit 1: some neighbour is on a finer time level (only then can an ACTIVE face change).
__global__ void __launch_bounds__(256, GHOST_MINB) k_blk_ghosts(const __grid_constant__ Dev Dv, const __grid_constant__ Bufs B,
                                                    const __grid_constant__ LevT lt, int role, long long s_u, int all,
                                                    int zero_ctop) {
  // grid: x covers the padded locations of one block, y the blocks of the launch; 32-bit index arithmetic
  const Lay& L = Dv.L;
  const int e3 = L.n[2] + 2 * NG + 1;
  const unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (unsigned)(L.e1 * L.e2 * e3)) return;
  const int b = __ldg(Dv.B.list + blockIdx.y);
  if (zero_ctop && t == 0) Dv.B.ctopb[b * 3] = Dv.B.ctopb[b * 3 + 1] = Dv.B.ctopb[b * 3 + 2] = 0.0;
  int i0, i1, i2;
  if (!all && !(Dv.B.flags[b] & 2)) {
    // no finer neighbour: active storage is final, so only the ghost shell is enumerated (whole warps of ghost
    // slots instead of warps that are two thirds active zones).  Part A: the (i, j) columns outside the active
    // range, every k; part B: the active columns' 2 NG + 1 ghost slots in k.
    const int n0 = L.n[0], n1 = L.n[1], gj = 2 * NG + 1;
    const unsigned lo_rows = (unsigned)(NG * L.e2), mid_rows = (unsigned)(n0 * gj);
    const unsigned nA = (lo_rows + mid_rows + (unsigned)((NG + 1) * L.e2)) * (unsigned)e3;
    if (t < nA) {
      unsigned row = t / (unsigned)e3;
      i2 = (int)(t - row * e3) - NG;
      if (row < lo_rows) {
        i0 = (int)(row / (unsigned)L.e2) - NG; i1 = (int)(row % (unsigned)L.e2) - NG;
      } else if (row < lo_rows + mid_rows) {
        row -= lo_rows;
        i0 = (int)(row / (unsigned)gj);
        const int q = (int)(row - i0 * gj);
        i1 = q < NG ? q - NG : n1 + q - NG;
      } else {
        row -= lo_rows + mid_rows;
        i0 = n0 + (int)(row / (unsigned)L.e2); i1 = (int)(row % (unsigned)L.e2) - NG;
      }
    } else {
      const unsigned u = t - nA;
      const int q = (int)(u & 7);
      if (q == 7 || u >= (unsigned)(n0 * n1 * 8)) return;
      const unsigned col = u >> 3;
      i0 = (int)(col / (unsigned)n1); i1 = (int)(col - i0 * n1);
      i2 = q < NG ? q - NG : L.n[2] + q - NG;
    }
  } else {
    const unsigned tj = t / (unsigned)e3, ti = tj / (unsigned)L.e2;
    i0 = (int)ti - NG; i1 = (int)(tj - ti * L.e2) - NG; i2 = (int)(t - tj * e3) - NG;
  }
  const int id[3] = {i0, i1, i2};
  bool in_c[3], extra[3];
#pragma unroll
  for (int d = 0; d < 3; d++) { in_c[d] = id[d] >= 0 && id[d] < L.n[d]; extra[d] = id[d] == L.n[d] + NG; }
  const bool zone_active = in_c[0] && in_c[1] && in_c[2];
  const bool zone_slot = !(extra[0] || extra[1] || extra[2]);
  // Which ghosts anything reads: a sweep along d reads zones up to NG deep along d but only one layer out
  // in the other two dimensions (the transverse ghost layer whose face EMFs feed C-9), and the centre EMFs
  // are needed one layer out.  Ghost zones more than one layer out in two or more dimensions are never
  // read and are left alone; ghost FACE storage is only read as the normal field of faces 0..n along d
  // in that one transverse layer (a ghost zone's B_c is built here from the fetched face values).
  int ndeep = 0;
  bool shell1[3];
#pragma unroll
  for (int d = 0; d < 3; d++) {
    ndeep += (id[d] < -1 || id[d] > L.n[d]) ? 1 : 0;
    shell1[d] = id[d] >= -1 && id[d] <= L.n[d];
  }
  if (ndeep >= 2) return;
  const int flags = Dv.B.flags[b];
  if (zone_active && !all && !(flags & 2)) return;   // no finer neighbour: active storage is final
  const int cur = Dv.B.cur[b];
  const int own = role == 0 ? cur : 1;
  const long long z = (long long)b * Dv.B.blen + L.idx(id[0], id[1], id[2]);
  const int* nb = Dv.B.nbr + b * NNBR;

  if ((flags & 1) && !all) {
    // ---- fast path: plain copies from same-level neighbours ------------------------------------------
    int oc[3], lc[3];
#pragma unroll
    for (int d = 0; d < 3; d++) {
      oc[d] = id[d] < 0 ? -1 : (id[d] >= L.n[d] ? 1 : 0);
      lc[d] = id[d] - oc[d] * L.n[d];
    }
    // all loads are issued before the first store (the stores may alias the loads as far as the compiler
    // knows; interleaving them would serialise eleven DRAM round trips)
    const Fields& fo = own == 0 ? B.s[0] : (own == 1 ? B.s[1] : B.s[2]);
    double vP[5], vB[3], vF[3];
    bool wF[3];
    // C-15: phi-ghost slots of derefined rows are in group units (x2-face arrays: their face's grouping)
    int mj = 1, Mj = 1;
    if (Dv.mrow && oc[2] != 0) {
      const int J = Dv.B.info[b].w + id[1];
      mj = __ldg(Dv.mrow + J + NG);
      Mj = max(mj, __ldg(Dv.mrow + max(J - 1, -NG) + NG));
      if (mj > 1) lc[2] = deref_ghost_k(id[2], L.n[2], mj);
    }
    if (zone_slot) {
      const int q = __ldg(nb + (oc[0] + 1) * 9 + (oc[1] + 1) * 3 + (oc[2] + 1));
      const int bq = role == 0 ? Dv.B.cur[q] : 1;
      const long long zq = (long long)q * Dv.B.blen + L.idx(lc[0], lc[1], lc[2]);
      const Fields& fq = bq == 0 ? B.s[0] : (bq == 1 ? B.s[1] : B.s[2]);
#pragma unroll
      for (int c = 0; c < 5; c++) vP[c] = fq.P[c][zq];
#pragma unroll
      for (int c = 0; c < 3; c++) vB[c] = fq.Bc[c][zq];
    }
#pragma unroll
    for (int d = 0; d < 3; d++) {
      const int o1 = (d + 1) % 3, o2 = (d + 2) % 3;
      int of[3] = {oc[0], oc[1], oc[2]}, lf[3] = {lc[0], lc[1], lc[2]};
      if (d == 1 && oc[2] != 0 && Mj > 1) lf[2] = deref_ghost_k(id[2], L.n[2], Mj);
      if (id[d] == L.n[d]) { of[d] = 0; lf[d] = id[d]; }    // the block's own high face
      wF[d] = shell1[o1] && shell1[o2] && id[d] >= 0 && id[d] <= L.n[d] && (of[0] | of[1] | of[2]) != 0;
      vF[d] = 0.0;
      if (wF[d]) {
        const int q = __ldg(nb + (of[0] + 1) * 9 + (of[1] + 1) * 3 + (of[2] + 1));
        const int bq = role == 0 ? Dv.B.cur[q] : 1;
        vF[d] = buf_arr(B, bq, 5 + d)[(long long)q * Dv.B.blen + L.idx(lf[0], lf[1], lf[2])];
      }
    }
    if (zone_slot) {
#pragma unroll
      for (int c = 0; c < 5; c++) fo.P[c][z] = vP[c];
#pragma unroll
      for (int c = 0; c < 3; c++) fo.Bc[c][z] = vB[c];
    }
#pragma unroll
    for (int d = 0; d < 3; d++)
      if (wF[d]) fo.Bf[d][z] = vF[d];
    return;
  }

  // ---- general path --------------------------------------------------------------------------------
  // zones two or more layers inside the block have nothing to do
  bool deep = true;
#pragma unroll
  for (int d = 0; d < 3; d++) deep = deep && id[d] >= 1 && id[d] <= L.n[d] - 2;
  if (deep && !all) return;
  const int phys = __ldg(Dv.B.phys + b);
  // bit 2: all neighbours on the block's own level: no finer-block faces, and every sample is a plain copy
  // of the neighbour's stage source (its time-n state for a predictor, its predictor state for a corrector)
  const bool same = (flags & 4) != 0;
  // the block's part of the ghost-source table and this thread's location in it (its neighbours: fixed strides)
  const unsigned long long* tb = Dv.B.gsrc ? Dv.B.gsrc + (size_t)b * 4 * Dv.B.gloc : nullptr;
  const int lst[3] = {L.e2 * e3, e3, 1};
  const int loc0 = ((id[0] + NG) * L.e2 + id[1] + NG) * e3 + id[2] + NG;
  int lastq = -1;
  QTime qt;
  qt.b0 = 0; qt.b1 = -1; qt.w = 0.0;
  const int levb = Dv.B.info[b].y;
  auto fetch = [&](int kind, const GSrc& gs) {
    return gs.ref ? blk_fetch_ref(Dv, B, lt, levb, kind, gs, s_u) : blk_fetch(Dv, B, b, own, kind, gs, qt);
  };
  auto qtime = [&](int q) {
    QTime r;
    if (same) { r.b0 = role == 0 ? Dv.B.cur[q] : 1; r.b1 = -1; r.w = 0.0; return r; }
    return blk_qtime(Dv, lt, q, s_u);
  };
  // loads first, stores last (see the fast path)
  double vP[5], vB[3];
  const bool wP = zone_slot && !zone_active;
  // pure: a ghost zone that is simply a same-level neighbour's zone (no boundary map, no refinement, no time
  // interpolation): its B_c is the neighbour's own B_c (same faces, same geometry), which saves the six face
  // look-ups that would rebuild it.  Safe for the reason the fast path is: every block touching the zones read
  // here is a neighbour of b on b's own level, so none of them rewrites those zones in this launch.
  bool pure = false;
  if (wP) {
    const GSrc s = blk_src_tab(Dv, tb, loc0, b, phys, -1, id, same);
    if (s.ghost) { qt = qtime(s.q); lastq = s.q; }
#pragma unroll
    for (int c = 0; c < 5; c++) vP[c] = fetch(c, s);
    pure = same && !all && s.ghost && !s.ref && !s.moved && !s.zero;
    if (pure) {
      const Fields& fq = qt.b0 == 0 ? B.s[0] : (qt.b0 == 1 ? B.s[1] : B.s[2]);
      const long long zq = (long long)s.q * Dv.B.blen + s.zl;
#pragma unroll
      for (int d = 0; d < 3; d++) vB[d] = fq.Bc[d][zq];
    }
  }
  double lo[3], hi[3];
  bool wF[3] = {false, false, false};
  bool anymod = false;
#pragma unroll
  for (int d = 0; d < 3; d++) {
    const int o1 = (d + 1) % 3, o2 = (d + 2) % 3;
    if (extra[o1] || extra[o2]) { lo[d] = hi[d] = 0.0; continue; }
    const bool face_read = shell1[o1] && shell1[o2] && id[d] >= 0 && id[d] <= L.n[d];   // a flux kernel reads this face
    if (pure && !face_read) { lo[d] = hi[d] = 0.0; continue; }
    GSrc s = blk_src_tab(Dv, tb, loc0, b, phys, d, id, same);
    if (s.ghost && s.q != lastq) { qt = qtime(s.q); lastq = s.q; }
    lo[d] = fetch(5 + d, s);
    if (s.mod) { wF[d] = face_read; anymod = true; }
    hi[d] = 0.0;
    if (!extra[d] && !pure) {
      int idp[3] = {id[0], id[1], id[2]};
      idp[d] += 1;
      s = blk_src_tab(Dv, tb, loc0 + lst[d], b, phys, d, idp, same);
      if (s.ghost && s.q != lastq) { qt = qtime(s.q); lastq = s.q; }
      hi[d] = fetch(5 + d, s);
      anymod = anymod || s.mod;
    }
  }
  if (wP) {
#pragma unroll
    for (int c = 0; c < 5; c++) const_cast<double*>(buf_arr(B, own, c))[z] = vP[c];
  }
#pragma unroll
  for (int d = 0; d < 3; d++)
    if (wF[d]) const_cast<double*>(buf_arr(B, own, 5 + d))[z] = lo[d];
  if (pure) {
#pragma unroll
    for (int d = 0; d < 3; d++) {
      double* bc = own == 0 ? B.s[0].Bc[d] : (own == 1 ? B.s[1].Bc[d] : B.s[2].Bc[d]);
      bc[z] = vB[d];
    }
  } else if (zone_slot && (!zone_active || all || anymod)) {
    const int4 inf = __ldg(Dv.B.info + b);
    const double g = __ldg(Dv.gcA + inf.y * Dv.B.tlevA + (size_t)(inf.x + id[0] * Dv.B.ge2 + id[1]) * NREC_C + CREC_GDET);
    if (Dv.mrow) {
      const int J = inf.w + id[1], n3 = L.n[2];
      const int m = __ldg(Dv.mrow + J + NG);
      if (id[2] >= 0 && id[2] < n3) {
        if (m > 1) {   // C-15: B_c^3 of a phi-derefined row is the group's value, from the group's two outer x3-faces
          const int k0 = id[2] - id[2] % m;
          int ig[3] = {id[0], id[1], k0};
          GSrc s = blk_src_tab(Dv, tb, loc0 + (k0 - id[2]), b, phys, 2, ig, same);
          if (s.ghost && s.q != lastq) { qt = qtime(s.q); lastq = s.q; }
          lo[2] = fetch(7, s);
          ig[2] = k0 + m;
          s = blk_src_tab(Dv, tb, loc0 + (k0 + m - id[2]), b, phys, 2, ig, same);
          if (s.ghost && s.q != lastq) { qt = qtime(s.q); lastq = s.q; }
          hi[2] = fetch(7, s);
        }
      } else {
        // a phi-ghost slot holds a whole group of THIS row; its two x2-faces are stored in their faces' groupings
        const int Mlo = max(m, __ldg(Dv.mrow + max(J - 1, -NG) + NG));
        const int Mhi = max(m, __ldg(Dv.mrow + min(J + 1, Dv.B.n2g + NG) + NG));
        if (Mlo != m) {
          int ig[3] = {id[0], id[1], deref_face2_slot(id[2], n3, m, Mlo)};
          const GSrc s = blk_src_tab(Dv, tb, loc0 + (ig[2] - id[2]), b, phys, 1, ig, same);
          if (s.ghost && s.q != lastq) { qt = qtime(s.q); lastq = s.q; }
          lo[1] = fetch(6, s);
        }
        if (Mhi != m) {
          int ig[3] = {id[0], id[1] + 1, deref_face2_slot(id[2], n3, m, Mhi)};
          const GSrc s = blk_src_tab(Dv, tb, loc0 + lst[1] + (ig[2] - id[2]), b, phys, 1, ig, same);
          if (s.ghost && s.q != lastq) { qt = qtime(s.q); lastq = s.q; }
          hi[1] = fetch(6, s);
        }
      }
    }
#pragma unroll
    for (int d = 0; d < 3; d++) {
      double* bc = own == 0 ? B.s[0].Bc[d] : (own == 1 ? B.s[1].Bc[d] : B.s[2].Bc[d]);
      bc[z] = (lo[d] + hi[d]) / (2.0 * g);
    }
  }
}

// C-17 registers: R2 = sum over the steps inside one step of the next coarser level of dt_b F and
// dt_b E of the corrector pass, on the faces and edges of the block boundary only.
template <bool ENT>
__global__ void __launch_bounds__(128) k_blk_registers(Dev Dv, int first, double dtfac) {
  const Lay& L = Dv.L;
  const int c2 = L.n[2] + 1, c1 = L.n[1] + 1;
  const unsigned per = (unsigned)(L.n[0] + 1) * c1 * c2;
  unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= per * Dv.B.nact) return;
  const int bslot = (int)(t / per);
  t -= bslot * per;
  const int b = __ldg(Dv.B.list + bslot);
  const unsigned tj = t / (unsigned)c2, ti = tj / (unsigned)c1;
  const int id[3] = {(int)ti, (int)(tj - ti * c1), (int)(t - tj * c2)};
  bool onb[3];
  for (int d = 0; d < 3; d++) onb[d] = id[d] == 0 || id[d] == L.n[d];
  if (!(onb[0] || onb[1] || onb[2])) return;
  const long long z = (long long)b * Dv.B.blen + L.idx(id[0], id[1], id[2]);
  const double dtb = dtfac * Dv.scal[S_DT];
#pragma unroll
  for (int d = 0; d < 3; d++) {
    const int e = (d + 1) % 3, f = (d + 2) % 3;
    if (onb[d] && id[e] < L.n[e] && id[f] < L.n[f]) {  // a boundary face along d
#pragma unroll
      for (int c = 0; c < 5; c++) {
        const double v = dtb * Dv.F[d][c][z];
        Dv.B.FA2[d][c][z] = first ? v : Dv.B.FA2[d][c][z] + v;
      }
      if (ENT) {   // C-18: the entropy flux is one more flux of the face
        const double v = dtb * Dv.FK[d][z];
        Dv.B.FKA2[d][z] = first ? v : Dv.B.FKA2[d][z] + v;
      }
    }
    // edge along d lies on the boundary if either transverse index does
    if (id[d] < L.n[d] && (onb[e] || onb[f])) {
      const double v = dtb * Dv.Ee[d][z];
      Dv.B.EA2[d][z] = first ? v : Dv.B.EA2[d][z] + v;
    }
  }
}

// time-integrated EMF on edge f at index id[] of block c (time level tc, step dtc): the accumulated
// register of a block on level tc - 1 that shares the edge (across the face, the other face, or the
// diagonal, in that order), else the block's own dtc * E.  rep: the former.
__device__ __forceinline__ double blk_edge_ec(const Dev& Dv, int c, int tc, int f, const int id[3], double dtc,
                                              bool& rep) {
  const Lay& L = Dv.L;
  const int d = (f + 1) % 3, e = (f + 2) % 3;
  const int od = id[d] == 0 ? -1 : (id[d] == L.n[d] ? 1 : 0);
  const int oe = id[e] == 0 ? -1 : (id[e] == L.n[e] ? 1 : 0);
  rep = false;
  if (od != 0 || oe != 0) {
    const int cand[3][2] = {{od, 0}, {0, oe}, {od, oe}};
#pragma unroll
    for (int t = 0; t < 3; t++) {
      if (cand[t][0] == 0 && cand[t][1] == 0) continue;
      int o[3] = {0, 0, 0};
      o[d] = cand[t][0]; o[e] = cand[t][1];
      const int q = __ldg(Dv.B.nbr + c * NNBR + (o[0] + 1) * 9 + (o[1] + 1) * 3 + (o[2] + 1));
      if (q < 0 || Dv.B.tau[q] != tc - 1) continue;
      int lq[3] = {id[0], id[1], id[2]};
      lq[d] -= o[d] * L.n[d];
      lq[e] -= o[e] * L.n[e];
      rep = true;
      return Dv.B.EA2[f][(long long)q * Dv.B.blen + L.idx(lq[0], lq[1], lq[2])];
    }
  }
  return dtc * Dv.Ee[f][(long long)c * Dv.B.blen + L.idx(id[0], id[1], id[2])];
}

// is the d-face at id[] of block c rebuilt by the correction, and with what?  Returns true and the new
// value: base - curl(EC) if one of its four edges is shared with a finer block; the finer face
// neighbour's own normal field on a face shared with it (C-17 correct(), steps 1-3 for the field).
__device__ __forceinline__ bool blk_face_corr(const Dev& Dv, const Bufs& B, int c, int tc, int curc, int d,
                                              const int id[3], double dtc, bool want_value, double& val) {
  const Lay& L = Dv.L;
  const int e = (d + 1) % 3, f = (d + 2) % 3;
  // shared with a finer face neighbour: copy its field (it has completed both steps: its time-n state
  // is at the coarse block's new time)
  if (id[d] == 0 || id[d] == L.n[d]) {
    int o[3] = {0, 0, 0};
    o[d] = id[d] == 0 ? -1 : 1;
    const int q = __ldg(Dv.B.nbr + c * NNBR + (o[0] + 1) * 9 + (o[1] + 1) * 3 + (o[2] + 1));
    if (q >= 0 && Dv.B.tau[q] == tc - 1) {
      if (want_value) {
        int lq[3] = {id[0], id[1], id[2]};
        lq[d] = id[d] == 0 ? L.n[d] : 0;
        val = buf_arr(B, Dv.B.cur[q], 5 + d)[(long long)q * Dv.B.blen + L.idx(lq[0], lq[1], lq[2])];
      }
      return true;
    }
  }
  const int4 inf = __ldg(Dv.B.info + c);
  if (d == 1 && Dv.metric == HAMR_METRIC_KERR_SCHILD && (inf.w + id[1] == 0 || inf.w + id[1] == Dv.B.n2g))
    return false;  // pole faces stay 0
  int ie[3] = {id[0], id[1], id[2]}, jf[3] = {id[0], id[1], id[2]};
  ie[e] += 1;
  jf[f] += 1;
  bool r0, r1, r2, r3;
  const double Ef0 = blk_edge_ec(Dv, c, tc, f, id, dtc, r0), Ef1 = blk_edge_ec(Dv, c, tc, f, ie, dtc, r1);
  const double Ee0 = blk_edge_ec(Dv, c, tc, e, id, dtc, r2), Ee1 = blk_edge_ec(Dv, c, tc, e, jf, dtc, r3);
  if (!(r0 || r1 || r2 || r3)) return false;
  if (want_value) {
    const double dxd[3] = {inf.y ? 0.5 * Dv.dx[0] : Dv.dx[0], Dv.dx[1], Dv.dx[2]};
    const double curl = (Ef1 - Ef0) / dxd[e] - (Ee1 - Ee0) / dxd[f];
    val = buf_arr(B, curc, 5 + d)[(long long)c * Dv.B.blen + L.idx(id[0], id[1], id[2])] - curl;
  }
  return true;
}

// correct(tau-1 -> tau), field part: rewrites the faces of the listed (level tau) blocks' new state
__global__ void __launch_bounds__(128) k_blk_correct_faces(Dev Dv, Bufs B, int tc, double dtfac) {
  const Lay& L = Dv.L;
  const int c2 = L.n[2] + 1, c1 = L.n[1] + 1;
  const unsigned per = (unsigned)(L.n[0] + 1) * c1 * c2;
  unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= per * Dv.B.nact) return;
  const int bslot = (int)(t / per);
  t -= bslot * per;
  const int c = __ldg(Dv.B.list + bslot);
  const unsigned tj = t / (unsigned)c2, ti = tj / (unsigned)c1;
  const int id[3] = {(int)ti, (int)(tj - ti * c1), (int)(t - tj * c2)};
  // only faces within one zone of the block boundary can be touched
  bool near = false;
  for (int d = 0; d < 3; d++) near = near || id[d] <= 1 || id[d] >= L.n[d] - 1;
  if (!near) return;
  const int curc = Dv.B.cur[c];
  const double dtc = dtfac * Dv.scal[S_DT];
  const long long z = (long long)c * Dv.B.blen + L.idx(id[0], id[1], id[2]);
#pragma unroll
  for (int d = 0; d < 3; d++) {
    const int e = (d + 1) % 3, f = (d + 2) % 3;
    if (id[e] >= L.n[e] || id[f] >= L.n[f]) continue;
    double v;
    if (blk_face_corr(Dv, B, c, tc, curc, d, id, dtc, true, v))
      const_cast<double*>(buf_arr(B, 2 - curc, 5 + d))[z] = v;
  }
}

// correct(tau-1 -> tau), zone part: flux difference into the boundary zones, new cell-centred field,
// re-inversion of every touched zone
// ROB: the grid carries the entropy row and / or the drift-frame floors (C-18, C-19, C-21)
template <bool ROB>
__global__ void __launch_bounds__(128) k_blk_correct_zones(Dev Dv, Bufs B, int tc, double dtfac) {
  const Lay& L = Dv.L;
  const unsigned per = (unsigned)L.n[0] * L.n[1] * L.n[2];
  unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  int nfail = 0, nrf = 0, nuf = 0, ngc = 0, bad = 0, nent = 0, nait = 0;
  if (t < per * Dv.B.nact) {
    const int bslot = (int)(t / per);
    t -= bslot * per;
    const int c = __ldg(Dv.B.list + bslot);
    const unsigned tj = t / (unsigned)L.n[2], ti = tj / (unsigned)L.n[1];
    const int id[3] = {(int)ti, (int)(tj - ti * L.n[1]), (int)(t - tj * L.n[2])};
    bool near = false;
    for (int d = 0; d < 3; d++) near = near || id[d] == 0 || id[d] == L.n[d] - 1;
    if (near) {
      const int curc = Dv.B.cur[c];
      const double dtc = dtfac * Dv.scal[S_DT];
      const int4 inf = __ldg(Dv.B.info + c);
      const double dxd[3] = {inf.y ? 0.5 * Dv.dx[0] : Dv.dx[0], Dv.dx[1], Dv.dx[2]};
      const long long S[3] = {L.S1, L.S2, 1};
      const long long z = (long long)c * Dv.B.blen + L.idx(id[0], id[1], id[2]);
      bool touched = false;
      double dU[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, dUS = 0.0;
#pragma unroll
      for (int d = 0; d < 3; d++) {
#pragma unroll
        for (int side = 0; side < 2; side++) {
          int fi[3] = {id[0], id[1], id[2]};
          fi[d] += side;
          double dummy;
          if (blk_face_corr(Dv, B, c, tc, curc, d, fi, dtc, false, dummy)) touched = true;
          // flux difference on a face shared with a finer face neighbour
          if ((side == 0 && id[d] == 0) || (side == 1 && id[d] == L.n[d] - 1)) {
            int o[3] = {0, 0, 0};
            o[d] = side ? 1 : -1;
            const int q = __ldg(Dv.B.nbr + c * NNBR + (o[0] + 1) * 9 + (o[1] + 1) * 3 + (o[2] + 1));
            if (q >= 0 && Dv.B.tau[q] == tc - 1) {
              int lq[3] = {id[0], id[1], id[2]};
              lq[d] = side ? 0 : L.n[d];
              const long long zq = (long long)q * Dv.B.blen + L.idx(lq[0], lq[1], lq[2]);
              const long long zf = z + side * S[d];
#pragma unroll
              for (int cc = 0; cc < 5; cc++) {
                const double dF = Dv.B.FA2[d][cc][zq] - dtc * Dv.F[d][cc][zf];
                // U_new = U - (dt F_hi - dt F_lo)/dx: the high face enters with -, the low face with +
                dU[cc] += (side ? -dF : dF) / dxd[d];
              }
              if (ROB && Dv.entropy) {   // C-18: the entropy row is corrected like the others
                const double dF = Dv.B.FKA2[d][zq] - dtc * Dv.FK[d][zf];
                dUS += (side ? -dF : dF) / dxd[d];
              }
              touched = true;
            }
          }
        }
      }
      if (touched) {
        const int q2 = inf.x + id[0] * Dv.B.ge2 + id[1];
        const CGeo G = load_cgeo(Dv.gcA + inf.y * Dv.B.tlevA + (size_t)q2 * NREC_C);
        double P[8], U[5], Bn[3], Pn[5];
        const int nw = 2 - curc;
#pragma unroll
        for (int cc = 0; cc < 5; cc++) P[cc] = buf_arr(B, nw, cc)[z];
#pragma unroll
        for (int d = 0; d < 3; d++) {
          double* bc = nw == 0 ? B.s[0].Bc[d] : B.s[2].Bc[d];
          P[5 + d] = bc[z];
          const double* bf = buf_arr(B, nw, 5 + d);
          Bn[d] = (bf[z] + bf[z + S[d]]) / (2.0 * G.gdet);
          bc[z] = Bn[d];
        }
        St Sx;
        get_state(P, G, Sx);
        prim_to_U5(P, Sx, G.gdet, Dv.gam, U);
        // C-18 under LAT: kappa was reset from the zone's new primitives, so its entropy row before the correction is its
        // density row times kappa(P)
        const double US = (ROB && Dv.entropy) ? U[0] * kappa_of(P[0], P[1], Dv.gam) + dUS : 0.0;
#pragma unroll
        for (int cc = 0; cc < 5; cc++) U[cc] += dU[cc];
        int rc = con2prim(U, Bn, G, Dv.gam, P, Pn);
        if (ROB && Dv.entropy && (rc != 0 || !(Pn[0] > 0.0) || !(Pn[1] >= 0.0))) {   // the chain of the update (C-21, C-18)
          double Pe[5], Uc[5], Bc[3], Pc[5];
          CGeo Gc = G;
#pragma unroll
          for (int cc = 0; cc < 5; cc++) { Uc[cc] = U[cc]; Pc[cc] = P[cc]; }
#pragma unroll
          for (int cc = 0; cc < 3; cc++) Bc[cc] = Bn[cc];
          if (rc != 0 && con2prim_aitken(Uc, Bc, &Gc, Dv.gam, Pc, Pe) == 0) {
#pragma unroll
            for (int cc = 0; cc < 5; cc++) Pn[cc] = Pe[cc];
            rc = 0;
            nait = 1;
          }
          if ((rc != 0 || !(Pn[0] > 0.0) || !(Pn[1] >= 0.0)) && con2prim_entropy(Uc, US, Bc, &Gc, Dv.gam, Pc, Pe) == 0) {
#pragma unroll
            for (int cc = 0; cc < 5; cc++) Pn[cc] = Pe[cc];
            rc = 0;
            nent = 1;
          }
        }
        if (rc != 0) {
          nfail = 1;
#pragma unroll
          for (int cc = 0; cc < 5; cc++) Pn[cc] = P[cc];
        }
        const int fi = inf.z + id[0] + NG + inf.y * Dv.B.flev;
        const double rfl = __ldg(Dv.rho_fl + fi), ufl = __ldg(Dv.u_fl + fi);
        if (ROB && Dv.drift) {   // C-19
          nrf = Pn[0] < rfl;
          nuf = Pn[1] < ufl;
          if (nrf | nuf) floors_drift(G, Bn, Dv.gam, nrf ? rfl : Pn[0], nuf ? ufl : Pn[1], Pn);
          ceiling_only(G, Dv.gamma_max, Pn, ngc);
        } else {
          floors_ceiling(G, rfl, ufl, Dv.gamma_max, Pn, nrf, nuf, ngc);
        }
#pragma unroll
        for (int cc = 0; cc < 5; cc++) {
          const_cast<double*>(buf_arr(B, nw, cc))[z] = Pn[cc];
          if (!isfinite(Pn[cc])) bad = 1;
        }
      }
    }
  }
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

// the listed blocks finished a step: their new state becomes their time-n state
__global__ void k_blk_rotate(Dev Dv) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= Dv.B.nact) return;
  const int b = Dv.B.list[t];
  Dv.B.cur[b] = 2 - Dv.B.cur[b];
}

// C-14 on a block grid with one global dt: per-direction maximum of ctop / dx over the blocks, then
// the harmonic sum (PAPER.md:93 fn. 2).  One CTA.  mode 0: set dt; 1: advance t by the dt just used first.
__global__ void __launch_bounds__(256) k_blk_dt(Dev Dv, int mode) {
  __shared__ double sm[3][8];
  double m[3] = {0.0, 0.0, 0.0};
  for (int b = threadIdx.x; b < Dv.B.nblk; b += blockDim.x) {
    const int lev = Dv.B.info[b].y;
    m[0] = fmax(m[0], Dv.B.ctopb[b * 3] / (lev ? 0.5 * Dv.dx[0] : Dv.dx[0]));
    m[1] = fmax(m[1], Dv.B.ctopb[b * 3 + 1] / Dv.dx[1]);
    m[2] = fmax(m[2], Dv.B.ctopb[b * 3 + 2] / Dv.dx[2]);
  }
  for (int d = 0; d < 3; d++) {
    m[d] = warp_max(m[d]);
    if ((threadIdx.x & 31) == 0) sm[d][threadIdx.x >> 5] = m[d];
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double* s = Dv.scal;
    if (mode == 1) { s[S_T] += s[S_DT]; s[S_DTLAST] = s[S_DT]; }
    double sum = 0.0;
    for (int d = 0; d < 3; d++) {
      double v = 0.0;
      for (int w = 0; w < (int)(blockDim.x >> 5); w++) v = fmax(v, sm[d][w]);
      sum += v;
    }
    s[S_DT] = Dv.cour / sum;
  }
}

// LAT: one coarse step of 2^tmax finest steps has been taken; the host sets the next dt_0
__global__ void k_blk_time(Dev Dv, double fac) {
  Dv.scal[S_T] += fac * Dv.scal[S_DT];
  Dv.scal[S_DTLAST] = Dv.scal[S_DT];
}

// dense global arrays <-> blocks (grids without x1 refinement).  stag: -1 zone-centred, else the face dim;
// a face shared by two blocks is stored in both.
__global__ void __launch_bounds__(256) k_blk_pack(Dev Dv, const double* __restrict__ dense, double* __restrict__ s0,
                                                  double* __restrict__ s2, int stag, int zero_pole, int ng0, int ng1,
                                                  int ng2) {
  const Lay& L = Dv.L;
  int m[3] = {L.n[0], L.n[1], L.n[2]};
  int M[3] = {ng0, ng1, ng2};
  if (stag >= 0) { m[stag] += 1; M[stag] += 1; }
  const long long per = (long long)m[0] * m[1] * m[2];
  long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= per * Dv.B.nblk) return;
  const int b = (int)(t / per);
  t -= b * per;
  const int k = (int)(t % m[2]), j = (int)((t / m[2]) % m[1]), i = (int)(t / ((long long)m[2] * m[1]));
  const int4 inf = __ldg(Dv.B.info + b);
  const int K0 = __ldg(Dv.B.K0 + b);
  double v = dense ? dense[((long long)(inf.z + i) * M[1] + (inf.w + j)) * M[2] + (K0 + k)] : 0.0;
  if (zero_pole && Dv.metric == HAMR_METRIC_KERR_SCHILD && (inf.w + j == 0 || inf.w + j == Dv.B.n2g)) v = 0.0;
  (Dv.B.cur[b] ? s2 : s0)[(long long)b * Dv.B.blen + L.idx(i, j, k)] = v;
}

__global__ void __launch_bounds__(256) k_blk_unpack(Dev Dv, const double* __restrict__ s0, const double* __restrict__ s2,
                                                    double* __restrict__ dense, int stag, int ng0, int ng1, int ng2) {
  const Lay& L = Dv.L;
  int m[3] = {L.n[0], L.n[1], L.n[2]};
  int M[3] = {ng0, ng1, ng2};
  if (stag >= 0) { m[stag] += 1; M[stag] += 1; }
  const long long per = (long long)m[0] * m[1] * m[2];
  long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= per * Dv.B.nblk) return;
  const int b = (int)(t / per);
  t -= b * per;
  const int k = (int)(t % m[2]), j = (int)((t / m[2]) % m[1]), i = (int)(t / ((long long)m[2] * m[1]));
  const int4 inf = __ldg(Dv.B.info + b);
  const int K0 = __ldg(Dv.B.K0 + b);
  dense[((long long)(inf.z + i) * M[1] + (inf.w + j)) * M[2] + (K0 + k)] =
      (Dv.B.cur[b] ? s2 : s0)[(long long)b * Dv.B.blen + L.idx(i, j, k)];
}

// ---- diagnostics on a block grid (C-11 div B, conserved totals, finite check) ----------------------------
__global__ void __launch_bounds__(256) k_blk_diag(Dev Dv, Bufs B, int what) {
  // what 0: max denominator of C-11; 1: max |div| / den; 2: conserved totals; 3: finite check
  const Lay& L = Dv.L;
  const long long per = (long long)L.n[0] * L.n[1] * L.n[2];
  long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  double val = 0.0, U[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
  int bad = 0;
  if (t < per * Dv.B.nblk) {
    const int b = (int)(t / per);
    t -= b * per;
    const int k = (int)(t % L.n[2]), j = (int)((t / L.n[2]) % L.n[1]), i = (int)(t / ((long long)L.n[2] * L.n[1]));
    const long long z = (long long)b * Dv.B.blen + L.idx(i, j, k);
    const long long S[3] = {L.S1, L.S2, 1};
    const int cur = Dv.B.cur[b];
    const int4 inf = __ldg(Dv.B.info + b);
    const double dxd[3] = {inf.y ? 0.5 * Dv.dx[0] : Dv.dx[0], Dv.dx[1], Dv.dx[2]};
    const Fields& s = cur ? B.s[2] : B.s[0];
    if (what <= 1) {
      double div = 0.0, den = 0.0;
      for (int d = 0; d < 3; d++) {
        const double lo = s.Bf[d][z], hi = s.Bf[d][z + S[d]];
        div += (hi - lo) / dxd[d];
        den += (fabs(hi) + fabs(lo)) / (2.0 * dxd[d]);
      }
      if (what == 0) val = den;
      else if (den > 1e-12 * Dv.scal[S_DENMAX]) val = fabs(div) / den;
    } else if (what == 2) {
      const CGeo G = load_cgeo(Dv.gcA + inf.y * Dv.B.tlevA + (size_t)(inf.x + i * Dv.B.ge2 + j) * NREC_C);
      double P[8];
      for (int c = 0; c < 5; c++) P[c] = s.P[c][z];
      for (int c = 0; c < 3; c++) P[5 + c] = s.Bc[c][z];
      St Sx;
      get_state(P, G, Sx);
      prim_to_U5(P, Sx, G.gdet, Dv.gam, U);
      const double dV = dxd[0] * dxd[1] * dxd[2];
      for (int c = 0; c < 5; c++) U[c] *= dV;
    } else {
      for (int c = 0; c < 5; c++) bad |= !isfinite(s.P[c][z]);
      for (int c = 0; c < 3; c++) bad |= !isfinite(s.Bc[c][z]);
    }
  }
  if (what <= 1) {
    val = warp_max(val);
    if ((threadIdx.x & 31) == 0 && val > 0.0) atomic_max_pos(Dv.scal + (what == 0 ? S_DENMAX : S_DIVB), val);
  } else if (what == 2) {
    for (int c = 0; c < 5; c++) {
      double v = U[c];
      for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
      if ((threadIdx.x & 31) == 0) atomicAdd(Dv.scal + S_TOT0 + c, v);
    }
  } else {
    const unsigned m = __ballot_sync(0xffffffffu, bad);
    if ((threadIdx.x & 31) == 0 && m) atomicAdd(Dv.cnt + N_NONFINITE, (unsigned long long)__popc(m));
  }
}

__global__ void k_blk_zero_scal(Dev Dv, int first, int count) {
  for (int c = 0; c < count; c++) Dv.scal[first + c] = 0.0;
}

// C-16: where a coarse and a fine block on the same time level share the x1 interface, the fine block's F^1
// and the edge EMFs E_2, E_3 lying in the interface plane are authoritative: the coarse block overwrites its
// own with them before its update (equal face areas and edge lengths: plain copies).
__global__ void __launch_bounds__(128) k_blk_iface(Dev Dv) {
  const Lay& L = Dv.L;
  const int c2 = L.n[2] + 1, c1 = L.n[1] + 1;
  const unsigned per = 2u * c1 * c2;
  unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= per * Dv.B.nact) return;
  const int bslot = (int)(t / per);
  t -= bslot * per;
  const int c = __ldg(Dv.B.list + bslot);
  if (Dv.B.info[c].y != 0) return;
  const int side = (int)(t / (unsigned)(c1 * c2));
  t -= side * c1 * c2;
  const int j = (int)(t / (unsigned)c2), k = (int)(t - (t / (unsigned)c2) * c2);
  const int q = __ldg(Dv.B.nbr + c * NNBR + (side ? 2 : 0) * 9 + 4);
  if (q < 0 || Dv.B.info[q].y == 0 || Dv.B.tau[q] != Dv.B.tau[c]) return;
  const long long zc = (long long)c * Dv.B.blen + L.idx(side ? L.n[0] : 0, j, k);
  const long long zq = (long long)q * Dv.B.blen + L.idx(side ? 0 : L.n[0], j, k);
  if (j < L.n[1] && k < L.n[2]) {
#pragma unroll
    for (int cc = 0; cc < 5; cc++) Dv.F[0][cc][zc] = Dv.F[0][cc][zq];
    if (Dv.entropy) Dv.FK[0][zc] = Dv.FK[0][zq];   // C-18: the entropy flux is one more flux of the face
  }
  if (j < L.n[1]) Dv.Ee[1][zc] = Dv.Ee[1][zq];
  if (k < L.n[2]) Dv.Ee[2][zc] = Dv.Ee[2][zq];
}

// one block's dense arrays <-> its padded storage (grids with x1 refinement are set and read block by block)
__global__ void __launch_bounds__(256) k_blk_pack1(Dev Dv, int b, const double* __restrict__ dense, double* __restrict__ s0,
                                                   double* __restrict__ s2, int stag, int zero_pole, int unpack) {
  const Lay& L = Dv.L;
  int m[3] = {L.n[0], L.n[1], L.n[2]};
  if (stag >= 0) m[stag] += 1;
  // b < 0: every block, the dense arrays of the blocks back to back in block order
  const unsigned per = (unsigned)(m[0] * m[1] * m[2]);
  const unsigned tg = blockIdx.x * blockDim.x + threadIdx.x;
  if (tg >= (b < 0 ? per * (unsigned)Dv.B.nblk : per)) return;
  unsigned t = tg;
  if (b < 0) { b = (int)(tg / per); t = tg - (unsigned)b * per; }
  const unsigned tj = t / (unsigned)m[2], ti = tj / (unsigned)m[1];
  const int k = (int)(t - tj * m[2]), j = (int)(tj - ti * m[1]), i = (int)ti;
  double* a = Dv.B.cur[b] ? s2 : s0;
  const long long z = (long long)b * Dv.B.blen + L.idx(i, j, k);
  if (unpack) { const_cast<double*>(dense)[tg] = a[z]; return; }
  double v = dense ? dense[tg] : 0.0;
  const int J = Dv.B.info[b].w + j;
  if (zero_pole && Dv.metric == HAMR_METRIC_KERR_SCHILD && (J == 0 || J == Dv.B.n2g)) v = 0.0;
  a[z] = v;
}

// ==== host side ==============================================================================================

static Bufs bufs_of(const hamr_grid* g) {
  Bufs B;
  for (int i = 0; i < 3; i++) B.s[i] = g->s[i];
  return B;
}

static LevT clocks_of(const hamr_grid* g) {
  LevT lt;
  for (int i = 0; i < 4; i++) { lt.tb[i] = g->bh.tb_u[i]; lt.dtu[i] = g->bh.dt_u[i]; lt.hasnew[i] = g->bh.has_new[i]; }
  return lt;
}

// Dev of a launch over the blocks of list `which` (0..3: time level; 4: every block)
static Dev dev_list(const hamr_grid* g, int which) {
  Dev D = g->D;
  D.B.list = g->bh.d_lists + (size_t)which * g->bh.nblk;
  D.B.nact = which == 4 ? g->bh.nblk : g->bh.nlist[which];
  D.B.dlist = g->bh.d_dlists + (size_t)which * g->bh.nblk;
  D.B.ndact = g->bh.ndlist[which];
  return D;
}

// per-block ghost-fill flags from the current time levels (see k_blk_ghosts) into pinned memory, then upload
static cudaError_t blk_upload_flags(hamr_grid* g) {
  BlkHost& H = g->bh;
  int* hf = H.h_ints + (size_t)9 * H.nblk;
  for (int b = 0; b < H.nblk; b++) {
    bool same = true, finer = false;
    for (int a = 0; a < NNBR; a++) {
      const int q = H.nbr[(size_t)b * NNBR + a];
      if (q < 0) continue;
      if (H.tau[q] != H.tau[b] || H.lev1[q] != H.lev1[b]) same = false;
      if (H.tau[q] < H.tau[b]) finer = true;
    }
    hf[b] = ((same && H.phys[b] == 0) ? 1 : 0) | (finer ? 2 : 0) | (same ? 4 : 0);
  }
  return cudaMemcpyAsync(g->D.B.flags, hf, (size_t)H.nblk * 4, cudaMemcpyHostToDevice, g->stream);
}

// (re)builds the ghost-source table if the time levels differ from those it was built for; the flags and levels must
// have been uploaded on the stream before
static void blk_build_gsrc(hamr_grid* g) {
  BlkHost& H = g->bh;
  if (!H.d_gsrc || H.gsrc_tau == H.tau) return;
  const Dev D = dev_list(g, 4);
  Launch l_(g, K_OTHER);
  k_blk_src_table<<<dim3((D.B.gloc + 255) / 256, H.nblk), 256, 0, g->stream>>>(D, H.d_gsrc);
  H.gsrc_tau = H.tau;
}

// C-16 x1 slots: a base block column whose x1-centre has r < r_refine_max (x1 itself on the Cartesian map)
// is replaced by two children with dx1 / 2 (per-dimension splitting).  Returns the number of
// refined columns (they must be contiguous from the low x1 side), -1 if they are not.
static int blk_refined_columns(const hamr_params& p, int ncol, int bn0) {
  if (!(p.r_refine_max > 0.0)) return 0;
  const bool ks = p.metric == HAMR_METRIC_KERR_SCHILD;
  const double lo = ks ? std::log(p.xmin[0]) : p.xmin[0], hi = ks ? std::log(p.xmax[0]) : p.xmax[0];
  const double dx0 = (hi - lo) / p.n[0];
  int nref = 0;
  bool seen_coarse = false;
  for (int col = 0; col < ncol; col++) {
    const double xc = lo + ((double)col + 0.5) * bn0 * dx0;
    const bool refined = (ks ? std::exp(xc) : xc) < p.r_refine_max;
    if (refined && seen_coarse) return -1;
    if (refined) nref++;
    else seen_coarse = true;
  }
  return nref;
}

// per list (time levels 0..3, every block), the blocks that hold phi-derefined rows: the C-15 kernels run on
// these only.  Uses the pinned staging area (the stream must be idle with respect to it).
static cudaError_t blk_upload_dlists(hamr_grid* g) {
  BlkHost& H = g->bh;
  const int nblk = H.nblk;
  int* hd = H.h_ints + (size_t)10 * nblk;
  for (int i = 0; i < 5; i++) H.ndlist[i] = 0;
  for (int b = 0; b < nblk; b++) {
    if (!H.hasderef[b]) continue;
    const int t = H.tau[b];
    hd[(size_t)t * nblk + H.ndlist[t]++] = b;
    hd[(size_t)4 * nblk + H.ndlist[4]++] = b;
  }
  return cudaMemcpyAsync(H.d_dlists, hd, (size_t)5 * nblk * 4, cudaMemcpyHostToDevice, g->stream);
}

int blk_count(const hamr_params& p, int nslot[3], int bn[3]) {
  long long nb = 1;
  for (int d = 0; d < 3; d++) {
    bn[d] = p.nb[d] > 0 ? p.nb[d] : p.n[d];
    if (bn[d] < NG || p.n[d] % bn[d] != 0) return 0;
    nslot[d] = p.n[d] / bn[d];
  }
  const int nref = blk_refined_columns(p, nslot[0], bn[0]);
  if (nref < 0) return 0;
  if (nref > 0 && bn[0] < 2 * NG) return 0;   // a coarse ghost layer of 3 zones covers 6 fine zones
  nslot[0] += nref;
  for (int d = 0; d < 3; d++) nb *= nslot[d];
  return nb > (1 << 20) ? 0 : (int)nb;
}

int blk_has_refinement(const hamr_params& p) {
  int ns[3], bn[3];
  if (blk_count(p, ns, bn) <= 0) return 0;
  return blk_refined_columns(p, p.n[0] / bn[0], bn[0]) > 0 ? 1 : 0;
}

// the ghost-source table is kept when it stays below 4 GB (cfg 4: 1472 blocks x 12167 locations x 32 B = 0.57 GB; a grid
// of a few huge blocks has few ghost zones per zone and computes the sources on the fly)
static size_t blk_gsrc_bytes(int nblk, long long nloc) {
  const unsigned long long bytes = (unsigned long long)nblk * 4ull * (unsigned long long)nloc * 8ull;
  return (bytes <= (4ull << 30) && nloc < (1ll << 31) && nblk <= 65535) ? (size_t)bytes : 0;   // grid.y carries the block id
}

size_t blk_table_bytes(int nblk, long long nloc) {
  // info (int4), nbr (NNBR), phys, K0, tau, cur, flags, 5 lists, 4 correction lists, ctopb (3 doubles), source table
  return ((size_t)nblk * (16 + 4 * (NNBR + 5 + 5 + 4 + 5) + 24) + 1024 + 255) / 256 * 256 + blk_gsrc_bytes(nblk, nloc) + 256;
}

// C-16: block lattice, neighbour table (periodic dimensions close through it), per-block table offsets
int blk_setup(hamr_grid* g, void* tables) {
  BlkHost& H = g->bh;
  const hamr_params& p = g->par;
  int bn[3];
  const int nblk = blk_count(p, H.nslot, bn);
  if (nblk <= 0) return HAMR_EINVAL;
  H.on = true;
  H.nblk = nblk;
  H.tmax = p.lat_max_level > 0 ? p.lat_max_level : 0;
  H.nbr.assign((size_t)nblk * NNBR, -1);
  H.lev1.assign(nblk, 0);
  H.tau.assign(nblk, 0);
  H.I0.assign((size_t)nblk * 3, 0);
  H.forced.clear();
  H.phys.clear();
  BlkDev& B = g->D.B;
  const int ge2 = p.n[1] + 2 * NG + 1;
  std::vector<int> info((size_t)nblk * 4), phys(nblk), K0(nblk);
  auto id_of = [&](int s0, int s1, int s2) { return (s0 * H.nslot[1] + s1) * H.nslot[2] + s2; };
  const int nref = blk_refined_columns(p, p.n[0] / bn[0], bn[0]);   // slots 0 .. 2 nref - 1 are fine children
  H.refined = nref > 0;
  for (int s0 = 0; s0 < H.nslot[0]; s0++)
    for (int s1 = 0; s1 < H.nslot[1]; s1++)
      for (int s2 = 0; s2 < H.nslot[2]; s2++) {
        const int b = id_of(s0, s1, s2);
        const int sl[3] = {s0, s1, s2};
        // x1 index of the block's first zone in zones of its own level
        const int lev = s0 < 2 * nref ? 1 : 0;
        const int I0[3] = {lev ? s0 * bn[0] : (s0 - nref) * bn[0], s1 * bn[1], s2 * bn[2]};
        H.lev1[b] = lev;
        for (int d = 0; d < 3; d++) H.I0[(size_t)b * 3 + d] = I0[d];
        info[(size_t)b * 4 + 0] = (I0[0] + NG) * ge2 + I0[1] + NG;
        info[(size_t)b * 4 + 1] = lev;
        info[(size_t)b * 4 + 2] = I0[0];
        info[(size_t)b * 4 + 3] = I0[1];
        K0[b] = I0[2];
        int ph = 0;
        for (int d = 0; d < 3; d++) {
          if (sl[d] == 0 && p.bc_lo[d] != HAMR_BC_PERIODIC) ph |= 1 << d;
          if (sl[d] == H.nslot[d] - 1 && p.bc_hi[d] != HAMR_BC_PERIODIC) ph |= 8 << d;
        }
        phys[b] = ph;
        H.phys.push_back(ph);
        for (int o0 = -1; o0 <= 1; o0++)
          for (int o1 = -1; o1 <= 1; o1++)
            for (int o2 = -1; o2 <= 1; o2++) {
              const int o[3] = {o0, o1, o2};
              int q[3];
              bool inside = true;
              for (int d = 0; d < 3; d++) {
                q[d] = sl[d] + o[d];
                if (q[d] < 0 || q[d] >= H.nslot[d]) {
                  if (p.bc_lo[d] == HAMR_BC_PERIODIC) q[d] = (q[d] + H.nslot[d]) % H.nslot[d];
                  else inside = false;
                }
              }
              H.nbr[(size_t)b * NNBR + (o0 + 1) * 9 + (o1 + 1) * 3 + (o2 + 1)] = inside ? id_of(q[0], q[1], q[2]) : -1;
            }
        // NEXT-1 on blocks that cut x3: the rows beyond a transmissive pole lie in the block half a turn away
        const bool xpole = H.nslot[2] > 1 && ((s1 == 0 && p.bc_lo[1] == HAMR_BC_POLAR_TRANSMIT) ||
                                              (s1 == H.nslot[1] - 1 && p.bc_hi[1] == HAMR_BC_POLAR_TRANSMIT));
        for (int o0 = -1; o0 <= 1; o0++)
          for (int o2 = -1; o2 <= 1; o2++) {
            const int q0 = s0 + o0, q2 = ((s2 + H.nslot[2] / 2 + o2) % H.nslot[2] + H.nslot[2]) % H.nslot[2];
            H.nbr[(size_t)b * NNBR + 27 + (o0 + 1) * 3 + (o2 + 1)] =
                (xpole && q0 >= 0 && q0 < H.nslot[0]) ? id_of(q0, s1, q2) : -1;
          }
      }
  char* t = (char*)tables;
  auto take = [&](size_t bytes) { char* r = t; t += (bytes + 15) / 16 * 16; return r; };
  int4* d_info = (int4*)take((size_t)nblk * 16);
  int* d_nbr = (int*)take((size_t)nblk * NNBR * 4);
  int* d_phys = (int*)take((size_t)nblk * 4);
  int* d_K0 = (int*)take((size_t)nblk * 4);
  B.tau = (int*)take((size_t)nblk * 4);
  B.cur = (int*)take((size_t)nblk * 4);
  H.d_lists = (int*)take((size_t)nblk * 5 * 4);
  H.d_clists = (int*)take((size_t)nblk * 4 * 4);
  H.d_dlists = (int*)take((size_t)nblk * 5 * 4);
  H.hasderef.assign(nblk, 0);
  for (int b = 0; b < nblk; b++)
    for (int J = H.I0[(size_t)b * 3 + 1] - 1; J <= H.I0[(size_t)b * 3 + 1] + bn[1]; J++)
      if (deref_row_factor(p, J) > 1) H.hasderef[b] = 1;
  B.flags = (int*)take((size_t)nblk * 4);
  B.ctopb = (double*)take((size_t)nblk * 24);
  {
    const Lay& L = g->D.L;
    const long long nloc = (long long)L.e1 * L.e2 * (L.n[2] + 2 * NG + 1);
    const size_t gb = blk_gsrc_bytes(nblk, nloc);
    H.d_gsrc = gb ? (unsigned long long*)take(gb) : nullptr;
    H.gsrc_tau.clear();
    B.gsrc = H.d_gsrc;
    B.gloc = (int)nloc;
  }
  B.info = d_info; B.nbr = d_nbr; B.phys = d_phys; B.K0 = d_K0;
  B.list = H.d_lists; B.nact = 0;
  if (cudaMallocHost((void**)&H.h_ctop, (size_t)nblk * 3 * sizeof(double)) != cudaSuccess) return HAMR_ECUDA;
  if (cudaMallocHost((void**)&H.h_ints, (size_t)nblk * 16 * sizeof(int)) != cudaSuccess) return HAMR_ECUDA;
  std::vector<int> all(nblk);
  for (int b = 0; b < nblk; b++) all[b] = b;
  cudaStream_t st = g->stream;
  cudaError_t e = cudaSuccess;
  auto up = [&](void* dst, const void* src, size_t bytes) {
    if (e == cudaSuccess) e = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, st);
  };
  up(d_info, info.data(), (size_t)nblk * 16);
  up(d_nbr, H.nbr.data(), (size_t)nblk * NNBR * 4);
  up(d_phys, phys.data(), (size_t)nblk * 4);
  up(d_K0, K0.data(), (size_t)nblk * 4);
  up(H.d_lists, all.data(), (size_t)nblk * 4);                       // level 0 list (every block at tau = 0)
  up(H.d_lists + (size_t)4 * nblk, all.data(), (size_t)nblk * 4);    // the list of every block
  if (e == cudaSuccess) e = cudaMemsetAsync(B.tau, 0, (size_t)nblk * 4, st);
  if (e == cudaSuccess) e = cudaMemsetAsync(B.cur, 0, (size_t)nblk * 4, st);
  if (e == cudaSuccess) e = blk_upload_flags(g);
  if (e == cudaSuccess) e = blk_upload_dlists(g);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);               // the host vectors go out of scope
  for (int i = 0; i < 4; i++) { H.nlist[i] = 0; H.nclist[i] = 0; H.tb_u[i] = 0; H.dt_u[i] = 2 << i; H.has_new[i] = 0; }
  H.nlist[0] = nblk;
  H.dt0 = 0.0;
  return e == cudaSuccess ? HAMR_OK : HAMR_ECUDA;
}

void blk_pack(hamr_grid* g, const double* dense, int kind, int stag, bool zero_pole) {
  const Dev D = dev_list(g, 4);
  const Lay& L = D.L;
  int m[3] = {L.n[0], L.n[1], L.n[2]};
  if (stag >= 0) m[stag] += 1;
  const long long tot = (long long)m[0] * m[1] * m[2] * D.B.nblk;
  double* a0 = kind < 5 ? g->s[0].P[kind] : g->s[0].Bf[kind - 5];
  double* a2 = kind < 5 ? g->s[2].P[kind] : g->s[2].Bf[kind - 5];
  Launch l_(g, K_OTHER);
  k_blk_pack<<<(unsigned)((tot + 255) / 256), 256, 0, g->stream>>>(D, dense, a0, a2, stag, zero_pole ? 1 : 0,
                                                                   g->par.n[0], g->par.n[1], g->par.n[2]);
}

void blk_unpack(hamr_grid* g, int kind, double* dense) {
  const Dev D = dev_list(g, 4);
  const Lay& L = D.L;
  const int stag = kind >= 8 ? kind - 8 : -1;
  int m[3] = {L.n[0], L.n[1], L.n[2]};
  if (stag >= 0) m[stag] += 1;
  const long long tot = (long long)m[0] * m[1] * m[2] * D.B.nblk;
  auto arr = [&](int buf) -> const double* {
    const Fields& f = g->s[buf];
    return kind < 5 ? f.P[kind] : (kind < 8 ? f.Bc[kind - 5] : f.Bf[kind - 8]);
  };
  Launch l_(g, K_OTHER);
  k_blk_unpack<<<(unsigned)((tot + 255) / 256), 256, 0, g->stream>>>(D, arr(0), arr(2), dense, stag, g->par.n[0],
                                                                     g->par.n[1], g->par.n[2]);
}

void blk_pack_one(hamr_grid* g, int b, const double* dense, int kind, int stag, bool zero_pole) {
  const Lay& L = g->D.L;
  int m[3] = {L.n[0], L.n[1], L.n[2]};
  if (stag >= 0) m[stag] += 1;
  const long long tot = (long long)m[0] * m[1] * m[2] * (b < 0 ? g->bh.nblk : 1);
  double* a0 = kind < 5 ? g->s[0].P[kind] : g->s[0].Bf[kind - 5];
  double* a2 = kind < 5 ? g->s[2].P[kind] : g->s[2].Bf[kind - 5];
  Launch l_(g, K_OTHER);
  k_blk_pack1<<<(unsigned)((tot + 255) / 256), 256, 0, g->stream>>>(g->D, b, dense, a0, a2, stag, zero_pole ? 1 : 0, 0);
}

void blk_unpack_one(hamr_grid* g, int b, int kind, double* dense) {
  const Lay& L = g->D.L;
  const int stag = kind >= 8 ? kind - 8 : -1;
  int m[3] = {L.n[0], L.n[1], L.n[2]};
  if (stag >= 0) m[stag] += 1;
  const long long tot = (long long)m[0] * m[1] * m[2] * (b < 0 ? g->bh.nblk : 1);
  auto arr = [&](int buf) -> double* {
    const Fields& f = g->s[buf];
    return kind < 5 ? f.P[kind] : (kind < 8 ? f.Bc[kind - 5] : f.Bf[kind - 8]);
  };
  Launch l_(g, K_OTHER);
  k_blk_pack1<<<(unsigned)((tot + 255) / 256), 256, 0, g->stream>>>(g->D, b, dense, arr(0), arr(2), stag, 0, 1);
}

static void blk_ghosts(hamr_grid* g, const Dev& D, int role, long long s_u, bool all, bool zero_ctop) {
  if (D.B.nact == 0) return;
  const Lay& L = D.L;
  const int per = L.e1 * L.e2 * (L.n[2] + 2 * NG + 1);
  Launch l_(g, K_GHOSTS);
  for (int first = 0; first < D.B.nact; first += 65535) {   // grid.y limit
    Dev Dc = D;
    Dc.B.list = D.B.list + first;
    Dc.B.nact = std::min(65535, D.B.nact - first);
    k_blk_ghosts<<<dim3((per + 255) / 256, Dc.B.nact), 256, 0, g->stream>>>(Dc, bufs_of(g), clocks_of(g), role, s_u,
                                                                         all ? 1 : 0, zero_ctop ? 1 : 0);
  }
}

// one stage of C-12 on every block of time level tau (C-17)
static void blk_stage(hamr_grid* g, int tau, bool corrector) {
  BlkHost& H = g->bh;
  const Dev D = dev_list(g, tau);
  if (D.B.nact > 0) {
    const long long s_u = H.tb_u[tau] + (corrector ? H.dt_u[tau] / 2 : 0);
    blk_ghosts(g, D, corrector ? 1 : 0, s_u, false, corrector);
    const Fields& s0 = g->s[0];
    const Fields& s1 = g->s[1];
    const Fields& s2 = g->s[2];
    if (D.entropy) launch_kappa(g, D, corrector ? s1 : s0, corrector ? s1 : s2);   // C-18: kappa of the level's stage sources
    launch_flux_on(g, D, corrector ? s1 : s0, corrector ? s1 : s2, corrector, true);
    launch_ct_on(g, D, corrector ? s1 : s0, corrector ? s1 : s2);
    launch_deref_fix_edges(g, D);
    if (H.refined) {   // C-16: same-time flux / EMF agreement on the refinement interface
      const Lay& L = D.L;
      const long long tot = 2LL * (L.n[1] + 1) * (L.n[2] + 1) * D.B.nact;
      Launch l_(g, K_OTHER);
      k_blk_iface<<<(unsigned)((tot + 127) / 128), 128, 0, g->stream>>>(D);
    }
    const double lev_fac = (double)(1 << tau);   // dt_b = 2^tau dt_0
    if (corrector && tau < H.tmax) {
      const int first = (H.tb_u[tau] % (2LL * H.dt_u[tau])) == 0 ? 1 : 0;
      const Lay& L = D.L;
      const long long tot = (long long)(L.n[0] + 1) * (L.n[1] + 1) * (L.n[2] + 1) * D.B.nact;
      Launch l_(g, K_OTHER);
      if (D.entropy) k_blk_registers<true><<<(unsigned)((tot + 127) / 128), 128, 0, g->stream>>>(D, first, lev_fac);
      else k_blk_registers<false><<<(unsigned)((tot + 127) / 128), 128, 0, g->stream>>>(D, first, lev_fac);
    }
    if (!corrector) {
      const Roles ra = {s0, s0, s1}, rb = {s2, s2, s1};
      launch_update_on(g, D, ra, rb, 0.5 * lev_fac, true);
      launch_deref_sync(g, D, s1, s1);
    } else {
      const Roles ra = {s1, s0, s2}, rb = {s1, s2, s0};
      launch_update_on(g, D, ra, rb, lev_fac, false);
      launch_deref_sync(g, D, s2, s0);
    }
  }
  if (corrector) H.has_new[tau] = 1;
}

// C-17 correct(tau-1 -> tau) on the level-tau blocks that touch a level tau-1 block
static void blk_correct(hamr_grid* g, int tau) {
  BlkHost& H = g->bh;
  if (H.nclist[tau] == 0) return;
  Dev D = g->D;
  D.B.list = H.d_clists + (size_t)tau * H.nblk;
  D.B.nact = H.nclist[tau];
  const Lay& L = D.L;
  const double lev_fac = (double)(1 << tau);
  long long tot = (long long)(L.n[0] + 1) * (L.n[1] + 1) * (L.n[2] + 1) * D.B.nact;
  {
    Launch l_(g, K_OTHER);
    k_blk_correct_faces<<<(unsigned)((tot + 127) / 128), 128, 0, g->stream>>>(D, bufs_of(g), tau, lev_fac);
  }
  tot = (long long)L.n[0] * L.n[1] * L.n[2] * D.B.nact;
  {
    Launch l_(g, K_OTHER);
    if (D.entropy || D.drift) k_blk_correct_zones<true><<<(unsigned)((tot + 127) / 128), 128, 0, g->stream>>>(D, bufs_of(g), tau, lev_fac);
    else k_blk_correct_zones<false><<<(unsigned)((tot + 127) / 128), 128, 0, g->stream>>>(D, bufs_of(g), tau, lev_fac);
  }
  launch_deref_sync(g, D, g->s[2], g->s[0]);   // the corrected new state of a block with cur == 0 / 2
}

static void blk_rotate(hamr_grid* g, int tau) {
  BlkHost& H = g->bh;
  const Dev D = dev_list(g, tau);
  if (D.B.nact > 0) {
    Launch l_(g, K_OTHER);
    k_blk_rotate<<<(D.B.nact + 127) / 128, 128, 0, g->stream>>>(D);
  }
  H.tb_u[tau] += H.dt_u[tau];
  H.has_new[tau] = 0;
}

// C-17: advance(tau) = predictor, first half of the finer levels, corrector, second half, correction
static void blk_advance(hamr_grid* g, int tau) {
  blk_stage(g, tau, false);
  if (tau > 0) blk_advance(g, tau - 1);
  blk_stage(g, tau, true);
  if (tau > 0) {
    blk_advance(g, tau - 1);
    blk_correct(g, tau);
  }
  blk_rotate(g, tau);
}

// C-14 / C-17: the next dt and, under LAT, every block's time level.  after_step: a coarse step was just taken.
static int blk_assign(hamr_grid* g, bool after_step) {
  BlkHost& H = g->bh;
  const int nblk = H.nblk;
  cudaStream_t st = g->stream;
  if (H.tmax == 0) {  // one global dt, found on the device; every block stays on level 0
    Launch l_(g, K_DT);
    k_blk_dt<<<1, 256, 0, st>>>(dev_list(g, 4), after_step ? 1 : 0);
    for (int i = 0; i < 4; i++) { H.tb_u[i] = 0; H.dt_u[i] = 2 << i; H.has_new[i] = 0; }
    return HAMR_OK;
  }
  if (after_step) {
    Launch l_(g, K_DT);
    k_blk_time<<<1, 1, 0, st>>>(g->D, (double)(1 << H.tmax));
  }
  if (cudaMemcpyAsync(H.h_ctop, g->D.B.ctopb, (size_t)nblk * 24, cudaMemcpyDeviceToHost, st) != cudaSuccess) return HAMR_ECUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return HAMR_ECUDA;
  // per-block Courant step (PAPER.md:93 fn. 2), levels in factors of two above the smallest
  std::vector<double> dtb(nblk);
  double dt0 = 1e300;
  for (int b = 0; b < nblk; b++) {
    double s = 0.0;
    for (int d = 0; d < 3; d++) {
      const double dx = (d == 0 && H.lev1[b]) ? 0.5 * g->D.dx[0] : g->D.dx[d];
      s += H.h_ctop[(size_t)b * 3 + d] / dx;
    }
    dtb[b] = g->D.cour / s;
    dt0 = std::min(dt0, dtb[b]);
  }
  if (!H.forced.empty()) {
    dt0 = 1e300;
    for (int b = 0; b < nblk; b++) {
      H.tau[b] = std::min(H.tmax, std::max(0, H.forced[b]));
      dt0 = std::min(dt0, dtb[b] / (double)(1 << H.tau[b]));
    }
  } else {
    for (int b = 0; b < nblk; b++) {
      int tau = 0;
      double lim = 2.0 * dt0;
      while (tau < H.tmax && dtb[b] >= lim) { tau++; lim *= 2.0; }
      H.tau[b] = tau;
    }
  }
  // neighbours across faces, edges and corners differ by at most one level
  std::vector<int> nt(nblk);
  for (bool changed = true; changed;) {
    changed = false;
    for (int b = 0; b < nblk; b++) {
      int t = H.tau[b];
      for (int a = 0; a < NNBR; a++) {
        const int q = H.nbr[(size_t)b * NNBR + a];
        if (q >= 0) t = std::min(t, H.tau[q] + 1);
      }
      nt[b] = t;
      if (t != H.tau[b]) changed = true;
    }
    H.tau = nt;
  }
  // lists per level; correction lists; upload
  int* hl = H.h_ints;                       // [4][nblk] lists, [4][nblk] correction lists, [nblk] tau
  for (int i = 0; i < 4; i++) { H.nlist[i] = 0; H.nclist[i] = 0; }
  for (int b = 0; b < nblk; b++) {
    const int t = H.tau[b];
    hl[(size_t)t * nblk + H.nlist[t]++] = b;
    bool any = false;
    for (int a = 0; a < 27 && !any; a++) {   // (a block across the pole shares no face or edge)
      const int q = H.nbr[(size_t)b * NNBR + a];
      any = q >= 0 && H.tau[q] == t - 1;
    }
    if (any) hl[(size_t)(4 + t) * nblk + H.nclist[t]++] = b;
    hl[(size_t)8 * nblk + b] = t;
  }
  cudaError_t e = cudaMemcpyAsync(H.d_lists, hl, (size_t)4 * nblk * 4, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(H.d_clists, hl + (size_t)4 * nblk, (size_t)4 * nblk * 4, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(g->D.B.tau, hl + (size_t)8 * nblk, (size_t)nblk * 4, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = blk_upload_flags(g);
  if (e == cudaSuccess) e = blk_upload_dlists(g);
  if (e == cudaSuccess) blk_build_gsrc(g);
  H.dt0 = dt0;
  g->h_pinned[56] = dt0;
  if (e == cudaSuccess) e = cudaMemcpyAsync(g->D.scal + S_DT, g->h_pinned + 56, sizeof(double), cudaMemcpyHostToDevice, st);
  for (int i = 0; i < 4; i++) { H.tb_u[i] = 0; H.dt_u[i] = 2 << i; H.has_new[i] = 0; }
  return e == cudaSuccess ? HAMR_OK : HAMR_ECUDA;
}

int blk_set_levels(hamr_grid* g, const int* tau) {
  BlkHost& H = g->bh;
  if (!H.on) return HAMR_EINVAL;
  H.forced.clear();
  if (tau) H.forced.assign(tau, tau + H.nblk);
  return HAMR_OK;
}

// after the state has been packed: every block on level 0, ghost fill, one flux pass for the first dt (C-14)
int blk_initial(hamr_grid* g) {
  BlkHost& H = g->bh;
  cudaStream_t st = g->stream;
  std::fill(H.tau.begin(), H.tau.end(), 0);
  for (int i = 0; i < 4; i++) { H.nlist[i] = 0; H.nclist[i] = 0; H.tb_u[i] = 0; H.dt_u[i] = 2 << i; H.has_new[i] = 0; }
  H.nlist[0] = H.nblk;
  if (cudaMemsetAsync(g->D.B.tau, 0, (size_t)H.nblk * 4, st) != cudaSuccess) return HAMR_ECUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return HAMR_ECUDA;   // the pinned staging area is reused
  if (blk_upload_flags(g) != cudaSuccess) return HAMR_ECUDA;
  if (blk_upload_dlists(g) != cudaSuccess) return HAMR_ECUDA;
  blk_build_gsrc(g);
  // level-0 list = every block
  if (cudaMemcpyAsync(H.d_lists, H.d_lists + (size_t)4 * H.nblk, (size_t)H.nblk * 4, cudaMemcpyDeviceToDevice, st) != cudaSuccess)
    return HAMR_ECUDA;
  const Dev D = dev_list(g, 4);
  launch_deref_project(g, D, g->s[0], g->s[2]);
  launch_deref_sync(g, D, g->s[0], g->s[2]);
  blk_ghosts(g, D, 0, 0, true, true);
  if (D.entropy) launch_kappa(g, D, g->s[0], g->s[2]);
  launch_flux_on(g, D, g->s[0], g->s[2], true);
  return blk_assign(g, false);
}

int blk_step(hamr_grid* g, int nsteps) {
  for (int s = 0; s < nsteps; s++) {
    blk_advance(g, g->bh.tmax);
    const int rc = blk_assign(g, true);
    if (rc != HAMR_OK) return rc;
  }
  return HAMR_OK;
}

static void blk_diag(hamr_grid* g, int what) {
  const Dev D = dev_list(g, 4);
  const Lay& L = D.L;
  const long long tot = (long long)L.n[0] * L.n[1] * L.n[2] * D.B.nblk;
  Launch l_(g, K_OTHER);
  k_blk_diag<<<(unsigned)((tot + 255) / 256), 256, 0, g->stream>>>(D, bufs_of(g), what);
}

void blk_divb(hamr_grid* g) {
  g->launches++;
  k_blk_zero_scal<<<1, 1, 0, g->stream>>>(g->D, S_DENMAX, 2);
  blk_diag(g, 0);
  blk_diag(g, 1);
}

void blk_totals(hamr_grid* g) {
  g->launches++;
  k_blk_zero_scal<<<1, 1, 0, g->stream>>>(g->D, S_TOT0, 5);
  blk_diag(g, 2);
}

void blk_check_finite(hamr_grid* g) { blk_diag(g, 3); }

// ---- C-20 (the x1-only part): regridding of the x1 refinement level --------------------------------
// refinement criterion "a cutoff on the maximum density in each block"; "(de-)refinement ...
// including the divergence-free prolongation and restriction of magnetic fields (Balsara 2001)".  The refined block
// columns are contiguous from the inner x1 edge (C-16), so a regrid moves the outer edge of the refined region: a new
// grid is created with another r_refine_max and the state is transferred on the device.

// maximum density over the active zones of every block: one CTA per block, result to out[b]
__global__ void __launch_bounds__(256) k_blk_max_rho(Dev Dv, Bufs B, double* __restrict__ out) {
  const Lay& L = Dv.L;
  const int b = blockIdx.x;
  const double* rho = buf_arr(B, Dv.B.cur[b], 0) + (long long)b * Dv.B.blen;
  const int tot = L.n[0] * L.n[1] * L.n[2];
  double m = 0.0;
  for (int t = threadIdx.x; t < tot; t += blockDim.x) {
    const int k = t % L.n[2], j = (t / L.n[2]) % L.n[1], i = t / (L.n[2] * L.n[1]);
    m = fmax(m, rho[L.idx(i, j, k)]);
  }
  __shared__ double wm[8];
  m = warp_max(m);
  if ((threadIdx.x & 31) == 0) wm[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 8; w++) m = fmax(m, wm[w]);
    out[b] = m;
  }
}

// State transfer between two lattices of the same blocks that differ in the refined columns.  map[bn] = {kind, q0, q1,
// child}: kind 0 copy of old block q0; 1 prolongation of old coarse block q0, this block being its child `child`;
// 2 restriction of the old fine blocks q0 (low half) and q1 (high half).  One thread per zone / face location
// (i <= n0, j <= n1, k <= n2) of every new block; the old state must have its x1 ghost zones filled.
//   prolongation: hydro piecewise linear in x1 with the MC-limited slope of the coarse values, a quarter of a coarse
//   zone off the coarse centre (the operator of the ghost fill, C-16); x1-faces: coincident ones copied, the new face
//   in the middle of a coarse zone the mean of that zone's two faces; transverse faces: the coarse zone's value for both
//   children: every child keeps the coarse zone's divergence.  restriction: means of the two fine values; x1-faces the
//   coincident fine faces.
__global__ void __launch_bounds__(256) k_blk_regrid(Dev Do, Bufs Bo, Dev Dn, Fields sn, const int4* __restrict__ map) {
  const Lay& L = Dn.L;
  const int n0 = L.n[0], n1 = L.n[1], n2 = L.n[2];
  const int c2 = n2 + 1, c1 = n1 + 1;
  const unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (unsigned)((n0 + 1) * c1 * c2)) return;
  const int bn = blockIdx.y;
  const int4 m = __ldg(map + bn);
  const unsigned tj = t / (unsigned)c2;
  const int k = (int)(t - tj * c2), i = (int)(tj / (unsigned)c1), j = (int)(tj - (unsigned)i * c1);
  const bool zi = i < n0, zj = j < n1, zk = k < n2;
  const long long zn = (long long)bn * Dn.B.blen + L.idx(i, j, k);
  if (m.x == 0) {
    const int cur = Do.B.cur[m.y];
    const long long zo = (long long)m.y * Do.B.blen + L.idx(i, j, k);
    if (zi && zj && zk)
      for (int c = 0; c < 5; c++) sn.P[c][zn] = buf_arr(Bo, cur, c)[zo];
    if (zj && zk) sn.Bf[0][zn] = buf_arr(Bo, cur, 5)[zo];
    if (zi && zk) sn.Bf[1][zn] = buf_arr(Bo, cur, 6)[zo];
    if (zi && zj) sn.Bf[2][zn] = buf_arr(Bo, cur, 7)[zo];
  } else if (m.x == 1) {
    const int cur = Do.B.cur[m.y];
    const long long base = (long long)m.y * Do.B.blen;
    const int c0 = m.w * (n0 / 2), ic = c0 + i / 2;
    if (zi && zj && zk)
      for (int c = 0; c < 5; c++) {
        const double* a = buf_arr(Bo, cur, c) + base;
        const double am = a[L.idx(ic - 1, j, k)], a0 = a[L.idx(ic, j, k)], ap = a[L.idx(ic + 1, j, k)];
        const double dl = a0 - am, dr = ap - a0;
        double sl = 0.0;
        if (dl * dr > 0.0) {
          sl = fmin(0.5 * fabs(ap - am), 2.0 * fmin(fabs(dl), fabs(dr)));
          if (dl < 0.0) sl = -sl;
        }
        sn.P[c][zn] = 0.5 * (a0 + ((i & 1) ? a0 + 0.5 * sl : a0 - 0.5 * sl));
      }
    if (zj && zk) {
      const double* a = buf_arr(Bo, cur, 5) + base;
      const int f2 = 2 * c0 + i;
      sn.Bf[0][zn] = (f2 & 1) ? 0.5 * (a[L.idx(f2 / 2, j, k)] + a[L.idx(f2 / 2 + 1, j, k)]) : a[L.idx(f2 / 2, j, k)];
    }
    if (zi && zk) sn.Bf[1][zn] = buf_arr(Bo, cur, 6)[base + L.idx(ic, j, k)];
    if (zi && zj) sn.Bf[2][zn] = buf_arr(Bo, cur, 7)[base + L.idx(ic, j, k)];
  } else {
    const int hh = (i == n0) ? 1 : ((i < n0 / 2) ? 0 : 1);
    const int q = hh ? m.z : m.y;
    const int cur = Do.B.cur[q];
    const long long base = (long long)q * Do.B.blen;
    const int i0 = 2 * i - hh * n0;
    const long long za = base + L.idx(i0, j, k), zb = base + L.idx(i0 + 1, j, k);
    if (zi && zj && zk)
      for (int c = 0; c < 5; c++) { const double* a = buf_arr(Bo, cur, c); sn.P[c][zn] = 0.5 * (a[za] + a[zb]); }
    if (zj && zk) sn.Bf[0][zn] = buf_arr(Bo, cur, 5)[za];
    if (zi && zk) { const double* a = buf_arr(Bo, cur, 6); sn.Bf[1][zn] = 0.5 * (a[za] + a[zb]); }
    if (zi && zj) { const double* a = buf_arr(Bo, cur, 7); sn.Bf[2][zn] = 0.5 * (a[za] + a[zb]); }
  }
}

// the refinement criterion as the r_refine_max it asks for: every block column up to the outermost one that holds a
// zone with rho >= rho_cut (0: none).  Synchronises the stream (one read-back of a double per block).
int blk_refine_radius(hamr_grid* g, double rho_cut, double* r_new) {
  BlkHost& H = g->bh;
  const hamr_params& p = g->par;
  if (g->stage_doubles < (size_t)H.nblk) return HAMR_ENOMEM;
  {
    Launch l_(g, K_OTHER);
    k_blk_max_rho<<<H.nblk, 256, 0, g->stream>>>(g->D, bufs_of(g), stage_take(g));
  }
  // h_ctop is pinned, [nblk][3] doubles, idle between steps
  if (cudaMemcpyAsync(H.h_ctop, g->stage, (size_t)H.nblk * 8, cudaMemcpyDeviceToHost, g->stream) != cudaSuccess) return HAMR_ECUDA;
  if (cudaStreamSynchronize(g->stream) != cudaSuccess) return HAMR_ECUDA;
  const int nb0 = g->D.L.n[0], ncol = p.n[0] / nb0;
  int cmax = -1;
  for (int b = 0; b < H.nblk; b++) {
    const int c = H.I0[(size_t)b * 3] / nb0, col = H.lev1[b] ? c / 2 : c;
    if (H.h_ctop[b] >= rho_cut) cmax = std::max(cmax, col);
  }
  if (cmax < 0) { *r_new = 0.0; return HAMR_OK; }
  const bool ks = p.metric == HAMR_METRIC_KERR_SCHILD;
  const double lo = ks ? std::log(p.xmin[0]) : p.xmin[0], hi = ks ? std::log(p.xmax[0]) : p.xmax[0];
  const double edge = lo + (hi - lo) * (double)(cmax + 1) / (double)ncol;
  *r_new = ks ? std::exp(edge) : edge;
  return HAMR_OK;
}

// state of go (between coarse steps) onto gn, created with the same parameters but for r_refine_max; gn's stream
int blk_regrid(hamr_grid* go, hamr_grid* gn) {
  BlkHost& Ho = go->bh;
  BlkHost& Hn = gn->bh;
  const Lay& L = go->D.L;
  const int nb0 = L.n[0], ncol = go->par.n[0] / nb0;
  const int nref_o = (Ho.nslot[0] - ncol), nref_n = (Hn.nslot[0] - ncol);
  if (nref_o != nref_n && (nb0 & 1)) return HAMR_EINVAL;
  // x1 ghost zones of the old state: the slopes of the prolongation read one zone beyond a block (all clocks are 0
  // between coarse steps, so every sample is a plain copy of a time-n state)
  blk_ghosts(go, dev_list(go, 4), 0, 0, false, false);
  std::vector<int> map((size_t)Hn.nblk * 4);
  auto old_id = [&](int s0, int s1, int s2) { return (s0 * Ho.nslot[1] + s1) * Ho.nslot[2] + s2; };
  for (int s0 = 0; s0 < Hn.nslot[0]; s0++)
    for (int s1 = 0; s1 < Hn.nslot[1]; s1++)
      for (int s2 = 0; s2 < Hn.nslot[2]; s2++) {
        const int bn = (s0 * Hn.nslot[1] + s1) * Hn.nslot[2] + s2;
        const bool fine = s0 < 2 * nref_n;
        const int col = fine ? s0 / 2 : s0 - nref_n, child = fine ? s0 & 1 : 0;
        const bool old_fine = col < nref_o;
        int* m = &map[(size_t)bn * 4];
        if (fine == old_fine) { m[0] = 0; m[1] = old_id(old_fine ? 2 * col + child : col + nref_o, s1, s2); m[2] = -1; m[3] = 0; }
        else if (fine) { m[0] = 1; m[1] = old_id(col + nref_o, s1, s2); m[2] = -1; m[3] = child; }
        else { m[0] = 2; m[1] = old_id(2 * col, s1, s2); m[2] = old_id(2 * col + 1, s1, s2); m[3] = 0; }
      }
  // the map travels through the new grid's staging buffer (it is free until the state is committed)
  if (gn->stage_doubles * 8 < map.size() * 4) return HAMR_ENOMEM;
  int4* d_map = (int4*)gn->stage;
  cudaError_t e = cudaMemcpyAsync(d_map, map.data(), map.size() * 4, cudaMemcpyHostToDevice, go->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(gn->D.B.cur, 0, (size_t)Hn.nblk * sizeof(int), go->stream);
  if (e != cudaSuccess) return HAMR_ECUDA;
  {
    Launch l_(go, K_OTHER);
    const int per = (L.n[0] + 1) * (L.n[1] + 1) * (L.n[2] + 1);
    k_blk_regrid<<<dim3((per + 255) / 256, Hn.nblk), 256, 0, go->stream>>>(go->D, bufs_of(go), gn->D, gn->s[0], d_map);
  }
  // the old grid's stream has written the new grid's arrays: finish before the new grid's stream goes on
  if (cudaStreamSynchronize(go->stream) != cudaSuccess) return HAMR_ECUDA;
  return cudaGetLastError() == cudaSuccess ? HAMR_OK : HAMR_ECUDA;
}

}  // namespace hamr
