// sweep.cuh — the two hot kernels: the active-cell sub-sweep (Algorithm 2) and the cell
// shift / re-bin (Algorithm 4), re-designed for sm_100a.  See DESIGN.md "Kernels".
#pragma once
#include "common.cuh"

namespace mpmc {

#ifndef MPMC_SUB_THREADS
#define MPMC_SUB_THREADS 128
#endif
#ifndef MPMC_SUB_MINB
#define MPMC_SUB_MINB 1
#endif
constexpr int SUB_THREADS = MPMC_SUB_THREADS;
constexpr int SUB_MINB = MPMC_SUB_MINB;      // minimum resident blocks per SM asked of ptxas (register cap)
constexpr int SHIFT_THREADS = 256;

// ---------------------------------------------------------------------------------------------------------
// Sub-sweep kernel.  One thread per cell of the active checkerboard set (the paper's mapping, L158/L260),
// over the dense colour plane so that a warp's 32 cells are contiguous.
//
//  * the cell's own <= 4 disks and the first NF disks of each of the 8 neighbour cells are loaded ONCE into
//    registers, neighbours already translated into the active cell's frame (q = l_j + s, L154/L196), and are
//    reused by all n_s moves; empty entries hold a far-away sentinel so the overlap loop has a fixed trip
//    count and no divergence (the paper's (-10,-10) trick, L295/L346);
//  * entries are kept NEGATED and in pairs, so that one overlap test of two disks is four packed fp32x2
//    instructions of sm_100a (FADD2, FADD2, FMUL2, FFMA2: D = M + (-q), r^2 = fma(Dx, Dx, Dy*Dy)) and two
//    compares; every lane of a packed instruction is one IEEE rn operation, so results are unchanged
//    (-(a+b) = (-a)+(-b) exactly under round-to-nearest-even).  fp64 uses the same code with scalar pairs;
//  * NF = 2 covers every neighbour at w ~ sigma except a rare few (occupancy 0/1/2); neighbours with more
//    than NF disks set a bit in `big` and their remaining slots are re-read from L1/L2 inside the move loop;
//    NF = 4 is the instantiation for the paper's own regime w ~ 1.4 sigma (L152);
//  * Philox4x32-10 keyed on (seed; cell, sweep, move) replaces the per-thread Saru stream (L180, L262);
//  * accept/reject is computed without early exit: all lanes run the same instruction stream.
//  * NS > 0 fixes n_s at compile time (4 and 8, the BASELINE configs): the n_s Philox calls, which depend
//    only on (seed, sweep, cell, s), are issued up front and interleaved (4-8 independent dependency chains
//    instead of one), and the move loop is fully unrolled; NS = 0 is the generic run-time loop;
// SETK: index into Ctl::order (0..3) or, for the test hook, 4 + explicit set.
// ---------------------------------------------------------------------------------------------------------
template <typename P, int NF, int NS, bool DEBUG>
__global__ void __launch_bounds__(SUB_THREADS, SUB_MINB)
k_sub_sweep(const __grid_constant__ Params p, const uint32_t setk) {
  using R = Real<P>;
  using P2 = typename R::T2;
  using Pair = typename R::Pair;
  constexpr int NPN = 8 * NF / 2;        // neighbour pairs
  const Ctl* __restrict__ ctl = p.ctl;
  const uint32_t Q = setk < 4 ? ctl->order[setk] : (setk & 3u);
  const unsigned long long t = ctl->t;
  const uint32_t cur = ctl->cur;
  const uint32_t offx = Q & 1u, offy = Q >> 1;
  const uint32_t ci_raw = blockIdx.x * SUB_THREADS + threadIdx.x;
  const bool valid = ci_raw < p.Mq;
  const uint32_t ci = valid ? ci_raw : p.Mq - 1u;      // clamped: every lane may prefetch
  const uint32_t t_lo = (uint32_t)t, t_hi = (uint32_t)(t >> 32);

  // base pointers of the current buffer; planes are addressed with 32-bit element indices
  const uint8_t* __restrict__ cntb = p.cnt[cur];
  P2* __restrict__ posb = reinterpret_cast<P2*>(p.pos[cur]);
  const uint32_t Mqp = p.Mqp;

  // ---- cell and neighbour indices in the colour planes, with periodic wrap ----
  const uint32_t ya = div_hx(p, ci), xa = ci - ya * p.hx;
  const uint32_t cell = (2u * ya + offy) * p.mx + (2u * xa + offx);   // canonical cell id y*mx + x
  const uint32_t xl = offx ? xa : (xa == 0 ? p.hx - 1 : xa - 1);        // plane column of cell x-1
  const uint32_t xr = offx ? (xa + 1 == p.hx ? 0 : xa + 1) : xa;        // ... of cell x+1
  const uint32_t yd = offy ? ya : (ya == 0 ? p.hy - 1 : ya - 1);
  const uint32_t yu = offy ? (ya + 1 == p.hy ? 0 : ya + 1) : ya;
  const uint32_t rowd = yd * p.hx, rowa = ya * p.hx, rowu = yu * p.hx;

  // ---- level-1 loads, all independent: count and slot 0 of the 3x3 cells (idx 4 = own cell) ----
  uint32_t cidx[9], cj[9];
  P2 v0[9];
#pragma unroll
  for (int idx = 0; idx < 9; ++idx) {
    const int ox = idx % 3 - 1, oy = idx / 3 - 1;
    const uint32_t qn = ((offy ^ (uint32_t)(oy & 1)) << 1) | (offx ^ (uint32_t)(ox & 1));
    const uint32_t cn = (oy < 0 ? rowd : oy > 0 ? rowu : rowa) + (ox < 0 ? xl : ox > 0 ? xr : xa);
    cidx[idx] = qn * Mqp + cn;                       // count index; slot s of the cell is at 4*qn*Mqp + s*Mqp + cn
    cj[idx] = ld_u8_early(cntb + cidx[idx]);
    v0[idx] = ld_pos_early(posb + (cidx[idx] + 3u * qn * Mqp));
  }

  // ---- arithmetic that needs no memory, issued while the loads are in flight: the Philox words of the
  //      shuffle (Alg. 2 line 9) and of the first half of the displacements (line 12, L190; A2, A9) ----
  const P dmax = R::d(p);
  // Philox block q serves moves 2q (words 0, 1) and 2q + 1 (words 2, 3)  (reading A9)
  auto displacement2 = [&](uint32_t q, P& ax, P& ay, P& bx, P& by) {
    uint32_t Rw[4];
    philox4x32_10(cell, t_lo, t_hi, q, p.seed_lo, p.seed_hi, Rw);
    ax = R::mul(dmax, R::sym(Rw[0])); ay = R::mul(dmax, R::sym(Rw[1]));
    bx = R::mul(dmax, R::sym(Rw[2])); by = R::mul(dmax, R::sym(Rw[3]));
  };
  uint32_t S[4];
  philox4x32_10(cell, t_lo, t_hi, SLOT_SHUFFLE, p.seed_lo, p.seed_hi, S);
  static_assert(NS % 4 == 0, "compile-time n_s must be a multiple of 4");
  constexpr int NSA = NS > 0 ? NS : 2;
  P ddx[NSA], ddy[NSA];
  if (NS > 0) {
#pragma unroll
    for (int q = 0; q < NS / 4; ++q) displacement2((uint32_t)q, ddx[2 * q], ddy[2 * q], ddx[2 * q + 1], ddy[2 * q + 1]);
  }

  uint32_t n_acc = 0, n_rb = 0, n_ro = 0;
  // Empty cells (and the clamped lanes past the end) run the same instruction stream on sentinels and are
  // masked out of the counters and the write-back: no lane-dependent branch stands between the loads above
  // and their first use, so the loads are issued before the Philox arithmetic and overlap it.  (Skipping an
  // empty cell saves nothing unless all 32 cells of a warp are empty; Alg. 2 lines 4-7, L181-185.)
  if (!valid) cj[4] = 0u;
  const uint32_t n = cj[4];
  const uint32_t nv = n > 0u ? n : 1u;                 // visiting modulus; an empty cell "visits" a sentinel

  {
    const P wx = R::wx(p), wy = R::wy(p), sigma2 = R::sigma2(p);
    const P FAR = R::far_away();
    const Pair MINUS1 = R::pair((P)-1, (P)-1);

    // ---- level-2 loads: the occupied higher slots (rare at w ~ sigma) ----
    P2 v1[9], v2[9], v3[9];
    uint32_t big = 0;          // bit idx set: neighbour idx holds more than NF disks
#pragma unroll
    for (int idx = 0; idx < 9; ++idx) {
      const int ox = idx % 3 - 1, oy = idx / 3 - 1;
      const uint32_t qn = ((offy ^ (uint32_t)(oy & 1)) << 1) | (offx ^ (uint32_t)(ox & 1));
      const uint32_t s0 = cidx[idx] + 3u * qn * Mqp;
      v1[idx].x = FAR; v1[idx].y = FAR; v2[idx] = v1[idx]; v3[idx] = v1[idx];
      if (cj[idx] > 1u) v1[idx] = posb[s0 + Mqp];
      if (idx == 4 || NF == 4) {
        if (cj[idx] > 2u) v2[idx] = posb[s0 + 2u * Mqp];
        if (cj[idx] > 3u) v3[idx] = posb[s0 + 3u * Mqp];
      } else if (cj[idx] > (uint32_t)NF) {
        big |= 1u << idx;
      }
      if (cj[idx] == 0u) { v0[idx].x = FAR; v0[idx].y = FAR; }
    }
    if (NS > 0) {
#pragma unroll
      for (int q = NS / 4; q < NS / 2; ++q) displacement2((uint32_t)q, ddx[2 * q], ddy[2 * q], ddx[2 * q + 1], ddy[2 * q + 1]);
    }

    // ---- own cell (Alg. 2 line 8, L186), negated, as pairs (slot 0,1) and (slot 2,3) ----
    Pair nox[2], noy[2];
    nox[0] = R::pair(-v0[4].x, -v1[4].x); nox[1] = R::pair(-v2[4].x, -v3[4].x);
    noy[0] = R::pair(-v0[4].y, -v1[4].y); noy[1] = R::pair(-v2[4].y, -v3[4].y);

    // ---- neighbours, translated into this cell's frame (s = (ox wx, oy wy), L154, L196), negated:
    //      -(l_j + s) = fma(l_j, -1, -s), one rn operation ----
    Pair nqx[NPN], nqy[NPN];
#pragma unroll
    for (int idx = 0; idx < 9; ++idx) {
      if (idx == 4) continue;
      const int e = idx < 4 ? idx : idx - 1;
      const int ox = idx % 3 - 1, oy = idx / 3 - 1;
      const P nsx = ox < 0 ? wx : ox > 0 ? -wx : (P)0;
      const P nsy = oy < 0 ? wy : oy > 0 ? -wy : (P)0;
      nqx[e * (NF / 2)] = R::pfma(R::pair(v0[idx].x, v1[idx].x), MINUS1, R::pair(nsx, nsx));
      nqy[e * (NF / 2)] = R::pfma(R::pair(v0[idx].y, v1[idx].y), MINUS1, R::pair(nsy, nsy));
      if (NF == 4) {
        nqx[e * (NF / 2) + NF / 2 - 1] = R::pfma(R::pair(v2[idx].x, v3[idx].x), MINUS1, R::pair(nsx, nsx));
        nqy[e * (NF / 2) + NF / 2 - 1] = R::pfma(R::pair(v2[idx].y, v3[idx].y), MINUS1, R::pair(nsy, nsy));
      }
    }

    // ---- shuffle (Alg. 2 line 9, L187), kept as a visiting permutation packed in nibbles ----
    uint32_t perm = 0x3210u;
#pragma unroll
    for (int step = 0; step < NMAX - 1; ++step) {
      if ((uint32_t)step + 1u < n) {
        const uint32_t i = n - 1u - (uint32_t)step;
        const uint32_t j = bounded(S[step], i + 1u);
        const uint32_t a = (perm >> (4u * i)) & 15u, b = (perm >> (4u * j)) & 15u;
        const uint32_t x = a ^ b;
        perm ^= (x << (4u * i)) ^ (x << (4u * j));
      }
    }

    // ---- n_s trial moves (Alg. 2 lines 11-32, L189-230) ----
    uint32_t amask = 0, vi = 0;
    auto trial_move = [&](const uint32_t s, const P dx, const P dy) {
      const uint32_t k = (perm >> (4u * vi)) & 3u;               // p <- particles[s mod n]  (L75)
      vi = (vi + 1u == nv) ? 0u : vi + 1u;                       // lines 28-32 (L224-230)
      const P nlx = k == 0 ? nox[0].x : k == 1 ? nox[0].y : k == 2 ? nox[1].x : nox[1].y;
      const P nly = k == 0 ? noy[0].x : k == 1 ? noy[0].y : k == 2 ? noy[1].x : noy[1].y;
      const P Mx = R::sub(dx, nlx);                              // D_move = l + displacement
      const P My = R::sub(dy, nly);
      const bool inside = (Mx > (P)0) && (Mx <= wx) && (My > (P)0) && (My <= wy);   // (0, w]  (A3)
      const Pair MMx = R::pair(Mx, Mx), MMy = R::pair(My, My);
      bool ov = false;
      // the other disks of the own cell (line 17 skips i = j, L201); s = 0 so q = l_j
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const Pair Dx = R::padd(MMx, nox[h]), Dy = R::padd(MMy, noy[h]);
        const Pair r2 = R::pfma(Dx, Dx, R::pmul(Dy, Dy));
        ov |= (r2.x < sigma2) && ((uint32_t)(2 * h) != k);
        ov |= (r2.y < sigma2) && ((uint32_t)(2 * h + 1) != k);
      }
      // neighbour disks held in registers: |D_move - (D + s)|^2 < sigma^2 (line 19, L204)
#pragma unroll
      for (int e = 0; e < NPN; ++e) {
        const Pair Dx = R::padd(MMx, nqx[e]), Dy = R::padd(MMy, nqy[e]);
        const Pair r2 = R::pfma(Dx, Dx, R::pmul(Dy, Dy));
        ov |= (r2.x < sigma2) || (r2.y < sigma2);
      }
      if (NF < NMAX && big != 0 && inside && !ov) {              // rare: neighbours with more than NF disks
#pragma unroll 1
        for (int idx = 0; idx < 9; ++idx) {
          if (!((big >> idx) & 1u)) continue;
          const int ox = idx % 3 - 1, oy = idx / 3 - 1;
          const uint32_t qn = ((offy ^ (uint32_t)(oy & 1)) << 1) | (offx ^ (uint32_t)(ox & 1));
          const uint32_t cn = (oy < 0 ? rowd : oy > 0 ? rowu : rowa) + (ox < 0 ? xl : ox > 0 ? xr : xa);
          const uint32_t nj = cntb[qn * Mqp + cn];
          const P sx = ox < 0 ? -wx : ox > 0 ? wx : (P)0;
          const P sy = oy < 0 ? -wy : oy > 0 ? wy : (P)0;
          for (uint32_t i = NF; i < nj; ++i) {
            const P2 v = posb[(qn * NMAX + i) * Mqp + cn];
            const P Dx = R::sub(Mx, R::add(v.x, sx)), Dy = R::sub(My, R::add(v.y, sy));
            const P r2 = R::fma(Dx, Dx, R::mul(Dy, Dy));
            ov |= r2 < sigma2;
          }
        }
      }
      if (!inside) {
        ++n_rb;                                                  // leaves the cell: rejected (L79, L118)
      } else if (ov) {
        ++n_ro;
      } else {                                                   // lines 24-27 (L215-222)
        ++n_acc;
        amask |= 1u << (s & 31u);
        const P nMx = -Mx, nMy = -My;
        if (k == 0) { nox[0].x = nMx; noy[0].x = nMy; }
        if (k == 1) { nox[0].y = nMx; noy[0].y = nMy; }
        if (k == 2) { nox[1].x = nMx; noy[1].x = nMy; }
        if (k == 3) { nox[1].y = nMx; noy[1].y = nMy; }
      }
    };
    if (NS > 0) {
#pragma unroll
      for (int s = 0; s < NS; ++s) trial_move((uint32_t)s, ddx[s], ddy[s]);
    } else {
      for (uint32_t s = 0; s < p.n_s; s += 2) {
        displacement2(s >> 1, ddx[0], ddy[0], ddx[1], ddy[1]);
        trial_move(s, ddx[0], ddy[0]);
        if (s + 1 < p.n_s) trial_move(s + 1, ddx[1], ddy[1]);
      }
    }

    // ---- write back (line 34, L234) ----
    if (amask != 0) {
      const P vx[NMAX] = {nox[0].x, nox[0].y, nox[1].x, nox[1].y};
      const P vy[NMAX] = {noy[0].x, noy[0].y, noy[1].x, noy[1].y};
#pragma unroll
      for (int i = 0; i < NMAX; ++i)
        if ((uint32_t)i < n) { P2 v; v.x = -vx[i]; v.y = -vy[i]; posb[(Q * NMAX + i) * Mqp + ci] = v; }
    }
    if (DEBUG && valid) {
      p.mask[cell] = amask;
      if (n > 0u) atomicAdd(&p.ctl->digest, mix64(mix64(t) ^ (((unsigned long long)cell << 32) | amask)));
    }
  }
  if (n == 0u) n_rb = 0u;        // a sentinel never passes the in-cell test; empty cells attempt nothing (A10)

  // ---- counters: warp reduce, then three fire-and-forget 64-bit reductions per warp into one of CTR_SLOTS
  //      counter rows (spread so that same-address atomics do not serialise); no block barrier ----
  n_acc = __reduce_add_sync(0xFFFFFFFFu, n_acc);
  n_rb = __reduce_add_sync(0xFFFFFFFFu, n_rb);
  n_ro = __reduce_add_sync(0xFFFFFFFFu, n_ro);
  if ((threadIdx.x & 31) == 0) {
    unsigned long long* row = p.ctl->counters[(blockIdx.x * (SUB_THREADS / 32) + (threadIdx.x >> 5)) % CTR_SLOTS];
    if (n_acc) atomicAdd(&row[0], (unsigned long long)n_acc);
    if (n_rb) atomicAdd(&row[1], (unsigned long long)n_rb);
    if (n_ro) atomicAdd(&row[2], (unsigned long long)n_ro);
  }
}

// ---------------------------------------------------------------------------------------------------------
// Cell shift (Algorithm 4, pull form).  One thread per NEW cell (L350): its own old disks that stay, in slot
// order, then the disks of the one old neighbour in direction f that left it.  l' = rn(l - f*delta) is the
// same single operation on both sides, and the +-w translation of an entrant is a separate operation after
// the test (L352), so no disk is lost or duplicated.  Writes the other buffer (L350).  The last block to
// finish flips the buffer, advances the sweep index, moves the grid origin and draws the next sweep's set
// order and shift, so a sweep needs no host involvement.
// ovr: 0 = use Ctl's draws and advance the sweep; 1 = test hook (explicit dir/delta, sweep index unchanged).
// ---------------------------------------------------------------------------------------------------------
// one new cell; ALONG_X and POSITIVE are uniform across the grid, so the caller branches once
template <typename P, bool ALONG_X, bool POSITIVE>
__device__ __forceinline__ void shift_cell(const Params& p, Ctl* ctl, const uint32_t cur, const uint32_t Q,
                                           const uint32_t ci, const P delta) {
  using R = Real<P>;
  using P2 = typename R::T2;
  const uint32_t nxt = cur ^ 1u, Mqp = p.Mqp;
  const uint8_t* __restrict__ cntc = p.cnt[cur];
  const P2* __restrict__ posc = reinterpret_cast<const P2*>(p.pos[cur]);
  const uint32_t* __restrict__ idsc = p.ids[cur];
  P2* __restrict__ posn = reinterpret_cast<P2*>(p.pos[nxt]);
  uint32_t* __restrict__ idsn = p.ids[nxt];
  const P w = ALONG_X ? R::wx(p) : R::wy(p);
  const P step = POSITIVE ? -delta : delta;     // l' = l - f*delta   (L303)
  const P back = POSITIVE ? w : -w;             // entrant translation (L332)
  const uint32_t offx = Q & 1u, offy = Q >> 1;
  // the old neighbour in direction f (lines 15-16, L314-317)
  uint32_t qn, cn;
  if (ALONG_X) {
    const uint32_t ya = div_hx(p, ci), xa = ci - ya * p.hx;
    qn = Q ^ 1u;
    const uint32_t xn = POSITIVE ? (offx ? (xa + 1 == p.hx ? 0 : xa + 1) : xa)
                                 : (offx ? xa : (xa == 0 ? p.hx - 1 : xa - 1));
    cn = ci - xa + xn;
  } else {
    qn = Q ^ 2u;
    // one row up or down in the other colour: +-hx with wrap over the Mq = hx*hy cells of the plane
    if (POSITIVE) cn = offy ? (ci + p.hx >= p.Mq ? ci + p.hx - p.Mq : ci + p.hx) : ci;
    else          cn = offy ? ci : (ci < p.hx ? ci + p.Mq - p.hx : ci - p.hx);
  }
  const uint32_t own0 = Q * NMAX * Mqp + ci, nb0 = qn * NMAX * Mqp + cn;
  const uint32_t n0 = cntc[Q * Mqp + ci], n1 = cntc[qn * Mqp + cn];
  uint32_t nn = 0;
  // lines 7-14 (L299-312): own disks that stay, in slot order
#pragma unroll
  for (int i = 0; i < NMAX; ++i) {
    if ((uint32_t)i < n0) {
      P2 v = posc[own0 + i * Mqp];
      const uint32_t id = idsc[own0 + i * Mqp];
      const P a = R::add(ALONG_X ? v.x : v.y, step);
      if (a > (P)0 && a <= w) {
        if (ALONG_X) v.x = a; else v.y = a;
        posn[own0 + nn * Mqp] = v;
        idsn[own0 + nn * Mqp] = id;
        ++nn;
      }
    }
  }
  // lines 17-27 (L319-339): disks of the neighbour that left it enter here
#pragma unroll
  for (int i = 0; i < NMAX; ++i) {
    if ((uint32_t)i < n1) {
      P2 v = posc[nb0 + i * Mqp];
      const P a = R::add(ALONG_X ? v.x : v.y, step);
      if (!(a > (P)0 && a <= w)) {              // else: stays in the neighbour (L326-328)
        const P b = R::add(a, back);            // L332: a separate operation after the test (L352)
        if (nn < (uint32_t)NMAX) {
          if (ALONG_X) v.x = b; else v.y = b;
          posn[own0 + nn * Mqp] = v;
          idsn[own0 + nn * Mqp] = idsc[nb0 + i * Mqp];
        }
        ++nn;
      }
    }
  }
  if (nn > (uint32_t)NMAX) { atomicOr(&ctl->err, ERRBIT_OVERFLOW); nn = NMAX; }
  p.cnt[nxt][Q * Mqp + ci] = (uint8_t)nn;        // L280, L342
}

template <typename P>
__global__ void __launch_bounds__(SHIFT_THREADS)
k_shift(const __grid_constant__ Params p, const uint32_t ovr, const uint32_t ovr_dir, const double ovr_delta) {
  using R = Real<P>;
  Ctl* ctl = p.ctl;
  const uint32_t cur = ctl->cur, nxt = cur ^ 1u;
  const uint32_t dir = ovr ? ovr_dir : ctl->dir;
  const bool along_x = dir < 2, positive = (dir & 1u) == 0;
  const P w = along_x ? R::wx(p) : R::wy(p);
  // Alg. 1 line 15 (L90): delta = uniform(0, w/2) = rn(rn(0.5 w) * u01)
  const P delta = ovr ? (P)ovr_delta : R::mul(R::mul((P)0.5, w), R::unit(ctl->dist_word));
  const unsigned long long t = ctl->t;

  const uint32_t Q = blockIdx.y;
  const uint32_t ci = blockIdx.x * SHIFT_THREADS + threadIdx.x;
  if (ci < p.Mq) {
    if (along_x) {
      if (positive) shift_cell<P, true, true>(p, ctl, cur, Q, ci, delta);
      else          shift_cell<P, true, false>(p, ctl, cur, Q, ci, delta);
    } else {
      if (positive) shift_cell<P, false, true>(p, ctl, cur, Q, ci, delta);
      else          shift_cell<P, false, false>(p, ctl, cur, Q, ci, delta);
    }
  }

  // ---- last block done: advance the control block ----
  __shared__ uint32_t last;
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    const uint32_t total = gridDim.x * gridDim.y;
    last = (atomicAdd(&ctl->ticket, 1u) == total - 1u) ? 1u : 0u;
  }
  __syncthreads();
  if (last && threadIdx.x == 0) {
    ctl->ticket = 0;
    ctl->cur = nxt;
    const double L = along_x ? p.Lx_eff : p.Ly_eff;
    double o = ctl->origin[along_x ? 0 : 1];
    o = __dadd_rn(o, positive ? (double)delta : -(double)delta);
    if (o >= L) o = __dsub_rn(o, L);
    if (o < 0.0) o = __dadd_rn(o, L);
    ctl->origin[along_x ? 0 : 1] = o;
    if (!ovr) {
      ctl->t = t + 1ull;
      draw_sweep(p, t + 1ull, ctl);
    }
  }
}

}  // namespace mpmc
