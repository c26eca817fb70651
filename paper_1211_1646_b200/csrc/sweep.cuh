// sweep.cuh — the two hot kernels: the active-cell sub-sweep (Algorithm 2) and the cell
// shift / re-bin (Algorithm 4), re-designed for sm_100a.  See DESIGN.md "Kernels".
#pragma once
#include "common.cuh"

namespace mpmc {

constexpr int SUB_THREADS = 128;
constexpr int SHIFT_THREADS = 256;

// ---------------------------------------------------------------------------------------------------------
// Sub-sweep kernel.  One thread per cell of the active checkerboard set (the paper's mapping, L158/L260),
// over the dense colour plane so that a warp's 32 cells are contiguous.
//
//  * the cell's own <= 4 disks and the first NF disks of each of the 8 neighbour cells are loaded ONCE into
//    registers (neighbours already translated into the active cell's frame, q = l_j + s, L154/L196) and
//    reused by all n_s moves; empty entries hold a far-away sentinel so the overlap loop has a fixed trip
//    count and no divergence (the paper's (-10,-10) trick, L295/L346);
//  * NF = 2 covers every neighbour at w ~ sigma except a rare few (occupancy 0/1/2); neighbours with more
//    than NF disks set a bit in `big` and their remaining slots are re-read from L1/L2 inside the move loop;
//    NF = 4 is the instantiation for the paper's own regime w ~ 1.4 sigma (L152);
//  * Philox4x32-10 keyed on (seed; cell, sweep, move) replaces the per-thread Saru stream (L180, L262);
//  * accept/reject is computed without early exit: all lanes run the same instruction stream.
// SETK: index into Ctl::order (0..3) or, for the test hook, 4 + explicit set.
// ---------------------------------------------------------------------------------------------------------
template <typename P, int NF, bool DEBUG>
__global__ void __launch_bounds__(SUB_THREADS)
k_sub_sweep(const __grid_constant__ Params p, const uint32_t setk) {
  using R = Real<P>;
  using P2 = typename R::T2;
  const Ctl* __restrict__ ctl = p.ctl;
  const uint32_t Q = setk < 4 ? ctl->order[setk] : (setk & 3u);
  const unsigned long long t = ctl->t;
  const uint32_t cur = ctl->cur;
  const uint32_t offx = Q & 1u, offy = Q >> 1;
  const uint32_t ci = blockIdx.x * SUB_THREADS + threadIdx.x;
  const bool valid = ci < p.Mq;

  uint32_t n_acc = 0, n_rb = 0, n_ro = 0;
  uint32_t n = 0;
  if (valid) n = cnt_plane(p, cur, Q)[ci];

  if (n > 0) {
    const uint32_t ya = ci / p.hx, xa = ci - ya * p.hx;
    const uint32_t cell = (2u * ya + offy) * p.mx + (2u * xa + offx);   // canonical cell id y*mx + x
    const P wx = R::wx(p), wy = R::wy(p), sigma2 = R::sigma2(p), dmax = R::d(p);
    const P FAR = R::far_away();

    // ---- own cell (Alg. 2 line 8, L186) ----
    P ox_[NMAX], oy_[NMAX];
#pragma unroll
    for (int i = 0; i < NMAX; ++i) {
      ox_[i] = FAR; oy_[i] = FAR;
      if ((uint32_t)i < n) { const P2 v = pos_plane<P>(p, cur, Q, i)[ci]; ox_[i] = v.x; oy_[i] = v.y; }
    }

    // ---- neighbour cells: index in their colour plane, with periodic wrap ----
    const uint32_t xl = offx ? xa : (xa == 0 ? p.hx - 1 : xa - 1);        // plane column of cell x-1
    const uint32_t xr = offx ? (xa + 1 == p.hx ? 0 : xa + 1) : xa;        // ... of cell x+1
    const uint32_t yd = offy ? ya : (ya == 0 ? p.hy - 1 : ya - 1);
    const uint32_t yu = offy ? (ya + 1 == p.hy ? 0 : ya + 1) : ya;

    P qx[8 * NF], qy[8 * NF];
    uint32_t big = 0;          // bit e set: neighbour e holds more than NF disks
    uint32_t ncnt = 0;         // 4 bits per neighbour: its count
    {
      int e = 0;
#pragma unroll
      for (int oy = -1; oy <= 1; ++oy) {
#pragma unroll
        for (int ox = -1; ox <= 1; ++ox) {
          if (ox == 0 && oy == 0) continue;
          const uint32_t qn = ((offy ^ (uint32_t)(oy & 1)) << 1) | (offx ^ (uint32_t)(ox & 1));
          const uint32_t xn = ox < 0 ? xl : ox > 0 ? xr : xa;
          const uint32_t yn = oy < 0 ? yd : oy > 0 ? yu : ya;
          const uint32_t cn = yn * p.hx + xn;
          const uint32_t nj = cnt_plane(p, cur, qn)[cn];
          ncnt |= nj << (4 * e);
          if (nj > (uint32_t)NF) big |= 1u << e;
          const P sx = ox < 0 ? -wx : ox > 0 ? wx : (P)0;     // translation s (L154, L196)
          const P sy = oy < 0 ? -wy : oy > 0 ? wy : (P)0;
#pragma unroll
          for (int i = 0; i < NF; ++i) {
            P ax = FAR, ay = FAR;
            if ((uint32_t)i < nj) {
              const P2 v = pos_plane<P>(p, cur, qn, i)[cn];
              ax = R::add(v.x, sx);                              // q = rn(l_j + s)
              ay = R::add(v.y, sy);
            }
            qx[e * NF + i] = ax; qy[e * NF + i] = ay;
          }
          ++e;
        }
      }
    }

    // ---- shuffle (Alg. 2 line 9, L187), kept as a visiting permutation packed in nibbles ----
    uint32_t perm = 0x3210u;
    if (n >= 2) {
      uint32_t S[4];
      philox4x32_10(cell, (uint32_t)t, (uint32_t)(t >> 32), SLOT_SHUFFLE, p.seed_lo, p.seed_hi, S);
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
    }

    // ---- n_s trial moves (Alg. 2 lines 11-32, L189-230) ----
    uint32_t amask = 0, vi = 0;
    bool changed = false;
    for (uint32_t s = 0; s < p.n_s; ++s) {
      const uint32_t k = (perm >> (4u * vi)) & 3u;               // p <- particles[s mod n]  (L75)
      vi = (vi + 1u == n) ? 0u : vi + 1u;                        // lines 28-32 (L224-230)
      uint32_t Rw[4];
      philox4x32_10(cell, (uint32_t)t, (uint32_t)(t >> 32), s, p.seed_lo, p.seed_hi, Rw);
      const P lx = k == 0 ? ox_[0] : k == 1 ? ox_[1] : k == 2 ? ox_[2] : ox_[3];
      const P ly = k == 0 ? oy_[0] : k == 1 ? oy_[1] : k == 2 ? oy_[2] : oy_[3];
      const P Mx = R::add(lx, R::mul(dmax, R::sym(Rw[0])));      // line 12 (L190); square proposal (A2)
      const P My = R::add(ly, R::mul(dmax, R::sym(Rw[1])));
      const bool inside = (Mx > (P)0) && (Mx <= wx) && (My > (P)0) && (My <= wy);   // (0, w]  (A3)
      bool ov = false;
      // the other disks of the own cell (line 17 skips i = j, L201); s = 0 so q = l_j
#pragma unroll
      for (int j = 0; j < NMAX; ++j) {
        const P Dx = R::sub(Mx, ox_[j]), Dy = R::sub(My, oy_[j]);
        const P r2 = R::fma(Dx, Dx, R::mul(Dy, Dy));
        ov |= (r2 < sigma2) && ((uint32_t)j != k);
      }
      // neighbour disks held in registers
#pragma unroll
      for (int e = 0; e < 8 * NF; ++e) {
        const P Dx = R::sub(Mx, qx[e]), Dy = R::sub(My, qy[e]);
        const P r2 = R::fma(Dx, Dx, R::mul(Dy, Dy));             // |D_move - (D + s)|^2 < sigma^2 (line 19, L204)
        ov |= r2 < sigma2;
      }
      if (NF < NMAX && big != 0 && inside && !ov) {              // rare: neighbours with more than NF disks
        int e = 0;
        for (int oy = -1; oy <= 1; ++oy)
          for (int ox = -1; ox <= 1; ++ox) {
            if (ox == 0 && oy == 0) continue;
            if ((big >> e) & 1u) {
              const uint32_t qn = ((offy ^ (uint32_t)(oy & 1)) << 1) | (offx ^ (uint32_t)(ox & 1));
              const uint32_t xn = ox < 0 ? xl : ox > 0 ? xr : xa;
              const uint32_t yn = oy < 0 ? yd : oy > 0 ? yu : ya;
              const uint32_t cn = yn * p.hx + xn;
              const uint32_t nj = (ncnt >> (4 * e)) & 15u;
              const P sx = ox < 0 ? -wx : ox > 0 ? wx : (P)0;
              const P sy = oy < 0 ? -wy : oy > 0 ? wy : (P)0;
              for (uint32_t i = NF; i < nj; ++i) {
                const P2 v = pos_plane<P>(p, cur, qn, i)[cn];
                const P Dx = R::sub(Mx, R::add(v.x, sx)), Dy = R::sub(My, R::add(v.y, sy));
                const P r2 = R::fma(Dx, Dx, R::mul(Dy, Dy));
                ov |= r2 < sigma2;
              }
            }
            ++e;
          }
      }
      if (!inside) {
        ++n_rb;                                                  // leaves the cell: rejected (L79, L118)
      } else if (ov) {
        ++n_ro;
      } else {                                                   // lines 24-27 (L215-222)
        ++n_acc;
        amask |= 1u << (s & 31u);
        changed = true;
#pragma unroll
        for (int j = 0; j < NMAX; ++j)
          if ((uint32_t)j == k) { ox_[j] = Mx; oy_[j] = My; }
      }
    }

    // ---- write back (line 34, L234) ----
    if (changed) {
#pragma unroll
      for (int i = 0; i < NMAX; ++i)
        if ((uint32_t)i < n) { P2 v; v.x = ox_[i]; v.y = oy_[i]; pos_plane<P>(p, cur, Q, i)[ci] = v; }
    }
    if (DEBUG) {
      p.mask[cell] = amask;
      atomicAdd(&p.ctl->digest, mix64(mix64(t) ^ (((unsigned long long)cell << 32) | amask)));
    }
  } else if (DEBUG && valid) {
    const uint32_t ya = ci / p.hx, xa = ci - ya * p.hx;
    p.mask[(2u * ya + offy) * p.mx + (2u * xa + offx)] = 0u;
  }

  // ---- counters: warp reduce, one shared atomic per warp, three global atomics per block ----
  __shared__ uint32_t sh[3];
  if (threadIdx.x < 3) sh[threadIdx.x] = 0;
  __syncthreads();
  n_acc = __reduce_add_sync(0xFFFFFFFFu, n_acc);
  n_rb = __reduce_add_sync(0xFFFFFFFFu, n_rb);
  n_ro = __reduce_add_sync(0xFFFFFFFFu, n_ro);
  if ((threadIdx.x & 31) == 0) {
    if (n_acc) atomicAdd(&sh[0], n_acc);
    if (n_rb) atomicAdd(&sh[1], n_rb);
    if (n_ro) atomicAdd(&sh[2], n_ro);
  }
  __syncthreads();
  if (threadIdx.x < 3 && sh[threadIdx.x]) atomicAdd(&p.ctl->counters[threadIdx.x], (unsigned long long)sh[threadIdx.x]);
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
template <typename P>
__global__ void __launch_bounds__(SHIFT_THREADS)
k_shift(const __grid_constant__ Params p, const uint32_t ovr, const uint32_t ovr_dir, const double ovr_delta) {
  using R = Real<P>;
  using P2 = typename R::T2;
  Ctl* ctl = p.ctl;
  const uint32_t cur = ctl->cur, nxt = cur ^ 1u;
  const uint32_t dir = ovr ? ovr_dir : ctl->dir;
  const bool along_x = dir < 2, positive = (dir & 1u) == 0;
  const P w = along_x ? R::wx(p) : R::wy(p);
  // Alg. 1 line 15 (L90): delta = uniform(0, w/2) = rn(rn(0.5 w) * u01)
  const P delta = ovr ? (P)ovr_delta : R::mul(R::mul((P)0.5, w), R::unit(ctl->dist_word));
  const P step = positive ? -delta : delta;     // l' = l - f*delta   (L303)
  const P back = positive ? w : -w;             // entrant translation (L332)
  const unsigned long long t = ctl->t;

  const uint32_t Q = blockIdx.y;
  const uint32_t ci = blockIdx.x * SHIFT_THREADS + threadIdx.x;
  if (ci < p.Mq) {
    const uint32_t offx = Q & 1u, offy = Q >> 1;
    const uint32_t ya = ci / p.hx, xa = ci - ya * p.hx;
    uint32_t nn = 0;
    // lines 7-14 (L299-312): own disks that stay
    const uint32_t n0 = cnt_plane(p, cur, Q)[ci];
    for (uint32_t i = 0; i < n0; ++i) {
      P2 v = pos_plane<P>(p, cur, Q, i)[ci];
      P a = R::add(along_x ? v.x : v.y, step);
      if (a > (P)0 && a <= w) {
        if (along_x) v.x = a; else v.y = a;
        pos_plane<P>(p, nxt, Q, nn)[ci] = v;
        ids_plane(p, nxt, Q, nn)[ci] = ids_plane(p, cur, Q, i)[ci];
        ++nn;
      }
    }
    // lines 15-27 (L314-339): the neighbour in direction f
    uint32_t qn, cn;
    if (along_x) {
      qn = Q ^ 1u;
      const uint32_t xn = positive ? (offx ? (xa + 1 == p.hx ? 0 : xa + 1) : xa)
                                   : (offx ? xa : (xa == 0 ? p.hx - 1 : xa - 1));
      cn = ya * p.hx + xn;
    } else {
      qn = Q ^ 2u;
      const uint32_t yn = positive ? (offy ? (ya + 1 == p.hy ? 0 : ya + 1) : ya)
                                   : (offy ? ya : (ya == 0 ? p.hy - 1 : ya - 1));
      cn = yn * p.hx + xa;
    }
    const uint32_t n1 = cnt_plane(p, cur, qn)[cn];
    for (uint32_t i = 0; i < n1; ++i) {
      P2 v = pos_plane<P>(p, cur, qn, i)[cn];
      P a = R::add(along_x ? v.x : v.y, step);
      if (a > (P)0 && a <= w) continue;         // stays in the neighbour (L326-328)
      a = R::add(a, back);                      // L332
      if (nn < (uint32_t)NMAX) {
        if (along_x) v.x = a; else v.y = a;
        pos_plane<P>(p, nxt, Q, nn)[ci] = v;
        ids_plane(p, nxt, Q, nn)[ci] = ids_plane(p, cur, qn, i)[cn];
      }
      ++nn;
    }
    if (nn > (uint32_t)NMAX) { atomicOr(&ctl->err, ERRBIT_OVERFLOW); nn = NMAX; }
    cnt_plane(p, nxt, Q)[ci] = (uint8_t)nn;      // L280, L342
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
