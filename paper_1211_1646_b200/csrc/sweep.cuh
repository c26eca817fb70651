// sweep.cuh — the general path: the cell update (Algorithm 2) in two register-resident forms and
// the cell shift / re-bin (Algorithm 4) on the colour planes in global memory, driven by the persistent
// cooperative kernel k_sweeps (any cell width up to sqrt(2) sigma, any n_s).  The fused tile kernel for w ~ sigma
// (tile.cuh) reuses shift_pair, the tallies and the visiting permutation from here.  See DESIGN.md "Kernels".
#pragma once
#include "common.cuh"

namespace mpmc {

constexpr int SUB_THREADS = 128;
constexpr int SUB_MINB = 1;                  // minimum resident blocks per SM asked of ptxas (register cap)
constexpr int FAST_MINB = 6;
constexpr int SHIFT_THREADS = 256;

// ---------------------------------------------------------------------------------------------------------
// Where an active cell and its 3x3 neighbourhood live in the colour planes (periodic wrap).
// ---------------------------------------------------------------------------------------------------------
struct Where {
  uint32_t Q, offx, offy, ci, cell;
  uint32_t xl, xa, xr, rowd, rowa, rowu;
  bool valid;
};
__device__ __forceinline__ Where locate_active(const Params& p, const uint32_t Q, const uint32_t ci_raw, const bool valid) {
  Where w;
  w.Q = Q; w.offx = Q & 1u; w.offy = Q >> 1;
  w.valid = valid;
  w.ci = w.valid ? ci_raw : p.Mq - 1u;             // clamped: every lane may prefetch
  const uint32_t ya = div_hx(p, w.ci);
  w.xa = w.ci - ya * p.hx;
  w.cell = (2u * ya + w.offy) * p.mx + (2u * w.xa + w.offx);        // canonical cell id y*mx + x
  w.xl = w.offx ? w.xa : (w.xa == 0 ? p.hx - 1 : w.xa - 1);          // plane column of cell x-1
  w.xr = w.offx ? (w.xa + 1 == p.hx ? 0 : w.xa + 1) : w.xa;          // ... of cell x+1
  const uint32_t yd = w.offy ? ya : (ya == 0 ? p.hy - 1 : ya - 1);
  const uint32_t yu = w.offy ? (ya + 1 == p.hy ? 0 : ya + 1) : ya;
  w.rowd = yd * p.hx; w.rowa = ya * p.hx; w.rowu = yu * p.hx;
  return w;
}
// colour and in-plane index of the neighbour at offset (ox, oy), ox, oy in {-1, 0, 1}
__device__ __forceinline__ void neighbour(const Where& w, int ox, int oy, uint32_t& qn, uint32_t& cn) {
  qn = ((w.offy ^ (uint32_t)(oy & 1)) << 1) | (w.offx ^ (uint32_t)(ox & 1));
  cn = (oy < 0 ? w.rowd : oy > 0 ? w.rowu : w.rowa) + (ox < 0 ? w.xl : ox > 0 ? w.xr : w.xa);
}

// Fisher-Yates of the cell's n disks (Alg. 2 line 9, L187) as a visiting permutation packed in nibbles
__device__ __forceinline__ uint32_t visiting_permutation(const Params& p, const uint32_t n, const uint32_t (&S)[4]) {
  uint32_t perm = 0x3210u;
  if (p.flags & FLAG_NO_PARTICLE_SHUFFLE) return perm;        // ablation (Table 1): slot order
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
  return perm;
}

// ---------------------------------------------------------------------------------------------------------
// Generic cell update: Algorithm 2 line by line on the slots in global memory, any occupancy up to n_max.
// Used by update_cell_fast for the rare cells whose 3x3 neighbourhood holds a cell with more than 2 disks.
// Deliberately compact (rolled loops, scalar arithmetic): it runs for a handful of lanes.
// ---------------------------------------------------------------------------------------------------------
template <typename P>
__device__ __forceinline__ void cell_update_generic(const Params& p, const Where& w, const uint8_t* cntb, P* posb,
                                                    const uint32_t n, const uint32_t n_s, const uint32_t t_lo,
                                                    const uint32_t t_hi, uint32_t& n_acc, uint32_t& n_rb,
                                                    uint32_t& n_ro, uint32_t& amask) {
  using R = Real<P>;
  const uint32_t Mqp = p.Mqp;
  const P wx = R::wx(p), wy = R::wy(p), sigma2 = R::sigma2(p), dmax = R::d(p);
  uint32_t perm = 0x3210u;
  if (n >= 2u) {
    uint32_t S[4];
    philox4x32_10(w.cell, t_lo, t_hi, SLOT_SHUFFLE, p.seed_lo, p.seed_hi, S);
    perm = visiting_permutation(p, n, S);
  }
  const uint32_t own = 2u * w.Q * Mqp + w.ci;           // half-0 index of the own cell
  uint32_t vi = 0;
  uint32_t Rw[4] = {0, 0, 0, 0};
#pragma unroll 1
  for (uint32_t s = 0; s < n_s; ++s) {
    if ((s & 1u) == 0u) philox4x32_10(w.cell, t_lo, t_hi, s >> 1, p.seed_lo, p.seed_hi, Rw);
    const uint32_t k = (perm >> (4u * vi)) & 3u;                 // p <- particles[s mod n]  (L75)
    vi = (vi + 1u == n) ? 0u : vi + 1u;                          // lines 28-32 (L224-230)
    const uint32_t r0 = (s & 1u) ? Rw[2] : Rw[0], r1 = (s & 1u) ? Rw[3] : Rw[1];
    P* slot_k = posb + ((size_t)(own + (k >> 1) * Mqp) * 4 + (k & 1u));
    const P Mx = R::add(slot_k[0], R::mul(dmax, R::sym(r0)));    // D_move = l + displacement (line 12, L190)
    const P My = R::add(slot_k[2], R::mul(dmax, R::sym(r1)));
    if (!((Mx > (P)0) && (Mx <= wx) && (My > (P)0) && (My <= wy))) { ++n_rb; continue; }   // (0, w]  (A3; L79)
    bool ov = false;
#pragma unroll 1
    for (int idx = 0; idx < 9; ++idx) {
      const int ox = idx % 3 - 1, oy = idx / 3 - 1;
      uint32_t qn, cn;
      neighbour(w, ox, oy, qn, cn);
      const uint32_t nj = cntb[qn * Mqp + cn];
      const P sx = ox < 0 ? -wx : ox > 0 ? wx : (P)0;            // s = (ox wx, oy wy)  (L154, L196)
      const P sy = oy < 0 ? -wy : oy > 0 ? wy : (P)0;
      for (uint32_t j = 0; j < nj; ++j) {
        if (idx == 4 && j == k) continue;                        // line 17 (L201)
        const P* sj = posb + ((size_t)(2u * qn * Mqp + (j >> 1) * Mqp + cn) * 4 + (j & 1u));
        const P Dx = R::sub(Mx, R::add(sj[0], sx)), Dy = R::sub(My, R::add(sj[2], sy));
        ov |= R::fma(Dx, Dx, R::mul(Dy, Dy)) < sigma2;           // line 19 (L204), strict (A4)
      }
    }
    if (ov) { ++n_ro; }
    else { ++n_acc; amask |= 1u << (s & 31u); slot_k[0] = Mx; slot_k[2] = My; }   // lines 24-27 (L215-222)
  }
}

// Move counters of one thread, accumulated over a whole launch (many cells, many sweeps) and flushed once:
// warp reduce, then three fire-and-forget 64-bit reductions per warp into one of CTR_SLOTS counter rows.
struct Tally { uint32_t acc = 0, rb = 0, ro = 0; };
__device__ __forceinline__ void flush_tally(const Params& p, const Tally& tl) {
  const uint32_t n_acc = __reduce_add_sync(0xFFFFFFFFu, tl.acc);
  const uint32_t n_rb = __reduce_add_sync(0xFFFFFFFFu, tl.rb);
  const uint32_t n_ro = __reduce_add_sync(0xFFFFFFFFu, tl.ro);
  if ((threadIdx.x & 31) == 0) {
    unsigned long long* row = p.ctl->counters[(blockIdx.x * (blockDim.x / 32) + (threadIdx.x >> 5)) % CTR_SLOTS];
    if (n_acc) atomicAdd(&row[0], (unsigned long long)n_acc);
    if (n_rb) atomicAdd(&row[1], (unsigned long long)n_rb);
    if (n_ro) atomicAdd(&row[2], (unsigned long long)n_ro);
  }
}

// ---------------------------------------------------------------------------------------------------------
// Fast cell update for cell widths w ~ sigma (occupancy 0/1/2 per cell), one thread per cell of the active
// checkerboard set (the paper's mapping, L158/L260) over the dense colour plane in global memory, so a warp's 32 cells
// are contiguous.  (The tile kernel's tile_update_cell is the same arithmetic on shared memory.)
//
//  * each of the 3x3 cells is ONE load of its slot pair {x0, x1, y0, y1} (128 bit in fp32), issued up front and
//    unconditionally; empty slots hold the far-away sentinel (the paper's (-10,-10) trick, L295/L346), so the
//    two register pairs of a neighbour are, after one packed fma that translates them into this cell's frame and
//    negates them (-(l_j + s), s = (ox wx, oy wy), L154/L196), directly the operands of the packed fp32x2
//    overlap test (FADD2, FADD2, FMUL2, FFMA2: D = M + (-q), r^2 = fma(Dx, Dx, Dy*Dy)); every lane of a packed
//    instruction is one IEEE rn operation and -(a+b) = (-a)+(-b) exactly, so results are those of the scalar
//    formula.  No count-dependent select, no branch, no divergence: the verdict of a move is min r^2 < sigma^2;
//  * the two own disks are kept in VISITING order (A = the disk the next move acts on, B = the other one or the
//    sentinel): the shuffle (Alg. 2 line 9, L187) swaps them once up front, and after every move they swap iff
//    n = 2 (the s mod n cycling, L75, L224-230) — no dynamic slot index anywhere;
//  * Philox4x32-10 keyed on (seed; cell, sweep, block) replaces the per-thread Saru stream (L180, L262); the
//    NS/2 blocks depend on nothing loaded and are computed while the loads are in flight; d*u is evaluated as
//    (d 2^-24) * integer, the same real product, hence the same rounding;
//  * the rare cell with more than 2 disks in its 3x3 neighbourhood takes cell_update_generic (lane-divergent).
// ---------------------------------------------------------------------------------------------------------
template <typename P, int NS, bool DEBUG>
__device__ __forceinline__ void update_cell_fast(const Params& p, const uint32_t Q, const unsigned long long t,
                                                 const uint32_t cur, const uint32_t ci_raw, const bool valid,
                                                 Tally& tally) {
  using R = Real<P>;
  using Pair = typename R::Pair;
  static_assert(NS > 0 && NS % 2 == 0, "compile-time n_s must be even");
  const uint32_t t_lo = (uint32_t)t, t_hi = (uint32_t)(t >> 32);
  const Where w = locate_active(p, Q, ci_raw, valid);
  const uint8_t* cntb = p.cnt[cur];
  P* posb = reinterpret_cast<P*>(p.pos[cur]);
  const uint32_t Mqp = p.Mqp;

  // ---- all loads, independent and unconditional: count and slot pair 0 of the 3x3 cells (idx 4 = own) ----
  uint32_t cj[9];
  Half<P> h[9];
#pragma unroll
  for (int idx = 0; idx < 9; ++idx) {
    uint32_t qn, cn;
    neighbour(w, idx % 3 - 1, idx / 3 - 1, qn, cn);
    cj[idx] = ld_u8_early(cntb + (qn * Mqp + cn));
    h[idx] = ld_half_early(posb, 2u * qn * Mqp + cn);
  }

  // ---- arithmetic that needs no memory: the displacements of all NS moves (line 12, L190; A2, A9) ----
  P ddx[NS], ddy[NS];
#pragma unroll
  for (int q = 0; q < NS / 2; ++q) {
    uint32_t Rw[4];
    philox4x32_10(w.cell, t_lo, t_hi, (uint32_t)q, p.seed_lo, p.seed_hi, Rw);
    ddx[2 * q] = R::scaled_sym(p, Rw[0]); ddy[2 * q] = R::scaled_sym(p, Rw[1]);
    ddx[2 * q + 1] = R::scaled_sym(p, Rw[2]); ddy[2 * q + 1] = R::scaled_sym(p, Rw[3]);
  }

  uint32_t n_acc = 0, n_rb = 0, n_ro = 0, amask = 0;
  const uint32_t n = w.valid ? cj[4] : 0u;
  // largest count in the neighbourhood: above 2 the slot pair does not hold the whole cell
  uint32_t cmax = cj[0];
#pragma unroll
  for (int idx = 1; idx < 9; ++idx) cmax = max(cmax, cj[idx]);

  if (cmax > 2u) {
    if (n > 0u) cell_update_generic<P>(p, w, cntb, posb, n, (uint32_t)NS, t_lo, t_hi, n_acc, n_rb, n_ro, amask);
  } else {
    const P wx = R::wx(p), wy = R::wy(p), sigma2 = R::sigma2(p);
    const Pair MINUS1 = R::pair((P)-1, (P)-1);
    // ---- neighbours, translated into this cell's frame and negated: -(l_j + s) = fma(l_j, -1, -s) ----
    Pair nqx[8], nqy[8];
#pragma unroll
    for (int idx = 0; idx < 9; ++idx) {
      if (idx == 4) continue;
      const int e = idx < 4 ? idx : idx - 1;
      const int ox = idx % 3 - 1, oy = idx / 3 - 1;
      const P nsx = ox < 0 ? wx : ox > 0 ? -wx : (P)0;
      const P nsy = oy < 0 ? wy : oy > 0 ? -wy : (P)0;
      nqx[e] = R::pfma(h[idx].x, MINUS1, R::pair(nsx, nsx));
      nqy[e] = R::pfma(h[idx].y, MINUS1, R::pair(nsy, nsy));
    }
    // ---- own cell in visiting order (Alg. 2 lines 8-9, L186-187) ----
    P Ax = h[4].x.x, Ay = h[4].y.x, Bx = h[4].x.y, By = h[4].y.y;
    const bool two = n == 2u;
    bool flip = false;                   // true: A is slot 1
    if (two) {                           // n = 2: Fisher-Yates is one draw, j = bounded(S0, 2); j = 0 swaps
      uint32_t S[4];
      philox4x32_10(w.cell, t_lo, t_hi, SLOT_SHUFFLE, p.seed_lo, p.seed_hi, S);
      flip = bounded(S[0], 2u) == 0u && !(p.flags & FLAG_NO_PARTICLE_SHUFFLE);
    }
    if (flip) { P tx = Ax, ty = Ay; Ax = Bx; Ay = By; Bx = tx; By = ty; }

    // ---- NS trial moves (Alg. 2 lines 11-32, L189-230) ----
#pragma unroll
    for (int s = 0; s < NS; ++s) {
      const P Mx = R::add(Ax, ddx[s]), My = R::add(Ay, ddy[s]);              // D_move = l + displacement
      const bool inside = (Mx > (P)0) && (Mx <= wx) && (My > (P)0) && (My <= wy);   // (0, w]  (A3; L79, L118)
      const P Dbx = R::sub(Mx, Bx), Dby = R::sub(My, By);                    // the other own disk (s = 0)
      P rmin = R::fma(Dbx, Dbx, R::mul(Dby, Dby));
      const Pair MMx = R::pair(Mx, Mx), MMy = R::pair(My, My);
#pragma unroll
      for (int e = 0; e < 8; ++e) {                                          // |D_move - (D + s)|^2  (line 19, L204)
        const Pair Dx = R::padd(MMx, nqx[e]), Dy = R::padd(MMy, nqy[e]);
        const Pair r2 = R::pfma(Dx, Dx, R::pmul(Dy, Dy));
        rmin = R::min3(rmin, r2.x, r2.y);
      }
      const bool ov = rmin < sigma2;                                         // strict (A4)
      const bool acc = inside && !ov;
      if (acc) { Ax = Mx; Ay = My; amask |= 1u << s; }                       // lines 24-27 (L215-222)
      n_rb += inside ? 0u : 1u;                                              // leaves the cell: rejected
      n_acc += acc ? 1u : 0u;
      if (two) { const P tx = Ax, ty = Ay; Ax = Bx; Ay = By; Bx = tx; By = ty; }   // s mod n cycling (L75)
    }
    // a sentinel never passes the in-cell test; empty cells (and the clamped lanes past the end) attempt nothing (A10)
    if (n == 0u) { n_rb = 0u; n_acc = 0u; amask = 0u; }
    else { n_ro = (uint32_t)NS - n_acc - n_rb; }
    // ---- write back (line 34, L234): the slot pair in slot order ----
    if (amask != 0u) {
      if (two && (NS & 1)) flip = !flip;
      Half<P> o;
      o.x = flip ? R::pair(Bx, Ax) : R::pair(Ax, Bx);
      o.y = flip ? R::pair(By, Ay) : R::pair(Ay, By);
      st_half(posb, 2u * Q * Mqp + w.ci, o);
    }
  }
  if (DEBUG && w.valid) {
    p.mask[w.cell] = amask;
    if (n > 0u) atomicAdd(&p.ctl->digest, mix64(mix64(t) ^ (((unsigned long long)w.cell << 32) | amask)));
  }
  tally.acc += n_acc; tally.rb += n_rb; tally.ro += n_ro;
}

// The moves of one cell with up to n_max = 4 disks (Algorithm 2 lines 9-32) on registers: h0 / h1 = slot pairs 0 / 1 of
// the 3x3 cells (idx 4 = own cell; empty slots = sentinel), n = the own count, cell = canonical cell id (Philox counter).
// Returns the own cell's slot pairs after the moves, the accept mask and the three tallies.  Shared by the general
// kernel (operands from global memory) and the 4-slot tile kernel (operands from shared memory).
template <typename P, int NS, bool DISC>
__device__ __forceinline__ void cell_moves_general(const Params& p, const Half<P> (&h0)[9], const Half<P> (&h1)[9],
                                                   const uint32_t n, const uint32_t cell, const uint32_t t_lo,
                                                   const uint32_t t_hi, Half<P>& o0, Half<P>& o1, uint32_t& amask,
                                                   uint32_t& n_acc, uint32_t& n_rb, uint32_t& n_ro) {
  using R = Real<P>;
  using Pair = typename R::Pair;
  static_assert(NS % 2 == 0, "compile-time n_s must be even");
  // ---- Philox words of the shuffle and of the displacements, while the loads are in flight ----
  constexpr int NSA = NS > 0 ? NS : 2;
  P ddx[NSA], ddy[NSA];
  auto displacement2 = [&](uint32_t q, int at) {       // block q serves moves 2q and 2q + 1 (reading A9)
    uint32_t Rw[4];
    philox4x32_10(cell, t_lo, t_hi, q, p.seed_lo, p.seed_hi, Rw);
    ddx[at] = R::scaled_sym(p, Rw[0]); ddy[at] = R::scaled_sym(p, Rw[1]);
    ddx[at + 1] = R::scaled_sym(p, Rw[2]); ddy[at + 1] = R::scaled_sym(p, Rw[3]);
  };
  // DISC: the paper's proposal, uniform in the disc of radius d (rng.inCircle(d), L190), by rejection from the square:
  // block (s | j << 16) serves the candidate pairs 2j (words 0, 1) and 2j + 1 (words 2, 3) of move s; the first pair
  // with fma(ux, ux, uy*uy) <= 1 is taken (reading A2)
  auto displacement_disc = [&](uint32_t s, int at) {
    // both pairs of the first block are evaluated without a branch (one of them is inside the disc 95 % of the time);
    // the rare lanes that need more go through further blocks in a structured loop
    uint32_t Rw[4];
    philox4x32_10(cell, t_lo, t_hi, s, p.seed_lo, p.seed_hi, Rw);
    const P ax = R::sym(Rw[0]), ay = R::sym(Rw[1]), bx = R::sym(Rw[2]), by = R::sym(Rw[3]);
    const bool oka = R::fma(ax, ax, R::mul(ay, ay)) <= (P)1, okb = R::fma(bx, bx, R::mul(by, by)) <= (P)1;
    P ux = oka ? ax : bx, uy = oka ? ay : by;
    bool found = oka || okb;
    uint32_t blk = 1;
    while (!found) {
      philox4x32_10(cell, t_lo, t_hi, s | (blk << 16), p.seed_lo, p.seed_hi, Rw);
      const P cx = R::sym(Rw[0]), cy = R::sym(Rw[1]), ex = R::sym(Rw[2]), ey = R::sym(Rw[3]);
      const bool okc = R::fma(cx, cx, R::mul(cy, cy)) <= (P)1, oke = R::fma(ex, ex, R::mul(ey, ey)) <= (P)1;
      ux = okc ? cx : ex; uy = okc ? cy : ey;
      found = okc || oke;
      ++blk;
    }
    ddx[at] = R::mul(R::d(p), ux); ddy[at] = R::mul(R::d(p), uy);
  };
  uint32_t S[4];
  philox4x32_10(cell, t_lo, t_hi, SLOT_SHUFFLE, p.seed_lo, p.seed_hi, S);
  if (NS > 0) {
    if (DISC) {
      if constexpr (NS == 4) {
        // The four moves' first blocks without a branch (one of a block's two candidate pairs is inside the disc 95 % of
        // the time), then ONE loop for whatever is still missing: a lane takes its first unserved move and that move's
        // next block.  Served move by move, a warp ran a nearly empty extra round for 80 % of its moves (some lane of 32
        // needs it); together the expected number of such rounds is ~1.4 per cell instead of ~3.3.  Same blocks, same
        // pairs, same order per move (reading A2): the same displacements.
        P ux[4], uy[4];
        uint32_t pend = 0u, nextblk = 0x01010101u;       // bit s: move s has no pair yet; byte s: its next block index j
#pragma unroll
        for (int s = 0; s < 4; ++s) {
          uint32_t Rw[4];
          philox4x32_10(cell, t_lo, t_hi, (uint32_t)s, p.seed_lo, p.seed_hi, Rw);
          const P ax = R::sym(Rw[0]), ay = R::sym(Rw[1]), bx = R::sym(Rw[2]), by = R::sym(Rw[3]);
          const bool oka = R::fma(ax, ax, R::mul(ay, ay)) <= (P)1, okb = R::fma(bx, bx, R::mul(by, by)) <= (P)1;
          ux[s] = oka ? ax : bx; uy[s] = oka ? ay : by;
          pend |= (oka || okb) ? 0u : 1u << s;
        }
        while (pend != 0u) {
          const uint32_t s = (uint32_t)__ffs((int)pend) - 1u, j = (nextblk >> (8u * s)) & 0xFFu;
          uint32_t Rw[4];
          philox4x32_10(cell, t_lo, t_hi, s | (j << 16), p.seed_lo, p.seed_hi, Rw);
          const P cx = R::sym(Rw[0]), cy = R::sym(Rw[1]), ex = R::sym(Rw[2]), ey = R::sym(Rw[3]);
          const bool okc = R::fma(cx, cx, R::mul(cy, cy)) <= (P)1, oke = R::fma(ex, ex, R::mul(ey, ey)) <= (P)1;
          const P vx = okc ? cx : ex, vy = okc ? cy : ey;
          if (okc || oke) {
            if (s == 0u) { ux[0] = vx; uy[0] = vy; }
            if (s == 1u) { ux[1] = vx; uy[1] = vy; }
            if (s == 2u) { ux[2] = vx; uy[2] = vy; }
            if (s == 3u) { ux[3] = vx; uy[3] = vy; }
            pend &= pend - 1u;
          }
          nextblk += 1u << (8u * s);
        }
#pragma unroll
        for (int s = 0; s < 4; ++s) { ddx[s] = R::mul(R::d(p), ux[s]); ddy[s] = R::mul(R::d(p), uy[s]); }
      } else {
#pragma unroll
        for (int s = 0; s < NS; ++s) displacement_disc((uint32_t)s, s);
      }
    } else {
#pragma unroll
      for (int q = 0; q < NS / 2; ++q) displacement2((uint32_t)q, 2 * q);
    }
  }

  n_acc = 0; n_rb = 0; n_ro = 0; amask = 0;
  const uint32_t nv = n > 0u ? n : 1u;                 // visiting modulus; an empty cell "visits" a sentinel
  const P wx = R::wx(p), wy = R::wy(p), sigma2 = R::sigma2(p);
  const P FAR = R::far_away();
  const Pair MINUS1 = R::pair((P)-1, (P)-1);

  // ---- own cell (Alg. 2 line 8, L186), negated, as pairs (slot 0,1) and (slot 2,3) ----
  Pair nox[2], noy[2];
  nox[0] = R::pair(-h0[4].x.x, -h0[4].x.y); nox[1] = R::pair(-h1[4].x.x, -h1[4].x.y);
  noy[0] = R::pair(-h0[4].y.x, -h0[4].y.y); noy[1] = R::pair(-h1[4].y.x, -h1[4].y.y);

  // ---- neighbours, translated into this cell's frame (s = (ox wx, oy wy), L154, L196), negated ----
  Pair nqx[16], nqy[16];
#pragma unroll
  for (int idx = 0; idx < 9; ++idx) {
    if (idx == 4) continue;
    const int e = idx < 4 ? idx : idx - 1;
    const int ox = idx % 3 - 1, oy = idx / 3 - 1;
    const P nsx = ox < 0 ? wx : ox > 0 ? -wx : (P)0;
    const P nsy = oy < 0 ? wy : oy > 0 ? -wy : (P)0;
    nqx[2 * e] = R::pfma(h0[idx].x, MINUS1, R::pair(nsx, nsx));
    nqy[2 * e] = R::pfma(h0[idx].y, MINUS1, R::pair(nsy, nsy));
    nqx[2 * e + 1] = R::pfma(h1[idx].x, MINUS1, R::pair(nsx, nsx));
    nqy[2 * e + 1] = R::pfma(h1[idx].y, MINUS1, R::pair(nsy, nsy));
  }

  const uint32_t perm = visiting_permutation(p, n, S);    // Alg. 2 line 9 (L187)

  // ---- n_s trial moves (Alg. 2 lines 11-32, L189-230) ----
  uint32_t vi = 0;
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
    for (int hh = 0; hh < 2; ++hh) {
      const Pair Dx = R::padd(MMx, nox[hh]), Dy = R::padd(MMy, noy[hh]);
      const Pair r2 = R::pfma(Dx, Dx, R::pmul(Dy, Dy));
      ov |= (r2.x < sigma2) && ((uint32_t)(2 * hh) != k);
      ov |= (r2.y < sigma2) && ((uint32_t)(2 * hh + 1) != k);
    }
    // neighbour disks: |D_move - (D + s)|^2 < sigma^2 (line 19, L204)
    P rmin = FAR;
#pragma unroll
    for (int e = 0; e < 16; ++e) {
      const Pair Dx = R::padd(MMx, nqx[e]), Dy = R::padd(MMy, nqy[e]);
      const Pair r2 = R::pfma(Dx, Dx, R::pmul(Dy, Dy));
      rmin = R::min3(rmin, r2.x, r2.y);
    }
    ov |= rmin < sigma2;
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
      if (DISC) { displacement_disc(s, 0); if (s + 1 < p.n_s) displacement_disc(s + 1, 1); }
      else displacement2(s >> 1, 0);
      trial_move(s, ddx[0], ddy[0]);
      if (s + 1 < p.n_s) trial_move(s + 1, ddx[1], ddy[1]);
    }
  }
  if (n == 0u) { n_rb = 0u; n_acc = 0u; n_ro = 0u; amask = 0u; }   // empty cells attempt nothing (A10)
  o0.x = R::pair(-nox[0].x, -nox[0].y); o0.y = R::pair(-noy[0].x, -noy[0].y);
  o1.x = R::pair(-nox[1].x, -nox[1].y); o1.y = R::pair(-noy[1].x, -noy[1].y);
}

// ---------------------------------------------------------------------------------------------------------
// General cell update: any occupancy up to n_max = 4 per cell — the paper's own regime, w up to
// sqrt(2) sigma (L152) — and any n_s.  Same mapping and arithmetic; all four slots of the 3x3 cells are kept
// in registers (own cell as two negated pairs, each neighbour as two translated, negated pairs; slot pair 1 is
// loaded only where n > 2), and the disk a move acts on is chosen with select chains from the visiting
// permutation.  NS > 0 fixes n_s at compile time (Philox blocks issued up front, move loop unrolled); NS = 0 is
// the run-time loop.
// ---------------------------------------------------------------------------------------------------------
template <typename P, int NS, bool DEBUG, bool DISC>
__device__ __forceinline__ void update_cell_general(const Params& p, const uint32_t Q, const unsigned long long t,
                                                    const uint32_t cur, const uint32_t ci_raw, const bool valid,
                                                    Tally& tally) {
  using R = Real<P>;
  const uint32_t t_lo = (uint32_t)t, t_hi = (uint32_t)(t >> 32);
  const Where w = locate_active(p, Q, ci_raw, valid);
  const uint8_t* cntb = p.cnt[cur];
  P* posb = reinterpret_cast<P*>(p.pos[cur]);
  const uint32_t Mqp = p.Mqp;

  // ---- level-1 loads, all independent: count and slot pair 0 of the 3x3 cells (idx 4 = own cell) ----
  uint32_t cj[9], pidx[9];
  Half<P> h0[9];
#pragma unroll
  for (int idx = 0; idx < 9; ++idx) {
    uint32_t qn, cn;
    neighbour(w, idx % 3 - 1, idx / 3 - 1, qn, cn);
    pidx[idx] = 2u * qn * Mqp + cn;
    cj[idx] = ld_u8_early(cntb + (qn * Mqp + cn));
    h0[idx] = ld_half_early(posb, pidx[idx]);
  }

  // ---- slot pair 1 where n > 2 ----
  const P FAR = R::far_away();
  Half<P> h1[9];
#pragma unroll
  for (int idx = 0; idx < 9; ++idx) {
    h1[idx].x = R::pair(FAR, FAR); h1[idx].y = h1[idx].x;
    if (cj[idx] > 2u) h1[idx] = ld_half(posb, pidx[idx] + Mqp);
  }
  const uint32_t n = w.valid ? cj[4] : 0u;
  uint32_t n_acc, n_rb, n_ro, amask;
  Half<P> o0, o1;
  cell_moves_general<P, NS, DISC>(p, h0, h1, n, w.cell, t_lo, t_hi, o0, o1, amask, n_acc, n_rb, n_ro);

  // ---- write back (line 34, L234) ----
  if (amask != 0u) {
    st_half(posb, pidx[4], o0);
    if (n > 2u) st_half(posb, pidx[4] + Mqp, o1);
  }
  if (DEBUG && w.valid) {
    p.mask[w.cell] = amask;
    if (n > 0u) atomicAdd(&p.ctl->digest, mix64(mix64(t) ^ (((unsigned long long)w.cell << 32) | amask)));
  }
  tally.acc += n_acc; tally.rb += n_rb; tally.ro += n_ro;
}

// ---------------------------------------------------------------------------------------------------------
// Cell shift (Algorithm 4, pull form).  One thread per NEW cell (L350): its own old disks that stay, in slot
// order, then the disks of the one old neighbour in direction f that left it.  l' = rn(l - f*delta) is the
// same single operation on both sides, and the +-w translation of an entrant is a separate operation after
// the test (L352), so no disk is lost or duplicated.  Writes the other buffer (L350).  Both old cells are one
// slot-pair load each (+ ids), the new cell is compacted in registers and written as one slot pair (sentinel in
// the empty slots); cells with more than 2 disks take a rolled generic path.  The last block to finish flips
// the buffer, advances the sweep index, moves the grid origin and draws the next sweep's set order and shift,
// so a sweep needs no host involvement.
// ovr: 0 = use Ctl's draws and advance the sweep; 1 = test hook (explicit dir/delta, sweep index unchanged).
// ---------------------------------------------------------------------------------------------------------
template <typename P> struct Disk { P x, y; uint32_t id; };
template <typename P> __device__ __forceinline__ Disk<P> pick(bool c, const Disk<P>& a, const Disk<P>& b) {
  Disk<P> r; r.x = c ? a.x : b.x; r.y = c ? a.y : b.y; r.id = c ? a.id : b.id; return r;
}

// The new cell from the slot pairs of its own old cell (a, ids ia) and of the old neighbour in direction f (b, ib),
// both holding at most 2 disks (empty slot = sentinel): stayers in slot order, then entrants in slot order
// (reading A13), compacted in registers.  Returns the new count; o01/i01 = slots 0, 1 (empty slots = sentinel); `rest`
// is what shift_pair_rest makes slots 2, 3 of when the count exceeds 2.
template <typename P> struct ShiftRest { uint32_t ns; Disk<P> t0, t1; };   // what slots 2, 3 are made of (rarely needed)
template <typename P, bool ALONG_X>
__device__ __forceinline__ uint32_t shift_pair(const Half<P>& a, const Half<P>& b, const uint2 ia, const uint2 ib,
                                               const P step, const P back, const P w, Half<P>& o01, uint2& i01,
                                               ShiftRest<P>& rest) {
  using R = Real<P>;
  const P FAR = R::far_away(), HALF_FAR = FAR * (P)0.5;
  // lines 7-14 (L299-312): own disks that stay; a sentinel stays a sentinel and fails the test
  Disk<P> o0 = {a.x.x, a.y.x, ia.x}, o1 = {a.x.y, a.y.y, ia.y};
  const P a0 = R::add(ALONG_X ? o0.x : o0.y, step), a1 = R::add(ALONG_X ? o1.x : o1.y, step);
  if (ALONG_X) { o0.x = a0; o1.x = a1; } else { o0.y = a0; o1.y = a1; }
  const bool k0 = a0 > (P)0 && a0 <= w, k1 = a1 > (P)0 && a1 <= w;
  // lines 17-27 (L319-339): disks of the neighbour that left it enter here; L332 is a separate operation
  Disk<P> e0 = {b.x.x, b.y.x, ib.x}, e1 = {b.x.y, b.y.y, ib.y};
  const bool v0 = e0.x < HALF_FAR, v1 = e1.x < HALF_FAR;          // occupied slots of the neighbour
  const P b0 = R::add(ALONG_X ? e0.x : e0.y, step), b1 = R::add(ALONG_X ? e1.x : e1.y, step);
  const bool g0 = v0 && !(b0 > (P)0 && b0 <= w), g1 = v1 && !(b1 > (P)0 && b1 <= w);
  const P c0 = R::add(b0, back), c1 = R::add(b1, back);
  if (ALONG_X) { e0.x = c0; e1.x = c1; } else { e0.y = c0; e1.y = c1; }
  const Disk<P> none = {FAR, FAR, 0xFFFFFFFFu};
  const uint32_t ns = (k0 ? 1u : 0u) + (k1 ? 1u : 0u), ne = (g0 ? 1u : 0u) + (g1 ? 1u : 0u);
  const Disk<P> s0 = pick(k0, o0, o1);
  const Disk<P> t0 = pick(ne > 0u, pick(g0, e0, e1), none), t1 = pick(ne > 1u, e1, none);
  const Disk<P> r0 = pick(ns > 0u, s0, t0);
  const Disk<P> r1 = pick(ns == 2u, o1, pick(ns == 1u, t0, t1));
  o01.x = R::pair(r0.x, r1.x); o01.y = R::pair(r0.y, r1.y); i01 = make_uint2(r0.id, r1.id);
  rest.ns = ns; rest.t0 = t0; rest.t1 = t1;
  return ns + ne;
}
// slots 2, 3 of the new cell (count above 2): what is left of the entrants after slots 0, 1
template <typename P>
__device__ __forceinline__ void shift_pair_rest(const ShiftRest<P>& rest, Half<P>& o23, uint2& i23) {
  using R = Real<P>;
  const Disk<P> none = {R::far_away(), R::far_away(), 0xFFFFFFFFu};
  const Disk<P> r2 = pick(rest.ns == 2u, rest.t0, pick(rest.ns == 1u, rest.t1, none));
  const Disk<P> r3 = pick(rest.ns == 2u, rest.t1, none);
  o23.x = R::pair(r2.x, r3.x); o23.y = R::pair(r2.y, r3.y); i23 = make_uint2(r2.id, r3.id);
}

// The new cell from ALL FOUR slots of its own old cell (slot pairs ho0, ho1, ids io01, io23) and of the old neighbour in
// direction f (hn0, hn1, in01, in23); empty slots = sentinel.  Straight-line code on registers: eight candidates, four
// output slots filled by prefix count (stayers in slot order, then entrants in slot order, reading A13).  Returns the
// new count (may exceed n_max: the caller reports the overflow); o0/o1 and j01/j23 = the new slot pairs and ids.
template <typename P>
__device__ __forceinline__ uint32_t shift_eight(const Half<P>& ho0, const Half<P>& ho1, const Half<P>& hn0, const Half<P>& hn1,
                                                const uint2 io01, const uint2 io23, const uint2 in01, const uint2 in23,
                                                const bool along_x, const P step, const P back, const P w,
                                                Half<P>& o0, Half<P>& o1, uint2& j01, uint2& j23) {
  using R = Real<P>;
  const P FAR = R::far_away(), HALF_FAR = FAR * (P)0.5;
  P cx[8] = {ho0.x.x, ho0.x.y, ho1.x.x, ho1.x.y, hn0.x.x, hn0.x.y, hn1.x.x, hn1.x.y};
  P cy[8] = {ho0.y.x, ho0.y.y, ho1.y.x, ho1.y.y, hn0.y.x, hn0.y.y, hn1.y.x, hn1.y.y};
  const uint32_t cid[8] = {io01.x, io01.y, io23.x, io23.y, in01.x, in01.y, in23.x, in23.y};
  bool take[8];
  uint32_t pos[8], nn = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const bool occupied = cx[i] < HALF_FAR;
    P m = R::add(along_x ? cx[i] : cy[i], step);                 // l' = l - f*delta  (L303)
    const bool in = m > (P)0 && m <= w;
    take[i] = occupied && (i < 4 ? in : !in);                    // own disks that stay; the neighbour's that left it (L326-328)
    if (i >= 4) m = R::add(m, back);                             // L332, after the test (L352)
    if (along_x) cx[i] = m; else cy[i] = m;
    pos[i] = nn;
    nn += take[i] ? 1u : 0u;
  }
  P ox[NMAX], oy[NMAX]; uint32_t oid[NMAX];
#pragma unroll
  for (int j = 0; j < NMAX; ++j) {
    ox[j] = FAR; oy[j] = FAR; oid[j] = 0xFFFFFFFFu;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const bool here = take[i] && pos[i] == (uint32_t)j;
      ox[j] = here ? cx[i] : ox[j]; oy[j] = here ? cy[i] : oy[j]; oid[j] = here ? cid[i] : oid[j];
    }
  }
  o0.x = R::pair(ox[0], ox[1]); o0.y = R::pair(oy[0], oy[1]); j01 = make_uint2(oid[0], oid[1]);
  o1.x = R::pair(ox[2], ox[3]); o1.y = R::pair(oy[2], oy[3]); j23 = make_uint2(oid[2], oid[3]);
  return nn;
}

// one new cell; ALONG_X and POSITIVE are uniform across the grid, so the caller branches once
template <typename P, bool ALONG_X, bool POSITIVE>
__device__ __forceinline__ void shift_cell(const Params& p, Ctl* ctl, const uint32_t cur, const uint32_t Q,
                                           const uint32_t ci, const P delta, const uint32_t crowd_slot) {
  using R = Real<P>;
  const uint32_t nxt = cur ^ 1u, Mqp = p.Mqp;
  const uint8_t* cntc = p.cnt[cur];
  const P* posc = reinterpret_cast<const P*>(p.pos[cur]);
  const uint2* idsc = reinterpret_cast<const uint2*>(p.ids[cur]);
  P* posn = reinterpret_cast<P*>(p.pos[nxt]);
  uint2* idsn = reinterpret_cast<uint2*>(p.ids[nxt]);
  const P w = ALONG_X ? R::wx(p) : R::wy(p);
  const P step = POSITIVE ? -delta : delta;     // l' = l - f*delta   (L303)
  const P back = POSITIVE ? w : -w;             // entrant translation (L332)
  const P FAR = R::far_away();
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
  const uint32_t own = 2u * Q * Mqp + ci, nb = 2u * qn * Mqp + cn;       // slot-pair indices (half 0)
  const uint32_t n0 = cntc[Q * Mqp + ci], n1 = cntc[qn * Mqp + cn];
  const Half<P> a = ld_half(posc, own), b = ld_half(posc, nb);
  const uint2 ia = idsc[own], ib = idsc[nb];
  uint32_t nn;
  if (n0 <= 2u && n1 <= 2u) {
    Half<P> o01; uint2 i01; ShiftRest<P> rest;
    nn = shift_pair<P, ALONG_X>(a, b, ia, ib, step, back, w, o01, i01, rest);
    st_half(posn, own, o01);
    idsn[own] = i01;
    if (nn > 2u) {
      Half<P> o23; uint2 i23;
      shift_pair_rest<P>(rest, o23, i23);
      st_half(posn, own + Mqp, o23); idsn[own + Mqp] = i23;
    }
  } else {
    // generic: any occupancy, rolled loops, scalar accesses
    nn = 0;
    P* on = posn + (size_t)own * 4;                  // new cell: slot s at on[(s>>1)*4*Mqp + (s&1)], y at +2
    uint32_t* idn = p.ids[nxt] + (size_t)own * 2;
    const uint32_t* idc = p.ids[cur];
#pragma unroll 1
    for (uint32_t pass = 0; pass < 2u; ++pass) {
      const uint32_t src = pass ? nb : own, cnt = pass ? n1 : n0;
#pragma unroll 1
      for (uint32_t i = 0; i < cnt; ++i) {
        const size_t e = (size_t)(src + (i >> 1) * Mqp);
        P x = posc[e * 4 + (i & 1u)], y = posc[e * 4 + 2 + (i & 1u)];
        P m = R::add(ALONG_X ? x : y, step);
        const bool in = m > (P)0 && m <= w;
        if (pass ? in : !in) continue;               // own: leavers go elsewhere; neighbour: stayers stay (L326-328)
        if (pass) m = R::add(m, back);               // L332, after the test (L352)
        if (ALONG_X) x = m; else y = m;
        if (nn < (uint32_t)NMAX) {
          const size_t d = (size_t)(nn >> 1) * Mqp;
          on[d * 4 + (nn & 1u)] = x; on[d * 4 + 2 + (nn & 1u)] = y;
          idn[d * 2 + (nn & 1u)] = idc[e * 2 + (i & 1u)];
        }
        ++nn;
      }
    }
    const uint32_t fill_to = nn > 2u ? (uint32_t)NMAX : 2u;     // sentinel in the empty slots of the halves in use
    for (uint32_t s = nn; s < fill_to; ++s) {
      const size_t d = (size_t)(s >> 1) * Mqp;
      on[d * 4 + (s & 1u)] = FAR; on[d * 4 + 2 + (s & 1u)] = FAR;
      idn[d * 2 + (s & 1u)] = 0xFFFFFFFFu;
    }
  }
  if (nn > (uint32_t)NMAX) { atomicOr(&ctl->err, ERRBIT_OVERFLOW); nn = NMAX; }
  if (nn > 2u && p.track_crowded) {              // crowded cell of the new state (read by the 2-slot tile kernel only)
    const uint32_t ya = div_hx(p, ci), xa = ci - ya * p.hx;
    note_crowded(ctl, crowd_slot, (2u * ya + offy) * p.mx + (2u * xa + offx));
  }
  p.cnt[nxt][Q * Mqp + ci] = (uint8_t)nn;        // L280, L342
}


// ---------------------------------------------------------------------------------------------------------
// Grid-wide barrier for the persistent sweep kernel (all blocks co-resident: cooperative launch).  One arrival
// counter in L2 that only grows; barrier number i is passed when it reaches (i+1) * gridDim.x.  The fences make
// the phase's writes visible before the arrival and drop this SM's stale L1 lines after the release, so plain
// loads of the next phase see what other SMs wrote.  ~1 us, against ~3.3 us for a dependent kernel launch
// (measured: a sweep of five launches at N = 4096 takes 16.6 us in a CUDA graph).
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void grid_barrier(uint32_t* bar, uint32_t& target) {
  target += gridDim.x;
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    atomicAdd(bar, 1u);
    uint32_t seen;
    do {
      asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(bar) : "memory");
    } while ((int32_t)(seen - target) < 0);
    __threadfence();
  }
  __syncthreads();
}

constexpr uint32_t OP_SWEEPS = 0, OP_SUB_SWEEP = 1, OP_SHIFT = 2;

// ---------------------------------------------------------------------------------------------------------
// The persistent sweep kernel: any number of sweeps of Algorithm 1 (L60-93) in ONE cooperative launch.  Each sweep is four
// sub-sweep phases (the sets in the order drawn for this sweep, Alg. 1 line 2) and the shift phase (lines
// 15-17), separated by grid barriers.  Every block owns a contiguous range of the active plane per phase (equal
// shares, so the SMs finish together) and walks it blockDim.x cells at a time; the draws of a sweep are a pure
// function of (seed, sweep index) and are recomputed by every block, so nothing but the barrier counter is
// shared between blocks during the launch.  Block 0 writes the control block back at the end.
//   op = OP_SWEEPS: sweeps until the sweep index reaches t_end (none if it already has).  OP_SUB_SWEEP (test hook): one sub-sweep of set `arg` at the current sweep index.
//   OP_SHIFT (test hook): one shift with direction `arg` and distance `delta_in`; the sweep index stays.
// FAST selects update_cell_fast (w ~ sigma) or update_cell_general; DISC (general only) the disc-shaped proposal.
// ---------------------------------------------------------------------------------------------------------
template <typename P, int NS, bool DEBUG, bool FAST, bool DISC = false>
__global__ void __launch_bounds__(SUB_THREADS, FAST ? (sizeof(P) == 4 ? FAST_MINB : FAST_MINB / 2) : SUB_MINB)
k_sweeps(const __grid_constant__ Params p, const unsigned long long t_end, const uint32_t op, const uint32_t arg,
         const double delta_in) {
  using R = Real<P>;
  __shared__ Draws sdraw;
  Ctl* ctl = p.ctl;
  unsigned long long t = ctl->t;
  uint32_t cur = ctl->cur;
  double ox = ctl->origin[0], oy = ctl->origin[1];
  uint32_t target = 0;
  Tally tally;
  const uint32_t nb = gridDim.x, b = blockIdx.x;
  // equal contiguous shares of the Mq cells of a colour plane / of the 4 Mq cells of the whole grid
  const uint32_t sub_lo = (uint32_t)((unsigned long long)p.Mq * b / nb);
  const uint32_t sub_hi = (uint32_t)((unsigned long long)p.Mq * (b + 1) / nb);
  const uint32_t all_lo = (uint32_t)((unsigned long long)(4u * p.Mq) * b / nb);
  const uint32_t all_hi = (uint32_t)((unsigned long long)(4u * p.Mq) * (b + 1) / nb);
  const uint32_t warp0 = threadIdx.x & ~31u;

  auto sub_phase = [&](const uint32_t Q) {
    for (uint32_t base = sub_lo; base + warp0 < sub_hi; base += SUB_THREADS) {    // warp-uniform trip count
      const uint32_t ci = base + threadIdx.x;
      if constexpr (FAST) update_cell_fast<P, NS, DEBUG>(p, Q, t, cur, ci, ci < sub_hi, tally);
      else                update_cell_general<P, NS, DEBUG, DISC>(p, Q, t, cur, ci, ci < sub_hi, tally);
    }
  };
  auto shift_phase = [&](const uint32_t dir, const P delta, const uint32_t crowded) {
    const bool along_x = dir < 2, positive = (dir & 1u) == 0;
    for (uint32_t g = all_lo + threadIdx.x; g < all_hi; g += SUB_THREADS) {
      const uint32_t Q = g / p.Mq, ci = g - Q * p.Mq;
      if (along_x) {
        if (positive) shift_cell<P, true, true>(p, ctl, cur, Q, ci, delta, crowded);
        else          shift_cell<P, true, false>(p, ctl, cur, Q, ci, delta, crowded);
      } else {
        if (positive) shift_cell<P, false, true>(p, ctl, cur, Q, ci, delta, crowded);
        else          shift_cell<P, false, false>(p, ctl, cur, Q, ci, delta, crowded);
      }
    }
    // the grid origin follows the shift (X = origin + cell*w + local stays put)
    const double L = along_x ? p.Lx_eff : p.Ly_eff;
    double o = along_x ? ox : oy;
    o = __dadd_rn(o, positive ? (double)delta : -(double)delta);
    if (o >= L) o = __dsub_rn(o, L);
    if (o < 0.0) o = __dadd_rn(o, L);
    if (along_x) ox = o; else oy = o;
    cur ^= 1u;
  };

  if (op == OP_SUB_SWEEP) {
    sub_phase(arg & 3u);
  } else if (op == OP_SHIFT) {
    // the state changes at an unchanged sweep index: its crowded flag is recomputed from scratch
    if (b == 0 && threadIdx.x == 0) { ctl->crowded[t & 3u] = 0u; ctl->ccount[t & 3u] = 0u; }
    grid_barrier(&ctl->bar, target);
    shift_phase(arg & 3u, (P)delta_in, (uint32_t)(t & 3u));
  } else {
    const uint32_t k = t_end > t ? (uint32_t)(t_end - t) : 0u;
    for (uint32_t it = 0; it < k; ++it) {
      if (threadIdx.x == 0) {
        sdraw = draw_sweep(p, t);                              // Alg. 1 lines 2, 15, 16 (L64, L90-91)
        if (b == 0) { ctl->crowded[(t + 2ull) & 3u] = 0u; ctl->ccount[(t + 2ull) & 3u] = 0u; }   // sweep after next
      }
      __syncthreads();
      const uint32_t dir = sdraw.dir, dist_word = sdraw.dist_word;
#pragma unroll 1
      for (uint32_t ph = 0; ph < 4u; ++ph) {                   // lines 3-14 (L66-88)
        sub_phase(sdraw.order[ph]);
        grid_barrier(&ctl->bar, target);
      }
      // line 15 (L90): delta = uniform(0, w/2) = rn(rn(0.5 w) * u01)
      const P w = dir < 2 ? R::wx(p) : R::wy(p);
      shift_phase(dir, R::mul(R::mul((P)0.5, w), R::unit(dist_word)), (uint32_t)((t + 1ull) & 3u));
      t += 1ull;
      if (it + 1u < k) grid_barrier(&ctl->bar, target);
    }
  }
  flush_tally(p, tally);
  if (op == OP_SHIFT) grid_barrier(&ctl->bar, target);   // every block has read the control block before it changes
  if (b == 0 && threadIdx.x == 0) {
    if (op == OP_SWEEPS) ctl->path_sweeps[1] += t - ctl->t;
    ctl->t = t; ctl->cur = cur; ctl->origin[0] = ox; ctl->origin[1] = oy;
  }
}

}  // namespace mpmc
