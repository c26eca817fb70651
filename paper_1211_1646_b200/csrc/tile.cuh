// tile.cuh — the fused sweep kernel for cell widths w ~ sigma: one launch = one whole sweep of Algorithm 1
// (four sub-sweeps + cell shift) with the state of a tile resident in shared memory.
//
// The cell grid is cut into ntx x nty rectangular tiles, one CTA each.  A CTA loads its tile plus a halo of
// HALO = 5 cells into shared memory (slot pair 0 of every cell: 16 B in fp32), runs the four sub-sweeps there
// with __syncthreads() between them — where separate kernels cost a dependent launch (~3.3 us measured) or a
// grid barrier each — then performs the shift from shared memory straight into the other global buffer.  One
// pass over HBM/L2 per sweep instead of six, neighbour loads at shared-memory latency.
//
// Halo recompute: sub-sweep k (k = 1..4) updates the cells of its colour whose ring index
// (distance to the edge of the loaded region) is >= k.  A cell of ring r reads neighbours of ring >= r-1, and
// colours already updated this sweep are correct from ring j <= k-1 on, the others are untouched: by induction
// every value read is correct.  After sub-sweep 4 all cells of ring >= 4 are final; the shift of an interior
// cell (ring >= 5) reads itself and one neighbour (ring >= 4).  Halo cells are updated redundantly by the
// neighbouring CTAs with the same counter-based random numbers (Philox keyed on the GLOBAL cell id), hence with
// identical results: the trajectory is bit-identical to the one-kernel-per-sub-sweep path and to the oracle.
// Moves are tallied for interior cells only.
//
// Precondition: no cell of the system holds more than 2 disks (then slot pair 0 + sentinels is the whole state
// and counts are implied: a slot is empty iff it holds the sentinel).  The flag Ctl::crowded[t & 3] says whether
// the state at sweep t violates it; it is maintained by every kernel that writes cell counts.  A crowded state
// makes this kernel return at once, and the general persistent kernel (sweep.cuh k_sweeps), which mpmc_sweep
// always enqueues behind the tile kernels with the target sweep index, runs the remaining sweeps.
#pragma once
#include "common.cuh"
#include "sweep.cuh"

namespace mpmc {

// threads per CTA, one CTA per SM: 24 warps at <= 85 registers (fp32), 12 warps at <= 170 registers (fp64)
template <typename P> struct TileThreads { static constexpr int value = sizeof(P) == 4 ? 768 : 384; };
constexpr int HALO = 5;

__device__ __forceinline__ uint32_t wrap_cell(int v, uint32_t m, bool single) {
  if (single) { if (v < 0) v += (int)m; else if (v >= (int)m) v -= (int)m; return (uint32_t)v; }
  int r = v % (int)m; if (r < 0) r += (int)m; return (uint32_t)r;
}

template <typename P> struct SmemCell;                        // slot pair 0 of a cell: {x0, x1, y0, y1}
template <> struct SmemCell<float> { float4 v; };
template <> struct SmemCell<double> { double2 a, b; };
__device__ __forceinline__ Half<float> lds_half(const SmemCell<float>* s, uint32_t i) {
  const float4 v = s[i].v; Half<float> h; h.x.x = v.x; h.x.y = v.y; h.y.x = v.z; h.y.y = v.w; return h;
}
__device__ __forceinline__ Half<double> lds_half(const SmemCell<double>* s, uint32_t i) {
  const double2 a = s[i].a, b = s[i].b; Half<double> h; h.x.x = a.x; h.x.y = a.y; h.y.x = b.x; h.y.y = b.y; return h;
}
__device__ __forceinline__ void sts_half(SmemCell<float>* s, uint32_t i, const Half<float>& h) {
  s[i].v = make_float4(h.x.x, h.x.y, h.y.x, h.y.y);
}
__device__ __forceinline__ void sts_half(SmemCell<double>* s, uint32_t i, const Half<double>& h) {
  s[i].a = make_double2(h.x.x, h.x.y); s[i].b = make_double2(h.y.x, h.y.y);
}

// Geometry of one tile: interior [x0, x0+TX) x [y0, y0+TY) in cells (all even), loaded region = interior grown
// by HALO; shared-memory planes by LOCAL colour q = 2 (ly & 1) + (lx & 1), pw x ph cells each, stride PS.
struct TileBox {
  uint32_t x0, y0, TX, TY, w, h, pw, ph;
};
__device__ __forceinline__ TileBox tile_box(const Params& p, uint32_t tx, uint32_t ty) {
  TileBox b;
  b.x0 = 2u * (uint32_t)((unsigned long long)p.hx * tx / p.tl_ntx);
  b.y0 = 2u * (uint32_t)((unsigned long long)p.hy * ty / p.tl_nty);
  b.TX = 2u * (uint32_t)((unsigned long long)p.hx * (tx + 1) / p.tl_ntx) - b.x0;
  b.TY = 2u * (uint32_t)((unsigned long long)p.hy * (ty + 1) / p.tl_nty) - b.y0;
  b.w = b.TX + 2 * HALO; b.h = b.TY + 2 * HALO;
  b.pw = b.w / 2; b.ph = b.h / 2;
  return b;
}

// ---------------------------------------------------------------------------------------------------------
// One cell update (Algorithm 2) on the tile in shared memory: the arithmetic of update_cell_fast
// (sweep.cuh), neighbours read with one LDS.128 each.  (px, py): position in the plane of local colour q.
// ---------------------------------------------------------------------------------------------------------
template <typename P, int NS, bool DEBUG>
__device__ __forceinline__ void tile_update_cell(const Params& p, SmemCell<P>* sm, const TileBox& tb, const uint32_t q,
                                                 const uint32_t px, const uint32_t py, const bool active,
                                                 const unsigned long long t, const bool single, Tally& tally) {
  using R = Real<P>;
  using Pair = typename R::Pair;
  const uint32_t qx = q & 1u, qy = q >> 1, PS = p.tl_PS, pw = tb.pw;
  const uint32_t lx = 2u * px + qx, ly = 2u * py + qy;
  // ---- the 3x3 cells from shared memory (idx 4 = own) ----
  Half<P> h[9];
  uint32_t own_idx = 0;
#pragma unroll
  for (int idx = 0; idx < 9; ++idx) {
    const int ox = idx % 3 - 1, oy = idx / 3 - 1;
    const uint32_t qn = ((qy ^ (uint32_t)(oy & 1)) << 1) | (qx ^ (uint32_t)(ox & 1));
    const uint32_t pxn = px + (ox < 0 ? qx - 1u : ox > 0 ? qx : 0u);
    const uint32_t pyn = py + (oy < 0 ? qy - 1u : oy > 0 ? qy : 0u);
    const uint32_t si = qn * PS + pyn * pw + pxn;
    if (idx == 4) own_idx = si;
    h[idx] = lds_half(sm, si);
  }
  // ---- displacements of all NS moves from the GLOBAL cell id (line 12, L190; A2, A9) ----
  const uint32_t gx = wrap_cell((int)tb.x0 - HALO + (int)lx, p.mx, single);
  const uint32_t gy = wrap_cell((int)tb.y0 - HALO + (int)ly, p.my, single);
  const uint32_t cell = gy * p.mx + gx;
  const uint32_t t_lo = (uint32_t)t, t_hi = (uint32_t)(t >> 32);
  P ddx[NS], ddy[NS];
#pragma unroll
  for (int b = 0; b < NS / 2; ++b) {
    uint32_t Rw[4];
    philox4x32_10(cell, t_lo, t_hi, (uint32_t)b, p.seed_lo, p.seed_hi, Rw);
    ddx[2 * b] = R::scaled_sym(p, Rw[0]); ddy[2 * b] = R::scaled_sym(p, Rw[1]);
    ddx[2 * b + 1] = R::scaled_sym(p, Rw[2]); ddy[2 * b + 1] = R::scaled_sym(p, Rw[3]);
  }
  const P wx = R::wx(p), wy = R::wy(p), sigma2 = R::sigma2(p);
  const P HALF_FAR = R::far_away() * (P)0.5;
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
  // ---- own cell in visiting order (Alg. 2 lines 8-9, L186-187); a slot is empty iff it holds the sentinel ----
  P Ax = h[4].x.x, Ay = h[4].y.x, Bx = h[4].x.y, By = h[4].y.y;
  const uint32_t n = !active ? 0u : (Bx < HALF_FAR ? 2u : (Ax < HALF_FAR ? 1u : 0u));
  const bool two = n == 2u;
  bool flip = false;                   // true: A is slot 1
  if (two) {                           // n = 2: Fisher-Yates is one draw, j = bounded(S0, 2); j = 0 swaps
    uint32_t S[4];
    philox4x32_10(cell, t_lo, t_hi, SLOT_SHUFFLE, p.seed_lo, p.seed_hi, S);
    flip = bounded(S[0], 2u) == 0u;
  }
  if (flip) { P tx = Ax, ty = Ay; Ax = Bx; Ay = By; Bx = tx; By = ty; }
  uint32_t n_acc = 0, n_rb = 0, amask = 0;
#pragma unroll
  for (int s = 0; s < NS; ++s) {       // Alg. 2 lines 11-32 (L189-230)
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
    const bool acc = inside && !(rmin < sigma2);                           // strict (A4)
    if (acc) { Ax = Mx; Ay = My; amask |= 1u << s; }                       // lines 24-27 (L215-222)
    n_rb += inside ? 0u : 1u;
    n_acc += acc ? 1u : 0u;
    if (two) { const P tx = Ax, ty = Ay; Ax = Bx; Ay = By; Bx = tx; By = ty; }   // s mod n cycling (L75)
  }
  if (n == 0u) amask = 0u;             // empty cells (and idle lanes) attempt nothing (A10)
  if (amask != 0u) {                   // write back (line 34, L234): the slot pair in slot order
    if (two && (NS & 1)) flip = !flip;
    Half<P> o;
    o.x = flip ? R::pair(Bx, Ax) : R::pair(Ax, Bx);
    o.y = flip ? R::pair(By, Ay) : R::pair(Ay, By);
    sts_half(sm, own_idx, o);
  }
  // tallies, accept masks and the digest count every cell once: in the tile that owns it
  const bool interior = lx >= (uint32_t)HALO && lx < tb.TX + HALO && ly >= (uint32_t)HALO && ly < tb.TY + HALO;
  if (interior && n > 0u) {
    tally.acc += n_acc; tally.rb += n_rb; tally.ro += (uint32_t)NS - n_acc - n_rb;
  }
  if (DEBUG && interior && active) {
    p.mask[cell] = amask;
    if (n > 0u) atomicAdd(&p.ctl->digest, mix64(mix64(t) ^ (((unsigned long long)cell << 32) | amask)));
  }
}

// floor(n / d) for n < 2^16, 1 <= d < 2^16 with the per-phase constant inv = ceil(2^32 / d) (0 stands for d = 1)
__device__ __forceinline__ uint32_t small_div_magic(uint32_t d) { return d == 1u ? 0u : (uint32_t)(0xFFFFFFFFull / d) + 1u; }
__device__ __forceinline__ uint32_t small_div(uint32_t n, uint32_t inv) { return inv == 0u ? n : __umulhi(n, inv); }

// ---------------------------------------------------------------------------------------------------------
// The fused sweep kernel: one CTA per tile, one launch per sweep.  See the header of this file.
// Dynamic shared memory: 4 planes x tl_PS cells x sizeof(SmemCell<P>).
// ---------------------------------------------------------------------------------------------------------
template <typename P, int NS, bool DEBUG>
__global__ void __launch_bounds__(TileThreads<P>::value, 1)
k_tile_sweep(const __grid_constant__ Params p) {
  using R = Real<P>;
  constexpr uint32_t TILE_THREADS = TileThreads<P>::value;
  extern __shared__ __align__(16) unsigned char tile_smem[];
  SmemCell<P>* sm = reinterpret_cast<SmemCell<P>*>(tile_smem);
  __shared__ Draws sdraw;
  __shared__ uint32_t s_last;
  Ctl* ctl = p.ctl;
  const unsigned long long t = ctl->t;
  if (ctl->crowded[t & 3u] != 0u) return;        // a cell with more than 2 disks: the general kernel takes over
  const uint32_t cur = ctl->cur, nxt = cur ^ 1u;
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const uint32_t ty = blockIdx.x / p.tl_ntx, tx = blockIdx.x - ty * p.tl_ntx;
  const TileBox tb = tile_box(p, tx, ty);
  const bool single = p.tl_single != 0u;
  const uint32_t PS = p.tl_PS, pw = tb.pw, ph = tb.ph, Mqp = p.Mqp;
  if (tid == 0) {
    sdraw = draw_sweep(p, t);                    // Alg. 1 lines 2, 15, 16 (L64, L90-91)
    ctl->crowded[(t + 2ull) & 3u] = 0u;          // slot of the sweep after next: nobody uses it now
  }

  // ---- load the tile and its halo: one warp per plane row, lanes along the row (512 contiguous bytes) ----
  {
    const P* posc = reinterpret_cast<const P*>(p.pos[cur]);
    for (uint32_t row = warp; row < 4u * ph; row += TILE_THREADS / 32) {
      const uint32_t q = row / ph, py = row - q * ph;
      const uint32_t gy = wrap_cell((int)tb.y0 - HALO + (int)(2u * py + (q >> 1)), p.my, single);
      const uint32_t rowbase = (gy >> 1) * p.hx;
      for (uint32_t px = lane; px < pw; px += 32u) {
        const uint32_t gx = wrap_cell((int)tb.x0 - HALO + (int)(2u * px + (q & 1u)), p.mx, single);
        const uint32_t Qg = ((gy & 1u) << 1) | (gx & 1u);
        sts_half(sm, q * PS + py * pw + px, ld_half(posc, 2u * Qg * Mqp + rowbase + (gx >> 1)));
      }
    }
  }
  __syncthreads();
  const Draws dr = sdraw;
  Tally tally;

  // ---- four sub-sweeps (Alg. 1 lines 3-14, L66-88): sub-sweep k updates its colour at ring >= k ----
#pragma unroll 1
  for (uint32_t k = 1; k <= 4u; ++k) {
    const uint32_t Qg = k == 1u ? dr.order[0] : k == 2u ? dr.order[1] : k == 3u ? dr.order[2] : dr.order[3];
    const uint32_t q = Qg ^ 3u;                  // the region starts at an odd cell (x0 - 5, y0 - 5): colours flip
    const uint32_t qx = q & 1u, qy = q >> 1;
    const uint32_t px0 = (k - qx + 1u) >> 1, px1 = (tb.w - 1u - k - qx) >> 1;
    const uint32_t py0 = (k - qy + 1u) >> 1, py1 = (tb.h - 1u - k - qy) >> 1;
    const uint32_t nxp = px1 - px0 + 1u, count = nxp * (py1 - py0 + 1u);
    const uint32_t inv = small_div_magic(nxp);
    for (uint32_t idx = tid; idx < count; idx += TILE_THREADS) {
      const uint32_t ry = small_div(idx, inv), rx = idx - ry * nxp;
      tile_update_cell<P, NS, DEBUG>(p, sm, tb, q, px0 + rx, py0 + ry, true, t, single, tally);
    }
    __syncthreads();
  }

  // ---- cell shift (Alg. 1 lines 15-17; Algorithm 4) of the interior cells, shared memory -> other buffer ----
  {
    const uint32_t dir = dr.dir;
    const bool along_x = dir < 2u, positive = (dir & 1u) == 0u;
    const P w = along_x ? R::wx(p) : R::wy(p);
    const P delta = R::mul(R::mul((P)0.5, w), R::unit(dr.dist_word));   // line 15 (L90)
    const P step = positive ? -delta : delta;     // l' = l - f*delta   (L303)
    const P back = positive ? w : -w;             // entrant translation (L332)
    const uint2* idsc = reinterpret_cast<const uint2*>(p.ids[cur]);
    P* posn = reinterpret_cast<P*>(p.pos[nxt]);
    uint2* idsn = reinterpret_cast<uint2*>(p.ids[nxt]);
    uint8_t* cntn = p.cnt[nxt];
    const uint32_t hTX = tb.TX >> 1, per_plane = hTX * (tb.TY >> 1);
    const uint32_t inv = small_div_magic(hTX);
    const int dox = along_x ? (positive ? 1 : -1) : 0, doy = along_x ? 0 : (positive ? 1 : -1);
#pragma unroll 1
    for (uint32_t q = 0; q < 4u; ++q) {
      const uint32_t qx = q & 1u, qy = q >> 1;
      const uint32_t px0 = (HALO - qx + 1u) >> 1, py0 = (HALO - qy + 1u) >> 1;
      for (uint32_t idx = tid; idx < per_plane; idx += TILE_THREADS) {
        const uint32_t ry = small_div(idx, inv), rx = idx - ry * hTX;
        const uint32_t px = px0 + rx, py = py0 + ry;
        // the old neighbour in direction f (Alg. 4 lines 15-16, L314-317)
        const uint32_t qn = along_x ? (q ^ 1u) : (q ^ 2u);
        const uint32_t pxn = px + (dox < 0 ? qx - 1u : dox > 0 ? qx : 0u);
        const uint32_t pyn = py + (doy < 0 ? qy - 1u : doy > 0 ? qy : 0u);
        const Half<P> a = lds_half(sm, q * PS + py * pw + px), b = lds_half(sm, qn * PS + pyn * pw + pxn);
        const uint32_t gx = wrap_cell((int)tb.x0 - HALO + (int)(2u * px + qx), p.mx, true);   // interior: one wrap
        const uint32_t gy = wrap_cell((int)tb.y0 - HALO + (int)(2u * py + qy), p.my, true);
        const uint32_t gxn = wrap_cell((int)gx + dox, p.mx, true), gyn = wrap_cell((int)gy + doy, p.my, true);
        const uint32_t Qg = ((gy & 1u) << 1) | (gx & 1u), Qn = ((gyn & 1u) << 1) | (gxn & 1u);
        const uint32_t cig = (gy >> 1) * p.hx + (gx >> 1), cin = (gyn >> 1) * p.hx + (gxn >> 1);
        const uint32_t own = 2u * Qg * Mqp + cig;
        const uint2 ia = idsc[own], ib = idsc[2u * Qn * Mqp + cin];
        Half<P> o01, o23; uint2 i01, i23;
        uint32_t nn;
        if (along_x) nn = shift_pair<P, true>(a, b, ia, ib, step, back, w, o01, i01, o23, i23);
        else         nn = shift_pair<P, false>(a, b, ia, ib, step, back, w, o01, i01, o23, i23);
        st_half(posn, own, o01);
        idsn[own] = i01;
        if (nn > 2u) {                            // the next state needs the general kernel
          st_half(posn, own + Mqp, o23); idsn[own + Mqp] = i23;
          ctl->crowded[(t + 1ull) & 3u] = 1u;
        }
        cntn[Qg * Mqp + cig] = (uint8_t)nn;       // L280, L342
      }
    }
  }

  // ---- counters; the last CTA to finish advances the control block ----
  flush_tally(p, tally);
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    s_last = (atomicAdd(&ctl->ticket, 1u) == gridDim.x - 1u) ? 1u : 0u;
  }
  __syncthreads();
  if (s_last && tid == 0) {
    const uint32_t dir = dr.dir;
    const bool along_x = dir < 2u, positive = (dir & 1u) == 0u;
    const P w = along_x ? R::wx(p) : R::wy(p);
    const P delta = R::mul(R::mul((P)0.5, w), R::unit(dr.dist_word));
    const double L = along_x ? p.Lx_eff : p.Ly_eff;
    double o = ctl->origin[along_x ? 0 : 1];     // the grid origin follows the shift
    o = __dadd_rn(o, positive ? (double)delta : -(double)delta);
    if (o >= L) o = __dsub_rn(o, L);
    if (o < 0.0) o = __dadd_rn(o, L);
    ctl->origin[along_x ? 0 : 1] = o;
    ctl->ticket = 0u;
    ctl->cur = nxt;
    ctl->t = t + 1ull;
  }
}

}  // namespace mpmc
