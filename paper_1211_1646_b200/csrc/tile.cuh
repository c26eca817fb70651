// tile.cuh — the fused sweep kernel for cell widths w ~ sigma: one launch = one whole sweep of Algorithm 1
// (four sub-sweeps + cell shift) with the state of a tile resident in shared memory.
//
// The cell grid is cut into ntx x nty rectangular tiles, one CTA each.  A CTA loads its tile plus a halo of
// HALO = 5 cells into shared memory (slot pair 0 of every cell: 16 B in fp32), runs the four sub-sweeps there
// with __syncthreads() between them — where separate kernels cost a dependent launch (~3.3 us measured) or a
// grid barrier each — then performs the shift from shared memory straight into the other global buffer.  One
// pass over HBM/L2 per sweep instead of six, neighbour loads at shared-memory latency.  Within a phase the warps
// draw chunks of cells from shared counters (dynamic balance); dilute systems use a variant that compacts the
// non-empty cells into full warps.
//
// Halo recompute: sub-sweep k (k = 1..4) updates the cells of its colour whose ring index
// (distance to the edge of the loaded region) is >= k (>= k + 1 on the three sides the shift does not pull from, see
// sub_sweep_rect).  A cell of ring r reads neighbours of ring >= r-1, and
// colours already updated this sweep are correct from ring j <= k-1 on, the others are untouched: by induction
// every value read is correct.  After sub-sweep 4 all cells of ring >= 4 are final; the shift of an interior
// cell (ring >= 5) reads itself and one neighbour (ring >= 4).  Halo cells are updated redundantly by the
// neighbouring CTAs with the same counter-based random numbers (Philox keyed on the GLOBAL cell id), hence with
// identical results: the trajectory is bit-identical to the one-kernel-per-sub-sweep path and to the oracle.
// Moves are tallied for interior cells only.
//
// Cells with more than 2 disks ("crowded"; about one in a million at phi = 0.716, w ~ sigma): shared memory holds
// slot pair 0 only, where a slot is empty iff it holds the sentinel, so counts are implied.  The few crowded cells
// of the state are listed in the control block (Ctl::clist, maintained by every kernel that writes cell counts);
// a CTA copies those inside its region, with their slots 2 and 3, into a small shared-memory list; a cell whose 3x3
// neighbourhood touches a listed cell is updated by a whole warp (tile_update_cell_warp), and in the shift a cell that is
// listed or pulls from a listed cell goes through the eight-candidate routine (tile_shift_cell_general).
// With more than CROWD_CAP crowded cells (Ctl::crowded) this kernel returns at once, and the general persistent
// kernel (sweep.cuh k_sweeps), which mpmc_sweep always enqueues behind the tile kernels with the target sweep
// index, runs the remaining sweeps.  The host only tiles boxes in which a loaded region never overlaps itself
// (tile + 2 HALO <= box), so every cell appears at most once in a region.
#pragma once
#include "common.cuh"
#include "sweep.cuh"

namespace mpmc {

// threads per CTA, one CTA per SM: 24 warps at <= 85 registers (fp32), 12 warps at <= 170 registers (fp64)
template <typename P> struct TileThreads { static constexpr int value = sizeof(P) == 4 ? 768 : 384; };
constexpr int HALO = 5;
constexpr int SHIFT_U = 2;              // cells per lane and chunk in the shift (their id loads are in flight together)

// -DMPMC_PHASE_CLOCKS builds a variant that records clock64() at every phase boundary (phase_clocks.py).
#ifdef MPMC_PHASE_CLOCKS
constexpr uint32_t PHASE_TILES = 4096, PHASE_MARKS = 20;
__device__ unsigned long long g_phase_clocks[PHASE_TILES][PHASE_MARKS];
__device__ __forceinline__ unsigned long long globaltimer_ns() { unsigned long long v; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(v)); return v; }
// (the clock is read AFTER a shared-memory load that follows the barrier: a bare clock read right behind __syncthreads is
// issued before the barrier releases and would record this warp's arrival instead)
__device__ __forceinline__ unsigned long long clock_after(const volatile uint32_t* s) {
  const uint32_t v = *s; unsigned long long c;
  asm volatile("mov.u64 %0, %%clock64;" : "=l"(c) : "r"(v) : "memory");
  return c;
}
#define MPMC_PHASE_MARK_AT(i, mark_word) do { if (threadIdx.x == 0 && blockIdx.x < PHASE_TILES) g_phase_clocks[blockIdx.x][i] = ((i) == 0 || (i) == 8) ? globaltimer_ns() : clock_after(mark_word); } while (0)
#else
#define MPMC_PHASE_MARK_AT(i, mark_word) do { } while (0)
#endif

#define MPMC_PHASE_MARK(i) MPMC_PHASE_MARK_AT(i, &s_last)
// thread 0's own clock, no barrier implied (marks 11, 13-15: inside the load phase)
#ifdef MPMC_PHASE_CLOCKS
#define MPMC_PHASE_NOW(i) do { if (threadIdx.x == 0 && blockIdx.x < PHASE_TILES) g_phase_clocks[blockIdx.x][i] = clock_after(&s_last); } while (0)
#else
#define MPMC_PHASE_NOW(i) do { } while (0)
#endif
// thread 0's clock where no barrier precedes (marks 16-18: kernel entry, before and after the dependency wait)
#ifdef MPMC_PHASE_CLOCKS
#define MPMC_PHASE_RAW(i) do { if (threadIdx.x == 0 && blockIdx.x < PHASE_TILES) g_phase_clocks[blockIdx.x][i] = clock64(); } while (0)
#else
#define MPMC_PHASE_RAW(i) do { } while (0)
#endif
#ifdef MPMC_PHASE_CLOCKS
#define MPMC_PHASE_VALUE(i, v) do { if (threadIdx.x == 0 && blockIdx.x < PHASE_TILES) g_phase_clocks[blockIdx.x][i] = (unsigned long long)(v); } while (0)
#else
#define MPMC_PHASE_VALUE(i, v) do { } while (0)
#endif

// v in [-m, 2m) -> [0, m)
__device__ __forceinline__ uint32_t wrap_cell(int v, uint32_t m) {
  if (v < 0) v += (int)m;
  if (v >= (int)m) v -= (int)m;
  return (uint32_t)v;
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

// Bulk asynchronous copies global -> shared (cp.async.bulk, the TMA unit; SASS UBLKCP) that report to an mbarrier: ONE
// instruction moves a whole plane row of the tile (up to 1 KB), so the tile load costs a few hundred instructions per
// CTA instead of 13 LDGSTS per thread, and every warp is free for the sort while the bytes arrive.
__device__ __forceinline__ uint32_t smem_addr(const void* ptr) { return (uint32_t)__cvta_generic_to_shared(ptr); }
__device__ __forceinline__ void mbar_init_expect(const uint32_t mbar, const uint32_t bytes) {   // one thread, one phase
  asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(mbar) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_copy_g2s(const uint32_t dst, const void* src, const uint32_t bytes, const uint32_t mbar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               :: "r"(dst), "l"(src), "r"(bytes), "r"(mbar) : "memory");
}
__device__ __forceinline__ void mbar_wait(const uint32_t mbar, const uint32_t parity) {
  uint32_t done;
  do {
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(done) : "r"(mbar), "r"(parity) : "memory");
  } while (done == 0u);
}

__device__ __forceinline__ float lds_x0(const SmemCell<float>* s, uint32_t i) { return s[i].v.x; }     // x of slot 0
__device__ __forceinline__ double lds_x0(const SmemCell<double>* s, uint32_t i) { return s[i].a.x; }
__device__ __forceinline__ float lds_x1(const SmemCell<float>* s, uint32_t i) { return s[i].v.y; }     // x of slot 1
__device__ __forceinline__ double lds_x1(const SmemCell<double>* s, uint32_t i) { return s[i].a.y; }

// Geometry of one tile: interior [x0, x0+TX) x [y0, y0+TY) in cells (all even), loaded region = interior grown
// by HALO; shared-memory planes by LOCAL colour q = 2 (ly & 1) + (lx & 1), pw x ph cells each, stride PS.
struct TileBox {
  uint32_t x0, y0, TX, TY, w, h, pw, ph;
};
// Tile number b (= blockIdx.x).  The tiles form rows; the first tl_na rows hold tl_ntx tiles each and share the half-rows
// [0, tl_hyA) evenly, the remaining rows hold tl_ntx + 1 (narrower, taller) tiles each: with two tile shapes of equal
// loaded area the tile count can match the SM count (C3: 8 x 12 + 4 x 13 = 148) where a rectangular ntx x nty grid leaves
// SMs idle (12 x 12 = 144).
__device__ __forceinline__ TileBox tile_box(const Params& p, const uint32_t b) {
  TileBox t;                                     // (32-bit products, divisions by the host's magic numbers)
  const uint32_t nA = p.tl_na * p.tl_ntx;
  uint32_t tx, h0, h1, x0, x1;
  if (b < nA) {
    const uint32_t r = magic_div(b, p.tl_div[0]);
    tx = b - r * p.tl_ntx;
    h0 = magic_div(p.tl_hyA * r, p.tl_div[2]);
    h1 = magic_div(p.tl_hyA * (r + 1u), p.tl_div[2]);
    x0 = magic_div(p.hx * tx, p.tl_div[0]); x1 = magic_div(p.hx * (tx + 1u), p.tl_div[0]);
  } else {
    const uint32_t b2 = b - nA, hyB = p.hy - p.tl_hyA;
    const uint32_t r = magic_div(b2, p.tl_div[1]);
    tx = b2 - r * (p.tl_ntx + 1u);
    h0 = p.tl_hyA + magic_div(hyB * r, p.tl_div[3]);
    h1 = p.tl_hyA + magic_div(hyB * (r + 1u), p.tl_div[3]);
    x0 = magic_div(p.hx * tx, p.tl_div[1]); x1 = magic_div(p.hx * (tx + 1u), p.tl_div[1]);
  }
  t.x0 = 2u * x0; t.TX = 2u * x1 - t.x0;
  t.y0 = 2u * h0; t.TY = 2u * (h1 - h0);
  t.w = t.TX + 2 * HALO; t.h = t.TY + 2 * HALO;
  t.pw = t.w / 2; t.ph = t.h / 2;
  return t;
}

// The cells sub-sweep k (1..4) has to update, as a rectangle of local coordinates.  The shift of the interior (ring >= 5)
// reads one more column or row on the side the shift pulls from (direction dir), so after sub-sweep 4 the cells of
// S4 = interior + that one line must be final; sub-sweep k then needs its colour correct on S4 grown by 4 - k, whose
// neighbours (S4 grown by 5 - k) are correct from the earlier sub-sweeps by the same rule.  That is ring >= k on the side
// of the shift and ring >= k + 1 on the other three.
struct SubRect { uint32_t x_lo, x_hi, y_lo, y_hi; };
__device__ __forceinline__ SubRect sub_sweep_rect(const TileBox& tb, uint32_t k, uint32_t dir) {
  SubRect r;
  r.x_lo = k + (dir == 1u ? 0u : 1u); r.x_hi = tb.w - 1u - (k + (dir == 0u ? 0u : 1u));   // dir 0: +x pulls from x+1, 1: -x
  r.y_lo = k + (dir == 3u ? 0u : 1u); r.y_hi = tb.h - 1u - (k + (dir == 2u ? 0u : 1u));   // dir 2: +y, 3: -y
  return r;
}

// A crowded cell inside the loaded region: where it is, and its slots 2 and 3 (slot pair 1 of global memory).
template <typename P> struct CrowdEntry { uint32_t si; uint32_t lxly; Half<P> hi; };   // lxly = lx | ly << 16
template <typename P> struct CrowdList { uint32_t n; CrowdEntry<P> e[CROWD_CAP]; };

template <typename P>
__device__ __forceinline__ int crowd_find(const CrowdList<P>& cl, uint32_t nc, uint32_t si) {
  for (uint32_t i = 0; i < nc; ++i) if (cl.e[i].si == si) return (int)i;
  return -1;
}
// does the 3x3 neighbourhood of the cell at local coordinates (lx, ly) contain a listed cell?
template <typename P>
__device__ __forceinline__ bool crowd_near(const CrowdList<P>& cl, uint32_t nc, uint32_t lx, uint32_t ly) {
  bool near = false;
  for (uint32_t i = 0; i < nc; ++i) {
    const uint32_t v = cl.e[i].lxly;
    near |= (lx - (v & 0xFFFFu) + 1u <= 2u) && (ly - (v >> 16) + 1u <= 2u);
  }
  return near;
}

// floor(n / d) for n < 2^16, 1 <= d < 2^16 with the per-phase constant inv = ceil(2^32 / d) (0 stands for d = 1)
__device__ __forceinline__ uint32_t small_div_magic(uint32_t d) { return d == 1u ? 0u : 0xFFFFFFFFu / d + 1u; }
__device__ __forceinline__ uint32_t small_div(uint32_t n, uint32_t inv) { return inv == 0u ? n : __umulhi(n, inv); }

// shared-memory offsets of the 3x3 cells relative to an active cell of local colour q (uniform per phase)
__device__ __forceinline__ int neighbour_offset(uint32_t q, int ox, int oy, uint32_t PS, uint32_t pw) {
  const int qx = (int)(q & 1u), qy = (int)(q >> 1);
  const int qn = ((qy ^ (oy & 1)) << 1) | (qx ^ (ox & 1));
  const int dx = ox < 0 ? qx - 1 : ox > 0 ? qx : 0, dy = oy < 0 ? qy - 1 : oy > 0 ? qy : 0;
  return (qn - (int)q) * (int)PS + dy * (int)pw + dx;
}

// ---------------------------------------------------------------------------------------------------------
// General cell update on the tile (rare: a crowded cell in the 3x3 neighbourhood), done by a WHOLE WARP for one
// cell: Algorithm 2 line by line with up to 4 disks per cell (slots 0, 1 from the planes, slots 2, 3 from the crowd
// list).  Every lane runs the move sequence (identical values in all lanes); lane idx < 9 holds the disks of
// neighbour cell idx, tests them against the trial position, and the verdict is a warp vote — the overlap test as a
// warp-parallel any-reduction over the neighbour list.  All arguments are warp-uniform.
// ---------------------------------------------------------------------------------------------------------
template <typename P, bool DEBUG>
__device__ __noinline__ void tile_update_cell_warp(const Params& p, SmemCell<P>* sm, CrowdList<P>& cl, const uint32_t nc,
                                                   const uint32_t q, const uint32_t pw, const uint32_t si_own,
                                                   const uint32_t cell, const bool interior, const unsigned long long t,
                                                   Tally& tally) {
  using R = Real<P>;
  const uint32_t PS = p.tl_PS, lane = threadIdx.x & 31u;
  const P wx = R::wx(p), wy = R::wy(p), sigma2 = R::sigma2(p);
  const P FAR = R::far_away(), HALF_FAR = FAR * (P)0.5;
  const uint32_t t_lo = (uint32_t)t, t_hi = (uint32_t)(t >> 32);
  // own disks (Alg. 2 line 8, L186), in every lane
  P lx[NMAX], ly[NMAX];
  const Half<P> h0 = lds_half(sm, si_own);
  const int eo = crowd_find(cl, nc, si_own);
  lx[0] = h0.x.x; lx[1] = h0.x.y; ly[0] = h0.y.x; ly[1] = h0.y.y;
  lx[2] = lx[3] = ly[2] = ly[3] = FAR;
  if (eo >= 0) { lx[2] = cl.e[eo].hi.x.x; lx[3] = cl.e[eo].hi.x.y; ly[2] = cl.e[eo].hi.y.x; ly[3] = cl.e[eo].hi.y.y; }
  const uint32_t n = lx[0] < HALF_FAR ? (lx[1] < HALF_FAR ? (lx[2] < HALF_FAR ? (lx[3] < HALF_FAR ? 4u : 3u) : 2u) : 1u) : 0u;
  if (n == 0u) {                                                 // lines 4-7 (L181-185)
    if (DEBUG && interior && lane == 0u) p.mask[cell] = 0u;
    return;
  }
  // lane idx < 9, idx != 4: the disks of neighbour cell idx translated into this cell's frame, q = l_j + s,
  // s = (ox wx, oy wy) (L154, L196); empty slots keep the sentinel, which never overlaps
  P jx[NMAX] = {FAR, FAR, FAR, FAR}, jy[NMAX] = {FAR, FAR, FAR, FAR};
  if (lane < 9u && lane != 4u) {
    const int ox = (int)(lane % 3u) - 1, oy = (int)(lane / 3u) - 1;
    const P sx = ox < 0 ? -wx : ox > 0 ? wx : (P)0, sy = oy < 0 ? -wy : oy > 0 ? wy : (P)0;
    const uint32_t si = (uint32_t)((int)si_own + neighbour_offset(q, ox, oy, PS, pw));
    const Half<P> h = lds_half(sm, si);
    if (h.x.x < HALF_FAR) { jx[0] = R::add(h.x.x, sx); jy[0] = R::add(h.y.x, sy); }
    if (h.x.y < HALF_FAR) { jx[1] = R::add(h.x.y, sx); jy[1] = R::add(h.y.y, sy); }
    const int en = crowd_find(cl, nc, si);
    if (en >= 0) {
      const Half<P> g = cl.e[en].hi;
      if (g.x.x < HALF_FAR) { jx[2] = R::add(g.x.x, sx); jy[2] = R::add(g.y.x, sy); }
      if (g.x.y < HALF_FAR) { jx[3] = R::add(g.x.y, sx); jy[3] = R::add(g.y.y, sy); }
    }
  }
  uint32_t perm = 0x3210u;
  if (n >= 2u) {                                                 // line 9 (L187)
    uint32_t S[4];
    philox4x32_10_rk(p, cell, t_lo, t_hi, SLOT_SHUFFLE, S);
    perm = visiting_permutation(p, n, S);
  }
  uint32_t n_acc = 0, n_rb = 0, n_ro = 0, amask = 0, vi = 0;
  uint32_t Rw[4] = {0, 0, 0, 0};
#pragma unroll 1
  for (uint32_t s = 0; s < p.n_s; ++s) {                         // lines 11-32 (L189-230)
    if ((s & 1u) == 0u) philox4x32_10_rk(p, cell, t_lo, t_hi, s >> 1, Rw);
    const uint32_t k = (perm >> (4u * vi)) & 3u;                 // p <- particles[s mod n]  (L75)
    vi = (vi + 1u == n) ? 0u : vi + 1u;
    const uint32_t r0 = (s & 1u) ? Rw[2] : Rw[0], r1 = (s & 1u) ? Rw[3] : Rw[1];
    const P lkx = k == 0u ? lx[0] : k == 1u ? lx[1] : k == 2u ? lx[2] : lx[3];
    const P lky = k == 0u ? ly[0] : k == 1u ? ly[1] : k == 2u ? ly[2] : ly[3];
    const P Mx = R::add(lkx, R::scaled_sym(p, r0)), My = R::add(lky, R::scaled_sym(p, r1));
    if (!((Mx > (P)0) && (Mx <= wx) && (My > (P)0) && (My <= wy))) { ++n_rb; continue; }   // (0, w]  (A3)
    bool ov = false;
#pragma unroll
    for (int j = 0; j < NMAX; ++j) {
      // lane 4 tests the other disks of the own cell (s = 0, q = l_j; line 17 skips j = k), lanes 0-3, 5-8 theirs
      const P qx_ = lane == 4u ? ((uint32_t)j == k ? FAR : lx[j]) : jx[j];
      const P qy_ = lane == 4u ? ((uint32_t)j == k ? FAR : ly[j]) : jy[j];
      const P Dx = R::sub(Mx, qx_), Dy = R::sub(My, qy_);
      ov |= R::fma(Dx, Dx, R::mul(Dy, Dy)) < sigma2;             // line 19 (L204), strict (A4)
    }
    if (__any_sync(0xFFFFFFFFu, ov)) { ++n_ro; }
    else {                                                       // lines 24-27 (L215-222)
      ++n_acc; amask |= 1u << (s & 31u);
      if (k == 0u) { lx[0] = Mx; ly[0] = My; } else if (k == 1u) { lx[1] = Mx; ly[1] = My; }
      else if (k == 2u) { lx[2] = Mx; ly[2] = My; } else { lx[3] = Mx; ly[3] = My; }
    }
  }
  if (lane == 0u) {
    if (amask != 0u) {                                           // write back (line 34, L234)
      Half<P> o;
      o.x = R::pair(lx[0], lx[1]); o.y = R::pair(ly[0], ly[1]);
      sts_half(sm, si_own, o);
      if (eo >= 0) { cl.e[eo].hi.x = R::pair(lx[2], lx[3]); cl.e[eo].hi.y = R::pair(ly[2], ly[3]); }
    }
    if (interior) { tally.acc += n_acc; tally.rb += n_rb; tally.ro += n_ro; }
    if (DEBUG && interior) {
      p.mask[cell] = amask;
      atomicAdd(&p.ctl->digest, mix64(mix64(t) ^ (((unsigned long long)cell << 32) | amask)));
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// One cell update (Algorithm 2) on the tile in shared memory: the arithmetic of update_cell_fast
// (sweep.cuh), the 3x3 cells read with one LDS.128 each at si_own + noff[idx].  The local colour is a run-time value
// (the nine offsets are computed once per sub-sweep and are uniform): one copy serves the four sub-sweeps of both
// variants of the kernel.
// ---------------------------------------------------------------------------------------------------------
template <typename P, int NS, bool DEBUG>
__device__ __forceinline__ void tile_update_cell(const Params& p, SmemCell<P>* sm, const uint32_t si_own,
                                                    const int (&noff)[9], const uint32_t cell, const bool interior,
                                                 const unsigned long long t, Tally& tally) {
  using R = Real<P>;
  using Pair = typename R::Pair;
  Half<P> h[9];
  const SmemCell<P>* own = sm + si_own;            // the nine offsets are uniform per sub-sweep
#pragma unroll
  for (int idx = 0; idx < 9; ++idx) h[idx] = lds_half(own + noff[idx], 0u);
  // ---- displacements of all NS moves from the GLOBAL cell id (line 12, L190; A2, A9) ----
  const uint32_t t_lo = (uint32_t)t, t_hi = (uint32_t)(t >> 32);
  P ddx[NS], ddy[NS];
#pragma unroll
  for (int b = 0; b < NS / 2; ++b) {
    uint32_t Rw[4];
    philox4x32_10_rk(p, cell, t_lo, t_hi, (uint32_t)b, Rw);
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
  const uint32_t n = Bx < HALF_FAR ? 2u : (Ax < HALF_FAR ? 1u : 0u);
  const bool two = n == 2u;
  bool flip = false;                   // true: A is slot 1
  if (two) {                           // n = 2: Fisher-Yates is one draw, j = bounded(S0, 2); j = 0 swaps
    uint32_t S[4];
    philox4x32_10_rk(p, cell, t_lo, t_hi, SLOT_SHUFFLE, S);
    flip = bounded(S[0], 2u) == 0u && !(p.flags & FLAG_NO_PARTICLE_SHUFFLE);
  }
  if (flip) { P tx = Ax, ty = Ay; Ax = Bx; Ay = By; Bx = tx; By = ty; }
  uint32_t amask = 0, bmask = 0;       // bit s: move s accepted / left the cell
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
    if (!inside) bmask |= 1u << s;                                         // leaves the cell: rejected (L79, L118)
    if (two) { const P tx = Ax, ty = Ay; Ax = Bx; Ay = By; Bx = tx; By = ty; }   // s mod n cycling (L75)
  }
  if (n == 0u) amask = 0u;             // empty cells attempt nothing (A10)
  const uint32_t n_acc = __popc(amask), n_rb = __popc(bmask);
  if (amask != 0u) {                   // write back (line 34, L234): the slot pair in slot order
    if (two && (NS & 1)) flip = !flip;
    Half<P> o;
    o.x = flip ? R::pair(Bx, Ax) : R::pair(Ax, Bx);
    o.y = flip ? R::pair(By, Ay) : R::pair(Ay, By);
    sts_half(sm, si_own, o);
  }
  // tallies, accept masks and the digest count every cell once: in the tile that owns it
  if (interior && n > 0u) {
    tally.acc += n_acc; tally.rb += n_rb; tally.ro += (uint32_t)NS - n_acc - n_rb;
  }
  if (DEBUG && interior) {
    p.mask[cell] = amask;
    if (n > 0u) atomicAdd(&p.ctl->digest, mix64(mix64(t) ^ (((unsigned long long)cell << 32) | amask)));
  }
}

// General shift of one interior cell (rare: it or its source neighbour is crowded): Algorithm 4 with up to 4 disks
// in each of the two old cells.  Straight-line code on registers (eight candidates, four output slots filled by
// prefix count), because the whole tile waits for the thread that runs it.
template <typename P>
__device__ __noinline__ void tile_shift_cell_general(const Params& p, const SmemCell<P>* sm, const CrowdList<P>& cl,
                                                     const uint32_t nc, const uint32_t si_own, const uint32_t si_nb,
                                                     const uint32_t own_g, const uint32_t nb_g, const uint32_t cnt_g,
                                                     const uint32_t cell, const bool along_x, const P step, const P back,
                                                     const P w, const uint32_t cur, const uint32_t crowd_slot) {
  using R = Real<P>;
  const uint32_t nxt = cur ^ 1u, Mqp = p.Mqp;
  const P FAR = R::far_away(), HALF_FAR = FAR * (P)0.5;
  const uint2* idsc = reinterpret_cast<const uint2*>(p.ids[cur]);
  // candidates 0-3: the own old cell (stay if still inside), 4-7: the old neighbour in direction f (enter if they left it)
  const int eo = crowd_find(cl, nc, si_own), en = crowd_find(cl, nc, si_nb);
  const uint2 io01 = idsc[own_g], in01 = idsc[nb_g];
  uint2 io23 = make_uint2(0xFFFFFFFFu, 0xFFFFFFFFu), in23 = io23;
  if (eo >= 0) io23 = idsc[own_g + Mqp];
  if (en >= 0) in23 = idsc[nb_g + Mqp];
  const Half<P> ho = lds_half(sm, si_own), hn = lds_half(sm, si_nb);
  Half<P> go, gn;
  go.x = R::pair(FAR, FAR); go.y = go.x; gn = go;
  if (eo >= 0) go = cl.e[eo].hi;
  if (en >= 0) gn = cl.e[en].hi;
  Half<P> o0, o1; uint2 j01, j23;
  uint32_t nn = shift_eight<P>(ho, go, hn, gn, io01, io23, in01, in23, along_x, step, back, w, o0, o1, j01, j23);
  if (nn > (uint32_t)NMAX) { atomicOr(&p.ctl->err, ERRBIT_OVERFLOW); nn = NMAX; }
  P* posn = reinterpret_cast<P*>(p.pos[nxt]);
  uint2* idsn = reinterpret_cast<uint2*>(p.ids[nxt]);
  st_half(posn, own_g, o0); idsn[own_g] = j01;
  if (nn > 2u) {
    st_half(posn, own_g + Mqp, o1); idsn[own_g + Mqp] = j23;
    note_crowded(p.ctl, crowd_slot, cell);
  }
  p.cnt[nxt][cnt_g] = (uint8_t)nn;
}

// The ordinary cells of sub-sweep k: the cells of local colour QL at ring >= k.  Warps draw chunks of 32 cells from a
// shared counter, so a warp that was busy with a crowded cell (or started late) simply takes fewer.
// The local colour QL is a run-time value and ONE copy of the update serves the four sub-sweeps: this variant runs the
// small and middle-sized systems, whose sub-sweeps are a single batch per warp — every phase a cold start — and with four
// specialised copies 30 % of the working warps' stall samples were instruction fetch (ncu at C2).
template <typename P, int NS, bool DEBUG>
__device__ __forceinline__ void tile_sub_sweep_cells(const Params& p, SmemCell<P>* sm, const CrowdList<P>& cl,
                                                     const uint32_t nc, const TileBox& tb, const uint32_t QL, const uint32_t k,
                                                     const uint32_t dir, const int gx0, const int gy0,
                                                     const unsigned long long t, uint32_t* next, Tally& tally) {
  const uint32_t qx = QL & 1u, qy = QL >> 1;
  const uint32_t PS = p.tl_PS, pw = tb.pw;
  int noff[9];
#pragma unroll
  for (int idx = 0; idx < 9; ++idx) noff[idx] = neighbour_offset(QL, idx % 3 - 1, idx / 3 - 1, PS, pw);
  const SubRect rc = sub_sweep_rect(tb, k, dir);
  const uint32_t px0 = (rc.x_lo - qx + 1u) >> 1, px1 = (rc.x_hi - qx) >> 1;
  const uint32_t py0 = (rc.y_lo - qy + 1u) >> 1, py1 = (rc.y_hi - qy) >> 1;
  const uint32_t nxp = px1 - px0 + 1u, count = nxp * (py1 - py0 + 1u);
  const uint32_t inv = small_div_magic(nxp);
  const uint32_t lane = threadIdx.x & 31u;
  for (;;) {                                                   // warps draw chunks of 32 cells until none is left
    uint32_t base = 0;
    if (lane == 0u) base = atomicAdd(next, 32u);
    base = __shfl_sync(0xFFFFFFFFu, base, 0);
    if (base >= count) break;
    const uint32_t idx = base + lane;
    if (idx >= count) continue;
    const uint32_t ry = small_div(idx, inv), rx = idx - ry * nxp;
    const uint32_t px = px0 + rx, py = py0 + ry, lx = 2u * px + qx, ly = 2u * py + qy;
    if (nc != 0u && crowd_near(cl, nc, lx, ly)) continue;      // done by a warp (tile_update_cell_warp)
    const uint32_t si = QL * PS + py * pw + px;
    const uint32_t cell = wrap_cell(gy0 + (int)ly, p.my) * p.mx + wrap_cell(gx0 + (int)lx, p.mx);
    const bool interior = lx - (uint32_t)HALO < tb.TX && ly - (uint32_t)HALO < tb.TY;
    tile_update_cell<P, NS, DEBUG>(p, sm, si, noff, cell, interior, t, tally);
  }
}

// ---------------------------------------------------------------------------------------------------------
// SORTED variant of the sub-sweeps.  The packed overlap test of tile_update_cell spends half of its lanes on slot 1 of
// the neighbour cells, which is empty in 96.5 % of them (w ~ sigma, phi = 0.716), and every warp pays the shuffle's
// Philox block as soon as one of its 32 cells holds two disks.  Occupancies do not change during the sub-sweeps (a move
// never leaves its cell), so ONCE per sweep, right after the load, the cells of the four sub-sweeps are sorted into
// three classes:
//   empty                       attempt nothing (A10): dropped — 11 % of the cells at phi = 0.716, 62 % at phi = 0.30;
//   simple  (61 % at C3)        one disk, and no cell of the 3x3 neighbourhood holds two: tile_update_simple tests the
//                               eight neighbour disks as FOUR packed pairs (slot 0 of two cells per pair), draws no shuffle
//                               word (Fisher-Yates of one element draws nothing, L187) and has no second own disk;
//   general (28 %)              everything else with at most two disks per cell: tile_update_cell as before.
// Cells next to a crowded cell stay with tile_update_cell_warp.  Each sub-sweep then runs on FULL warps of like cells.
// The sort has no atomics: the warps are dealt (sub-sweep, segment) jobs, a segment being a contiguous run of 32-cell
// chunks of the sub-sweep's rectangle; a job writes the plane indices of its simple cells upward from the start of its
// stretch of the sub-sweep's queue and of its general cells downward from the end, and leaves its two counts in shared
// memory.  A sub-sweep hands out batches of 32 entries, the general ones first, from one shared counter.
// ---------------------------------------------------------------------------------------------------------
// How the sort works (no per-cell arithmetic, no contended atomics): a plane row is at most 64 cells wide (the host sorts
// only such tilings), so the occupancy of a row is two 64-bit masks — bit px of occ / two: the cell holds >= 1 / 2 disks —
// taken with two ballots per row (phase A).  "A cell of the 3x3 neighbourhood holds two disks" is then nine shifted
// ORs of row masks, evaluated once per ROW of a sub-sweep's rectangle (phase B), which yields the row's simple and
// general masks; a prefix sum over the rows (phase C) places every row in the sub-sweep's queue, simple cells from the
// front, general cells from the back, and phase D writes the plane indices.  Phases end at __syncthreads().
struct QueueRect { uint32_t px_lo, px_hi, py_lo, py_hi; };     // plane coordinates of a sub-sweep's rectangle (inclusive)
__device__ __forceinline__ QueueRect queue_rect(const TileBox& tb, const uint32_t k, const uint32_t dir, const uint32_t q) {
  const uint32_t qx = q & 1u, qy = q >> 1;
  const SubRect rc = sub_sweep_rect(tb, k, dir);
  QueueRect g;
  g.px_lo = (rc.x_lo - qx + 1u) >> 1; g.py_lo = (rc.y_lo - qy + 1u) >> 1;
  g.px_hi = (rc.x_hi - qx) >> 1; g.py_hi = (rc.y_hi - qy) >> 1;
  return g;
}
// shared-memory work area of the sort, behind the queues: per plane row (q or sub-sweep k, row py) at index 4 * PH
struct SortArea {
  unsigned long long *occ, *two, *simple, *general;   // [4][PH]
  uint16_t *base1, *base2;                            // [4][PH]: queue position of the row's first simple / general cell
};
__device__ __forceinline__ SortArea sort_area(void* mem, const uint32_t PH) {
  SortArea a;
  a.occ = reinterpret_cast<unsigned long long*>(mem); a.two = a.occ + 4u * PH; a.simple = a.two + 4u * PH; a.general = a.simple + 4u * PH;
  a.base1 = reinterpret_cast<uint16_t*>(a.general + 4u * PH); a.base2 = a.base1 + 4u * PH;
  return a;
}
constexpr uint32_t SORT_ROW_BYTES = 4u * 8u + 2u * 2u;   // per plane row: four masks and two bases
constexpr uint32_t SORT_ROWS = 10;                       // plane rows a warp takes the count bytes of at a time (all of its rows up to 240 rows per tile)

__device__ __forceinline__ float2 lds_x01(const SmemCell<float>* s, uint32_t i) { return make_float2(s[i].v.x, s[i].v.y); }
__device__ __forceinline__ double2 lds_x01(const SmemCell<double>* s, uint32_t i) { return s[i].a; }
// T[px + a] as a mask over px, a in {-1, 0, +1}
__device__ __forceinline__ unsigned long long mask_shift(const unsigned long long T, const int a) { return a < 0 ? T << 1 : a > 0 ? T >> 1 : T; }

// barrier among the first `threads` threads of the CTA (the warps that sort while the others issue the tile's copies)
__device__ __forceinline__ void sort_barrier(const uint32_t threads) { asm volatile("bar.sync 1, %0;" :: "r"(threads) : "memory"); }

// Called by the first nws warps of the CTA (all of their threads).
template <typename P, bool DEBUG>
__device__ __forceinline__ void tile_sort_cells(const Params& p, const SmemCell<P>* sm, const CrowdList<P>& cl, const uint32_t nc,
                                                const TileBox& tb, const Draws& dr, const int gx0, const int gy0,
                                                uint16_t* queues, const SortArea sa, uint32_t (*s_cnt)[2], const uint32_t nws) {
  const uint32_t PS = p.tl_PS, PH = p.tl_PH, pw = tb.pw, ph = tb.ph;
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5, NW = nws;
  const uint32_t inv_ph = small_div_magic(ph);
  // (phase A — the occupancy masks of every plane row — was taken from the count bytes by the warps that copy the rows)
  MPMC_PHASE_MARK_AT(9, &s_cnt[0][0]);
  if (nc != 0u) {                                        // (uniform) cells next to a crowded cell are nobody's here: a
    for (uint32_t i = tid; i < 9u * nc; i += 32u * NW) {   // whole warp does them (tile_update_cell_warp)
      const uint32_t e = i / 9u, d = i - 9u * e;
      const uint32_t lx = (cl.e[e].lxly & 0xFFFFu) + d % 3u - 1u, ly = (cl.e[e].lxly >> 16) + d / 3u - 1u;   // may wrap below 0
      if (lx < tb.w && ly < tb.h)
        atomicAnd(&sa.occ[(((ly & 1u) << 1) | (lx & 1u)) * PH + (ly >> 1)], ~(1ull << (lx >> 1)));
    }
    sort_barrier(32u * NW);
  }
  // ---- B + C: one warp per sub-sweep, one LANE per row: the row's simple and general cells (nine shifted ORs of row
  //      masks), then the exclusive prefix sums over the rows that place every row in the sub-sweep's queue ----
  if (warp < 4u) {
    const uint32_t k = warp;
    const uint32_t Qg = k == 0u ? dr.order[0] : k == 1u ? dr.order[1] : k == 2u ? dr.order[2] : dr.order[3];
    const uint32_t q = Qg ^ 3u;                          // the region starts at an odd cell: colours flip
    const int qx = (int)(q & 1u), qy = (int)(q >> 1);
    const QueueRect g = queue_rect(tb, k + 1u, dr.dir, q);
    const unsigned long long in = (~0ull >> (63u - g.px_hi)) & (~0ull << g.px_lo);
    const unsigned long long* T = sa.two;
    const uint32_t q1 = q ^ 1u, q2 = q ^ 2u, q3 = q ^ 3u;
    // a lane takes the rows py = lane and lane + 32 (a plane has at most 64 rows... of interest: rows beyond hold no cell
    // of the rectangle), both in flight together
    uint32_t run1 = 0, run2 = 0;
    for (uint32_t r0 = 0; r0 < ph; r0 += 64u) {
      unsigned long long simple[2], general[2];
      uint32_t n1[2], n2[2], i1[2], i2[2];
#pragma unroll
      for (uint32_t h = 0; h < 2u; ++h) {
        const uint32_t py = r0 + lane + 32u * h;
        simple[h] = 0ull; general[h] = 0ull;
        if (py >= g.py_lo && py <= g.py_hi) {
          const uint32_t ra = py + (uint32_t)qy - 1u, rb = py + (uint32_t)qy;   // the plane rows of the cells below / above
          unsigned long long c = T[q * PH + py];
          c |= mask_shift(T[q1 * PH + py], qx - 1) | mask_shift(T[q1 * PH + py], qx);
          c |= T[q2 * PH + ra] | T[q2 * PH + rb];
          c |= mask_shift(T[q3 * PH + ra], qx - 1) | mask_shift(T[q3 * PH + ra], qx);
          c |= mask_shift(T[q3 * PH + rb], qx - 1) | mask_shift(T[q3 * PH + rb], qx);
          const unsigned long long o = sa.occ[q * PH + py] & in;
          simple[h] = o & ~c; general[h] = o & c;
        }
        n1[h] = (uint32_t)__popcll(simple[h]); n2[h] = (uint32_t)__popcll(general[h]);
        i1[h] = n1[h]; i2[h] = n2[h];
      }
#pragma unroll
      for (uint32_t d = 1; d < 32u; d <<= 1) {       // inclusive prefix sums over the lanes, the two halves side by side
        const uint32_t a0 = __shfl_up_sync(0xFFFFFFFFu, i1[0], d), b0 = __shfl_up_sync(0xFFFFFFFFu, i2[0], d);
        const uint32_t a1 = __shfl_up_sync(0xFFFFFFFFu, i1[1], d), b1 = __shfl_up_sync(0xFFFFFFFFu, i2[1], d);
        if (lane >= d) { i1[0] += a0; i2[0] += b0; i1[1] += a1; i2[1] += b1; }
      }
      const uint32_t t1 = __shfl_sync(0xFFFFFFFFu, i1[0], 31), t2 = __shfl_sync(0xFFFFFFFFu, i2[0], 31);
#pragma unroll
      for (uint32_t h = 0; h < 2u; ++h) {
        const uint32_t py = r0 + lane + 32u * h;
        if (py < ph) {
          sa.simple[k * PH + py] = simple[h]; sa.general[k * PH + py] = general[h];
          sa.base1[k * PH + py] = (uint16_t)(run1 + (h ? t1 : 0u) + i1[h] - n1[h]);
          sa.base2[k * PH + py] = (uint16_t)(run2 + (h ? t2 : 0u) + i2[h] - n2[h]);
        }
      }
      run1 += t1 + __shfl_sync(0xFFFFFFFFu, i1[1], 31); run2 += t2 + __shfl_sync(0xFFFFFFFFu, i2[1], 31);
    }
    if (lane == 0u) { s_cnt[k][0] = run1; s_cnt[k][1] = run2; }
  }
  sort_barrier(32u * NW);
  MPMC_PHASE_MARK_AT(10, &s_cnt[0][0]);
  // ---- D: the plane indices, a warp per row, a lane per cell: simple cells from the front of the sub-sweep's queue,
  //      general cells from its back ----
  const uint32_t below = (1u << lane) - 1u;
  for (uint32_t r = warp; r < 4u * ph; r += 2u * NW) {           // two rows per round: their loads are in flight together
    uint32_t k[2], py[2], at1[2], at2[2];
    unsigned long long m1[2], m2[2];
#pragma unroll
    for (uint32_t h = 0; h < 2u; ++h) {
      const uint32_t rr = min(r + h * NW, 4u * ph - 1u);
      const bool live = r + h * NW < 4u * ph;
      k[h] = small_div(rr, inv_ph); py[h] = rr - k[h] * ph;
      m1[h] = live ? sa.simple[k[h] * PH + py[h]] : 0ull; m2[h] = live ? sa.general[k[h] * PH + py[h]] : 0ull;
      at1[h] = sa.base1[k[h] * PH + py[h]]; at2[h] = PS - 1u - sa.base2[k[h] * PH + py[h]];
    }
#pragma unroll
    for (uint32_t h = 0; h < 2u; ++h) {
      uint16_t* qk = queues + k[h] * PS;
#pragma unroll
      for (uint32_t half = 0; half < 2u; ++half) {        // a cell is in at most one of the two classes: one store
        const uint32_t w1 = (uint32_t)(m1[h] >> (32u * half)), w2 = (uint32_t)(m2[h] >> (32u * half));
        const bool is1 = (w1 >> lane) & 1u, is2 = (w2 >> lane) & 1u;
        const uint32_t c = (uint32_t)__popc((is1 ? w1 : w2) & below);
        if (is1 || is2) qk[is1 ? at1[h] + c : at2[h] - c] = (uint16_t)(py[h] * pw + lane + 32u * half);
        if (half == 0u) { at1[h] += (uint32_t)__popc(w1); at2[h] -= (uint32_t)__popc(w2); }
      }
    }
  }
  sort_barrier(32u * NW);
}

// A simple cell (see above): one disk, no second disk anywhere in the 3x3 cells.  Same arithmetic per disk as
// tile_update_cell — q = fma(l_j, -1, -s), D = M + (-q), r^2 = fma(Dx, Dx, Dy Dy), overlap iff r^2 < sigma^2 — on half as
// many packed instructions: the two lanes of a pair are slot 0 of two different neighbour cells.  The slots left out
// hold the sentinel, whose r^2 ~ 1e36 never decides the minimum.
template <typename P, int NS, bool DEBUG>
__device__ __forceinline__ void tile_update_simple(const Params& p, SmemCell<P>* sm, const uint32_t si_own, const int (&noff)[9],
                                                   const uint32_t cell, const bool interior, const unsigned long long t,
                                                   Tally& tally) {
  using R = Real<P>;
  using Pair = typename R::Pair;
  Half<P> h[9];
  const SmemCell<P>* own = sm + si_own;
#pragma unroll
  for (int idx = 0; idx < 9; ++idx) h[idx] = lds_half(own + noff[idx], 0u);
  const uint32_t t_lo = (uint32_t)t, t_hi = (uint32_t)(t >> 32);
  P ddx[NS], ddy[NS];
#pragma unroll
  for (int b = 0; b < NS / 2; ++b) {                   // displacements of all NS moves (line 12, L190; A2, A9)
    uint32_t Rw[4];
    philox4x32_10_rk(p, cell, t_lo, t_hi, (uint32_t)b, Rw);
    ddx[2 * b] = R::scaled_sym(p, Rw[0]); ddy[2 * b] = R::scaled_sym(p, Rw[1]);
    ddx[2 * b + 1] = R::scaled_sym(p, Rw[2]); ddy[2 * b + 1] = R::scaled_sym(p, Rw[3]);
  }
  const P wx = R::wx(p), wy = R::wy(p), sigma2 = R::sigma2(p);
  // slot 0 of the eight neighbour cells, translated into this cell's frame and negated, two cells per pair
  Pair nqx[4], nqy[4];
  {
    P qx[8], qy[8];
#pragma unroll
    for (int idx = 0; idx < 9; ++idx) {
      if (idx == 4) continue;
      const int e = idx < 4 ? idx : idx - 1;
      const int ox = idx % 3 - 1, oy = idx / 3 - 1;
      const P nsx = ox < 0 ? wx : ox > 0 ? -wx : (P)0;
      const P nsy = oy < 0 ? wy : oy > 0 ? -wy : (P)0;
      qx[e] = R::fma(h[idx].x.x, (P)-1, nsx);          // -(l_j + s) = fma(l_j, -1, -s): one rn operation (L154, L196)
      qy[e] = R::fma(h[idx].y.x, (P)-1, nsy);
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) { nqx[j] = R::pair(qx[2 * j], qx[2 * j + 1]); nqy[j] = R::pair(qy[2 * j], qy[2 * j + 1]); }
  }
  P Ax = h[4].x.x, Ay = h[4].y.x;
  uint32_t amask = 0, bmask = 0;
#pragma unroll
  for (int s = 0; s < NS; ++s) {                       // Alg. 2 lines 11-32 (L189-230) with n = 1
    const P Mx = R::add(Ax, ddx[s]), My = R::add(Ay, ddy[s]);
    const bool inside = (Mx > (P)0) && (Mx <= wx) && (My > (P)0) && (My <= wy);   // (0, w]  (A3; L79, L118)
    const Pair MMx = R::pair(Mx, Mx), MMy = R::pair(My, My);
    P rmin = R::far_away();
#pragma unroll
    for (int j = 0; j < 4; ++j) {                      // |D_move - (D + s)|^2  (line 19, L204)
      const Pair Dx = R::padd(MMx, nqx[j]), Dy = R::padd(MMy, nqy[j]);
      const Pair r2 = R::pfma(Dx, Dx, R::pmul(Dy, Dy));
      rmin = R::min3(rmin, r2.x, r2.y);
    }
    const bool acc = inside && !(rmin < sigma2);       // strict (A4)
    if (acc) { Ax = Mx; Ay = My; amask |= 1u << s; }
    if (!inside) bmask |= 1u << s;
  }
  const uint32_t n_acc = __popc(amask), n_rb = __popc(bmask);
  if (amask != 0u) {                                   // write back (line 34, L234); slot 1 keeps its sentinel
    Half<P> o;
    o.x = R::pair(Ax, h[4].x.y); o.y = R::pair(Ay, h[4].y.y);
    sts_half(sm, si_own, o);
  }
  if (interior) { tally.acc += n_acc; tally.rb += n_rb; tally.ro += (uint32_t)NS - n_acc - n_rb; }
  if (DEBUG && interior) {
    p.mask[cell] = amask;
    atomicAdd(&p.ctl->digest, mix64(mix64(t) ^ (((unsigned long long)cell << 32) | amask)));
  }
}

// One sub-sweep of the SORTED variant: batches of 32 queued cells, the general ones first (they take longer).
template <typename P, int NS, bool DEBUG>
__device__ __forceinline__ void tile_run_sorted(const Params& p, SmemCell<P>* sm, const TileBox& tb, const uint32_t q,
                                                const int gx0, const int gy0, const unsigned long long t,
                                                const uint16_t* qk, const uint32_t n_simple, const uint32_t n_general,
                                                uint32_t* next, Tally& tally) {
  const uint32_t PS = p.tl_PS, pw = tb.pw, lane = threadIdx.x & 31u;
  const uint32_t qx = q & 1u, qy = q >> 1, inv_pw = small_div_magic(pw);
  int noff[9];
#pragma unroll
  for (int idx = 0; idx < 9; ++idx) noff[idx] = neighbour_offset(q, idx % 3 - 1, idx / 3 - 1, PS, pw);
  const uint32_t total2 = (n_general + 31u) >> 5, total = total2 + ((n_simple + 31u) >> 5);
  for (;;) {
    uint32_t b = 0;
    if (lane == 0u) b = atomicAdd(next, 1u);
    b = __shfl_sync(0xFFFFFFFFu, b, 0);
    if (b >= total) break;
    const bool general = b < total2;
    const uint32_t e = 32u * (general ? b : b - total2) + lane;
    if (e >= (general ? n_general : n_simple)) continue;
    const uint32_t v = general ? qk[PS - 1u - e] : qk[e];
    const uint32_t py = small_div(v, inv_pw), px = v - py * pw, lx = 2u * px + qx, ly = 2u * py + qy;
    const uint32_t cell = wrap_cell(gy0 + (int)ly, p.my) * p.mx + wrap_cell(gx0 + (int)lx, p.mx);
    const bool interior = lx - (uint32_t)HALO < tb.TX && ly - (uint32_t)HALO < tb.TY;
    if (general) tile_update_cell<P, NS, DEBUG>(p, sm, q * PS + v, noff, cell, interior, t, tally);
    else         tile_update_simple<P, NS, DEBUG>(p, sm, q * PS + v, noff, cell, interior, t, tally);
  }
}

// ---------------------------------------------------------------------------------------------------------
// The shift of the interior cells of a tile (Algorithm 4, pull form: one thread per NEW cell, L350), from the
// planes in shared memory to the other global buffer.  Warps draw chunks of 64 cells of one local colour plane
// from shared counters, two cells per lane: the four id loads of a lane are in flight together, and consecutive
// lanes write consecutive cells of one global colour plane.  Everything that depends only on the plane (colours,
// the neighbour's offset, the index constants) is uniform.
// ---------------------------------------------------------------------------------------------------------
template <typename P, bool ALONG_X>
__device__ __forceinline__ void tile_shift_cells(const Params& p, const SmemCell<P>* sm, const CrowdList<P>& cl,
                                                 const uint32_t nc, const TileBox& tb, const int gx0, const int gy0,
                                                 const bool positive, const P delta, const uint32_t cur,
                                                 const uint32_t crowd_slot, uint32_t* next) {
  using R = Real<P>;
  const uint32_t nxt = cur ^ 1u, Mqp = p.Mqp, PS = p.tl_PS, pw = tb.pw, lane = threadIdx.x & 31u;
  const P w = ALONG_X ? R::wx(p) : R::wy(p);
  const P step = positive ? -delta : delta;     // l' = l - f*delta   (L303)
  const P back = positive ? w : -w;             // entrant translation (L332)
  const uint2* idsc = reinterpret_cast<const uint2*>(p.ids[cur]);
  P* posn = reinterpret_cast<P*>(p.pos[nxt]);
  uint2* idsn = reinterpret_cast<uint2*>(p.ids[nxt]);
  uint8_t* cntn = p.cnt[nxt];
  const uint32_t hTX = tb.TX >> 1, per_plane = hTX * (tb.TY >> 1);
  const uint32_t inv = small_div_magic(hTX);
  const int dox = ALONG_X ? (positive ? 1 : -1) : 0, doy = ALONG_X ? 0 : (positive ? 1 : -1);
  // The few interior cells that are crowded or pull from a crowded cell take the rolled general routine; they are
  // done first, by the first threads, so that its latency overlaps the chunks the other warps draw meanwhile.
  for (uint32_t pi = threadIdx.x; pi < 2u * nc; pi += blockDim.x) {
    const uint32_t e = pi >> 1, role = pi & 1u;                      // role 0: the listed cell; role 1: the cell pulling from it
    const uint32_t lx = (cl.e[e].lxly & 0xFFFFu) - (role ? (uint32_t)dox : 0u);
    const uint32_t ly = (cl.e[e].lxly >> 16) - (role ? (uint32_t)doy : 0u);
    if (!(lx - (uint32_t)HALO < tb.TX && ly - (uint32_t)HALO < tb.TY)) continue;      // not an interior cell of this tile
    const uint32_t q = ((ly & 1u) << 1) | (lx & 1u);
    const uint32_t si = q * PS + (ly >> 1) * pw + (lx >> 1), sn = (uint32_t)((int)si + neighbour_offset(q, dox, doy, PS, pw));
    if (role && crowd_find(cl, nc, si) >= 0) continue;               // listed itself: done in its own role 0
    const uint32_t gx = (uint32_t)(gx0 + (int)lx), gy = (uint32_t)(gy0 + (int)ly);    // interior: no wrap
    const uint32_t gxn = wrap_cell((int)gx + dox, p.mx), gyn = wrap_cell((int)gy + doy, p.my);
    const uint32_t Qg = ((gy & 1u) << 1) | (gx & 1u), Qn = ((gyn & 1u) << 1) | (gxn & 1u);
    const uint32_t cig = (gy >> 1) * p.hx + (gx >> 1), cin = (gyn >> 1) * p.hx + (gxn >> 1);
    tile_shift_cell_general<P>(p, sm, cl, nc, si, sn, 2u * Qg * Mqp + cig, 2u * Qn * Mqp + cin, Qg * Mqp + cig, gy * p.mx + gx,
                               ALONG_X, step, back, w, cur, crowd_slot);
  }
#pragma unroll 1
  for (uint32_t q = 0; q < 4u; ++q) {
    const uint32_t qx = q & 1u, qy = q >> 1;
    const uint32_t px0 = (HALO - qx + 1u) >> 1, py0 = (HALO - qy + 1u) >> 1;
    const int nboff = neighbour_offset(q, dox, doy, PS, pw);         // the old neighbour in direction f (L314-317)
    // the region starts at an odd cell, so the global colour of local colour q is q ^ 3 and, with arithmetic shifts,
    // gx >> 1 = px + ((gx0 + qx) >> 1): the index of an interior cell in its global plane is py*hx + px + constant
    const uint32_t Qg = q ^ 3u, Qn = Qg ^ (ALONG_X ? 1u : 2u);
    const int chx = (gx0 + (int)qx) >> 1, chy = (gy0 + (int)qy) >> 1;
    const int cbase = chy * (int)p.hx + chx;
    // the neighbour's index in ITS plane: same half-coordinate or the next/previous one, by the parity of this colour
    const int bit = ALONG_X ? (int)(Qg & 1u) : (int)(Qg >> 1);
    const int dh = positive ? bit : bit - 1;                         // (g + 1) >> 1 - (g >> 1) = bit; (g - 1) >> 1 - (g >> 1) = bit - 1
    const int hn = ALONG_X ? (int)p.hx : (int)p.hy;                  // half-cells along the shift axis
    // The cells of this plane that take the general routine above: the listed cells of the plane and the cells that pull
    // from a listed cell of the plane they pull from.  Normally none, or one or two plane indices kept in registers
    // (a per-cell search of the list cost 2 900 cycles per tile with a crowded cell, measured); more: search the list.
    uint32_t sp0 = 0xFFFFFFFFu, sp1 = 0xFFFFFFFFu, nsp = 0u;
    for (uint32_t e = 0; e < nc; ++e) {
      const uint32_t v = cl.e[e].si;
      const uint32_t pe = (v >= 2u * PS ? 2u : 0u) + ((v >= 3u * PS || (v >= PS && v < 2u * PS)) ? 1u : 0u);
      if (pe == q) { if (nsp == 0u) sp0 = v; else if (nsp == 1u) sp1 = v; ++nsp; }
      if (pe == (q ^ (ALONG_X ? 1u : 2u))) {
        const uint32_t w = (uint32_t)((int)v - nboff);
        if (nsp == 0u) sp0 = w; else if (nsp == 1u) sp1 = w;
        ++nsp;
      }
    }
    for (;;) {
      uint32_t base = 0;
      if (lane == 0u) base = atomicAdd(&next[q], 32u * SHIFT_U);
      base = __shfl_sync(0xFFFFFFFFu, base, 0);
      if (base >= per_plane) break;
      uint32_t si[SHIFT_U], sn[SHIFT_U], own[SHIFT_U], nbg[SHIFT_U], cell[SHIFT_U];
      bool ok[SHIFT_U], general[SHIFT_U];
      uint2 ia[SHIFT_U], ib[SHIFT_U];
#pragma unroll
      for (int u = 0; u < SHIFT_U; ++u) {
        const uint32_t idx = base + lane + 32u * (uint32_t)u;
        ok[u] = idx < per_plane;
        const uint32_t id2 = ok[u] ? idx : 0u;
        const uint32_t ry = small_div(id2, inv), rx = id2 - ry * hTX;
        const uint32_t px = px0 + rx, py = py0 + ry;
        si[u] = q * PS + py * pw + px; sn[u] = (uint32_t)((int)si[u] + nboff);
        const int hxg = (int)px + chx, hyg = (int)py + chy;            // half-coordinates in the global plane
        const int cig = (int)(py * p.hx + px) + cbase;
        int hnb = (ALONG_X ? hxg : hyg) + dh;                          // neighbour's half-coordinate, wrapped
        hnb = hnb < 0 ? hnb + hn : (hnb >= hn ? hnb - hn : hnb);
        const int cin = ALONG_X ? hyg * (int)p.hx + hnb : hnb * (int)p.hx + hxg;
        own[u] = 2u * Qg * Mqp + (uint32_t)cig; nbg[u] = 2u * Qn * Mqp + (uint32_t)cin;
        cell[u] = (uint32_t)(2 * hyg + (int)(Qg >> 1)) * p.mx + (uint32_t)(2 * hxg + (int)(Qg & 1u));
        general[u] = nsp <= 2u ? (si[u] == sp0 || si[u] == sp1)
                               : (crowd_find(cl, nc, si[u]) >= 0 || crowd_find(cl, nc, sn[u]) >= 0);
        if (ok[u] && !general[u]) { ia[u] = idsc[own[u]]; ib[u] = idsc[nbg[u]]; }
      }
#pragma unroll
      for (int u = 0; u < SHIFT_U; ++u) {
        if (!ok[u]) continue;
        const uint32_t cnt_g = own[u] - Qg * Mqp;                      // Qg*Mqp + cig
        if (general[u]) continue;                                      // done above
        const Half<P> a = lds_half(sm, si[u]), b = lds_half(sm, sn[u]);
        Half<P> o01; uint2 i01; ShiftRest<P> rest;
        const uint32_t nn = shift_pair<P, ALONG_X>(a, b, ia[u], ib[u], step, back, w, o01, i01, rest);
        st_half(posn, own[u], o01);
        idsn[own[u]] = i01;
        if (nn > 2u) {                            // a crowded cell of the new state
          Half<P> o23; uint2 i23;
          shift_pair_rest<P>(rest, o23, i23);
          st_half(posn, own[u] + Mqp, o23); idsn[own[u] + Mqp] = i23;
          note_crowded(p.ctl, crowd_slot, cell[u]);
        }
        cntn[cnt_g] = (uint8_t)nn;                // L280, L342
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// The fused sweep kernel: one CTA per tile, one launch per sweep.  See the header of this file.
// Dynamic shared memory: 4 planes x tl_PS cells x sizeof(SmemCell<P>).
// ---------------------------------------------------------------------------------------------------------
template <typename P, int NS, bool DEBUG, bool SORTED = false>
__global__ void __launch_bounds__(TileThreads<P>::value, 1)
k_tile_sweep(const __grid_constant__ Params p, const unsigned long long t, const Draws dr_host, const uint32_t cur) {
  using R = Real<P>;
  const uint32_t TILE_THREADS = blockDim.x;           // at most TileThreads<P>::value (the host may launch fewer)
  extern __shared__ __align__(16) unsigned char tile_smem[];
  SmemCell<P>* sm = reinterpret_cast<SmemCell<P>*>(tile_smem);
  __shared__ CrowdList<P> cl;
#ifdef MPMC_PHASE_CLOCKS
  __shared__ uint32_t s_last;                    // (the word the phase marks read behind a barrier)
#endif
  __shared__ __align__(8) unsigned long long s_mbar;   // completion of the tile load (bulk copies)
  __shared__ uint32_t s_next[8];                 // chunk counters: sub-sweeps 1-4, shift planes 0-3
  __shared__ uint32_t s_cnt[4][2];               // SORTED: simple / general cells queued per sub-sweep
  Ctl* ctl = p.ctl;
  // The sweep index comes as a kernel argument (the host counts launches), and with it the draws of this sweep — a pure
  // function of (seed, t), Alg. 1 lines 2, 15, 16 (L64, L90-91), evaluated by the host with the same draw_sweep (common.cuh)
  // — so all they decide are uniform values from the constant bank.  The code ahead of the wait is on the critical path of
  // the SM that finished the previous sweep last (24 warps computing the same uniform values took 3 400 cycles there:
  // measured), hence host-made draws, divisions by magic numbers and nothing done twice.  Launched with programmatic stream serialisation (mpmc.cu): everything below the wait reads what the previous
  // sweep wrote.  If the state is not at sweep t (an earlier launch left its sweep to the general kernel), return.
  MPMC_PHASE_RAW(16);
  Draws dr;                                      // (a copy in registers: a parameter whose address is taken lives in local memory)
  dr.order[0] = dr_host.order[0]; dr.order[1] = dr_host.order[1]; dr.order[2] = dr_host.order[2]; dr.order[3] = dr_host.order[3];
  dr.dir = dr_host.dir; dr.dist_word = dr_host.dist_word;
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const TileBox tb = tile_box(p, blockIdx.x);
  const uint32_t PS = p.tl_PS, pw = tb.pw, ph = tb.ph, Mqp = p.Mqp;
  const int gx0 = (int)tb.x0 - HALO, gy0 = (int)tb.y0 - HALO;       // global cell of the region's corner (unwrapped)
  const uint32_t nrows = 4u * ph, inv_ph = small_div_magic(ph), NW = TILE_THREADS / 32;
  const uint32_t mbar = smem_addr(&s_mbar);
  const uint32_t NPROD = NW >= 12u ? NW / 6u : 1u, NWS = NW - NPROD;   // SORTED: warps that issue the copies / that sort
  // SORTED: where this lane's cells px = lane (.x) and lane + 32 (.y) of a plane row sit in the row's global colour planes,
  // for rows of local colours with qx = 0 (col0) and qx = 1 (col1)
  uint2 col0 = make_uint2(0u, 0u), col1 = col0;
  if (SORTED) {
    const uint32_t g00 = wrap_cell(gx0 + (int)(2u * lane), p.mx), g01 = wrap_cell(gx0 + (int)(2u * (lane + 32u)), p.mx);
    const uint32_t g10 = wrap_cell(gx0 + (int)(2u * lane + 1u), p.mx), g11 = wrap_cell(gx0 + (int)(2u * (lane + 32u) + 1u), p.mx);
    col0 = make_uint2((g00 & 1u) * Mqp + (g00 >> 1), (g01 & 1u) * Mqp + (g01 >> 1));
    col1 = make_uint2((g10 & 1u) * Mqp + (g10 >> 1), (g11 & 1u) * Mqp + (g11 >> 1));
  }
  if (tid == 0) {
    cl.n = 0u;
    for (int i = 0; i < 8; ++i) s_next[i] = 0u;
    mbar_init_expect(mbar, nrows * pw * (uint32_t)sizeof(SmemCell<P>));   // the bytes of the whole region
  }
  // SORTED: a sorting warp takes blocks of rpw consecutive plane rows; lane j works out where row j of the block lies (the
  // loops of the load phase fetch that with a shuffle).  The first block is set up here, ahead of the wait.
  const uint32_t rpw = min(SORT_ROWS, (nrows + NWS - 1u) / NWS);
  uint32_t my_off = 0u, my_q = 0u, my_py = 0u;
  auto row_setup = [&](const uint32_t r0) {
    my_off = 0u; my_q = 0u; my_py = 0u;
    if (r0 + lane < nrows && lane < rpw) {
      my_q = small_div(r0 + lane, inv_ph); my_py = r0 + lane - my_q * ph;
      const uint32_t gy = wrap_cell(gy0 + (int)(2u * my_py + (my_q >> 1)), p.my);
      my_off = 2u * (((gy & 1u) << 1) * Mqp + (gy >> 1) * p.hx) + (my_q & 1u);     // (bit 0: the row's qx; the host tiles grids
                                                                                 // of fewer than 2^30 cells only)
    }
  };
  if (SORTED) row_setup(warp * rpw);
  __syncthreads();
  // ---- everything above is a function of the launch parameters; what follows reads what the previous sweep wrote ----
  MPMC_PHASE_RAW(17);
  asm volatile("griddepcontrol.wait;" ::: "memory");
  MPMC_PHASE_RAW(18);
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  // The head of the control block — sweep index, buffer parity, "too many crowded cells" — is one trip to L2 (~900 cycles).
  // The host knows which buffer holds the state of sweep t (every sweep flips it) and passes it as `cur`, so the sorted
  // variant requests the count bytes of its region at once and looks at the head when it has arrived (stale_launch below,
  // before anything is written or copied).  A head at sweep t with another parity cannot happen; it is reported.
  const uint32_t slot = (uint32_t)(t & 3u), slot1 = (uint32_t)((t + 1ull) & 3u), slot2 = (uint32_t)((t + 2ull) & 3u);
  const CtlHeader ch = ctl_header(ctl, slot);
  const uint32_t nxt = cur ^ 1u;
  auto stale_launch = [&]() -> bool {
    // the state is not at sweep t (an earlier launch left its sweep to the general kernel), or it has too many crowded
    // cells and the general kernel takes over
    if (ch.t == t && ch.cur != cur && threadIdx.x == 0) atomicOr(&ctl->err, ERRBIT_STATE);
    return ch.t != t || ch.crowded != 0u || ch.cur != cur;
  };
  if (!SORTED && stale_launch()) return;
  MPMC_PHASE_MARK(0); MPMC_PHASE_MARK(1);
  // plain variant: the list of crowded cells of this state, its first TILE_THREADS entries fetched NOW (the chain count ->
  // cell -> slots 2, 3 is three trips to L2; started here it ends under the tile load instead of behind it).  The sorted
  // variant finds the crowded cells of its region in the count bytes it reads anyway.
  uint32_t ng = 0u, my_listed = 0xFFFFFFFFu;
  if (!SORTED) {
    ng = ctl->ccount[slot];
    if (tid < ng) my_listed = ctl->clist[slot][tid];
  }
  MPMC_PHASE_NOW(11);

  // ---- load the tile and its halo: a plane row of the region is contiguous in its global colour plane (two pieces where
  //      it wraps around the box), so a row is ONE bulk copy global -> shared, issued by one thread and reported to the
  //      CTA's mbarrier; the phase runs at the L2 -> SM bandwidth all SMs share (measured 6 TB/s) with the issue slots free ----
  const P* posc = reinterpret_cast<const P*>(p.pos[cur]);
  // one bulk copy (two where the row wraps around the box) for plane row (q, py); called by ONE lane
  auto copy_row = [&](const uint32_t q, const uint32_t py) {
    const uint32_t gy = wrap_cell(gy0 + (int)(2u * py + (q >> 1)), p.my), gx = wrap_cell(gx0 + (int)(q & 1u), p.mx);
    const uint32_t first = gx >> 1, n1 = min(pw, p.hx - first);                // the box has an even number of cells: the
    const size_t row = (size_t)(2u * (((gy & 1u) << 1) | (gx & 1u))) * Mqp + (size_t)(gy >> 1) * p.hx;   // colour holds along the row
    const unsigned char* src = reinterpret_cast<const unsigned char*>(posc);
    const uint32_t dst = smem_addr(sm + q * PS + py * pw);
    bulk_copy_g2s(dst, src + (row + first) * sizeof(SmemCell<P>), n1 * (uint32_t)sizeof(SmemCell<P>), mbar);
    if (n1 < pw) bulk_copy_g2s(dst + n1 * (uint32_t)sizeof(SmemCell<P>), src + row * sizeof(SmemCell<P>), (pw - n1) * (uint32_t)sizeof(SmemCell<P>), mbar);
  };
  uint16_t* queues = reinterpret_cast<uint16_t*>(sm + 4u * PS);   // SORTED: the queues of the four sub-sweeps (behind the planes)
  if (SORTED) {
    // The sort needs occupancies, not positions: it works from the count bytes of the region (1 byte per cell against 16),
    // so the whole sort — row masks, classes, prefix sums, queues — runs under the copies of the positions, whose phase is
    // bound by L2 bandwidth and leaves the issue slots idle.  A count above 2 is a crowded cell of the region.
    // A warp takes a block of consecutive plane rows (row arithmetic by increments); lanes run along the row.
    const uint8_t* cntc = p.cnt[cur];
    const SortArea sa_load = sort_area(queues + 4u * PS, p.tl_PH);
    // Warp roles: the last NPROD warps only ISSUE the copies (a thread that issues bulk copies stalls while the copy
    // queue is full, i.e. for most of the load: measured), the other NWS warps sort.
    if (warp >= NWS) {
      asm volatile("bar.sync 2, %0;" :: "r"(TILE_THREADS) : "memory");   // (see below)
      if (stale_launch()) return;
      const uint32_t share = (nrows + NPROD - 1u) / NPROD, first = (warp - NWS) * share, last = min(nrows, first + share);
      for (uint32_t r = first + lane; r < last; r += 32u) { const uint32_t q = small_div(r, inv_ph); copy_row(q, r - q * ph); }
    }
    bool told = warp >= NWS;
    const bool has0 = lane < pw, has1 = lane + 32u < pw;
    for (uint32_t r0 = warp * rpw; warp < NWS && r0 < nrows; r0 += rpw * NWS) {
      const uint32_t nr = min(rpw, nrows - r0);
      if (r0 != warp * rpw) row_setup(r0);
      uint32_t c0[SORT_ROWS], c1[SORT_ROWS];     // counts of the cells px = lane, lane + 32 of the warp's rows
#pragma unroll
      for (uint32_t j = 0; j < SORT_ROWS; ++j) {
        c0[j] = 0u; c1[j] = 0u;
        if (j < nr) {                            // (warp-uniform)
          const uint32_t w = __shfl_sync(0xFFFFFFFFu, my_off, j), off = w >> 1;
          if (has0) c0[j] = ld_u8_early(cntc + (off + ((w & 1u) ? col1.x : col0.x)));
          if (has1) c1[j] = ld_u8_early(cntc + (off + ((w & 1u) ? col1.y : col0.y)));
        }
      }
      // the copies start once the count bytes have been REQUESTED: behind the copies' requests in the SM's queue to L2 they
      // would arrive with the last rows (measured)
      if (!told) {
        asm volatile("bar.arrive 2, %0;" :: "r"(TILE_THREADS) : "memory"); told = true;
        if (stale_launch()) return;              // (every thread of the CTA takes the same decision)
      }
      MPMC_PHASE_NOW(13);
      // phase A of the sort: the occupancy masks of these rows (lane j ends up with the masks of row j and stores them)
      uint2 m_occ = make_uint2(0u, 0u), m_two = m_occ;
      uint32_t most = 0u;
#pragma unroll
      for (uint32_t j = 0; j < SORT_ROWS; ++j) {
        if (j < nr) {
          const uint32_t b1a = __ballot_sync(0xFFFFFFFFu, c0[j] >= 1u), b1b = __ballot_sync(0xFFFFFFFFu, c1[j] >= 1u);
          const uint32_t b2a = __ballot_sync(0xFFFFFFFFu, c0[j] >= 2u), b2b = __ballot_sync(0xFFFFFFFFu, c1[j] >= 2u);
          if (lane == j) { m_occ = make_uint2(b1a, b1b); m_two = make_uint2(b2a, b2b); }
          most = max(most, max(c0[j], c1[j]));
        }
      }
      if (lane < nr) {
        reinterpret_cast<uint2*>(sa_load.occ)[my_q * p.tl_PH + my_py] = m_occ;
        reinterpret_cast<uint2*>(sa_load.two)[my_q * p.tl_PH + my_py] = m_two;
      }
      if (__any_sync(0xFFFFFFFFu, most > 2u)) {  // (rare) crowded cells: into the tile's list
#pragma unroll
        for (uint32_t j = 0; j < SORT_ROWS; ++j) {
          const uint32_t q = __shfl_sync(0xFFFFFFFFu, my_q, j), py = __shfl_sync(0xFFFFFFFFu, my_py, j);
#pragma unroll
          for (uint32_t half = 0; half < 2u; ++half) {
            if (j < nr && (half == 0u ? c0[j] : c1[j]) > 2u) {
              const uint32_t px = lane + 32u * half, e = atomicAdd(&cl.n, 1u);
              cl.e[e].si = q * PS + py * pw + px;
              cl.e[e].lxly = (2u * px + (q & 1u)) | ((2u * py + (q >> 1)) << 16);
            }
          }
        }
      }
      if (DEBUG) {                               // an empty cell of the tile: nothing accepted
#pragma unroll
        for (uint32_t j = 0; j < SORT_ROWS; ++j) {
          const uint32_t q = __shfl_sync(0xFFFFFFFFu, my_q, j), py = __shfl_sync(0xFFFFFFFFu, my_py, j);
#pragma unroll
          for (uint32_t half = 0; half < 2u; ++half) {
            const uint32_t px = lane + 32u * half, lx = 2u * px + (q & 1u), ly = 2u * py + (q >> 1);
            if (j < nr && px < pw && (half == 0u ? c0[j] : c1[j]) == 0u && lx - (uint32_t)HALO < tb.TX && ly - (uint32_t)HALO < tb.TY)
              p.mask[wrap_cell(gy0 + (int)ly, p.my) * p.mx + wrap_cell(gx0 + (int)lx, p.mx)] = 0u;
          }
        }
      }
    }
    if (!told) { asm volatile("bar.arrive 2, %0;" :: "r"(TILE_THREADS) : "memory"); if (stale_launch()) return; }
  } else {
    for (uint32_t r = warp; r < nrows; r += NW)
      if (lane == 0u) { const uint32_t q = small_div(r, inv_ph); copy_row(q, r - q * ph); }
    // the crowded cells of this state that lie in the region, with their slots 2 and 3: entry tid was fetched at the top;
    // the load of its slots 2, 3 is issued here and stored behind the tile's copies
    uint32_t my_entry = 0xFFFFFFFFu;
    Half<P> my_hi;
    if (my_listed != 0xFFFFFFFFu) {
      const uint32_t gy = my_listed / p.mx, gx = my_listed - gy * p.mx;
      const uint32_t lx = wrap_cell((int)gx - gx0, p.mx), ly = wrap_cell((int)gy - gy0, p.my);
      if (lx < tb.w && ly < tb.h) {
        my_entry = atomicAdd(&cl.n, 1u);
        cl.e[my_entry].si = (((ly & 1u) << 1) | (lx & 1u)) * PS + (ly >> 1) * pw + (lx >> 1);
        cl.e[my_entry].lxly = lx | (ly << 16);
        my_hi = ld_half(posc, (2u * (((gy & 1u) << 1) | (gx & 1u)) + 1u) * Mqp + (gy >> 1) * p.hx + (gx >> 1));
      }
    }
    if (my_entry != 0xFFFFFFFFu) cl.e[my_entry].hi = my_hi;
    for (uint32_t i = tid + TILE_THREADS; i < ng; i += TILE_THREADS) {        // (more listed cells than threads: never at w ~ sigma)
      const uint32_t cell = ctl->clist[slot][i];
      const uint32_t gy = cell / p.mx, gx = cell - gy * p.mx;
      const uint32_t lx = wrap_cell((int)gx - gx0, p.mx), ly = wrap_cell((int)gy - gy0, p.my);
      if (lx < tb.w && ly < tb.h) {
        const uint32_t e = atomicAdd(&cl.n, 1u);
        cl.e[e].si = (((ly & 1u) << 1) | (lx & 1u)) * PS + (ly >> 1) * pw + (lx >> 1);
        cl.e[e].lxly = lx | (ly << 16);
        cl.e[e].hi = ld_half(posc, (2u * (((gy & 1u) << 1) | (gx & 1u)) + 1u) * Mqp + (gy >> 1) * p.hx + (gx >> 1));
      }
    }
  }
  MPMC_PHASE_NOW(14);
  // ---- the control block of the next sweep.  Every CTA takes a ticket once it has read the block (above); the one that
  //      draws the last ticket knows that all have, and advances it right away — nothing below reads it, and the next
  //      launch waits for this one to complete — so no CTA waits for a counter at its end. ----
  const uint32_t dir = dr.dir;
  const bool along_x = dir < 2u, positive = (dir & 1u) == 0u;
  const P w = along_x ? R::wx(p) : R::wy(p);
  const P delta = R::mul(R::mul((P)0.5, w), R::unit(dr.dist_word));   // line 15 (L90)
  if (tid == TILE_THREADS - 32u) {               // (a thread of a warp that does not sort)
    ctl->crowded[slot2] = 0u; ctl->ccount[slot2] = 0u;   // slots of the sweep after next: nobody uses them now
  }
  if (tid == TILE_THREADS - 32u && atomicAdd(&ctl->ticket, 1u) == gridDim.x - 1u) {
    const double L = along_x ? p.Lx_eff : p.Ly_eff;
    double o = ctl->origin[along_x ? 0 : 1];     // the grid origin follows the shift
    o = __dadd_rn(o, positive ? (double)delta : -(double)delta);
    if (o >= L) o = __dsub_rn(o, L);
    if (o < 0.0) o = __dadd_rn(o, L);
    ctl->origin[along_x ? 0 : 1] = o;
    ctl->ticket = 0u;
    ctl->cur = nxt;
    ctl->t = t + 1ull;
    ctl->path_sweeps[0] += 1ull;
  }
  uint32_t nc;
  if (SORTED) {
    if (warp < NWS) {
      sort_barrier(32u * NWS);                   // row masks and the list of crowded cells are complete
      asm volatile("bar.arrive 3, %0;" :: "r"(TILE_THREADS) : "memory");
      tile_sort_cells<P, DEBUG>(p, sm, cl, cl.n, tb, dr, gx0, gy0, queues, sort_area(queues + 4u * PS, p.tl_PH), s_cnt, NWS);
    } else {                                     // the warps that issued the copies fetch slots 2 and 3 of the crowded cells
      asm volatile("bar.sync 3, %0;" :: "r"(TILE_THREADS) : "memory");
      const uint32_t ncs = cl.n;
      for (uint32_t i = tid - 32u * NWS; i < ncs; i += 32u * NPROD) {
        const uint32_t v = cl.e[i].lxly;
        const uint32_t gx = wrap_cell(gx0 + (int)(v & 0xFFFFu), p.mx), gy = wrap_cell(gy0 + (int)(v >> 16), p.my);
        cl.e[i].hi = ld_half(posc, (2u * (((gy & 1u) << 1) | (gx & 1u)) + 1u) * Mqp + (gy >> 1) * p.hx + (gx >> 1));
      }
    }
    MPMC_PHASE_NOW(15);
    mbar_wait(mbar, 0u);                         // the region has arrived
    __syncthreads();                             // ... the queues are written and the list is complete
    nc = cl.n;
  } else {
    mbar_wait(mbar, 0u);
    __syncthreads();
    nc = cl.n;
  }
  MPMC_PHASE_MARK(2);
  MPMC_PHASE_VALUE(12, nc);                      // crowded cells in this tile's region
  Tally tally;

  // ---- four sub-sweeps (Alg. 1 lines 3-14, L66-88): sub-sweep k updates its colour at ring >= k ----
#pragma unroll 1
  for (uint32_t k = 1; k <= 4u; ++k) {
    const uint32_t Qg = k == 1u ? dr.order[0] : k == 2u ? dr.order[1] : k == 3u ? dr.order[2] : dr.order[3];
    const uint32_t q = Qg ^ 3u;                  // the region starts at an odd cell (x0 - 5, y0 - 5): colours flip
    const uint32_t qx = q & 1u, qy = q >> 1;
    const SubRect rc = sub_sweep_rect(tb, k, dr.dir);
    // cells of this colour next to a crowded cell: one warp each, before the warp's share of the ordinary cells (a warp
    // update takes about as long as a batch of ordinary cells, so its warp simply draws one batch fewer; done at the
    // end of the sub-sweep instead, it delayed the barrier by its full length: measured)
    for (uint32_t pi = warp; pi < 9u * nc; pi += TILE_THREADS / 32) {      // (listed cell, 3x3 position) pairs
      const uint32_t e = pi / 9u, d = pi - 9u * e;
      const uint32_t elx = cl.e[e].lxly & 0xFFFFu, ely = cl.e[e].lxly >> 16;
      const uint32_t lx = elx + d % 3u - 1u, ly = ely + d / 3u - 1u;       // may wrap below 0: fails the tests
      if ((lx & 1u) != qx || (ly & 1u) != qy) continue;
      if (lx < rc.x_lo || lx > rc.x_hi || ly < rc.y_lo || ly > rc.y_hi) continue;               // not in this sub-sweep's rectangle
      bool first = true;                                         // a cell next to two listed cells is done once
      for (uint32_t e2 = 0; e2 < e; ++e2) {
        const uint32_t v = cl.e[e2].lxly;
        first &= !((lx - (v & 0xFFFFu) + 1u <= 2u) && (ly - (v >> 16) + 1u <= 2u));
      }
      if (!first) continue;
      const uint32_t si = q * PS + (ly >> 1) * pw + (lx >> 1);
      const uint32_t cell = wrap_cell(gy0 + (int)ly, p.my) * p.mx + wrap_cell(gx0 + (int)lx, p.mx);
      const bool interior = lx - (uint32_t)HALO < tb.TX && ly - (uint32_t)HALO < tb.TY;
      tile_update_cell_warp<P, DEBUG>(p, sm, cl, nc, q, pw, si, cell, interior, t, tally);
    }
    if (SORTED) {
      tile_run_sorted<P, NS, DEBUG>(p, sm, tb, q, gx0, gy0, t, queues + (k - 1u) * PS, s_cnt[k - 1u][0], s_cnt[k - 1u][1],
                                    &s_next[k - 1u], tally);
    } else {
      tile_sub_sweep_cells<P, NS, DEBUG>(p, sm, cl, nc, tb, q, k, dr.dir, gx0, gy0, t, &s_next[k - 1u], tally);
    }
    __syncthreads();
    MPMC_PHASE_MARK(2 + k);
  }

  // ---- cell shift (Alg. 1 lines 15-17; Algorithm 4) of the interior cells, shared memory -> other buffer ----
  if (along_x) tile_shift_cells<P, true>(p, sm, cl, nc, tb, gx0, gy0, positive, delta, cur, slot1, &s_next[4]);
  else         tile_shift_cells<P, false>(p, sm, cl, nc, tb, gx0, gy0, positive, delta, cur, slot1, &s_next[4]);
  flush_tally(p, tally);                         // counters
#ifdef MPMC_PHASE_CLOCKS
  __syncthreads();
  MPMC_PHASE_MARK(7);
  MPMC_PHASE_MARK(8);
#endif
}

}  // namespace mpmc
