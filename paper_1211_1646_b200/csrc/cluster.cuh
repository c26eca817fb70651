// cluster.cuh — small systems: any number of sweeps of Algorithm 1 in ONE
// launch of ONE thread-block cluster, with the whole state RESIDENT in the cluster's shared memory.
//
// Below ~2e4 cells the fused tile kernels (tile.cuh, tile4.cuh) are latency, not throughput: a launch per sweep, a tile load
// and a shift through L2 every sweep, a recomputed halo of 5 cells around tiles a few cells wide (6 x redundant work at
// N = 4096), and every phase a cold start.  Here the cell grid is cut into cx x cy tiles without halo, one CTA of the
// cluster each (up to 16 CTAs = 16 SMs); a CTA keeps its cells — all four slots and the ids — in its shared memory from the
// first sweep of the call to the last, reads the cells of the neighbouring tiles from the neighbouring CTAs' shared memory
// (distributed shared memory) and synchronises with the hardware cluster barrier: four sub-sweeps and the shift are five
// barriers per sweep, no launch, no global traffic, and the loop's code stays in the instruction cache.
//
// The arithmetic is that of the other kernels — the w ~ sigma cell update of update_cell_fast / tile_update_cell restated on
// registers (cl_moves_fast), cell_moves_general (Algorithm 2 with up to n_max = 4 disks per cell, any cell width, both
// proposals), shift_pair and shift_eight (Algorithm 4) from sweep.cuh — with Philox keyed on the global cell id, so the
// trajectory is bit-identical to every other path and to the oracle.
//
// A sub-sweep writes only cells of the active colour and reads only cells of the other colours besides the own cell, so it
// needs no barrier inside; the shift reads the old own cell and one old neighbour from one buffer and writes the new cell
// to the other (two buffers per CTA), so it needs none either.
//
// Measured (B200, us per sweep, this kernel / fused tile kernel): N = 1024-4096 fp32 w ~ sigma 4.9-5.2 / 11.7; C1 (N = 4096,
// fp64) 9.5 / 15.2; N = 4096 at w = 1.4 sigma with the disc proposal, fp32 13.1 / 16.1.  What a sweep costs here is latency:
// one warp per scheduler runs a dependent chain of ~700 (fp32) to ~900 (fp64) instructions per sub-sweep at ~0.3-0.4
// instructions per cycle (fp32 1 650 cycles, fp64 3 500), five barriers of ~400 cycles, a shift of 1 900-2 500.
#pragma once
#include <cooperative_groups.h>
#include <cstdio>

#include "common.cuh"
#include "sweep.cuh"
#include "tile.cuh"

namespace mpmc {

// threads per CTA; a CTA holds as many cells as its shared memory has room for (two buffers: the shift writes the other one)
template <typename P> struct ClThreads { static constexpr int value = sizeof(P) == 4 ? 384 : 256; };   // (~170 / ~255 registers)
constexpr uint32_t CL_MAX_CTAS = 16;
// Cells per CTA up to which the host chooses this kernel: while a sub-sweep is ONE pass of the CTA's threads with some
// margin.  Measured against the fused tile kernels on a B200 (us per sweep, resident / tile): fast fp32 1116 cells per CTA
// 10.5 / 12.1, 1732 15.0 / 12.9; fast fp64 621 14.5 / 15.3, 1116 23.4 / 15.3; general fp32 585 19.2 / 20.4, 910 21.1 / 21.1;
// general fp64 910 35.0 / 39.1, 1306 56.8 / 39.2.
template <typename P> constexpr uint32_t cluster_max_cells_per_cta(bool fast) {
  return fast ? (sizeof(P) == 4 ? 1152u : 640u) : (sizeof(P) == 4 ? 768u : 920u);
}

// shared memory of one CTA: two buffers of {slot pair 0, slot pair 1, ids of slots 0-1, ids of slots 2-3, count} per cell,
// row-major with the stride of the widest tile
template <typename P> constexpr size_t cluster_cell_bytes() { return 2 * (2 * sizeof(SmemCell<P>) + 2 * sizeof(uint2) + 1); }

template <typename P> struct ClTile {
  SmemCell<P>* s0;   // slot pair 0
  SmemCell<P>* s1;   // slot pair 1 (sentinels unless the cell holds more than 2 disks)
  uint2* i01;        // ids of slots 0, 1
  uint2* i23;        // ids of slots 2, 3 (0xFFFFFFFF unless in use)
  uint8_t* cnt;      // disks in the cell
};
// buffer b (0 / 1) of the CTA whose dynamic shared memory starts at base
template <typename P>
__device__ __forceinline__ ClTile<P> cl_tile(unsigned char* base, const uint32_t cap, const uint32_t b) {
  ClTile<P> t;
  t.s0 = reinterpret_cast<SmemCell<P>*>(base) + 2u * b * cap; t.s1 = t.s0 + cap;
  t.i01 = reinterpret_cast<uint2*>(reinterpret_cast<SmemCell<P>*>(base) + 4u * cap) + 2u * b * cap; t.i23 = t.i01 + cap;
  t.cnt = reinterpret_cast<uint8_t*>(reinterpret_cast<uint2*>(reinterpret_cast<SmemCell<P>*>(base) + 4u * cap) + 4u * cap) + b * cap;
  return t;
}

// -DMPMC_PHASE_CLOCKS (phase_clocks.py --resident): thread 0 of every CTA adds up the SM cycles it spends in the sub-sweeps,
// at the cluster barriers and in the shift; row = CTA, values = {sweeps, sub-sweeps, barriers, shift, whole loop}
#ifdef MPMC_PHASE_CLOCKS
constexpr uint32_t CL_CLOCK_MARKS = 5;
__device__ unsigned long long g_cluster_clocks[CL_MAX_CTAS][CL_CLOCK_MARKS];
#define MPMC_CL_CLOCK_START() long long ck_sub = 0, ck_bar = 0, ck_shift = 0, ck_a = clock64(); const long long ck_t0 = ck_a
#define MPMC_CL_CLOCK_ADD(v) do { const long long n_ = clock64(); v += n_ - ck_a; ck_a = n_; } while (0)
#else
#define MPMC_CL_CLOCK_START() do { } while (0)
#define MPMC_CL_CLOCK_ADD(v) do { } while (0)
#endif

// The random numbers of one cell's moves in the fast update: the NS displacements (Alg. 2 line 12, L190; A2, A9) and
// whether the shuffle of TWO disks swaps them (line 9, L187: Fisher-Yates of two is one draw, j = bounded(S0, 2); j = 0
// swaps; made only for a cell of two).  The displacement blocks depend on nothing loaded: they run under the loads.
template <typename P, int NS> struct ClDraws { P ddx[NS], ddy[NS]; bool swap2; };
template <typename P, int NS>
__device__ __forceinline__ void cl_draws_fast(const Params& p, const uint32_t cell, const uint32_t t_lo, const uint32_t t_hi,
                                              const bool two, ClDraws<P, NS>& d) {
  using R = Real<P>;
  static_assert(NS > 0 && NS % 2 == 0, "compile-time n_s must be even");
#pragma unroll
  for (int q = 0; q < NS / 2; ++q) {
    uint32_t Rw[4];
    philox4x32_10(cell, t_lo, t_hi, (uint32_t)q, p.seed_lo, p.seed_hi, Rw);
    d.ddx[2 * q] = R::scaled_sym(p, Rw[0]); d.ddy[2 * q] = R::scaled_sym(p, Rw[1]);
    d.ddx[2 * q + 1] = R::scaled_sym(p, Rw[2]); d.ddy[2 * q + 1] = R::scaled_sym(p, Rw[3]);
  }
  d.swap2 = false;
  if (two) {                                       // (a single disk is not shuffled: no draw is made)
    uint32_t S[4];
    philox4x32_10(cell, t_lo, t_hi, SLOT_SHUFFLE, p.seed_lo, p.seed_hi, S);
    d.swap2 = bounded(S[0], 2u) == 0u && !(p.flags & FLAG_NO_PARTICLE_SHUFFLE);
  }
}

// The moves of one cell whose 3 x 3 cells hold at most 2 disks each (w ~ sigma), on registers: h = slot pair 0 of the 3 x 3
// cells (idx 4 = own), n = the own count, d = the cell's draws.  The arithmetic of update_cell_fast (sweep.cuh) /
// tile_update_cell (tile.cuh), step for step: neighbours translated into this cell's frame and negated with one fma,
// -(l_j + s) = fma(l_j, -1, -s) (L154, L196); the two own disks in visiting order, swapped iff n = 2 (L75, L187); verdict of
// a move = in the cell and min r^2 >= sigma^2 (L79, L118, L194-204).  Returns the new slot pair in slot order, the accept
// mask and the tallies.
template <typename P, int NS>
__device__ __forceinline__ void cl_moves_fast(const Params& p, const Half<P> (&h)[9], const uint32_t n, const ClDraws<P, NS>& d,
                                              Half<P>& o, uint32_t& amask, uint32_t& n_acc, uint32_t& n_rb, uint32_t& n_ro) {
  using R = Real<P>;
  using Pair = typename R::Pair;
  n_acc = 0; n_rb = 0; n_ro = 0; amask = 0;
  const P wx = R::wx(p), wy = R::wy(p), sigma2 = R::sigma2(p);
  const Pair MINUS1 = R::pair((P)-1, (P)-1);
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
  P Ax = h[4].x.x, Ay = h[4].y.x, Bx = h[4].x.y, By = h[4].y.y;      // own cell in visiting order (Alg. 2 lines 8-9)
  const bool two = n == 2u;
  bool flip = two && d.swap2;                      // true: A is slot 1 (a single disk is not shuffled: no draw is used)
  if (flip) { const P tx = Ax, ty = Ay; Ax = Bx; Ay = By; Bx = tx; By = ty; }
#pragma unroll
  for (int s = 0; s < NS; ++s) {                   // NS trial moves (Alg. 2 lines 11-32, L189-230)
    const P Mx = R::add(Ax, d.ddx[s]), My = R::add(Ay, d.ddy[s]);
    const bool inside = (Mx > (P)0) && (Mx <= wx) && (My > (P)0) && (My <= wy);   // (0, w]  (A3; L79, L118)
    const P Dbx = R::sub(Mx, Bx), Dby = R::sub(My, By);                          // the other own disk
    OverlapAcc<P> ov(sigma2, R::fma(Dbx, Dbx, R::mul(Dby, Dby)));
    const Pair MMx = R::pair(Mx, Mx), MMy = R::pair(My, My);
#pragma unroll
    for (int e = 0; e < 8; ++e) {                  // |D_move - (D + s)|^2  (line 19, L204)
      const Pair Dx = R::padd(MMx, nqx[e]), Dy = R::padd(MMy, nqy[e]);
      const Pair r2 = R::pfma(Dx, Dx, R::pmul(Dy, Dy));
      if (e & 1) ov.template pair<1>(r2); else ov.template pair<0>(r2);
    }
    const bool acc = inside && !ov.overlap(sigma2);   // strict (A4)
    if (acc) { Ax = Mx; Ay = My; amask |= 1u << s; }
    n_rb += inside ? 0u : 1u;
    n_acc += acc ? 1u : 0u;
    if (two) { const P tx = Ax, ty = Ay; Ax = Bx; Ay = By; Bx = tx; By = ty; }   // s mod n cycling (L75)
  }
  if (n == 0u) { n_rb = 0u; n_acc = 0u; amask = 0u; }                            // empty cells attempt nothing (A10)
  else { n_ro = (uint32_t)NS - n_acc - n_rb; }
  if (two && (NS & 1)) flip = !flip;
  o.x = flip ? R::pair(Bx, Ax) : R::pair(Ax, Bx);
  o.y = flip ? R::pair(By, Ay) : R::pair(Ay, By);
}

// The barrier between the phases of a sweep.  What it has to order is SHARED memory only: a CTA's stores into its own tile
// before the other CTAs' loads from it (and their loads before its next stores).  cluster.sync() is a release at cluster
// scope, which this GPU implements as MEMBAR.ALL.GPU + ERRBAR (SASS; ~470 cycles per barrier, 18 % of a sweep at N = 4096:
// ncu).  A tile lives in ONE place, the shared memory of its SM, and remote loads are served there, uncached; so a fence at
// CTA scope (MEMBAR.ALL.CTA: this thread's stores are performed in that memory) followed by the relaxed arrive puts the
// stores before every load a CTA issues after its wait, and a thread has consumed its own loads before it arrives.  The
// PTX memory model asks for cluster scope here; -DMPMC_CLUSTER_SYNC_STRICT builds that version.  (Global memory is not
// ordered by this barrier: the kernel writes global memory only at its end, and the launch boundary orders that.)
__device__ __forceinline__ void cl_sync() {
#ifdef MPMC_CLUSTER_SYNC_STRICT
  cooperative_groups::this_cluster().sync();
#else
  asm volatile("fence.acq_rel.cta;\n\tbarrier.cluster.arrive.relaxed.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
#endif
}
__device__ __forceinline__ void cl_sync_arrive() {
#ifdef MPMC_CLUSTER_SYNC_STRICT
  cooperative_groups::this_cluster().barrier_arrive();
#else
  asm volatile("fence.acq_rel.cta;\n\tbarrier.cluster.arrive.relaxed.aligned;" ::: "memory");
#endif
}
__device__ __forceinline__ void cl_sync_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

// A CTA's tile and what it needs to know of its periodic neighbours (balanced split of the mx x my cells, every tile non-empty)
struct ClGeom { uint32_t wme, hme, wl, hb, stride, cap; };   // own width / height; width of the tile to the left, height of the
                                                             // tile below; row stride and capacity of every CTA's arrays
// where the cell next to local cell (lx, ly) in direction (ox, oy) lives: which of the 3 x 3 tiles around this one
// (3 sy + sx; 4 = this tile), and its index there.  One step to the left of column 0 is the LAST column of the left tile.
__device__ __forceinline__ void cl_neighbour(const ClGeom& g, const uint32_t lx, const uint32_t ly, const int ox, const int oy,
                                             uint32_t& which, uint32_t& li) {
  uint32_t sx = 1u, sy = 1u, nx = lx + (uint32_t)ox, ny = ly + (uint32_t)oy;
  if (ox < 0 && lx == 0u) { sx = 0u; nx = g.wl - 1u; } else if (ox > 0 && lx + 1u == g.wme) { sx = 2u; nx = 0u; }
  if (oy < 0 && ly == 0u) { sy = 0u; ny = g.hb - 1u; } else if (oy > 0 && ly + 1u == g.hme) { sy = 2u; ny = 0u; }
  which = 3u * sy + sx; li = ny * g.stride + nx;
}

// General update of local cell (lx, ly) in buffer b: Algorithm 2 with up to n_max = 4 disks per cell (cell_moves_general,
// sweep.cuh), all four slots of the 3 x 3 cells from the (distributed) shared memory.  Writes the own cell back.
template <typename P, int NS, bool DISC>
__device__ __forceinline__ void cl_update_general(const Params& p, unsigned char* const* s_base, const ClGeom& g, const uint32_t b,
                                                  const uint32_t lx, const uint32_t ly, const uint32_t cell, const uint32_t t_lo,
                                                  const uint32_t t_hi, uint32_t& amask, uint32_t& n_acc, uint32_t& n_rb,
                                                  uint32_t& n_ro) {
  using R = Real<P>;
  const P FAR = R::far_away();
  Half<P> h0[9], h1[9];
  uint32_t n = 0;
#pragma unroll
  for (int j = 0; j < 9; ++j) {
    uint32_t which, li;
    cl_neighbour(g, lx, ly, j % 3 - 1, j / 3 - 1, which, li);
    const ClTile<P> nt = cl_tile<P>(s_base[which], g.cap, b);
    const uint32_t cj = nt.cnt[li];
    h0[j] = lds_half(nt.s0, li);
    h1[j].x = R::pair(FAR, FAR); h1[j].y = h1[j].x;
    if (cj > 2u) h1[j] = lds_half(nt.s1, li);
    if (j == 4) n = cj;
  }
  Half<P> o0, o1;
  cell_moves_general<P, NS, DISC>(p, h0, h1, n, cell, t_lo, t_hi, o0, o1, amask, n_acc, n_rb, n_ro);
  if (amask != 0u) {                              // write back (Alg. 2 line 34, L234)
    const ClTile<P> me = cl_tile<P>(s_base[4], g.cap, b);
    const uint32_t li = ly * g.stride + lx;
    sts_half(me.s0, li, o0);
    if (n > 2u) sts_half(me.s1, li, o1);
  }
}
// the same as a call, for the rare cell of a w ~ sigma system with more than 2 disks somewhere in its 3 x 3 cells
template <typename P, int NS>
__device__ __noinline__ void cl_update_general_rare(const Params& p, unsigned char* const* s_base, const ClGeom g, const uint32_t b,
                                                    const uint32_t lx, const uint32_t ly, const uint32_t cell, const uint32_t t_lo,
                                                    const uint32_t t_hi, uint32_t* out4) {
  uint32_t amask, n_acc, n_rb, n_ro;
  cl_update_general<P, NS, false>(p, s_base, g, b, lx, ly, cell, t_lo, t_hi, amask, n_acc, n_rb, n_ro);
  out4[0] = amask; out4[1] = n_acc; out4[2] = n_rb; out4[3] = n_ro;
}

// ---------------------------------------------------------------------------------------------------------
// Sweeps from the state's sweep index up to t_end.  Launched as ONE cluster of p.cl_cx * p.cl_cy CTAs (grid = cluster);
// dynamic shared memory: p.cl_cap cells x cluster_cell_bytes<P>().  Reads the state from the current global buffer, writes
// it back to the SAME buffer at the end (Ctl::cur does not change) and advances Ctl::t and the grid origin.
// FAST: the w ~ sigma cell update (cells of 0/1/2 disks; the rare cell near a fuller one takes the general routine);
// otherwise the general update for every cell (any width, DISC = the disc-shaped proposal).
// ---------------------------------------------------------------------------------------------------------
template <typename P, int NS, bool DEBUG, bool DISC, bool FAST>
__global__ void __launch_bounds__(ClThreads<P>::value, 1)
k_cluster_sweeps(const __grid_constant__ Params p, const unsigned long long t_end) {
  namespace cg = cooperative_groups;
  using R = Real<P>;
  static_assert(!(FAST && DISC), "the fast update serves the square proposal only");
  cg::cluster_group cluster = cg::this_cluster();
  extern __shared__ __align__(16) unsigned char cl_smem[];
  __shared__ unsigned char* s_base[9];   // shared memory of the 3 x 3 tiles around this one (index 3 sy + sx; 4 = this tile)
  const uint32_t T = blockDim.x, tid = threadIdx.x;
  const uint32_t rank = cluster.block_rank(), cx = p.cl_cx, cy = p.cl_cy, cap = p.cl_cap;
  const uint32_t tx = rank % cx, ty = rank / cx;
  const uint32_t txm = tx == 0u ? cx - 1u : tx - 1u, tym = ty == 0u ? cy - 1u : ty - 1u;
  const uint32_t x0 = p.mx * tx / cx, x1 = p.mx * (tx + 1u) / cx, y0 = p.my * ty / cy, y1 = p.my * (ty + 1u) / cy;
  ClGeom g;
  g.wme = x1 - x0; g.hme = y1 - y0; g.stride = p.cl_stride; g.cap = cap;
  g.wl = p.mx * (txm + 1u) / cx - p.mx * txm / cx;
  g.hb = p.my * (tym + 1u) / cy - p.my * tym / cy;
  const uint32_t ncell = g.wme * g.hme;
  if (tid < 9u) {
    const uint32_t sx = tid % 3u, sy = tid / 3u;
    const uint32_t rtx = sx == 0u ? txm : sx == 1u ? tx : (tx + 1u == cx ? 0u : tx + 1u);
    const uint32_t rty = sy == 0u ? tym : sy == 1u ? ty : (ty + 1u == cy ? 0u : ty + 1u);
    s_base[tid] = cluster.map_shared_rank(cl_smem, rty * cx + rtx);
  }
  const uint32_t inv_w = small_div_magic(g.wme), Mqp = p.Mqp;
  const P FAR = R::far_away();
  const uint2 none = make_uint2(0xFFFFFFFFu, 0xFFFFFFFFu);
  Ctl* ctl = p.ctl;
  const unsigned long long t_start = ctl->t;
  const uint32_t cur = ctl->cur;
  double org_x = ctl->origin[0], org_y = ctl->origin[1];
  P* posc = reinterpret_cast<P*>(p.pos[cur]);
  uint2* idsc = reinterpret_cast<uint2*>(p.ids[cur]);
  uint8_t* cntc = p.cnt[cur];
  uint32_t b = 0;                                // the buffer that holds the state

  // ---- load this tile ----
  {
    const ClTile<P> me = cl_tile<P>(cl_smem, cap, 0u);
    for (uint32_t idx = tid; idx < ncell; idx += T) {
      const uint32_t ly = small_div(idx, inv_w), lx = idx - ly * g.wme, gx = x0 + lx, gy = y0 + ly;
      const uint32_t Qg = ((gy & 1u) << 1) | (gx & 1u), cig = (gy >> 1) * p.hx + (gx >> 1), g0 = 2u * Qg * Mqp + cig;
      const uint32_t n = cntc[Qg * Mqp + cig];
      Half<P> h1; h1.x = R::pair(FAR, FAR); h1.y = h1.x;
      uint2 j23 = none;
      if (n > 2u) { h1 = ld_half(posc, g0 + Mqp); j23 = idsc[g0 + Mqp]; }
      const uint32_t li = ly * g.stride + lx;
      sts_half(me.s0, li, ld_half(posc, g0)); sts_half(me.s1, li, h1);
      me.i01[li] = idsc[g0]; me.i23[li] = j23; me.cnt[li] = (uint8_t)n;
    }
  }
  cluster.sync();                                // every CTA of the cluster runs and has loaded its tile
  Tally tally;
  MPMC_CL_CLOCK_START();

  // The cells of checkerboard set Q in this tile: every second column from ax0, every second row from ay0.  The four sets'
  // figures are made once (a division each) and kept in shared memory.
  struct ActiveSet { uint32_t ax0, ay0, nax, na, inv_a; };
  __shared__ ActiveSet s_set[4];
  if (tid < 4u) {
    ActiveSet a;
    const uint32_t qx = tid & 1u, qy = tid >> 1;
    a.ax0 = x0 + ((x0 ^ qx) & 1u); a.ay0 = y0 + ((y0 ^ qy) & 1u);
    a.nax = a.ax0 < x1 ? (x1 - a.ax0 + 1u) >> 1 : 0u;
    const uint32_t nay = a.ay0 < y1 ? (y1 - a.ay0 + 1u) >> 1 : 0u;
    a.na = a.nax * nay; a.inv_a = small_div_magic(a.nax == 0u ? 1u : a.nax);
    s_set[tid] = a;
  }
  __syncthreads();
  auto active_set = [&](const uint32_t Q) { return s_set[Q]; };
  auto set_of = [](const Draws& d, const uint32_t k) { return k == 0u ? d.order[0] : k == 1u ? d.order[1] : k == 2u ? d.order[2] : d.order[3]; };
  // (Making a cell's draws while its thread waits at the barrier BEFORE the sub-sweep was tried: the Philox rounds already
  // run under the latency of the sub-sweep's loads, so nothing left the critical path and the barriers grew: C1 +3-7 %.)
  Draws dr = draw_sweep(p, t_start);             // Alg. 1 lines 2, 15, 16 (L64, L90-91): a pure function of (seed, t)

#pragma unroll 1
  for (unsigned long long t = t_start; t < t_end; ++t) {
    const uint32_t t_lo = (uint32_t)t, t_hi = (uint32_t)(t >> 32);
    const ClTile<P> me = cl_tile<P>(cl_smem, cap, b);
    // ---- four sub-sweeps (Alg. 1 lines 3-14, L66-88): a sub-sweep writes cells of its set only and reads, besides the
    //      own cell, cells of the other sets only, so there is nothing to order inside it ----
#pragma unroll 1
    for (uint32_t k = 0; k < 4u; ++k) {
      const ActiveSet as = active_set(set_of(dr, k));
      MPMC_CL_CLOCK_ADD(ck_shift);                 // (set-up of the sub-sweep: counted with the shift)
      for (uint32_t idx = tid; idx < as.na; idx += T) {
        const uint32_t iy = small_div(idx, as.inv_a), ix = idx - iy * as.nax;
        const uint32_t gx = as.ax0 + 2u * ix, gy = as.ay0 + 2u * iy, lx = gx - x0, ly = gy - y0;
        const uint32_t cell = gy * p.mx + gx;
        uint32_t amask, n_acc, n_rb, n_ro, n;
        if constexpr (FAST) {
          Half<P> h[9];
          uint32_t cj[9];
#pragma unroll
          for (int j = 0; j < 9; ++j) {            // counts and slot pair 0 of the 3 x 3 cells: independent loads
            uint32_t which, li;
            cl_neighbour(g, lx, ly, j % 3 - 1, j / 3 - 1, which, li);
            const ClTile<P> nt = cl_tile<P>(s_base[which], cap, b);
            cj[j] = nt.cnt[li];
            h[j] = lds_half(nt.s0, li);
          }
          n = cj[4];
          uint32_t cmax = cj[0];
#pragma unroll
          for (int j = 1; j < 9; ++j) cmax = max(cmax, cj[j]);
          if (cmax > 2u) {                         // (rare) the slot pair does not hold the whole cell
            uint32_t r4[4] = {0u, 0u, 0u, 0u};
            if (n > 0u) cl_update_general_rare<P, NS>(p, s_base, g, b, lx, ly, cell, t_lo, t_hi, r4);
            amask = r4[0]; n_acc = r4[1]; n_rb = r4[2]; n_ro = r4[3];
          } else {
            ClDraws<P, NS> pre;
            cl_draws_fast<P, NS>(p, cell, t_lo, t_hi, n == 2u, pre);
            Half<P> o;
            cl_moves_fast<P, NS>(p, h, n, pre, o, amask, n_acc, n_rb, n_ro);
            if (amask != 0u) sts_half(me.s0, ly * g.stride + lx, o);       // write back (Alg. 2 line 34, L234)
          }
        } else {
          n = me.cnt[ly * g.stride + lx];
          cl_update_general<P, NS, DISC>(p, s_base, g, b, lx, ly, cell, t_lo, t_hi, amask, n_acc, n_rb, n_ro);
        }
        tally.acc += n_acc; tally.rb += n_rb; tally.ro += n_ro;
        if (DEBUG) {
          p.mask[cell] = amask;
          if (n > 0u) atomicAdd(&ctl->digest, mix64(mix64(t) ^ (((unsigned long long)cell << 32) | amask)));
        }
      }
      MPMC_CL_CLOCK_ADD(ck_sub);
      cl_sync();
      MPMC_CL_CLOCK_ADD(ck_bar);
    }

    // ---- cell shift (Alg. 1 lines 15-17; Algorithm 4, pull form): new cell = stayers of the old own cell, then the disks
    //      that left the old neighbour in direction f; read from this buffer, written to the other one ----
    const uint32_t dir = dr.dir;
    const bool along_x = dir < 2u, positive = (dir & 1u) == 0u;
    const P w = along_x ? R::wx(p) : R::wy(p);
    const P delta = R::mul(R::mul((P)0.5, w), R::unit(dr.dist_word));   // line 15 (L90)
    const P step = positive ? -delta : delta;     // l' = l - f*delta   (L303)
    const P back = positive ? w : -w;             // entrant translation (L332)
    const int dox = along_x ? (positive ? 1 : -1) : 0, doy = along_x ? 0 : (positive ? 1 : -1);
    const ClTile<P> to = cl_tile<P>(cl_smem, cap, b ^ 1u);
    // two cells per thread and round (tiles of more cells than threads): the loads of both are in flight together
    struct ShiftIn { Half<P> a0, b0; uint2 ia, ib; uint32_t c_own, c_nb, li, ni, which; };
    auto shift_load = [&](const uint32_t idx) {
      ShiftIn in;
      const uint32_t ly = small_div(idx, inv_w), lx = idx - ly * g.wme;
      in.li = ly * g.stride + lx;
      cl_neighbour(g, lx, ly, dox, doy, in.which, in.ni);
      const ClTile<P> nt = cl_tile<P>(s_base[in.which], cap, b);
      in.c_own = me.cnt[in.li]; in.c_nb = nt.cnt[in.ni];
      in.a0 = lds_half(me.s0, in.li); in.b0 = lds_half(nt.s0, in.ni);
      in.ia = me.i01[in.li]; in.ib = nt.i01[in.ni];
      return in;
    };
    auto shift_store = [&](const ShiftIn& in) {
      Half<P> o0, o1; uint2 j01, j23;
      uint32_t nn;
      if (in.c_own <= 2u && in.c_nb <= 2u) {
        ShiftRest<P> rest;
        nn = along_x ? shift_pair<P, true>(in.a0, in.b0, in.ia, in.ib, step, back, w, o0, j01, rest)
                     : shift_pair<P, false>(in.a0, in.b0, in.ia, in.ib, step, back, w, o0, j01, rest);
        o1.x = R::pair(FAR, FAR); o1.y = o1.x; j23 = none;
        if (nn > 2u) shift_pair_rest<P>(rest, o1, j23);
      } else {
        const ClTile<P> nt = cl_tile<P>(s_base[in.which], cap, b);
        nn = shift_eight<P>(in.a0, lds_half(me.s1, in.li), in.b0, lds_half(nt.s1, in.ni), in.ia, me.i23[in.li], in.ib,
                            nt.i23[in.ni], along_x, step, back, w, o0, o1, j01, j23);
        if (nn > (uint32_t)NMAX) { atomicOr(&ctl->err, ERRBIT_OVERFLOW); nn = NMAX; }
      }
      sts_half(to.s0, in.li, o0); sts_half(to.s1, in.li, o1);
      to.i01[in.li] = j01; to.i23[in.li] = j23; to.cnt[in.li] = (uint8_t)nn;     // L280, L342
    };
    for (uint32_t idx = tid; idx < ncell; idx += 2u * T) {
      const bool second = idx + T < ncell;
      const ShiftIn in0 = shift_load(idx);
      ShiftIn in1 = in0;
      if (second) in1 = shift_load(idx + T);
      shift_store(in0);
      if (second) shift_store(in1);
    }
    b ^= 1u;
    MPMC_CL_CLOCK_ADD(ck_shift);
    cl_sync_arrive();
    {                                             // the grid origin follows the shift (X = origin + cell*w + local stays put)
      const double L = along_x ? p.Lx_eff : p.Ly_eff;
      double o = along_x ? org_x : org_y;
      o = __dadd_rn(o, positive ? (double)delta : -(double)delta);
      if (o >= L) o = __dsub_rn(o, L);
      if (o < 0.0) o = __dadd_rn(o, L);
      if (along_x) org_x = o; else org_y = o;
    }
    if (t + 1ull < t_end) dr = draw_sweep(p, t + 1ull);     // the draws of the next sweep, under the barrier
    cl_sync_wait();
    MPMC_CL_CLOCK_ADD(ck_bar);
  }

#ifdef MPMC_PHASE_CLOCKS
  if (tid == 0u && rank < CL_MAX_CTAS) {
    g_cluster_clocks[rank][0] = t_end - t_start; g_cluster_clocks[rank][1] = (unsigned long long)ck_sub;
    g_cluster_clocks[rank][2] = (unsigned long long)ck_bar; g_cluster_clocks[rank][3] = (unsigned long long)ck_shift;
    g_cluster_clocks[rank][4] = (unsigned long long)(clock64() - ck_t0);
  }
#endif
  // ---- write the tile back to the global buffer it came from; rank 0 advances the control block ----
  {
    const ClTile<P> me = cl_tile<P>(cl_smem, cap, b);
    for (uint32_t idx = tid; idx < ncell; idx += T) {
      const uint32_t ly = small_div(idx, inv_w), lx = idx - ly * g.wme, gx = x0 + lx, gy = y0 + ly, li = ly * g.stride + lx;
      const uint32_t Qg = ((gy & 1u) << 1) | (gx & 1u), cig = (gy >> 1) * p.hx + (gx >> 1), g0 = 2u * Qg * Mqp + cig;
      const uint32_t n = me.cnt[li];
      st_half(posc, g0, lds_half(me.s0, li)); idsc[g0] = me.i01[li];
      if (n > 2u) { st_half(posc, g0 + Mqp, lds_half(me.s1, li)); idsc[g0 + Mqp] = me.i23[li]; }
      cntc[Qg * Mqp + cig] = (uint8_t)n;
    }
  }
  flush_tally(p, tally);
  if (rank == 0u && tid == 0u && t_end > t_start) {
    ctl->origin[0] = org_x; ctl->origin[1] = org_y;
    ctl->path_sweeps[0] += t_end - t_start;
    ctl->t = t_end;
  }
}

}  // namespace mpmc
