// aux.cuh — kernels off the per-sweep path: cell-list build (mpmc_load_positions), unpack
// (mpmc_get_positions), contact histogram (mpmc_pressure_contact), canonical export (mpmc_debug_state).
#pragma once
#include "common.cuh"

namespace mpmc {

constexpr int AUX_THREADS = 256;

__global__ void k_reset(const __grid_constant__ Params p) {
  // clear the u32 build counters and the control block
  const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
  const uint32_t total = 4u * p.Mqp;
  for (uint32_t i = g; i < total; i += gridDim.x * blockDim.x) p.cnt32[i] = 0;
  if (g == 0) {
    Ctl* c = p.ctl;
    c->t = 0; c->cur = 0; c->err = 0; c->bar = 0; c->ticket = 0; c->pad0[0] = c->pad0[1] = 0;
    for (int i = 0; i < 4; ++i) { c->crowded[i] = 0; c->ccount[i] = 0; }
    c->origin[0] = 0.0; c->origin[1] = 0.0;
    c->digest = 0; c->path_sweeps[0] = c->path_sweeps[1] = 0;
    for (uint32_t r = 0; r < CTR_SLOTS; ++r) c->counters[r][0] = c->counters[r][1] = c->counters[r][2] = c->counters[r][3] = 0;
  }
}

// per coordinate, in double: c = floor(X / w), l = fma(-c, w, X); cast to P; one +-w step into (0, w]
template <typename P>
__device__ __forceinline__ void to_local(double X, double w_d, P w, uint32_t m, uint32_t& c, P& l) {
  using R = Real<P>;
  const double cf = floor(__ddiv_rn(X, w_d));
  const double ld = __fma_rn(-cf, w_d, X);
  long long ci = (long long)cf;
  l = (P)ld;
  if (!(l > (P)0)) { l = R::add(l, w); ci -= 1; }
  else if (l > w) { l = R::sub(l, w); ci += 1; }
  ci %= (long long)m;
  if (ci < 0) ci += (long long)m;
  c = (uint32_t)ci;
}

// Cell-list build, pass 1: one thread per disk appends to its cell with an atomic slot
// counter (arrival order); pass 2 (k_load_sort) puts each cell's slots in ascending disk index (reading A13).
template <typename P>
__global__ void __launch_bounds__(AUX_THREADS) k_load_bin(const __grid_constant__ Params p, const double* __restrict__ xy) {
  const uint32_t i = blockIdx.x * AUX_THREADS + threadIdx.x;
  if (i >= p.N) return;
  const double X = xy[2 * (size_t)i], Y = xy[2 * (size_t)i + 1];
  if (!(X >= 0.0 && X <= p.Lx_user * (1 + 1e-12) && Y >= 0.0 && Y <= p.Ly_user * (1 + 1e-12))) {
    atomicOr(&p.ctl->err, ERRBIT_RANGE);
    return;
  }
  uint32_t cx, cy; P lx, ly;
  to_local<P>(X, p.wx_d, Real<P>::wx(p), p.mx, cx, lx);
  to_local<P>(Y, p.wy_d, Real<P>::wy(p), p.my, cy, ly);
  const uint32_t Q = ((cy & 1u) << 1) | (cx & 1u);
  const uint32_t ci = (cy >> 1) * p.hx + (cx >> 1);
  const uint32_t slot = atomicAdd(&p.cnt32[Q * p.Mqp + ci], 1u);
  if (slot >= (uint32_t)NMAX) { atomicOr(&p.ctl->err, ERRBIT_OVERFLOW); return; }
  st_slot<P>(p, 0, Q, slot, ci, lx, ly);
  st_id(p, 0, Q, slot, ci, i);
}

// Pass 2: one thread per cell sorts its <= 4 (id, position) by id and writes the cell in its final form: u8
// count, slots ascending by id, empty slots of half 0 (and of half 1 when n > 2) = the far-away sentinel.
template <typename P>
__global__ void __launch_bounds__(AUX_THREADS) k_load_sort(const __grid_constant__ Params p) {
  using R = Real<P>;
  using P2 = typename R::T2;
  const uint32_t Q = blockIdx.y;
  const uint32_t ci = blockIdx.x * AUX_THREADS + threadIdx.x;
  if (ci >= p.Mq) return;
  uint32_t n = p.cnt32[Q * p.Mqp + ci];
  if (n > (uint32_t)NMAX) n = NMAX;
  cnt_plane(p, 0, Q)[ci] = (uint8_t)n;
  if (n > 2u && p.track_crowded) {               // crowded cell of the state at sweep 0 (tile.cuh)
    const uint32_t ya = div_hx(p, ci), xa = ci - ya * p.hx;
    note_crowded(p.ctl, 0u, (2u * ya + (Q >> 1)) * p.mx + (2u * xa + (Q & 1u)));
  }
  uint32_t id[NMAX]; P2 v[NMAX];
#pragma unroll
  for (int i = 0; i < NMAX; ++i) {
    id[i] = 0xFFFFFFFFu; v[i].x = R::far_away(); v[i].y = R::far_away();
    if ((uint32_t)i < n) { id[i] = ld_id(p, 0, Q, i, ci); v[i] = ld_slot<P>(p, 0, Q, i, ci); }
  }
#define MPMC_CSWAP(a, b) if (id[a] > id[b]) { uint32_t ti = id[a]; id[a] = id[b]; id[b] = ti; P2 tv = v[a]; v[a] = v[b]; v[b] = tv; }
  MPMC_CSWAP(0, 1) MPMC_CSWAP(2, 3) MPMC_CSWAP(0, 2) MPMC_CSWAP(1, 3) MPMC_CSWAP(1, 2)
#undef MPMC_CSWAP
#pragma unroll
  for (int i = 0; i < NMAX; ++i)
    if (i < 2 || n > 2u) { st_id(p, 0, Q, i, ci, id[i]); st_slot<P>(p, 0, Q, i, ci, v[i].x, v[i].y); }
}

// colour-plane location of the cell (x + ox, y + oy) with periodic wrap; |ox| < mx and |oy| < my unless `tiny`
// (a box narrower than the neighbourhood, where a cell is met at several image offsets)
__device__ __forceinline__ void locate(const Params& p, uint32_t x, uint32_t y, int ox, int oy, bool tiny, uint32_t& Q, uint32_t& ci) {
  int xn = (int)x + ox, yn = (int)y + oy;
  if (tiny) {
    xn %= (int)p.mx; yn %= (int)p.my;
    if (xn < 0) xn += (int)p.mx;
    if (yn < 0) yn += (int)p.my;
  } else {
    xn = xn < 0 ? xn + (int)p.mx : (xn >= (int)p.mx ? xn - (int)p.mx : xn);
    yn = yn < 0 ? yn + (int)p.my : (yn >= (int)p.my ? yn - (int)p.my : yn);
  }
  Q = (((uint32_t)yn & 1u) << 1) | ((uint32_t)xn & 1u);
  ci = ((uint32_t)yn >> 1) * p.hx + ((uint32_t)xn >> 1);
}

// the four slots of a cell as two slot pairs; the second pair is stored only while n > 2, otherwise it reads as sentinels
template <typename P>
__device__ __forceinline__ void ld_cell(const Params& p, const P* pos, const uint8_t* cnt, uint32_t Q, uint32_t ci,
                                        uint32_t& n, Half<P>& h0, Half<P>& h1) {
  using R = Real<P>;
  n = cnt[Q * p.Mqp + ci];
  h0 = ld_half(pos, 2u * Q * p.Mqp + ci);
  h1.x = R::pair(R::far_away(), R::far_away()); h1.y = h1.x;
  if (n > 2u) h1 = ld_half(pos, (2u * Q + 1u) * p.Mqp + ci);
}

// Reject overlapping input with the predicate of the cell update (Alg. 2 line 19, L204: |D_move - (D + s)|^2 < sigma^2
// in the working precision), evaluated from every disk's own frame: one thread per cell tests its disks against the
// 3x3 cells; a cell is two vector loads, empty slots are sentinels that never overlap.
template <typename P>
__global__ void __launch_bounds__(AUX_THREADS) k_load_check(const __grid_constant__ Params p) {
  using R = Real<P>;
  const uint32_t Q = blockIdx.y;
  const uint32_t ci = blockIdx.x * AUX_THREADS + threadIdx.x;
  if (ci >= p.Mq) return;
  const P* pos = reinterpret_cast<const P*>(p.pos[0]);
  const uint8_t* cnt = p.cnt[0];
  uint32_t n; Half<P> a0, a1;
  ld_cell<P>(p, pos, cnt, Q, ci, n, a0, a1);
  if (n == 0) return;
  const P ax[NMAX] = {a0.x.x, a0.x.y, a1.x.x, a1.x.y}, ay[NMAX] = {a0.y.x, a0.y.y, a1.y.x, a1.y.y};
  const uint32_t ya = div_hx(p, ci), xa = ci - ya * p.hx;
  const uint32_t x = 2u * xa + (Q & 1u), y = 2u * ya + (Q >> 1);
  const P wx = R::wx(p), wy = R::wy(p), sigma2 = R::sigma2(p);
  const bool tiny = p.mx < 3u || p.my < 3u;
  bool bad = false;
  for (int oy = -1; oy <= 1; ++oy)
    for (int ox = -1; ox <= 1; ++ox) {
      uint32_t qn, cn, nj; Half<P> b0, b1;
      locate(p, x, y, ox, oy, tiny, qn, cn);
      ld_cell<P>(p, pos, cnt, qn, cn, nj, b0, b1);
      const P sx = R::mul((P)ox, wx), sy = R::mul((P)oy, wy);          // s = (ox wx, oy wy)  (L154, L196)
      const P bx[NMAX] = {b0.x.x, b0.x.y, b1.x.x, b1.x.y}, by[NMAX] = {b0.y.x, b0.y.y, b1.y.x, b1.y.y};
#pragma unroll
      for (int j = 0; j < NMAX; ++j) {
        if (j >= 2 && nj <= 2u) break;
        const P qx = R::add(bx[j], sx), qy = R::add(by[j], sy);         // a sentinel stays far away
#pragma unroll
        for (int k = 0; k < NMAX; ++k) {
          if (k >= 2 && n <= 2u) break;
          if (ox == 0 && oy == 0 && j == k) continue;                   // line 17 (L201)
          const P Dx = R::sub(ax[k], qx), Dy = R::sub(ay[k], qy);
          bad |= (uint32_t)k < n && R::fma(Dx, Dx, R::mul(Dy, Dy)) < sigma2;
        }
      }
    }
  if (bad) atomicOr(&p.ctl->err, ERRBIT_OVERLAP);
}

// Unpack: X = wrap(origin + cell*w + local) into [0, L_eff), written at the disk's index.
template <typename P>
__global__ void __launch_bounds__(AUX_THREADS) k_unpack(const __grid_constant__ Params p, double* __restrict__ xy) {
  using P2 = typename Real<P>::T2;
  const uint32_t Q = blockIdx.y;
  const uint32_t ci = blockIdx.x * AUX_THREADS + threadIdx.x;
  if (ci >= p.Mq) return;
  const uint32_t cur = p.ctl->cur;
  const uint32_t n = cnt_plane(p, cur, Q)[ci];
  const uint32_t ya = div_hx(p, ci), xa = ci - ya * p.hx;
  const double bx = __fma_rn((double)(2u * xa + (Q & 1u)), p.wx_d, p.ctl->origin[0]);
  const double by = __fma_rn((double)(2u * ya + (Q >> 1)), p.wy_d, p.ctl->origin[1]);
  for (uint32_t i = 0; i < n; ++i) {
    const P2 v = ld_slot<P>(p, cur, Q, i, ci);
    double X = __dadd_rn(bx, (double)v.x), Y = __dadd_rn(by, (double)v.y);
    if (X >= p.Lx_eff) X = __dsub_rn(X, p.Lx_eff);
    if (Y >= p.Ly_eff) Y = __dsub_rn(Y, p.Ly_eff);
    const uint32_t who = ld_id(p, cur, Q, i, ci);
    reinterpret_cast<double2*>(xy)[who] = make_double2(X, Y);
  }
}

// Canonical export for mpmc_debug_state: cell c = y*mx + x.
template <typename P>
__global__ void __launch_bounds__(AUX_THREADS) k_export(const __grid_constant__ Params p, uint32_t* counts, P* slab, uint32_t* ids) {
  using P2 = typename Real<P>::T2;
  const uint32_t Q = blockIdx.y;
  const uint32_t ci = blockIdx.x * AUX_THREADS + threadIdx.x;
  if (ci >= p.Mq) return;
  const uint32_t cur = p.ctl->cur;
  const uint32_t n = cnt_plane(p, cur, Q)[ci];
  const uint32_t ya = div_hx(p, ci), xa = ci - ya * p.hx;
  const size_t c = (size_t)(2u * ya + (Q >> 1)) * p.mx + (2u * xa + (Q & 1u));
  if (counts) counts[c] = n;
  for (uint32_t i = 0; i < (uint32_t)NMAX; ++i) {
    P2 v; v.x = 0; v.y = 0; uint32_t id = 0xFFFFFFFFu;
    if (i < n) { v = ld_slot<P>(p, cur, Q, i, ci); id = ld_id(p, cur, Q, i, ci); }
    if (slab) { slab[(c * NMAX + i) * 2] = v.x; slab[(c * NMAX + i) * 2 + 1] = v.y; }
    if (ids) ids[c * NMAX + i] = id;
  }
}

// Pair-distance histogram near contact (eq. 5): unordered pairs with r in [sigma, sigma + nbins*dr),
// the distance in double from the stored locals exactly as the oracle forms it, neighbourhood radius Rc cells (reading
// A12).  Two stages, so that the double-precision square root and division run on full warps of pairs that matter:
//   1. one thread per cell walks the HALF neighbourhood (the cell itself, then the offsets with oy > 0, or oy = 0 and
//      ox > 0: every unordered pair of cell images once; offsets whose cells cannot hold a pair closer than rmax are
//      skipped: bit mask `keep` from the host) and tests its slots against the neighbour's in fp32 with a safety margin
//      (packed fp32x2: both own slots at once; a cell is one vector load, empty slots are sentinels).  A
//      (cell, neighbour) with a candidate goes into the warp's queue in shared memory (ballot + prefix count).
//   2. whenever 32 records are queued the warp takes one each: D = (b + o w) - a in double seen from the disk with the
//      LOWER index (the oracle counts a pair from that disk's frame; in fp64 the rounding depends on the frame),
//      r = sqrt(Dx Dx + Dy Dy) without FMA, bin = floor((r - sigma) / dr), shared-memory histogram.
// This kernel serves any radius; k_contact_hist_tile below is the fast path for radius 1 and 2.
// Per-block histograms are flushed with 64-bit atomics.
constexpr int HIST_THREADS = 256;
constexpr int HIST_QUEUE = 64;             // records per warp queue: fewer than 32 left over + at most 32 new ones

struct HistQueue { uint32_t own[HIST_QUEUE], nb[HIST_QUEUE], code[HIST_QUEUE]; };

// offsets of the half neighbourhood in visiting order: e = 0 is the cell itself, then (1..Rc, 0), then rows oy = 1..Rc
__host__ __device__ inline int hist_offset_index(int ox, int oy, int Rc) { return oy == 0 ? ox : Rc + (oy - 1) * (2 * Rc + 1) + (ox + Rc) + 1; }

template <typename P>
__device__ __forceinline__ void hist_pairs_exact(const Params& p, const P* pos, const uint32_t* ids, const uint32_t own_g,
                                                 const uint32_t nb_g, const uint32_t code, const double dr,
                                                 const uint32_t nbins, const double rmax2, uint32_t* sh_hist) {
  const int ox = (int)(code & 0xFFu) - 128, oy = (int)((code >> 8) & 0xFFu) - 128;
  uint32_t cm = code >> 16;                                    // bit 4 i + j: own slot i against the neighbour's slot j
  const double sx = __dmul_rn((double)ox, p.wx_d), sy = __dmul_rn((double)oy, p.wy_d);
  while (cm != 0u) {
    const uint32_t b = (uint32_t)__ffs((int)cm) - 1u;
    cm &= cm - 1u;
    const uint32_t i = b >> 2, j = b & 3u;
    const size_t ea = (size_t)own_g + (i >> 1) * p.Mqp, eb = (size_t)nb_g + (j >> 1) * p.Mqp;
    const uint32_t ida = ids[ea * 2 + (i & 1u)], idb = ids[eb * 2 + (j & 1u)];
    const double ax = (double)pos[ea * 4 + (i & 1u)], ay = (double)pos[ea * 4 + 2 + (i & 1u)];
    const double bx = (double)pos[eb * 4 + (j & 1u)], by = (double)pos[eb * 4 + 2 + (j & 1u)];
    if (ida == idb) continue;                                  // a disk and its own periodic image (boxes of a few cells)
    double Dx, Dy;
    if (ida < idb) {                                           // from a's frame: b sits at offset (ox, oy)
      Dx = __dsub_rn(__dadd_rn(bx, sx), ax); Dy = __dsub_rn(__dadd_rn(by, sy), ay);
    } else {                                                   // from b's frame: a sits at offset (-ox, -oy)
      Dx = __dsub_rn(__dadd_rn(ax, -sx), bx); Dy = __dsub_rn(__dadd_rn(ay, -sy), by);
    }
    const double r2 = __dadd_rn(__dmul_rn(Dx, Dx), __dmul_rn(Dy, Dy));
    if (!(r2 < rmax2)) continue;                               // beyond the last bin by a margin far above the rounding
    const double r = sqrt(r2);
    const double bin = floor(__ddiv_rn(__dsub_rn(r, p.sigma_d), dr));
    if (bin >= 0.0 && bin < (double)nbins) atomicAdd(&sh_hist[(uint32_t)bin], 1u);
  }
}

template <typename P, int RC>
__global__ void __launch_bounds__(HIST_THREADS) k_contact_hist(const __grid_constant__ Params p, const double dr,
                                                               const uint32_t nbins, const int Rc_arg, const double rmax,
                                                               const unsigned long long keep, unsigned long long* out) {
  using F = Real<float>;
  extern __shared__ uint32_t sh_hist[];
  __shared__ HistQueue s_queue[HIST_THREADS / 32];
  for (uint32_t b = threadIdx.x; b < nbins; b += HIST_THREADS) sh_hist[b] = 0;
  __syncthreads();
  const int Rc = RC > 0 ? RC : Rc_arg;
  const uint32_t lane = threadIdx.x & 31u;
  HistQueue& q = s_queue[threadIdx.x >> 5];
  const uint32_t Q = blockIdx.y;
  const uint32_t ci_raw = blockIdx.x * HIST_THREADS + threadIdx.x;
  const bool valid = ci_raw < p.Mq;
  const uint32_t ci = valid ? ci_raw : p.Mq - 1u;                 // clamped: every lane takes part in the warp votes
  const uint32_t cur = p.ctl->cur;
  const P* pos = reinterpret_cast<const P*>(p.pos[cur]);
  const uint8_t* cnt = p.cnt[cur];
  const uint32_t* ids = p.ids[cur];
  const float FARF = 1.0e18f;
  // the fp32 image of a slot coordinate (the sentinel of an fp64 slot would convert to infinity)
  auto f = [&](P v) { const float r = (float)v; return sizeof(P) == 4 ? r : fminf(r, FARF); };
  // own cell; an empty own slot is moved to -FAR (an empty neighbour slot sits at +FAR): no pair with an empty slot
  // ever passes the filter
  uint32_t n; Half<P> a0, a1;
  ld_cell<P>(p, pos, cnt, Q, ci, n, a0, a1);
  if (!valid) n = 0u;
  const bool own4 = n > 2u;
  const F::Pair nax01 = F::pair(n > 0u ? -f(a0.x.x) : FARF, n > 1u ? -f(a0.x.y) : FARF);      // negated own slots 0, 1
  const F::Pair nay01 = F::pair(-f(a0.y.x), -f(a0.y.y));
  const F::Pair nax23 = F::pair(n > 2u ? -f(a1.x.x) : FARF, n > 3u ? -f(a1.x.y) : FARF);
  const F::Pair nay23 = F::pair(-f(a1.y.x), -f(a1.y.y));
  const uint32_t ya = div_hx(p, ci), xa = ci - ya * p.hx;
  const uint32_t x = 2u * xa + (Q & 1u), y = 2u * ya + (Q >> 1);
  const uint32_t own_g = 2u * Q * p.Mqp + ci;
  const uint32_t own_rows = 0x1111u & ((1u << (4u * n)) - 1u);    // bit 4 i for every own slot i < n
  const bool tiny = (uint32_t)Rc >= p.mx || (uint32_t)Rc >= p.my;
  // fp32 pre-filter: r^2 below (rmax (1 + 1e-3))^2; the fp32 images are off by a few 1e-7 at most
  const float thr2 = (float)(rmax * rmax * 1.002);
  const float wxf = (float)p.wx_d, wyf = (float)p.wy_d;
  const double rmax2 = rmax * rmax * 1.000001;
  uint32_t qn = 0;                                                // records in the warp's queue (warp-uniform)

  // squared fp32 distances of own slots (i, i + 1) to the point (bx, by): one packed evaluation
  auto r2_pair = [&](const F::Pair nax, const F::Pair nay, const float bx, const float by) {
    const F::Pair Dx = F::padd(F::pair(bx, bx), nax), Dy = F::padd(F::pair(by, by), nay);
    return F::pfma(Dx, Dx, F::pmul(Dy, Dy));
  };
  auto drain = [&]() {                                            // a full warp of records
    hist_pairs_exact<P>(p, pos, ids, q.own[lane], q.nb[lane], q.code[lane], dr, nbins, rmax2, sh_hist);
    const uint32_t o = q.own[lane + 32u], b = q.nb[lane + 32u], c = q.code[lane + 32u];
    __syncwarp();
    if (lane + 32u < qn) { q.own[lane] = o; q.nb[lane] = b; q.code[lane] = c; }   // the rest moves to the front
    qn -= 32u;
    __syncwarp();
  };
  auto enqueue = [&](const bool has, const uint32_t nb_g, const int ox, const int oy, const uint32_t cm) {
    const uint32_t m = __ballot_sync(0xFFFFFFFFu, has);
    if (m == 0u) return;
    if (has) {
      const uint32_t at = qn + __popc(m & ((1u << lane) - 1u));
      q.own[at] = own_g; q.nb[at] = nb_g;
      q.code[at] = (uint32_t)(ox + 128) | ((uint32_t)(oy + 128) << 8) | (cm << 16);
    }
    qn += __popc(m);
    __syncwarp();
    if (qn >= 32u) drain();
  };
  auto visit = [&](const int ox, const int oy) {
    uint32_t qc, cn, nj; Half<P> b0, b1;
    locate(p, x, y, ox, oy, tiny, qc, cn);
    ld_cell<P>(p, pos, cnt, qc, cn, nj, b0, b1);
    const float sx = (float)ox * wxf, sy = (float)oy * wyf;
    const float bx0 = f(b0.x.x) + sx, bx1 = f(b0.x.y) + sx, by0 = f(b0.y.x) + sy, by1 = f(b0.y.y) + sy;
    const F::Pair r0 = r2_pair(nax01, nay01, bx0, by0), r1 = r2_pair(nax01, nay01, bx1, by1);
    float rmin = fminf(F::min3(r0.x, r0.y, r1.x), r1.y);
    if (__any_sync(0xFFFFFFFFu, own4 || nj > 2u)) {               // slots 2, 3 somewhere in the warp (rare at w ~ sigma)
      const float bx2 = f(b1.x.x) + sx, bx3 = f(b1.x.y) + sx, by2 = f(b1.y.x) + sy, by3 = f(b1.y.y) + sy;
      const F::Pair r2 = r2_pair(nax01, nay01, bx2, by2), r3 = r2_pair(nax01, nay01, bx3, by3);
      const F::Pair r4 = r2_pair(nax23, nay23, bx0, by0), r5 = r2_pair(nax23, nay23, bx1, by1);
      const F::Pair r6 = r2_pair(nax23, nay23, bx2, by2), r7 = r2_pair(nax23, nay23, bx3, by3);
      rmin = fminf(rmin, fminf(fminf(F::min3(r2.x, r2.y, r3.x), F::min3(r3.y, r4.x, r4.y)),
                               fminf(F::min3(r5.x, r5.y, r6.x), F::min3(r6.y, r7.x, r7.y))));
    }
    // every pair of occupied slots goes to stage 2, which filters exactly
    enqueue(rmin < thr2, 2u * qc * p.Mqp + cn, ox, oy, own_rows * ((1u << nj) - 1u));
  };

  // the pairs inside the cell, each once (j > i)
  {
    const F::Pair r0 = r2_pair(nax01, nay01, -nax01.y, -nay01.y);                    // r0.x: slots (0, 1)
    float rmin = n >= 2u ? r0.x : FARF;
    if (__any_sync(0xFFFFFFFFu, own4)) {
      const F::Pair r2 = r2_pair(nax01, nay01, -nax23.x, -nay23.x), r3 = r2_pair(nax01, nay01, -nax23.y, -nay23.y);
      const F::Pair r6 = r2_pair(nax23, nay23, -nax23.y, -nay23.y);                  // r6.x: slots (2, 3)
      if (own4) rmin = fminf(fminf(rmin, r6.x), fminf(fminf(r2.x, r2.y), fminf(r3.x, r3.y)));
    }
    enqueue(rmin < thr2, own_g, 0, 0, own_rows * ((1u << n) - 1u) & 0x08CEu);
  }
  if (RC > 0) {
#pragma unroll
    for (int oy = 0; oy <= RC; ++oy)
#pragma unroll
      for (int ox = -RC; ox <= RC; ++ox) {
        if (oy == 0 && ox <= 0) continue;
        if ((keep >> hist_offset_index(ox, oy, RC)) & 1ull) visit(ox, oy);
      }
  } else {
    for (int oy = 0; oy <= Rc; ++oy)
      for (int ox = (oy == 0 ? 1 : -Rc); ox <= Rc; ++ox) {
        // the nearest points of the two cells are (|o| - 1) w apart along each axis: skip offsets out of reach
        const int gi = (ox < 0 ? -ox : ox) - 1, gj = oy - 1;
        const double gx = (double)(gi > 0 ? gi : 0) * p.wx_d, gy = (double)(gj > 0 ? gj : 0) * p.wy_d;
        if (gx * gx + gy * gy < rmax2) visit(ox, oy);
      }
  }
  if (lane < qn) hist_pairs_exact<P>(p, pos, ids, q.own[lane], q.nb[lane], q.code[lane], dr, nbins, rmax2, sh_hist);
  __syncthreads();
  for (uint32_t b = threadIdx.x; b < nbins; b += HIST_THREADS)
    if (sh_hist[b]) atomicAdd(&out[b], (unsigned long long)sh_hist[b]);
}

// ---------------------------------------------------------------------------------------------------------
// The same histogram for neighbourhood radius RC = 1 or 2 (every configuration whose bins end below 2 cell widths: all
// BASELINE configs and the paper's estimator, L382) with the cells of a tile staged in shared memory: a block owns
// HT_W x HT_H cells, a warp a row at a time (its queue of candidates carries over from row to row); the tile plus a halo of RC cells to the left, to the right and
// above is loaded once (fp32 images of the slots as float4 {x0, x1, y0, y1}, the global slot-pair index and the count
// of every cell), so a neighbour is ONE shared-memory vector load at a compile-time offset from the own cell and
// stage 1 is ~25 instructions per neighbour instead of ~100.  Stage 2 is hist_pairs_exact, as above.
// ---------------------------------------------------------------------------------------------------------
constexpr int HT_W = 32, HT_H = 16, HT_THREADS = 256;      // a warp per row, HT_H / 8 rows per warp

template <typename P, int RC>
__global__ void __launch_bounds__(HT_THREADS) k_contact_hist_tile(const __grid_constant__ Params p, const double dr,
                                                                   const uint32_t nbins, const double rmax,
                                                                   const unsigned long long keep, unsigned long long* out) {
  using F = Real<float>;
  constexpr int CW = HT_W + 2 * RC, CH = HT_H + RC, NT = HT_THREADS;
  extern __shared__ uint32_t sh_hist[];
  __shared__ float4 s01[CH * CW], s23[CH * CW];      // fp32 images of slots 0, 1 and 2, 3 (empty slot: +FAR)
  __shared__ uint32_t sg[CH * CW];                   // global index of the cell's slot pair 0
  __shared__ uint8_t sn[CH * CW];                    // its count
  __shared__ uint32_t q_pair[NT / 32][96], q_code[NT / 32][96];    // per warp: fewer than 32 records left over + at most 64 new ones
  const uint32_t tid = threadIdx.x, lane = tid & 31u, ty = tid >> 5;
  for (uint32_t b = tid; b < nbins; b += NT) sh_hist[b] = 0;
  const uint32_t cur = p.ctl->cur;
  const P* pos = reinterpret_cast<const P*>(p.pos[cur]);
  const uint8_t* cnt = p.cnt[cur];
  const uint32_t* ids = p.ids[cur];
  const float FARF = 1.0e18f;
  auto f = [&](P v) { const float r = (float)v; return sizeof(P) == 4 ? r : fminf(r, FARF); };
  const uint32_t x0 = blockIdx.x * HT_W, y0 = blockIdx.y * HT_H;
  // ---- load the tile and its halo (periodic wrap; a box narrower than the region is met at several images) ----
  bool any4 = false;
  for (uint32_t idx = tid; idx < (uint32_t)(CH * CW); idx += NT) {
    const uint32_t r = idx / CW, c = idx - r * CW;
    const uint32_t gx = (x0 + p.mx * (uint32_t)RC + c - (uint32_t)RC) % p.mx, gy = (y0 + r) % p.my;
    const uint32_t Qc = ((gy & 1u) << 1) | (gx & 1u), cc = (gy >> 1) * p.hx + (gx >> 1);
    uint32_t n; Half<P> h0, h1;
    ld_cell<P>(p, pos, cnt, Qc, cc, n, h0, h1);
    s01[idx] = make_float4(n > 0u ? f(h0.x.x) : FARF, n > 1u ? f(h0.x.y) : FARF, f(h0.y.x), f(h0.y.y));
    s23[idx] = make_float4(n > 2u ? f(h1.x.x) : FARF, n > 3u ? f(h1.x.y) : FARF, f(h1.y.x), f(h1.y.y));
    sg[idx] = 2u * Qc * p.Mqp + cc;
    sn[idx] = (uint8_t)n;
    any4 |= n > 2u;
  }
  const bool crowded = __syncthreads_or(any4) != 0;   // slots 2, 3 in use somewhere in the region (rare at w ~ sigma)

  // ---- stage 1: one thread per cell of a tile row, the warps take the rows in turn ----
  const float thr2 = (float)(rmax * rmax * 1.002);                // fp32 pre-filter with a margin of 1e-3 in r
  const float wxf = (float)p.wx_d, wyf = (float)p.wy_d;
  const double rmax2 = rmax * rmax * 1.000001;
  uint32_t qn = 0;
  uint32_t* qp = q_pair[ty];
  uint32_t* qc = q_code[ty];
  // squared fp32 distances of the own slots (i, i + 1) to the two points of B (packed: both points at once)
  auto r2_two = [&](const float ax_neg, const float ay_neg, const F::Pair Bx, const F::Pair By) {
    const F::Pair Dx = F::padd(Bx, F::pair(ax_neg, ax_neg)), Dy = F::padd(By, F::pair(ay_neg, ay_neg));
    return F::pfma(Dx, Dx, F::pmul(Dy, Dy));
  };
  auto exact = [&](const uint32_t pair, const uint32_t code) {
    hist_pairs_exact<P>(p, pos, ids, sg[pair >> 16], sg[pair & 0xFFFFu], code, dr, nbins, rmax2, sh_hist);
  };
  // A thread owns TWO cells, one in each of its warp's rows (row, row + NT / 32): the per-offset work of a visit (the
  // neighbour's index offset, its translation, the loop and the queue bookkeeping) is shared by both, and their
  // arithmetic interleaves.
  constexpr uint32_t NR = 2u, WARPS = NT / 32;
  static_assert(HT_H % (NR * WARPS) == 0, "rows per warp");
  struct OwnCell { uint32_t idx, rows; bool own4; F::Pair nax01, nay01, nax23, nay23; };
  auto drain = [&]() {                                            // a full warp of records
    exact(qp[lane], qc[lane]);
    uint32_t a[2], c[2];
#pragma unroll
    for (uint32_t j = 0; j < 2u; ++j) { a[j] = qp[lane + 32u * (j + 1u)]; c[j] = qc[lane + 32u * (j + 1u)]; }
    __syncwarp();
#pragma unroll
    for (uint32_t j = 0; j < 2u; ++j)
      if (lane + 32u * (j + 1u) < qn) { qp[lane + 32u * j] = a[j]; qc[lane + 32u * j] = c[j]; }   // the rest moves to the front
    qn -= 32u;
    __syncwarp();
  };
#pragma unroll 1
  for (uint32_t row0 = ty; row0 < (uint32_t)HT_H; row0 += NR * WARPS) {
    OwnCell o[NR];
#pragma unroll
    for (uint32_t c = 0; c < NR; ++c) {
      const uint32_t row = row0 + c * WARPS;
      const uint32_t own = row * CW + lane + RC;
      const bool valid = x0 + lane < p.mx && y0 + row < p.my;
      const uint32_t n = valid ? sn[own] : 0u;
      const float4 a01 = s01[own], a23 = s23[own];
      // negated own slots; an empty own slot goes to -FAR (empty neighbour slots sit at +FAR): no pair with an empty
      // slot ever passes the filter
      o[c].idx = own; o[c].own4 = n > 2u;
      o[c].nax01 = F::pair(n > 0u ? -a01.x : FARF, n > 1u ? -a01.y : FARF); o[c].nay01 = F::pair(-a01.z, -a01.w);
      o[c].nax23 = F::pair(n > 2u ? -a23.x : FARF, n > 3u ? -a23.y : FARF); o[c].nay23 = F::pair(-a23.z, -a23.w);
      o[c].rows = 0x1111u & ((1u << (4u * n)) - 1u);              // bit 4 i for every own slot i < n
    }
    // both cells' candidates of one offset go into the queue in one round (at most 64 new records on top of < 32)
    auto enqueue = [&](const bool (&has)[NR], const uint32_t (&nb)[NR], const int ox, const int oy, const bool self) {
      uint32_t m[NR];
#pragma unroll
      for (uint32_t c = 0; c < NR; ++c) m[c] = __ballot_sync(0xFFFFFFFFu, has[c]);
      if ((m[0] | m[1]) == 0u) return;
      uint32_t at = qn + __popc(m[0] & ((1u << lane) - 1u));
#pragma unroll
      for (uint32_t c = 0; c < NR; ++c) {
        if (has[c]) {
          uint32_t cm = o[c].rows * ((1u << sn[nb[c]]) - 1u);     // every pair of occupied slots; stage 2 filters exactly
          if (self) cm &= 0x08CEu;                                // inside a cell: each pair once (j > i)
          qp[at] = (o[c].idx << 16) | nb[c];
          qc[at] = (uint32_t)(ox + 128) | ((uint32_t)(oy + 128) << 8) | (cm << 16);
        }
        if (c == 0u) at = qn + __popc(m[0]) + __popc(m[1] & ((1u << lane) - 1u));
      }
      qn += __popc(m[0]) + __popc(m[1]);
      __syncwarp();
      while (qn >= 32u) drain();
    };
    auto visit = [&](const int ox, const int oy) {
      const int dnb = oy * CW + ox;
      const float sx = (float)ox * wxf, sy = (float)oy * wyf;
      bool has[NR]; uint32_t nb[NR];
#pragma unroll
      for (uint32_t c = 0; c < NR; ++c) {
        nb[c] = (uint32_t)((int)o[c].idx + dnb);
        const float4 b01 = s01[nb[c]];
        const F::Pair Bx = F::padd(F::pair(b01.x, b01.y), F::pair(sx, sx)), By = F::padd(F::pair(b01.z, b01.w), F::pair(sy, sy));
        const F::Pair r0 = r2_two(o[c].nax01.x, o[c].nay01.x, Bx, By), r1 = r2_two(o[c].nax01.y, o[c].nay01.y, Bx, By);
        float rmin = fminf(F::min3(r0.x, r0.y, r1.x), r1.y);
        if (crowded) {
          const float4 b23 = s23[nb[c]];
          const F::Pair Cx = F::padd(F::pair(b23.x, b23.y), F::pair(sx, sx)), Cy = F::padd(F::pair(b23.z, b23.w), F::pair(sy, sy));
          const F::Pair r2 = r2_two(o[c].nax01.x, o[c].nay01.x, Cx, Cy), r3 = r2_two(o[c].nax01.y, o[c].nay01.y, Cx, Cy);
          const F::Pair r4 = r2_two(o[c].nax23.x, o[c].nay23.x, Bx, By), r5 = r2_two(o[c].nax23.y, o[c].nay23.y, Bx, By);
          const F::Pair r6 = r2_two(o[c].nax23.x, o[c].nay23.x, Cx, Cy), r7 = r2_two(o[c].nax23.y, o[c].nay23.y, Cx, Cy);
          rmin = fminf(rmin, fminf(fminf(F::min3(r2.x, r2.y, r3.x), F::min3(r3.y, r4.x, r4.y)),
                                   fminf(F::min3(r5.x, r5.y, r6.x), F::min3(r6.y, r7.x, r7.y))));
        }
        has[c] = rmin < thr2;
      }
      enqueue(has, nb, ox, oy, false);
    };

    // the pairs inside the cells, each once
    {
      bool has[NR]; uint32_t nb[NR];
#pragma unroll
      for (uint32_t c = 0; c < NR; ++c) {
        nb[c] = o[c].idx;
        // own slots 1, 2, 3 as points (un-negated); an empty one sits at -FAR
        const F::Pair Bx = F::pair(-o[c].nax01.y, -o[c].nax23.x), By = F::pair(-o[c].nay01.y, -o[c].nay23.x);
        const F::Pair r0 = r2_two(o[c].nax01.x, o[c].nay01.x, Bx, By);                     // (0, 1), (0, 2)
        float rmin = r0.x;                                        // huge unless slots 0 and 1 are both occupied
        if (crowded) {
          const F::Pair r1 = r2_two(o[c].nax01.y, o[c].nay01.y, Bx, By);                   // (1, 1) = 0, (1, 2)
          const F::Pair Cx = F::pair(-o[c].nax23.y, -o[c].nax23.y), Cy = F::pair(-o[c].nay23.y, -o[c].nay23.y);   // own slot 3
          const F::Pair r3 = r2_two(o[c].nax01.x, o[c].nay01.x, Cx, Cy), r4 = r2_two(o[c].nax01.y, o[c].nay01.y, Cx, Cy),
                        r5 = r2_two(o[c].nax23.x, o[c].nay23.x, Cx, Cy);
          if (o[c].own4) rmin = fminf(fminf(fminf(rmin, r0.y), fminf(r1.y, r3.x)), fminf(r4.x, r5.x));
        }
        has[c] = rmin < thr2 && (o[c].rows & 0x10u) != 0u;         // (at least two disks in the cell)
      }
      enqueue(has, nb, 0, 0, true);
    }
    // (rolled: one copy of the visit keeps the loop inside the instruction cache; the unrolled form stalled 30 % of its
    // cycles on instruction fetch)
#pragma unroll 1
    for (int oy = 0; oy <= RC; ++oy)
#pragma unroll 1
      for (int ox = (oy == 0 ? 1 : -RC); ox <= RC; ++ox)
        if ((keep >> hist_offset_index(ox, oy, RC)) & 1ull) visit(ox, oy);
  }
  if (lane < qn) exact(qp[lane], qc[lane]);
  __syncthreads();
  for (uint32_t b = tid; b < nbins; b += NT)
    if (sh_hist[b]) atomicAdd(&out[b], (unsigned long long)sh_hist[b]);
}

__global__ void k_philox_test(const uint32_t* __restrict__ ctr, uint32_t k0, uint32_t k1, uint32_t* __restrict__ out, uint32_t n) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  uint32_t o[4];
  philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], k0, k1, o);
  out[4 * i] = o[0]; out[4 * i + 1] = o[1]; out[4 * i + 2] = o[2]; out[4 * i + 3] = o[3];
}

}  // namespace mpmc
