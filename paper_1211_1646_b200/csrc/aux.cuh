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

// colour-plane location of the cell (x + ox, y + oy) with periodic wrap, for arbitrary small offsets
__device__ __forceinline__ void locate(const Params& p, uint32_t x, uint32_t y, int ox, int oy, uint32_t& Q, uint32_t& ci) {
  long long xn = ((long long)x + ox) % (long long)p.mx; if (xn < 0) xn += p.mx;
  long long yn = ((long long)y + oy) % (long long)p.my; if (yn < 0) yn += p.my;
  Q = (((uint32_t)yn & 1u) << 1) | ((uint32_t)xn & 1u);
  ci = ((uint32_t)yn >> 1) * p.hx + ((uint32_t)xn >> 1);
}

// Reject overlapping input with the predicate of the cell update, evaluated from every disk's own frame.
template <typename P>
__global__ void __launch_bounds__(AUX_THREADS) k_load_check(const __grid_constant__ Params p) {
  using R = Real<P>;
  using P2 = typename R::T2;
  const uint32_t Q = blockIdx.y;
  const uint32_t ci = blockIdx.x * AUX_THREADS + threadIdx.x;
  if (ci >= p.Mq) return;
  const uint32_t n = cnt_plane(p, 0, Q)[ci];
  if (n == 0) return;
  const uint32_t ya = div_hx(p, ci), xa = ci - ya * p.hx;
  const uint32_t x = 2u * xa + (Q & 1u), y = 2u * ya + (Q >> 1);
  const P wx = R::wx(p), wy = R::wy(p), sigma2 = R::sigma2(p);
  bool bad = false;
  for (uint32_t k = 0; k < n; ++k) {
    const P2 m = ld_slot<P>(p, 0, Q, k, ci);
    for (int oy = -1; oy <= 1; ++oy)
      for (int ox = -1; ox <= 1; ++ox) {
        uint32_t qn, cn;
        locate(p, x, y, ox, oy, qn, cn);
        const uint32_t nj = cnt_plane(p, 0, qn)[cn];
        const P sx = R::mul((P)ox, wx), sy = R::mul((P)oy, wy);
        for (uint32_t j = 0; j < nj; ++j) {
          if (ox == 0 && oy == 0 && j == k) continue;
          const P2 v = ld_slot<P>(p, 0, qn, j, cn);
          const P Dx = R::sub(m.x, R::add(v.x, sx)), Dy = R::sub(m.y, R::add(v.y, sy));
          if (R::fma(Dx, Dx, R::mul(Dy, Dy)) < sigma2) bad = true;
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

// Pair-distance histogram near contact: unordered pairs with r in [sigma, sigma + nbins*dr),
// all arithmetic in double from the stored locals, neighbourhood radius Rc cells (reading A12).  One thread
// per cell; per-block histogram in shared memory, flushed with 64-bit atomics.
template <typename P>
__global__ void __launch_bounds__(AUX_THREADS) k_contact_hist(const __grid_constant__ Params p, const double dr,
                                                              const uint32_t nbins, const int Rc) {
  using P2 = typename Real<P>::T2;
  extern __shared__ uint32_t sh_hist[];
  for (uint32_t b = threadIdx.x; b < nbins; b += AUX_THREADS) sh_hist[b] = 0;
  __syncthreads();
  const uint32_t Q = blockIdx.y;
  const uint32_t ci = blockIdx.x * AUX_THREADS + threadIdx.x;
  if (ci < p.Mq) {
    const uint32_t cur = p.ctl->cur;
    const uint32_t n = cnt_plane(p, cur, Q)[ci];
    const uint32_t ya = div_hx(p, ci), xa = ci - ya * p.hx;
    const uint32_t x = 2u * xa + (Q & 1u), y = 2u * ya + (Q >> 1);
    for (uint32_t i = 0; i < n; ++i) {
      const P2 a = ld_slot<P>(p, cur, Q, i, ci);
      const uint32_t ida = ld_id(p, cur, Q, i, ci);
      for (int oy = -Rc; oy <= Rc; ++oy)
        for (int ox = -Rc; ox <= Rc; ++ox) {
          uint32_t qn, cn;
          locate(p, x, y, ox, oy, qn, cn);
          const uint32_t nj = cnt_plane(p, cur, qn)[cn];
          for (uint32_t j = 0; j < nj; ++j) {
            if (!(ida < ld_id(p, cur, qn, j, cn))) continue;     // each unordered pair image once
            const P2 b = ld_slot<P>(p, cur, qn, j, cn);
            const double Dx = __dsub_rn(__dadd_rn((double)b.x, __dmul_rn((double)ox, p.wx_d)), (double)a.x);
            const double Dy = __dsub_rn(__dadd_rn((double)b.y, __dmul_rn((double)oy, p.wy_d)), (double)a.y);
            const double r = sqrt(__dadd_rn(__dmul_rn(Dx, Dx), __dmul_rn(Dy, Dy)));
            const double bin = floor(__ddiv_rn(__dsub_rn(r, p.sigma_d), dr));
            if (bin >= 0.0 && bin < (double)nbins) atomicAdd(&sh_hist[(uint32_t)bin], 1u);
          }
        }
    }
  }
  __syncthreads();
  for (uint32_t b = threadIdx.x; b < nbins; b += AUX_THREADS)
    if (sh_hist[b]) atomicAdd(&p.hist[b], (unsigned long long)sh_hist[b]);
}

__global__ void k_philox_test(const uint32_t* __restrict__ ctr, uint32_t k0, uint32_t k1, uint32_t* __restrict__ out, uint32_t n) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  uint32_t o[4];
  philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], k0, k1, o);
  out[4 * i] = o[0]; out[4 * i + 1] = o[1]; out[4 * i + 2] = o[2]; out[4 * i + 3] = o[3];
}

}  // namespace mpmc
