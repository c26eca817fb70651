// tile4.cuh — the fused sweep kernel for the paper's own regime: cell widths up to sqrt(2) sigma, where a cell holds up
// to n_max = 4 disks and 3-4 disks per cell are the norm.  Same plan as tile.cuh — one launch = one
// whole sweep of Algorithm 1 (L60-93) on a tile + halo of 5 cells held in shared memory, halo recompute, warps drawing
// chunks of 32 cells, shift straight into the other global buffer, last CTA advances the control block — but shared
// memory holds BOTH slot pairs of every cell (32 B in fp32; empty slots = sentinel, so counts are implied), the cell
// update is the register-resident general one (cell_moves_general, sweep.cuh: 16 neighbour pairs + 2 own pairs per
// move) and the shift compacts eight candidates (shift_eight).  No list of crowded cells is needed.  Serves the square
// and the disc-shaped proposal (MPMC_DISC, L190).
#pragma once
#include "common.cuh"
#include "sweep.cuh"
#include "tile.cuh"

namespace mpmc {

// Threads per CTA, one CTA per SM.  fp32: the update needs ~150 registers; 12 warps at <= 170 leave three warps per
// scheduler to hide a long dependent chain behind (ncu at P1536: issue slots 43 % busy, wait 22 %, long_scoreboard 16 %), 16
// warps at <= 128 registers spill 4 bytes and run P1536 / P3072 12-13 % faster (measured; 20 warps at 96 registers spill 700
// bytes and lose) — so tiles with more cells of a set than 384 take the WIDE instantiation, small tiles (one pass either
// way: latency, where the tighter register budget costs 3 %) the narrow one.  fp64: 8 warps at <= 255 registers (12 at 168
// spill 836 bytes).
template <typename P, bool WIDE> struct Tile4Threads { static constexpr int value = sizeof(P) == 4 ? (WIDE ? 512 : 384) : 256; };
constexpr uint32_t TILE4_WIDE_MIN_PLANE = 385;   // cells per colour plane of a tile region from which the wide instantiation is used

// The cells of sub-sweep k: local colour QL at ring >= k, in chunks of 32 drawn from a shared counter.
template <typename P, int NS, bool DEBUG, bool DISC>
__device__ __forceinline__ void tile4_sub_sweep_cells(const Params& p, SmemCell<P>* sm0, SmemCell<P>* sm1, const TileBox& tb,
                                                      const uint32_t QL, const uint32_t k, const uint32_t dir, const int gx0,
                                                      const int gy0, const unsigned long long t, uint32_t* next, Tally& tally) {
  using R = Real<P>;
  const uint32_t qx = QL & 1u, qy = QL >> 1;
  const uint32_t PS = p.tl_PS, pw = tb.pw;
  const SubRect rc = sub_sweep_rect(tb, k, dir);
  const uint32_t px0 = (rc.x_lo - qx + 1u) >> 1, px1 = (rc.x_hi - qx) >> 1;
  const uint32_t py0 = (rc.y_lo - qy + 1u) >> 1, py1 = (rc.y_hi - qy) >> 1;
  const uint32_t nxp = px1 - px0 + 1u, count = nxp * (py1 - py0 + 1u);
  const uint32_t inv = small_div_magic(nxp);
  const uint32_t lane = threadIdx.x & 31u;
  const uint32_t t_lo = (uint32_t)t, t_hi = (uint32_t)(t >> 32);
  const P HALF_FAR = R::far_away() * (P)0.5;
  int noff[9];                                   // the 3 x 3 cells relative to a cell of this colour (uniform)
#pragma unroll
  for (int j = 0; j < 9; ++j) noff[j] = neighbour_offset(QL, j % 3 - 1, j / 3 - 1, PS, pw);
  for (;;) {
    uint32_t base = 0;
    if (lane == 0u) base = atomicAdd(next, 32u);
    base = __shfl_sync(0xFFFFFFFFu, base, 0);
    if (base >= count) break;
    const uint32_t idx = base + lane;
    if (idx >= count) continue;
    const uint32_t ry = small_div(idx, inv), rx = idx - ry * nxp;
    const uint32_t px = px0 + rx, py = py0 + ry, lx = 2u * px + qx, ly = 2u * py + qy;
    const uint32_t si = QL * PS + py * pw + px;
    const uint32_t cell = wrap_cell(gy0 + (int)ly, p.my) * p.mx + wrap_cell(gx0 + (int)lx, p.mx);
    const bool interior = lx - (uint32_t)HALO < tb.TX && ly - (uint32_t)HALO < tb.TY;
    Half<P> h0[9], h1[9];
#pragma unroll
    for (int j = 0; j < 9; ++j) {
      h0[j] = lds_half(sm0 + si + noff[j], 0u);
      h1[j] = lds_half(sm1 + si + noff[j], 0u);
    }
    // slots fill in order, so the count is the number of occupied slots
    const uint32_t n = h0[4].x.x < HALF_FAR ? (h0[4].x.y < HALF_FAR ? (h1[4].x.x < HALF_FAR ? (h1[4].x.y < HALF_FAR ? 4u : 3u) : 2u) : 1u) : 0u;
    uint32_t amask, n_acc, n_rb, n_ro;
    Half<P> o0, o1;
    cell_moves_general<P, NS, DISC>(p, h0, h1, n, cell, t_lo, t_hi, o0, o1, amask, n_acc, n_rb, n_ro);
    if (amask != 0u) {                              // write back (Alg. 2 line 34, L234)
      sts_half(sm0, si, o0);
      if (n > 2u) sts_half(sm1, si, o1);
    }
    if (interior) { tally.acc += n_acc; tally.rb += n_rb; tally.ro += n_ro; }
    if (DEBUG && interior) {
      p.mask[cell] = amask;
      if (n > 0u) atomicAdd(&p.ctl->digest, mix64(mix64(t) ^ (((unsigned long long)cell << 32) | amask)));
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// The fused sweep kernel, four slots per cell.  Dynamic shared memory: 2 slot pairs x 4 planes x tl_PS cells.
// ---------------------------------------------------------------------------------------------------------
template <typename P, int NS, bool DEBUG, bool DISC, bool WIDE = false>
__global__ void __launch_bounds__(Tile4Threads<P, WIDE>::value, 1)
k_tile4_sweep(const __grid_constant__ Params p, const unsigned long long t, const Draws dr_host, const uint32_t cur) {
  using R = Real<P>;
  extern __shared__ __align__(16) unsigned char tile_smem[];
  const uint32_t PS = p.tl_PS;
  SmemCell<P>* sm0 = reinterpret_cast<SmemCell<P>*>(tile_smem);     // slot pair 0 of the four local colour planes
  SmemCell<P>* sm1 = sm0 + 4u * PS;                                 // slot pair 1
  __shared__ uint32_t s_next[8];                 // chunk counters: sub-sweeps 1-4, shift planes 0-3
  Ctl* ctl = p.ctl;
  // The sweep index comes as a kernel argument (the host counts launches), and with it the draws of this sweep — a pure
  // function of (seed, t), Alg. 1 lines 2, 15, 16 (L64, L90-91), evaluated by the host with the same draw_sweep — and the
  // buffer that holds the sweep's state (every sweep flips it): uniform values, so the tile's geometry and the counters are
  // set up before the wait.  Launched with programmatic stream serialisation (mpmc.cu): everything below the wait reads
  // what the previous sweep wrote.
  Draws dr;                                      // (a copy in registers: a parameter whose address is taken lives in local memory)
  dr.order[0] = dr_host.order[0]; dr.order[1] = dr_host.order[1]; dr.order[2] = dr_host.order[2]; dr.order[3] = dr_host.order[3];
  dr.dir = dr_host.dir; dr.dist_word = dr_host.dist_word;
  const uint32_t nxt = cur ^ 1u;
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5, NW = blockDim.x >> 5;
  const TileBox tb = tile_box(p, blockIdx.x);
  const uint32_t pw = tb.pw, ph = tb.ph, Mqp = p.Mqp;
  const int gx0 = (int)tb.x0 - HALO, gy0 = (int)tb.y0 - HALO;       // global cell of the region's corner (unwrapped)
  const P FAR = R::far_away(), HALF_FAR = FAR * (P)0.5;
  const uint32_t dir = dr.dir;
  const bool along_x = dir < 2u, positive = (dir & 1u) == 0u;
  const P w = along_x ? R::wx(p) : R::wy(p);
  const P delta = R::mul(R::mul((P)0.5, w), R::unit(dr.dist_word));   // line 15 (L90)
  if (tid == 0) {
    for (int i = 0; i < 8; ++i) s_next[i] = 0u;
  }
  __syncthreads();
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  // the head of the control block, one trip to L2: a launch whose sweep index is not the state's returns (nothing has been
  // written); the state's buffer is the one the host named (anything else cannot happen and is reported)
  {
    const CtlHeader ch = ctl_header(ctl, (uint32_t)(t & 3u));
    if (ch.t == t && ch.cur != cur && tid == 0) atomicOr(&ctl->err, ERRBIT_STATE);
    if (ch.t != t || ch.cur != cur) return;
  }
  // Every CTA takes a ticket once it has read the control block; the one that draws the last ticket knows that all have,
  // and advances the block right away — nothing below reads it, and the next launch waits for this one to complete — so no
  // CTA waits for a counter at its end.
  if (tid == 0 && atomicAdd(&ctl->ticket, 1u) == gridDim.x - 1u) {
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

  // ---- load the tile and its halo: warps take plane rows, lanes run along the row; slot pair 1 only where n > 2 ----
  {
    const P* posc = reinterpret_cast<const P*>(p.pos[cur]);
    const uint8_t* cntc = p.cnt[cur];
    const uint32_t nrows = 4u * ph, inv_ph = small_div_magic(ph);
    for (uint32_t c0 = 0; c0 < pw; c0 += 32u) {
      for (uint32_t r0 = warp; r0 < nrows; r0 += 4u * NW) {
        Half<P> v[4];
        uint32_t sidx[4], gidx[4], cnt[4];
        bool ok[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const uint32_t r = r0 + (uint32_t)j * NW, rr = r < nrows ? r : 0u;
          const uint32_t q = small_div(rr, inv_ph), py = rr - q * ph, px = c0 + lane;
          ok[j] = r < nrows && px < pw;
          const uint32_t gy = wrap_cell(gy0 + (int)(2u * py + (q >> 1)), p.my);
          const uint32_t gx = wrap_cell(gx0 + (int)(2u * (ok[j] ? px : 0u) + (q & 1u)), p.mx);
          const uint32_t Qg = ((gy & 1u) << 1) | (gx & 1u), cig = (gy >> 1) * p.hx + (gx >> 1);
          sidx[j] = q * PS + py * pw + px; gidx[j] = 2u * Qg * Mqp + cig;
          cnt[j] = 0u;
          if (ok[j]) { cnt[j] = cntc[Qg * Mqp + cig]; v[j] = ld_half(posc, gidx[j]); }
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          if (!ok[j]) continue;
          Half<P> hi; hi.x = R::pair(FAR, FAR); hi.y = hi.x;
          if (cnt[j] > 2u) hi = ld_half(posc, gidx[j] + Mqp);
          sts_half(sm0, sidx[j], v[j]);
          sts_half(sm1, sidx[j], hi);
        }
      }
    }
  }
  __syncthreads();
  Tally tally;

  // ---- four sub-sweeps (Alg. 1 lines 3-14, L66-88): sub-sweep k updates its colour at ring >= k ----
#pragma unroll 1
  for (uint32_t k = 1; k <= 4u; ++k) {
    const uint32_t Qg = k == 1u ? dr.order[0] : k == 2u ? dr.order[1] : k == 3u ? dr.order[2] : dr.order[3];
    // the region starts at an odd cell (x0 - 5, y0 - 5): colours flip.  ONE copy of the update for the four colours (the
    // local colour is a run-time value): a quarter of the code for the instruction cache
    tile4_sub_sweep_cells<P, NS, DEBUG, DISC>(p, sm0, sm1, tb, Qg ^ 3u, k, dr.dir, gx0, gy0, t, &s_next[k - 1u], tally);
    __syncthreads();
  }

  // ---- cell shift (Alg. 1 lines 15-17; Algorithm 4) of the interior cells, shared memory -> other buffer ----
  {
    const P step = positive ? -delta : delta;     // l' = l - f*delta   (L303)
    const P back = positive ? w : -w;             // entrant translation (L332)
    const uint2* idsc = reinterpret_cast<const uint2*>(p.ids[cur]);
    P* posn = reinterpret_cast<P*>(p.pos[nxt]);
    uint2* idsn = reinterpret_cast<uint2*>(p.ids[nxt]);
    uint8_t* cntn = p.cnt[nxt];
    const uint32_t hTX = tb.TX >> 1, per_plane = hTX * (tb.TY >> 1);
    const uint32_t inv = small_div_magic(hTX);
    const int dox = along_x ? (positive ? 1 : -1) : 0, doy = along_x ? 0 : (positive ? 1 : -1);
    const uint2 none = make_uint2(0xFFFFFFFFu, 0xFFFFFFFFu);
#pragma unroll 1
    for (uint32_t q = 0; q < 4u; ++q) {
      const uint32_t qx = q & 1u, qy = q >> 1;
      const uint32_t px0 = (HALO - qx + 1u) >> 1, py0 = (HALO - qy + 1u) >> 1;
      const int nboff = neighbour_offset(q, dox, doy, PS, pw);       // the old neighbour in direction f (L314-317)
      for (;;) {
        uint32_t base = 0;
        if (lane == 0u) base = atomicAdd(&s_next[4u + q], 32u);
        base = __shfl_sync(0xFFFFFFFFu, base, 0);
        if (base >= per_plane) break;
        const uint32_t idx = base + lane;
        if (idx >= per_plane) continue;
        const uint32_t ry = small_div(idx, inv), rx = idx - ry * hTX;
        const uint32_t px = px0 + rx, py = py0 + ry, lx = 2u * px + qx, ly = 2u * py + qy;
        const uint32_t si = q * PS + py * pw + px, sn = (uint32_t)((int)si + nboff);
        const uint32_t gx = (uint32_t)(gx0 + (int)lx), gy = (uint32_t)(gy0 + (int)ly);      // interior: no wrap
        const uint32_t gxn = wrap_cell((int)gx + dox, p.mx), gyn = wrap_cell((int)gy + doy, p.my);
        const uint32_t Qg = ((gy & 1u) << 1) | (gx & 1u), Qn = ((gyn & 1u) << 1) | (gxn & 1u);
        const uint32_t cig = (gy >> 1) * p.hx + (gx >> 1), cin = (gyn >> 1) * p.hx + (gxn >> 1);
        const uint32_t own = 2u * Qg * Mqp + cig, nbg = 2u * Qn * Mqp + cin;
        const Half<P> ho0 = lds_half(sm0, si), ho1 = lds_half(sm1, si), hn0 = lds_half(sm0, sn), hn1 = lds_half(sm1, sn);
        const uint2 io01 = idsc[own], in01 = idsc[nbg];
        uint2 io23 = none, in23 = none;
        if (ho1.x.x < HALF_FAR) io23 = idsc[own + Mqp];            // slots 2, 3 in use: their ids are valid
        if (hn1.x.x < HALF_FAR) in23 = idsc[nbg + Mqp];
        Half<P> o0, o1; uint2 j01, j23;
        uint32_t nn = shift_eight<P>(ho0, ho1, hn0, hn1, io01, io23, in01, in23, along_x, step, back, w, o0, o1, j01, j23);
        if (nn > (uint32_t)NMAX) { atomicOr(&ctl->err, ERRBIT_OVERFLOW); nn = NMAX; }
        st_half(posn, own, o0); idsn[own] = j01;
        if (nn > 2u) { st_half(posn, own + Mqp, o1); idsn[own + Mqp] = j23; }
        cntn[Qg * Mqp + cig] = (uint8_t)nn;       // L280, L342
      }
    }
  }

  flush_tally(p, tally);                         // counters
}

}  // namespace mpmc
