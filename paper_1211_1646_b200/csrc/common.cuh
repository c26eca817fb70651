// common.cuh — data layout, control block, Philox4x32-10 and variates for the sm_100a MPMC kernels.
//
// Product code (CUDA path).  Shares nothing with oracle/.  Compile with -fmad=false: every floating-point
// operation below is ONE IEEE round-to-nearest operation, and the only fused multiply-add of the method (the
// squared distance) is written __fma_rn / __fmaf_rn explicitly, so results are bit-identical to a plain CPU
// evaluation of the same formulas.
//
// Layout in HBM ("colour-split slot-pair planes"): the four checkerboard sets of
// PAPER.md eq. 1 (L43) are stored as four dense sub-grids of hx x hy = (mx/2) x (my/2) cells, cell (x, y) at
//   colour Q = 2 (y & 1) + (x & 1),   index ci = (y >> 1) * hx + (x >> 1),
// and the n_max = 4 slots of a cell (L150, L152) are two planes of slot PAIRS (half h = slots 2h, 2h+1):
//   cnt[buf][Q][ci]            u8        number of disks n[x, y]
//   pos[buf][Q][h][ci]         real x 4  {x_a, x_b, y_a, y_b}: cell-local coordinates (L154) of slots a = 2h, b = 2h+1
//   ids[buf][Q][h][ci]         u32 x 2   original disk indices of the two slots
// Invariant: an EMPTY slot of half 0 holds the far-away sentinel (the paper's (-10,-10) trick, L295/L346), so
// a neighbour cell is ONE 128-bit load (fp32) whose two register pairs are directly the operands of the packed
// fp32x2 overlap test, with no count-dependent select.  Half 1 is valid (and sentinel-filled) only while
// n > 2; it is never touched at w ~ sigma.  A warp that works on 32 consecutive active cells reads 512
// contiguous bytes per neighbour cell row.  This generalises the even/odd-x split of the paper's Algorithm 3
// (L241-258) to both axes.  buf = 0/1 is the double buffer of the cell shift (L350).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <cstddef>

namespace mpmc {

constexpr int NMAX = 4;                       // n_max
constexpr uint32_t SLOT_SHUFFLE = 0x80000000u;  // Philox counter word 3 for the cell's shuffle words
constexpr uint32_t CELL_GLOBAL = 0xFFFFFFFFu;   // counter word 0 for per-sweep draws
constexpr uint32_t SLOT_ORDER = 0xFFFFFFFFu;    // set order + shift direction
constexpr uint32_t SLOT_DIST = 0xFFFFFFFEu;     // shift distance

// sticky device error bits (Ctl::err)
constexpr uint32_t ERRBIT_OVERFLOW = 1u;  // a cell would hold more than NMAX disks
constexpr uint32_t ERRBIT_RANGE = 2u;     // loaded coordinate NaN or outside [0, L]
constexpr uint32_t ERRBIT_OVERLAP = 4u;   // loaded positions overlap
constexpr uint32_t ERRBIT_STATE = 8u;     // internal: a launch was given the wrong buffer parity for its sweep index
constexpr uint32_t FLAG_NO_PARTICLE_SHUFFLE = 8u, FLAG_NO_SET_SHUFFLE = 16u;   // = MPMC_NO_* of mpmc.h
constexpr uint32_t CTR_SLOTS = 64;        // rows of move counters (summed on read)
constexpr uint32_t CROWD_CAP = 256;       // cells with more than 2 disks the tile kernel can carry per state

// Device-resident control block: the state that survives between launches.  Inside a launch the sweep index,
// buffer parity, grid origin and per-sweep draws live in registers / shared memory (sweep.cuh, k_sweeps).
struct Ctl {
  // ---- the first 32 bytes are what a tile-kernel launch reads before it does anything: two 16-byte loads (ctl_header) ----
  unsigned long long t;            // sweep index
  uint32_t cur;                    // which buffer holds the current state
  uint32_t err;                    // sticky error bits
  // Cells holding more than 2 disks ("crowded") in the state at sweep t, kept per (t & 3): ccount = how many,
  // clist = their canonical ids y*mx+x in no particular order; crowded != 0: more than CROWD_CAP of them, the
  // list is incomplete and the tile kernel (tile.cuh) must leave this state to the general kernel.  Written by
  // whichever kernel produces the state; a slot is cleared two sweeps ahead of its use.
  uint32_t crowded[4];
  uint32_t ccount[4];
  uint32_t bar;                    // arrival counter of the grid barrier (zeroed by the host before a launch)
  uint32_t ticket;                 // blocks-started counter of the tile kernels
  uint32_t pad0[2];
  uint32_t clist[4][CROWD_CAP];
  double origin[2];                // grid origin: X = origin + cell * w + local
  unsigned long long digest;       // accept-sequence digest (MPMC_DEBUG)
  unsigned long long path_sweeps[2];  // sweeps done by the tile kernel / by the general kernel since the last load
  unsigned long long counters[CTR_SLOTS][4];  // per row: accepted, rejected_boundary, rejected_overlap, -
};

// Kernel parameters (by value, __grid_constant__): geometry and the workspace pointers.
struct Params {
  uint32_t mx, my, hx, hy;   // cells; hx = mx/2, hy = my/2
  uint32_t Mq, Mqp;          // cells per colour; plane stride (Mq rounded up to 64)
  uint32_t n_s, N;
  uint32_t flags;            // MPMC_* creation flags (the ablation switches are read on the device)
  uint32_t tune;             // tuning word for experiments (builds with -DMPMC_EXPERIMENT read it from MPMC_TUNE); unused by default
  uint32_t track_crowded;    // 1: kernels that write cell counts list the cells with more than 2 disks (for tile.cuh)
  uint32_t hx_magic, hx_sh1, hx_sh2;  // ci / hx without a divide (Granlund-Montgomery; host: div_magic)
  uint32_t tl_ntx, tl_nty, tl_PS;       // tile kernel: tiles per row (first tl_na rows), rows of tiles, shared-memory plane stride (cells)
  uint32_t tl_na, tl_hyA;               // the first tl_na rows of tiles cover the half-rows [0, tl_hyA) with tl_ntx tiles each, the
                                        // other rows the rest with tl_ntx + 1 tiles each (uniform tiling: tl_na = tl_nty, tl_hyA = hy)
  uint32_t tl_PH;                       // ... rows of the tallest tile's planes (sorted variant: stride of its row tables)
  uint32_t tl_div[4][3];                // n / d without a divide (host: div_magic) for d = tl_ntx, tl_ntx + 1, tl_na, tl_nty - tl_na
  uint32_t cl_cx, cl_cy, cl_cap, cl_stride;   // cluster-resident kernel (cluster.cuh): tiles per row / column = CTAs of the cluster, cells a CTA
                                        // has room for, row stride of a CTA's cell arrays (the widest tile)
  uint32_t seed_lo, seed_hi;
  uint32_t rk0[10], rk1[10];            // Philox round keys seed + r * Weyl constant (philox4x32_10_rk)
  float wx_f, wy_f, sigma2_f, d_f;      // working-precision constants (fp32 mode)
  double wx_p, wy_p, sigma2_p, d_p;     // working-precision constants (fp64 mode)
  float dsc_f; double dsc_p;            // d 2^-24 (fp32) / d 2^-32 (fp64): displacement = dsc * odd integer
  double wx_d, wy_d;                    // (double) of the working-precision widths
  double Lx_eff, Ly_eff, sigma_d;
  double Lx_user, Ly_user;              // the caller's box (input range check)
  Ctl* ctl;
  uint8_t* cnt[2];
  void* pos[2];
  uint32_t* ids[2];
  uint32_t* cnt32;                      // scratch: u32 counters for the cell-list build
  unsigned long long* hist;             // scratch: contact histogram
  uint32_t* mask;                       // MPMC_DEBUG: accept masks, canonical index y*mx+x; else nullptr
};

template <typename P> struct Real;
template <> struct Real<float> {
  using T2 = float2;
  static __device__ __forceinline__ float wx(const Params& p) { return p.wx_f; }
  static __device__ __forceinline__ float wy(const Params& p) { return p.wy_f; }
  static __device__ __forceinline__ float sigma2(const Params& p) { return p.sigma2_f; }
  static __device__ __forceinline__ float d(const Params& p) { return p.d_f; }
  static __device__ __forceinline__ float add(float a, float b) { return __fadd_rn(a, b); }
  static __device__ __forceinline__ float sub(float a, float b) { return __fsub_rn(a, b); }
  static __device__ __forceinline__ float mul(float a, float b) { return __fmul_rn(a, b); }
  static __device__ __forceinline__ float fma(float a, float b, float c) { return __fmaf_rn(a, b, c); }
  // symmetric unit variate: odd integer of magnitude < 2^24 times 2^-24 (exact; never 0)
  static __device__ __forceinline__ float sym(uint32_t R) {
    return __fmul_rn((float)((int)(2u * (R >> 8) + 1u) - (1 << 24)), 0x1p-24f);
  }
  static __device__ __forceinline__ float unit(uint32_t R) { return __fmul_rn((float)(R >> 8), 0x1p-24f); }
  // d * sym(R) as (d 2^-24) * integer: the same real product, so the same rounded value (host checks d 2^-24 is normal)
  static __device__ __forceinline__ float scaled_sym(const Params& p, uint32_t R) {
    return __fmul_rn((float)((int)((R >> 7) | 1u) - (1 << 24)), p.dsc_f);   // (R >> 7) | 1 = 2 (R >> 8) + 1
  }
  static __device__ __forceinline__ float min3(float a, float b, float c) { return fminf(fminf(a, b), c); }
  static __device__ __forceinline__ float far_away() { return 1.0e18f; }   // sentinel: never overlaps
  // Two lanes at once: sm_100a packed fp32x2 instructions (FADD2 / FMUL2 / FFMA2), each lane one IEEE rn op.
  using Pair = float2;
  static __device__ __forceinline__ Pair pair(float a, float b) { return make_float2(a, b); }
  static __device__ __forceinline__ Pair padd(Pair a, Pair b) { return __fadd2_rn(a, b); }
  static __device__ __forceinline__ Pair pmul(Pair a, Pair b) { return __fmul2_rn(a, b); }
  static __device__ __forceinline__ Pair pfma(Pair a, Pair b, Pair c) { return __ffma2_rn(a, b, c); }
};
template <> struct Real<double> {
  using T2 = double2;
  static __device__ __forceinline__ double wx(const Params& p) { return p.wx_p; }
  static __device__ __forceinline__ double wy(const Params& p) { return p.wy_p; }
  static __device__ __forceinline__ double sigma2(const Params& p) { return p.sigma2_p; }
  static __device__ __forceinline__ double d(const Params& p) { return p.d_p; }
  static __device__ __forceinline__ double add(double a, double b) { return __dadd_rn(a, b); }
  static __device__ __forceinline__ double sub(double a, double b) { return __dsub_rn(a, b); }
  static __device__ __forceinline__ double mul(double a, double b) { return __dmul_rn(a, b); }
  static __device__ __forceinline__ double fma(double a, double b, double c) { return __fma_rn(a, b, c); }
  static __device__ __forceinline__ double sym(uint32_t R) {
    return __dmul_rn((double)(2ll * (long long)R + 1ll - (1ll << 32)), 0x1p-32);
  }
  static __device__ __forceinline__ double unit(uint32_t R) { return __dmul_rn((double)R, 0x1p-32); }
  static __device__ __forceinline__ double scaled_sym(const Params& p, uint32_t R) {
    return __dmul_rn((double)(2ll * (long long)R + 1ll - (1ll << 32)), p.dsc_p);
  }
  static __device__ __forceinline__ double min3(double a, double b, double c) { return fmin(fmin(a, b), c); }
  static __device__ __forceinline__ double far_away() { return 1.0e150; }
  struct Pair { double x, y; };             // no packed fp64 instruction: two scalar ops
  static __device__ __forceinline__ Pair pair(double a, double b) { Pair r; r.x = a; r.y = b; return r; }
  static __device__ __forceinline__ Pair padd(Pair a, Pair b) { return pair(__dadd_rn(a.x, b.x), __dadd_rn(a.y, b.y)); }
  static __device__ __forceinline__ Pair pmul(Pair a, Pair b) { return pair(__dmul_rn(a.x, b.x), __dmul_rn(a.y, b.y)); }
  static __device__ __forceinline__ Pair pfma(Pair a, Pair b, Pair c) { return pair(__fma_rn(a.x, b.x, c.x), __fma_rn(a.y, b.y, c.y)); }
};

// "Does the trial position overlap one of these disks": min r^2 < sigma^2 over the distances fed in (L194-204, strict: A4).
// fp32 keeps a running minimum (one 3-input FMNMX per pair of distances).  In fp64 a minimum is DSETP.MIN + two FSEL and the
// running minimum of 17 values a dependent chain of 16 of them per move (~900 cycles of a 3 500-cycle sub-sweep pass at
// N = 4096: measured); min r^2 < s is the same verdict as "some r^2 < s" (no NaN occurs: every operand is finite), so fp64
// compares each distance and ORs the predicates, on two independent accumulators.  Used where a sub-sweep is ONE pass of
// one warp per scheduler (cluster.cuh: C1 14 020 -> 13 390 cycles); on the tile kernels, whose fp64 sub-sweeps are bound by
// the DP pipe's throughput rather than by the chain, the running minimum is faster (C2: 18.9 against 20.0 us per sweep).
template <typename P> struct OverlapAcc;
template <> struct OverlapAcc<float> {
  float rmin;
  __device__ __forceinline__ OverlapAcc(float, float first) : rmin(first) {}      // first = the first distance
  template <int E> __device__ __forceinline__ void pair(float2 r2) { rmin = fminf(fminf(rmin, r2.x), r2.y); }
  __device__ __forceinline__ bool overlap(float sigma2) const { return rmin < sigma2; }
};
template <> struct OverlapAcc<double> {
  double s2; bool a, b;
  __device__ __forceinline__ OverlapAcc(double sigma2, double first) : s2(sigma2), a(first < sigma2), b(false) {}
  template <int E> __device__ __forceinline__ void pair(Real<double>::Pair r2) {      // E: which accumulator (parity)
    if (E & 1) b |= (r2.x < s2) | (r2.y < s2); else a |= (r2.x < s2) | (r2.y < s2);
  }
  __device__ __forceinline__ bool overlap(double) const { return a | b; }
};

// Philox4x32-10 (Salmon et al., SC'11).  Ten rounds of two 32x32->64 multiplies and xors; the key schedule
// adds the Weyl constants.  counter = (c0..c3), key = (k0, k1).
__host__ __device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t (&out)[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const unsigned long long p0 = (unsigned long long)0xD2511F53u * c0;
    const unsigned long long p1 = (unsigned long long)0xCD9E8D57u * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    c1 = (uint32_t)p1;
    c3 = (uint32_t)p0;
    c0 = n0;
    c2 = n2;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// The same function with the ten round keys of the run's seed taken from the kernel parameters (constant bank):
// the key schedule costs no instruction.
__device__ __forceinline__ void philox4x32_10_rk(const Params& p, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                 uint32_t (&out)[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const unsigned long long p0 = (unsigned long long)0xD2511F53u * c0;
    const unsigned long long p1 = (unsigned long long)0xCD9E8D57u * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ p.rk0[r];
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ p.rk1[r];
    c1 = (uint32_t)p1;
    c3 = (uint32_t)p0;
    c0 = n0;
    c2 = n2;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// The head of the control block as two independent loads, issued together: {t, cur, err} (16 bytes) and crowded[slot].
struct CtlHeader { unsigned long long t; uint32_t cur, err, crowded; };
__device__ __forceinline__ CtlHeader ctl_header(const Ctl* ctl, const uint32_t slot) {
  uint32_t a0, a1, a2, a3, b;
  asm volatile("ld.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(a0), "=r"(a1), "=r"(a2), "=r"(a3) : "l"(ctl) : "memory");
  asm volatile("ld.global.u32 %0, [%1];" : "=r"(b) : "l"(reinterpret_cast<const unsigned char*>(ctl) + 16 + 4 * slot) : "memory");
  CtlHeader h;
  h.t = ((unsigned long long)a1 << 32) | a0; h.cur = a2; h.err = a3; h.crowded = b;
  return h;
}
static_assert(offsetof(Ctl, cur) == 8 && offsetof(Ctl, crowded) == 16 && offsetof(Ctl, ccount) == 32, "ctl_header reads this layout");

// a kernel that writes a cell with more than 2 disks into the state of sweep slot `slot` records it here
__device__ __forceinline__ void note_crowded(Ctl* ctl, uint32_t slot, uint32_t cell) {
  const uint32_t i = atomicAdd(&ctl->ccount[slot], 1u);
  if (i < CROWD_CAP) ctl->clist[slot][i] = cell; else ctl->crowded[slot] = 1u;
}

__host__ __device__ __forceinline__ uint32_t bounded(uint32_t word, uint32_t bound) {
  return (uint32_t)(((unsigned long long)word * bound) >> 32);
}

// Per-sweep draws (Alg. 1 lines 2, 15, 16; reading A9): Fisher-Yates of the four sets with
// words G0..G2, direction from the top two bits of G3, distance word from a second counter.  A pure function of
// (seed, sweep index), so every block computes it for itself.
struct Draws { uint32_t order[4]; uint32_t dir; uint32_t dist_word; };
__host__ __device__ __forceinline__ Draws draw_sweep(const uint32_t seed_lo, const uint32_t seed_hi, const uint32_t flags,
                                                     const unsigned long long t) {
  uint32_t G[4], H[4];
  philox4x32_10(CELL_GLOBAL, (uint32_t)t, (uint32_t)(t >> 32), SLOT_ORDER, seed_lo, seed_hi, G);
  uint32_t o[4] = {0, 1, 2, 3};
#pragma unroll
  for (int i = 3; i >= 1 && !(flags & FLAG_NO_SET_SHUFFLE); --i) {
    const uint32_t j = bounded(G[3 - i], (uint32_t)i + 1u);
    const uint32_t a = o[i];
    // o[j] with j dynamic: select chain keeps o[] in registers
    const uint32_t b = j == 0 ? o[0] : j == 1 ? o[1] : j == 2 ? o[2] : o[3];
    if (j == 0) o[0] = a; else if (j == 1) o[1] = a; else if (j == 2) o[2] = a; else o[3] = a;
    o[i] = b;
  }
  philox4x32_10(CELL_GLOBAL, (uint32_t)t, (uint32_t)(t >> 32), SLOT_DIST, seed_lo, seed_hi, H);
  Draws d;
  d.order[0] = o[0]; d.order[1] = o[1]; d.order[2] = o[2]; d.order[3] = o[3];
  d.dir = G[3] >> 30;
  d.dist_word = H[0];
  return d;
}
__device__ __forceinline__ Draws draw_sweep(const Params& p, unsigned long long t) { return draw_sweep(p.seed_lo, p.seed_hi, p.flags, t); }

// n / d for any 32-bit n with the numbers div_magic (mpmc.cu) made for d
__device__ __forceinline__ uint32_t magic_div(const uint32_t n, const uint32_t (&m)[3]) {
  const uint32_t t = __umulhi(m[0], n);
  return (t + ((n - t) >> m[1])) >> m[2];
}
// ya = ci / hx, xa = ci - ya * hx with the precomputed magic numbers of Params
__device__ __forceinline__ uint32_t div_hx(const Params& p, uint32_t ci) {
  const uint32_t t = __umulhi(p.hx_magic, ci);
  return (t + ((ci - t) >> p.hx_sh1)) >> p.hx_sh2;
}

// Prefetching loads.  `asm volatile` keeps the compiler from sinking them into the branch that consumes them,
// so they are issued up front and their latency overlaps the Philox arithmetic (sweep.cuh, level-1 loads).
__device__ __forceinline__ uint32_t ld_u8_early(const uint8_t* ptr) {
  uint32_t v;
  asm volatile("ld.global.u8 %0, [%1];" : "=r"(v) : "l"(ptr) : "memory");
  return v;
}

// ---- slot-pair planes: wide accessors for the hot kernels (index i = (Q*2 + h)*Mqp + ci, in cells) ----
template <typename P> struct Half { typename Real<P>::Pair x, y; };   // (x_a, x_b), (y_a, y_b)

// `asm volatile` keeps the compiler from sinking the load into a branch that consumes it: it is issued up front
__device__ __forceinline__ Half<float> ld_half_early(const float* pos, uint32_t i) {
  Half<float> h;
  asm volatile("ld.global.v4.f32 {%0, %1, %2, %3}, [%4];"
               : "=f"(h.x.x), "=f"(h.x.y), "=f"(h.y.x), "=f"(h.y.y) : "l"(reinterpret_cast<const float4*>(pos) + i) : "memory");
  return h;
}
__device__ __forceinline__ Half<double> ld_half_early(const double* pos, uint32_t i) {
  Half<double> h;
  const double2* q = reinterpret_cast<const double2*>(pos) + 2 * (size_t)i;
  asm volatile("ld.global.v2.f64 {%0, %1}, [%2];" : "=d"(h.x.x), "=d"(h.x.y) : "l"(q) : "memory");
  asm volatile("ld.global.v2.f64 {%0, %1}, [%2];" : "=d"(h.y.x), "=d"(h.y.y) : "l"(q + 1) : "memory");
  return h;
}
__device__ __forceinline__ Half<float> ld_half(const float* pos, uint32_t i) {
  const float4 v = reinterpret_cast<const float4*>(pos)[i];
  Half<float> h; h.x.x = v.x; h.x.y = v.y; h.y.x = v.z; h.y.y = v.w; return h;
}
__device__ __forceinline__ Half<double> ld_half(const double* pos, uint32_t i) {
  const double2* q = reinterpret_cast<const double2*>(pos) + 2 * (size_t)i;
  const double2 a = q[0], b = q[1];
  Half<double> h; h.x.x = a.x; h.x.y = a.y; h.y.x = b.x; h.y.y = b.y; return h;
}
__device__ __forceinline__ void st_half(float* pos, uint32_t i, const Half<float>& h) {
  reinterpret_cast<float4*>(pos)[i] = make_float4(h.x.x, h.x.y, h.y.x, h.y.y);
}
__device__ __forceinline__ void st_half(double* pos, uint32_t i, const Half<double>& h) {
  double2* q = reinterpret_cast<double2*>(pos) + 2 * (size_t)i;
  q[0] = make_double2(h.x.x, h.x.y); q[1] = make_double2(h.y.x, h.y.y);
}

// ---- scalar accessors (kernels off the per-sweep path, and the rare generic paths) ----
__device__ __forceinline__ size_t slot_index(const Params& p, uint32_t Q, uint32_t slot, uint32_t ci) {
  return (size_t)((Q * 2u + (slot >> 1)) * p.Mqp + ci);       // in slot pairs
}
template <typename P>
__device__ __forceinline__ typename Real<P>::T2 ld_slot(const Params& p, uint32_t buf, uint32_t Q, uint32_t slot, uint32_t ci) {
  const P* b = reinterpret_cast<const P*>(p.pos[buf]) + (slot_index(p, Q, slot, ci) * 4 + (slot & 1u));
  typename Real<P>::T2 v; v.x = b[0]; v.y = b[2]; return v;
}
template <typename P>
__device__ __forceinline__ void st_slot(const Params& p, uint32_t buf, uint32_t Q, uint32_t slot, uint32_t ci, P x, P y) {
  P* b = reinterpret_cast<P*>(p.pos[buf]) + (slot_index(p, Q, slot, ci) * 4 + (slot & 1u));
  b[0] = x; b[2] = y;
}
__device__ __forceinline__ uint32_t ld_id(const Params& p, uint32_t buf, uint32_t Q, uint32_t slot, uint32_t ci) {
  return p.ids[buf][slot_index(p, Q, slot, ci) * 2 + (slot & 1u)];
}
__device__ __forceinline__ void st_id(const Params& p, uint32_t buf, uint32_t Q, uint32_t slot, uint32_t ci, uint32_t id) {
  p.ids[buf][slot_index(p, Q, slot, ci) * 2 + (slot & 1u)] = id;
}
__device__ __forceinline__ uint8_t* cnt_plane(const Params& p, uint32_t buf, uint32_t Q) {
  return p.cnt[buf] + (size_t)Q * p.Mqp;
}

__device__ __forceinline__ unsigned long long mix64(unsigned long long z) {  // splitmix64 finaliser (digest only)
  z += 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

}  // namespace mpmc
