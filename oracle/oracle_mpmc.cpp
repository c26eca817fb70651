// ORACLE — TEST INFRASTRUCTURE ONLY.  Not part of the product path.
//
// Plain, slow, single-threaded CPU restatement of the hot path of
//   Anderson, Jankowski, Grubb, Engel, Glotzer, "Massively parallel Monte Carlo for many-particle
//   simulations on GPUs" (arxiv 1211.1646; /root/reference/PAPER.md),
// i.e. the checkerboard cell sweep for hard disks: Algorithm 1 with the cell update
// of Algorithm 2 (L164-236) and the cell shift of Algorithm 4 (L270-342), plus the pair-distance
// histogram near contact used by the pressure estimator (L366-382, eq. 4-6).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use
// this file.  It shares no code, header, table or helper with paper_1211_1646_b200/csrc (the CUDA
// path); neither includes or imports the other.  Every loop below follows the paper's order and
// notation; there is no blocking, fusion or reordering.  The readings of the points where the paper
// is silent or garbled are SURVEY.md §8(c) A1-A15 and are restated in DESIGN.md "Readings".
//
// Precision P is float or double.  rn(.) below means ONE IEEE-754 round-to-nearest-even operation in
// P.  Build with -ffp-contract=off so the compiler contracts nothing; the one FMA of the method (the
// squared distance) is written std::fma.
//
// Options beside the default reading: the paper's disc-shaped displacement (OR_DISC, L190) and the two ablations of
// Table 1 (OR_NO_PARTICLE_SHUFFLE, OR_NO_SET_SHUFFLE, L134-142).
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): Philox known answers; the visiting-order example
// of PAPER.md L112; bookkeeping invariants (L152, L354); overlap-free configurations checked
// independently in numpy; isolated-disk acceptance closed form; N=2 / N=3 sampling law (chi^2);
// agreement with a separately written serial MC (Fig. 1); virial-series pressure;
// the polynomial fit on the paper's model distribution (L382); for the disc proposal the isolated-disk closed form of
// the disc, the displacement law and the two-disk law; for the ablations the slot-order and set-order behaviour.
// No function here is "parity unpinned".

#include <cmath>
#include <cstdint>
#include <cstring>
#include <new>
#include <vector>

namespace {

constexpr int NMAX = 4;  // n_max: at most four centres fit a cell of width w < sqrt(2) sigma (Fig. 3)

enum {
  OR_OK = 0,
  OR_ERR_ARG = -1,
  OR_ERR_BOX = -2,
  OR_ERR_OVERLAP = -4,
  OR_ERR_CELL_OVERFLOW = -5,
  OR_ERR_STATE = -7,
};
enum { OR_FP64 = 1u, OR_FP32 = 2u, OR_DISC = 4u,
       // ablations of PAPER.md section 2.4 / Table 1 (L114-142): leave out the particle shuffle / the checkerboard-set shuffle
       OR_NO_PARTICLE_SHUFFLE = 8u, OR_NO_SET_SHUFFLE = 16u,
       // pitfall 1 of section 2.4 (L118-122): a trial move whose centre leaves the cell is NOT rejected for that; the disk
       // is handed to the cell it lands in (appended to that cell's list, L123).  The paper reports that this breaks
       // detailed balance (the reverse sequence of moves cannot be generated); oracle-only ablation, see cell_update
       OR_LEAVE_CELL = 32u };   // OR_DISC: trial displacement uniform in the disc of radius d (L190)

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): 10 rounds; multipliers 0xD2511F53, 0xCD9E8D57;
// key increments (Weyl) 0x9E3779B9, 0xBB67AE85.  Replaces the paper's unpublished Saru hash
// (reading A9): a stateless stream keyed on (seed; cell, sweep, slot).
// ---------------------------------------------------------------------------------------------
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    const uint32_t n0 = hi1 ^ c1 ^ k0;
    const uint32_t n1 = lo1;
    const uint32_t n2 = hi0 ^ c3 ^ k1;
    const uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Counter layout (reading A9): counter = (cell_id, t_lo, t_hi, slot), key = (seed_lo, seed_hi).
//   slot q in [0, ceil(n_s/2)): the displacement words of trial moves 2q (words 0, 1 = x, y) and
//                             2q + 1 (words 2, 3 = x, y) — all four words of a Philox block are used
//   with the disc proposal (flag OR_DISC; the paper's rng.inCircle(d), L190): block (s | j << 16), j = 0, 1, ...,
//                             serves the candidate pairs 2j (words 0, 1) and 2j + 1 (words 2, 3) of trial move s; the
//                             first pair inside the unit disc is taken (rejection from the square)
//   slot 0x80000000         : the shuffle words of the cell
//   cell 0xFFFFFFFF, slot 0xFFFFFFFF : per-sweep set order + shift direction
//   cell 0xFFFFFFFF, slot 0xFFFFFFFE : per-sweep shift distance
constexpr uint32_t SLOT_SHUFFLE = 0x80000000u;
constexpr uint32_t CELL_GLOBAL = 0xFFFFFFFFu;
constexpr uint32_t SLOT_ORDER = 0xFFFFFFFFu;
constexpr uint32_t SLOT_DIST = 0xFFFFFFFEu;

void draw(uint64_t seed, uint32_t cell, uint64_t t, uint32_t slot, uint32_t out[4]) {
  const uint32_t ctr[4] = {cell, (uint32_t)t, (uint32_t)(t >> 32), slot};
  const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  philox4x32_10(ctr, key, out);
}

// bounded integer in [0, bound): high 32 bits of word * bound
inline uint32_t bounded(uint32_t word, uint32_t bound) {
  return (uint32_t)(((uint64_t)word * (uint64_t)bound) >> 32);
}

// Variates.  Symmetric unit variate u in (-1, 1): an odd integer of magnitude < 2^24 (fp32) or
// < 2^32 (fp64) times 2^-24 / 2^-32 — exactly representable, symmetric about 0, never 0.
// Unit-interval variate in [0, 1): (R >> 8) 2^-24 (fp32), R 2^-32 (fp64).
template <typename P> struct Variate;
template <> struct Variate<float> {
  static float sym(uint32_t R) {
    const int32_t v = (int32_t)(2u * (R >> 8) + 1u) - (int32_t)(1 << 24);
    return (float)v * 0x1p-24f;
  }
  static float unit(uint32_t R) { return (float)(R >> 8) * 0x1p-24f; }
};
template <> struct Variate<double> {
  static double sym(uint32_t R) {
    const int64_t v = 2 * (int64_t)R + 1 - ((int64_t)1 << 32);
    return (double)v * 0x1p-32;
  }
  static double unit(uint32_t R) { return (double)R * 0x1p-32; }
};

// Visiting order of the n_M (= n_s) moves of a cell: "p <- c.particles[mod(s, len(c.particles))]"
// (Alg. 1 line 7; Alg. 2 lines 28-32, L224-230) applied to the shuffled list.
// Reading A1: the shuffle is kept as a visiting permutation perm[] over the slots.
inline uint32_t visit(const uint32_t* perm, uint32_t n, uint32_t s) { return perm[s % n]; }

// Durstenfeld / Fisher-Yates (ref [35]): for i = n-1 .. 1: j = bounded(word, i+1); swap.
inline void fisher_yates(uint32_t* a, uint32_t n, const uint32_t* words) {
  for (uint32_t i = n - 1; i >= 1; --i) {
    const uint32_t j = bounded(words[n - 1 - i], i + 1);
    const uint32_t tmp = a[i]; a[i] = a[j]; a[j] = tmp;
  }
}

struct SweepDraws {
  uint32_t order[4];  // checkerboard sets in the order they run; 0=a(0,0) 1=b(1,0) 2=c(0,1) 3=d(1,1) (eq. 1)
  uint32_t dir;       // 0:+x 1:-x 2:+y 3:-y  (Alg. 1 line 16, L91)
  uint32_t dist_word; // the word the shift distance is made of (Alg. 1 line 15, L90)
};

SweepDraws sweep_draws(uint64_t seed, uint64_t t, bool shuffle_sets = true) {
  SweepDraws D;
  uint32_t G[4], H[4];
  draw(seed, CELL_GLOBAL, t, SLOT_ORDER, G);
  for (uint32_t q = 0; q < 4; ++q) D.order[q] = q;
  if (shuffle_sets) fisher_yates(D.order, 4, G);   // uses G[0], G[1], G[2]   (Alg. 1 line 2, L64)
  D.dir = G[3] >> 30;
  draw(seed, CELL_GLOBAL, t, SLOT_DIST, H);
  D.dist_word = H[0];
  return D;
}

// ---------------------------------------------------------------------------------------------
struct Base {
  virtual ~Base() {}
  virtual int load(const double* xy) = 0;
  virtual int sweep(uint64_t k) = 0;
  virtual int get(double* xy) const = 0;
  virtual int debug(uint32_t* counts, void* slab, uint32_t* ids, uint32_t* mask, double origin[2],
                    uint64_t* sweep_index, uint64_t* digest) const = 0;
  virtual int histogram(double dr, uint32_t nbins, uint64_t* hist) const = 0;
  virtual int cell_update_only(uint32_t set) = 0;
  virtual int shift_only(uint32_t dir, double delta) = 0;
  uint64_t N = 0;
  uint32_t mx = 0, my = 0, n_s = 0, flags = 0;
  uint64_t seed = 0, t = 0;
  double wx_d = 0, wy_d = 0, Lx_eff = 0, Ly_eff = 0, sigma_d = 0, d_d = 0;
  double origin[2] = {0, 0};
  uint64_t counters[4] = {0, 0, 0, 0};  // attempted, accepted, rej_boundary, rej_overlap
  uint64_t digest = 0;                  // sum over (sweep, cell) of mix(t, cell, accept mask)  (test aid)
  bool loaded = false;
  int sticky = OR_OK;
};

inline uint64_t mix64(uint64_t z) {  // splitmix64 finaliser; only feeds the accept-sequence digest
  z += 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

template <typename P>
struct Sim : Base {
  P wx, wy, sigma, sigma2, d;
  std::vector<uint32_t> n;       // n[x,y]
  std::vector<P> lx, ly;         // disk[x,y,i], cell-local coordinates (L150, L154)
  std::vector<uint32_t> id;      // original disk index, travels with the position
  std::vector<uint32_t> mask;    // accept mask of the cell in the sweep just finished (bit s = move s accepted)
  std::vector<uint32_t> n_dbl; std::vector<P> lx_dbl, ly_dbl; std::vector<uint32_t> id_dbl;  // L350

  size_t cell(uint32_t x, uint32_t y) const { return (size_t)y * mx + x; }

  // A local coordinate is in the cell iff 0 < l <= w (Alg. 4 lines 10 and 21, L305, L326; reading A3).
  static bool inside(P l, P w) { return l > (P)0 && l <= w; }

  // |D_move - (D + s)| < sigma, strict (Alg. 2 line 19, L204; reading A4), as r^2 < sigma^2 with
  //   q = rn(l_j + s), Delta = rn(M - q), r^2 = fma(Dx, Dx, rn(Dy*Dy)).
  bool overlaps(P Mx, P My, P ljx, P ljy, P sx, P sy) const {
    const P qx = ljx + sx, qy = ljy + sy;
    const P Dx = Mx - qx, Dy = My - qy;
    const P yy = Dy * Dy;
    const P r2 = std::fma(Dx, Dx, yy);
    return r2 < sigma2;
  }

  // ---- Algorithm 2: update of one active cell ------------------------------
  // The move counters and the digest go to an accumulator the caller names (the cells of a set are independent, L48: the
  // OpenMP strip baseline of L390, strip_omp.cpp, gives every thread its own); the plain form adds to the members.
  struct Acc { uint64_t counters[4] = {0, 0, 0, 0}; uint64_t digest = 0; };
  void cell_update(uint32_t x, uint32_t y) {
    Acc a;
    cell_update(x, y, a);
    for (int i = 0; i < 4; ++i) counters[i] += a.counters[i];
    digest += a.digest;
  }
  void cell_update(uint32_t x, uint32_t y, Acc& acc) {
    uint64_t (&counters)[4] = acc.counters;
    uint64_t& digest = acc.digest;
    const size_t c = cell(x, y);
    const uint32_t nc = n[c];
    mask[c] = 0;
    if (nc == 0) return;                                        // lines 4-7 (L181-185); reading A10
    uint32_t perm[NMAX] = {0, 1, 2, 3};
    if (nc >= 2 && !(flags & OR_NO_PARTICLE_SHUFFLE)) {          // line 9 (L187): rng.shuffle
      uint32_t S[4];
      draw(seed, (uint32_t)c, t, SLOT_SHUFFLE, S);
      fisher_yates(perm, nc, S);
    }
    uint32_t m = 0;
    // OR_LEAVE_CELL only: where the disk that started in slot i sits now (slots close up behind a disk that left), -1 = left
    int cur[NMAX] = {0, 1, 2, 3};
    for (uint32_t s = 0; s < n_s; ++s) {                        // line 11 (L189)
      uint32_t k = visit(perm, nc, s);
      if (flags & OR_LEAVE_CELL) {
        if (cur[k] < 0) continue;                               // this disk has left the cell: nothing to move
        k = (uint32_t)cur[k];
      }
      uint32_t R[4];
      P ddx, ddy;
      if (!(flags & OR_DISC)) {
        draw(seed, (uint32_t)c, t, s >> 1, R);                  // reading A9: block s/2 serves moves 2q, 2q+1
        const uint32_t h = 2u * (s & 1u);
        // line 12 (L190); reading A2: uniform in the square [-d, d]^2
        ddx = d * Variate<P>::sym(R[h]);
        ddy = d * Variate<P>::sym(R[h + 1]);
      } else {
        // line 12 as printed: rng.inCircle(d) (L190), uniform in the disc of radius d, by rejection from the square:
        // candidate pairs (ux, uy) in order until rn(fma(ux, ux, rn(uy*uy))) <= 1
        for (uint32_t j = 0;; ++j) {
          if ((j & 1u) == 0u) draw(seed, (uint32_t)c, t, s | ((j >> 1) << 16), R);
          const P ux = Variate<P>::sym(R[2u * (j & 1u)]), uy = Variate<P>::sym(R[2u * (j & 1u) + 1u]);
          const P yy = uy * uy;
          if (std::fma(ux, ux, yy) <= (P)1) { ddx = d * ux; ddy = d * uy; break; }
        }
      }
      const P Mx = lx[c * NMAX + k] + ddx;
      const P My = ly[c * NMAX + k] + ddy;
      counters[0] += 1;
      if (!(inside(Mx, wx) && inside(My, wy))) {                // line 25 (L217), L79, L118
        if (!(flags & OR_LEAVE_CELL)) {
          counters[2] += 1;
          continue;
        }
        // ---- ablation (L118-122): the disk may leave.  It lands in the adjacent cell (d < w), at N = M - e w in that
        //      cell's frame; the Metropolis test is made there, against the 3x3 cells around the cell it lands in ----
        const int ex = Mx > wx ? 1 : (Mx > (P)0 ? 0 : -1), ey = My > wy ? 1 : (My > (P)0 ? 0 : -1);
        const P Nx = Mx - (P)ex * wx, Ny = My - (P)ey * wy;
        const uint32_t xd = (uint32_t)(((int64_t)x + ex + mx) % mx), yd = (uint32_t)(((int64_t)y + ey + my) % my);
        const size_t cd = cell(xd, yd);
        const uint32_t nk = n[c];
        if (n[cd] >= (uint32_t)NMAX || !(inside(Nx, wx) && inside(Ny, wy))) { counters[2] += 1; continue; }   // no room there
        bool ov = false;
        for (int oy = -1; oy <= 1; ++oy)
          for (int ox = -1; ox <= 1; ++ox) {
            const uint32_t xn = (uint32_t)(((int64_t)xd + ox + mx) % mx), yn = (uint32_t)(((int64_t)yd + oy + my) % my);
            const size_t cn = cell(xn, yn);
            const P sx = (P)ox * wx, sy = (P)oy * wy;
            for (uint32_t j = 0; j < n[cn]; ++j) {
              if (cn == c && j == k && (int)xn == (int)x && (int)yn == (int)y && ox == -ex && oy == -ey) continue;   // itself
              if (overlaps(Nx, Ny, lx[cn * NMAX + j], ly[cn * NMAX + j], sx, sy)) ov = true;
            }
          }
        if (ov) { counters[3] += 1; continue; }
        const uint32_t moved_id = id[c * NMAX + k];
        for (uint32_t j = k; j + 1 < nk; ++j) {                 // the list of the cell it leaves closes up
          lx[c * NMAX + j] = lx[c * NMAX + j + 1]; ly[c * NMAX + j] = ly[c * NMAX + j + 1]; id[c * NMAX + j] = id[c * NMAX + j + 1];
        }
        lx[c * NMAX + nk - 1] = (P)0; ly[c * NMAX + nk - 1] = (P)0; id[c * NMAX + nk - 1] = 0xFFFFFFFFu;
        n[c] = nk - 1;
        for (int i = 0; i < NMAX; ++i) { if (cur[i] == (int)k) cur[i] = -1; else if (cur[i] > (int)k) cur[i] -= 1; }
        lx[cd * NMAX + n[cd]] = Nx; ly[cd * NMAX + n[cd]] = Ny; id[cd * NMAX + n[cd]] = moved_id;   // added at the end (L123)
        n[cd] += 1;
        counters[1] += 1;
        m |= (1u << (s & 31));
        continue;
      }
      bool overlap = false;                                     // line 13 (L193)
      for (int oy = -1; oy <= 1; ++oy) {                        // line 14 (L194): neighbourhood of (x, y)
        for (int ox = -1; ox <= 1; ++ox) {
          const uint32_t xn = (uint32_t)(((int64_t)x + ox + mx) % mx);
          const uint32_t yn = (uint32_t)(((int64_t)y + oy + my) % my);
          const size_t cn = cell(xn, yn);
          const P sx = (P)ox * wx, sy = (P)oy * wy;             // line 15 (L196), L154
          for (uint32_t j = 0; j < n[cn]; ++j) {                // line 16 (L198)
            if (ox == 0 && oy == 0 && j == k) continue;         // line 17 (L201)
            if (overlaps(Mx, My, lx[cn * NMAX + j], ly[cn * NMAX + j], sx, sy)) overlap = true;  // 18-21
          }
        }
      }
      if (overlap) {
        counters[3] += 1;
      } else {                                                  // lines 24-27 (L215-222)
        lx[c * NMAX + k] = Mx;
        ly[c * NMAX + k] = My;
        counters[1] += 1;
        m |= (1u << (s & 31));
      }
    }
    mask[c] = m;
    digest += mix64(mix64(t) ^ (((uint64_t)c << 32) | (uint64_t)m));
  }

  // one sub-sweep: every cell of checkerboard set Q (eq. 1); cells of a set are independent (L48)
  void sub_sweep(uint32_t Q) {
    const uint32_t offx = Q & 1u, offy = Q >> 1;
    for (uint32_t y = offy; y < my; y += 2)
      for (uint32_t x = offx; x < mx; x += 2) cell_update(x, y);
  }

  // ---- Algorithm 4, pull form: one pass per NEW cell -----------------------
  // dir 0:+x 1:-x 2:+y 3:-y.  Disks are translated by -f*delta (L303, L350); those that leave (0, w]
  // enter the adjacent cell with a SEPARATE +-w translation after the test (L332, L352).
  int shift(uint32_t dir, P delta) {
    const bool along_x = dir < 2;
    const bool positive = (dir & 1u) == 0;
    const P w = along_x ? wx : wy;
    const P step = positive ? -delta : delta;        // l' = l - f*delta
    const P back = positive ? w : -w;                // entrant: l'' = l' + w (from +f neighbour), l' - w (from -f)
    int status = OR_OK;
    for (uint32_t y = 0; y < my; ++y) {
      for (uint32_t x = 0; x < mx; ++x) {
        const size_t c = cell(x, y);
        uint32_t nn = 0;
        P nx[NMAX + 1], ny[NMAX + 1]; uint32_t nid[NMAX + 1];
        // lines 7-14 (L299-312): own disks that stay
        for (uint32_t i = 0; i < n[c]; ++i) {
          P ax = lx[c * NMAX + i], ay = ly[c * NMAX + i];
          P& a = along_x ? ax : ay;
          a = a + step;
          if (inside(a, w)) {
            if (nn < NMAX) { nx[nn] = ax; ny[nn] = ay; nid[nn] = id[c * NMAX + i]; }
            ++nn;
          }
        }
        // lines 15-27 (L314-339): disks of the neighbour in direction f that left it
        uint32_t xn = x, yn = y;
        if (along_x) xn = positive ? (x + 1) % mx : (x + mx - 1) % mx;
        else         yn = positive ? (y + 1) % my : (y + my - 1) % my;
        const size_t cn = cell(xn, yn);
        for (uint32_t i = 0; i < n[cn]; ++i) {
          P ax = lx[cn * NMAX + i], ay = ly[cn * NMAX + i];
          P& a = along_x ? ax : ay;
          a = a + step;
          if (inside(a, w)) continue;                // stays in the neighbour (L326-328)
          a = a + back;                              // L332
          if (nn < NMAX) { nx[nn] = ax; ny[nn] = ay; nid[nn] = id[cn * NMAX + i]; }
          ++nn;
        }
        if (nn > NMAX) { status = OR_ERR_CELL_OVERFLOW; nn = NMAX; }
        n_dbl[c] = nn;                               // L280, L342
        for (uint32_t i = 0; i < NMAX; ++i) {
          lx_dbl[c * NMAX + i] = i < nn ? nx[i] : (P)0;
          ly_dbl[c * NMAX + i] = i < nn ? ny[i] : (P)0;
          id_dbl[c * NMAX + i] = i < nn ? nid[i] : 0xFFFFFFFFu;
        }
      }
    }
    n.swap(n_dbl); lx.swap(lx_dbl); ly.swap(ly_dbl); id.swap(id_dbl);   // L350
    // the grid origin follows the cell boundaries: X = origin + cell*w + l is unchanged
    const double L = along_x ? Lx_eff : Ly_eff;
    double& o = origin[along_x ? 0 : 1];
    o = o + (positive ? (double)delta : -(double)delta);
    if (o >= L) o = o - L;
    if (o < 0.0) o = o + L;
    return status;
  }

  // ---- Algorithm 1: k sweeps -------------------------------------------------
  int sweep(uint64_t k) override {
    if (!loaded) return OR_ERR_STATE;
    for (uint64_t it = 0; it < k; ++it) {
      const SweepDraws D = sweep_draws(seed, t, !(flags & OR_NO_SET_SHUFFLE));
      for (uint32_t q = 0; q < 4; ++q) sub_sweep(D.order[q]);            // lines 3-14
      const bool along_x = D.dir < 2;
      const P half = (P)0.5 * (along_x ? wx : wy);                        // line 15: uniform(0, w/2)
      const P delta = half * Variate<P>::unit(D.dist_word);
      const int st = shift(D.dir, delta);                                 // line 17
      if (st != OR_OK && sticky == OR_OK) sticky = st;
      t += 1;
    }
    return sticky;
  }

  int cell_update_only(uint32_t set) override {  // test hook: one sub-sweep of set `set` at sweep index t
    if (!loaded) return OR_ERR_STATE;
    sub_sweep(set & 3u);
    return OR_OK;
  }
  int shift_only(uint32_t dir, double delta) override {  // test hook: one cell shift
    if (!loaded) return OR_ERR_STATE;
    return shift(dir & 3u, (P)delta);
  }

  // ---- cell-list build: global double coordinates -> (cell, local) ----------
  int load(const double* xy) override {
    const size_t M = (size_t)mx * my;
    std::fill(n.begin(), n.end(), 0u);
    std::fill(lx.begin(), lx.end(), (P)0); std::fill(ly.begin(), ly.end(), (P)0);
    std::fill(id.begin(), id.end(), 0xFFFFFFFFu);
    std::fill(mask.begin(), mask.end(), 0u);
    origin[0] = origin[1] = 0.0;
    loaded = false;
    const double Lx_user = wx_d0 * mx, Ly_user = wy_d0 * my;
    for (uint64_t i = 0; i < N; ++i) {           // ascending id => slots ascending by id (reading A13)
      const double X = xy[2 * i], Y = xy[2 * i + 1];
      if (!(X >= 0.0 && X <= Lx_user * (1 + 1e-12) && Y >= 0.0 && Y <= Ly_user * (1 + 1e-12))) return OR_ERR_OVERLAP;
      int64_t cx, cy; P px, py;
      to_local(X, wx_d, wx, mx, cx, px);
      to_local(Y, wy_d, wy, my, cy, py);
      const size_t c = cell((uint32_t)cx, (uint32_t)cy);
      if (n[c] >= NMAX) return OR_ERR_CELL_OVERFLOW;
      lx[c * NMAX + n[c]] = px; ly[c * NMAX + n[c]] = py; id[c * NMAX + n[c]] = (uint32_t)i;
      n[c] += 1;
    }
    // reject overlapping input with the predicate of the cell update, from both disks' frames
    for (uint32_t y = 0; y < my; ++y)
      for (uint32_t x = 0; x < mx; ++x) {
        const size_t c = cell(x, y);
        for (uint32_t k = 0; k < n[c]; ++k)
          for (int oy = -1; oy <= 1; ++oy)
            for (int ox = -1; ox <= 1; ++ox) {
              const size_t cn = cell((uint32_t)(((int64_t)x + ox + mx) % mx), (uint32_t)(((int64_t)y + oy + my) % my));
              for (uint32_t j = 0; j < n[cn]; ++j) {
                if (ox == 0 && oy == 0 && j == k) continue;
                if (overlaps(lx[c * NMAX + k], ly[c * NMAX + k], lx[cn * NMAX + j], ly[cn * NMAX + j],
                             (P)ox * wx, (P)oy * wy)) return OR_ERR_OVERLAP;
              }
            }
      }
    (void)M;
    t = 0; digest = 0; sticky = OR_OK;
    counters[0] = counters[1] = counters[2] = counters[3] = 0;
    loaded = true;
    return OR_OK;
  }

  // per coordinate, in double: c = floor(X / w), l = fma(-c, w, X); cast to P; one +-w step into (0, w]
  static void to_local(double X, double w_d, P w, uint32_t m, int64_t& c, P& l) {
    const double cf = std::floor(X / w_d);
    const double ld = std::fma(-cf, w_d, X);
    c = (int64_t)cf;
    l = (P)ld;
    if (!(l > (P)0)) { l = l + w; c -= 1; }
    else if (l > w) { l = l - w; c += 1; }
    c %= (int64_t)m;
    if (c < 0) c += (int64_t)m;
  }

  // unpack: X = wrap(origin + c*w + l) into [0, L_eff), written at index id (L154)
  int get(double* xy) const override {
    if (!loaded) return OR_ERR_STATE;
    for (uint32_t y = 0; y < my; ++y)
      for (uint32_t x = 0; x < mx; ++x) {
        const size_t c = cell(x, y);
        for (uint32_t i = 0; i < n[c]; ++i) {
          double X = std::fma((double)x, wx_d, origin[0]) + (double)lx[c * NMAX + i];
          double Y = std::fma((double)y, wy_d, origin[1]) + (double)ly[c * NMAX + i];
          if (X >= Lx_eff) X = X - Lx_eff;
          if (Y >= Ly_eff) Y = Y - Ly_eff;
          const uint32_t who = id[c * NMAX + i];
          xy[2 * (size_t)who] = X; xy[2 * (size_t)who + 1] = Y;
        }
      }
    return OR_OK;
  }

  int debug(uint32_t* counts, void* slab, uint32_t* ids, uint32_t* mask_out, double origin_out[2],
            uint64_t* sweep_index, uint64_t* digest_out) const override {
    const size_t M = (size_t)mx * my;
    if (counts) std::memcpy(counts, n.data(), M * sizeof(uint32_t));
    if (slab) {
      P* s = (P*)slab;   // canonical [M][NMAX][2]
      for (size_t c = 0; c < M; ++c)
        for (int i = 0; i < NMAX; ++i) {
          const bool used = (uint32_t)i < n[c];
          s[(c * NMAX + i) * 2 + 0] = used ? lx[c * NMAX + i] : (P)0;
          s[(c * NMAX + i) * 2 + 1] = used ? ly[c * NMAX + i] : (P)0;
        }
    }
    if (ids)
      for (size_t c = 0; c < M; ++c)
        for (int i = 0; i < NMAX; ++i) ids[c * NMAX + i] = (uint32_t)i < n[c] ? id[c * NMAX + i] : 0xFFFFFFFFu;
    if (mask_out) std::memcpy(mask_out, mask.data(), M * sizeof(uint32_t));
    if (origin_out) { origin_out[0] = origin[0]; origin_out[1] = origin[1]; }
    if (sweep_index) *sweep_index = t;
    if (digest_out) *digest_out = digest;
    return OR_OK;
  }

  // ---- pair-distance histogram near contact: n[r_i] for r in [sigma, sigma+nbins*dr) ----
  // Unordered pairs; all arithmetic in double from the stored locals; neighbourhood radius
  // Rc = ceil((sigma + nbins*dr) / min(wx, wy)) cells (reading A12: 3x3 is not enough at w ~ sigma).
  int histogram(double dr, uint32_t nbins, uint64_t* hist) const override {
    if (!loaded) return OR_ERR_STATE;
    if (!(dr > 0.0) || nbins == 0) return OR_ERR_ARG;
    for (uint32_t b = 0; b < nbins; ++b) hist[b] = 0;
    const double rmax = sigma_d + (double)nbins * dr;
    const double wmin = wx_d < wy_d ? wx_d : wy_d;
    const int Rc = (int)std::ceil(rmax / wmin);
    for (uint32_t y = 0; y < my; ++y)
      for (uint32_t x = 0; x < mx; ++x) {
        const size_t c = cell(x, y);
        for (uint32_t i = 0; i < n[c]; ++i)
          for (int oy = -Rc; oy <= Rc; ++oy)
            for (int ox = -Rc; ox <= Rc; ++ox) {
              const int64_t xn = (((int64_t)x + ox) % mx + mx) % mx, yn = (((int64_t)y + oy) % my + my) % my;
              const size_t cn = cell((uint32_t)xn, (uint32_t)yn);
              for (uint32_t j = 0; j < n[cn]; ++j) {
                if (!(id[c * NMAX + i] < id[cn * NMAX + j])) continue;   // each unordered pair image once
                const double Dx = ((double)lx[cn * NMAX + j] + (double)ox * wx_d) - (double)lx[c * NMAX + i];
                const double Dy = ((double)ly[cn * NMAX + j] + (double)oy * wy_d) - (double)ly[c * NMAX + i];
                const double xx = Dx * Dx, yy = Dy * Dy;
                const double r = std::sqrt(xx + yy);
                const double b = std::floor((r - sigma_d) / dr);
                if (b >= 0.0 && b < (double)nbins) hist[(uint32_t)b] += 1;
              }
            }
      }
    return OR_OK;
  }

  double wx_d0 = 0, wy_d0 = 0;   // Lx/mx, Ly/my before rounding to P
};

template <typename P, typename SimT = Sim<P>>
int make(Base** out, uint64_t N, const double box[2], double sigma, double d, uint32_t n_s, uint64_t seed,
         uint32_t flags, double w_target) {
  SimT* S = new (std::nothrow) SimT();
  if (!S) return OR_ERR_ARG;
  S->N = N; S->n_s = n_s; S->seed = seed; S->flags = flags; S->sigma_d = sigma; S->d_d = d;
  S->sigma = (P)sigma; S->sigma2 = S->sigma * S->sigma; S->d = (P)d;
  // Setup (reading A11): mx, my = largest even integers with w = P(L/m) >= max(sigma, w_target)
  const double wmin = (w_target > sigma) ? w_target : sigma;
  uint32_t m[2]; P w[2]; double w0[2];
  for (int a = 0; a < 2; ++a) {
    const double q = std::floor(box[a] / (2.0 * wmin));
    if (!(q >= 1.0) || q > 1e9) { delete S; return OR_ERR_BOX; }
    int64_t mm = 2 * (int64_t)q;
    while (mm >= 2 && (P)(box[a] / (double)mm) < (P)wmin) mm -= 2;
    if (mm < 2) { delete S; return OR_ERR_BOX; }
    m[a] = (uint32_t)mm; w0[a] = box[a] / (double)mm; w[a] = (P)w0[a];
  }
  if ((uint64_t)m[0] * m[1] >= 0xFFFFFFFFull / NMAX) { delete S; return OR_ERR_BOX; }
  S->mx = m[0]; S->my = m[1]; S->wx = w[0]; S->wy = w[1];
  S->wx_d0 = w0[0]; S->wy_d0 = w0[1];
  S->wx_d = (double)w[0]; S->wy_d = (double)w[1];
  S->Lx_eff = (double)m[0] * S->wx_d; S->Ly_eff = (double)m[1] * S->wy_d;
  const size_t M = (size_t)m[0] * m[1];
  S->n.assign(M, 0); S->n_dbl.assign(M, 0); S->mask.assign(M, 0);
  S->lx.assign(M * NMAX, (P)0); S->ly.assign(M * NMAX, (P)0); S->id.assign(M * NMAX, 0xFFFFFFFFu);
  S->lx_dbl.assign(M * NMAX, (P)0); S->ly_dbl.assign(M * NMAX, (P)0); S->id_dbl.assign(M * NMAX, 0xFFFFFFFFu);
  *out = S;
  return OR_OK;
}

}  // namespace

// =============================================================================================
// C ABI (host pointers only).  Mirrors the product's call list so one harness can drive both.
// =============================================================================================
extern "C" {

struct oracle_ctx { Base* sim; };

int oracle_create(oracle_ctx** out, uint64_t N, const double box[2], double sigma, double d, uint32_t n_s,
                  uint64_t seed, uint32_t flags, double w_target) {
  if (!out || !box || N == 0 || N >= 0xFFFFFFFFull || !(sigma > 0) || !(d > 0) || n_s > 32) return OR_ERR_ARG;
  const bool f64 = (flags & OR_FP64) != 0, f32 = (flags & OR_FP32) != 0;
  if ((flags & OR_DISC) && n_s > 0xFFFFu) return OR_ERR_ARG;     // the move index shares the counter word with the attempt
  if (f64 == f32) return OR_ERR_ARG;
  Base* b = nullptr;
  const int st = f32 ? make<float>(&b, N, box, sigma, d, n_s, seed, flags, w_target)
                     : make<double>(&b, N, box, sigma, d, n_s, seed, flags, w_target);
  if (st != OR_OK) return st;
  *out = new oracle_ctx{b};
  return OR_OK;
}
int oracle_destroy(oracle_ctx* c) { if (c) { delete c->sim; delete c; } return OR_OK; }
int oracle_geometry(const oracle_ctx* c, uint32_t m[2], double w[2], double L_eff[2]) {
  m[0] = c->sim->mx; m[1] = c->sim->my; w[0] = c->sim->wx_d; w[1] = c->sim->wy_d;
  L_eff[0] = c->sim->Lx_eff; L_eff[1] = c->sim->Ly_eff;
  return OR_OK;
}
int oracle_load_positions(oracle_ctx* c, const double* xy) { return c->sim->load(xy); }
int oracle_sweep(oracle_ctx* c, uint64_t k) { return c->sim->sweep(k); }
int oracle_get_positions(const oracle_ctx* c, double* xy) { return c->sim->get(xy); }
int oracle_acceptance(const oracle_ctx* c, uint64_t out[4]) {
  for (int i = 0; i < 4; ++i) out[i] = c->sim->counters[i];
  return c->sim->sticky;
}
int oracle_contact_histogram(const oracle_ctx* c, double dr, uint32_t nbins, uint64_t* hist) {
  return c->sim->histogram(dr, nbins, hist);
}
int oracle_debug_state(const oracle_ctx* c, uint32_t* counts, void* slab, uint32_t* ids, uint32_t* mask,
                       double origin[2], uint64_t* sweep_index, uint64_t* digest) {
  return c->sim->debug(counts, slab, ids, mask, origin, sweep_index, digest);
}
// test hooks: the pieces of Algorithm 1 one at a time
int oracle_sub_sweep(oracle_ctx* c, uint32_t set) { return c->sim->cell_update_only(set); }
int oracle_shift(oracle_ctx* c, uint32_t dir, double delta) { return c->sim->shift_only(dir, delta); }
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) { philox4x32_10(ctr, key, out); }
void oracle_sweep_draws(uint64_t seed, uint64_t t, uint32_t order[4], uint32_t* dir, uint32_t* dist_word) {
  const SweepDraws D = sweep_draws(seed, t);
  for (int i = 0; i < 4; ++i) order[i] = D.order[i];
  *dir = D.dir; *dist_word = D.dist_word;
}
void oracle_visit_sequence(const uint32_t* perm, uint32_t n, uint32_t n_moves, uint32_t* out) {
  for (uint32_t s = 0; s < n_moves; ++s) out[s] = visit(perm, n, s);
}
void oracle_fisher_yates(uint32_t* a, uint32_t n, const uint32_t* words) { if (n >= 2) fisher_yates(a, n, words); }
float oracle_variate_sym_f32(uint32_t R) { return Variate<float>::sym(R); }
double oracle_variate_sym_f64(uint32_t R) { return Variate<double>::sym(R); }
float oracle_variate_unit_f32(uint32_t R) { return Variate<float>::unit(R); }
double oracle_variate_unit_f64(uint32_t R) { return Variate<double>::unit(R); }

}  // extern "C"
