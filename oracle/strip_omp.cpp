// CPU BASELINE — TEST / BENCH INFRASTRUCTURE ONLY (bench.py's cpu_baseline leg and tests/).  Not part of the product path.
//
// The paper's multi-core CPU implementation (section 5): "the same algorithm is parallelised with OpenMP:
// each thread processes a single horizontal strip of cells, and the innermost loop follows Algorithm 2".  This file is
// that program: the oracle's Algorithm 2 (cell_update) and Algorithm 4 (the shift's per-cell body), unchanged, with the
// rows of a checkerboard set — and the rows of the new grid in the shift — divided into one contiguous strip per OpenMP
// thread (schedule(static)).  Cells of a set are independent (L48) and the shift is double-buffered (L350), so the
// trajectory is the oracle's, bit for bit, whatever the thread count (checked by tests/test_strip_baseline.py and by
// bench.py on every run).  Move counters are per thread and summed after each sub-sweep.
//
// Build: g++ -O2 -fopenmp -ffp-contract=off (oracle.py: build_strip).  Exports strip_* with the oracle's call list.
#include "oracle_mpmc.cpp"

#include <omp.h>

namespace {

template <typename P>
struct StripSim : Sim<P> {
  using S = Sim<P>;
  using typename S::Acc;

  // one sub-sweep: every cell of checkerboard set Q (eq. 1), one strip of rows per thread
  void sub_sweep_strips(uint32_t Q) {
    const uint32_t offx = Q & 1u, offy = Q >> 1;
    const int rows = (int)((this->my - offy + 1u) / 2u);
    uint64_t c0 = 0, c1 = 0, c2 = 0, c3 = 0, dg = 0;
#pragma omp parallel reduction(+ : c0, c1, c2, c3, dg)
    {
      Acc acc;
#pragma omp for schedule(static)
      for (int r = 0; r < rows; ++r) {
        const uint32_t y = offy + 2u * (uint32_t)r;
        for (uint32_t x = offx; x < this->mx; x += 2) this->cell_update(x, y, acc);      // Algorithm 2
      }
      c0 += acc.counters[0]; c1 += acc.counters[1]; c2 += acc.counters[2]; c3 += acc.counters[3]; dg += acc.digest;
    }
    this->counters[0] += c0; this->counters[1] += c1; this->counters[2] += c2; this->counters[3] += c3;
    this->digest += dg;
  }

  // Algorithm 4, pull form, one strip of new-grid rows per thread.  The per-cell body is the oracle's (Sim::shift),
  // restated here because there it is the inside of a serial double loop.
  int shift_strips(uint32_t dir, P delta) {
    const bool along_x = dir < 2, positive = (dir & 1u) == 0;
    const P w = along_x ? this->wx : this->wy;
    const P step = positive ? -delta : delta;        // l' = l - f*delta  (L303)
    const P back = positive ? w : -w;                // entrant translation (L332), a separate operation (L352)
    const uint32_t mx = this->mx, my = this->my;
    int overflow = 0;
#pragma omp parallel for schedule(static) reduction(| : overflow)
    for (int yy = 0; yy < (int)my; ++yy) {
      const uint32_t y = (uint32_t)yy;
      for (uint32_t x = 0; x < mx; ++x) {
        const size_t c = this->cell(x, y);
        uint32_t nn = 0;
        P nx[NMAX + 1], ny[NMAX + 1]; uint32_t nid[NMAX + 1];
        for (uint32_t i = 0; i < this->n[c]; ++i) {            // lines 7-14 (L299-312): own disks that stay
          P ax = this->lx[c * NMAX + i], ay = this->ly[c * NMAX + i];
          P& a = along_x ? ax : ay;
          a = a + step;
          if (S::inside(a, w)) {
            if (nn < NMAX) { nx[nn] = ax; ny[nn] = ay; nid[nn] = this->id[c * NMAX + i]; }
            ++nn;
          }
        }
        uint32_t xn = x, yn = y;                               // lines 15-27 (L314-339): the neighbour's leavers
        if (along_x) xn = positive ? (x + 1) % mx : (x + mx - 1) % mx;
        else         yn = positive ? (y + 1) % my : (y + my - 1) % my;
        const size_t cn = this->cell(xn, yn);
        for (uint32_t i = 0; i < this->n[cn]; ++i) {
          P ax = this->lx[cn * NMAX + i], ay = this->ly[cn * NMAX + i];
          P& a = along_x ? ax : ay;
          a = a + step;
          if (S::inside(a, w)) continue;
          a = a + back;
          if (nn < NMAX) { nx[nn] = ax; ny[nn] = ay; nid[nn] = this->id[cn * NMAX + i]; }
          ++nn;
        }
        if (nn > NMAX) { overflow |= 1; nn = NMAX; }
        this->n_dbl[c] = nn;
        for (uint32_t i = 0; i < NMAX; ++i) {
          this->lx_dbl[c * NMAX + i] = i < nn ? nx[i] : (P)0;
          this->ly_dbl[c * NMAX + i] = i < nn ? ny[i] : (P)0;
          this->id_dbl[c * NMAX + i] = i < nn ? nid[i] : 0xFFFFFFFFu;
        }
      }
    }
    this->n.swap(this->n_dbl); this->lx.swap(this->lx_dbl); this->ly.swap(this->ly_dbl); this->id.swap(this->id_dbl);
    const double L = along_x ? this->Lx_eff : this->Ly_eff;
    double& o = this->origin[along_x ? 0 : 1];
    o = o + (positive ? (double)delta : -(double)delta);
    if (o >= L) o = o - L;
    if (o < 0.0) o = o + L;
    return overflow ? OR_ERR_CELL_OVERFLOW : OR_OK;
  }

  // Algorithm 1 (L60-93)
  int sweep(uint64_t k) override {
    if (!this->loaded) return OR_ERR_STATE;
    for (uint64_t it = 0; it < k; ++it) {
      const SweepDraws D = sweep_draws(this->seed, this->t, !(this->flags & OR_NO_SET_SHUFFLE));
      for (uint32_t q = 0; q < 4; ++q) sub_sweep_strips(D.order[q]);
      const bool along_x = D.dir < 2;
      const P half = (P)0.5 * (along_x ? this->wx : this->wy);
      const P delta = half * Variate<P>::unit(D.dist_word);
      const int st = shift_strips(D.dir, delta);
      if (st != OR_OK && this->sticky == OR_OK) this->sticky = st;
      this->t += 1;
    }
    return this->sticky;
  }
};

}  // namespace

extern "C" {

int strip_create(oracle_ctx** out, uint64_t N, const double box[2], double sigma, double d, uint32_t n_s, uint64_t seed,
                 uint32_t flags, double w_target, int threads) {
  if (!out || !box || N == 0 || N >= 0xFFFFFFFFull || !(sigma > 0) || !(d > 0) || n_s > 32) return OR_ERR_ARG;
  const bool f64 = (flags & OR_FP64) != 0, f32 = (flags & OR_FP32) != 0;
  if (f64 == f32) return OR_ERR_ARG;
  if (threads > 0) omp_set_num_threads(threads);
  Base* b = nullptr;
  const int st = f32 ? make<float, StripSim<float>>(&b, N, box, sigma, d, n_s, seed, flags, w_target)
                     : make<double, StripSim<double>>(&b, N, box, sigma, d, n_s, seed, flags, w_target);
  if (st != OR_OK) return st;
  *out = new oracle_ctx{b};
  return OR_OK;
}
int strip_threads(void) { return omp_get_max_threads(); }

}  // extern "C"
