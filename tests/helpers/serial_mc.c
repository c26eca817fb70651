/* Test comparator, independent of oracle/ and of the CUDA path: the textbook SERIAL hard-disk Monte Carlo
 * of PAPER.md L25 (Fig. 1): "(i) Select a single disk at random, (ii) apply a random displacement to it,
 * and (iii) accept the move if it generates no overlaps ... A sweep is defined as N consecutive trial
 * moves".  No cell list (all-pairs minimum-image check), no checkerboard, no grid shift; its own RNG
 * (xoshiro256** seeded by splitmix64).  Displacement uniform in the square [-d, d]^2.
 * Output: per-sample histograms of unordered pair distances r in [sigma, rmax). */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

static uint64_t s[4];
static uint64_t rotl(uint64_t x, int k) { return (x << k) | (x >> (64 - k)); }
static uint64_t next(void) {
  const uint64_t r = rotl(s[1] * 5, 7) * 9, t = s[1] << 17;
  s[2] ^= s[0]; s[3] ^= s[1]; s[1] ^= s[2]; s[0] ^= s[3]; s[2] ^= t; s[3] = rotl(s[3], 45);
  return r;
}
static void seed_rng(uint64_t z) {
  for (int i = 0; i < 4; ++i) {
    z += 0x9E3779B97F4A7C15ull;
    uint64_t x = z;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    s[i] = x ^ (x >> 31);
  }
}
static double u01(void) { return (double)(next() >> 11) * 0x1p-53; }

int serial_mc_pair_histograms(int N, double Lx, double Ly, double sigma, double d, const double* xy0,
                              uint64_t seed, long equil_sweeps, long nsamples, long stride, double rmax,
                              int nbins, double* hist /* [nsamples][nbins] */, double* acceptance) {
  double* x = (double*)malloc(sizeof(double) * N), *y = (double*)malloc(sizeof(double) * N);
  if (!x || !y) return -1;
  for (int i = 0; i < N; ++i) { x[i] = xy0[2 * i]; y[i] = xy0[2 * i + 1]; }
  seed_rng(seed);
  const double s2 = sigma * sigma, bw = (rmax - sigma) / nbins;
  long tried = 0, accepted = 0;
  for (long sweep = 0; sweep < equil_sweeps + nsamples * stride; ++sweep) {
    for (int m = 0; m < N; ++m) {
      const int i = (int)(u01() * N);
      double nx = x[i] + d * (2.0 * u01() - 1.0), ny = y[i] + d * (2.0 * u01() - 1.0);
      nx -= Lx * floor(nx / Lx); ny -= Ly * floor(ny / Ly);
      int ok = 1;
      for (int j = 0; j < N && ok; ++j) {
        if (j == i) continue;
        double dx = nx - x[j], dy = ny - y[j];
        dx -= Lx * rint(dx / Lx); dy -= Ly * rint(dy / Ly);
        if (dx * dx + dy * dy < s2) ok = 0;
      }
      ++tried;
      if (ok) { x[i] = nx; y[i] = ny; ++accepted; }
    }
    if (sweep >= equil_sweeps && (sweep - equil_sweeps + 1) % stride == 0) {
      double* h = hist + ((sweep - equil_sweeps + 1) / stride - 1) * nbins;
      for (int b = 0; b < nbins; ++b) h[b] = 0.0;
      for (int i = 0; i < N; ++i)
        for (int j = i + 1; j < N; ++j) {
          double dx = x[i] - x[j], dy = y[i] - y[j];
          dx -= Lx * rint(dx / Lx); dy -= Ly * rint(dy / Ly);
          const double r = sqrt(dx * dx + dy * dy);
          const int b = (int)floor((r - sigma) / bw);
          if (b >= 0 && b < nbins) h[b] += 1.0;
        }
    }
  }
  if (acceptance) *acceptance = (double)accepted / (double)tried;
  free(x); free(y);
  return 0;
}
