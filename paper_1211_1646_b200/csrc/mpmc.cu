// mpmc.cu — host side of the C ABI declared in include/mpmc.h.  Product code (CUDA path); no CPU fallback.
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -fmad=false -lineinfo -shared (see ../build.py).
#include "../../include/mpmc.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "aux.cuh"
#include "common.cuh"
#include "sweep.cuh"
#include "tile.cuh"
#include "tile4.cuh"
#include "cluster.cuh"
#include "kernels.h"

using namespace mpmc;

// Scratch of mpmc_contact_histogram_noalloc (include/mpmc.h): the device histogram the contact-histogram kernels add their
// counts to, as a file-scope device array instead of a piece of the caller's workspace, so that the call allocates nothing.
// Every GPU that loads the library holds these 8 KB until the process exits.  In HOST code this name is a host-side stand-in,
// not a device address (a kernel given it would fault, or silently use host memory where the GPU can reach it): the host
// passes what cudaGetSymbolAddress returns (noalloc_scratch below).
static __device__ __align__(256) unsigned long long g_noalloc_hist[MPMC_NOALLOC_MAX_BINS];

struct mpmc_ctx {
  Params p;
  uint64_t N;
  uint32_t flags;
  bool fp32, debug, loaded;
  int nf;                  // 2: w < 1.15 sigma, cells hold 0/1/2 disks -> fast sub-sweep kernel; 4: general kernel
  cudaStream_t stream;
  const void* kernel;      // the k_sweeps instantiation for this context
  uint32_t grid;           // co-resident blocks of the persistent kernel
  const void* tile_kernel; // the k_tile_sweep instantiation, or nullptr when the tile path does not apply
  uint32_t tile_grid;      // tiles = CTAs of the tile kernel
  size_t tile_smem;        // its dynamic shared memory
  uint32_t tile_threads;   // threads per CTA of the tile kernel
  bool tile_two_slot;      // the tile kernel is the 2-slot one (tile.cuh), which may hand a crowded state to the general kernel
  uint32_t sms;            // SMs of the device
  const void* cluster_kernel;  // the k_cluster_sweeps instantiation when the system is small enough to live in one cluster's
  uint32_t cl_ctas;            // shared memory (cluster.cuh), else nullptr; its CTAs (= cluster size), threads per CTA and
  uint32_t cl_threads;         // dynamic shared memory per CTA
  size_t cl_smem;
  uint64_t t_host;         // sweeps requested since the last load (the sweep index the device will reach)
  uint32_t cur_host;       // ... and the buffer that will hold that state (every sweep and every test-hook shift flips it)
  unsigned long long* hist_acc;   // device: histogram accumulated over samples (mpmc_pressure_accumulate)
  uint64_t acc_samples;    // samples in it
  double acc_dr; uint32_t acc_nbins;   // its bins (fixed by the first sample after a reset)
  int sticky;
};

namespace {

constexpr size_t ALIGN = 256;
constexpr uint32_t MAX_BINS = 4096;
constexpr uint32_t SORT_MIN_PLANE = 1000;   // cells per shared-memory colour plane from which the sorted tile kernel is used

inline size_t up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Geom {
  uint32_t m[2];
  double w0[2];    // L/m in double
  double wp[2];    // rounded to the working precision, as double
};

// Setup (reading A11): mx, my = largest even integers with w = P(L/m) >= P(max(sigma, w_target)).
int geometry(const double box[2], double sigma, double w_target, bool fp32, Geom* g) {
  if (!box || !(sigma > 0) || !(box[0] > 0) || !(box[1] > 0)) return MPMC_ERR_ARG;
  const double wmin = (w_target > sigma) ? w_target : sigma;
  for (int a = 0; a < 2; ++a) {
    const double q = std::floor(box[a] / (2.0 * wmin));
    if (!(q >= 1.0) || q > 1e9) return MPMC_ERR_BOX;
    long long mm = 2 * (long long)q;
    for (;;) {
      if (mm < 2) return MPMC_ERR_BOX;
      const double w0 = box[a] / (double)mm;
      const bool ok = fp32 ? ((float)w0 >= (float)wmin) : (w0 >= wmin);
      if (ok) break;
      mm -= 2;
    }
    g->m[a] = (uint32_t)mm;
    g->w0[a] = box[a] / (double)mm;
    g->wp[a] = fp32 ? (double)(float)g->w0[a] : g->w0[a];
  }
  if ((uint64_t)g->m[0] * g->m[1] >= 0xFFFFFFFFull / NMAX) return MPMC_ERR_BOX;
  return MPMC_OK;
}

struct Layout {
  uint32_t Mq, Mqp;
  size_t off_ctl, off_hist, off_hist_acc, off_cnt32, off_cnt[2], off_pos[2], off_ids[2], off_mask, total;
};

Layout layout(const Geom& g, bool fp32, bool debug) {
  Layout L;
  L.Mq = (g.m[0] / 2) * (g.m[1] / 2);
  L.Mqp = (uint32_t)up(L.Mq, 64);
  const size_t real2 = fp32 ? 8 : 16;
  size_t o = 0;
  L.off_ctl = o; o += up(sizeof(Ctl), ALIGN);
  L.off_hist = o; o += up((size_t)MAX_BINS * 8, ALIGN);
  L.off_hist_acc = o; o += up((size_t)MAX_BINS * 8, ALIGN);
  L.off_cnt32 = o; o += up((size_t)4 * L.Mqp * 4, ALIGN);
  for (int b = 0; b < 2; ++b) { L.off_cnt[b] = o; o += up((size_t)4 * L.Mqp, ALIGN); }
  for (int b = 0; b < 2; ++b) { L.off_pos[b] = o; o += up((size_t)4 * NMAX * L.Mqp * real2, ALIGN); }
  for (int b = 0; b < 2; ++b) { L.off_ids[b] = o; o += up((size_t)4 * NMAX * L.Mqp * 4, ALIGN); }
  L.off_mask = o;
  if (debug) o += up((size_t)g.m[0] * g.m[1] * 4, ALIGN);
  L.total = o;
  return L;
}

// unsigned division by an invariant d >= 1 (Granlund & Montgomery 1994): q = (t + ((n - t) >> sh1)) >> sh2,
// t = mulhi(magic, n)
void div_magic(uint32_t d, uint32_t* magic, uint32_t* sh1, uint32_t* sh2) {
  uint32_t l = 0;
  while ((1ull << l) < d) ++l;
  *magic = (uint32_t)(((1ull << 32) * ((1ull << l) - d)) / d + 1);
  *sh1 = l < 1 ? l : 1;
  *sh2 = l < 1 ? 0 : l - 1;
}

bool precision_ok(uint32_t flags) { return ((flags & MPMC_FP64) != 0) != ((flags & MPMC_FP32) != 0); }

int cuda_fail(cudaError_t e) {
  if (e == cudaSuccess) return MPMC_OK;
  std::fprintf(stderr, "[mpmc] CUDA error: %s\n", cudaGetErrorString(e));
  return MPMC_ERR_CUDA;
}
#define CU(x) do { cudaError_t e__ = (x); if (e__ != cudaSuccess) return cuda_fail(e__); } while (0)

dim3 cell_grid(const mpmc_ctx* c, int threads) { return dim3((c->p.Mq + threads - 1) / threads, 4, 1); }

// one cooperative launch: sweeps up to sweep index t_end, or one piece of a sweep (test hooks)
int launch_sweeps(mpmc_ctx* c, unsigned long long t_end, uint32_t op, uint32_t arg, double delta) {
  CU(cudaMemsetAsync(&c->p.ctl->bar, 0, sizeof(uint32_t), c->stream));
  void* args[] = {(void*)&c->p, (void*)&t_end, (void*)&op, (void*)&arg, (void*)&delta};
  CU(cudaLaunchCooperativeKernel(c->kernel, dim3(c->grid), dim3(SUB_THREADS), args, 0, c->stream));
  return MPMC_OK;
}

// Tiling of the tile kernels.  Tiles form rows of (nearly) equal even size; every loaded region (tile + 2 HALO) must fit
// the shared memory of one SM and must not overlap itself around the box.  Two families are searched for the least work
// on the busiest SM = waves * cells of the largest region: uniform ntx x nty grids, and — while the whole grid is one wave
// — MIXED tilings: na rows of a tiles over the half-rows [0, hyA) and nb rows of a + 1 narrower, taller tiles over the rest,
// hyA placed so that both shapes load the same area (C3 on 148 SMs: 8 x 12 + 4 x 13 = 148 tiles instead of 12 x 12 = 144).
// row_bytes / pw_max: the sorted variant of the 2-slot kernel also needs row_bytes of shared memory per plane row and plane
// rows of at most pw_max cells.  Returns false if no tiling exists (boxes under 12 cells across).
struct Tiling { uint32_t ntx, nty, na, hyA, PS, PH, tiles; };

bool choose_tiling(uint32_t hx, uint32_t hy, size_t cell_bytes, size_t smem_max, uint32_t sms, Tiling* out,
                   size_t row_bytes = 0, uint32_t pw_max = 0xFFFFFFFFu) {
  double best = 0; bool found = false;
  const uint32_t lim = 1024;
  auto fits = [&](uint32_t TX, uint32_t TY) {
    const uint32_t pw = (TX + 2 * HALO) / 2, ph = (TY + 2 * HALO) / 2;
    if (TX + 2 * HALO > 2 * hx || TY + 2 * HALO > 2 * hy) return false;     // a region must not overlap itself around the box
    const size_t bytes = (size_t)4 * pw * ph * cell_bytes + (size_t)4 * ph * row_bytes;
    return bytes <= smem_max && pw * ph < 16384u && pw <= pw_max;
  };
  for (uint32_t ax = 1; ax <= hx && ax <= lim; ++ax) {
    const uint32_t TX = 2 * ((hx + ax - 1) / ax);
    for (uint32_t ay = 1; ay <= hy && ay <= lim; ++ay) {
      const uint32_t TY = 2 * ((hy + ay - 1) / ay);
      if (!fits(TX, TY)) continue;
      const double waves = std::ceil((double)ax * ay / sms);
      const double cost = waves * (double)(TX + 2 * HALO) * (TY + 2 * HALO) + 1e-6 * ax * ay;
      if (!found || cost < best) {
        best = cost; found = true;
        *out = Tiling{ax, ay, ay, hy, ((TX + 2 * HALO) / 2) * ((TY + 2 * HALO) / 2), (TY + 2 * HALO) / 2, ax * ay};
      }
    }
  }
  // mixed tilings of at most one wave
  for (uint32_t a = 1; a + 1 <= hx && a < sms; ++a) {
    const uint32_t TXa = 2 * ((hx + a - 1) / a), TXb = 2 * ((hx + a) / (a + 1));
    for (uint32_t na = 1; na * a < sms; ++na) {
      for (uint32_t nb = 1; na * a + nb * (a + 1) <= sms; ++nb) {
        if (na + nb > hy) break;
        // equal loaded areas: (TXa + 10)(2 hyA / na + 10) = (TXb + 10)(2 (hy - hyA) / nb + 10)
        const double A = TXa + 2.0 * HALO, B = TXb + 2.0 * HALO;
        const double hA = (B * (2.0 * hy / nb + 2.0 * HALO) - 2.0 * HALO * A) / (2.0 * A / na + 2.0 * B / nb);
        for (int d = -1; d <= 1; ++d) {
          const long long h = (long long)std::floor(hA + 0.5) + d;
          if (h < (long long)na || h > (long long)hy - (long long)nb) continue;
          const uint32_t hyA = (uint32_t)h;
          const uint32_t TYa = 2 * ((hyA + na - 1) / na), TYb = 2 * ((hy - hyA + nb - 1) / nb);
          if (!fits(TXa, TYa) || !fits(TXb, TYb)) continue;
          const double ra = (double)(TXa + 2 * HALO) * (TYa + 2 * HALO), rb = (double)(TXb + 2 * HALO) * (TYb + 2 * HALO);
          const uint32_t tiles = na * a + nb * (a + 1);
          const double cost = (ra > rb ? ra : rb) + 1e-6 * tiles;
          if (!found || cost < best * (1.0 - 1e-3)) {            // (a uniform tiling wins ties: simpler index arithmetic)
            best = cost; found = true;
            const uint32_t psa = ((TXa + 2 * HALO) / 2) * ((TYa + 2 * HALO) / 2), psb = ((TXb + 2 * HALO) / 2) * ((TYb + 2 * HALO) / 2);
            const uint32_t pha = (TYa + 2 * HALO) / 2, phb = (TYb + 2 * HALO) / 2;
            *out = Tiling{a, na + nb, na, hyA, psa > psb ? psa : psb, pha > phb ? pha : phb, tiles};
          }
        }
      }
    }
  }
  return found;
}

int read_ctl(mpmc_ctx* c, Ctl* h) {
  CU(cudaMemcpyAsync(h, c->p.ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, c->stream));
  CU(cudaStreamSynchronize(c->stream));
  if (h->err & ERRBIT_OVERFLOW) c->sticky = MPMC_ERR_CELL_OVERFLOW;
  else if (h->err & (ERRBIT_OVERLAP | ERRBIT_RANGE)) c->sticky = MPMC_ERR_OVERLAP;
  else if (h->err & ERRBIT_STATE) c->sticky = MPMC_ERR_STATE;
  return c->sticky;
}

// Unweighted least-squares polynomial of the given degree through (t_i, y_i); returns the value at t = 0.
// Householder QR on the Vandermonde matrix (host, double).
bool polyfit_at_zero(const std::vector<double>& t, const std::vector<double>& y, uint32_t degree, double* value) {
  const size_t n = t.size(), m = degree + 1;
  if (n < m) return false;
  std::vector<double> A(n * m), b(y);
  for (size_t i = 0; i < n; ++i) { double pw = 1.0; for (size_t j = 0; j < m; ++j) { A[i * m + j] = pw; pw *= t[i]; } }
  for (size_t k = 0; k < m; ++k) {
    double norm = 0; for (size_t i = k; i < n; ++i) norm += A[i * m + k] * A[i * m + k];
    norm = std::sqrt(norm);
    if (norm == 0) return false;
    const double alpha = A[k * m + k] > 0 ? -norm : norm;
    std::vector<double> v(n - k);
    for (size_t i = k; i < n; ++i) v[i - k] = A[i * m + k];
    v[0] -= alpha;
    double vn = 0; for (double x : v) vn += x * x;
    if (vn == 0) continue;
    for (size_t j = k; j < m; ++j) {
      double s = 0; for (size_t i = k; i < n; ++i) s += v[i - k] * A[i * m + j];
      s = 2 * s / vn;
      for (size_t i = k; i < n; ++i) A[i * m + j] -= s * v[i - k];
    }
    double s = 0; for (size_t i = k; i < n; ++i) s += v[i - k] * b[i];
    s = 2 * s / vn;
    for (size_t i = k; i < n; ++i) b[i] -= s * v[i - k];
  }
  std::vector<double> c(m);
  for (size_t kk = m; kk-- > 0;) {
    double s = b[kk];
    for (size_t j = kk + 1; j < m; ++j) s -= A[kk * m + j] * c[j];
    if (A[kk * m + kk] == 0) return false;
    c[kk] = s / A[kk * m + kk];
  }
  *value = c[0];
  return true;
}

// eq. 5-6 (L374-379) on a histogram summed over `samples` configurations: g(R_i) = 2 H_i / (samples N rho 2 pi R_i dr),
// R_i = (2/3)(r_{i+1}^3 - r_i^3)/(r_{i+1}^2 - r_i^2); unweighted polynomial fit extrapolated to r = sigma (L382);
// P* = sigma^2 rho (1 + (pi/2) sigma^2 rho g(sigma+))  (eq. 4).  Host arithmetic.
int fit_contact(const mpmc_ctx* c, const uint64_t* H, uint64_t samples, double dr, uint32_t nbins, uint32_t degree,
                double* g_contact, double* p_star) {
  const Params& p = c->p;
  const double Nd = (double)c->N, rho = Nd / (p.Lx_eff * p.Ly_eff), sg = p.sigma_d;
  const double PI = 3.14159265358979323846;
  std::vector<double> t(nbins), g(nbins);
  for (uint32_t i = 0; i < nbins; ++i) {
    const double r0 = sg + dr * (double)i, r1 = sg + dr * (double)(i + 1);
    const double Ri = (2.0 / 3.0) * (r1 * r1 * r1 - r0 * r0 * r0) / (r1 * r1 - r0 * r0);
    t[i] = (Ri - sg) / (dr * (double)nbins);     // scaled abscissa; the value at 0 is unchanged
    g[i] = 2.0 * ((double)H[i] / (double)samples) / (Nd * rho * 2.0 * PI * Ri * dr);
  }
  double g0 = 0;
  if (!polyfit_at_zero(t, g, degree, &g0)) return MPMC_ERR_ARG;
  if (g_contact) *g_contact = g0;
  if (p_star) *p_star = sg * sg * rho * (1.0 + 0.5 * PI * sg * sg * rho * g0);
  return MPMC_OK;
}

// the pair-distance histogram of the current state, ADDED to `target` (device, nbins u64); asynchronous
int launch_histogram(mpmc_ctx* c, double dr, uint32_t nbins, unsigned long long* target) {
  const Params& p = c->p;
  const double rmax = p.sigma_d + (double)nbins * dr;
  const double wmin = p.wx_d < p.wy_d ? p.wx_d : p.wy_d;
  const int Rc = (int)std::ceil(rmax / wmin);
  if (Rc > 120) return MPMC_ERR_ARG;                     // the range must stay within a few cells (offsets are packed in 8 bits)
  // offsets of the half neighbourhood whose cells can hold a pair closer than rmax (radius 1 and 2: compile-time loops)
  unsigned long long keep = 0;
  const double rmax2 = rmax * rmax * 1.000001;
  if (Rc <= 2)
    for (int oy = 0; oy <= Rc; ++oy)
      for (int ox = -Rc; ox <= Rc; ++ox) {
        if (oy == 0 && ox <= 0) continue;
        const int gi = (ox < 0 ? -ox : ox) - 1, gj = oy - 1;
        const double gx = (gi > 0 ? gi : 0) * p.wx_d, gy = (gj > 0 ? gj : 0) * p.wy_d;
        if (gx * gx + gy * gy < rmax2) keep |= 1ull << hist_offset_index(ox, oy, Rc);
      }
  const size_t sh = (size_t)nbins * 4;
  if (Rc <= 2) {                     // tiles staged in shared memory
    const dim3 gT((p.mx + HT_W - 1) / HT_W, (p.my + HT_H - 1) / HT_H);
#define MPMC_HIST(P, RC) k_contact_hist_tile<P, RC><<<gT, HT_THREADS, sh, c->stream>>>(p, dr, nbins, rmax, keep, target)
    if (c->fp32) { if (Rc == 1) MPMC_HIST(float, 1); else MPMC_HIST(float, 2); }
    else         { if (Rc == 1) MPMC_HIST(double, 1); else MPMC_HIST(double, 2); }
#undef MPMC_HIST
  } else {
    const dim3 gC = cell_grid(c, HIST_THREADS);
    if (c->fp32) k_contact_hist<float, 0><<<gC, HIST_THREADS, sh, c->stream>>>(p, dr, nbins, Rc, rmax, keep, target);
    else         k_contact_hist<double, 0><<<gC, HIST_THREADS, sh, c->stream>>>(p, dr, nbins, Rc, rmax, keep, target);
  }
  CU(cudaGetLastError());
  return MPMC_OK;
}

// The device address of g_noalloc_hist on the context's device: resolved once per device, with that device current, and kept.
constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex g_noalloc_mutex;
unsigned long long* g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {};

int noalloc_scratch(const mpmc_ctx* c, unsigned long long** out) {
  int dev = -1;
  CU(cudaGetDevice(&dev));
  cudaPointerAttributes at;
  CU(cudaPointerGetAttributes(&at, c->p.ctl));             // the device the context's workspace lives on
  if (at.type != cudaMemoryTypeDevice || at.device != dev) return MPMC_ERR_ARG;   // ... must be the current one
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return MPMC_ERR_ARG;
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_ptr[dev]) {
    void* ptr = nullptr;
    CU(cudaGetSymbolAddress(&ptr, g_noalloc_hist));
    if (!ptr) return MPMC_ERR_CUDA;
    g_noalloc_ptr[dev] = static_cast<unsigned long long*>(ptr);
  }
  *out = g_noalloc_ptr[dev];
  return MPMC_OK;
}

}  // namespace

// =========================================================================================================
extern "C" {

size_t mpmc_workspace_bytes_ex(uint64_t N, const double box[2], double sigma, double w_target, uint32_t flags) {
  if (N == 0 || N >= 0xFFFFFFFFull || !precision_ok(flags)) return 0;
  Geom g;
  if (geometry(box, sigma, w_target, (flags & MPMC_FP32) != 0, &g) != MPMC_OK) return 0;
  return layout(g, (flags & MPMC_FP32) != 0, (flags & MPMC_DEBUG) != 0).total;
}
size_t mpmc_workspace_bytes(uint64_t N, const double box[2], double sigma, uint32_t flags) {
  return mpmc_workspace_bytes_ex(N, box, sigma, 0.0, flags);
}

int mpmc_create_ex(mpmc_ctx** out, uint64_t N, const double box[2], double sigma, double d, uint32_t n_s,
                   uint64_t seed, uint32_t flags, double w_target, void* workspace, size_t workspace_bytes,
                   void* cuda_stream) {
  if (!out || !box || N == 0 || N >= 0xFFFFFFFFull || !(sigma > 0) || !(d > 0) || n_s > 32 || !precision_ok(flags))
    return MPMC_ERR_ARG;
  const bool fp32 = (flags & MPMC_FP32) != 0, debug = (flags & MPMC_DEBUG) != 0, disc = (flags & MPMC_DISC) != 0;
  Geom g;
  const int st = geometry(box, sigma, w_target, fp32, &g);
  if (st != MPMC_OK) return st;
  // displacement = (d 2^-k) * odd integer must equal d * (integer 2^-k): the scaled d has to be a normal number
  if (fp32 ? !((float)d * 0x1p-24f >= 1.17549435e-38f) : !(d * 0x1p-32 >= 2.2250738585072014e-308)) return MPMC_ERR_ARG;
  const Layout L = layout(g, fp32, debug);
  if (!workspace || ((uintptr_t)workspace % ALIGN) != 0 || workspace_bytes < L.total) return MPMC_ERR_WORKSPACE;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return MPMC_ERR_CUDA; }

  mpmc_ctx* c = new (std::nothrow) mpmc_ctx();
  if (!c) return MPMC_ERR_ARG;
  std::memset(&c->p, 0, sizeof(Params));
  c->N = N; c->flags = flags; c->fp32 = fp32; c->debug = debug; c->loaded = false; c->sticky = MPMC_OK;
  c->stream = (cudaStream_t)cuda_stream;
  Params& p = c->p;
  p.mx = g.m[0]; p.my = g.m[1]; p.hx = g.m[0] / 2; p.hy = g.m[1] / 2;
  p.Mq = L.Mq; p.Mqp = L.Mqp; p.n_s = n_s; p.N = (uint32_t)N; p.flags = flags;
  div_magic(p.hx, &p.hx_magic, &p.hx_sh1, &p.hx_sh2);
  p.seed_lo = (uint32_t)seed; p.seed_hi = (uint32_t)(seed >> 32);
  for (uint32_t r = 0; r < 10; ++r) { p.rk0[r] = p.seed_lo + r * 0x9E3779B9u; p.rk1[r] = p.seed_hi + r * 0xBB67AE85u; }
  p.wx_f = (float)g.w0[0]; p.wy_f = (float)g.w0[1];
  p.sigma2_f = (float)sigma * (float)sigma; p.d_f = (float)d;
  p.dsc_f = p.d_f * 0x1p-24f; p.dsc_p = d * 0x1p-32;
  p.wx_p = g.w0[0]; p.wy_p = g.w0[1]; p.sigma2_p = sigma * sigma; p.d_p = d;
  p.wx_d = g.wp[0]; p.wy_d = g.wp[1];
  p.Lx_eff = (double)g.m[0] * g.wp[0]; p.Ly_eff = (double)g.m[1] * g.wp[1];
  p.sigma_d = sigma;
  p.Lx_user = g.w0[0] * g.m[0]; p.Ly_user = g.w0[1] * g.m[1];
  char* base = (char*)workspace;
  p.ctl = (Ctl*)(base + L.off_ctl);
  p.hist = (unsigned long long*)(base + L.off_hist);
  c->hist_acc = (unsigned long long*)(base + L.off_hist_acc);
  c->acc_samples = 0; c->acc_dr = 0.0; c->acc_nbins = 0;
  p.cnt32 = (uint32_t*)(base + L.off_cnt32);
  for (int b = 0; b < 2; ++b) {
    p.cnt[b] = (uint8_t*)(base + L.off_cnt[b]);
    p.pos[b] = (void*)(base + L.off_pos[b]);
    p.ids[b] = (uint32_t*)(base + L.off_ids[b]);
  }
  p.mask = debug ? (uint32_t*)(base + L.off_mask) : nullptr;
  // fast kernel while at most 2 disks fit a cell nearly always (w < ~1.15 sigma; rarer cells take its generic
  // path); general kernel in the paper's regime (w up to sqrt(2) sigma, L152).
  const double wmax = g.wp[0] > g.wp[1] ? g.wp[0] : g.wp[1];
  c->nf = (wmax < 1.15 * sigma) ? 2 : 4;
  {
    const bool fast = c->nf == 2 && (n_s == 4 || n_s == 8);
    c->kernel = fp32 ? pick_kernel_f32(debug, fast, disc, n_s) : pick_kernel_f64(debug, fast, disc, n_s);
  }
  // grid of the persistent kernel: every block co-resident (cooperative launch), no more blocks than chunks
  int dev = 0, sms = 0, occ = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, c->kernel, SUB_THREADS, 0) != cudaSuccess || occ < 1) {
    cudaGetLastError(); delete c; return MPMC_ERR_CUDA;
  }
  const uint32_t chunks = (L.Mq + SUB_THREADS - 1) / SUB_THREADS;
  c->sms = (uint32_t)sms;
  c->grid = (uint32_t)sms * (uint32_t)occ;
  if (c->grid > chunks) c->grid = chunks;
  // The fused tile kernels: tile.cuh (2 slots per cell in shared memory) where cells hold 0/1/2 disks (w < 1.15 sigma),
  // the square proposal and n_s in {4, 8}; otherwise tile4.cuh (all 4 slots; any width, both proposals) for n_s = 4.
  c->tile_kernel = nullptr; c->tile_grid = 0; c->tile_smem = 0; c->t_host = 0; c->cur_host = 0; c->tile_threads = 0;
  const bool two_slot = c->nf == 2 && (n_s == 4 || n_s == 8) && !disc;
  c->tile_two_slot = two_slot;
  p.tune = 0u;
  // the tile kernel variant that sorts the cells of a sweep into empty / simple / general ones (tile.cuh, SORTED)
  bool compact = true;
#ifdef MPMC_EXPERIMENT
  if (const char* e = std::getenv("MPMC_TUNE")) p.tune = (uint32_t)std::strtoul(e, nullptr, 0);
  if (const char* e = std::getenv("MPMC_COMPACT")) compact = e[0] == '1';
#endif
  p.track_crowded = two_slot ? 1u : 0u;      // only the 2-slot tile kernel reads the list of crowded cells
  // the sorted variant of the 2-slot kernel first; the plain one if no tiling with plane rows of <= 64 cells fits
  for (int attempt = 0; attempt < 2 && !c->tile_kernel; ++attempt) {
    const bool sorted = two_slot && compact && attempt == 0;
    if (attempt == 1 && !(two_slot && compact)) break;
    const void* tk = two_slot ? (fp32 ? pick_tile_kernel_f32(debug, n_s, sorted) : pick_tile_kernel_f64(debug, n_s, sorted))
                              : (fp32 ? pick_tile4_kernel_f32(debug, disc, false, n_s) : pick_tile4_kernel_f64(debug, disc, false, n_s));
    if (!tk) break;
    int smem_optin = 0;
    cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    // per cell of a shared-memory plane: the slot pair(s), and in the sorted 2-slot kernel one u16 queue entry
    const size_t cell_bytes = (fp32 ? sizeof(SmemCell<float>) : sizeof(SmemCell<double>)) * (two_slot ? 1 : 2)
                              + (sorted ? sizeof(uint16_t) : 0);
    const size_t stat = (two_slot ? (fp32 ? sizeof(CrowdList<float>) : sizeof(CrowdList<double>)) : 0) + 512;   // static shared memory
    const size_t smem_max = (size_t)smem_optin > stat ? (size_t)smem_optin - stat : 0;
    Tiling tl = {};
    const size_t row_bytes = sorted ? SORT_ROW_BYTES : 0;
    c->tile_threads = two_slot ? (fp32 ? TileThreads<float>::value : TileThreads<double>::value)
                               : (fp32 ? Tile4Threads<float, false>::value : Tile4Threads<double, false>::value);
    bool have = choose_tiling(p.hx, p.hy, cell_bytes, smem_max, (uint32_t)sms, &tl, row_bytes, sorted ? 64u : 0xFFFFFFFFu);
    // the sort is a fixed cost of ~8 000 cycles per tile and sweep (measured, phase_clocks.py): it pays from about a
    // thousand cells per colour plane on; smaller tiles (systems below ~2e5 cells) keep the plain variant
    if (sorted && have && tl.PS < SORT_MIN_PLANE) have = false;
#ifdef MPMC_EXPERIMENT
    if (const char* e = std::getenv("MPMC_TILE")) {        // "ntx,nty,threads" (whole warps)
      unsigned a = 0, b = 0, th = 0;
      if (std::sscanf(e, "%u,%u,%u", &a, &b, &th) == 3 && a && b && th >= 32 && th % 32 == 0 && th <= c->tile_threads && a <= p.hx && b <= p.hy) {
        const uint32_t pw = (2 * ((p.hx + a - 1) / a) + 2 * HALO) / 2, ph = (2 * ((p.hy + b - 1) / b) + 2 * HALO) / 2;
        if ((size_t)4 * pw * ph * cell_bytes + (size_t)4 * ph * row_bytes <= smem_max) { tl = Tiling{a, b, b, p.hy, pw * ph, ph, a * b}; c->tile_threads = th; have = true; }
      }
    }
#endif
    if (have && !two_slot && fp32 && tl.PS >= TILE4_WIDE_MIN_PLANE) {      // large tiles: the 512-thread instantiation (tile4.cuh)
      tk = pick_tile4_kernel_f32(debug, disc, true, n_s);
      c->tile_threads = Tile4Threads<float, true>::value;
    }
    if (have) {
      c->tile_kernel = tk;
      c->tile_grid = tl.tiles;
      c->tile_smem = (size_t)4 * tl.PS * cell_bytes + (size_t)4 * tl.PH * row_bytes;
      p.tl_ntx = tl.ntx; p.tl_nty = tl.nty; p.tl_PS = tl.PS; p.tl_PH = tl.PH; p.tl_na = tl.na; p.tl_hyA = tl.hyA;
      {
        const uint32_t dv[4] = {tl.ntx, tl.ntx + 1u, tl.na, tl.nty > tl.na ? tl.nty - tl.na : 1u};
        for (int i = 0; i < 4; ++i) div_magic(dv[i], &p.tl_div[i][0], &p.tl_div[i][1], &p.tl_div[i][2]);
      }
      // The attribute belongs to the kernel function, not to this context: set it to the most any tiling can ask for
      // (the opt-in maximum minus the kernel's static shared memory), so that live contexts with different tilings
      // of the same instantiation do not undo each other's setting.
      cudaFuncAttributes fa;
      if (cudaFuncGetAttributes(&fa, c->tile_kernel) != cudaSuccess ||
          (size_t)smem_optin < fa.sharedSizeBytes + c->tile_smem ||
          cudaFuncSetAttribute(c->tile_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                               smem_optin - (int)fa.sharedSizeBytes) != cudaSuccess) {
        cudaGetLastError(); delete c; return MPMC_ERR_CUDA;
      }
    }
  }
  // Small systems: the whole state resident in the shared memory of ONE cluster of up to 16 CTAs (cluster.cuh), all sweeps
  // of a call in one launch.  Chosen while a CTA's tile stays within cluster_max_cells_per_cta (beyond that the fused tile
  // kernels, which use all SMs, are faster: measured, cluster.cuh).  MPMC_NO_RESIDENT turns it off.
  c->cluster_kernel = nullptr; c->cl_ctas = 0; c->cl_threads = 0; c->cl_smem = 0;
  p.cl_cx = p.cl_cy = p.cl_cap = p.cl_stride = 0;
  if (!(flags & MPMC_NO_RESIDENT)) {
    const bool cfast = c->nf == 2 && !disc;
    const void* ck = fp32 ? pick_cluster_kernel_f32(debug, disc, cfast, n_s) : pick_cluster_kernel_f64(debug, disc, cfast, n_s);
    const uint32_t threads = fp32 ? ClThreads<float>::value : ClThreads<double>::value;
    const size_t cell_bytes = fp32 ? cluster_cell_bytes<float>() : cluster_cell_bytes<double>();
    const uint32_t cap_max = fp32 ? cluster_max_cells_per_cta<float>(cfast) : cluster_max_cells_per_cta<double>(cfast);
    int smem_optin = 0, cluster_ok = 0;
    cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    cudaDeviceGetAttribute(&cluster_ok, cudaDevAttrClusterLaunch, dev);
    // the largest cluster (most SMs), then the squarest tiles, whose tiles fit; sizes above 8 are "non-portable" and
    // depend on the GPU's partitioning, so every candidate is checked with the occupancy query
    for (uint32_t nc = CL_MAX_CTAS; ck && cluster_ok && nc >= 1 && !c->cluster_kernel; nc >>= 1) {
      uint32_t best_cx = 0, best_cap = 0, best_stride = 0; double best_aspect = 0;
      for (uint32_t cx = 1; cx <= nc; ++cx) {
        if (nc % cx) continue;
        const uint32_t cy = nc / cx;
        if (cx > p.mx || cy > p.my) continue;
        const uint32_t tw = (p.mx + cx - 1) / cx, th = (p.my + cy - 1) / cy, cap = tw * th;
        if (cap > cap_max || cap * cell_bytes + 1024 > (size_t)smem_optin) continue;
        const double aspect = tw > th ? (double)tw / th : (double)th / tw;
        if (!best_cx || aspect < best_aspect) { best_cx = cx; best_cap = cap; best_stride = tw; best_aspect = aspect; }
      }
      if (!best_cx) continue;
      const size_t smem = (size_t)best_cap * cell_bytes;
      cudaFuncAttributes fa;                      // (a per-function attribute: set to the most any context can ask for)
      if (cudaFuncGetAttributes(&fa, ck) != cudaSuccess || (size_t)smem_optin < fa.sharedSizeBytes + smem ||
          cudaFuncSetAttribute(ck, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin - (int)fa.sharedSizeBytes) != cudaSuccess ||
          (nc > 8 && cudaFuncSetAttribute(ck, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess)) {
        cudaGetLastError(); continue;
      }
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3(nc); cfg.blockDim = dim3(threads); cfg.dynamicSmemBytes = smem;
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeClusterDimension;
      at[0].val.clusterDim.x = nc; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
      cfg.attrs = at; cfg.numAttrs = 1;
      int nclusters = 0;
      if (cudaOccupancyMaxActiveClusters(&nclusters, ck, &cfg) != cudaSuccess || nclusters < 1) { cudaGetLastError(); continue; }
      c->cluster_kernel = ck; c->cl_ctas = nc; c->cl_threads = threads; c->cl_smem = smem;
      p.cl_cx = best_cx; p.cl_cy = nc / best_cx; p.cl_cap = best_cap; p.cl_stride = best_stride;
    }
  }
  *out = c;
  return MPMC_OK;
}

int mpmc_create(mpmc_ctx** out, uint64_t N, const double box[2], double sigma, double d, uint32_t n_s,
                uint64_t seed, uint32_t flags, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  return mpmc_create_ex(out, N, box, sigma, d, n_s, seed, flags, 0.0, workspace, workspace_bytes, cuda_stream);
}

int mpmc_destroy(mpmc_ctx* c) {
  if (!c) return MPMC_OK;
  delete c;
  return MPMC_OK;
}

int mpmc_geometry(const mpmc_ctx* c, uint32_t m[2], double w[2], double L_eff[2]) {
  if (!c) return MPMC_ERR_ARG;
  if (m) { m[0] = c->p.mx; m[1] = c->p.my; }
  if (w) { w[0] = c->p.wx_d; w[1] = c->p.wy_d; }
  if (L_eff) { L_eff[0] = c->p.Lx_eff; L_eff[1] = c->p.Ly_eff; }
  return MPMC_OK;
}

int mpmc_load_positions(mpmc_ctx* c, const double* xy) {
  if (!c || !xy) return MPMC_ERR_ARG;
  c->loaded = false;
  c->sticky = MPMC_OK;
  c->t_host = 0; c->cur_host = 0;
  k_reset<<<c->sms * 4, 256, 0, c->stream>>>(c->p);
  const dim3 gN((c->p.N + AUX_THREADS - 1) / AUX_THREADS), gC = cell_grid(c, AUX_THREADS);
  if (c->fp32) {
    k_load_bin<float><<<gN, AUX_THREADS, 0, c->stream>>>(c->p, xy);
    k_load_sort<float><<<gC, AUX_THREADS, 0, c->stream>>>(c->p);
    k_load_check<float><<<gC, AUX_THREADS, 0, c->stream>>>(c->p);
  } else {
    k_load_bin<double><<<gN, AUX_THREADS, 0, c->stream>>>(c->p, xy);
    k_load_sort<double><<<gC, AUX_THREADS, 0, c->stream>>>(c->p);
    k_load_check<double><<<gC, AUX_THREADS, 0, c->stream>>>(c->p);
  }
  CU(cudaGetLastError());
  if (c->debug) CU(cudaMemsetAsync(c->p.mask, 0, (size_t)c->p.mx * c->p.my * 4, c->stream));
  Ctl h;
  const int st = read_ctl(c, &h);
  if (st != MPMC_OK) return st;
  c->loaded = true;
  return MPMC_OK;
}

int mpmc_sweep(mpmc_ctx* c, uint64_t k) {
  if (!c) return MPMC_ERR_ARG;
  if (!c->loaded) return MPMC_ERR_STATE;
  if (k == 0) return c->sticky;
  if (c->cluster_kernel) {
    // small systems: ONE launch of one cluster runs all k sweeps on the state resident in its shared memory (cluster.cuh);
    // the state returns to the buffer it came from, so the buffer parity does not change
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(c->cl_ctas); cfg.blockDim = dim3(c->cl_threads);
    cfg.dynamicSmemBytes = c->cl_smem; cfg.stream = c->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = c->cl_ctas; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    unsigned long long t_end = c->t_host + k;
    void* args[] = {(void*)&c->p, (void*)&t_end};
    CU(cudaLaunchKernelExC(&cfg, c->cluster_kernel, args));
    c->t_host += k;
    return c->sticky;
  }
  if (c->tile_kernel) {
    // one tile-kernel launch per sweep; each returns at once if the state has become crowded (tile.cuh) ...
    // Programmatic dependent launch: the CTAs of sweep t+1 become resident as the SMs of sweep t free up and park at
    // griddepcontrol.wait until sweep t has completed and flushed, which hides the launch latency (~4 us of ~50).
    bool pdl = c->stream != nullptr;
#ifdef MPMC_EXPERIMENT
    if (const char* e = std::getenv("MPMC_PDL")) pdl = pdl && e[0] != '0';      // A/B timing
#endif
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(c->tile_grid);
    cfg.blockDim = dim3(c->tile_threads);
    cfg.dynamicSmemBytes = c->tile_smem; cfg.stream = c->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    unsigned long long t = c->t_host;              // sweep index of each launch (kernel argument: uniform on the device)
    Draws dr;                                      // ... and its draws (read by the 2-slot kernel; the 4-slot kernel makes its own)
    uint32_t cur = c->cur_host;                    // ... and the buffer its state is in
    void* args[] = {(void*)&c->p, (void*)&t, (void*)&dr, (void*)&cur};
    for (uint64_t i = 0; i < k; ++i, ++t, cur ^= 1u) {
      dr = draw_sweep(c->p.seed_lo, c->p.seed_hi, c->p.flags, t);
      const cudaError_t e = cudaLaunchKernelExC(&cfg, c->tile_kernel, args);
      if (e != cudaSuccess) {                      // the device stays at the sweeps launched so far
        c->t_host += i; c->cur_host ^= (uint32_t)(i & 1u);
        return cuda_fail(e);
      }
    }
  }
  c->t_host += k; c->cur_host ^= (uint32_t)(k & 1u);
  // ... and the general kernel runs whatever is left up to the target sweep index: everything without a tile kernel,
  // normally nothing behind the 2-slot tile kernel (it hands over only a state with too many crowded cells), never
  // anything behind the 4-slot tile kernel, which takes every state
  if (c->tile_kernel && !c->tile_two_slot) return c->sticky;
  const int st = launch_sweeps(c, c->t_host, OP_SWEEPS, 0, 0.0);
  return st != MPMC_OK ? st : c->sticky;
}

int mpmc_get_positions(mpmc_ctx* c, double* xy_out) {
  if (!c || !xy_out) return MPMC_ERR_ARG;
  if (!c->loaded) return MPMC_ERR_STATE;
  const dim3 gC = cell_grid(c, AUX_THREADS);
  if (c->fp32) k_unpack<float><<<gC, AUX_THREADS, 0, c->stream>>>(c->p, xy_out);
  else         k_unpack<double><<<gC, AUX_THREADS, 0, c->stream>>>(c->p, xy_out);
  CU(cudaGetLastError());
  return c->sticky;
}

int mpmc_acceptance(mpmc_ctx* c, uint64_t out[4]) {
  if (!c || !out) return MPMC_ERR_ARG;
  if (!c->loaded) return MPMC_ERR_STATE;
  Ctl h;
  const int st = read_ctl(c, &h);
  out[1] = out[2] = out[3] = 0;
  for (uint32_t r = 0; r < CTR_SLOTS; ++r) { out[1] += h.counters[r][0]; out[2] += h.counters[r][1]; out[3] += h.counters[r][2]; }
  out[0] = out[1] + out[2] + out[3];
  return st;
}

int mpmc_pressure_contact(mpmc_ctx* c, double dr, uint32_t nbins, uint32_t degree, uint64_t* hist_out,
                          double* g_contact, double* p_star) {
  if (!c || !(dr > 0) || nbins == 0 || nbins > MAX_BINS) return MPMC_ERR_ARG;
  if ((g_contact || p_star) && degree + 1 > nbins) return MPMC_ERR_ARG;
  if (!c->loaded) return MPMC_ERR_STATE;
  CU(cudaMemsetAsync(c->p.hist, 0, (size_t)nbins * 8, c->stream));
  const int st = launch_histogram(c, dr, nbins, c->p.hist);
  if (st != MPMC_OK) return st;
  std::vector<uint64_t> H(nbins);
  CU(cudaMemcpyAsync(H.data(), c->p.hist, (size_t)nbins * 8, cudaMemcpyDeviceToHost, c->stream));
  CU(cudaStreamSynchronize(c->stream));
  if (hist_out) std::memcpy(hist_out, H.data(), (size_t)nbins * 8);
  if (g_contact || p_star) {
    const int fs = fit_contact(c, H.data(), 1, dr, nbins, degree, g_contact, p_star);
    if (fs != MPMC_OK) return fs;
  }
  return c->sticky;
}

int mpmc_contact_histogram_noalloc(mpmc_ctx* c, double dr, uint32_t nbins, uint64_t* hist_out) {
  if (!c || !hist_out || !(dr > 0) || nbins == 0) return MPMC_ERR_ARG;
  if (nbins > MPMC_NOALLOC_MAX_BINS) return MPMC_ERR_TOO_LARGE;
  if (!c->loaded) return MPMC_ERR_STATE;
  unsigned long long* scratch = nullptr;
  const int ss = noalloc_scratch(c, &scratch);
  if (ss != MPMC_OK) return ss;
  // the array keeps the last call's counts, and the kernels ADD: clear the bins this call uses
  CU(cudaMemsetAsync(scratch, 0, (size_t)nbins * 8, c->stream));
  const int st = launch_histogram(c, dr, nbins, scratch);
  if (st != MPMC_OK) return st;
  static_assert(sizeof(unsigned long long) == sizeof(uint64_t), "");
  CU(cudaMemcpyAsync(hist_out, scratch, (size_t)nbins * 8, cudaMemcpyDeviceToDevice, c->stream));
  return c->sticky;
}

int mpmc_pressure_accumulate(mpmc_ctx* c, double dr, uint32_t nbins) {
  if (!c || !(dr > 0) || nbins == 0 || nbins > MAX_BINS) return MPMC_ERR_ARG;
  if (!c->loaded) return MPMC_ERR_STATE;
  if (c->acc_samples == 0) {                     // the first sample after a reset fixes the bins
    CU(cudaMemsetAsync(c->hist_acc, 0, (size_t)MAX_BINS * 8, c->stream));
    c->acc_dr = dr; c->acc_nbins = nbins;
  } else if (dr != c->acc_dr || nbins != c->acc_nbins) {
    return MPMC_ERR_ARG;
  }
  const int st = launch_histogram(c, dr, nbins, c->hist_acc);      // the kernels ADD to their target
  if (st != MPMC_OK) return st;
  c->acc_samples += 1;
  return c->sticky;
}

int mpmc_pressure_accumulated(mpmc_ctx* c, uint32_t degree, uint64_t* hist_out, uint64_t* samples, double* g_contact,
                              double* p_star) {
  if (!c) return MPMC_ERR_ARG;
  if (!c->loaded) return MPMC_ERR_STATE;
  if (samples) *samples = c->acc_samples;
  if (c->acc_samples == 0) return (hist_out || g_contact || p_star) ? MPMC_ERR_STATE : c->sticky;
  if ((g_contact || p_star) && degree + 1 > c->acc_nbins) return MPMC_ERR_ARG;
  std::vector<uint64_t> H(c->acc_nbins);
  CU(cudaMemcpyAsync(H.data(), c->hist_acc, (size_t)c->acc_nbins * 8, cudaMemcpyDeviceToHost, c->stream));
  CU(cudaStreamSynchronize(c->stream));
  if (hist_out) std::memcpy(hist_out, H.data(), (size_t)c->acc_nbins * 8);
  if (g_contact || p_star) {
    const int fs = fit_contact(c, H.data(), c->acc_samples, c->acc_dr, c->acc_nbins, degree, g_contact, p_star);
    if (fs != MPMC_OK) return fs;
  }
  return c->sticky;
}

int mpmc_pressure_reset(mpmc_ctx* c) {
  if (!c) return MPMC_ERR_ARG;
  c->acc_samples = 0; c->acc_dr = 0.0; c->acc_nbins = 0;
  return MPMC_OK;
}

int mpmc_pressure_from_histogram(const mpmc_ctx* c, const uint64_t* hist, uint64_t samples, double dr, uint32_t nbins,
                                 uint32_t degree, double* g_contact, double* p_star) {
  if (!c || !hist || samples == 0 || !(dr > 0) || nbins == 0 || degree + 1 > nbins) return MPMC_ERR_ARG;
  return fit_contact(c, hist, samples, dr, nbins, degree, g_contact, p_star);
}

int mpmc_debug_sub_sweep(mpmc_ctx* c, uint32_t set) {
  if (!c || set > 3) return MPMC_ERR_ARG;
  if (!c->loaded) return MPMC_ERR_STATE;
  const int st = launch_sweeps(c, 0, OP_SUB_SWEEP, set, 0.0);
  return st != MPMC_OK ? st : c->sticky;
}

int mpmc_debug_shift(mpmc_ctx* c, uint32_t direction, double delta) {
  if (!c || direction > 3 || !(delta >= 0)) return MPMC_ERR_ARG;
  // Algorithm 1 draws delta from [0, w/2) (L90); the pull form takes entrants from ONE neighbour, so delta must stay below w
  if (!(delta < (direction < 2 ? c->p.wx_d : c->p.wy_d))) return MPMC_ERR_ARG;
  if (!c->loaded) return MPMC_ERR_STATE;
  const int st = launch_sweeps(c, 0, OP_SHIFT, direction, delta);
  if (st == MPMC_OK) c->cur_host ^= 1u;            // the shifted state is in the other buffer
  return st != MPMC_OK ? st : c->sticky;
}

int mpmc_debug_state(mpmc_ctx* c, void* counts, void* slab, void* ids, void* accept_mask, double origin[2],
                     uint64_t* sweep, uint64_t* digest) {
  if (!c) return MPMC_ERR_ARG;
  if (!c->loaded) return MPMC_ERR_STATE;
  if (accept_mask && !c->debug) return MPMC_ERR_ARG;
  const dim3 gC = cell_grid(c, AUX_THREADS);
  if (counts || slab || ids) {
    if (c->fp32) k_export<float><<<gC, AUX_THREADS, 0, c->stream>>>(c->p, (uint32_t*)counts, (float*)slab, (uint32_t*)ids);
    else         k_export<double><<<gC, AUX_THREADS, 0, c->stream>>>(c->p, (uint32_t*)counts, (double*)slab, (uint32_t*)ids);
    CU(cudaGetLastError());
  }
  if (accept_mask)
    CU(cudaMemcpyAsync(accept_mask, c->p.mask, (size_t)c->p.mx * c->p.my * 4, cudaMemcpyDeviceToDevice, c->stream));
  Ctl h;
  const int st = read_ctl(c, &h);
  if (origin) { origin[0] = h.origin[0]; origin[1] = h.origin[1]; }
  if (sweep) *sweep = h.t;
  if (digest) *digest = h.digest;
  return st;
}

int mpmc_debug_path(mpmc_ctx* c, uint64_t out[2]) {
  if (!c || !out) return MPMC_ERR_ARG;
  if (!c->loaded) return MPMC_ERR_STATE;
  Ctl h;
  const int st = read_ctl(c, &h);
  out[0] = h.path_sweeps[0]; out[1] = h.path_sweeps[1];
  return st;
}

int mpmc_debug_config(const mpmc_ctx* c, uint32_t out[12]) {
  if (!c || !out) return MPMC_ERR_ARG;
  out[0] = c->tile_kernel ? (c->tile_two_slot ? 2u : 4u) : 0u;
  out[1] = c->tile_kernel ? c->tile_grid : 0u;
  out[2] = c->p.tl_ntx; out[3] = c->p.tl_nty;
  out[4] = c->tile_kernel ? c->tile_threads : 0u;
  out[5] = (uint32_t)c->tile_smem;
  out[6] = c->grid; out[7] = (uint32_t)SUB_THREADS;
  out[8] = c->cluster_kernel ? c->cl_ctas : 0u; out[9] = c->p.cl_cx; out[10] = c->p.cl_cy; out[11] = (uint32_t)c->cl_smem;
  return MPMC_OK;
}

int mpmc_debug_phase_clocks(mpmc_ctx* c, uint64_t* out, uint32_t max_tiles, uint32_t* marks) {
  if (!c || !out || !marks) return MPMC_ERR_ARG;
  if (c->loaded && c->cluster_kernel) {               // the cluster-resident kernel: one row per CTA (cluster.cuh)
    const uint32_t ctas = c->cl_ctas < max_tiles ? c->cl_ctas : max_tiles;
    const int m = c->fp32 ? cluster_clocks_f32((unsigned long long*)out, ctas, c->stream) : cluster_clocks_f64((unsigned long long*)out, ctas, c->stream);
    if (m < 0) return MPMC_ERR_CUDA;
    *marks = (uint32_t)m;
    return MPMC_OK;
  }
  if (!c->loaded || !c->tile_kernel || !c->tile_two_slot) return MPMC_ERR_STATE;
  const uint32_t tiles = c->tile_grid < max_tiles ? c->tile_grid : max_tiles;
  static_assert(sizeof(unsigned long long) == sizeof(uint64_t), "");
  const int m = c->fp32 ? phase_clocks_f32((unsigned long long*)out, tiles, c->stream) : phase_clocks_f64((unsigned long long*)out, tiles, c->stream);
  if (m < 0) return MPMC_ERR_CUDA;
  *marks = (uint32_t)m;
  return MPMC_OK;
}

int mpmc_debug_tiling(uint32_t hx, uint32_t hy, size_t cell_bytes, size_t smem_max, uint32_t sms, uint32_t out[6]) {
  if (!out || hx == 0 || hy == 0 || cell_bytes == 0 || sms == 0) return MPMC_ERR_ARG;
  Tiling tl = {};
  if (!choose_tiling(hx, hy, cell_bytes, smem_max, sms, &tl)) return MPMC_ERR_BOX;
  out[0] = tl.ntx; out[1] = tl.nty; out[2] = tl.PS; out[3] = tl.na; out[4] = tl.hyA; out[5] = tl.tiles;
  return MPMC_OK;
}

int mpmc_debug_philox(const uint32_t* ctr, const uint32_t key[2], uint32_t* out, uint32_t n, void* cuda_stream) {
  if (!ctr || !key || !out) return MPMC_ERR_ARG;
  if (n == 0) return MPMC_OK;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  k_philox_test<<<(n + 127) / 128, 128, 0, s>>>(ctr, key[0], key[1], out, n);
  CU(cudaGetLastError());
  CU(cudaStreamSynchronize(s));
  return MPMC_OK;
}

const char* mpmc_strerror(int code) {
  switch (code) {
    case MPMC_OK: return "ok";
    case MPMC_ERR_ARG: return "bad argument";
    case MPMC_ERR_BOX: return "box too small for two cells of width >= sigma per axis (or too many cells)";
    case MPMC_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
    case MPMC_ERR_OVERLAP: return "loaded positions overlap or lie outside the box";
    case MPMC_ERR_CELL_OVERFLOW: return "more than n_max = 4 disks in one cell";
    case MPMC_ERR_CUDA: return "CUDA error (no device, or a launch failed)";
    case MPMC_ERR_STATE: return "no positions loaded";
    case MPMC_ERR_TOO_LARGE: return "size beyond the fixed capacity of the no-allocation entry point (mpmc_contact_histogram_noalloc: at most MPMC_NOALLOC_MAX_BINS = 1024 bins)";
    default: return "unknown error";
  }
}
const char* mpmc_version(void) { return "mpmc-b200 0.1 (sm_100a)"; }

}  // extern "C"
