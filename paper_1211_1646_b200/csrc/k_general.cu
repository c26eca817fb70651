// k_general.cu — instantiations of the general persistent kernel k_sweeps (sweep.cuh) for one precision:
// compile with -DMPMC_P=float -DMPMC_SUFFIX=f32 or -DMPMC_P=double -DMPMC_SUFFIX=f64 (see ../build.py).
#include "kernels.h"
#include "sweep.cuh"

#define MPMC_CAT2(a, b) a##b
#define MPMC_CAT(a, b) MPMC_CAT2(a, b)

namespace mpmc {
namespace {
template <typename P, bool DEBUG>
const void* pick(bool fast, bool disc, uint32_t n_s) {
  if (disc) {           // the paper's disc-shaped proposal: general cell update only
    if (n_s == 4) return (const void*)k_sweeps<P, 4, DEBUG, false, true>;
    return (const void*)k_sweeps<P, 0, DEBUG, false, true>;
  }
  if (fast && n_s == 4) return (const void*)k_sweeps<P, 4, DEBUG, true>;
  if (fast && n_s == 8) return (const void*)k_sweeps<P, 8, DEBUG, true>;
  if (n_s == 4) return (const void*)k_sweeps<P, 4, DEBUG, false>;
  if (n_s == 8) return (const void*)k_sweeps<P, 8, DEBUG, false>;
  return (const void*)k_sweeps<P, 0, DEBUG, false>;
}
}  // namespace
const void* MPMC_CAT(pick_kernel_, MPMC_SUFFIX)(bool debug, bool fast, bool disc, uint32_t n_s) {
  return debug ? pick<MPMC_P, true>(fast, disc, n_s) : pick<MPMC_P, false>(fast, disc, n_s);
}
}  // namespace mpmc
