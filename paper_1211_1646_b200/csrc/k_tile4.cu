// k_tile4.cu — instantiations of the fused 4-slot tile kernel k_tile4_sweep (tile4.cuh) for one precision:
// compile with -DMPMC_P=float -DMPMC_SUFFIX=f32 or -DMPMC_P=double -DMPMC_SUFFIX=f64 (see ../build.py).
#include "kernels.h"
#include "tile4.cuh"

#define MPMC_CAT2(a, b) a##b
#define MPMC_CAT(a, b) MPMC_CAT2(a, b)

namespace mpmc {
namespace {
template <bool DEBUG, bool WIDE>
const void* pick(bool disc) {
  return disc ? (const void*)k_tile4_sweep<MPMC_P, 4, DEBUG, true, WIDE> : (const void*)k_tile4_sweep<MPMC_P, 4, DEBUG, false, WIDE>;
}
}  // namespace
const void* MPMC_CAT(pick_tile4_kernel_, MPMC_SUFFIX)(bool debug, bool disc, bool wide, uint32_t n_s) {
  if (n_s != 4) return nullptr;
  if constexpr (sizeof(MPMC_P) == 4) {         // (fp64 has one thread count: no second instantiation)
    if (wide) return debug ? pick<true, true>(disc) : pick<false, true>(disc);
  }
  return debug ? pick<true, false>(disc) : pick<false, false>(disc);
}
}  // namespace mpmc
