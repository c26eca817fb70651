// k_tile2.cu — instantiations of the fused 2-slot tile kernel k_tile_sweep (tile.cuh) for one precision:
// compile with -DMPMC_P=float -DMPMC_SUFFIX=f32 or -DMPMC_P=double -DMPMC_SUFFIX=f64 (see ../build.py).
#include "kernels.h"
#include "tile.cuh"

#define MPMC_CAT2(a, b) a##b
#define MPMC_CAT(a, b) MPMC_CAT2(a, b)

namespace mpmc {
namespace {
template <typename P, bool DEBUG>
const void* pick(uint32_t n_s, bool compact) {
  // dilute systems (most cells empty): the variant that runs the cell update on compacted warps of non-empty cells
  if (compact && n_s == 4) return (const void*)k_tile_sweep<P, 4, DEBUG, true>;
  if (compact && n_s == 8) return (const void*)k_tile_sweep<P, 8, DEBUG, true>;
  if (n_s == 4) return (const void*)k_tile_sweep<P, 4, DEBUG>;
  if (n_s == 8) return (const void*)k_tile_sweep<P, 8, DEBUG>;
  return nullptr;
}
}  // namespace
const void* MPMC_CAT(pick_tile_kernel_, MPMC_SUFFIX)(bool debug, uint32_t n_s, bool compact) {
  return debug ? pick<MPMC_P, true>(n_s, compact) : pick<MPMC_P, false>(n_s, compact);
}
}  // namespace mpmc
