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

// -DMPMC_PHASE_CLOCKS: copy the phase marks of the last launch to the host (tiles x PHASE_MARKS values)
int MPMC_CAT(phase_clocks_, MPMC_SUFFIX)(unsigned long long* out, uint32_t tiles, void* stream) {
#ifdef MPMC_PHASE_CLOCKS
  if (tiles > PHASE_TILES) tiles = PHASE_TILES;
  if (cudaMemcpyFromSymbolAsync(out, g_phase_clocks, (size_t)tiles * PHASE_MARKS * 8, 0, cudaMemcpyDeviceToHost, (cudaStream_t)stream) != cudaSuccess) return -1;
  if (cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess) return -1;
  return (int)PHASE_MARKS;
#else
  (void)out; (void)tiles; (void)stream;
  return 0;
#endif
}
}  // namespace mpmc
