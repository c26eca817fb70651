// k_cluster.cu — instantiations of the cluster-resident small-system kernel k_cluster_sweeps (cluster.cuh) for one precision:
// compile with -DMPMC_P=float -DMPMC_SUFFIX=f32 or -DMPMC_P=double -DMPMC_SUFFIX=f64 (see ../build.py).
#include "kernels.h"
#include "cluster.cuh"

#define MPMC_CAT2(a, b) a##b
#define MPMC_CAT(a, b) MPMC_CAT2(a, b)

namespace mpmc {
namespace {
template <bool DEBUG>
const void* pick(bool disc, bool fast) {
  if (disc) return (const void*)k_cluster_sweeps<MPMC_P, 4, DEBUG, true, false>;
  return fast ? (const void*)k_cluster_sweeps<MPMC_P, 4, DEBUG, false, true> : (const void*)k_cluster_sweeps<MPMC_P, 4, DEBUG, false, false>;
}
}  // namespace
const void* MPMC_CAT(pick_cluster_kernel_, MPMC_SUFFIX)(bool debug, bool disc, bool fast, uint32_t n_s) {
  if (n_s != 4) return nullptr;
  return debug ? pick<true>(disc, fast) : pick<false>(disc, fast);
}

// -DMPMC_PHASE_CLOCKS: the cycle sums k_cluster_sweeps took in its last launch, copied to the host (ctas x marks values)
int MPMC_CAT(cluster_clocks_, MPMC_SUFFIX)(unsigned long long* out, uint32_t ctas, void* stream) {
#ifdef MPMC_PHASE_CLOCKS
  if (ctas > CL_MAX_CTAS) ctas = CL_MAX_CTAS;
  if (cudaMemcpyFromSymbolAsync(out, g_cluster_clocks, (size_t)ctas * CL_CLOCK_MARKS * 8, 0, cudaMemcpyDeviceToHost, (cudaStream_t)stream) != cudaSuccess) return -1;
  if (cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess) return -1;
  return (int)CL_CLOCK_MARKS;
#else
  (void)out; (void)ctas; (void)stream;
  return 0;
#endif
}
}  // namespace mpmc
