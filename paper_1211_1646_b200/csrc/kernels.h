// kernels.h — the per-sweep kernels are compiled in translation units of their own (one per kernel family and
// precision, so the library builds in parallel); the host code in mpmc.cu picks an instantiation through these.
#pragma once
#include <stdint.h>

namespace mpmc {

// k_sweeps<P, NS, DEBUG, FAST, DISC> (sweep.cuh): fast = the w ~ sigma cell update (occupancy 0/1/2, compile-time
// n_s in {4, 8}); otherwise the general one
const void* pick_kernel_f32(bool debug, bool fast, bool disc, uint32_t n_s);
const void* pick_kernel_f64(bool debug, bool fast, bool disc, uint32_t n_s);
// k_tile_sweep<P, NS, DEBUG, COMPACT> (tile.cuh); nullptr if there is no instantiation for n_s
const void* pick_tile_kernel_f32(bool debug, uint32_t n_s, bool compact);
const void* pick_tile_kernel_f64(bool debug, uint32_t n_s, bool compact);
// builds with -DMPMC_PHASE_CLOCKS: the clock marks k_tile_sweep took at its phase boundaries in its last launch, copied to
// the host (tiles x marks values); returns the number of marks per tile, 0 in an ordinary build, -1 on a CUDA error
int phase_clocks_f32(unsigned long long* out, uint32_t tiles, void* stream);
int phase_clocks_f64(unsigned long long* out, uint32_t tiles, void* stream);
// k_tile4_sweep<P, 4, DEBUG, DISC, WIDE> (tile4.cuh); wide = the 512-thread instantiation (fp32 only); nullptr unless n_s = 4
const void* pick_tile4_kernel_f32(bool debug, bool disc, bool wide, uint32_t n_s);
const void* pick_tile4_kernel_f64(bool debug, bool disc, bool wide, uint32_t n_s);

// k_cluster_sweeps<P, 4, DEBUG, DISC, FAST> (cluster.cuh): the whole state resident in one cluster's shared memory; fast = the
// w ~ sigma cell update (square proposal only); nullptr unless n_s = 4
const void* pick_cluster_kernel_f32(bool debug, bool disc, bool fast, uint32_t n_s);
const void* pick_cluster_kernel_f64(bool debug, bool disc, bool fast, uint32_t n_s);
// builds with -DMPMC_PHASE_CLOCKS: cycle sums of the last k_cluster_sweeps launch (ctas x marks); marks per CTA, 0, or -1
int cluster_clocks_f32(unsigned long long* out, uint32_t ctas, void* stream);
int cluster_clocks_f64(unsigned long long* out, uint32_t ctas, void* stream);

}  // namespace mpmc
