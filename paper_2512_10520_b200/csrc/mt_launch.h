// mt_launch.h — launcher interface between mt_lib.cu (host logic) and mt_kernels.cu (kernels).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "mt_params.h"

#ifndef MT_MAX_THREADS
#define MT_MAX_THREADS 768      // largest block the transport kernels are compiled for: one CTA of 768 threads
#endif                          // or three of 256 per SM -> at most 85 registers per thread
#ifndef MT_MIN_BLOCKS
#define MT_MIN_BLOCKS 1
#endif

struct MtLaunchCfg {
  unsigned grid, block;
  size_t smem_bytes;
  int pack;        // 32 or 64 (bits per packed alias cell)
  bool tab_smem;   // the hot prefix of the tables (P.hot_cells > 0) is staged in shared memory
  int sched;       // MT_SCHED_STATIC / _REFILL / _WAVEFRONT
  bool joint;      // MT_HIST_JOINT tables (pack64, never staged)
  int field;       // MT_FIELD_* of the geometry
  bool lean;       // P.lean == MT_LEAN_ALL and a LEAN kernel exists for this combination (mt_has_lean)
};
// LEAN variants exist for: voxel grids under WAVEFRONT (every field mode, marginal or joint tables from L2; marginal
// 4-byte cells staged in shared memory with the trilinear frozen field); regions and polyhedra under REFILL and WAVEFRONT
// (tables from L2, or 4-byte cells staged in shared memory)
bool mt_has_lean(int mode, const MtLaunchCfg& cfg);

// the transport kernel for a launch configuration; each picker lives in the translation unit that instantiates its kernels
typedef void (*mt_kernel_fn)(const MtParams);
mt_kernel_fn mt_pick_regions(const MtLaunchCfg& cfg);
mt_kernel_fn mt_pick_poly(const MtLaunchCfg& cfg);
mt_kernel_fn mt_pick_voxel_a(const MtLaunchCfg& cfg);   // field frozen over the step
mt_kernel_fn mt_pick_voxel_b(const MtLaunchCfg& cfg);   // field at every Runge-Kutta stage
mt_kernel_fn mt_pick_lean(const MtLaunchCfg& cfg);      // only where mt_has_lean() holds

cudaError_t mt_launch_transport(const MtParams& P, const MtLaunchCfg& cfg, cudaStream_t stream);
cudaError_t mt_occupancy(const MtParams& P, const MtLaunchCfg& cfg, int* blocks_per_sm);
// WAVEFRONT helpers: key + rank of the input muons; scan of the key histogram followed by the permutation that
// puts the parked records (P.sort_key) in sorted order (P.perm)
cudaError_t mt_launch_wave_bin(const MtParams& P, unsigned grid, cudaStream_t stream);
cudaError_t mt_launch_wave_sort(const MtParams& P, int n_keys, unsigned grid, cudaStream_t stream);
// item-mode passes: spread tallies [MT_COUNTER_SLOTS][8] -> the caller's counters [8] (and cleared)
cudaError_t mt_launch_reduce_counters(unsigned long long* spread, unsigned long long* counters, cudaStream_t stream);
// d_material_cells: [256] counters (zeroed by the caller) of grid cells per material id
cudaError_t mt_launch_repack(const uint8_t* mat, const float* fld, MtCellPair* out, int nx, int ny, int nz,
                             unsigned long long* d_material_cells, cudaStream_t stream);
cudaError_t mt_launch_debug_sample(int pack, bool joint, const void* tab, uint32_t N, const uint32_t* words,
                                   uint64_t n, uint32_t* out, cudaStream_t stream);
cudaError_t mt_launch_debug_lookup(const MtParams& P, size_t smem_bytes, const float* xyz, uint64_t n, int32_t* mat_out,
                                   float* b_out, cudaStream_t stream);
cudaError_t mt_launch_debug_philox(uint32_t k0, uint32_t k1, uint64_t id_base, uint32_t step, uint64_t n,
                                   uint32_t* out, cudaStream_t stream);
