// mt_inst_voxel_b.cu — transport-kernel instantiations for voxel grids (MT_GEOM_VOXEL), field at every Runge-Kutta stage: trilinear or nearest-neighbour.
#include "mt_kernels.cuh"

mt_kernel_fn mt_pick_voxel_b(const MtLaunchCfg& cfg) {
  return (cfg.field & 1) ? pick_tables<1, 3>(cfg) : pick_tables<1, 2>(cfg);
}
