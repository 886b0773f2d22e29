// mt_inst_voxel_a.cu — transport-kernel instantiations for voxel grids (MT_GEOM_VOXEL), field frozen over the step: trilinear or nearest-neighbour.
#include "mt_kernels.cuh"

mt_kernel_fn mt_pick_voxel_a(const MtLaunchCfg& cfg) {
  return (cfg.field & 1) ? pick_tables<1, 1>(cfg) : pick_tables<1, 0>(cfg);
}
