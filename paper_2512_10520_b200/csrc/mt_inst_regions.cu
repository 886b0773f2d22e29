// mt_inst_regions.cu — transport-kernel instantiations for box regions (MT_GEOM_REGIONS): every table kind and schedule, field frozen or per stage.
#include "mt_kernels.cuh"

mt_kernel_fn mt_pick_regions(const MtLaunchCfg& cfg) {
  if (cfg.lean) return (cfg.field & 2) ? pick_tables_lean<0, 2>(cfg) : pick_tables_lean<0, 0>(cfg);
  return (cfg.field & 2) ? pick_tables<0, 2>(cfg) : pick_tables<0, 0>(cfg);
}
