// mt_inst_poly.cu — transport-kernel instantiations for convex polyhedra (MT_GEOM_POLY): every table kind and schedule, field frozen or per stage.
#include "mt_kernels.cuh"

mt_kernel_fn mt_pick_poly(const MtLaunchCfg& cfg) {
  if (cfg.lean) return (cfg.field & 2) ? pick_tables_lean<2, 2>(cfg) : pick_tables_lean<2, 0>(cfg);
  return (cfg.field & 2) ? pick_tables<2, 2>(cfg) : pick_tables<2, 0>(cfg);
}
