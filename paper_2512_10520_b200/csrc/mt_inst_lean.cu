// mt_inst_lean.cu — transport-kernel instantiations for the LEAN variants: WAVEFRONT schedule on a voxel grid, tables gathered from L2 (and, for the default mode, staged in shared memory).
#include "mt_kernels.cuh"

mt_kernel_fn mt_pick_lean(const MtLaunchCfg& cfg) {
  if (cfg.tab_smem) return wave_transport_kernel<1, 32, true, false, 0, true>;   // 4-byte cells, trilinear frozen only
  switch ((cfg.field & 3) | (cfg.joint ? 8 : (cfg.pack == 32 ? 0 : 4))) {
    case 0: return wave_transport_kernel<1, 32, false, false, 0, true>;
    case 1: return wave_transport_kernel<1, 32, false, false, 1, true>;
    case 2: return wave_transport_kernel<1, 32, false, false, 2, true>;
    case 3: return wave_transport_kernel<1, 32, false, false, 3, true>;
    case 4: return wave_transport_kernel<1, 64, false, false, 0, true>;
    case 5: return wave_transport_kernel<1, 64, false, false, 1, true>;
    case 6: return wave_transport_kernel<1, 64, false, false, 2, true>;
    case 7: return wave_transport_kernel<1, 64, false, false, 3, true>;
    case 8: return wave_transport_kernel<1, 64, false, true, 0, true>;
    case 9: return wave_transport_kernel<1, 64, false, true, 1, true>;
    case 10: return wave_transport_kernel<1, 64, false, true, 2, true>;
    default: return wave_transport_kernel<1, 64, false, true, 3, true>;
  }
}
