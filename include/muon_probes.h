/* muon_probes.h — C ABI of libmuon_probes.so: the measurement probes that bench.py's roofline is reported against.
 *
 * NOT part of the transport library.  SURVEY.md §8(d) asks for peaks measured in the benchmark's own process ("measure the
 * FFMA peak in the same process ... L2 bandwidth with a random-sector gather") and north_star subsystem (5) for a
 * comparison of the ways a field corner can be fetched; both are experiments about the device, not steps of Algorithm 1,
 * so they live in a library of their own that only bench.py and tests/test_gpu_probes.py load.  libmuon_transport.so
 * (include/muon_transport.h) exports neither.  Both calls return 0 or one of muon_transport.h's negative MT_ERR_* codes
 * (MT_ERR_INVALID_ARG -1, MT_ERR_CUDA -5, MT_ERR_NOMEM -6), allocate their own temporary device memory, free it, and
 * synchronise the device.
 */
#ifndef MUON_PROBES_H_
#define MUON_PROBES_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Measured peaks of device `cuda_device`, for the roofline the transport kernels are reported against (SURVEY.md §8(d):
 * "measure the FFMA peak in the same process ... L2 bandwidth with a random-sector gather").  Runs a few short probe
 * kernels (about 50 ms in all, 1.4 GB of temporary device memory) and synchronises.  Not on the transport path.
 *   *_thread_ops_per_s   lanes x warp instructions per second over the whole GPU for an instruction stream of that one
 *                        kind with no dependency stalls (8 warps per scheduler, 8 independent chains per thread):
 *                        fma.rn.f32 / lop3.b32 / mad.lo.u32 / mul.hi.u32 / rsqrt.approx.f32 (the conversion unit)
 *   gather_*_bytes_per_s 32-byte sectors per second x 32 for one random sector per lane out of a working set of
 *                        64 KB (L1-resident), 675 KB and 64 MB (L2-resident), 1400 MB (HBM)
 *   mix_*                the same count for mixed streams, 8 fma.rn.f32 to 4 lop3.b32 / 4 mad.lo.u32 / 2 mul.wide.u32 per
 *                        group: a pipe that runs beside the FP32 stream leaves the total near the fma rate, one that takes
 *                        its place pulls it down by its own cycles                                                      */
typedef struct {
  int32_t sm_count;
  double sm_clock_mhz_nominal;
  double ffma_thread_ops_per_s, ffma_warp_instr_per_s_per_smsp;
  double lop3_thread_ops_per_s, imad_thread_ops_per_s, mulhi_thread_ops_per_s, mufu_thread_ops_per_s;
  double gather_l1_bytes_per_s, gather_675k_bytes_per_s, gather_64m_bytes_per_s, gather_1400m_bytes_per_s;
  double mix_ffma8_lop3_4_thread_ops_per_s, mix_ffma8_imad4_thread_ops_per_s, mix_ffma8_mulwide2_thread_ops_per_s;
} mt_peaks;
int mt_measure_peaks(int cuda_device, mt_peaks* out);

/* The three ways of serving the trilinear field corners that north_star subsystem (5) names, timed on one synthetic
 * access pattern (csrc/mt_probe_field.cu): read-only 256-bit global loads (what the transport kernels use), point-sampled
 * 3D texture fetches, and a shared-memory window staged by TMA (cp.async.bulk.tensor).  Rates are 32-byte corner records
 * per second over the whole GPU; tma_records_per_s = 0 if the driver offers no cuTensorMapEncodeTiled.  ~100 MB of
 * temporary device memory; synchronises.  Not on the transport path. */
typedef struct {
  double records_per_launch;
  double ldg_records_per_s, tex_records_per_s, tma_records_per_s;
} mt_field_paths;
int mt_probe_field_paths(int cuda_device, mt_field_paths* out);

#ifdef __cplusplus
}
#endif
#endif /* MUON_PROBES_H_ */
