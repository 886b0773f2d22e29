// mt_probe.cu — measured peaks of THIS device for the roofline that bounds the transport kernels (SURVEY.md §8(d):
// "measure the FFMA peak in the same process"; "measure [L2 bandwidth] with a random-sector gather over an L2-resident
// buffer (675 KB and 64 MB) and over a 1.4 GB buffer (HBM)").  Behind mt_measure_peaks() in include/muon_transport.h;
// bench.py prints the numbers under roofline.measured_peaks.  Nothing here is on the transport path.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/muon_probes.h"
#include "../../include/muon_transport.h"      // (the MT_ERR_* codes)
#include "mt_launch.h"

namespace {

constexpr int kChains = 8;            // independent dependency chains per thread (latency 4, so 8 hide it twice over)
constexpr int kUnroll = 32;           // instructions per chain per loop trip

// ---- issue-rate probes: `iters` trips of kChains x kUnroll instructions of one kind, operands in registers
enum { OP_FFMA = 0, OP_LOP3 = 1, OP_IMAD = 2, OP_IMAD_WIDE = 3, OP_MUFU = 4 };

template <int OP>
__global__ void __launch_bounds__(256) probe_issue_kernel(int iters, uint32_t seed, uint32_t* sink) {
  float f[kChains];
  uint32_t u[kChains];
  const float a = 1.0f + 1e-7f * (float)(seed & 7u), b = 1e-9f * (float)(threadIdx.x & 3);
  const uint32_t m = 0x9E3779B9u ^ seed, k = threadIdx.x | 1u;
#pragma unroll
  for (int c = 0; c < kChains; ++c) { f[c] = 1.0f + 0.001f * (float)(c + (threadIdx.x & 1)); u[c] = seed + 77u * c + threadIdx.x; }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int j = 0; j < kUnroll; ++j) {
#pragma unroll
      for (int c = 0; c < kChains; ++c) {
        if (OP == OP_FFMA) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[c]) : "f"(a), "f"(b));
        else if (OP == OP_LOP3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(u[c]) : "r"(m), "r"(k));
        else if (OP == OP_IMAD) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(u[c]) : "r"(m), "r"(k));
        else if (OP == OP_IMAD_WIDE) asm volatile("mul.hi.u32 %0, %0, %1;" : "+r"(u[c]) : "r"(m));   // Philox's wide product
        else asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(f[c]));        // MUFU: the conversion / special-function unit
      }
    }
  }
  uint32_t acc = 0;
#pragma unroll
  for (int c = 0; c < kChains; ++c) acc ^= u[c] ^ __float_as_uint(f[c]);
  if (acc == 0x12345678u) sink[0] = acc;          // never true in practice: keeps the chains alive
}

// ---- mixed streams: per group 8 fma.rn.f32 and NI instructions of another kind, all on independent chains.  They tell
// which pipes run beside the FP32 stream and which take its place: lop3 (ALU pipe) overlaps it, mad.lo and
// mul.wide (the FMA pipe's integer half) add their own 2 and 4 cycles per warp instruction.
enum { MIX_LOP3 = 0, MIX_IMAD = 1, MIX_MULWIDE = 2 };
template <int NI, int KIND>
__global__ void __launch_bounds__(256) probe_mix_kernel(int iters, uint32_t seed, uint32_t* sink) {
  float f[kChains];
  uint32_t u[kChains];
  uint64_t w[kChains];
  const float a = 1.0f + 1e-7f * (float)(seed & 7u), b = 1e-9f * (float)(threadIdx.x & 3);
  const uint32_t m = 0x9E3779B9u ^ seed, k = threadIdx.x | 1u;
#pragma unroll
  for (int c = 0; c < kChains; ++c) { f[c] = 1.0f + 0.001f * (float)(c + (threadIdx.x & 1)); u[c] = seed + 77u * c + threadIdx.x; w[c] = u[c]; }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int j = 0; j < 8; ++j) {
#pragma unroll
      for (int c = 0; c < kChains; ++c) {
        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[c]) : "f"(a), "f"(b));
        if (c < NI) {
          if (KIND == MIX_LOP3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(u[c]) : "r"(m), "r"(k));
          else if (KIND == MIX_IMAD) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(u[c]) : "r"(m), "r"(k));
          else asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(w[c]) : "r"((uint32_t)(w[c] >> 32)), "r"(m));
        }
      }
    }
  }
  uint32_t acc = 0;
#pragma unroll
  for (int c = 0; c < kChains; ++c) acc ^= u[c] ^ __float_as_uint(f[c]) ^ (uint32_t)w[c] ^ (uint32_t)(w[c] >> 32);
  if (acc == 0x12345678u) sink[0] = acc;
}

// ---- gather probe: every lane reads one 32-byte sector (the size of a field-grid record) at a
// pseudo-random position of a buffer of `n_sectors` sectors; four loads in flight per thread.  Positions come from a
// multiplicative hash of (thread, trip), so a warp's 32 sectors are unrelated: the worst case the step loop can meet.
__global__ void __launch_bounds__(256) probe_gather_kernel(const uint4* __restrict__ buf, uint32_t n_sectors, int iters,
                                                           uint32_t seed, uint32_t* sink) {
  uint32_t h = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + seed;
  float acc = 0.0f;
  for (int it = 0; it < iters; ++it) {
    float v[4][8];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      h = h * 1664525u + 1013904223u;
      const uint4* p = buf + 2 * (size_t)__umulhi(h, n_sectors);
      // the step loop's own load: one 256-bit read-only load per record (mt_step.cuh: ldg_pair)
      asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                   : "=f"(v[j][0]), "=f"(v[j][1]), "=f"(v[j][2]), "=f"(v[j][3]), "=f"(v[j][4]), "=f"(v[j][5]), "=f"(v[j][6]), "=f"(v[j][7])
                   : "l"(p));
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) acc += v[j][0] + v[j][3] + v[j][5] + v[j][6];
  }
  if (acc == 0.12345678f) sink[0] = 1u;
}

template <class F> cudaError_t time_best(F&& launch, int reps, float* best_ms) {
  cudaEvent_t e0, e1;
  cudaError_t e = cudaEventCreate(&e0);
  if (e != cudaSuccess) return e;
  e = cudaEventCreate(&e1);
  if (e != cudaSuccess) { cudaEventDestroy(e0); return e; }
  *best_ms = 1e30f;
  for (int r = 0; r < reps + 1 && e == cudaSuccess; ++r) {           // the first run warms up
    cudaEventRecord(e0, 0);
    launch();
    cudaEventRecord(e1, 0);
    e = cudaEventSynchronize(e1);
    float ms = 0.0f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    if (e == cudaSuccess && r > 0 && ms < *best_ms) *best_ms = ms;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  if (e == cudaSuccess) e = cudaGetLastError();
  return e;
}

template <int OP> cudaError_t issue_rate(int sm_count, uint32_t* sink, double* warp_instr_per_s_per_smsp, double* thread_ops_per_s) {
  const int grid = sm_count * 8, block = 256, iters = 400;           // 8 warps per scheduler
  float ms = 0.0f;
  cudaError_t e = time_best([&] { probe_issue_kernel<OP><<<grid, block>>>(iters, 12345u, sink); }, 3, &ms);
  if (e != cudaSuccess) return e;
  const double per_thread = (double)iters * kUnroll * kChains;
  const double warps = (double)grid * block / 32.0;
  *thread_ops_per_s = per_thread * grid * block / (ms * 1e-3);
  *warp_instr_per_s_per_smsp = per_thread * warps / (ms * 1e-3) / (sm_count * 4.0);
  return cudaSuccess;
}

template <int NI, int KIND> cudaError_t mix_rate(int sm_count, uint32_t* sink, double* thread_ops_per_s) {
  const int grid = sm_count * 8, block = 256, iters = 1000;
  float ms = 0.0f;
  cudaError_t e = time_best([&] { probe_mix_kernel<NI, KIND><<<grid, block>>>(iters, 12345u, sink); }, 3, &ms);
  if (e != cudaSuccess) return e;
  *thread_ops_per_s = (double)iters * 8 * (kChains + NI) * grid * block / (ms * 1e-3);
  return cudaSuccess;
}

}  // namespace

extern "C" int mt_measure_peaks(int cuda_device, mt_peaks* out) {
  if (!out) return MT_ERR_INVALID_ARG;
  int n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || cuda_device < 0 || cuda_device >= n_dev) { cudaGetLastError(); return MT_ERR_CUDA; }
  int prev = 0;
  cudaGetDevice(&prev);
  cudaSetDevice(cuda_device);
  cudaDeviceProp prop;
  int rc = MT_OK;
  uint32_t* sink = nullptr;
  uint4* buf = nullptr;
  do {
    if (cudaGetDeviceProperties(&prop, cuda_device) != cudaSuccess) { rc = MT_ERR_CUDA; break; }
    if (cudaMalloc(&sink, 256) != cudaSuccess) { rc = MT_ERR_NOMEM; break; }
    const int sms = prop.multiProcessorCount;
    int clock_khz = 0;
    cudaDeviceGetAttribute(&clock_khz, cudaDevAttrClockRate, cuda_device);
    out->sm_count = sms;
    out->sm_clock_mhz_nominal = clock_khz * 1e-3;
    double per_smsp = 0.0;
    if (issue_rate<OP_FFMA>(sms, sink, &per_smsp, &out->ffma_thread_ops_per_s) != cudaSuccess) { rc = MT_ERR_CUDA; break; }
    out->ffma_warp_instr_per_s_per_smsp = per_smsp;
    if (issue_rate<OP_LOP3>(sms, sink, &per_smsp, &out->lop3_thread_ops_per_s) != cudaSuccess) { rc = MT_ERR_CUDA; break; }
    if (issue_rate<OP_IMAD>(sms, sink, &per_smsp, &out->imad_thread_ops_per_s) != cudaSuccess) { rc = MT_ERR_CUDA; break; }
    if (issue_rate<OP_IMAD_WIDE>(sms, sink, &per_smsp, &out->mulhi_thread_ops_per_s) != cudaSuccess) { rc = MT_ERR_CUDA; break; }
    if (issue_rate<OP_MUFU>(sms, sink, &per_smsp, &out->mufu_thread_ops_per_s) != cudaSuccess) { rc = MT_ERR_CUDA; break; }
    if (mix_rate<4, MIX_LOP3>(sms, sink, &out->mix_ffma8_lop3_4_thread_ops_per_s) != cudaSuccess) { rc = MT_ERR_CUDA; break; }
    if (mix_rate<4, MIX_IMAD>(sms, sink, &out->mix_ffma8_imad4_thread_ops_per_s) != cudaSuccess) { rc = MT_ERR_CUDA; break; }
    if (mix_rate<2, MIX_MULWIDE>(sms, sink, &out->mix_ffma8_mulwide2_thread_ops_per_s) != cudaSuccess) { rc = MT_ERR_CUDA; break; }
    // gathers: one buffer of the largest size, the smaller working sets are prefixes of it
    const size_t sizes[4] = {(size_t)64 << 10, (size_t)675 << 10, (size_t)64 << 20, (size_t)1400 << 20};
    if (cudaMalloc(&buf, sizes[3]) != cudaSuccess) { cudaGetLastError(); rc = MT_ERR_NOMEM; break; }
    if (cudaMemset(buf, 1, sizes[3]) != cudaSuccess) { rc = MT_ERR_CUDA; break; }
    double* dst[4] = {&out->gather_l1_bytes_per_s, &out->gather_675k_bytes_per_s, &out->gather_64m_bytes_per_s,
                      &out->gather_1400m_bytes_per_s};
    for (int i = 0; i < 4 && rc == MT_OK; ++i) {
      const uint32_t n_sectors = (uint32_t)(sizes[i] / 32);
      const int grid = sms * 8, block = 256, iters = (i == 3) ? 64 : 256;
      float ms = 0.0f;
      if (time_best([&] { probe_gather_kernel<<<grid, block>>>(buf, n_sectors, iters, 99u + i, sink); }, 3, &ms) != cudaSuccess) {
        rc = MT_ERR_CUDA; break;
      }
      *dst[i] = (double)grid * block * iters * 4.0 * 32.0 / (ms * 1e-3);
    }
  } while (0);
  if (buf) cudaFree(buf);
  if (sink) cudaFree(sink);
  cudaSetDevice(prev);
  return rc;
}
