// mt_kernels.cu — the transport kernels and their launchers (sm_100a).
//
// One kernel template runs Algorithm 1 under three schedules:
//   STATIC     one lane per muon for its whole life (the paper's own mapping, L59, L174);
//   REFILL     persistent warps; lanes whose muon has terminated take new muons from a global counter;
//   WAVEFRONT  like REFILL, but over a compacted list of live muons and only until each muon leaves the
//              current z-slab; the caller launches one pass per slab, so every resident muon reads the same
//              few z-layers of the field grid (L2/L1-resident) instead of the whole 1.9 GB grid.
// The per-step arithmetic is mt_step.cuh; results do not depend on the schedule.
#include <cuda_runtime.h>
#include <stdint.h>
#include "mt_launch.h"
#include "mt_step.cuh"

namespace {

using namespace mt;

enum { SCHED_STATIC = 1, SCHED_REFILL = 2, SCHED_WAVEFRONT = 3 };
constexpr int kInnerSteps = 8;        // steps between two refill checks
constexpr unsigned kFull = 0xFFFFFFFFu;

extern __shared__ __align__(16) unsigned char mt_smem[];

template <int PACK, bool TAB_SMEM>
MT_DEV View<PACK> stage_view(const MtParams& P) {
  // const blob (edges, step lengths, regions) -> shared memory; tables too when they fit
  float* sblob = reinterpret_cast<float*>(mt_smem);
  for (int i = threadIdx.x; i < P.bl.n_words; i += blockDim.x) sblob[i] = __ldg(P.blob + i);
  View<PACK> V;
  V.edges = sblob;
  V.steps = sblob + P.bl.off_steps;
  V.zlo = sblob + P.bl.off_zlo;
  V.regions = reinterpret_cast<const MtRegionDev*>(sblob + P.bl.off_regions);
  const uint32_t* gtab = (PACK == 32) ? P.tab32 : reinterpret_cast<const uint32_t*>(P.tab64);
  if (TAB_SMEM) {
    uint32_t* stab = reinterpret_cast<uint32_t*>(sblob + ((P.bl.n_words + 3) & ~3));
    for (int i = threadIdx.x; i < P.table_words; i += blockDim.x) stab[i] = __ldg(gtab + i);
    V.tab = reinterpret_cast<const typename Tab<PACK>::cell_t*>(stab);
  } else {
    V.tab = reinterpret_cast<const typename Tab<PACK>::cell_t*>(gtab);
  }
  __syncthreads();
  return V;
}

template <int GEOM, int PACK, bool TAB_SMEM, int SCHED>
__global__ void __launch_bounds__(MT_MAX_THREADS, MT_MIN_BLOCKS)
transport_kernel(const __grid_constant__ MtParams P) {
  const View<PACK> V = stage_view<PACK, TAB_SMEM>(P);
  const unsigned lane = threadIdx.x & 31u;
  const unsigned lt_mask = (1u << lane) - 1u;

  // number of work items: muons (STATIC/REFILL) or live-list entries (WAVEFRONT)
  uint64_t n_items = P.n;
  if (SCHED == SCHED_WAVEFRONT && P.live_in_count) n_items = *P.live_in_count;

  Muon m;
  m.x = m.y = m.z = m.q = m.px = m.py = m.pz = 0.0f;
  m.step = 0;
  uint32_t idx = 0;              // muon index within this call
  bool active = false;
  bool exhausted = false;        // warp-uniform: the work counter has run past n_items
  unsigned long long acc_steps = 0;
  unsigned acc_f1 = 0, acc_f2 = 0, acc_f3 = 0, acc_f4 = 0;     // muons terminated per flag by this lane

  auto load = [&](uint64_t item) {
    if (SCHED == SCHED_WAVEFRONT) {
      idx = P.live_in ? P.live_in[item] : (uint32_t)item;
      if (P.first_pass) {
        const float4 a = __ldg(P.in_pos_q + idx), b = __ldg(P.in_mom + idx);
        m.x = a.x; m.y = a.y; m.z = a.z; m.q = a.w; m.px = b.x; m.py = b.y; m.pz = b.z; m.step = 0;
      } else {
        const float4 a = P.out_pos_flag[idx], b = P.out_mom_steps[idx];
        m.x = a.x; m.y = a.y; m.z = a.z; m.q = a.w; m.px = b.x; m.py = b.y; m.pz = b.z;
        m.step = __float_as_int(b.w);
      }
    } else {
      idx = (uint32_t)item;
      const float4 a = __ldg(P.in_pos_q + idx), b = __ldg(P.in_mom + idx);
      m.x = a.x; m.y = a.y; m.z = a.z; m.q = a.w; m.px = b.x; m.py = b.y; m.pz = b.z; m.step = 0;
    }
    active = true;
  };

  if (SCHED == SCHED_STATIC) {
    const uint64_t item = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (item < n_items) load(item);
    exhausted = true;
  }

  for (;;) {
    // ---- refill idle lanes from the global work counter (warp-aggregated: one atomic per warp)
    if (SCHED != SCHED_STATIC && !exhausted) {
      const unsigned idle = __ballot_sync(kFull, !active);
      const int n_idle = __popc(idle);
      if (n_idle >= P.refill_min_idle || idle == kFull) {
        unsigned long long base = 0;
        if (lane == 0) base = atomicAdd(P.work_counter, (unsigned long long)n_idle);
        base = __shfl_sync(kFull, base, 0);
        if (!active) {
          const uint64_t item = base + (unsigned)__popc(idle & lt_mask);
          if (item < n_items) load(item);
        }
        if (base + (unsigned)n_idle >= n_items) exhausted = true;
      }
    }
    if (!__any_sync(kFull, active)) {
      if (exhausted) break;
      continue;
    }

    // ---- a few steps for every active lane; the loop itself stays warp-uniform
#pragma unroll 1
    for (int k = 0; k < kInnerSteps; ++k) {
      int flag = 0;
      // WAVEFRONT: a live muon at or beyond the end of the slab waits for the next pass
      const bool parked = (SCHED == SCHED_WAVEFRONT) && active && m.z >= P.slab_z_end;
      if (active && !parked) {
        const uint64_t id = P.id_base + idx;
        flag = step_once<GEOM, PACK, !TAB_SMEM>(P, V, m, (uint32_t)id, (uint32_t)(id >> 32));
        if (flag == 0) acc_steps += 1;
      }
      // exit-plane records through one atomic per warp (north_star subsystem 6)
      if (P.exit_rec) {
        const bool ex = (flag == 2);
        const unsigned em = __ballot_sync(kFull, ex);
        if (em) {
          const int leader = __ffs(em) - 1;
          unsigned base = 0;
          if ((int)lane == leader) base = atomicAdd(P.exit_count, (unsigned)__popc(em));
          base = __shfl_sync(kFull, base, leader);
          if (ex) {
            const unsigned slot = base + (unsigned)__popc(em & lt_mask);
            if (slot < P.exit_capacity) {
              P.exit_rec[2 * (size_t)slot] = make_float4(m.x, m.y, m.z, __uint_as_float(idx));
              P.exit_rec[2 * (size_t)slot + 1] = make_float4(m.px, m.py, m.pz, __int_as_float(m.step));
            }
          }
        }
      }
      if (flag) {
        P.out_pos_flag[idx] = make_float4(m.x, m.y, m.z, __int_as_float(flag));
        P.out_mom_steps[idx] = make_float4(m.px, m.py, m.pz, __int_as_float(m.step));
        acc_f1 += (flag == 1); acc_f2 += (flag == 2); acc_f3 += (flag == 3); acc_f4 += (flag == 4);
        active = false;
      }
      if (SCHED == SCHED_WAVEFRONT) {
        const unsigned pm = __ballot_sync(kFull, parked);
        if (pm) {
          const int leader = __ffs(pm) - 1;
          unsigned base = 0;
          if ((int)lane == leader) base = atomicAdd(P.live_out_count, (unsigned)__popc(pm));
          base = __shfl_sync(kFull, base, leader);
          if (parked) {
            P.live_out[base + (unsigned)__popc(pm & lt_mask)] = idx;
            P.out_pos_flag[idx] = make_float4(m.x, m.y, m.z, m.q);
            P.out_mom_steps[idx] = make_float4(m.px, m.py, m.pz, __int_as_float(m.step));
            active = false;
          }
        }
      }
      if (!__any_sync(kFull, active)) break;
    }
    if (SCHED == SCHED_STATIC && !__any_sync(kFull, active)) break;
  }

  // ---- per-call counters: total steps and muons per flag
  if (P.counters) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc_steps += __shfl_xor_sync(kFull, acc_steps, o);
    acc_f1 = __reduce_add_sync(kFull, acc_f1); acc_f2 = __reduce_add_sync(kFull, acc_f2);
    acc_f3 = __reduce_add_sync(kFull, acc_f3); acc_f4 = __reduce_add_sync(kFull, acc_f4);
    if (lane == 0) {
      if (acc_steps) atomicAdd(P.counters + 0, acc_steps);
      if (acc_f1) atomicAdd(P.counters + 1, (unsigned long long)acc_f1);
      if (acc_f2) atomicAdd(P.counters + 2, (unsigned long long)acc_f2);
      if (acc_f3) atomicAdd(P.counters + 3, (unsigned long long)acc_f3);
      if (acc_f4) atomicAdd(P.counters + 4, (unsigned long long)acc_f4);
    }
  }
}

// ---- voxel repack: {material u8, field f32x3} -> one float4 per cell; also reports the largest material id
__global__ void repack_kernel(const uint8_t* __restrict__ mat, const float* __restrict__ fld, float4* __restrict__ out,
                              size_t n_cells, int* __restrict__ max_material) {
  int local_max = 0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_cells; i += (size_t)gridDim.x * blockDim.x) {
    const int mval = mat[i];
    out[i] = make_float4(fld[3 * i], fld[3 * i + 1], fld[3 * i + 2], __int_as_float(mval));
    local_max = max(local_max, mval);
  }
  for (int o = 16; o > 0; o >>= 1) local_max = max(local_max, __shfl_xor_sync(kFull, local_max, o));
  if ((threadIdx.x & 31) == 0 && local_max > 0) atomicMax(max_material, local_max);
}

template <int PACK>
__global__ void debug_sample_kernel(const typename Tab<PACK>::cell_t* tab, uint32_t N, const uint32_t* words,
                                    uint64_t n, uint32_t* out) {
  const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = Tab<PACK>::template draw<true>(tab, N, words[i]);
}

__global__ void debug_philox_kernel(uint32_t k0, uint32_t k1, uint64_t id_base, uint32_t step, uint64_t n,
                                    uint32_t* out) {
  const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint64_t id = id_base + i;
  uint32_t w[4];
  philox4x32_10((uint32_t)id, (uint32_t)(id >> 32), step, 0u, k0, k1, w);
  reinterpret_cast<uint4*>(out)[i] = make_uint4(w[0], w[1], w[2], w[3]);
}

typedef void (*kernel_fn)(const MtParams);

template <int GEOM, int PACK, bool TAB_SMEM>
kernel_fn pick_sched(int sched) {
  switch (sched) {
    case SCHED_STATIC: return transport_kernel<GEOM, PACK, TAB_SMEM, SCHED_STATIC>;
    case SCHED_REFILL: return transport_kernel<GEOM, PACK, TAB_SMEM, SCHED_REFILL>;
    default: return transport_kernel<GEOM, PACK, TAB_SMEM, SCHED_WAVEFRONT>;
  }
}
template <int GEOM>
kernel_fn pick_pack(int pack, bool tab_smem, int sched) {
  if (pack == 32) return tab_smem ? pick_sched<GEOM, 32, true>(sched) : pick_sched<GEOM, 32, false>(sched);
  return tab_smem ? pick_sched<GEOM, 64, true>(sched) : pick_sched<GEOM, 64, false>(sched);
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// launchers (called from mt_lib.cu)
// ------------------------------------------------------------------------------------------------
cudaError_t mt_launch_transport(const MtParams& P, const MtLaunchCfg& cfg, cudaStream_t stream) {
  kernel_fn fn = (P.mode == 0) ? pick_pack<0>(cfg.pack, cfg.tab_smem, cfg.sched)
                               : pick_pack<1>(cfg.pack, cfg.tab_smem, cfg.sched);
  cudaError_t e = cudaFuncSetAttribute((const void*)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.smem_bytes);
  if (e != cudaSuccess) return e;
  void* args[] = {(void*)&P};
  return cudaLaunchKernel((const void*)fn, dim3(cfg.grid), dim3(cfg.block), args, cfg.smem_bytes, stream);
}

cudaError_t mt_occupancy(const MtParams& P, const MtLaunchCfg& cfg, int* blocks_per_sm) {
  kernel_fn fn = (P.mode == 0) ? pick_pack<0>(cfg.pack, cfg.tab_smem, cfg.sched)
                               : pick_pack<1>(cfg.pack, cfg.tab_smem, cfg.sched);
  cudaError_t e = cudaFuncSetAttribute((const void*)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.smem_bytes);
  if (e != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, (const void*)fn, cfg.block, cfg.smem_bytes);
}

cudaError_t mt_launch_repack(const uint8_t* mat, const float* fld, float4* out, size_t n_cells, int* d_max_material,
                             cudaStream_t stream) {
  repack_kernel<<<148 * 8, 256, 0, stream>>>(mat, fld, out, n_cells, d_max_material);
  return cudaGetLastError();
}

cudaError_t mt_launch_debug_sample(int pack, const void* tab, uint32_t N, const uint32_t* words, uint64_t n,
                                   uint32_t* out, cudaStream_t stream) {
  if (n == 0) return cudaSuccess;
  const unsigned grid = (unsigned)((n + 255) / 256);
  if (pack == 32) debug_sample_kernel<32><<<grid, 256, 0, stream>>>((const uint32_t*)tab, N, words, n, out);
  else debug_sample_kernel<64><<<grid, 256, 0, stream>>>((const uint2*)tab, N, words, n, out);
  return cudaGetLastError();
}

cudaError_t mt_launch_debug_philox(uint32_t k0, uint32_t k1, uint64_t id_base, uint32_t step, uint64_t n,
                                   uint32_t* out, cudaStream_t stream) {
  if (n == 0) return cudaSuccess;
  debug_philox_kernel<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(k0, k1, id_base, step, n, out);
  return cudaGetLastError();
}
