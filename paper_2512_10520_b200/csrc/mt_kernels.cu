// mt_kernels.cu — the helper kernels (index sort of the WAVEFRONT schedule, grid repack, test hooks), the choice of the
// transport kernel for a launch configuration, and all launchers (sm_100a).  The transport kernels themselves are the
// templates of mt_kernels.cuh, instantiated in the mt_inst_*.cu files.
#include <cuda_runtime.h>
#include <limits.h>
#include <stdint.h>
#include <algorithm>
#include <map>
#include <mutex>
#include <tuple>
#include <utility>
#include "mt_kernels.cuh"

namespace {

// pass "-1": key and rank of every input muon (the first transport pass reads the state from the caller's arrays)
__global__ void __launch_bounds__(256) wave_bin_kernel(const __grid_constant__ MtParams P) {
  const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < P.n; i += stride) {
    const float4 a = __ldg(P.in_pos_q + i), b = __ldg(P.in_mom + i);
    const uint32_t key = sort_key(P, a.x, a.y, b.x, b.y, b.z);
    MT_CHECK(P, key < P.n_keys, MT_CHK_SORT_KEY);
    const uint32_t rank = atomicAdd(P.hist + key, 1u);
    P.sort_key[i] = make_uint2(key, rank);
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) *P.live_out_count = (uint32_t)P.n;
}

// exclusive scan of the key histogram (one CTA; n_keys <= 2^18), which it zeroes for the next pass.  STAGE: the
// histogram passes through shared memory so that global traffic is coalesced (thread t owns `per` consecutive
// keys, `per` odd -> conflict-free); otherwise (histograms above the shared-memory size) each thread walks its
// keys in global memory.
template <bool STAGE>
__global__ void __launch_bounds__(1024) wave_scan_kernel(uint32_t* __restrict__ hist, uint32_t* __restrict__ offset,
                                                         int n_keys) {
  __shared__ uint32_t warp_sum[32];
  uint32_t* sh = reinterpret_cast<uint32_t*>(mt_smem);
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int per = ((n_keys + 1023) / 1024) | 1;
  const int k0 = min(tid * per, n_keys), k1 = min(k0 + per, n_keys);
  if (STAGE) {
    for (int k = tid; k < n_keys; k += 1024) { sh[k] = hist[k]; hist[k] = 0u; }
    __syncthreads();
  }
  const uint32_t* src = STAGE ? sh : hist;
  uint32_t sum = 0;
  for (int k = k0; k < k1; ++k) sum += src[k];
  uint32_t inc = sum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t v = __shfl_up_sync(kFull, inc, o);
    if (lane >= o) inc += v;
  }
  if (lane == 31) warp_sum[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    uint32_t w = warp_sum[lane];
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t v = __shfl_up_sync(kFull, w, o);
      if (lane >= o) w += v;
    }
    warp_sum[lane] = w;
  }
  __syncthreads();
  uint32_t run = inc - sum + (wid ? warp_sum[wid - 1] : 0u);
  if (STAGE) {
    for (int k = k0; k < k1; ++k) { const uint32_t v = sh[k]; sh[k] = run; run += v; }
    __syncthreads();
    for (int k = tid; k < n_keys; k += 1024) offset[k] = sh[k];
  } else {
    for (int k = k0; k < k1; ++k) { const uint32_t v = hist[k]; offset[k] = run; run += v; hist[k] = 0u; }
  }
}

// sorted order of the parked records: perm[first position of the key + rank within the key] = record.  The 4-byte
// scattered writes land in a 40 MB array that stays in L2; the records themselves do not move.
__global__ void __launch_bounds__(256) wave_perm_kernel(const __grid_constant__ MtParams P) {
  const uint32_t n = *P.live_out_count;
  const uint32_t stride = gridDim.x * blockDim.x;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const uint2 k = P.sort_key[i];
    MT_CHECK(P, k.x < P.n_keys, MT_CHK_SORT_KEY);
    MT_CHECK(P, P.key_offset[k.x] + k.y < n, MT_CHK_PERM_SLOT);
    P.perm[P.key_offset[k.x] + k.y] = i;
  }
}

// item-mode passes add their tallies to MT_COUNTER_SLOTS spread copies (mt_kernels.cuh: Tally::flush); this folds them into
// the caller's counters at the end of a lane's work and clears them for the next call
__global__ void reduce_counters_kernel(unsigned long long* __restrict__ spread, unsigned long long* __restrict__ counters) {
  const int c = threadIdx.x;
  if (c >= 8) return;
  unsigned long long sum = 0;
  for (int k = 0; k < MT_COUNTER_SLOTS; ++k) { sum += spread[8 * k + c]; spread[8 * k + c] = 0ull; }
  if (sum) atomicAdd(counters + c, sum);
}

// ---- voxel repack: {material u8, field f32x3} -> one 32-byte record {cell x, cell x+1 minus cell x} per cell of a grid with a
// one-cell border that replicates the faces (so the clamped corner indices of DESIGN.md §3.3 need no clamps in
// the step loop and an x-pair of corners is one load); also counts the cells of each material
__global__ void repack_kernel(const uint8_t* __restrict__ mat, const float* __restrict__ fld, MtCellPair* __restrict__ out,
                              int nx, int ny, int nz, unsigned long long* __restrict__ material_cells) {
  __shared__ unsigned hist[256];
  for (int i = threadIdx.x; i < 256; i += blockDim.x) hist[i] = 0u;
  __syncthreads();
  const int px = nx + 2, py = ny + 2;
  const size_t n_padded = (size_t)px * py * (nz + 2);
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_padded; i += (size_t)gridDim.x * blockDim.x) {
    const int x = (int)(i % px), y = (int)((i / px) % py), z = (int)(i / ((size_t)px * py));
    const int sx = min(max(x - 1, 0), nx - 1), sx1 = min(max(x, 0), nx - 1);
    const int sy = min(max(y - 1, 0), ny - 1), sz = min(max(z - 1, 0), nz - 1);
    const size_t row = ((size_t)sz * ny + sy) * nx;
    const size_t s0 = row + sx, s1 = row + sx1;
    MtCellPair r;
    r.a = make_float4(fld[3 * s0], fld[3 * s0 + 1], fld[3 * s0 + 2], __int_as_float((int)mat[s0]));
    // .b holds the x-difference of §3.3's first lerp, v(x+1) - v(x) rounded once — the very subtraction the contract
    // asks for, done here once per cell instead of once per step (0 at the replicated faces)
    r.b = make_float4(__fsub_rn(fld[3 * s1], r.a.x), __fsub_rn(fld[3 * s1 + 1], r.a.y), __fsub_rn(fld[3 * s1 + 2], r.a.z),
                      __int_as_float((int)mat[s1]));
    out[i] = r;
    if (x >= 1 && x <= nx && y >= 1 && y <= ny && z >= 1 && z <= nz) atomicAdd(&hist[mat[s0]], 1u);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < 256; i += blockDim.x)
    if (hist[i]) atomicAdd(material_cells + i, (unsigned long long)hist[i]);
}

template <int PACK>
__global__ void debug_sample_kernel(const typename Tab<PACK>::cell_t* tab, uint32_t N, const uint32_t* words,
                                    uint64_t n, uint32_t* out) {
  const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  MtParams P;                       // only hot_cells is read: nothing staged here
  P.hot_cells = 0u;
  P.check = nullptr; P.n_tab_cells = 0xFFFFFFFFu;      // checked build: the caller passes a table of N cells, k < N
  View<PACK> V;
  V.tab = tab;
  V.hot = tab;
  out[i] = draw<PACK, false>(P, V, 0u, N, words[i]);
}

// Both forms of the block: the textbook one with the key schedule inline, and the hot path's own (philox4x32_10_rk, round
// keys from the host exactly as run_transport fills them).  The hook returns the hot path's words; if the two ever
// differed it would return the textbook words XOR 0xFFFFFFFF, which no oracle comparison survives.
struct MtRoundKeys { uint32_t rk[20]; };
__global__ void debug_philox_kernel(uint32_t k0, uint32_t k1, const __grid_constant__ MtRoundKeys keys, uint64_t id_base,
                                    uint32_t step, uint64_t n, uint32_t* out) {
  const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint64_t id = id_base + i;
  uint32_t w[4], v[4];
  philox4x32_10((uint32_t)id, (uint32_t)(id >> 32), step, 0u, k0, k1, w);
  philox4x32_10_rk((uint32_t)id, (uint32_t)(id >> 32), step, 0u, keys.rk, v);
  const bool same = (w[0] == v[0]) & (w[1] == v[1]) & (w[2] == v[2]) & (w[3] == v[3]);
  reinterpret_cast<uint4*>(out)[i] = same ? make_uint4(v[0], v[1], v[2], v[3]) : make_uint4(~w[0], ~w[1], ~w[2], ~w[3]);
}

// two-word draw of the joint tables: words[i] selects, words[n + i] accepts
__global__ void debug_sample_joint_kernel(const uint2* tab, uint32_t N, const uint32_t* words, uint64_t n, uint32_t* out) {
  const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t k = __umulhi(words[i], N);
  const uint2 e = __ldg(tab + k);
  out[i] = ((words[n + i] >> 8) < e.x) ? k : e.y;
}

// test hook: material and field at arbitrary points through the same lookups as the step loop
template <int GEOM, bool NEAREST>
__global__ void __launch_bounds__(256) debug_lookup_kernel(const __grid_constant__ MtParams P, const float* __restrict__ xyz,
                                                           uint64_t n, int32_t* __restrict__ mat_out, float* __restrict__ b_out) {
  const View<32> V = stage_view<32, false>(P);
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
    const float x = xyz[3 * i], y = xyz[3 * i + 1], z = xyz[3 * i + 2];
    int material;
    float bx, by, bz;
    if (GEOM == 0) lookup_regions<32>(P, V, x, y, z, material, bx, by, bz);
    else if (GEOM == 2) lookup_poly<32>(P, V, x, y, z, material, bx, by, bz);
    else lookup_voxel<NEAREST, true>(P, x, y, z, material, bx, by, bz);
    mat_out[i] = material;
    b_out[3 * i] = bx; b_out[3 * i + 1] = by; b_out[3 * i + 2] = bz;
  }
}

mt_kernel_fn pick_kernel(int mode, const MtLaunchCfg& cfg) {
  MtLaunchCfg c = cfg;
  c.lean = cfg.lean && mt_has_lean(mode, cfg);
  if (mode == 1 && c.lean) return mt_pick_lean(c);
  if (mode == 0) return mt_pick_regions(c);
  if (mode == 2) return mt_pick_poly(c);
  return (cfg.field & 2) ? mt_pick_voxel_b(cfg) : mt_pick_voxel_a(cfg);
}

}  // namespace

bool mt_has_lean(int mode, const MtLaunchCfg& cfg) {
  const bool staged_ok = !cfg.tab_smem || (cfg.pack == 32 && !cfg.joint);
  if (mode == 1) return cfg.sched == SCHED_WAVEFRONT && staged_ok && (!cfg.tab_smem || (cfg.field & 3) == 0);
  return (cfg.sched == SCHED_REFILL || cfg.sched == SCHED_WAVEFRONT) && staged_ok;
}

// ------------------------------------------------------------------------------------------------
// launchers (called from mt_lib.cu)
// ------------------------------------------------------------------------------------------------
// Function attributes of the transport kernels.  Both the dynamic shared-memory limit and the preferred carveout are state
// of (device, kernel), shared by every context and thread of the process, and an occupancy query answers for whatever is
// set at that moment.  So what is set is tracked here per (device, kernel) under one lock, the plan of a launch
// configuration — its occupancy with shared memory unrestricted and the carveout sized from it — is worked out once per
// (device, kernel, block, shared bytes) and kept, and an attribute is written only when it has to change: after the first
// call at a configuration neither mt_occupancy nor a launch touches the attributes again (a z-slab batch used to make
// two cudaFuncSetAttribute calls per pass and five resetting probes per call).
namespace {

struct FnPlanKey {
  int device; const void* fn; unsigned block; size_t smem;
  bool operator<(const FnPlanKey& o) const {
    return std::tie(device, fn, block, smem) < std::tie(o.device, o.fn, o.block, o.smem);
  }
};
struct FnPlan { int occ, carve; };
struct FnApplied { long long smem = -1; int carve = INT_MIN; };       // what the (device, kernel) attributes hold now

std::mutex g_fn_lock;
std::map<FnPlanKey, FnPlan> g_fn_plans;
std::map<std::pair<int, const void*>, FnApplied> g_fn_applied;

cudaError_t apply_attrs(int device, const void* fn, size_t smem, int carve) {
  FnApplied& a = g_fn_applied[std::make_pair(device, fn)];
  if (a.smem != (long long)smem) {
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    a.smem = (long long)smem;
  }
  if (a.carve != carve) {
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributePreferredSharedMemoryCarveout, carve);
    if (e != cudaSuccess) return e;
    a.carve = carve;
  }
  return cudaSuccess;
}

// (caller holds g_fn_lock)
cudaError_t fn_plan(const void* fn, unsigned block, size_t smem, int* device_out, FnPlan* out) {
  int device = 0;
  cudaError_t e = cudaGetDevice(&device);
  if (e != cudaSuccess) return e;
  *device_out = device;
  const FnPlanKey key = {device, fn, block, smem};
  auto it = g_fn_plans.find(key);
  if (it != g_fn_plans.end()) { *out = it->second; return cudaSuccess; }
  // the occupancy wanted is the one with shared memory unrestricted: the carveout is sized from it
  e = apply_attrs(device, fn, smem, (int)cudaSharedmemCarveoutDefault);
  if (e != cudaSuccess) return e;
  FnPlan plan = {0, (int)cudaSharedmemCarveoutDefault};
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&plan.occ, fn, (int)block, smem);
  if (e != cudaSuccess) return e;
  // As much L1 as the resident CTAs' shared memory leaves: the alias tables live there (mt_step.cuh: MT_GRID_HINT).  The
  // carveout is a preference the driver may honour at the cost of occupancy, so it is sized for the number of CTAs that fit
  // an SM when shared memory is not restricted (1 KB per CTA is the system's own), never below that.
  int sm_bytes = 0;
  e = cudaDeviceGetAttribute(&sm_bytes, cudaDevAttrMaxSharedMemoryPerMultiprocessor, device);
  if (e != cudaSuccess) return e;
  const size_t need = (size_t)std::max(plan.occ, 1) * (smem + 1024);
  if (sm_bytes == 228 * 1024) {
    // sm_100's shared-memory configurations (KB); the preference is a percentage of the SM's 228 KB that the driver rounds
    // UP to one of them, so the smallest configuration that holds `need` is asked for by its own size rounded DOWN to a percent
    static const int kb[] = {8, 16, 32, 64, 100, 132, 164, 196, 228};
    int pick = 228;
    for (int c : kb) if ((size_t)c * 1024 >= need) { pick = c; break; }
    plan.carve = std::max(1, pick * 100 / 228);
  } else if (sm_bytes > 0) {
    // another SM: its configurations are not known here; ask for the share that holds `need` (the driver rounds up)
    plan.carve = (int)std::min<size_t>(100, std::max<size_t>(1, (need * 100 + (size_t)sm_bytes - 1) / (size_t)sm_bytes));
  }
  g_fn_plans[key] = plan;
  *out = plan;
  return cudaSuccess;
}

}  // namespace

cudaError_t mt_launch_transport(const MtParams& P, const MtLaunchCfg& cfg, cudaStream_t stream) {
  mt_kernel_fn fn = pick_kernel(P.mode, cfg);
  std::lock_guard<std::mutex> lock(g_fn_lock);              // attributes and launch as one step: another thread's launch of
  int device = 0;                                           // the same kernel may want other values
  FnPlan plan;
  cudaError_t e = fn_plan((const void*)fn, cfg.block, cfg.smem_bytes, &device, &plan);
  if (e != cudaSuccess) return e;
  e = apply_attrs(device, (const void*)fn, cfg.smem_bytes, plan.carve);
  if (e != cudaSuccess) return e;
  void* args[] = {(void*)&P};
  return cudaLaunchKernel((const void*)fn, dim3(cfg.grid), dim3(cfg.block), args, cfg.smem_bytes, stream);
}

cudaError_t mt_occupancy(const MtParams& P, const MtLaunchCfg& cfg, int* blocks_per_sm) {
  mt_kernel_fn fn = pick_kernel(P.mode, cfg);
  std::lock_guard<std::mutex> lock(g_fn_lock);
  int device = 0;
  FnPlan plan;
  cudaError_t e = fn_plan((const void*)fn, cfg.block, cfg.smem_bytes, &device, &plan);
  if (e != cudaSuccess) return e;
  *blocks_per_sm = plan.occ;
  return cudaSuccess;
}

cudaError_t mt_launch_wave_bin(const MtParams& P, unsigned grid, cudaStream_t stream) {
  wave_bin_kernel<<<grid, 256, 0, stream>>>(P);
  return cudaGetLastError();
}

cudaError_t mt_launch_wave_sort(const MtParams& P, int n_keys, unsigned grid, cudaStream_t stream) {
  const size_t stage_b = (size_t)n_keys * sizeof(uint32_t);
  cudaError_t e;
  if (stage_b <= 200 * 1024) {
    e = cudaFuncSetAttribute((const void*)wave_scan_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)stage_b);
    if (e != cudaSuccess) return e;
    wave_scan_kernel<true><<<1, 1024, stage_b, stream>>>(P.hist, P.key_offset, n_keys);
  } else {
    wave_scan_kernel<false><<<1, 1024, 0, stream>>>(P.hist, P.key_offset, n_keys);
  }
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  wave_perm_kernel<<<grid, 256, 0, stream>>>(P);
  return cudaGetLastError();
}

cudaError_t mt_launch_reduce_counters(unsigned long long* spread, unsigned long long* counters, cudaStream_t stream) {
  reduce_counters_kernel<<<1, 32, 0, stream>>>(spread, counters);
  return cudaGetLastError();
}

cudaError_t mt_launch_repack(const uint8_t* mat, const float* fld, MtCellPair* out, int nx, int ny, int nz,
                             unsigned long long* d_material_cells, cudaStream_t stream) {
  repack_kernel<<<148 * 8, 256, 0, stream>>>(mat, fld, out, nx, ny, nz, d_material_cells);
  return cudaGetLastError();
}

cudaError_t mt_launch_debug_sample(int pack, bool joint, const void* tab, uint32_t N, const uint32_t* words, uint64_t n,
                                   uint32_t* out, cudaStream_t stream) {
  if (n == 0) return cudaSuccess;
  const unsigned grid = (unsigned)((n + 255) / 256);
  if (joint) debug_sample_joint_kernel<<<grid, 256, 0, stream>>>((const uint2*)tab, N, words, n, out);
  else if (pack == 32) debug_sample_kernel<32><<<grid, 256, 0, stream>>>((const uint32_t*)tab, N, words, n, out);
  else debug_sample_kernel<64><<<grid, 256, 0, stream>>>((const uint2*)tab, N, words, n, out);
  return cudaGetLastError();
}

cudaError_t mt_launch_debug_lookup(const MtParams& P, size_t smem_bytes, const float* xyz, uint64_t n, int32_t* mat_out,
                                   float* b_out, cudaStream_t stream) {
  if (n == 0) return cudaSuccess;
  typedef void (*fn_t)(const MtParams, const float*, uint64_t, int32_t*, float*);
  fn_t fn = (P.mode == 0) ? debug_lookup_kernel<0, false>
          : (P.mode == 2) ? debug_lookup_kernel<2, false>
          : (P.field_mode & 1) ? debug_lookup_kernel<1, true> : debug_lookup_kernel<1, false>;
  cudaError_t e = cudaFuncSetAttribute((const void*)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
  if (e != cudaSuccess) return e;
  const unsigned grid = (unsigned)std::min<uint64_t>((n + 255) / 256, 148 * 8);
  fn<<<grid, 256, smem_bytes, stream>>>(P, xyz, n, mat_out, b_out);
  return cudaGetLastError();
}

cudaError_t mt_launch_debug_philox(uint32_t k0, uint32_t k1, uint64_t id_base, uint32_t step, uint64_t n,
                                   uint32_t* out, cudaStream_t stream) {
  if (n == 0) return cudaSuccess;
  MtRoundKeys keys;
  for (uint32_t r = 0; r < 10; ++r) {                       // as run_transport fills MtParams::rk
    keys.rk[2 * r] = k0 + r * 0x9E3779B9u;
    keys.rk[2 * r + 1] = k1 + r * 0xBB67AE85u;
  }
  debug_philox_kernel<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(k0, k1, keys, id_base, step, n, out);
  return cudaGetLastError();
}
