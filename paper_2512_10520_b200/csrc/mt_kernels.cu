// mt_kernels.cu — the transport kernels and their launchers (sm_100a).
//
// Algorithm 1 runs under three schedules; the per-step arithmetic is
// mt_step.cuh and results do not depend on the schedule:
//   STATIC     one lane per muon for its whole life (the paper's own mapping, L59, L174);
//   REFILL     persistent warps; lanes whose muon has terminated take new muons from a global counter;
//   WAVEFRONT  one pass per z-slab over the live muons, which are re-sorted by xy cell between passes
//              (counting sort of record indices: wave_bin / wave_scan / wave_perm).  A warp then holds 32 muons of the same
//              cell column at the same z, so its eight field-corner gathers fall into one or two cache lines
//              instead of 32, and the slab's few z-layers of the 1.9 GB grid stay L1/L2-resident.
#include <cuda_runtime.h>
#include <algorithm>
#include <stdint.h>
#include "mt_launch.h"
#include "mt_step.cuh"

namespace {

using namespace mt;

enum { SCHED_STATIC = 1, SCHED_REFILL = 2, SCHED_WAVEFRONT = 3 };
constexpr int kInnerSteps = 8;        // REFILL: steps between two refill checks
constexpr unsigned kFull = 0xFFFFFFFFu;

extern __shared__ __align__(16) unsigned char mt_smem[];

template <int PACK, bool TAB_SMEM>
MT_DEV View<PACK> stage_view(const MtParams& P) {
  // const blob (edges, step lengths, axes, regions) -> shared memory, then the hot prefix of the packed tables
  float* sblob = reinterpret_cast<float*>(mt_smem);
  for (int i = threadIdx.x; i < P.bl.n_words; i += blockDim.x) sblob[i] = __ldg(P.blob + i);
  View<PACK> V;
  V.edges = sblob;
  V.edges_open = sblob + P.bl.off_edges_open;
  V.steps = sblob + P.bl.off_steps;
  V.axes = reinterpret_cast<const float4*>(sblob + P.bl.off_axes);
  V.zlo = sblob + P.bl.off_zlo;
  V.regions = reinterpret_cast<const MtRegionDev*>(sblob + P.bl.off_regions);
  V.blocks = reinterpret_cast<const MtBlockDev*>(sblob + P.bl.off_blocks);
  const uint32_t* gtab = (PACK == 32) ? P.tab32 : reinterpret_cast<const uint32_t*>(P.tab64);
  V.tab = reinterpret_cast<const typename Tab<PACK>::cell_t*>(gtab);
  uint4* stab = reinterpret_cast<uint4*>(sblob + ((P.bl.n_words + 3) & ~3));
  V.hot = reinterpret_cast<const typename Tab<PACK>::cell_t*>(stab);
  if (TAB_SMEM) {
    const uint32_t n16 = (P.hot_cells * (PACK / 8) + 15u) / 16u;          // the device array is padded to 16 bytes
    const uint4* src = reinterpret_cast<const uint4*>(gtab);
    for (uint32_t i = threadIdx.x; i < n16; i += blockDim.x) stab[i] = __ldg(src + i);
  }
  __syncthreads();
  return V;
}

// per-lane tallies of a call, reduced per warp and added to the caller's counters at kernel end
struct Tally {
  unsigned long long steps = 0;
  unsigned f1 = 0, f2 = 0, f3 = 0, f4 = 0;
  MT_DEV void count(int flag) { f1 += (flag == 1); f2 += (flag == 2); f3 += (flag == 3); f4 += (flag == 4); }
  MT_DEV void flush(unsigned long long* counters, unsigned lane) {
    if (!counters) return;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) steps += __shfl_xor_sync(kFull, steps, o);
    f1 = __reduce_add_sync(kFull, f1); f2 = __reduce_add_sync(kFull, f2);
    f3 = __reduce_add_sync(kFull, f3); f4 = __reduce_add_sync(kFull, f4);
    if (lane == 0) {
      if (steps) atomicAdd(counters + 0, steps);
      if (f1) atomicAdd(counters + 1, (unsigned long long)f1);
      if (f2) atomicAdd(counters + 2, (unsigned long long)f2);
      if (f3) atomicAdd(counters + 3, (unsigned long long)f3);
      if (f4) atomicAdd(counters + 4, (unsigned long long)f4);
    }
  }
};

// final state of a terminated muon -> dense outputs; exit-plane hits also go to the compact list through one
// atomic per warp (north_star subsystem 6).  Called by all 32 lanes; `flag` is 0 on lanes with nothing to write.
MT_DEV void write_final(const MtParams& P, const Muon& m, uint32_t idx, int flag, unsigned lane) {
  if (flag) {
    P.out_pos_flag[idx] = make_float4(m.x, m.y, m.z, __int_as_float(flag));
    P.out_mom_steps[idx] = make_float4(m.px, m.py, m.pz, __int_as_float(m.step));
  }
  if (P.exit_rec) {
    const bool ex = (flag == 2);
    const unsigned em = __ballot_sync(kFull, ex);
    if (em) {
      const int leader = __ffs(em) - 1;
      unsigned base = 0;
      if ((int)lane == leader) base = atomicAdd(P.exit_count, (unsigned)__popc(em));
      base = __shfl_sync(kFull, base, leader);
      if (ex) {
        const unsigned slot = base + (unsigned)__popc(em & ((1u << lane) - 1u));
        if (slot < P.exit_capacity) {
          P.exit_rec[2 * (size_t)slot] = make_float4(m.x, m.y, m.z, __uint_as_float(idx));
          P.exit_rec[2 * (size_t)slot + 1] = make_float4(m.px, m.py, m.pz, __int_as_float(m.step));
        }
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// STATIC and REFILL
// ------------------------------------------------------------------------------------------------
template <int GEOM, int PACK, bool TAB_SMEM, bool JOINT, int FIELD, int SCHED>
__global__ void __launch_bounds__(MT_MAX_THREADS, MT_MIN_BLOCKS)
transport_kernel(const __grid_constant__ MtParams P) {
  const View<PACK> V = stage_view<PACK, TAB_SMEM>(P);
  const unsigned lane = threadIdx.x & 31u;
  const unsigned lt_mask = (1u << lane) - 1u;
  const uint64_t n_items = P.n;

  Muon m;
  m.x = m.y = m.z = m.q = m.px = m.py = m.pz = 0.0f;
  m.step = 0;
  uint32_t idx = 0;              // muon index within this call
  bool active = false;
  bool exhausted = false;        // warp-uniform: the work counter has run past n_items
  Tally tally;

  auto load = [&](uint64_t item) {
    idx = (uint32_t)item;
    const float4 a = __ldg(P.in_pos_q + idx), b = __ldg(P.in_mom + idx);
    m.x = a.x; m.y = a.y; m.z = a.z; m.q = a.w; m.px = b.x; m.py = b.y; m.pz = b.z; m.step = 0;
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
      if (active) {
        const uint64_t id = P.id_base + idx;
        flag = step_once<GEOM, PACK, TAB_SMEM, false, JOINT, FIELD>(P, V, m, (uint32_t)id, (uint32_t)(id >> 32));
        if (flag == 0) tally.steps += 1;
      }
      write_final(P, m, idx, flag, lane);
      if (flag) {
        tally.count(flag);
        active = false;
      }
      if (!__any_sync(kFull, active)) break;
    }
    if (SCHED == SCHED_STATIC && !__any_sync(kFull, active)) break;
  }
  tally.flush(P.counters, lane);
}

// ------------------------------------------------------------------------------------------------
// WAVEFRONT: sorted z-slab passes
// ------------------------------------------------------------------------------------------------
MT_DEV uint32_t sort_key(const MtParams& P, float x, float y, float px, float py, float pz) {
  // any mapping works (the order never changes results); NaN and far-away positions land in a border cell.
  // The key is the xy cell the muon will be in after key_look metres of z on a straight line (about mid-slab), so
  // that the muons of a warp fan out around a common cell instead of away from it.
  const float t = __fdividef(P.key_look, fmaxf(pz, 0.05f));
  x = fmaf(px, t, x);
  y = fmaf(py, t, y);
  const float fx = fminf(fmaxf((x - P.key_x0) * P.key_inv, 0.0f), (float)(P.key_nx - 1));
  const float fy = fminf(fmaxf((y - P.key_y0) * P.key_inv, 0.0f), (float)(P.key_ny - 1));
  return (uint32_t)((int)fy * P.key_nx + (int)fx);
}

// pass "-1": key and rank of every input muon (the first transport pass reads the state from the caller's arrays)
__global__ void __launch_bounds__(256) wave_bin_kernel(const __grid_constant__ MtParams P) {
  const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < P.n; i += stride) {
    const float4 a = __ldg(P.in_pos_q + i), b = __ldg(P.in_mom + i);
    const uint32_t key = sort_key(P, a.x, a.y, b.x, b.y, b.z);
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
    P.perm[P.key_offset[k.x] + k.y] = i;
  }
}

template <int GEOM, int PACK, bool TAB_SMEM, bool JOINT, int FIELD, bool LEAN = false>
__global__ void __launch_bounds__(MT_MAX_THREADS, MT_MIN_BLOCKS)
wave_transport_kernel(const __grid_constant__ MtParams P) {
  const View<PACK> V = stage_view<PACK, TAB_SMEM>(P);
  const unsigned lane = threadIdx.x & 31u;
  const unsigned lt_mask = (1u << lane) - 1u;
  const uint32_t n_items = *P.live_in_count;
  Tally tally;

  for (;;) {
    // ---- the warp takes the next 32 muons of the sorted list
    unsigned long long base = 0;
    if (lane == 0) base = atomicAdd(P.work_counter, 32ull);
    base = __shfl_sync(kFull, base, 0);
    if (base >= n_items) break;
    const uint32_t item = (uint32_t)base + lane;
    Muon m;
    uint32_t idx = 0;
    int flag = -1;                                    // -1: no muon on this lane
    m.x = m.y = m.z = m.q = m.px = m.py = m.pz = 0.0f;
    m.step = 0;
    if (item < n_items) {
      const uint32_t rec = P.perm[item];
      float4 a, b;
      if (P.first_pass) {
        a = __ldg(P.in_pos_q + rec); b = __ldg(P.in_mom + rec);
        b.w = __int_as_float(0);
        idx = rec;
      } else {
        const float4* r = P.rec_in + 3 * (size_t)rec;
        a = __ldg(r); b = __ldg(r + 1);
        idx = __ldg(reinterpret_cast<const uint32_t*>(r + 2));
      }
      m.x = a.x; m.y = a.y; m.z = a.z; m.q = a.w; m.px = b.x; m.py = b.y; m.pz = b.z;
      m.step = __float_as_int(b.w);
      flag = 0;
    }
    const uint64_t id = P.id_base + idx;
    const uint32_t id_lo = (uint32_t)id, id_hi = (uint32_t)(id >> 32);
    const int step_in = m.step;

    // ---- step until every lane has terminated or reached the end of the slab
    for (;;) {
      if (flag == 0) flag = step_once<GEOM, PACK, TAB_SMEM, true, JOINT, FIELD, true, LEAN>(P, V, m, id_lo, id_hi, P.slab_z_end);
      if (!__any_sync(kFull, flag == 0)) break;
    }
    tally.steps += (unsigned)(m.step - step_in);

    // ---- terminated muons: final state; parked muons: state, sort key and rank for the next pass
    const int fin = (flag >= 1 && flag <= 4) ? flag : 0;
    write_final(P, m, idx, fin, lane);
    tally.count(fin);
    const bool parked = (flag == MT_PARK);
    const unsigned pm = __ballot_sync(kFull, parked);
    if (pm) {
      const int leader = __ffs(pm) - 1;
      unsigned slot0 = 0;
      if ((int)lane == leader) slot0 = atomicAdd(P.live_out_count, (unsigned)__popc(pm));
      slot0 = __shfl_sync(kFull, slot0, leader);
      if (parked) {
        const uint32_t key = sort_key(P, m.x, m.y, m.px, m.py, m.pz);
        const unsigned peers = __match_any_sync(pm, key);
        const int pl = __ffs(peers) - 1;
        unsigned r0 = 0;
        if ((int)lane == pl) r0 = atomicAdd(P.hist + key, (unsigned)__popc(peers));
        r0 = __shfl_sync(peers, r0, pl);
        const unsigned slot = slot0 + (unsigned)__popc(pm & lt_mask);
        float4* r = P.rec_out + 3 * (size_t)slot;                       // a warp's records are contiguous: full sectors
        r[0] = make_float4(m.x, m.y, m.z, m.q);
        r[1] = make_float4(m.px, m.py, m.pz, __int_as_float(m.step));
        r[2] = make_float4(__uint_as_float(idx), 0.0f, 0.0f, 0.0f);
        P.sort_key[slot] = make_uint2(key, r0 + (unsigned)__popc(peers & lt_mask));
      }
    }
  }
  tally.flush(P.counters, lane);
}

// ---- voxel repack: {material u8, field f32x3} -> one 32-byte record {cell x, cell x+1} per cell of a grid with a
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
    r.b = make_float4(fld[3 * s1], fld[3 * s1 + 1], fld[3 * s1 + 2], __int_as_float((int)mat[s1]));
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
  View<PACK> V;
  V.tab = tab;
  V.hot = tab;
  out[i] = draw<PACK, false>(P, V, 0u, N, words[i]);
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

typedef void (*kernel_fn)(const MtParams);

// Instantiated combinations: geometry x table kind {pack32, pack32 + shared prefix, pack64, pack64 + shared prefix,
// joint (pack64)} x field mode {trilinear / region, per-stage; voxel only: nearest, nearest per-stage} x schedule.
template <int GEOM, int PACK, bool TAB_SMEM, bool JOINT, int FIELD>
kernel_fn pick_sched(int sched) {
  switch (sched) {
    case SCHED_STATIC: return transport_kernel<GEOM, PACK, TAB_SMEM, JOINT, FIELD, SCHED_STATIC>;
    case SCHED_REFILL: return transport_kernel<GEOM, PACK, TAB_SMEM, JOINT, FIELD, SCHED_REFILL>;
    default: return wave_transport_kernel<GEOM, PACK, TAB_SMEM, JOINT, FIELD>;
  }
}
template <int GEOM, int FIELD>
kernel_fn pick_tables(const MtLaunchCfg& cfg) {
  if (cfg.joint) return pick_sched<GEOM, 64, false, true, FIELD>(cfg.sched);
  if (cfg.pack == 32) return cfg.tab_smem ? pick_sched<GEOM, 32, true, false, FIELD>(cfg.sched)
                                          : pick_sched<GEOM, 32, false, false, FIELD>(cfg.sched);
  return cfg.tab_smem ? pick_sched<GEOM, 64, true, false, FIELD>(cfg.sched)
                      : pick_sched<GEOM, 64, false, false, FIELD>(cfg.sched);
}
kernel_fn pick_kernel(int mode, const MtLaunchCfg& cfg) {
  if (cfg.lean && mt_has_lean(mode, cfg)) {
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
  if (mode == 0) return (cfg.field & 2) ? pick_tables<0, 2>(cfg) : pick_tables<0, 0>(cfg);
  if (mode == 2) return (cfg.field & 2) ? pick_tables<2, 2>(cfg) : pick_tables<2, 0>(cfg);
  switch (cfg.field & 3) {
    case 1: return pick_tables<1, 1>(cfg);
    case 2: return pick_tables<1, 2>(cfg);
    case 3: return pick_tables<1, 3>(cfg);
    default: return pick_tables<1, 0>(cfg);
  }
}

}  // namespace

bool mt_has_lean(int mode, const MtLaunchCfg& cfg) {
  return mode == 1 && cfg.sched == SCHED_WAVEFRONT && !cfg.tab_smem;
}

// ------------------------------------------------------------------------------------------------
// launchers (called from mt_lib.cu)
// ------------------------------------------------------------------------------------------------
cudaError_t mt_launch_transport(const MtParams& P, const MtLaunchCfg& cfg, cudaStream_t stream) {
  kernel_fn fn = pick_kernel(P.mode, cfg);
  cudaError_t e = cudaFuncSetAttribute((const void*)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.smem_bytes);
  if (e != cudaSuccess) return e;
  void* args[] = {(void*)&P};
  return cudaLaunchKernel((const void*)fn, dim3(cfg.grid), dim3(cfg.block), args, cfg.smem_bytes, stream);
}

cudaError_t mt_occupancy(const MtParams& P, const MtLaunchCfg& cfg, int* blocks_per_sm) {
  kernel_fn fn = pick_kernel(P.mode, cfg);
  cudaError_t e = cudaFuncSetAttribute((const void*)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.smem_bytes);
  if (e != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, (const void*)fn, cfg.block, cfg.smem_bytes);
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
  debug_philox_kernel<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(k0, k1, id_base, step, n, out);
  return cudaGetLastError();
}
