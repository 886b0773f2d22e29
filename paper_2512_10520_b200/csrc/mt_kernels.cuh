// mt_kernels.cuh — the transport kernels as templates (sm_100a), included by the translation units that instantiate
// them: mt_inst_regions.cu, mt_inst_voxel_a.cu, mt_inst_voxel_b.cu, mt_inst_poly.cu, mt_inst_lean.cu (split so that they
// compile in parallel) and by mt_kernels.cu for the staging helper.
//
// Algorithm 1 runs under three schedules; the per-step arithmetic is
// mt_step.cuh and results do not depend on the schedule:
//   STATIC     one lane per muon for its whole life (the paper's own mapping, L59, L174);
//   REFILL     persistent warps; lanes whose muon has terminated take new muons from a global counter;
//   WAVEFRONT  one pass per z-slab over the live muons, which are re-sorted by xy cell between passes
//              (counting sort of record indices: wave_bin / wave_scan / wave_perm in mt_kernels.cu).  A warp then
//              holds 32 muons of the same cell column at the same z, so its eight field-corner gathers fall into one
//              or two cache lines instead of 32, and the slab's few z-layers of the 3.9 GB grid stay L1/L2-resident.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "mt_launch.h"
#include "mt_step.cuh"

namespace {

using namespace mt;

enum { SCHED_STATIC = 1, SCHED_REFILL = 2, SCHED_WAVEFRONT = 3 };
// Muon records stream: a pass reads each once and writes each survivor once, 480 MB at the first pass against 126 MB of
// L2 that should keep the slab's field layers, so they go through cache-streaming (evict-first) loads and stores
// (ld.global.cs / st.global.cs: 142.6 -> 142.1 ms per 10^7 muons; -DMT_NO_STREAM restores plain accesses).
#ifndef MT_NO_STREAM
#define MT_LD(p) __ldcs(p)
#define MT_ST(p, v) __stcs(p, v)
#else
#define MT_LD(p) __ldg(p)
#define MT_ST(p, v) (*(p) = (v))
#endif
constexpr int kInnerSteps = 8;        // REFILL: steps between two refill checks
constexpr unsigned kFull = 0xFFFFFFFFu;

extern __shared__ __align__(16) unsigned char mt_smem[];

template <int PACK, bool TAB_SMEM>
MT_DEV View<PACK> stage_view(const MtParams& P) {
  // const blob (edges, step lengths, axes, regions) -> shared memory, then the hot prefix of the packed tables
  // (the per-table axes, by far the largest part, are NOT staged: one 128-bit read-only load per step serves them from
  // L1, and a CTA then starts after copying ~1.5 KB instead of ~7 KB — what makes small CTAs and item-mode passes cheap)
  float* sblob = reinterpret_cast<float*>(mt_smem);
  const int cut = MT_AXES_GLOBAL ? P.bl.off_zlo - P.bl.off_axes : 0;      // words of the blob that are not staged (a multiple of 4)
  for (int i = threadIdx.x; i < P.bl.n_words; i += blockDim.x) {
    if (i < P.bl.off_axes) sblob[i] = __ldg(P.blob + i);
    else if (i >= P.bl.off_zlo) sblob[i - cut] = __ldg(P.blob + i);
    else if (!MT_AXES_GLOBAL) sblob[i] = __ldg(P.blob + i);
  }
  View<PACK> V;
  V.edges = sblob;
  V.edges_open = sblob + P.bl.off_edges_open;
  V.steps = sblob + P.bl.off_steps;
  V.axes = MT_AXES_GLOBAL ? reinterpret_cast<const float4*>(P.blob + P.bl.off_axes)
                          : reinterpret_cast<const float4*>(sblob + P.bl.off_axes);
  V.zlo = sblob + (P.bl.off_zlo - cut);
  V.regions = reinterpret_cast<const MtRegionDev*>(sblob + (P.bl.off_regions - cut));
  V.blocks = reinterpret_cast<const MtBlockDev*>(sblob + (P.bl.off_blocks - cut));
  V.binlut = reinterpret_cast<const uint16_t*>(sblob + (P.bl.off_binlut - cut));
  V.zlut = reinterpret_cast<const int16_t*>(sblob + (P.bl.off_zlut - cut));
  const uint32_t* gtab = (PACK == 32) ? P.tab32 : reinterpret_cast<const uint32_t*>(P.tab64);
  V.tab = reinterpret_cast<const typename Tab<PACK>::cell_t*>(gtab);
  uint4* stab = reinterpret_cast<uint4*>(sblob + ((MT_STAGED_WORDS(P.bl) + 3) & ~3));
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
#ifdef MT_SLOT_STATS
  // diagnostic build (-DMT_SLOT_STATS; profiles/r2c_summary.md): lane-steps a WAVEFRONT pass had room for, and where the
  // unused ones went.  counters[5] += 32 x (steps of the item's slowest lane), [6] += steps that lanes whose muon
  // terminated in the item sat out, [7] += steps that parked lanes waited for the slowest one
  unsigned slots = 0, idle_fin = 0, idle_park = 0;
  MT_DEV void slot_stats(unsigned own, bool fin, bool parked) {
    const unsigned mx = __reduce_max_sync(kFull, own);
    slots += mx; idle_fin += fin ? mx - own : 0u; idle_park += parked ? mx - own : 0u;
  }
#endif
  MT_DEV void count(int flag) { f1 += (flag == 1); f2 += (flag == 2); f3 += (flag == 3); f4 += (flag == 4); }
  // `spread`: slot of 8 counters to add to (item-mode kernels flush once per warp-item, hundreds of thousands of times
  // per pass: the adds are spread over MT_COUNTER_SLOTS copies and summed by reduce_counters_kernel at the end of the call)
  MT_DEV void flush(unsigned long long* counters, unsigned lane, unsigned spread = 0) {
    if (!counters) return;
    counters += 8 * spread;
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
#ifdef MT_SLOT_STATS
    slots = __reduce_add_sync(kFull, slots); idle_fin = __reduce_add_sync(kFull, idle_fin); idle_park = __reduce_add_sync(kFull, idle_park);
    if (lane == 0) {
      atomicAdd(counters + 5, (unsigned long long)slots); atomicAdd(counters + 6, (unsigned long long)idle_fin);
      atomicAdd(counters + 7, (unsigned long long)idle_park);
    }
#endif
  }
};

// final state of a terminated muon -> dense outputs; exit-plane hits also go to the compact list through one
// atomic per warp (north_star subsystem 6).  Called by all 32 lanes; `flag` is 0 on lanes with nothing to write.
MT_DEV void write_final(const MtParams& P, const Muon& m, uint32_t idx, int flag, unsigned lane) {
  if (flag) {
    MT_CHECK(P, idx < P.n, MT_CHK_OUTPUT);
    MT_ST(P.out_pos_flag + idx, make_float4(m.x, m.y, m.z, __int_as_float(flag)));
    MT_ST(P.out_mom_steps + idx, make_float4(m.px, m.py, m.pz, __int_as_float(m.step)));
  }
  if (P.exit_count) {
    // the counter advances for every exit-plane hit (a caller may pass exit_count alone to count them); records are
    // written while there is a list and room in it
    const bool hit = (flag == 2);
    const unsigned em = __ballot_sync(kFull, hit);
    if (em) {
      const int leader = __ffs(em) - 1;
      unsigned base = 0;
      if ((int)lane == leader) base = atomicAdd(P.exit_count, (unsigned)__popc(em));
      base = __shfl_sync(kFull, base, leader);
      const unsigned slot = base + (unsigned)__popc(em & ((1u << lane) - 1u));
      if (hit && P.exit_rec && slot < P.exit_capacity) {
        float ex = m.x, ey = m.y, ez = m.z;
        if (P.exit_mode == 1 && m.pz > 0.0f) {
          // §3.13: back onto the plane along the final direction (one IEEE division, two fma)
          const float s = __fdiv_rn(mt::sub(m.z, P.z_exit), m.pz);
          ex = mt::fma(-s, m.px, m.x); ey = mt::fma(-s, m.py, m.y); ez = P.z_exit;
        }
        P.exit_rec[2 * (size_t)slot] = make_float4(ex, ey, ez, __uint_as_float(idx + P.idx_base));
        P.exit_rec[2 * (size_t)slot + 1] = make_float4(m.px, m.py, m.pz, __int_as_float(m.step));
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// STATIC and REFILL
// ------------------------------------------------------------------------------------------------
template <int GEOM, int PACK, bool TAB_SMEM, bool JOINT, int FIELD, int SCHED, bool LEAN = false>
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
    MT_CHECK(P, item < P.n, MT_CHK_INPUT);
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

    // ---- a few steps for every active lane; the loop itself stays warp-uniform.  Nothing but the step happens on a step
    // in which no lane of the warp terminates (one vote tells).
#pragma unroll 1
    for (int k = 0; k < kInnerSteps; ++k) {
      int flag = 0;
      if (active) {
        // two steps per warp vote, as in the z-slab passes
        const uint64_t id = P.id_base + idx;
        flag = step_once<GEOM, PACK, TAB_SMEM, false, JOINT, FIELD, true, LEAN>(P, V, m, (uint32_t)id, (uint32_t)(id >> 32));
        if (flag == 0) {
          tally.steps += 1;
          flag = step_once<GEOM, PACK, TAB_SMEM, false, JOINT, FIELD, true, LEAN>(P, V, m, (uint32_t)id, (uint32_t)(id >> 32));
          if (flag == 0) tally.steps += 1;
        }
      }
      if (__any_sync(kFull, flag != 0)) {
        write_final(P, m, idx, flag, lane);
        if (flag) {
          tally.count(flag);
          active = false;
        }
        if (!__any_sync(kFull, active)) break;
      }
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

template <int GEOM, int PACK, bool TAB_SMEM, bool JOINT, int FIELD, bool LEAN = false>
__global__ void __launch_bounds__(MT_MAX_THREADS, MT_MIN_BLOCKS)
wave_transport_kernel(const __grid_constant__ MtParams P) {
  const uint32_t n_items = *P.live_in_count;
  // item mode (P.persistent == 0): warp w of CTA b owns the 32 muons from (b * warps + w) * 32 and the CTA exits when its
  // warps are done, so that the CTAs of another lane's pass (or of this lane's sort) take the freed slots at once; the
  // grid covers the lane's muon count, CTAs beyond the live count leave before staging anything
  const unsigned warps_per_cta = blockDim.x >> 5;
  if (!P.persistent && (uint64_t)blockIdx.x * warps_per_cta * 32u >= n_items) return;
  const View<PACK> V = stage_view<PACK, TAB_SMEM>(P);
  const unsigned lane = threadIdx.x & 31u;
  const unsigned lt_mask = (1u << lane) - 1u;
  Tally tally;
  bool first = true;

  for (;;) {
    // ---- the warp takes the next 32 muons of the sorted list
    unsigned long long base = 0;
    if (P.persistent) {
      if (lane == 0) base = atomicAdd(P.work_counter, 32ull);
      base = __shfl_sync(kFull, base, 0);
    } else {
      if (!first) break;
      first = false;
      base = ((unsigned long long)blockIdx.x * warps_per_cta + (threadIdx.x >> 5)) * 32ull;
    }
    if (base >= n_items) break;
    const uint32_t item = (uint32_t)base + lane;
    Muon m;
    uint32_t idx = 0;
    int flag = -1;                                    // -1: no muon on this lane
    m.x = m.y = m.z = m.q = m.px = m.py = m.pz = 0.0f;
    m.step = 0;
    if (item < n_items) {
      MT_CHECK(P, item < P.n, MT_CHK_PERM);
      const uint32_t rec = P.sorted_in ? P.perm[item] : item;      // unsorted pass: the records in the order they were parked
      MT_CHECK(P, rec < (P.first_pass ? P.n : (uint64_t)n_items), MT_CHK_RECORD);
      float4 a, b;
      if (P.first_pass) {
        a = MT_LD(P.in_pos_q + rec); b = MT_LD(P.in_mom + rec);
        b.w = __int_as_float(0);
        idx = rec;
      } else {
        const float4* r = P.rec_in + 3 * (size_t)rec;
        a = MT_LD(r); b = MT_LD(r + 1);
        idx = MT_LD(reinterpret_cast<const uint32_t*>(r + 2));
        MT_CHECK(P, idx < P.n, MT_CHK_RECORD);
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
      if (flag == 0) flag = step_once<GEOM, PACK, TAB_SMEM, true, JOINT, FIELD, true, LEAN>(P, V, m, id_lo, id_hi, P.slab_z_end);
      if (!__any_sync(kFull, flag == 0)) break;
    }
    tally.steps += (unsigned)(m.step - step_in);

    // ---- terminated muons: final state; parked muons: state, sort key and rank for the next pass
    const int fin = (flag >= 1 && flag <= 4) ? flag : 0;
    write_final(P, m, idx, fin, lane);
    tally.count(fin);
    const bool parked = (flag == MT_PARK);
#ifdef MT_SLOT_STATS
    tally.slot_stats((unsigned)(m.step - step_in), fin != 0, parked);
#endif
    const unsigned pm = __ballot_sync(kFull, parked);
    if (pm) {
      const int leader = __ffs(pm) - 1;
      unsigned slot0 = 0;
      if ((int)lane == leader) slot0 = atomicAdd(P.live_out_count, (unsigned)__popc(pm));
      slot0 = __shfl_sync(kFull, slot0, leader);
      if (parked) {
        const unsigned slot = slot0 + (unsigned)__popc(pm & lt_mask);
        MT_CHECK(P, slot < P.n, MT_CHK_PARK_SLOT);
        float4* r = P.rec_out + 3 * (size_t)slot;                       // a warp's records are contiguous: full sectors
        MT_ST(r, make_float4(m.x, m.y, m.z, m.q));
        MT_ST(r + 1, make_float4(m.px, m.py, m.pz, __int_as_float(m.step)));
        MT_ST(r + 2, make_float4(__uint_as_float(idx), 0.0f, 0.0f, 0.0f));
        if (P.sort_out) {                                               // the next pass reads them sorted: key and rank
          const uint32_t key = sort_key(P, m.x, m.y, m.px, m.py, m.pz);
          MT_CHECK(P, key < P.n_keys, MT_CHK_SORT_KEY);
          const unsigned peers = __match_any_sync(pm, key);
          const int pl = __ffs(peers) - 1;
          unsigned r0 = 0;
          if ((int)lane == pl) r0 = atomicAdd(P.hist + key, (unsigned)__popc(peers));
          r0 = __shfl_sync(peers, r0, pl);
          P.sort_key[slot] = make_uint2(key, r0 + (unsigned)__popc(peers & lt_mask));
        }
      }
    }
  }
  tally.flush(P.persistent ? P.counters : P.counters_spread, lane, P.persistent ? 0u : (blockIdx.x & (MT_COUNTER_SLOTS - 1)));
}

// Instantiated combinations: geometry x table kind {pack32, pack32 + shared prefix, pack64, pack64 + shared prefix,
// joint (pack64)} x field mode {trilinear / region, per-stage; voxel only: nearest, nearest per-stage} x schedule.
template <int GEOM, int PACK, bool TAB_SMEM, bool JOINT, int FIELD>
mt_kernel_fn pick_sched(int sched) {
  switch (sched) {
    case SCHED_STATIC: return transport_kernel<GEOM, PACK, TAB_SMEM, JOINT, FIELD, SCHED_STATIC>;
    case SCHED_REFILL: return transport_kernel<GEOM, PACK, TAB_SMEM, JOINT, FIELD, SCHED_REFILL>;
    default: return wave_transport_kernel<GEOM, PACK, TAB_SMEM, JOINT, FIELD>;
  }
}
template <int GEOM, int FIELD>
mt_kernel_fn pick_tables(const MtLaunchCfg& cfg) {
  if (cfg.joint) return pick_sched<GEOM, 64, false, true, FIELD>(cfg.sched);
  if (cfg.pack == 32) return cfg.tab_smem ? pick_sched<GEOM, 32, true, false, FIELD>(cfg.sched)
                                          : pick_sched<GEOM, 32, false, false, FIELD>(cfg.sched);
  return cfg.tab_smem ? pick_sched<GEOM, 64, true, false, FIELD>(cfg.sched)
                      : pick_sched<GEOM, 64, false, false, FIELD>(cfg.sched);
}
// LEAN variants of a region / polyhedra geometry (MT_LEAN_AXES only): REFILL and WAVEFRONT; joint, 8-byte or 4-byte
// cells from L2, 4-byte cells staged in shared memory (mt_has_lean)
template <int GEOM, int PACK, bool TAB_SMEM, bool JOINT, int FIELD>
mt_kernel_fn pick_sched_lean(int sched) {
  if (sched == SCHED_REFILL) return transport_kernel<GEOM, PACK, TAB_SMEM, JOINT, FIELD, SCHED_REFILL, true>;
  return wave_transport_kernel<GEOM, PACK, TAB_SMEM, JOINT, FIELD, true>;
}
template <int GEOM, int FIELD>
mt_kernel_fn pick_tables_lean(const MtLaunchCfg& cfg) {
  if (cfg.joint) return pick_sched_lean<GEOM, 64, false, true, FIELD>(cfg.sched);
  if (cfg.pack == 32) return cfg.tab_smem ? pick_sched_lean<GEOM, 32, true, false, FIELD>(cfg.sched)
                                          : pick_sched_lean<GEOM, 32, false, false, FIELD>(cfg.sched);
  return pick_sched_lean<GEOM, 64, false, false, FIELD>(cfg.sched);
}

}  // namespace
